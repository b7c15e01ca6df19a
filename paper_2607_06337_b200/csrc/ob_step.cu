// ob_step.cu -- k_step, the product kernel (sm_100a): n physics steps of every world in one launch.
//
// One CTA per world in flight (persistent, work queue per size class), three CTAs of 128 threads per SM at the
// headline size.  Everything the level-synchronous tree sweeps touch lives in SHARED MEMORY as one 112-byte
// record of seven float4 per link (stride 7 x 16 B: 128-bit accesses of consecutive links are conflict-free),
// so the sweep code exists once, is about a thousand instructions long (it has to stay inside the instruction
// cache: the first versions of this kernel were no_instruction-stalled) and runs over any number of links.
// The apple block is staged by one TMA bulk copy (UBLKCP) and written back the same way; q, qd and the PCG start
// vectors stay in global memory (L2): only the once-per-step phases touch them.
//
//   A0  flat:      joint transforms R_rel = Q Rx Ry (Eq. 3) in fp64; E = R_rel^T rounded for the dynamics
//   A1  top-down:  forward kinematics in fp64 (world rotations and positions), hang points of the apples
//   A2  top-down:  velocities, bias accelerations, bias force of every link incl. tether reactions (Eq. 6 / Eq. 7,
//                  PAPER.md:149-161) and user wrenches; leaves finish at once
//   B1  bottom-up: bias torques of the inner links -> rhs b
//   B2  bottom-up: composite inertia -> exact diagonal of M for the Jacobi preconditioner (every kDiagRefresh-th
//                  step; in between the stored diagonal + the current spring-damper terms), effective link inertia
//   C   matrix-free Jacobi-PCG on (M + M_teth + diag(arm + hD + h^2 K)) dqd = b  (north_star), started from the
//                  cubic extrapolation of the last four solutions; M v = acceleration-only inverse dynamics:
//                  top-down a_i, bottom-up f_i, project on S_i
//   D   integrate joints and apples; rupture (Eq. 5) and detach predicates
//
// Order.  Links are in plain breadth-first order: levels contiguous, the children of a link contiguous.  In the
// PCG sweeps the leading levels that fit into 32 links (n_top of them) are swept by ONE warp, lane = link, own
// record in registers, parents and children by shuffle, no barrier; every other level ends with one block
// barrier; only the deepest level turns around inside the top-down pass (all of its links are leaves).  In the
// once-per-step sweeps warp 0 takes the leading levels with __syncwarp and every leaf turns around.
//
// Record of link i (P[7 i + j]); record Np is never written and stays zero: the trunk's parent, missing children.
//   0, 1  M0, M1   A0: R_rel (fp64); A1: world rotation R (fp64 for an inner link, fp32 for a leaf); A2: parked bias
//                  force / (n, f) for the parent; B2: composite inertia for the parent; C: (alpha, a) on the way
//                  down, (n, f) on the way up, A p in M1.zw
//   2     PD       (p, diagonal terms arm + (h c_d + h^2) K); A0, A1: more of R_rel, R; B2 borrows .xy
//   3..5  C0..C2   E (parent -> link rotation, row-major), c2, s2, parent length
//   6     C3       effective link inertia (m, m c, I about the joint, I_zz) incl. on-axis virtual tether masses
//                  (A15); A0, A1: the rest of R_rel, R
// Beside the records: G (float2: the ninth entry of R_rel / R as a double, then b, then 1 / diag(A)), T (packed topology word:
// parent | first child << 11 | children << 22 | flags), and one region shared by the A2 overflow (12 floats per
// inner link: velocity and bias acceleration for the children) and the PCG's (x, r) (one float4 per link).
//
// Spatial vectors are [angular; linear at the link origin] in link coordinates.  Link frame: origin at the
// proximal joint, +z along the link.  Joint i: R_rel = Q_i Rx(theta1) Ry(theta2); E_i = R_rel^T maps parent
// coordinates to link coordinates; the joint sits at r = (0,0,L_parent) in the parent frame.
#include <math.h>

#include "ob_device.h"
#include "ob_internal.h"

namespace ob {

// packed topology word
constexpr uint32_t kParMask = 0x7ffu, kChShift = 11, kNcShift = 22, kNcMask = 0xfu;
constexpr uint32_t kHasApples = 1u << 26, kOffax = 1u << 27, kSnapped = 1u << 28, kRuptured = 1u << 29, kTrunk = 1u << 30;

// ------------------------------------------------------------------------------------------------------
// shared-memory view of one world
// ------------------------------------------------------------------------------------------------------
struct Sm {
  int Np, Ap, NIp;
  float4 *P;                          // records: P[7 * i + j], j = 0 M0, 1 M1, 2 PD, 3..5 C0..C2, 6 C3
  float2 *G;
  uint32_t *T;
  float4 *ovf;                        // ovf[j * NIp + inner slot], j = 0..2
  float4 *XR;                         // [Np] (x, r) of the PCG; same memory as ovf (phase A2 / B1 only)
  int *lev;                           // level offsets [n_levels + 1]
  // apple block (TMA)
  float *u, *v;                       // [3][Ap]
  unsigned char *att, *cA, *cB;
  float *ao, *ak, *am, *ac, *afd;     // ao = [3][Ap]
  float *ft, *fsn;                    // tether force [3][Ap], |f_s| [Ap] (phase A2 -> phase D)
  float *hd;                          // [6][Ap] anchor - x_hang of every apple, fp64 as (hi, lo) pairs (phase A1 -> A2);
                                      // aliases ft, fsn (see carve)
  WrenchSlots *wr;
};

// The functions that are not inlined carve the CTA's dynamic shared memory again from the sizes (World) instead of
// taking pointers: pointers handed over through memory are generic, and the sweeps then run on LD.E / ST.E with
// 64-bit address arithmetic instead of LDS / STS.
extern __shared__ __align__(128) unsigned char ob_smem[];

__device__ __forceinline__ Sm carve(unsigned char *base, const int Np, const int Ap, const int NIp, const int n_levels) {
  Sm s;
  s.Np = Np; s.Ap = Ap; s.NIp = NIp;
  unsigned char *p = base;
  s.P = reinterpret_cast<float4 *>(p); p += step_planes_bytes(Np);
  s.G = reinterpret_cast<float2 *>(p); p += r16(8 * (Np + 1));
  s.T = reinterpret_cast<uint32_t *>(p); p += r16(4 * (Np + 1));
  s.ovf = reinterpret_cast<float4 *>(p); s.XR = s.ovf; p += step_ovf_bytes(Np, NIp);
  s.lev = reinterpret_cast<int *>(p); p += r16(4 * (n_levels + 1));
  float *f = reinterpret_cast<float *>(p);
  s.u = f; s.v = f + 3 * Ap;
  s.att = p + 24 * Ap; s.cA = s.att + Ap; s.cB = s.cA + Ap;
  f = reinterpret_cast<float *>(p + apple_state_bytes(Ap));
  s.ao = f; s.ak = f + 3 * Ap; s.am = f + 4 * Ap; s.ac = f + 5 * Ap; s.afd = f + 6 * Ap;
  p += r16(apple_block_bytes(Ap));
  f = reinterpret_cast<float *>(p);
  s.ft = f; f += 3 * Ap;
  s.fsn = f; f += Ap;
  s.hd = s.ft; f += 2 * Ap;             // hd[0..3] share the memory of ft[0..2], fsn: per apple, phase A2 reads hd, then writes them
  s.wr = reinterpret_cast<WrenchSlots *>(f);
  return s;
}

// per-link data of one world in global memory (L2-resident; only the once-per-step phases read it)
struct Gm {
  float2 *q2, *w2;                  // state (link block)
  unsigned char *rupt, *rc;
  const float4 *c4;                 // (m, m c, I about the joint, I_zz)
  const float *K, *rz;              // joint stiffness (Eq. 4), parent length
  const double2 *quatd;             // rest quaternions, normalised, fp64: (w, x), (y, z) of link i at 2 i, 2 i + 1
  const double *anchor;             // [k * Ap + a] rest hang points, world frame, fp64
  const float *Mmax;
  float2 *mdiag;                    // diag(M) as last computed by phase B2 (the Jacobi preconditioner may lag)
  float2 *hist;                     // [4][sum_np]: dqd of the last four steps, slot = step & 3
  const float *arm;                 // [k * Np + i] or nullptr
  const int4 *topo2;                // x = first apple | n_apples << 16, y = inner slot | parent's inner slot << 16
};

// block-wide sum of two values, result broadcast to every thread; one barrier per call (double-buffered stage)
template <int NT>
struct Reducer {
  float2 *stage;   // [2][32]
  int flip, tid;   // tid = the thread's LOGICAL index (otid): the sum must not depend on which warp is the top warp
  __device__ __forceinline__ float2 sum(float a, float b) {
    // five shuffles for the pair: the two halves of the warp trade a for b first
    const bool hi = (tid & 16) != 0;
    const float send = hi ? a : b;
    const float got = __shfl_xor_sync(0xffffffffu, send, 16);
    float v = (hi ? b : a) + got;              // lanes 0..15 carry a, lanes 16..31 carry b
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    float *st = reinterpret_cast<float *>(stage + 32 * flip);
    flip ^= 1;
    if ((tid & 15) == 0) st[2 * (tid >> 5) + (hi ? 1 : 0)] = v;
    __syncthreads();
    float sa = 0.f, sb = 0.f;
    if (NT % 64 == 0) {
      const float4 *s4 = reinterpret_cast<const float4 *>(st);
#pragma unroll
      for (int k = 0; k < NT / 64; k++) { const float4 t = s4[k]; sa += t.x + t.z; sb += t.y + t.w; }
    } else {
      const float2 *s2 = reinterpret_cast<const float2 *>(st);
#pragma unroll
      for (int k = 0; k < NT / 32; k++) { const float2 t = s2[k]; sa += t.x; sb += t.y; }
    }
    return make_float2(sa, sb);
  }
};

__device__ __forceinline__ void push_event(const DevCtx &c, int world, int step, int kind, int index, float value,
                                           float thr) {
  const int slot = atomicAdd(c.ev_count, 1);
  if (slot < c.ev_cap) {
    ob_event e;
    e.world = world; e.step = step; e.kind = kind; e.index = index; e.value = value; e.threshold = thr;
    c.events[slot] = e;
  } else {
    c.ev_count[1] = 1;
  }
}

// joint transform of one link as the sweeps use it
struct Jt {
  M3 E;                // parent -> link rotation
  float c2, s2, rz;
};
__device__ __forceinline__ Jt load_jt(const float4 *P, const int i) {
  const float4 e0 = P[7 * i + 3], e1 = P[7 * i + 4], e2 = P[7 * i + 5];
  Jt j;
  j.E.a[0] = e0.x; j.E.a[1] = e0.y; j.E.a[2] = e0.z; j.E.a[3] = e0.w;
  j.E.a[4] = e1.x; j.E.a[5] = e1.y; j.E.a[6] = e1.z; j.E.a[7] = e1.w;
  j.E.a[8] = e2.x; j.c2 = e2.y; j.s2 = e2.z; j.rz = e2.w;
  return j;
}
__device__ __forceinline__ void store_jt(float4 *P, const int i, const Jt &j) {
  P[7 * i + 3] = make_float4(j.E.a[0], j.E.a[1], j.E.a[2], j.E.a[3]);
  P[7 * i + 4] = make_float4(j.E.a[4], j.E.a[5], j.E.a[6], j.E.a[7]);
  P[7 * i + 5] = make_float4(j.E.a[8], j.c2, j.s2, j.rz);
}

// ------------------------------------------------------------------------------------------------------
// phase C: A v for one link.  mv_down: accelerations from the parent (the trunk reads the zero column).
// mv_up: f = I a + children, project on S (+ diagonal terms) -> A p (M1[i].zw), publish (n, f) in the parent
// frame; returns p . (A p) of this link.  Mailbox: M0[i] = (x, y, z of the angular part, x of the linear part),
// M1[i].xy = (y, z of the linear part).
// ------------------------------------------------------------------------------------------------------
// virtual tether masses off the link axis (rare: the workloads hang apples on the axis), one by one.  Everything
// goes in and out by value so that nothing of the caller is forced into local memory.
struct Force6 { float3 n, f; };
__device__ __noinline__ Force6 offaxis_tethers(const int4 t2, const float3 al, const float3 a, const unsigned char *att,
                                               const float *ao, const float *ak, const int Ap, const float hh) {
  Force6 r;
  r.n = f3(0, 0, 0); r.f = f3(0, 0, 0);
  const int ast = t2.x & 0xffff, nap = t2.x >> 16;
  for (int q = ast; q < ast + nap; q++) {
    if (!att[q]) continue;
    const float3 o = f3(ao[q], ao[Ap + q], ao[2 * Ap + q]);
    if (o.x == 0.f && o.y == 0.f) continue;                 // already inside (m, mc, Io)
    const float mv = hh * ak[q];
    const float3 fp = mv * (a + cross(al, o));
    r.f = r.f + fp;
    r.n = r.n + cross(o, fp);
  }
  return r;
}

__device__ __forceinline__ void mv_down(const Jt &j, const float4 *P, const uint32_t tw, const float4 pd, float3 &al,
                                        float3 &a) {
  const float4 *par = P + 7 * (int)(tw & kParMask);
  const float4 u = par[0], v = par[1];
  const float3 alp = f3(u.x, u.y, u.z), ap = f3(u.w, v.x, v.y);
  al = mul(j.E, alp) + f3(j.c2 * pd.x, pd.y, j.s2 * pd.x);
  a = mul(j.E, f3(ap.x + alp.y * j.rz, ap.y - alp.x * j.rz, ap.z));
}

// children of a link out of shared memory, added in ascending order: the first four with all loads in flight
// at once (a missing child reads the zero record), the rest one by one
__device__ __forceinline__ void gather_children(const float4 *P, const float4 *zero_rec, const int fc, const int nc,
                                                float3 &n, float3 &f) {
  const float4 *ch = P + 7 * fc;
  float4 cu[4], cv[4];
#pragma unroll
  for (int k = 0; k < 4; k++) {
    const float4 *q = k < nc ? ch + 7 * k : zero_rec;
    cu[k] = q[0]; cv[k] = q[1];
  }
#pragma unroll
  for (int k = 0; k < 4; k++) {
    n = n + f3(cu[k].x, cu[k].y, cu[k].z);
    f = f + f3(cu[k].w, cv[k].x, cv[k].y);
  }
#pragma unroll 1
  for (int k = 4; k < nc; k++) {
    const float4 u = ch[7 * k], v = ch[7 * k + 1];
    n = n + f3(u.x, u.y, u.z);
    f = f + f3(u.w, v.x, v.y);
  }
}

template <bool GATHER>
__device__ __forceinline__ float mv_up(const Jt &j, float4 *P, const float4 *zero_rec, const int i, const uint32_t tw,
                                       const float4 pd, const float3 al, const float3 a, const Sm &s, const Gm &g,
                                       const DevCtx &c) {
  float4 *rec = P + 7 * i;
  const float4 I = rec[6];                                    // (m, m c, I about the joint, I_zz)
  float3 n = f3(I.z * al.x - I.y * a.y, I.z * al.y + I.y * a.x, I.w * al.z);
  float3 f = f3(I.x * a.x + I.y * al.y, I.x * a.y - I.y * al.x, I.x * a.z);
  if (tw & kOffax) {
    const Force6 t = offaxis_tethers(__ldg(g.topo2 + i), al, a, s.att, s.ao, s.ak, s.Ap, c.P.h * c.P.h);
    n = n + t.n; f = f + t.f;
  }
  if (GATHER) gather_children(P, zero_rec, (int)((tw >> kChShift) & kParMask), (int)((tw >> kNcShift) & kNcMask), n, f);
  const float t1 = j.c2 * n.x + j.s2 * n.z + pd.z * pd.x;     // pd = (p0, p1, dt0, dt1)
  const float t2 = n.y + pd.w * pd.y;
  const float3 fp = mulT(j.E, f);                             // the trunk publishes into its own column, which nobody reads
  float3 np = mulT(j.E, n);
  np.x -= j.rz * fp.y; np.y += j.rz * fp.x;
  rec[0] = make_float4(np.x, np.y, np.z, fp.x);
  rec[1] = make_float4(fp.y, fp.z, t1, t2);
  return pd.x * t1 + pd.y * t2;
}

// ------------------------------------------------------------------------------------------------------
// The once-per-step phases, cut into passes that each keep a small working set in registers (a spilled
// register costs an L2 round trip here: the three CTAs of an SM leave the L1 only ~28 KB):
//   A0  flat      per link, no dependence on other links: R_rel = Q Rx Ry in fp64 (-> slots 0, 1, 2, 6, G),
//                 E = R_rel^T rounded (-> C0..C2)
//   A1  top-down  FK in fp64: R, p of every link (an inner link publishes twelve doubles: slots 0, 1, 2, 6, G and the
//                 overflow), hang points of the apples (-> hd), snapped flags
//   A2  top-down  velocities and bias accelerations (inner links publish 12 floats in the overflow); own bias
//                 force of every link incl. tethers and wrenches; a leaf finishes at once, an inner link
//                 parks (n, f) in M0, M1.xy
//   B1  bottom-up inner links: own (n, f) + children -> rhs b (-> G), (n, f) for the parent
// ------------------------------------------------------------------------------------------------------

// the views of the world every thread of the CTA shares (in shared memory, filled once per world)
struct World { Gm g; int N, Np, Ap, NIp, nlev, ntop; };
__device__ __forceinline__ Sm carve(const World *wd) { return carve(ob_smem, wd->Np, wd->Ap, wd->NIp, wd->nlev); }
// PCG start vector: cubic extrapolation of the last four solutions (x1 = the latest)
#define OB_X0(x1, x2, x3, x4) (4.f * ((x1) + (x3)) - 6.f * (x2) - (x4))

// a double carried as two floats (hi + lo): 48 bits, plenty for a displacement summed along <= 2000 links
__device__ __forceinline__ float2 split2(const double v) {
  const float hi = (float)v;
  return make_float2(hi, (float)(v - (double)hi));
}
__device__ __forceinline__ double join2(const float hi, const float lo) { return (double)hi + (double)lo; }

// ---- A0 ----  R_rel = Q Rx(th1) Ry(th2) of one link in fp64 -> the link's own record slots 0, 1, 2, 6 and G (they are
//               free until the link's turn in A1); E = R_rel^T rounded to fp32, cos / sin th2 and the parent length
//               -> C0..C2 for the dynamics
__device__ __forceinline__ void link_joint(const int i, const Sm &s, const Gm &g) {
  const float2 th = __ldcg(g.q2 + i);
  const double2 qa = __ldg(g.quatd + 2 * i), qb = __ldg(g.quatd + 2 * i + 1);
  const float rzf = (s.T[i] & kTrunk) ? 0.f : __ldg(g.rz + i);
  double Q[9], X[9], Rrel[9];
  {
    const double w = qa.x, x = qa.y, y = qb.x, z = qb.y;
    Q[0] = 1 - 2 * (y * y + z * z); Q[1] = 2 * (x * y - w * z);     Q[2] = 2 * (x * z + w * y);
    Q[3] = 2 * (x * y + w * z);     Q[4] = 1 - 2 * (x * x + z * z); Q[5] = 2 * (y * z - w * x);
    Q[6] = 2 * (x * z - w * y);     Q[7] = 2 * (y * z + w * x);     Q[8] = 1 - 2 * (x * x + y * y);
  }
  double s1, c1, s2, c2;
  sincos((double)th.x, &s1, &c1);
  sincos((double)th.y, &s2, &c2);
  X[0] = c2;       X[1] = 0.0; X[2] = s2;                           // Rx(th1) Ry(th2)
  X[3] = s1 * s2;  X[4] = c1;  X[5] = -s1 * c2;
  X[6] = -c1 * s2; X[7] = s1;  X[8] = c1 * c2;
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int cc = 0; cc < 3; cc++) Rrel[3 * r + cc] = Q[3 * r] * X[cc] + Q[3 * r + 1] * X[3 + cc] + Q[3 * r + 2] * X[6 + cc];
  Jt j;                                                              // E = Rrel^T, rounded once
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int cc = 0; cc < 3; cc++) j.E.a[3 * r + cc] = (float)Rrel[3 * cc + r];
  j.c2 = (float)c2; j.s2 = (float)s2; j.rz = rzf;
  store_jt(s.P, i, j);
  double2 *pr = reinterpret_cast<double2 *>(s.P + 7 * i);
  pr[0] = make_double2(Rrel[0], Rrel[1]); pr[1] = make_double2(Rrel[2], Rrel[3]); pr[2] = make_double2(Rrel[4], Rrel[5]);
  pr[6] = make_double2(Rrel[6], Rrel[7]);
  *reinterpret_cast<double *>(s.G + i) = Rrel[8];
}

// ---- A1 ----  forward kinematics in fp64 (Eq. 3): R_i = R_p Q_i Rx(th1) Ry(th2),
//               p_i = p_p + R_p (0,0,L_p).  The tether stretch x_a - x_hang is a millimetre-sized difference of
//               metre-sized positions, k_s = 2e3 N/m turns 1e-8 m of it into the whole error budget of a 3 mm twig:
//               rest rotations, sin / cos of the joint angles and the chain of products are therefore fp64, and the
//               hang point of every apple is formed here, where the fp64 pose is at hand.  The dynamics get the
//               fp32-rounded joint transform E = R_rel^T.
// Publish of an inner link for its children (twelve doubles): R[0..7] in the record slots 0, 1, 2, 6, R[8] in G,
// p in the overflow slot.  A leaf keeps its fp32 rotation in slots 0, 1, 2.x for phase A2.
__device__ __forceinline__ void link_fk(const int i, const Sm &s, const Gm &g) {
  float4 *rec = s.P + 7 * i;
  uint32_t tw = s.T[i];
  const int4 t2 = __ldg(g.topo2 + i);
  const bool trunk = (tw & kTrunk) != 0u;
  double Rrel[9];                                   // Q Rx(th1) Ry(th2) in fp64: phase A0 left it in the link's own slots
  {
    const double2 *pr = reinterpret_cast<const double2 *>(rec);
    const double2 a0 = pr[0], a1 = pr[1], a2 = pr[2], a3 = pr[6];
    Rrel[0] = a0.x; Rrel[1] = a0.y; Rrel[2] = a1.x; Rrel[3] = a1.y; Rrel[4] = a2.x; Rrel[5] = a2.y; Rrel[6] = a3.x;
    Rrel[7] = a3.y; Rrel[8] = *reinterpret_cast<const double *>(s.G + i);
  }
  const float rzf = rec[5].w;                       // parent length (0 for the trunk), stored with E by phase A0
  double Rp[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1}, pp[3] = {0, 0, 0};
  uint32_t snapped_p = 0u;
  if (!trunk) {
    const int par = (int)(tw & kParMask), ps = (int)((uint32_t)t2.y >> 16);
    const double2 *pr = reinterpret_cast<const double2 *>(s.P + 7 * par);
    const double2 a0 = pr[0], a1 = pr[1], a2 = pr[2], a3 = pr[6];
    Rp[0] = a0.x; Rp[1] = a0.y; Rp[2] = a1.x; Rp[3] = a1.y; Rp[4] = a2.x; Rp[5] = a2.y; Rp[6] = a3.x; Rp[7] = a3.y;
    Rp[8] = *reinterpret_cast<const double *>(s.G + par);
    const double2 b0 = *reinterpret_cast<const double2 *>(s.ovf + ps);
    pp[0] = b0.x; pp[1] = b0.y; pp[2] = *reinterpret_cast<const double *>(s.ovf + s.NIp + ps);
    snapped_p = s.T[par] & kSnapped;
  }
  double R[9], pw[3];
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int cc = 0; cc < 3; cc++) R[3 * r + cc] = Rp[3 * r] * Rrel[cc] + Rp[3 * r + 1] * Rrel[3 + cc] + Rp[3 * r + 2] * Rrel[6 + cc];
  const double rz = (double)rzf;
  pw[0] = pp[0] + rz * Rp[2]; pw[1] = pp[1] + rz * Rp[5]; pw[2] = pp[2] + rz * Rp[8];
  tw = (tw & ~kSnapped) | (((tw & kRuptured) || snapped_p) ? kSnapped : 0u);
  s.T[i] = tw;
  // hang points of the apples on this link: anchor - x_hang (the anchor is the rest hang point, fp64)
  if (tw & kHasApples) {
    const int Ap = s.Ap, ast = t2.x & 0xffff, nap = t2.x >> 16;
    for (int a = ast; a < ast + nap; a++) {
      const double ox = s.ao[a], oy = s.ao[Ap + a], oz = s.ao[2 * Ap + a];
#pragma unroll
      for (int k = 0; k < 3; k++) {
        const double xh = pw[k] + R[3 * k] * ox + R[3 * k + 1] * oy + R[3 * k + 2] * oz;
        const float2 dd = split2(__ldg(g.anchor + (size_t)k * Ap + a) - xh);
        s.hd[(2 * k) * Ap + a] = dd.x; s.hd[(2 * k + 1) * Ap + a] = dd.y;
      }
    }
  }
  if ((tw >> kNcShift) & kNcMask) {
    const int is = t2.y & 0xffff;
    double2 *pr = reinterpret_cast<double2 *>(rec);
    pr[0] = make_double2(R[0], R[1]); pr[1] = make_double2(R[2], R[3]); pr[2] = make_double2(R[4], R[5]);
    pr[6] = make_double2(R[6], R[7]);
    *reinterpret_cast<double *>(s.G + i) = R[8];
    *reinterpret_cast<double2 *>(s.ovf + is) = make_double2(pw[0], pw[1]);
    *reinterpret_cast<double *>(s.ovf + s.NIp + is) = pw[2];
  } else {
    rec[0] = make_float4((float)R[0], (float)R[1], (float)R[2], (float)R[3]);
    rec[1] = make_float4((float)R[4], (float)R[5], (float)R[6], (float)R[7]);
    rec[2] = make_float4((float)R[8], 0.f, 0.f, 0.f);
  }
}

// tether reactions (Eq. 6 / Eq. 7) and user wrenches on one link, subtracted from its bias
// force (n, f); also leaves the tether force and |f_s| of each apple for phase D.  Only links that carry apples or
// a wrench come here.
// (Not inlined.  It takes the World in shared memory, not references to the caller's copies: a reference would
// force those copies into local memory, and every pointer fetched from there is an L2 round trip.)
__device__ __noinline__ Force6 external_forces(const int i, const float3 om, const float3 vl, const uint32_t tw,
                                               const int apples, const World *wd, const DevCtx &c) {
  const Sm s = carve(wd);
  const ob_params &P = c.P;
  const int Ap = s.Ap;
  Force6 out;
  out.n = f3(0, 0, 0); out.f = f3(0, 0, 0);
  M3 R;                                   // world rotation of the link (phase A1): fp64 publish of an inner link, fp32 of a leaf
  if ((tw >> kNcShift) & kNcMask) {
    const double2 *pr = reinterpret_cast<const double2 *>(s.P + 7 * i);
    const double2 a0 = pr[0], a1 = pr[1], a2 = pr[2], a3 = pr[6];
    R.a[0] = (float)a0.x; R.a[1] = (float)a0.y; R.a[2] = (float)a1.x; R.a[3] = (float)a1.y; R.a[4] = (float)a2.x;
    R.a[5] = (float)a2.y; R.a[6] = (float)a3.x; R.a[7] = (float)a3.y;
    R.a[8] = (float)*reinterpret_cast<const double *>(s.G + i);
  } else {
    const float4 *rec = s.P + 7 * i;
    const float4 r0 = rec[0], r1 = rec[1];
    R.a[0] = r0.x; R.a[1] = r0.y; R.a[2] = r0.z; R.a[3] = r0.w;
    R.a[4] = r1.x; R.a[5] = r1.y; R.a[6] = r1.z; R.a[7] = r1.w; R.a[8] = rec[2].x;
  }
  const int ast = apples & 0xffff, nap = apples >> 16;          // first apple | count << 16 (topo2.x, loaded by the caller)
  const float eta_h = P.tether_implicit ? P.h : 0.f;
  for (int a = ast; a < ast + nap; a++) {
    if (!s.att[a]) continue;
    const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
    const float ks = s.ak[a], cdamp = s.ac[a], ma = s.am[a];
    // x_a - x_hang = (anchor - x_hang) + sag + u: the apple is stored as u = x_a - (anchor + sag), sag = m g / k_s,
    // and phase A1 left anchor - x_hang in fp64 (as two floats)
    const double mk = (double)ma / (double)ks;               // one fp64 division; sag = (m / k_s) g to ~1e-19 m of m g / k_s
    const float3 st = f3((float)(join2(s.hd[a], s.hd[Ap + a]) + mk * (double)P.gravity[0] + (double)s.u[a]),
                         (float)(join2(s.hd[2 * Ap + a], s.hd[3 * Ap + a]) + mk * (double)P.gravity[1] + (double)s.u[Ap + a]),
                         (float)(join2(s.hd[4 * Ap + a], s.hd[5 * Ap + a]) + mk * (double)P.gravity[2] + (double)s.u[2 * Ap + a]));
    const float3 vh = mul(R, vl + cross(om, o));                          // world velocity of the hang point
    const float3 fs = (-ks) * st;
    const float3 va = f3(s.v[a], s.v[Ap + a], s.v[2 * Ap + a]);
    s.ft[a] = fs.x - cdamp * va.x; s.ft[Ap + a] = fs.y - cdamp * va.y; s.ft[2 * Ap + a] = fs.z - cdamp * va.z;
    s.fsn[a] = sqrtf(dot(fs, fs));
    float3 fr = f3(ks * (st.x - eta_h * vh.x) - ma * P.gravity[0], ks * (st.y - eta_h * vh.y) - ma * P.gravity[1],
                   ks * (st.z - eta_h * vh.z) - ma * P.gravity[2]);
    const float nr = sqrtf(dot(fr, fr));
    if (nr > P.react_max) fr = (P.react_max / nr) * fr;                   // clamp
    const float3 fl = mulT(R, fr);
    out.f = out.f - fl;
    out.n = out.n - cross(o, fl);
  }
  // user wrenches on this link (disabled on snapped sub-trees)
  const int nwr = s.wr->n;
  for (int q = 0; q < nwr; q++) {
    if (s.wr->body[q] != i) continue;
    if ((tw & kSnapped) && P.forces_off_on_snapped) continue;
    const float3 fl = mulT(R, f3(s.wr->force[q][0], s.wr->force[q][1], s.wr->force[q][2]));
    const float3 pt = f3(s.wr->point[q][0], s.wr->point[q][1], s.wr->point[q][2]);
    out.f = out.f - fl;
    out.n = out.n - cross(pt, fl);
  }
  return out;
}

// project the accumulated bias force on the joint axes -> rhs b (G[i]), the diagonal terms of both DoF (PD[i].zw),
// and publish (n, f) in the parent frame (M0[i], M1[i].xy)
// (th, w, Ki = q, qd, K of the joint: the caller loads them at the top of its turn, with its other global inputs)
__device__ __forceinline__ void finish_bias(const Jt &j, const int i, const uint32_t tw, const float2 th, const float2 w,
                                            const float Ki, float3 n, float3 f, const Sm &s, const Gm &g,
                                            const DevCtx &c) {
  const ob_params &P = c.P;
  float4 *rec = s.P + 7 * i;
  // spring-damper part of the rhs and of the diagonal (Eq. 4); a ruptured joint has K = D = 0
  const float Kt = (tw & kRuptured) ? 0.f : Ki, Dt = P.c_d * Kt;
  const float2 kq = make_float2(Kt * th.x + (Dt + P.h * Kt) * w.x, Kt * th.y + (Dt + P.h * Kt) * w.y);
  s.G[i] = make_float2(P.h * (-(j.c2 * n.x + j.s2 * n.z) - kq.x), P.h * (-n.y - kq.y));
  float dt0 = (P.h * P.c_d + P.h * P.h) * Kt, dt1 = dt0;
  if (g.arm) {
    dt0 += __ldg(g.arm + i);
    dt1 += __ldg(g.arm + s.Np + i);
  }
  reinterpret_cast<float2 *>(rec + 2)[1] = make_float2(dt0, dt1);            // arm + (h c_d + h^2) K per DoF
  if (!(tw & kTrunk)) {
    const float3 fp = mulT(j.E, f);
    float3 np = mulT(j.E, n);
    np.x -= j.rz * fp.y; np.y += j.rz * fp.x;
    rec[0] = make_float4(np.x, np.y, np.z, fp.x);
    *reinterpret_cast<float2 *>(rec + 1) = make_float2(fp.y, fp.z);
  }
}

// ---- A2 ----  velocity, bias acceleration (gravity as base acceleration), own bias force
//               f = I a + v x* I v - tether reactions - user wrenches  (RNEA with qdd = 0)
__device__ __forceinline__ void link_bias(const int i, const World *wd, const Sm &s, const Gm &g, const DevCtx &c) {
  const ob_params &P = c.P;
  const int NIp = s.NIp;
  const uint32_t tw = s.T[i];
  const float2 w = __ldcg(g.w2 + i), th = __ldcg(g.q2 + i);       // all global inputs of the link's turn at once
  const float4 c4 = __ldg(g.c4 + i);
  const float Ki = __ldg(g.K + i);
  const int4 t2g = __ldg(g.topo2 + i);
  const int ty = t2g.y;                                           // inner slot | parent's inner slot << 16
  const Jt j = load_jt(s.P, i);
  float3 wp = f3(0, 0, 0), vp = f3(0, 0, 0), alp = f3(0, 0, 0);
  float3 ap = f3(-P.gravity[0], -P.gravity[1], -P.gravity[2]);   // world = parent of the trunk: at rest, (0; -g)
  if (!(tw & kTrunk)) {
    const int ps = (int)((uint32_t)ty >> 16);
    const float4 t0 = s.ovf[ps], t1 = s.ovf[NIp + ps], t2 = s.ovf[2 * NIp + ps];
    wp = f3(t0.x, t0.y, t0.z); vp = f3(t0.w, t1.x, t1.y);
    alp = f3(t1.z, t1.w, t2.x); ap = f3(t2.y, t2.z, t2.w);
  }
  const float rz = j.rz, c2 = j.c2, s2 = j.s2;
  const float3 vJ = f3(c2 * w.x, w.y, s2 * w.x);
  const float3 om = mul(j.E, wp) + vJ;
  const float3 vl = mul(j.E, f3(vp.x + wp.y * rz, vp.y - wp.x * rz, vp.z));
  const float ww = w.x * w.y;
  // mass-proportional damping (A32): its generalized force -alpha M qd enters the bias pass as the
  // joint acceleration alpha qd, i.e. alpha S qd = alpha vJ on top of the velocity-product terms
  const float3 al = mul(j.E, alp) + f3(-s2 * ww, 0.f, c2 * ww) + cross(om, vJ) + P.mass_damping * vJ;
  const float3 aln = mul(j.E, f3(ap.x + alp.y * rz, ap.y - alp.x * rz, ap.z)) + cross(vl, vJ);
  const bool inner = ((tw >> kNcShift) & kNcMask) != 0u;
  if (inner) {
    const int is = ty & 0xffff;
    s.ovf[is] = make_float4(om.x, om.y, om.z, vl.x);
    s.ovf[NIp + is] = make_float4(vl.y, vl.z, al.x, al.y);
    s.ovf[2 * NIp + is] = make_float4(al.z, aln.x, aln.y, aln.z);
  }
  // f = I a + v x* I v  (cylinder: com on +z)
  const float m = c4.x, mc = c4.y, Io = c4.z, Iz = c4.w;
  float3 n = f3(Io * al.x - mc * aln.y, Io * al.y + mc * aln.x, Iz * al.z);
  float3 f = f3(m * aln.x + mc * al.y, m * aln.y - mc * al.x, m * aln.z);
  const float3 hn = f3(Io * om.x - mc * vl.y, Io * om.y + mc * vl.x, Iz * om.z);
  const float3 hf = f3(m * vl.x + mc * om.y, m * vl.y - mc * om.x, m * vl.z);
  n = n + cross(om, hn) + cross(vl, hf);
  f = f + cross(om, hf);
  bool ext = (tw & kHasApples) != 0u;
  for (int q = 0; q < s.wr->n; q++) ext |= s.wr->body[q] == i;
  if (ext) {
    const Force6 e = external_forces(i, om, vl, tw, t2g.x, wd, c);
    n = n + e.n; f = f + e.f;
  }
  if (inner) {                                                    // parked until B1 adds the children
    s.P[7 * i] = make_float4(n.x, n.y, n.z, f.x);
    *reinterpret_cast<float2 *>(s.P + 7 * i + 1) = make_float2(f.y, f.z);
  } else {
    finish_bias(j, i, tw, th, w, Ki, n, f, s, g, c);
  }
}

// ---- B1 ----  one inner link: its parked bias force plus what its children sent up
__device__ __forceinline__ void link_bias_up(const int i, const uint32_t tw, const Sm &s, const Gm &g, const DevCtx &c) {
  const float2 th = __ldcg(g.q2 + i), w = __ldcg(g.w2 + i);
  const float Ki = __ldg(g.K + i);
  const float4 u0 = s.P[7 * i];
  const float2 v0 = *reinterpret_cast<const float2 *>(s.P + 7 * i + 1);
  float3 n = f3(u0.x, u0.y, u0.z), f = f3(u0.w, v0.x, v0.y);
  gather_children(s.P, s.P + 7 * s.Np, (int)((tw >> kChShift) & kParMask), (int)((tw >> kNcShift) & kNcMask), n, f);
  finish_bias(load_jt(s.P, i), i, tw, th, w, Ki, n, f, s, g, c);
}

// ------------------------------------------------------------------------------------------------------
// phase B2 for one link: composite rigid-body inertia about the link origin (mass, first moment h, symmetric
// I) -> exact diagonal of M -> Jacobi factors (G[i]); effective link inertia for A v (C3[i]); publish the
// composite inertia in the parent frame (M0[i], M1[i], PD[i].xy)
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void up_inertia(const int i, const Sm &s, const Gm &g, const DevCtx &c) {
  const int Ap = s.Ap;
  const ob_params &P = c.P;
  uint32_t tw = s.T[i];
  float4 c4 = __ldg(g.c4 + i);
  {                                  // mass-proportional damping, implicit: the operator carries (1 + h alpha) M
    const float sc = 1.f + P.h * P.mass_damping;
    c4.x *= sc; c4.y *= sc; c4.z *= sc; c4.w *= sc;
  }
  float cm = c4.x;
  float3 ch3 = f3(0.f, 0.f, c4.y);
  float Ixx = c4.z, Iyy = c4.z, Izz = c4.w, Ixy = 0.f, Ixz = 0.f, Iyz = 0.f;
  float4 eff = c4;
  if (P.tether_implicit && (tw & kHasApples)) {
    tw &= ~kOffax;
    const int4 t2 = __ldg(g.topo2 + i);
    const int ast = t2.x & 0xffff, nap = t2.x >> 16;
    for (int a = ast; a < ast + nap; a++) {
      if (!s.att[a]) continue;
      const float mv = P.h * P.h * s.ak[a];                     // virtual point mass h^2 k_s at the hang point
      const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
      cm += mv; ch3 = ch3 + mv * o;
      Ixx += mv * (o.y * o.y + o.z * o.z); Iyy += mv * (o.x * o.x + o.z * o.z); Izz += mv * (o.x * o.x + o.y * o.y);
      Ixy -= mv * o.x * o.y; Ixz -= mv * o.x * o.z; Iyz -= mv * o.y * o.z;
      if (o.x == 0.f && o.y == 0.f) { eff.x += mv; eff.y += mv * o.z; eff.z += mv * o.z * o.z; }   // stays a body of revolution
      else tw |= kOffax;
    }
    s.T[i] = tw;
  }
  s.P[7 * i + 6] = eff;
  const int fc = (int)((tw >> kChShift) & kParMask), nc = (int)((tw >> kNcShift) & kNcMask);
  for (int ch = fc; ch < fc + nc; ch++) {
    const float4 u0 = s.P[7 * ch];
    const float4 u1 = s.P[7 * ch + 1];
    const float2 u2 = *reinterpret_cast<const float2 *>(s.P + 7 * ch + 2);
    cm += u0.x;
    ch3 = ch3 + f3(u0.y, u0.z, u0.w);
    Ixx += u1.x; Iyy += u1.y; Izz += u1.z; Ixy += u1.w; Ixz += u2.x; Iyz += u2.y;
  }
  const Jt j = load_jt(s.P, i);
  const float c2 = j.c2, s2 = j.s2;
  const float2 dt = reinterpret_cast<const float2 *>(s.P + 7 * i + 2)[1];
  const float m1 = c2 * c2 * Ixx + 2.f * c2 * s2 * Ixz + s2 * s2 * Izz, m2 = Iyy;
  g.mdiag[i] = make_float2(m1, m2);
  float2 id = make_float2(1.f, 1.f);
  if (P.precond == 1) id = make_float2(1.f / (m1 + dt.x), 1.f / (m2 + dt.y));
  s.G[i] = id;
  if (!(tw & kTrunk)) {
    const M3 &E = j.E;
    const float rz = j.rz;
    // composite inertia into the parent frame: rotate by Rrel = E^T, then move the origin by r = (0,0,rz)
    const float3 hp = mulT(E, ch3);
    M3 I, T, Ip;
    I.a[0] = Ixx; I.a[1] = Ixy; I.a[2] = Ixz; I.a[3] = Ixy; I.a[4] = Iyy; I.a[5] = Iyz; I.a[6] = Ixz; I.a[7] = Iyz; I.a[8] = Izz;
#pragma unroll
    for (int r = 0; r < 3; r++)
#pragma unroll
      for (int cc = 0; cc < 3; cc++) T.a[3 * r + cc] = E.a[r] * I.a[cc] + E.a[3 + r] * I.a[3 + cc] + E.a[6 + r] * I.a[6 + cc];
    Ip = mul(T, E);
    const float sh = 2.f * rz * hp.z + cm * rz * rz;
    s.P[7 * i] = make_float4(cm, hp.x, hp.y, hp.z + cm * rz);
    s.P[7 * i + 1] = make_float4(Ip.a[0] + sh, Ip.a[4] + sh, Ip.a[8], Ip.a[1]);
    *reinterpret_cast<float2 *>(s.P + 7 * i + 2) = make_float2(Ip.a[2] - rz * hp.x, Ip.a[5] - rz * hp.y);
  }
}

// phase B2 on the steps between two recomputations of diag(M): the effective link inertia (it is part of A and must
// be exact: it changes when an apple detaches, and phase A1 borrows its slot) and the Jacobi factors from the stored
// diag(M) plus the CURRENT diagonal spring-damper terms.  A lagging preconditioner changes the number of PCG
// iterations, never the system that is solved.
__device__ __forceinline__ void link_inertia_lagged(const int i, float4 eff, const float2 md, const Sm &s, const Gm &g,
                                                    const DevCtx &c) {
  const ob_params &P = c.P;
  const int Ap = s.Ap;
  uint32_t tw = s.T[i];
  {
    const float sc = 1.f + P.h * P.mass_damping;
    eff.x *= sc; eff.y *= sc; eff.z *= sc; eff.w *= sc;
  }
  if (P.tether_implicit && (tw & kHasApples)) {
    tw &= ~kOffax;
    const int4 t2 = __ldg(g.topo2 + i);
    const int ast = t2.x & 0xffff, nap = t2.x >> 16;
    for (int a = ast; a < ast + nap; a++) {
      if (!s.att[a]) continue;
      const float mv = P.h * P.h * s.ak[a];
      const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
      if (o.x == 0.f && o.y == 0.f) { eff.x += mv; eff.y += mv * o.z; eff.z += mv * o.z * o.z; }
      else tw |= kOffax;
    }
    s.T[i] = tw;
  }
  s.P[7 * i + 6] = eff;
  const float2 dt = reinterpret_cast<const float2 *>(s.P + 7 * i + 2)[1];
  float2 id = make_float2(1.f, 1.f);
  if (P.precond == 1) id = make_float2(1.f / (md.x + dt.x), 1.f / (md.y + dt.y));
  s.G[i] = id;
}

// fence after level l of a top-down sweep / after level l of a bottom-up sweep (see "Order" above)
#define OB_FENCE_DOWN(l) { if ((l) + 1 < ntop) __syncwarp(); else __syncthreads(); }
#define OB_FENCE_UP(l) { if ((l) < ntop) __syncwarp(); else __syncthreads(); }

// ------------------------------------------------------------------------------------------------------
// the once-per-step sweeps as functions of their own (not inlined): their register pressure (24 kinematic
// quantities per link in flight) stays out of the allocation of the PCG loop.  The views of the world live in
// shared memory (World), the context is the kernel's __grid_constant__ parameter.
// ------------------------------------------------------------------------------------------------------
#define OB_COLD_ATTR __noinline__

__device__ OB_COLD_ATTR void sweep_bias(const World *wd, const DevCtx &c, const int nt) {
  const Sm s = carve(wd);
  const Gm g = wd->g;
  const int nlev = wd->nlev, ntop = wd->ntop, tid = threadIdx.x;
  const int l_first_down = tid < 32 ? 0 : ntop - 1, l_last_up = tid < 32 ? 0 : ntop;
  // ---- A0: joint transforms in fp64, flat (the two double sincos and Q Rx Ry are the expensive part of the FK and
  //      depend on nothing but the link's own q: kept out of the level-by-level chain) ----
#pragma unroll 1
  for (int i = tid; i < wd->N; i += nt) link_joint(i, s, g);
  __syncthreads();
  // ---- A1: forward kinematics in fp64, joint transforms, hang points, top-down ----
#pragma unroll 1
  for (int l = l_first_down; l < nlev; l++) {
    const int le = s.lev[l + 1];
#pragma unroll 1
    for (int i = s.lev[l] + tid; i < le; i += nt) link_fk(i, s, g);
    OB_FENCE_DOWN(l)
  }
  // ---- A2 (+ B1 for leaves): velocities, bias accelerations, bias forces, top-down ----
#pragma unroll 1
  for (int l = l_first_down; l < nlev; l++) {
    const int le = s.lev[l + 1];
#pragma unroll 1
    for (int i = s.lev[l] + tid; i < le; i += nt) link_bias(i, wd, s, g, c);
    OB_FENCE_DOWN(l)
  }
  // ---- B1: bias forces bottom-up over the inner links -> rhs b ----
#pragma unroll 1
  for (int l = nlev - 2; l >= l_last_up; l--) {
    const int le = s.lev[l + 1];
#pragma unroll 1
    for (int i = s.lev[l] + tid; i < le; i += nt) {
      const uint32_t tw = s.T[i];
      if ((tw >> kNcShift) & kNcMask) link_bias_up(i, tw, s, g, c);
    }
    OB_FENCE_UP(l)
  }
  __syncthreads();
}

__device__ OB_COLD_ATTR void sweep_inertia(const World *wd, const DevCtx &c, const int nt, const int otid,
                                           const bool refresh) {
  const Sm s = carve(wd);
  const Gm g = wd->g;
  const int nlev = wd->nlev, ntop = wd->ntop, N = wd->N, tid = threadIdx.x;
  if (!refresh) {
#pragma unroll 1
    for (int i0 = otid; i0 < N; i0 += 4 * nt) {          // four links per trip to L2
      float4 c4v[4];
      float2 mdv[4];
#pragma unroll
      for (int k = 0; k < 4; k++) {
        const int i = min(i0 + k * nt, N - 1);
        c4v[k] = __ldg(g.c4 + i); mdv[k] = __ldcg(g.mdiag + i);
      }
#pragma unroll
      for (int k = 0; k < 4; k++)
        if (i0 + k * nt < N) link_inertia_lagged(i0 + k * nt, c4v[k], mdv[k], s, g, c);
    }
    __syncthreads();
    return;
  }
  const int l_last_up = tid < 32 ? 0 : ntop;
  // ---- B2: composite inertia bottom-up -> Jacobi factors, effective inertia (all leaves first) ----
#pragma unroll 1
  for (int i = otid; i < N; i += nt)                       // flat ownership: G[i] was just read by this thread
    if (((s.T[i] >> kNcShift) & kNcMask) == 0u) up_inertia(i, s, g, c);
  __syncthreads();
#pragma unroll 1
  for (int l = nlev - 2; l >= l_last_up; l--) {
    const int le = s.lev[l + 1];
#pragma unroll 1
    for (int i = s.lev[l] + tid; i < le; i += nt)
      if ((s.T[i] >> kNcShift) & kNcMask) up_inertia(i, s, g, c);
    OB_FENCE_UP(l)
  }
  __syncthreads();
}

// ------------------------------------------------------------------------------------------------------
// phase C as a function of its own (not inlined): its registers are allocated for the PCG loop alone, and what
// it needs of the world comes out of shared memory (World).  Returns the number of iterations; *flags gets
// OB_STATUS_CG_MAXITER, bit 30 = non-finite.
// ------------------------------------------------------------------------------------------------------
constexpr int kPcgBad = 1 << 30;

template <int NT, int LPT>
__device__ __noinline__ int pcg_solve(const World *wd, const DevCtx &c, float2 *stage, int *flipp, const int otid,
                                      const bool top_warp, const float bb, const float bz, int *flags) {
  const Sm s = carve(wd);
  const Gm g = wd->g;
  const ob_params &P = c.P;
  const int tid = threadIdx.x, lane = tid & 31;
  const int Np = s.Np, N = wd->N, nlev = wd->nlev, ntop = wd->ntop;
  float4 *const PL = s.P;
  float4 *const XR = s.XR;
  Reducer<NT> red;
  red.stage = stage; red.flip = *flipp; red.tid = otid;
  int status = 0;
  // lanes of the top warp <-> links of the n_top leading levels: level of the lane's link, widest child list
  // that stays inside the warp
  const int ntopN = s.lev[ntop];
  int top_lvl = -1, top_maxc = 0;
  if (lane < ntopN) {
    for (int l = 0; l < ntop; l++)
      if (lane >= s.lev[l]) top_lvl = l;
    if (top_lvl < ntop - 1) top_maxc = (int)((s.T[lane] >> kNcShift) & kNcMask);
  }
  top_maxc = __reduce_max_sync(0xffffffffu, top_maxc);
  int it = 0;
  bool bad = false;
  if (bb == 0.f) {
#pragma unroll
    for (int k = 0; k < LPT; k++) {
      const int i = otid + k * NT;
      if (i < N) XR[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  } else if (!(bb < INFINITY)) {
    bad = true;
  } else {
#pragma unroll
    for (int k = 0; k < LPT; k++) {                 // first product: A x, i.e. p = x
      const int i = otid + k * NT;
      if (i < N) *reinterpret_cast<float2 *>(PL + 7 * i + 2) = *reinterpret_cast<const float2 *>(XR + i);
    }
    bool first = true;
    float rz = 0.f, rr = 0.f;
    // stopping rule: |r| <= tol |b| in the 2-norm (cg_norm 0) or in the preconditioned norm (cg_norm 1)
    const float tol2 = P.cg_tol * P.cg_tol * (P.cg_norm ? bz : bb);
    for (;;) {
      // ---- A p.  The n_top leading levels live in warp 0, lane = link: own record in registers, parents
      //      and children by shuffle, no barrier.  The other levels are swept by the whole CTA, one block
      //      barrier per level; the deepest level turns around at once ----
      float pAp_part = 0.f;
      if (top_warp) {
        const int me = lane < ntopN ? lane : Np;             // idle lanes work on the zero record
        const uint32_t tw = s.T[me];
        float4 *rec = PL + 7 * me;
        const float4 pd = rec[2];
        const Jt j = load_jt(PL, me);
        const int parl = (tw & kTrunk) ? lane : (int)(tw & kParMask);   // the trunk's "parent" is all zero at level 0
        const float3 sp = f3(j.c2 * pd.x, pd.y, j.s2 * pd.x);
        float3 al = f3(0, 0, 0), a = f3(0, 0, 0);
#pragma unroll 1
        for (int l = 0; l < ntop; l++) {                      // branch-free: every lane computes, level l commits
          float3 alp, ap;
          alp.x = __shfl_sync(0xffffffffu, al.x, parl); alp.y = __shfl_sync(0xffffffffu, al.y, parl);
          alp.z = __shfl_sync(0xffffffffu, al.z, parl);
          ap.x = __shfl_sync(0xffffffffu, a.x, parl); ap.y = __shfl_sync(0xffffffffu, a.y, parl);
          ap.z = __shfl_sync(0xffffffffu, a.z, parl);
          const float3 nal = mul(j.E, alp) + sp;
          const float3 na = mul(j.E, f3(ap.x + alp.y * j.rz, ap.y - alp.x * j.rz, ap.z));
          const bool mine = top_lvl == l;
          al.x = mine ? nal.x : al.x; al.y = mine ? nal.y : al.y; al.z = mine ? nal.z : al.z;
          a.x = mine ? na.x : a.x; a.y = mine ? na.y : a.y; a.z = mine ? na.z : a.z;
        }
        if (lane < ntopN) {
          rec[0] = make_float4(al.x, al.y, al.z, a.x);
          *reinterpret_cast<float2 *>(rec + 1) = make_float2(a.y, a.z);
        }
      }
      __syncthreads();
#pragma unroll 1
      for (int l = ntop; l < nlev; l++) {
        const int le = s.lev[l + 1];
        const bool deepest = l == nlev - 1;
#pragma unroll 1
        for (int i = s.lev[l] + otid; i < le; i += NT) {
          const uint32_t tw = s.T[i];
          float4 *rec = PL + 7 * i;
          const float4 pd = rec[2];
          const Jt j = load_jt(PL, i);
          float3 al, a;
          mv_down(j, PL, tw, pd, al, a);
          if (deepest) {
            pAp_part += mv_up<false>(j, PL, PL + 7 * Np, i, tw, pd, al, a, s, g, c);
          } else {
            rec[0] = make_float4(al.x, al.y, al.z, a.x);
            *reinterpret_cast<float2 *>(rec + 1) = make_float2(a.y, a.z);
          }
        }
        __syncthreads();
      }
#pragma unroll 1
      for (int l = nlev - 2; l >= ntop; l--) {
        const int le = s.lev[l + 1];
#pragma unroll 1
        for (int i = s.lev[l] + otid; i < le; i += NT) {
          const uint32_t tw = s.T[i];
          const float4 *rec = PL + 7 * i;
          const float4 pd = rec[2];
          const Jt j = load_jt(PL, i);
          const float4 u = rec[0], v = rec[1];
          pAp_part += mv_up<true>(j, PL, PL + 7 * Np, i, tw, pd, f3(u.x, u.y, u.z), f3(u.w, v.x, v.y), s, g, c);
        }
        __syncthreads();
      }
      if (top_warp) {
        const int me = lane < ntopN ? lane : Np;
        const uint32_t tw = s.T[me];
        float4 *rec = PL + 7 * me;
        const float4 pd = rec[2], I = rec[6];
        const Jt j = load_jt(PL, me);
        const float4 u = rec[0], v = rec[1];
        const float3 al = f3(u.x, u.y, u.z), a = f3(u.w, v.x, v.y);
        const int fc = (int)((tw >> kChShift) & kParMask), nc = (int)((tw >> kNcShift) & kNcMask);
        // own inertia force; the children of the last top level are in shared memory, all others are lanes
        float3 n0 = f3(I.z * al.x - I.y * a.y, I.z * al.y + I.y * a.x, I.w * al.z);
        float3 f0 = f3(I.x * a.x + I.y * al.y, I.x * a.y - I.y * al.x, I.x * a.z);
        if (tw & kOffax) {
          const Force6 t = offaxis_tethers(__ldg(g.topo2 + me), al, a, s.att, s.ao, s.ak, s.Ap, P.h * P.h);
          n0 = n0 + t.n; f0 = f0 + t.f;
        }
        if (top_lvl == ntop - 1) gather_children(PL, PL + 7 * Np, fc, nc, n0, f0);
        const int nct = (top_lvl >= 0 && top_lvl < ntop - 1) ? nc : 0;
        float3 un = f3(0, 0, 0), uf = f3(0, 0, 0);           // (n, f) of this link in its parent's frame
        float t1 = 0.f, t2 = 0.f;
#pragma unroll 1
        for (int l = ntop - 1; l >= 0; l--) {                // branch-free: every lane computes, level l commits
          float3 n = n0, f = f0;
#pragma unroll
          for (int k = 0; k < 4; k++) {
            const int src = min(fc + k, 31);
            const float c0 = __shfl_sync(0xffffffffu, un.x, src), c1 = __shfl_sync(0xffffffffu, un.y, src),
                        c2 = __shfl_sync(0xffffffffu, un.z, src), c3 = __shfl_sync(0xffffffffu, uf.x, src),
                        c4 = __shfl_sync(0xffffffffu, uf.y, src), c5 = __shfl_sync(0xffffffffu, uf.z, src);
            const bool on = k < nct;
            n.x += on ? c0 : 0.f; n.y += on ? c1 : 0.f; n.z += on ? c2 : 0.f;
            f.x += on ? c3 : 0.f; f.y += on ? c4 : 0.f; f.z += on ? c5 : 0.f;
          }
          if (top_maxc > 4) {                                // uniform over the warp; wide fans are rare
#pragma unroll 1
            for (int k = 4; k < top_maxc; k++) {
              const int src = min(fc + k, 31);
              const float c0 = __shfl_sync(0xffffffffu, un.x, src), c1 = __shfl_sync(0xffffffffu, un.y, src),
                          c2 = __shfl_sync(0xffffffffu, un.z, src), c3 = __shfl_sync(0xffffffffu, uf.x, src),
                          c4 = __shfl_sync(0xffffffffu, uf.y, src), c5 = __shfl_sync(0xffffffffu, uf.z, src);
              const bool on = k < nct;
              n.x += on ? c0 : 0.f; n.y += on ? c1 : 0.f; n.z += on ? c2 : 0.f;
              f.x += on ? c3 : 0.f; f.y += on ? c4 : 0.f; f.z += on ? c5 : 0.f;
            }
          }
          const float nt1 = j.c2 * n.x + j.s2 * n.z + pd.z * pd.x;
          const float nt2 = n.y + pd.w * pd.y;
          const float3 nuf = mulT(j.E, f);
          float3 nun = mulT(j.E, n);
          nun.x -= j.rz * nuf.y; nun.y += j.rz * nuf.x;
          const bool mine = top_lvl == l;
          t1 = mine ? nt1 : t1; t2 = mine ? nt2 : t2;
          un.x = mine ? nun.x : un.x; un.y = mine ? nun.y : un.y; un.z = mine ? nun.z : un.z;
          uf.x = mine ? nuf.x : uf.x; uf.y = mine ? nuf.y : uf.y; uf.z = mine ? nuf.z : uf.z;
        }
        if (lane < ntopN) {
          reinterpret_cast<float2 *>(rec + 1)[1] = make_float2(t1, t2);
          pAp_part += pd.x * t1 + pd.y * t2;
        }
      }
      float rz_p = 0.f, rr_p = 0.f;
      if (first) {                                 // r = b - A x, z = P^-1 r, p = z
        first = false;
        __syncthreads();
#pragma unroll
        for (int k = 0; k < LPT; k++) {
          const int i = otid + k * NT;
          if (i < N) {
            const float2 ap = reinterpret_cast<const float2 *>(PL + 7 * i + 1)[1];
            const float2 idg = s.G[i];
            float2 r = reinterpret_cast<const float2 *>(XR + i)[1];
            r.x -= ap.x; r.y -= ap.y;
            reinterpret_cast<float2 *>(XR + i)[1] = r;
            const float za = r.x * idg.x, zb = r.y * idg.y;
            *reinterpret_cast<float2 *>(PL + 7 * i + 2) = make_float2(za, zb);
            rz_p += r.x * za + r.y * zb; rr_p += r.x * r.x + r.y * r.y;
          }
        }
        const float2 t = red.sum(rz_p, rr_p);
        rz = t.x; rr = P.cg_norm ? t.x : t.y;
      } else {
        const float pAp = red.sum(pAp_part, 0.f).x;
        const float alpha = rz / pAp;
        float2 z[LPT], pk[LPT];
#pragma unroll
        for (int k = 0; k < LPT; k++) {
          const int i = otid + k * NT;
          z[k] = make_float2(0.f, 0.f); pk[k] = make_float2(0.f, 0.f);
          if (i < N) {
            const float2 ap = reinterpret_cast<const float2 *>(PL + 7 * i + 1)[1];
            const float2 idg = s.G[i];
            pk[k] = *reinterpret_cast<const float2 *>(PL + 7 * i + 2);
            float4 xr = XR[i];
            xr.x += alpha * pk[k].x; xr.y += alpha * pk[k].y;
            xr.z -= alpha * ap.x; xr.w -= alpha * ap.y;
            XR[i] = xr;
            z[k] = make_float2(xr.z * idg.x, xr.w * idg.y);
            rz_p += xr.z * z[k].x + xr.w * z[k].y; rr_p += xr.z * xr.z + xr.w * xr.w;
          }
        }
        const float2 t = red.sum(rz_p, rr_p);
        const float beta = t.x / rz;
        rz = t.x; rr = P.cg_norm ? t.x : t.y;
#pragma unroll
        for (int k = 0; k < LPT; k++) {
          const int i = otid + k * NT;
          if (i < N)
            *reinterpret_cast<float2 *>(PL + 7 * i + 2) = make_float2(z[k].x + beta * pk[k].x, z[k].y + beta * pk[k].y);
        }
        it++;
      }
      if (!(rr > tol2 && it < P.cg_max_iter)) break;
    }
    if (!(rr <= tol2)) {
      if (rr == rr && rr < INFINITY) status |= OB_STATUS_CG_MAXITER;
      else bad = true;
    }
  }
  *flipp = red.flip;
  *flags = status | (bad ? kPcgBad : 0);
  return it;
}

// ------------------------------------------------------------------------------------------------------
// k_step<NT, LPT>
// ------------------------------------------------------------------------------------------------------
template <int NT, int LPT, int MINB>
__global__ void __launch_bounds__(NT, MINB)
k_step(const __grid_constant__ DevCtx c, const int32_t *__restrict__ order, int n_in_class, int32_t *queue, int n_steps,
       int top_rot, int n_chunks, int32_t *progress) {
  unsigned char *const smem = ob_smem;
  __shared__ __align__(8) uint64_t s_bar;
  __shared__ int s_next;
  __shared__ World s_world;
  __shared__ __align__(16) float2 s_stage[64];
  const int tid = threadIdx.x;
  // the warp that sweeps the top levels of the PCG products: rotated over the CTAs that share an SM, so that these
  // serial stretches do not all land on the same warp scheduler.  Everything arithmetic is indexed by the logical
  // thread index otid (a rotation of tid by whole warps), so the results do not depend on the rotation: a world
  // gives the same bits whichever CTA of the queue picks it up
  const int topw = (int)((blockIdx.x / (unsigned)top_rot) % (NT / 32));
  const bool top_warp = (tid >> 5) == topw;
  // flat ownership: thread otid + k * NT <-> link; the top warp owns links 0..31, i.e. exactly its lanes' links
  const int otid = (tid - 32 * topw + NT) % NT;
  const ob_params &P = c.P;
  uint32_t parity = 0;
  if (tid == 0) mbar_init(&s_bar, 1);
  __syncthreads();
  Reducer<NT> red;
  red.stage = s_stage;
  red.flip = 0;
  red.tid = otid;

  for (;;) {
    if (tid == 0) s_next = atomicAdd(queue, 1);
    __syncthreads();
    const int qi = s_next;
    __syncthreads();
    if (qi >= n_in_class * n_chunks) break;
    // The n steps of a launch are cut into n_chunks queue items per world (all first chunks, then all second ones,
    // ...): the tail of the launch, where CTAs run out of work, is a fraction of a chunk instead of a fraction of
    // the whole launch.  A later chunk of a world waits until the earlier one (taken by a resident CTA before,
    // the queue is in order) has published its state; all state crosses in global memory (L2: __ldcg loads).
    const int chunk = qi / n_in_class;
    const int w = order[qi - chunk * n_in_class];
    const int n_my = (int)(((long long)n_steps * (chunk + 1)) / n_chunks - ((long long)n_steps * chunk) / n_chunks);
    if (chunk > 0) {
      if (tid == 0) {
        while (*reinterpret_cast<volatile int32_t *>(progress + w) < chunk) __nanosleep(200);
        __threadfence();
      }
      __syncthreads();
    }
    const WorldDesc d = c.desc[w];
    WorldInfo *info = c.info + w;
    int status = __ldcg(&info->status);
    if ((status & OB_STATUS_NONFINITE) || n_my == 0) {      // frozen world (or nothing to do): pass the baton
      if (tid == 0) { __threadfence(); atomicExch(progress + w, chunk + 1); }
      continue;
    }
    const Sm s = carve(smem, d.Np, d.Ap, d.NIp, d.n_levels);
    const int Np = d.Np, N = d.N;
    const int nlev = d.n_levels, ntop = d.n_top;
    float4 *const PL = s.P;
    Gm g;
    {
      unsigned char *lb = c.link_blk + d.link_blk_off;
      g.q2 = reinterpret_cast<float2 *>(lb); g.w2 = g.q2 + Np;
      g.rupt = lb + kLinkStateFloats * 4 * Np; g.rc = g.rupt + Np;
      const unsigned char *cst = c.link_cst + (size_t)link_const_bytes(1) * d.link_base;
      g.c4 = reinterpret_cast<const float4 *>(cst);
      g.K = reinterpret_cast<const float *>(cst) + 4 * Np;
      g.rz = g.K + Np;
      g.quatd = reinterpret_cast<const double2 *>(c.quatd) + 2 * (size_t)d.link_base;
      g.anchor = c.anchor + 3 * (size_t)d.apple_base;
      g.Mmax = c.Mmax + d.link_base;
      g.mdiag = c.mdiag + d.link_base;
      g.hist = c.xprev + d.link_base;
      g.arm = c.arm ? c.arm + 2 * (size_t)d.link_base : nullptr;
      g.topo2 = c.topo2 + d.link_base;
    }
    if (tid == 0) {
      s_world.g = g; s_world.N = N; s_world.Np = Np; s_world.Ap = d.Ap; s_world.NIp = d.NIp; s_world.nlev = nlev;
      s_world.ntop = ntop;
    }

    // ---- stage the world: the apple block by one TMA bulk copy; topology words, level offsets, wrench slots ----
    if (tid == 0 && d.Ap) {
      fence_proxy_async();
      const uint32_t ab = (uint32_t)apple_block_bytes(d.Ap);
      mbar_expect_tx(&s_bar, ab);
      tma_load(s.u, c.apple_blk + d.apple_blk_off, ab, &s_bar);
    }
    {
      const int32_t *src = reinterpret_cast<const int32_t *>(c.wrench + w);
      int32_t *dst = reinterpret_cast<int32_t *>(s.wr);
      for (int k = tid; k < (int)(sizeof(WrenchSlots) / 4); k += NT) dst[k] = __ldg(src + k);
      if (tid < 7) PL[7 * Np + tid] = make_float4(0.f, 0.f, 0.f, 0.f);            // the zero column
      for (int k = tid; k <= nlev; k += NT) s.lev[k] = __ldg(c.level_off + d.level_base + k);
      for (int i = tid; i <= Np; i += NT) {
        uint32_t tw = (uint32_t)Np | kTrunk;
        if (i < N) {
          const int4 tp = __ldg(c.topo + d.link_base + i);
          const int4 t2 = __ldg(g.topo2 + i);
          const uint32_t nc = (uint32_t)tp.w, fc = nc ? (uint32_t)tp.y : 0u;
          tw = (tp.x >= 0 ? (uint32_t)tp.x : ((uint32_t)Np | kTrunk)) | (fc << kChShift) | (nc << kNcShift) |
               ((t2.x >> 16) ? kHasApples : 0u) | (__ldcg(g.rupt + i) ? kRuptured : 0u);
        }
        s.T[i] = tw;
      }
    }
    float4 *const XR = s.XR;                           // (x, r) of the PCG per link; aliases the phase-A overflow
    if (d.Ap) {
      mbar_wait(&s_bar, parity);
      parity ^= 1;
    }
    __syncthreads();
    int step0 = __ldcg(&info->step), steps_done = 0, last_iters = 0, diag_age = __ldcg(&info->diag_age);
    unsigned long long iters_total = 0;
    for (int sidx = 0; sidx < n_my; sidx++) {
      sweep_bias(&s_world, c, NT);                      // A, B1
      {                                                 // r = b; x = cubic extrapolation of the last four solutions
        const int t = step0 + sidx;                     // (ring of four in global memory, slot = step & 3)
        float2 h1[LPT], h2[LPT], h3[LPT], h4[LPT];
#pragma unroll
        for (int k = 0; k < LPT; k++) {
          const int i = min(otid + k * NT, N - 1);
          h1[k] = __ldcg(g.hist + ((t - 1) & 3) * (size_t)c.sum_np + i);
          h2[k] = __ldcg(g.hist + ((t - 2) & 3) * (size_t)c.sum_np + i);
          h3[k] = __ldcg(g.hist + ((t - 3) & 3) * (size_t)c.sum_np + i);
          h4[k] = __ldcg(g.hist + (t & 3) * (size_t)c.sum_np + i);
        }
#pragma unroll
        for (int k = 0; k < LPT; k++) {
          const int i = otid + k * NT;
          if (i < N) {
            const float2 b = s.G[i];
            XR[i] = make_float4(OB_X0(h1[k].x, h2[k].x, h3[k].x, h4[k].x), OB_X0(h1[k].y, h2[k].y, h3[k].y, h4[k].y), b.x, b.y);
          }
        }
      }
      sweep_inertia(&s_world, c, NT, otid, diag_age == 0);
      diag_age = diag_age + 1 >= kDiagRefresh ? 0 : diag_age + 1;   // (B2 first rewrites G[i] by the thread that just read it)
      float bb_part = 0.f, bz_part = 0.f;
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = otid + k * NT;
        if (i < N) {
          const float2 idg = s.G[i];
          const float4 xr = XR[i];
          bb_part += xr.z * xr.z + xr.w * xr.w;
          bz_part += xr.z * xr.z * idg.x + xr.w * xr.w * idg.y;
        }
      }
      const float2 bbz = red.sum(bb_part, bz_part);
      const float bb = bbz.x, bz = bbz.y;
      // ---- C: PCG, warm-started from the previous dqd (x) ----
      int pcg_flags = 0;
      const int it = pcg_solve<NT, LPT>(&s_world, c, s_stage, &red.flip, otid, top_warp, bb, bz, &pcg_flags);
      status |= pcg_flags & OB_STATUS_CG_MAXITER;
      const bool bad = (pcg_flags & kPcgBad) != 0;
      // a non-finite solve freezes the world at its last finite state
      int nf = 0;
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = otid + k * NT;
        if (i < N) {
          const float2 x = *reinterpret_cast<const float2 *>(XR + i);
          nf |= !(fabsf(x.x) < INFINITY) || !(fabsf(x.y) < INFINITY);
        }
      }
      if (__syncthreads_or(nf || bad)) { status |= OB_STATUS_NONFINITE; break; }

      // ---- D: integrate, predicates ----
      const int step_now = step0 + sidx;
      // (all global loads of the thread's links first: a store between two loads would serialise their L2 round trips)
      float2 dw0[LPT], dq0[LPT];
      float dK[LPT], dMx[LPT];
      int drc[LPT];
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = min(otid + k * NT, N - 1);
        dw0[k] = __ldcg(g.w2 + i); dq0[k] = __ldcg(g.q2 + i);
        dK[k] = __ldg(g.K + i); dMx[k] = __ldg(g.Mmax + i);
        drc[k] = __ldcg(g.rc + i);
      }
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = otid + k * NT;
        if (i >= N) continue;
        const float2 w0 = dw0[k], q0 = dq0[k];
        const float2 x = *reinterpret_cast<const float2 *>(XR + i);
        g.hist[(step_now & 3) * (size_t)c.sum_np + i] = x;
        float wa = w0.x + x.x, wb = w0.y + x.y;
        if (P.qd_max > 0.f) {
          wa = fminf(fmaxf(wa, -P.qd_max), P.qd_max);
          wb = fminf(fmaxf(wb, -P.qd_max), P.qd_max);
        }
        const float qa = fmaf(P.h, wa, q0.x), qb = fmaf(P.h, wb, q0.y);
        g.w2[i] = make_float2(wa, wb); g.q2[i] = make_float2(qa, qb);
        const uint32_t tw = s.T[i];
        if (!(tw & kRuptured)) {
          const float Ki = dK[k], Mx = dMx[k];
          const float mu = Ki * sqrtf(qa * qa + qb * qb);                   // Eq. 5
          const int rc0 = drc[k];
          const int rcn = mu > Mx ? rc0 + 1 : 0;
          if (rcn >= P.rupture_frames) {
            g.rupt[i] = 1; g.rc[i] = 0;
            s.T[i] = tw | kRuptured;
            push_event(c, w, step_now, 0, __ldg(c.link_ext + d.link_base + i), mu, Mx);
          } else if (rcn != rc0) {
            g.rc[i] = (unsigned char)rcn;
          }
        }
      }
      for (int a = tid; a < d.A; a += NT) {
        const int Ap = d.Ap;
        const bool att = s.att[a] != 0;
        const float ma = s.am[a], inv_m = 1.f / ma;
        const float fdet = s.afd[a];
        float3 ft = att ? f3(s.ft[a], s.ft[Ap + a], s.ft[2 * Ap + a]) : f3(0, 0, 0);
        float3 fu = f3(0, 0, 0);                                            // user force on the apple (wrench slots)
        for (int k = 0; k < s.wr->n; k++)
          if (s.wr->body[k] == N + a) fu = fu + f3(s.wr->force[k][0], s.wr->force[k][1], s.wr->force[k][2]);
        float3 va = f3(s.v[a], s.v[Ap + a], s.v[2 * Ap + a]);
        const float3 v0 = va;                                               // F = -c_v m v on the apple
        va.x += P.h * (P.gravity[0] + (ft.x + fu.x) * inv_m - P.mass_damping * v0.x);
        va.y += P.h * (P.gravity[1] + (ft.y + fu.y) * inv_m - P.mass_damping * v0.y);
        va.z += P.h * (P.gravity[2] + (ft.z + fu.z) * inv_m - P.mass_damping * v0.z);
        s.v[a] = va.x; s.v[Ap + a] = va.y; s.v[2 * Ap + a] = va.z;
        s.u[a] = fmaf(P.h, va.x, s.u[a]); s.u[Ap + a] = fmaf(P.h, va.y, s.u[Ap + a]);
        s.u[2 * Ap + a] = fmaf(P.h, va.z, s.u[2 * Ap + a]);
        if (att) {
          const float fun = sqrtf(dot(fu, fu)), fsn = s.fsn[a], thrB = P.detach_kappa * fdet;
          const int ca = fun > fdet ? s.cA[a] + 1 : 0;
          const int cb = fsn > thrB ? s.cB[a] + 1 : 0;
          if (ca >= P.detach_frames_pull) {
            s.att[a] = 0; s.cA[a] = 0; s.cB[a] = 0;
            push_event(c, w, step_now, 1, __ldg(c.apple_ext + d.apple_base + a), fun, fdet);
          } else if (cb >= P.detach_frames_tension) {
            s.att[a] = 0; s.cA[a] = 0; s.cB[a] = 0;
            push_event(c, w, step_now, 1, __ldg(c.apple_ext + d.apple_base + a), fsn, thrB);
          } else {
            s.cA[a] = (unsigned char)ca; s.cB[a] = (unsigned char)cb;
          }
        }
      }
      if (tid == 0) atomicAdd(c.iter_hist + min(it, kIterHistBins - 1), 1ull);
      steps_done++;
      last_iters = it;
      iters_total += (unsigned long long)it;
      __syncthreads();
    }

    // ---- write the state back: the apple state by one TMA bulk store; a frozen world restarts from x = 0 ----
    if (status & OB_STATUS_NONFINITE) {
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = otid + k * NT;
        if (i < N)
          for (int q = 0; q < 4; q++) g.hist[q * (size_t)c.sum_np + i] = make_float2(0.f, 0.f);
      }
    }
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
      if (d.Ap) {
        tma_store(c.apple_blk + d.apple_blk_off, s.u, (uint32_t)apple_state_bytes(d.Ap));
        tma_store_commit_wait();
      }
      info->step = step0 + steps_done;
      info->last_iters = last_iters;
      info->status = status;
      info->diag_age = diag_age;
      info->steps_taken = __ldcg(&info->steps_taken) + steps_done;
      info->cg_iters = __ldcg(&info->cg_iters) + iters_total;
    }
    __syncthreads();                                 // every thread's global writes of this chunk are done
    if (tid == 0) { __threadfence(); atomicExch(progress + w, chunk + 1); }
  }
}

// ------------------------------------------------------------------------------------------------------
// launchers: one instantiation per size class (ob_internal.h: kStepClasses)
// ------------------------------------------------------------------------------------------------------
#define OB_FOR_CLASS(cls, CALL)                                     \
  switch (cls) {                                                    \
    case 0: { CALL(64, 4, 6); break; }                              \
    case 1: { CALL(128, 4, 3); break; }                             \
    case 2: { CALL(192, 4, 2); break; }                             \
    case 3: { CALL(256, 4, 1); break; }                             \
    case 4: { CALL(256, 6, 1); break; }                             \
    default: return cudaErrorInvalidValue;                          \
  }

cudaError_t step_kernel_setup(int cls, int smem_bytes, int *max_blocks_per_sm) {
#define OB_SETUP(NT, LPT, MINB)                                                                                   \
  cudaError_t e = cudaFuncSetAttribute(k_step<NT, LPT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize,        \
                                       smem_bytes);                                                               \
  if (e != cudaSuccess) return e;                                                                                 \
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(max_blocks_per_sm, k_step<NT, LPT, MINB>, NT, smem_bytes);
  OB_FOR_CLASS(cls, OB_SETUP)
#undef OB_SETUP
  return cudaSuccess;
}

cudaError_t launch_step(const DevCtx &c, int cls, const int32_t *order, int n_in_class, int32_t *queue, int n_steps,
                        int grid, int smem, int n_sm, int n_chunks, int32_t *progress, cudaStream_t s) {
#define OB_LAUNCH(NT, LPT, MINB)                                                                                   \
  k_step<NT, LPT, MINB><<<grid, NT, smem, s>>>(c, order, n_in_class, queue, n_steps, n_sm > 0 ? n_sm : 1, n_chunks, \
                                               progress);
  OB_FOR_CLASS(cls, OB_LAUNCH)
#undef OB_LAUNCH
  return cudaGetLastError();
}

}  // namespace ob
