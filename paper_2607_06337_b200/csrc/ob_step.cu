// ob_step.cu -- k_step, the product kernel (sm_100a): n physics steps of every world in one launch.
//
// One CTA per world in flight (persistent, work queue per size class), three CTAs of 128 threads per SM at the
// headline size.  Everything the level-synchronous tree sweeps touch lives in SHARED MEMORY as one 112-byte
// record of seven float4 per link (stride 7 x 16 B: 128-bit accesses of consecutive links are conflict-free),
// so the sweep code exists once and runs over any number of links.  The apple block is staged by one TMA bulk copy
// (UBLKCP) and written back the same way; q, qd and the PCG start vectors stay in global memory (L2): only the
// once-per-step phases touch them.
//
//   A0  flat:      joint rotations q_rel = Q qx(theta1) qy(theta2) (Eq. 3) as fp64 quaternions; the fp32
//                  copy is what the dynamics rotate with
//   A1  top-down:  forward kinematics in fp64 (world quaternion and position of every link), hang points of the apples
//   F   bottom-up: the preconditioner of the step.  precond = 2: articulated-body inertias of the tree whose joints
//                  carry the "armature" arm + h D + h^2 K, i.e. an exact O(N) factorisation of the system matrix
//                  A = M + M_teth + diag(arm + hD + h^2 K) (Featherstone's articulated-body recursion; A is the
//                  joint-space inertia of that tree), kept as K_i = U_i D_i^-1 and D_i^-1 per inner link;
//                  precond = 1: composite inertias -> exact diagonal of M (Jacobi)
//   A2  top-down:  velocities, bias accelerations, bias force of every link incl. tether reactions (Eq. 6 / Eq. 7,
//                  PAPER.md:149-161) and user wrenches; leaves finish at once
//   B1  bottom-up: bias torques of the inner links -> rhs b
//   C   matrix-free preconditioned CG on A dqd = b (north_star), started from the cubic extrapolation of the last
//                  four solutions; A v = acceleration-only inverse dynamics (top-down a_i, bottom-up f_i, project on
//                  S_i); with precond = 2, z = P^-1 r is one bottom-up and one top-down sweep of the same shape
//   D   integrate joints and apples; rupture (Eq. 5) and detach predicates
//
// Order.  Links are in plain breadth-first order: levels contiguous, the children of a link contiguous.  In the
// A v sweeps the leading levels that fit into 32 links (n_top of them) are swept by ONE warp, lane = link, own
// record in registers, parents and children by shuffle, no barrier; every other level ends with one block
// barrier; only the deepest level turns around inside the top-down pass (all of its links are leaves).  In the
// other sweeps that warp takes the leading levels with __syncwarp.
//
// Record of link i (P[7 i + j]); record Np is never written and stays zero: the trunk's parent, missing children.
//   0  QR   fp32 quaternion (w,x,y,z) of R_rel; E = R_rel^T maps parent coordinates to link coordinates
//   1  CS   cos theta2, sin theta2, parent length, packed topology word (parent | first child << 11 | children << 22 |
//           flags)
//   2  IN   effective link inertia (m, m c, I about the joint, I_zz) incl. on-axis virtual tether masses (A15)
//   3  PD   (p, diagonal terms arm + (h c_d + h^2) K)
//   4, 5  M0, M1   parent <-> child mailbox (six floats); M1.zw = A p, then the solve's D^-1 u, then z
//   6  XR   (x, r) of the PCG
// Before the PCG the slots double as mailboxes of the once-per-step sweeps: A0 -> A1 q_rel in fp64 (M0, M1); A1 the
// fp64 world pose of an inner link for its children (M0, M1, PD, XR.xy); F 21 floats of articulated inertia for the
// parent (IN, PD, M0, M1, XR + the X21 plane); A2 velocity and bias acceleration of an inner link for its children
// (XR, IN, PD.xy, M1.zw) beside its parked bias force (M0, M1.xy).  A2 / B1 then leave IN, PD.zw, XR.zw (= b) as the
// PCG wants them.
//
// Spatial vectors are [angular; linear at the link origin] in link coordinates.  Link frame: origin at the
// proximal joint, +z along the link.  Joint i: R_rel = Q_i Rx(theta1) Ry(theta2); the joint sits at
// r = (0,0,L_parent) in the parent frame; joint axes in link coordinates S = [(c2, 0, s2), (0, 1, 0)].
#include <math.h>

#include "ob_device.h"
#include "ob_internal.h"

namespace ob {

// packed topology word
constexpr uint32_t kParMask = 0x7ffu, kChShift = 11, kNcShift = 22, kNcMask = 0xfu;
constexpr uint32_t kHasApples = 1u << 26, kOffax = 1u << 27, kSnapped = 1u << 28, kRuptured = 1u << 29, kTrunk = 1u << 30;
constexpr int kQR = 0, kCS = 1, kIN = 2, kPD = 3, kM0 = 4, kM1 = 5, kXR = 6;
constexpr uint32_t kNoSlot = 0xffffu;

// ------------------------------------------------------------------------------------------------------
// shared-memory view of one world
// ------------------------------------------------------------------------------------------------------
struct Sm {
  int Np, Ap, NFp;
  float4 *P;                          // records
  float *X21;                         // [Np + 1] the 21st float of the F mailbox
  uint16_t *SL;                       // [Np + 1] factor slot of the link (inner links, off-axis tether links) or kNoSlot
  float4 *FAC;                        // precond 2: four planes [NFp]: K (6 x 2) and D^-1 per slot
  float2 *IDG;                        // precond 0 / 1: 1 / diag(A) per link (same memory as FAC)
  int *lev;                           // level offsets [n_levels + 1]
  // apple block (TMA)
  float *u, *v;                       // [3][Ap]
  unsigned char *att, *cA, *cB;
  float *ao, *ak, *am, *ac, *afd;     // ao = [3][Ap]
  const int *alnk;                    // [Ap] internal index of the link that carries the apple
  float *ft, *fsn;                    // tether force on the apple beyond its rest sag [3][Ap] (-k_s du - c_s v: the sag carries
                                      // the weight), |f_s| [Ap] (apple pass -> phase D)
  float *hd;                          // [6][Ap] anchor - x_hang of every apple, fp64 as (hi, lo) pairs (phase A1 -> apple
                                      // pass); aliases ft, fsn (see carve)
  float *aq;                          // [4][Ap] world quaternion (fp32) of the apple's link (phase A1 -> apple pass); then,
                                      // with hd[4], hd[5], the reaction of the apple on its link (apple pass -> B1)
  float4 *wq;                         // [OB_MAX_WRENCH] world quaternion of the link of each wrench slot
  WrenchSlots *wr;
};

// The functions that are not inlined carve the CTA's dynamic shared memory again from the sizes (World) instead of
// taking pointers: pointers handed over through memory are generic, and the sweeps then run on LD.E / ST.E with
// 64-bit address arithmetic instead of LDS / STS.
extern __shared__ __align__(128) unsigned char ob_smem[];

__device__ __forceinline__ Sm carve(unsigned char *base, const int Np, const int Ap, const int NFp, const int n_levels) {
  Sm s;
  s.Np = Np; s.Ap = Ap; s.NFp = NFp;
  unsigned char *p = base;
  s.P = reinterpret_cast<float4 *>(p); p += step_planes_bytes(Np);
  s.X21 = reinterpret_cast<float *>(p); p += r16(4 * (Np + 1));
  s.SL = reinterpret_cast<uint16_t *>(p); p += r16(2 * (Np + 1));
  s.FAC = reinterpret_cast<float4 *>(p); s.IDG = reinterpret_cast<float2 *>(p); p += step_fac_bytes(Np, NFp);
  s.lev = reinterpret_cast<int *>(p); p += r16(4 * (n_levels + 1));
  float *f = reinterpret_cast<float *>(p);
  s.u = f; s.v = f + 3 * Ap;
  s.att = p + 24 * Ap; s.cA = s.att + Ap; s.cB = s.cA + Ap;
  f = reinterpret_cast<float *>(p + apple_state_bytes(Ap));
  s.ao = f; s.ak = f + 3 * Ap; s.am = f + 4 * Ap; s.ac = f + 5 * Ap; s.afd = f + 6 * Ap;
  s.alnk = reinterpret_cast<const int *>(f + 7 * Ap);
  p += r16(apple_block_bytes(Ap));
  f = reinterpret_cast<float *>(p);
  s.ft = f; s.fsn = f + 3 * Ap; s.hd = f; f += 6 * Ap;   // hd[0..3] share the memory of ft[0..2], fsn: per apple, phase A2
  s.aq = f; f += 4 * Ap;                                 // reads hd, then writes them
  s.wq = reinterpret_cast<float4 *>(f); f += 4 * OB_MAX_WRENCH;
  s.wr = reinterpret_cast<WrenchSlots *>(f);
  return s;
}

// per-link data of one world in global memory (L2-resident; only the once-per-step phases read it)
struct Gm {
  float2 *q2, *w2;                  // state (link block)
  int32_t *rstep;                   // step during which the joint ruptured
  unsigned char *rupt, *rc;
  const float4 *c4;                 // (m, m c, I about the joint, I_zz)
  const float *K, *rz;              // joint stiffness (Eq. 4), parent length
  const double2 *quatd;             // rest quaternions, normalised, fp64: (w, x), (y, z) of link i at 2 i, 2 i + 1
  const double *anchor;             // [k * Ap + a] rest hang points, world frame, fp64
  const float *Mmax;
  float2 *hist;                     // [4][sum_np]: dqd of the last four steps, slot = step & 3
  const float *arm;                 // [k * Np + i] or nullptr
  const int4 *topo2;                // x = first apple | n_apples << 16, y = factor slot (or 0xffff)
};

// the views of the world every thread of the CTA shares (in shared memory, filled once per world)
struct World { Gm g; int N, A, Np, Ap, NFp, nlev, ntop, precond; };
__device__ __forceinline__ Sm carve(const World *wd) { return carve(ob_smem, wd->Np, wd->Ap, wd->NFp, wd->nlev); }

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

// ------------------------------------------------------------------------------------------------------
// joint transform of one link as the sweeps use it: the unit quaternion of R_rel (link -> parent), cos / sin theta2,
// the parent length, the topology word
// ------------------------------------------------------------------------------------------------------
struct Jt {
  float4 q;            // (w, x, y, z) in (.x, .y, .z, .w)
  float c2, s2, rz;
  uint32_t tw;
};
__device__ __forceinline__ Jt load_jt(const float4 *P, const int i) {
  const float4 q = P[7 * i + kQR], c = P[7 * i + kCS];
  Jt j;
  j.q = q; j.c2 = c.x; j.s2 = c.y; j.rz = c.z; j.tw = __float_as_uint(c.w);
  return j;
}
// R(q) x  (link -> parent) and R(q)^T x = E x  (parent -> link)
__device__ __forceinline__ float3 rot_up(const float4 q, const float3 x) {
  const float3 v = f3(q.y, q.z, q.w);
  const float3 t = cross(v, x);
  const float3 t2 = f3(t.x + t.x, t.y + t.y, t.z + t.z);
  return x + q.x * t2 + cross(v, t2);
}
__device__ __forceinline__ float3 rot_down(const float4 q, const float3 x) {
  const float3 v = f3(q.y, q.z, q.w);
  const float3 t = cross(v, x);
  const float3 t2 = f3(t.x + t.x, t.y + t.y, t.z + t.z);
  return x - q.x * t2 + cross(v, t2);
}
__device__ __forceinline__ M3 quat_mat(const float4 q) {   // R(q), row-major
  const float w = q.x, x = q.y, y = q.z, z = q.w;
  M3 R;
  R.a[0] = 1.f - 2.f * (y * y + z * z); R.a[1] = 2.f * (x * y - w * z);       R.a[2] = 2.f * (x * z + w * y);
  R.a[3] = 2.f * (x * y + w * z);       R.a[4] = 1.f - 2.f * (x * x + z * z); R.a[5] = 2.f * (y * z - w * x);
  R.a[6] = 2.f * (x * z - w * y);       R.a[7] = 2.f * (y * z + w * x);       R.a[8] = 1.f - 2.f * (x * x + y * y);
  return R;
}

struct Force6 { float3 n, f; };

// a spatial vector of the parent (motion) into the link frame: al = E alp, a = E (ap + alp x r), r = (0,0,rz)
__device__ __forceinline__ void motion_down(const Jt &j, const float3 alp, const float3 ap, float3 &al, float3 &a) {
  al = rot_down(j.q, alp);
  a = rot_down(j.q, f3(ap.x + alp.y * j.rz, ap.y - alp.x * j.rz, ap.z));
}
// the same with the rotation matrix R(q) at hand (a turn that rotates four or more vectors builds it once: 21 + 9 per
// vector instead of 21 per vector)
__device__ __forceinline__ void motion_down_m(const M3 &R, const float rz, const float3 alp, const float3 ap, float3 &al,
                                              float3 &a) {
  al = mulT(R, alp);
  a = mulT(R, f3(ap.x + alp.y * rz, ap.y - alp.x * rz, ap.z));
}
__device__ __forceinline__ void force_up_m(const M3 &R, const float rz, const float3 n, const float3 f, float3 &np,
                                           float3 &fp) {
  fp = mul(R, f);
  np = mul(R, n);
  np.x -= rz * fp.y; np.y += rz * fp.x;
}
// a spatial force of the link into the parent frame: fp = E^T f, np = E^T n + r x fp
__device__ __forceinline__ void force_up(const Jt &j, const float3 n, const float3 f, float3 &np, float3 &fp) {
  fp = rot_up(j.q, f);
  np = rot_up(j.q, n);
  np.x -= j.rz * fp.y; np.y += j.rz * fp.x;
}

// ------------------------------------------------------------------------------------------------------
// phase C: A v for one link.  mv_down: accelerations from the parent (the trunk reads the zero column).
// mv_up: f = I a + children, project on S (+ diagonal terms) -> A p (M1[i].zw), publish (n, f) in the parent
// frame; returns p . (A p) of this link.  Mailbox: M0[i] = (x, y, z of the angular part, x of the linear part),
// M1[i].xy = (y, z of the linear part).
// ------------------------------------------------------------------------------------------------------
// virtual tether masses off the link axis (rare: the workloads hang apples on the axis), one by one.  Everything
// goes in and out by value so that nothing of the caller is forced into local memory.
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

__device__ __forceinline__ void mv_down(const Jt &j, const float4 *P, const float4 pd, float3 &al, float3 &a) {
  const float4 *par = P + 7 * (int)(j.tw & kParMask);
  const float4 u = par[kM0], v = par[kM1];
  motion_down(j, f3(u.x, u.y, u.z), f3(u.w, v.x, v.y), al, a);
  al = al + f3(j.c2 * pd.x, pd.y, j.s2 * pd.x);
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
    cu[k] = q[kM0]; cv[k] = q[kM1];
  }
#pragma unroll
  for (int k = 0; k < 4; k++) {
    n = n + f3(cu[k].x, cu[k].y, cu[k].z);
    f = f + f3(cu[k].w, cv[k].x, cv[k].y);
  }
#pragma unroll 1
  for (int k = 4; k < nc; k++) {
    const float4 u = ch[7 * k + kM0], v = ch[7 * k + kM1];
    n = n + f3(u.x, u.y, u.z);
    f = f + f3(u.w, v.x, v.y);
  }
}

// inertia force of the link's own effective inertia (a body of revolution about +z through the joint)
__device__ __forceinline__ void own_inertia_force(const float4 I, const float3 al, const float3 a, float3 &n, float3 &f) {
  n = f3(I.z * al.x - I.y * a.y, I.z * al.y + I.y * a.x, I.w * al.z);
  f = f3(I.x * a.x + I.y * al.y, I.x * a.y - I.y * al.x, I.x * a.z);
}

template <bool GATHER>
__device__ __forceinline__ float mv_up(const Jt &j, float4 *P, const float4 *zero_rec, const int i, const float4 pd,
                                       const float3 al, const float3 a, const Sm &s, const Gm &g, const DevCtx &c) {
  float4 *rec = P + 7 * i;
  float3 n, f;
  own_inertia_force(rec[kIN], al, a, n, f);
  if (j.tw & kOffax) {
    const Force6 t = offaxis_tethers(__ldg(g.topo2 + i), al, a, s.att, s.ao, s.ak, s.Ap, c.P.h * c.P.h);
    n = n + t.n; f = f + t.f;
  }
  if (GATHER) gather_children(P, zero_rec, (int)((j.tw >> kChShift) & kParMask), (int)((j.tw >> kNcShift) & kNcMask), n, f);
  const float t1 = j.c2 * n.x + j.s2 * n.z + pd.z * pd.x;     // pd = (p0, p1, dt0, dt1)
  const float t2 = n.y + pd.w * pd.y;
  float3 np, fp;                                              // the trunk publishes into its own record, which nobody reads
  force_up(j, n, f, np, fp);
  rec[kM0] = make_float4(np.x, np.y, np.z, fp.x);
  rec[kM1] = make_float4(fp.y, fp.z, t1, t2);
  return pd.x * t1 + pd.y * t2;
}

// ------------------------------------------------------------------------------------------------------
// precond = 2: z = P^-1 r with the factors of phase F.  K = U D^-1 (6 x 2: columns k1, k2 as (angular, linear)) and
// D^-1 (symmetric 2 x 2) of one link: out of the factor planes for a link with a slot; for a plain leaf (its
// articulated inertia is its own effective inertia) from the closed form
//   U1 = (I c2, 0, Izz s2; 0, -mc c2, 0), U2 = (0, I, 0; mc, 0, 0), D = diag(I c2^2 + Izz s2^2 + dt0, I + dt1)
// ------------------------------------------------------------------------------------------------------
struct Kf { float3 k1n, k1f, k2n, k2f; float d11, d12, d22; };
__device__ __forceinline__ Kf load_kf(const Sm &s, const int i, const Jt &j, const float4 I, const float dt0, const float dt1) {
  Kf k;
  const uint32_t slot = s.SL[i];
  if (slot != kNoSlot) {
    const float4 a = s.FAC[slot], b = s.FAC[s.NFp + slot], cc = s.FAC[2 * s.NFp + slot], d = s.FAC[3 * s.NFp + slot];
    k.k1n = f3(a.x, a.y, a.z); k.k1f = f3(a.w, b.x, b.y);
    k.k2n = f3(b.z, b.w, cc.x); k.k2f = f3(cc.y, cc.z, cc.w);
    k.d11 = d.x; k.d12 = d.y; k.d22 = d.z;
  } else {
    const float i11 = __fdividef(1.f, j.c2 * j.c2 * I.z + j.s2 * j.s2 * I.w + dt0), i22 = __fdividef(1.f, I.z + dt1);
    k.k1n = f3(I.z * j.c2 * i11, 0.f, I.w * j.s2 * i11); k.k1f = f3(0.f, -I.y * j.c2 * i11, 0.f);
    k.k2n = f3(0.f, I.z * i22, 0.f); k.k2f = f3(I.y * i22, 0.f, 0.f);
    k.d11 = i11; k.d12 = 0.f; k.d22 = i22;
  }
  return k;
}

// bottom-up turn of one link: u = r - S^T p (p = what the children sent up), publish p + K u in the parent frame,
// keep y = D^-1 u (M1.zw)
template <bool GATHER>
__device__ __forceinline__ void solve_up(const int i, float4 *P, const Sm &s) {
  float4 *rec = P + 7 * i;
  const Jt j = load_jt(P, i);
  const float4 I = rec[kIN], pd = rec[kPD], xr = rec[kXR];
  const Kf k = load_kf(s, i, j, I, pd.z, pd.w);
  float3 n = f3(0, 0, 0), f = f3(0, 0, 0);
  if (GATHER) gather_children(P, P + 7 * s.Np, (int)((j.tw >> kChShift) & kParMask), (int)((j.tw >> kNcShift) & kNcMask), n, f);
  const float u0 = xr.z - (j.c2 * n.x + j.s2 * n.z), u1 = xr.w - n.y;
  n = n + u0 * k.k1n + u1 * k.k2n;
  f = f + u0 * k.k1f + u1 * k.k2f;
  float3 np, fp;
  force_up(j, n, f, np, fp);
  rec[kM0] = make_float4(np.x, np.y, np.z, fp.x);
  rec[kM1] = make_float4(fp.y, fp.z, k.d11 * u0 + k.d12 * u1, k.d12 * u0 + k.d22 * u1);
}

// top-down turn: a' = X a_parent, z = y - K^T a', a = a' + S z for the children; z -> M1.zw.
// FUSE (first PCG iteration: p = z): the accelerations this pass hands down ARE the top-down pass of the product A p
// for p = z, so the pass doubles as that: p -> PD.xy, every link keeps (al, a) for its turn in the product's bottom-up
// pass, and a link of the deepest level turns around at once (returns its p . A p).
template <bool FUSE>
__device__ __forceinline__ float solve_down(const int i, float4 *P, const Sm &s, const Gm &g, const DevCtx &c,
                                            const bool turn) {
  float4 *rec = P + 7 * i;
  const Jt j = load_jt(P, i);
  const float4 I = rec[kIN], pd = rec[kPD];
  const float4 m1 = rec[kM1];                                  // (128-bit accesses only: the 64-bit ones into the
  const float2 y = make_float2(m1.z, m1.w);                    // 112-byte records are 2-way bank conflicted)
  const Kf k = load_kf(s, i, j, I, pd.z, pd.w);
  const float4 *par = P + 7 * (int)(j.tw & kParMask);
  const float4 u = par[kM0], v = par[kM1];
  float3 al, a;
  motion_down(j, f3(u.x, u.y, u.z), f3(u.w, v.x, v.y), al, a);
  const float z0 = y.x - (dot(k.k1n, al) + dot(k.k1f, a)), z1 = y.y - (dot(k.k2n, al) + dot(k.k2f, a));
  al = al + f3(j.c2 * z0, z1, j.s2 * z0);
  if (FUSE) {
    rec[kPD] = make_float4(z0, z1, pd.z, pd.w);
    if (turn) return mv_up<false>(j, P, P + 7 * s.Np, i, make_float4(z0, z1, pd.z, pd.w), al, a, s, g, c);
    rec[kM0] = make_float4(al.x, al.y, al.z, a.x);
    rec[kM1] = make_float4(a.y, a.z, 0.f, 0.f);
  } else if ((j.tw >> kNcShift) & kNcMask) {
    rec[kM0] = make_float4(al.x, al.y, al.z, a.x);
    rec[kM1] = make_float4(a.y, a.z, z0, z1);
  } else {
    rec[kM1] = make_float4(0.f, 0.f, z0, z1);
  }
  return 0.f;
}

// ------------------------------------------------------------------------------------------------------
// The once-per-step phases, cut into passes that each keep a small working set in registers (a spilled
// register costs an L2 round trip here: the three CTAs of an SM leave the L1 only ~28 KB).
// ------------------------------------------------------------------------------------------------------
// PCG start vector: cubic extrapolation of the last four solutions (x1 = the latest)
#define OB_X0(x1, x2, x3, x4) (4.f * ((x1) + (x3)) - 6.f * (x2) - (x4))

// a double carried as two floats (hi + lo): 48 bits, plenty for a displacement summed along <= 2000 links
__device__ __forceinline__ float2 split2(const double v) {
  const float hi = (float)v;
  return make_float2(hi, (float)(v - (double)hi));
}
__device__ __forceinline__ double join2(const float hi, const float lo) { return (double)hi + (double)lo; }

struct Qd { double w, x, y, z; };
__device__ __forceinline__ Qd qmul(const Qd a, const Qd b) {
  Qd r;
  r.w = a.w * b.w - a.x * b.x - a.y * b.y - a.z * b.z;
  r.x = a.w * b.x + a.x * b.w + a.y * b.z - a.z * b.y;
  r.y = a.w * b.y - a.x * b.z + a.y * b.w + a.z * b.x;
  r.z = a.w * b.z + a.x * b.y - a.y * b.x + a.z * b.w;
  return r;
}
__device__ __forceinline__ void store_qd(float4 *rec, const Qd q) {
  double2 *pr = reinterpret_cast<double2 *>(rec + kM0);
  pr[0] = make_double2(q.w, q.x); pr[1] = make_double2(q.y, q.z);
}
__device__ __forceinline__ Qd load_qd(const float4 *rec) {
  const double2 *pr = reinterpret_cast<const double2 *>(rec + kM0);
  const double2 a = pr[0], b = pr[1];
  Qd q;
  q.w = a.x; q.x = a.y; q.y = b.x; q.z = b.y;
  return q;
}

// ---- A0 ----  q_rel = Q qx(th1) qy(th2) of one link in fp64 (Eq. 3: R_rel = Q Rx(th1) Ry(th2)) -> M0, M1 of the link's
//               own record for A1; its fp32 copy, cos / sin th2 and the parent length -> QR, CS for the dynamics
__device__ __forceinline__ void link_joint(const int i, const Sm &s, const Gm &g) {
  float4 *rec = s.P + 7 * i;
  const float2 th = __ldcg(g.q2 + i);
  const double2 qa = __ldg(g.quatd + 2 * i), qb = __ldg(g.quatd + 2 * i + 1);
  const uint32_t tw = __float_as_uint(rec[kCS].w);
  const float rzf = (tw & kTrunk) ? 0.f : __ldg(g.rz + i);
  double s1, c1, s2, c2;
  sincos(0.5 * (double)th.x, &s1, &c1);
  sincos(0.5 * (double)th.y, &s2, &c2);
  Qd Q, b;
  Q.w = qa.x; Q.x = qa.y; Q.y = qb.x; Q.z = qb.y;
  b.w = c1 * c2; b.x = s1 * c2; b.y = c1 * s2; b.z = s1 * s2;          // qx(th1) qy(th2)
  const Qd q = qmul(Q, b);
  rec[kQR] = make_float4((float)q.w, (float)q.x, (float)q.y, (float)q.z);
  rec[kCS] = make_float4((float)(c2 * c2 - s2 * s2), (float)(2.0 * s2 * c2), rzf, __uint_as_float(tw));
  store_qd(rec, q);
}

// Coulomb friction at a ruptured joint ("introduced at the break and ramped up ~5x over ~1.5 s as the
// torn fibres seize"; reading A34) as the damper D_f = T_f(t) / max(|qd|, v_eps) at the start-of-step joint speed,
// T_f(t) = fric_frac M_max (1 + (fric_ramp - 1) min(t / fric_time, 1)), t = h (step - step of the rupture)
// (out of line: cold unless fric_frac > 0 and the joint is ruptured)
__device__ __noinline__ float friction_damper(const int i, const float2 w, const int step, const Gm &g, const ob_params &P) {
  const float t = P.h * (float)(step - __ldcg(g.rstep + i));
  const float ramp = P.fric_time > 0.f ? fminf(t / P.fric_time, 1.f) : 1.f;
  const float Tf = P.fric_frac * __ldg(g.Mmax + i) * (1.f + (P.fric_ramp - 1.f) * ramp);
  return Tf / fmaxf(sqrtf(w.x * w.x + w.y * w.y), P.fric_veps);
}

// The global inputs of a level sweep are staged by a FLAT pass before it (one L2 round trip for the whole world
// instead of one per level of the sweep): the link's own inertia constants -> IN, (q, qd) -> XR, K -> PD.x (before
// phase F: -> X21, because A1 publishes through PD and XR.xy).  Each sweep reads them at the link's own turn, before it
// overwrites the slots with what it publishes.
// A ruptured joint has no K: its slot carries the friction damper D_f instead (split_kd sorts them out).
__device__ __forceinline__ void stage_link_inputs(const int i, const Sm &s, const Gm &g, const bool state, const int step,
                                                  const ob_params &P) {
  float4 *rec = s.P + 7 * i;
  const float4 c4 = __ldg(g.c4 + i);
  const float Ki = __ldg(g.K + i);
  const uint32_t tw = __float_as_uint(rec[kCS].w);
  const bool fric = (tw & kRuptured) && P.fric_frac > 0.f;
  float2 w = make_float2(0.f, 0.f);
  if (state || fric) w = __ldcg(g.w2 + i);
  const float kd = (tw & kRuptured) ? (fric ? friction_damper(i, w, step, g, P) : 0.f) : Ki;
  if (state) {
    const float2 th = __ldcg(g.q2 + i);
    rec[kXR] = make_float4(th.x, th.y, w.x, w.y);
    rec[kPD].x = kd;
    if (tw & kHasApples) s.X21[i] = __int_as_float(__ldg(g.topo2 + i).x);   // first apple | count << 16
  } else {
    s.X21[i] = kd;
  }
  rec[kIN] = c4;
}

// ---- A1 ----  forward kinematics in fp64 (Eq. 3): q_i = q_p q_rel, p_i = p_p + R(q_p) (0,0,L_p).
//               The tether stretch x_a - x_hang is a millimetre-sized difference of metre-sized positions, k_s = 2e3
//               N/m turns 1e-8 m of it into the whole error budget of a 3 mm twig: rest rotations, sin / cos of the
//               joint angles and the chain of products are therefore fp64, and the hang point of every apple is
//               formed here, where the fp64 pose is at hand.
// Publish of an inner link for its children (seven doubles): q in M0, M1, p in PD and XR.xy.
__device__ __forceinline__ void link_fk(const int i, const Sm &s, const Gm &g) {
  float4 *rec = s.P + 7 * i;
  const float4 cs = rec[kCS];
  uint32_t tw = __float_as_uint(cs.w);
  const Qd qrel = load_qd(rec);
  Qd qp;
  qp.w = 1.0; qp.x = 0.0; qp.y = 0.0; qp.z = 0.0;
  double pp[3] = {0, 0, 0};
  uint32_t snapped_p = 0u;
  if (!(tw & kTrunk)) {
    const float4 *par = s.P + 7 * (int)(tw & kParMask);
    qp = load_qd(par);
    const double2 b0 = *reinterpret_cast<const double2 *>(par + kPD);
    pp[0] = b0.x; pp[1] = b0.y; pp[2] = *reinterpret_cast<const double *>(par + kXR);
    snapped_p = __float_as_uint(par[kCS].w) & kSnapped;
  }
  const Qd q = qmul(qp, qrel);
  const double rz = (double)cs.z;
  double pw[3];
  pw[0] = pp[0] + rz * (2.0 * (qp.x * qp.z + qp.w * qp.y));
  pw[1] = pp[1] + rz * (2.0 * (qp.y * qp.z - qp.w * qp.x));
  pw[2] = pp[2] + rz * (1.0 - 2.0 * (qp.x * qp.x + qp.y * qp.y));
  tw = (tw & ~kSnapped) | (((tw & kRuptured) || snapped_p) ? kSnapped : 0u);
  rec[kCS].w = __uint_as_float(tw);
  const float4 qf = make_float4((float)q.w, (float)q.x, (float)q.y, (float)q.z);
  // hang points of the apples on this link: anchor - x_hang (the anchor is the rest hang point, fp64)
  if (tw & kHasApples) {
    const int4 t2 = __ldg(g.topo2 + i);
    const int Ap = s.Ap, ast = t2.x & 0xffff, nap = t2.x >> 16;
    double R[9];
    R[0] = 1 - 2 * (q.y * q.y + q.z * q.z); R[1] = 2 * (q.x * q.y - q.w * q.z);     R[2] = 2 * (q.x * q.z + q.w * q.y);
    R[3] = 2 * (q.x * q.y + q.w * q.z);     R[4] = 1 - 2 * (q.x * q.x + q.z * q.z); R[5] = 2 * (q.y * q.z - q.w * q.x);
    R[6] = 2 * (q.x * q.z - q.w * q.y);     R[7] = 2 * (q.y * q.z + q.w * q.x);     R[8] = 1 - 2 * (q.x * q.x + q.y * q.y);
    for (int a = ast; a < ast + nap; a++) {
      const double ox = s.ao[a], oy = s.ao[Ap + a], oz = s.ao[2 * Ap + a];
#pragma unroll
      for (int k = 0; k < 3; k++) {
        const double xh = pw[k] + R[3 * k] * ox + R[3 * k + 1] * oy + R[3 * k + 2] * oz;
        const float2 dd = split2(__ldg(g.anchor + (size_t)k * Ap + a) - xh);
        s.hd[(2 * k) * Ap + a] = dd.x; s.hd[(2 * k + 1) * Ap + a] = dd.y;
      }
      s.aq[a] = qf.x; s.aq[Ap + a] = qf.y; s.aq[2 * Ap + a] = qf.z; s.aq[3 * Ap + a] = qf.w;
    }
  }
  for (int k = 0; k < s.wr->n; k++)
    if (s.wr->body[k] == i) s.wq[k] = qf;
  if ((tw >> kNcShift) & kNcMask) {
    store_qd(rec, q);
    *reinterpret_cast<double2 *>(rec + kPD) = make_double2(pw[0], pw[1]);
    *reinterpret_cast<double *>(rec + kXR) = pw[2];
  }
}

// diagonal terms of the two DoF of a joint: arm + h (c_d K + D_f) + h^2 K (Eq. 4; a ruptured joint has K = 0 and only the
// post-rupture friction damper D_f, if any)
__device__ __forceinline__ float2 diag_terms(const int i, const uint32_t tw, const float kd, const Sm &s, const Gm &g,
                                             const ob_params &P) {
  const float Kt = (tw & kRuptured) ? 0.f : kd, Df = (tw & kRuptured) ? kd : 0.f;   // staged: K, or D_f of a ruptured joint
  float dt0 = P.h * (P.c_d * Kt + Df) + P.h * P.h * Kt, dt1 = dt0;
  if (g.arm) {
    dt0 += __ldg(g.arm + i);
    dt1 += __ldg(g.arm + s.Np + i);
  }
  return make_float2(dt0, dt1);
}

// velocity-proportional damping coefficient of a link (A32), reduced on snapped sub-trees (PAPER.md:141
// "a snapped sub-tree's linear drag is also reduced"; A35)
__device__ __forceinline__ float link_alpha(const uint32_t tw, const ob_params &P) {
  return (tw & kSnapped) ? P.mass_damping * P.snap_drag_scale : P.mass_damping;
}

// effective link inertia (m, m c, I about the joint, I_zz): the link's own, times (1 + h alpha) for the implicit
// mass-proportional damping (A32), plus the virtual tether masses h^2 k_s of the attached apples that hang on the
// link axis (A15).  Apples off the axis set kOffax in the returned topology word and are added one by one.
__device__ __forceinline__ float4 eff_inertia(const int i, uint32_t &tw, float4 c4, const Sm &s, const Gm &g,
                                              const ob_params &P) {
  const float sc = 1.f + P.h * link_alpha(tw, P);
  c4.x *= sc; c4.y *= sc; c4.z *= sc; c4.w *= sc;
  if (P.tether_implicit && (tw & kHasApples)) {
    tw &= ~kOffax;
    const int Ap = s.Ap;
    const int4 t2 = __ldg(g.topo2 + i);
    const int ast = t2.x & 0xffff, nap = t2.x >> 16;
    for (int a = ast; a < ast + nap; a++) {
      if (!s.att[a]) continue;
      const float mv = P.h * P.h * s.ak[a];                     // virtual point mass h^2 k_s at the hang point
      const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
      if (o.x == 0.f && o.y == 0.f) { c4.x += mv; c4.y += mv * o.z; c4.z += mv * o.z * o.z; }   // stays a body of revolution
      else tw |= kOffax;
    }
  }
  return c4;
}

// Tether of one apple (Eq. 6 / Eq. 7): the tether force and |f_s| for phase D, and the clamped
// reaction on the link as a spatial force (n, f) in link coordinates, which B1 subtracts from the link's bias force.
// A flat pass over the apples between A2 (which left the velocity of every apple-carrying link in its record) and B1:
// every lane has an apple, nothing of it sits in the level-by-level chain.
__device__ __forceinline__ void apple_forces(const int a, const Sm &s, const ob_params &P) {
  const int Ap = s.Ap;
  if (!s.att[a]) {
    s.aq[a] = 0.f; s.aq[Ap + a] = 0.f; s.aq[2 * Ap + a] = 0.f; s.aq[3 * Ap + a] = 0.f;
    s.hd[4 * Ap + a] = 0.f; s.hd[5 * Ap + a] = 0.f;
    return;
  }
  const float4 *rec = s.P + 7 * s.alnk[a];
  const float4 t0 = rec[kXR];
  const float4 t1 = rec[kIN];
  const float3 om = f3(t0.x, t0.y, t0.z), vl = f3(t0.w, t1.x, t1.y);
  const float4 qw = make_float4(s.aq[a], s.aq[Ap + a], s.aq[2 * Ap + a], s.aq[3 * Ap + a]);   // world rotation of the link
  const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
  const float ks = s.ak[a], cdamp = s.ac[a], ma = s.am[a];
  const float eta_h = P.tether_implicit ? P.h : 0.f;
  // x_a - x_hang = (anchor - x_hang) + sag + u: the apple is stored as u = x_a - (anchor + sag), sag = m g / k_s, and
  // phase A1 left anchor - x_hang in fp64 (as two floats).  At rest the spring force k_s sag and the weight m g cancel:
  // they are never formed.  With du = (anchor - x_hang) + u (millimetres), exactly:
  //   f_s = -k_s du - m g,   f_react = k_s (du - eta h v_hang)   (Eq. 7: the weight drops out),
  //   apple: g + (f_s - c_s v) / m = (-k_s du - c_s v) / m        (phase D adds the user force and integrates)
  // so a settled tree sees rounding of the small deviations only, not of two 2 N forces that cancel.
  const float3 du = f3((float)(join2(s.hd[a], s.hd[Ap + a]) + (double)s.u[a]),
                       (float)(join2(s.hd[2 * Ap + a], s.hd[3 * Ap + a]) + (double)s.u[Ap + a]),
                       (float)(join2(s.hd[4 * Ap + a], s.hd[5 * Ap + a]) + (double)s.u[2 * Ap + a]));
  const float3 vh = rot_up(qw, vl + cross(om, o));                      // world velocity of the hang point
  const float3 fe = (-ks) * du;                                          // elastic force beyond the rest sag
  const float3 fs = f3(fe.x - ma * P.gravity[0], fe.y - ma * P.gravity[1], fe.z - ma * P.gravity[2]);
  const float3 va = f3(s.v[a], s.v[Ap + a], s.v[2 * Ap + a]);
  s.ft[a] = fe.x - cdamp * va.x; s.ft[Ap + a] = fe.y - cdamp * va.y; s.ft[2 * Ap + a] = fe.z - cdamp * va.z;
  s.fsn[a] = sqrtf(dot(fs, fs));
  float3 fr = f3(ks * (du.x - eta_h * vh.x), ks * (du.y - eta_h * vh.y), ks * (du.z - eta_h * vh.z));
  const float nr = sqrtf(dot(fr, fr));
  if (nr > P.react_max) fr = (P.react_max / nr) * fr;                   // clamp
  const float3 fl = rot_down(qw, fr);
  const float3 nl = cross(o, fl);
  s.aq[a] = nl.x; s.aq[Ap + a] = nl.y; s.aq[2 * Ap + a] = nl.z; s.aq[3 * Ap + a] = fl.x;
  s.hd[4 * Ap + a] = fl.y; s.hd[5 * Ap + a] = fl.z;
}

// The three rails of PAPER.md:398 (App. B) on an applied force F on a FREE body of mass m moving with velocity v at the
// application point (reading A36): power fade of the part of F along v between rail_fade v_lim and v_lim; impulse cap
// |F| <= m max(v_lim - v . F^, 0) / h; speed brake - rail_brake m (|v| - v_lim) v^ above v_lim.
// (out of line: the callers come here only with rail_speed > 0)
__device__ __noinline__ float3 apply_rails(const ob_params &P, const float m, const float3 v, float3 F) {
  const float vl = P.rail_speed;
  const float vn = sqrtf(dot(v, v));
  float3 vh = f3(0, 0, 0);
  if (vn > 0.f) {
    vh = (1.f / vn) * v;
    const float Fp = dot(F, vh);
    if (Fp > 0.f) {
      const float vf = P.rail_fade * vl;
      const float fade = vn <= vf ? 1.f : (vn >= vl ? 0.f : (vl - vn) / (vl - vf));
      F = F - ((1.f - fade) * Fp) * vh;
    }
  }
  const float Fn = sqrtf(dot(F, F));
  if (Fn > 0.f) {
    const float vF = dot(v, F) / Fn;
    const float cap = m * fmaxf(vl - vF, 0.f) / P.h;
    if (Fn > cap) F = (cap / Fn) * F;
  }
  if (vn > vl) F = F - (P.rail_brake * m * (vn - vl)) * vh;
  return F;
}

// user wrenches on one link (disabled on snapped sub-trees; where they are not, a link of a snapped
// sub-tree is a free body and its wrench goes through the rails), subtracted from its bias force
__device__ __forceinline__ void wrench_forces(const int i, const uint32_t tw, const float m, const float3 om, const float3 vl,
                                              const Sm &s, const ob_params &P, float3 &n, float3 &f) {
  const int nwr = s.wr->n;
  for (int q = 0; q < nwr; q++) {
    if (s.wr->body[q] != i) continue;
    if ((tw & kSnapped) && P.forces_off_on_snapped) continue;
    float3 fl = rot_down(s.wq[q], f3(s.wr->force[q][0], s.wr->force[q][1], s.wr->force[q][2]));
    const float3 pt = f3(s.wr->point[q][0], s.wr->point[q][1], s.wr->point[q][2]);
    if ((tw & kSnapped) && P.rail_speed > 0.f) fl = apply_rails(P, m, vl + cross(om, pt), fl);   // all in link coordinates
    f = f - fl;
    n = n - cross(pt, fl);
  }
}

// project the accumulated bias force on the joint axes -> rhs b (XR[i].zw), the diagonal terms of both DoF (PD[i].zw),
// the effective inertia (IN[i]), and publish (n, f) in the parent frame (M0[i], M1[i].xy)
// (th, w, Ki, c4 = q, qd, K, inertia of the link: the caller loads them at the top of its turn, with its other global
// inputs)
__device__ __forceinline__ void finish_bias(const Jt &j, const M3 &R, const int i, const float2 th, const float2 w,
                                            const float Ki, const float4 c4, float3 n, float3 f, const Sm &s,
                                            const Gm &g, const DevCtx &c) {
  const ob_params &P = c.P;
  float4 *rec = s.P + 7 * i;
  uint32_t tw = j.tw;
  // spring-damper part of the rhs and of the diagonal (Eq. 4); a ruptured joint has K = D = 0
  const float Kt = (tw & kRuptured) ? 0.f : Ki, Dt = P.c_d * Kt + ((tw & kRuptured) ? Ki : 0.f);   // Ki: K, or D_f (staged)
  const float2 kq = make_float2(Kt * th.x + (Dt + P.h * Kt) * w.x, Kt * th.y + (Dt + P.h * Kt) * w.y);
  rec[kXR] = make_float4(0.f, 0.f, P.h * (-(j.c2 * n.x + j.s2 * n.z) - kq.x), P.h * (-n.y - kq.y));
  {
    const float2 dt = diag_terms(i, tw, Ki, s, g, P);
    rec[kPD] = make_float4(0.f, 0.f, dt.x, dt.y);
  }
  rec[kIN] = eff_inertia(i, tw, c4, s, g, P);
  if (tw != j.tw) rec[kCS].w = __uint_as_float(tw);
  if (!(tw & kTrunk)) {
    float3 np, fp;
    force_up_m(R, j.rz, n, f, np, fp);
    rec[kM0] = make_float4(np.x, np.y, np.z, fp.x);
    rec[kM1] = make_float4(fp.y, fp.z, 0.f, 0.f);
  }
}

// ---- A2 ----  velocity, bias acceleration (gravity as base acceleration), own bias force
//               f = I a + v x* I v - tether reactions - user wrenches  (RNEA with qdd = 0)
// An inner link leaves (om, vl, al, aln) for its children in XR, IN, PD.xy, M1.zw and parks its force in M0, M1.xy;
// so does a link that carries apples (the apple pass reads its velocity).
__device__ __forceinline__ void link_bias(const int i, const World *wd, const Sm &s, const Gm &g, const DevCtx &c) {
  const ob_params &P = c.P;
  float4 *rec = s.P + 7 * i;
  const float4 sq = rec[kXR], c4 = rec[kIN];                      // (q, qd), inertia, K: staged by the flat pass
  const float2 th = make_float2(sq.x, sq.y), w = make_float2(sq.z, sq.w);
  const float Ki = rec[kPD].x;
  const Jt j = load_jt(s.P, i);
  const uint32_t tw = j.tw;
  float3 wp = f3(0, 0, 0), vp = f3(0, 0, 0), alp = f3(0, 0, 0);
  float3 ap = f3(-P.gravity[0], -P.gravity[1], -P.gravity[2]);   // world = parent of the trunk: at rest, (0; -g)
  if (!(tw & kTrunk)) {
    const float4 *par = s.P + 7 * (int)(tw & kParMask);
    const float4 t0 = par[kXR], t1 = par[kIN];
    const float4 t2 = par[kPD], t3 = par[kM1];
    wp = f3(t0.x, t0.y, t0.z); vp = f3(t0.w, t1.x, t1.y);
    alp = f3(t1.z, t1.w, t2.x); ap = f3(t2.y, t3.z, t3.w);
  }
  const float c2 = j.c2, s2 = j.s2;
  const float3 vJ = f3(c2 * w.x, w.y, s2 * w.x);
  const M3 R = quat_mat(j.q);
  float3 om, vl, al, aln;
  motion_down_m(R, j.rz, wp, vp, om, vl);
  om = om + vJ;
  motion_down_m(R, j.rz, alp, ap, al, aln);
  const float ww = w.x * w.y;
  al = al + f3(-s2 * ww, 0.f, c2 * ww) + cross(om, vJ);
  aln = aln + cross(vl, vJ);
  // a link with children waits for them, a link with apples for the apple pass: both park
  const bool inner = (((tw >> kNcShift) & kNcMask) | (tw & kHasApples)) != 0u;
  // f = I a + v x* I v  (cylinder: com on +z)
  const float m = c4.x, mc = c4.y, Io = c4.z, Iz = c4.w;
  float3 n = f3(Io * al.x - mc * aln.y, Io * al.y + mc * aln.x, Iz * al.z);
  float3 f = f3(m * aln.x + mc * al.y, m * aln.y - mc * al.x, m * aln.z);
  const float3 hn = f3(Io * om.x - mc * vl.y, Io * om.y + mc * vl.x, Iz * om.z);
  const float3 hf = f3(m * vl.x + mc * om.y, m * vl.y - mc * om.x, m * vl.z);
  n = n + cross(om, hn) + cross(vl, hf);
  f = f + cross(om, hf);
  if (P.mass_damping != 0.f) {            // velocity-proportional damping F = -c_v m v, tau = -c_omega I omega (
    const float al_i = link_alpha(tw, P);   // A32, A35): minus alpha times the link's spatial momentum
    n = n + al_i * hn; f = f + al_i * hf;
  }
  wrench_forces(i, tw, c4.x, om, vl, s, P, n, f);
  if (inner) {                                                    // parked until B1 adds the children / the apples
    const float2 dt = diag_terms(i, tw, Ki, s, g, P);
    rec[kXR] = make_float4(om.x, om.y, om.z, vl.x);
    rec[kIN] = make_float4(vl.y, vl.z, al.x, al.y);
    rec[kPD] = make_float4(al.z, aln.x, dt.x, dt.y);
    rec[kM0] = make_float4(n.x, n.y, n.z, f.x);
    rec[kM1] = make_float4(f.y, f.z, aln.y, aln.z);
  } else {
    finish_bias(j, R, i, th, w, Ki, c4, n, f, s, g, c);
  }
}

// ---- B1 ----  one inner link: its parked bias force plus what its children sent up
__device__ __forceinline__ void link_bias_up(const int i, const Jt &j, const Sm &s, const Gm &g, const DevCtx &c) {
  const float4 sq = s.P[7 * i + kXR], c4 = s.P[7 * i + kIN];     // staged by the flat pass between A2 and B1
  const float2 th = make_float2(sq.x, sq.y), w = make_float2(sq.z, sq.w);
  const float Ki = s.P[7 * i + kPD].x;
  const float4 u0 = s.P[7 * i + kM0];
  const float4 v0 = s.P[7 * i + kM1];
  float3 n = f3(u0.x, u0.y, u0.z), f = f3(u0.w, v0.x, v0.y);
  gather_children(s.P, s.P + 7 * s.Np, (int)((j.tw >> kChShift) & kParMask), (int)((j.tw >> kNcShift) & kNcMask), n, f);
  if (j.tw & kHasApples) {                                  // the reactions of its apples, in apple order
    const int Ap = s.Ap, ap = __float_as_int(s.X21[i]), ast = ap & 0xffff, nap = ap >> 16;
    for (int a = ast; a < ast + nap; a++) {
      n = n - f3(s.aq[a], s.aq[Ap + a], s.aq[2 * Ap + a]);
      f = f - f3(s.aq[3 * Ap + a], s.hd[4 * Ap + a], s.hd[5 * Ap + a]);
    }
  }
  finish_bias(j, quat_mat(j.q), i, th, w, Ki, c4, n, f, s, g, c);
}

// ------------------------------------------------------------------------------------------------------
// phase F, precond = 2: articulated-body inertia of one link (Featherstone).  The system matrix
// A = M + M_teth + diag(arm + hD + h^2 K) is the joint-space inertia of the tree whose joints carry the armature
// d = arm + hD + h^2 K, so the articulated-body recursion factorises it exactly in O(N):
//   I^A_i = I_i + sum_children X^T I^a_c X,   U = I^A S,   D = S^T U + diag(d),   K = U D^-1,   I^a = I^A - K U^T.
// A spatial inertia is kept as three 3 x 3 blocks, n = A alpha + B a, f = B^T alpha + C a (A, C symmetric); the
// 21 floats of I^a go to the parent through the link's own record (IN, PD, M0, M1, XR) and the X21 plane, already
// rotated into the parent's frame and moved to the parent's origin.  K and D^-1 stay in the factor planes.
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void rot_block(const M3 &R, const float *M, float *out) {   // out = R M R^T (3 x 3, row-major)
  float T[9];
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int cc = 0; cc < 3; cc++) T[3 * r + cc] = R.a[3 * r] * M[cc] + R.a[3 * r + 1] * M[3 + cc] + R.a[3 * r + 2] * M[6 + cc];
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int cc = 0; cc < 3; cc++) out[3 * r + cc] = T[3 * r] * R.a[3 * cc] + T[3 * r + 1] * R.a[3 * cc + 1] + T[3 * r + 2] * R.a[3 * cc + 2];
}

__device__ __noinline__ void factor_link(const int i, const World *wd, const DevCtx &c) {
  const Sm s = carve(wd);
  const Gm g = wd->g;
  const ob_params &P = c.P;
  float4 *rec = s.P + 7 * i;
  const Jt j = load_jt(s.P, i);
  uint32_t tw = j.tw;
  const float Ki = s.X21[i];                                   // staged by the flat pass before the sweep
  const float4 eff = eff_inertia(i, tw, rec[kIN], s, g, P);
  const float2 dt = diag_terms(i, tw, Ki, s, g, P);
  if (tw != j.tw) rec[kCS].w = __uint_as_float(tw);
  // own inertia: body of revolution about +z through the joint
  float A[9] = {eff.z, 0, 0, 0, eff.z, 0, 0, 0, eff.w};
  float B[9] = {0, -eff.y, 0, eff.y, 0, 0, 0, 0, 0};
  float C[9] = {eff.x, 0, 0, 0, eff.x, 0, 0, 0, eff.x};
  if (tw & kOffax) {                                       // virtual tether masses off the axis: point masses
    const int Ap = s.Ap;
    const int4 t2 = __ldg(g.topo2 + i);
    const int ast = t2.x & 0xffff, nap = t2.x >> 16;
    for (int a = ast; a < ast + nap; a++) {
      if (!s.att[a]) continue;
      const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
      if (o.x == 0.f && o.y == 0.f) continue;
      const float mv = P.h * P.h * s.ak[a];
      const float oo = dot(o, o);
      A[0] += mv * (oo - o.x * o.x); A[4] += mv * (oo - o.y * o.y); A[8] += mv * (oo - o.z * o.z);
      A[1] -= mv * o.x * o.y; A[3] -= mv * o.x * o.y; A[2] -= mv * o.x * o.z; A[6] -= mv * o.x * o.z;
      A[5] -= mv * o.y * o.z; A[7] -= mv * o.y * o.z;
      B[1] -= mv * o.z; B[2] += mv * o.y; B[3] += mv * o.z; B[5] -= mv * o.x; B[6] -= mv * o.y; B[7] += mv * o.x;
      C[0] += mv; C[4] += mv; C[8] += mv;
    }
  }
  const int fc = (int)((tw >> kChShift) & kParMask), nc = (int)((tw >> kNcShift) & kNcMask);
#pragma unroll 1
  for (int k = 0; k < nc; k++) {                           // ascending order: a fixed summation order
    const float4 *ch = s.P + 7 * (fc + k);
    const float4 a0 = ch[kIN], a1 = ch[kPD], a2 = ch[kM0], a3 = ch[kM1], a4 = ch[kXR];
    const float a5 = s.X21[fc + k];
    A[0] += a0.x; A[4] += a0.y; A[8] += a0.z; A[1] += a0.w; A[3] += a0.w;
    A[2] += a1.x; A[6] += a1.x; A[5] += a1.y; A[7] += a1.y;
    C[0] += a1.z; C[4] += a1.w; C[8] += a2.x; C[1] += a2.y; C[3] += a2.y; C[2] += a2.z; C[6] += a2.z; C[5] += a2.w; C[7] += a2.w;
    B[0] += a3.x; B[1] += a3.y; B[2] += a3.z; B[3] += a3.w; B[4] += a4.x; B[5] += a4.y; B[6] += a4.z; B[7] += a4.w; B[8] += a5;
  }
  // U = I^A S, S = [(c2, 0, s2; 0), (0, 1, 0; 0)]
  const float c2 = j.c2, s2 = j.s2;
  const float3 u1n = f3(c2 * A[0] + s2 * A[2], c2 * A[3] + s2 * A[5], c2 * A[6] + s2 * A[8]);
  const float3 u1f = f3(c2 * B[0] + s2 * B[6], c2 * B[1] + s2 * B[7], c2 * B[2] + s2 * B[8]);      // B^T s1
  const float3 u2n = f3(A[1], A[4], A[7]);
  const float3 u2f = f3(B[3], B[4], B[5]);
  const float d11 = c2 * u1n.x + s2 * u1n.z + dt.x, d12 = u1n.y, d22 = u2n.y + dt.y;
  const float idet = __fdividef(1.f, d11 * d22 - d12 * d12);     // (a preconditioner: an approximate reciprocal will do)
  const float i11 = d22 * idet, i12 = -d12 * idet, i22 = d11 * idet;
  const float3 k1n = i11 * u1n + i12 * u2n, k1f = i11 * u1f + i12 * u2f;
  const float3 k2n = i12 * u1n + i22 * u2n, k2f = i12 * u1f + i22 * u2f;
  const uint32_t slot = s.SL[i];
  if (slot != kNoSlot) {
    s.FAC[slot] = make_float4(k1n.x, k1n.y, k1n.z, k1f.x);
    s.FAC[s.NFp + slot] = make_float4(k1f.y, k1f.z, k2n.x, k2n.y);
    s.FAC[2 * s.NFp + slot] = make_float4(k2n.z, k2f.x, k2f.y, k2f.z);
    s.FAC[3 * s.NFp + slot] = make_float4(i11, i12, i22, 0.f);
  }
  if (tw & kTrunk) return;
  // I^a = I^A - K U^T (upper triangles of A, C; mirrored below)
  const float k1na[3] = {k1n.x, k1n.y, k1n.z}, k2na[3] = {k2n.x, k2n.y, k2n.z}, k1fa[3] = {k1f.x, k1f.y, k1f.z}, k2fa[3] = {k2f.x, k2f.y, k2f.z};
  const float u1na[3] = {u1n.x, u1n.y, u1n.z}, u2na[3] = {u2n.x, u2n.y, u2n.z}, u1fa[3] = {u1f.x, u1f.y, u1f.z}, u2fa[3] = {u2f.x, u2f.y, u2f.z};
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int cc = 0; cc < 3; cc++) {
      B[3 * r + cc] -= k1na[r] * u1fa[cc] + k2na[r] * u2fa[cc];
      if (cc >= r) {
        A[3 * r + cc] -= k1na[r] * u1na[cc] + k2na[r] * u2na[cc];
        C[3 * r + cc] -= k1fa[r] * u1fa[cc] + k2fa[r] * u2fa[cc];
      }
    }
  A[3] = A[1]; A[6] = A[2]; A[7] = A[5]; C[3] = C[1]; C[6] = C[2]; C[7] = C[5];
  // into the parent's orientation, then from the joint (at r = (0,0,rz) of the parent) to the parent's origin:
  //   C' = C,  B' = B + r x C,  A' = A - B r x + r x B^T - r x C r x     (r x = rz [[0,-1,0],[1,0,0],[0,0,0]])
  const M3 R = quat_mat(j.q);
  float Ar[9], Br[9], Cr[9];
  rot_block(R, A, Ar); rot_block(R, B, Br); rot_block(R, C, Cr);
  const float z = j.rz, zz = z * z;
  // G = B r x: column 0 = z B[:,1], column 1 = -z B[:,0], column 2 = 0;  A' = A - G - G^T + z^2 [[C11, -C01, 0], [-C01, C00, 0], 0]
  const float g00 = z * Br[1], g10 = z * Br[4], g20 = z * Br[7], g01 = -z * Br[0], g11 = -z * Br[3], g21 = -z * Br[6];
  const float Axx = Ar[0] - 2.f * g00 + zz * Cr[4], Ayy = Ar[4] - 2.f * g11 + zz * Cr[0], Azz = Ar[8];
  const float Axy = Ar[1] - g01 - g10 - zz * Cr[1], Axz = Ar[2] - g20, Ayz = Ar[5] - g21;
  // B' = B + r x C: row 0 -= z C[1,:], row 1 += z C[0,:]
  const float B00 = Br[0] - z * Cr[3], B01 = Br[1] - z * Cr[4], B02 = Br[2] - z * Cr[5];
  const float B10 = Br[3] + z * Cr[0], B11 = Br[4] + z * Cr[1], B12 = Br[5] + z * Cr[2];
  rec[kIN] = make_float4(Axx, Ayy, Azz, Axy);
  rec[kPD] = make_float4(Axz, Ayz, Cr[0], Cr[4]);
  rec[kM0] = make_float4(Cr[8], Cr[1], Cr[2], Cr[5]);
  rec[kM1] = make_float4(B00, B01, B02, B10);
  rec[kXR] = make_float4(B11, B12, Br[6], Br[7]);
  s.X21[i] = Br[8];
}

// ------------------------------------------------------------------------------------------------------
// phase F, precond <= 1: composite rigid-body inertia about the link origin (mass, first moment h, symmetric I) ->
// exact diagonal of M -> Jacobi factors 1 / diag(A) (IDG[i]); composite inertia to the parent through M0, M1, PD.xy
// ------------------------------------------------------------------------------------------------------
__device__ __noinline__ void composite_link(const int i, const World *wd, const DevCtx &c) {
  const Sm s = carve(wd);
  const Gm g = wd->g;
  const int Ap = s.Ap;
  const ob_params &P = c.P;
  float4 *rec = s.P + 7 * i;
  const Jt j = load_jt(s.P, i);
  uint32_t tw = j.tw;
  float4 c4 = rec[kIN];                                        // staged by the flat pass before the sweep
  const float2 dt = diag_terms(i, tw, s.X21[i], s, g, P);
  {
    const float sc = 1.f + P.h * link_alpha(tw, P);
    c4.x *= sc; c4.y *= sc; c4.z *= sc; c4.w *= sc;
  }
  float cm = c4.x;
  float3 ch3 = f3(0.f, 0.f, c4.y);
  float Ixx = c4.z, Iyy = c4.z, Izz = c4.w, Ixy = 0.f, Ixz = 0.f, Iyz = 0.f;
  if (P.tether_implicit && (tw & kHasApples)) {
    const int4 t2 = __ldg(g.topo2 + i);
    const int ast = t2.x & 0xffff, nap = t2.x >> 16;
    for (int a = ast; a < ast + nap; a++) {
      if (!s.att[a]) continue;
      const float mv = P.h * P.h * s.ak[a];
      const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
      cm += mv; ch3 = ch3 + mv * o;
      Ixx += mv * (o.y * o.y + o.z * o.z); Iyy += mv * (o.x * o.x + o.z * o.z); Izz += mv * (o.x * o.x + o.y * o.y);
      Ixy -= mv * o.x * o.y; Ixz -= mv * o.x * o.z; Iyz -= mv * o.y * o.z;
    }
  }
  const int fc = (int)((tw >> kChShift) & kParMask), nc = (int)((tw >> kNcShift) & kNcMask);
  for (int ch = fc; ch < fc + nc; ch++) {
    const float4 u0 = s.P[7 * ch + kM0], u1 = s.P[7 * ch + kM1];
    const float2 u2 = *reinterpret_cast<const float2 *>(s.P + 7 * ch + kPD);
    cm += u0.x;
    ch3 = ch3 + f3(u0.y, u0.z, u0.w);
    Ixx += u1.x; Iyy += u1.y; Izz += u1.z; Ixy += u1.w; Ixz += u2.x; Iyz += u2.y;
  }
  const float c2 = j.c2, s2 = j.s2;
  const float m1 = c2 * c2 * Ixx + 2.f * c2 * s2 * Ixz + s2 * s2 * Izz, m2 = Iyy;
  s.IDG[i] = make_float2(1.f / (m1 + dt.x), 1.f / (m2 + dt.y));
  if (!(tw & kTrunk)) {
    // composite inertia into the parent frame: rotate by R_rel, then move the origin by r = (0,0,rz)
    const M3 R = quat_mat(j.q);
    const float rz = j.rz;
    const float3 hp = mul(R, ch3);
    const float I[9] = {Ixx, Ixy, Ixz, Ixy, Iyy, Iyz, Ixz, Iyz, Izz};
    float Ip[9];
    rot_block(R, I, Ip);
    const float sh = 2.f * rz * hp.z + cm * rz * rz;
    rec[kM0] = make_float4(cm, hp.x, hp.y, hp.z + cm * rz);
    rec[kM1] = make_float4(Ip[0] + sh, Ip[4] + sh, Ip[8], Ip[1]);
    *reinterpret_cast<float2 *>(rec + kPD) = make_float2(Ip[2] - rz * hp.x, Ip[5] - rz * hp.y);
  }
}

// fence after level l of a top-down sweep / after level l of a bottom-up sweep (see "Order" above)
#define OB_FENCE_DOWN(l) { if ((l) + 1 < ntop) __syncwarp(); else __syncthreads(); }
#define OB_FENCE_UP(l) { if ((l) < ntop) __syncwarp(); else __syncthreads(); }

// ------------------------------------------------------------------------------------------------------
// the once-per-step sweeps as functions of their own (not inlined): their register pressure stays out of the
// allocation of the PCG loop.  The views of the world live in shared memory (World), the context is the kernel's
// __grid_constant__ parameter.
// ------------------------------------------------------------------------------------------------------
__device__ __noinline__ void sweep_kinematics(const World *wd, const DevCtx &c, const int nt, const int step) {
  const Sm s = carve(wd);
  const Gm g = wd->g;
  const int nlev = wd->nlev, ntop = wd->ntop, tid = threadIdx.x;
  const int l_first_down = tid < 32 ? 0 : ntop - 1;
  // ---- A0: joint rotations in fp64, flat (the two double sincos depend on nothing but the link's own q: kept out
  //      of the level-by-level chain) ----
#pragma unroll 1
  for (int i = tid; i < wd->N; i += nt) {
    link_joint(i, s, g);
    stage_link_inputs(i, s, g, false, step, c.P);       // for phase F (A1 leaves IN and PD.x of every link alone)
  }
  __syncthreads();
  // ---- A1: forward kinematics in fp64, hang points, top-down ----
#pragma unroll 1
  for (int l = l_first_down; l < nlev; l++) {
    const int le = s.lev[l + 1];
#pragma unroll 1
    for (int i = s.lev[l] + tid; i < le; i += nt) link_fk(i, s, g);
    OB_FENCE_DOWN(l)
  }
}

__device__ __noinline__ void sweep_factor(const World *wd, const DevCtx &c, const int nt) {
  const Sm s = carve(wd);
  const int nlev = wd->nlev, ntop = wd->ntop, N = wd->N, tid = threadIdx.x;
  const int l_last_up = tid < 32 ? 0 : ntop;
  const bool tree = wd->precond == 2;
  // ---- F: all leaves first (flat, evenly spread), then the inner links bottom-up ----
#pragma unroll 1
  for (int i = tid; i < N; i += nt)
    if (((__float_as_uint(s.P[7 * i + kCS].w) >> kNcShift) & kNcMask) == 0u) {
      if (tree) factor_link(i, wd, c); else composite_link(i, wd, c);
    }
  __syncthreads();
#pragma unroll 1
  for (int l = nlev - 2; l >= l_last_up; l--) {
    const int le = s.lev[l + 1];
#pragma unroll 1
    for (int i = s.lev[l] + tid; i < le; i += nt)
      if ((__float_as_uint(s.P[7 * i + kCS].w) >> kNcShift) & kNcMask) {
        if (tree) factor_link(i, wd, c); else composite_link(i, wd, c);
      }
    OB_FENCE_UP(l)
  }
  __syncthreads();
}

__device__ __noinline__ void sweep_bias(const World *wd, const DevCtx &c, const int nt, const int step) {
  const Sm s = carve(wd);
  const Gm g = wd->g;
  const int nlev = wd->nlev, ntop = wd->ntop, tid = threadIdx.x;
  const int l_first_down = tid < 32 ? 0 : ntop - 1, l_last_up = tid < 32 ? 0 : ntop;
#pragma unroll 1
  for (int i = tid; i < wd->N; i += nt) stage_link_inputs(i, s, g, true, step, c.P);
  __syncthreads();
  // ---- A2 (+ B1 for leaves): velocities, bias accelerations, bias forces, top-down ----
#pragma unroll 1
  for (int l = l_first_down; l < nlev; l++) {
    const int le = s.lev[l + 1];
#pragma unroll 1
    for (int i = s.lev[l] + tid; i < le; i += nt) link_bias(i, wd, s, g, c);
    OB_FENCE_DOWN(l)
  }
  // ---- the apples: tether forces, reactions on their links ----
#pragma unroll 1
  for (int a = tid; a < wd->A; a += nt) apple_forces(a, s, c.P);
  __syncthreads();
  // ---- B1: bias forces bottom-up over the parked links -> rhs b ----
#pragma unroll 1
  for (int i = tid; i < wd->N; i += nt) {               // what A2 left in the record of a parked link is dead now
    const uint32_t tw = __float_as_uint(s.P[7 * i + kCS].w);
    if (((tw >> kNcShift) & kNcMask) | (tw & kHasApples)) stage_link_inputs(i, s, g, true, step, c.P);
  }
  __syncthreads();
#pragma unroll 1
  for (int l = nlev - 1; l >= l_last_up; l--) {
    const int le = s.lev[l + 1];
#pragma unroll 1
    for (int i = s.lev[l] + tid; i < le; i += nt) {
      const Jt j = load_jt(s.P, i);
      if (((j.tw >> kNcShift) & kNcMask) | (j.tw & kHasApples)) link_bias_up(i, j, s, g, c);
    }
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

// z = P^-1 r for precond = 2 (r in XR.zw, z -> M1.zw): one bottom-up and one top-down sweep with the factors of phase F.
// FUSE: z -> PD.xy (= p) and the top-down pass of A p is done with it (see solve_down); returns this thread's share of
// p . A p from the links that turned around.
template <int NT, bool FUSE>
__device__ __forceinline__ float tree_solve(const Sm &s, const Gm &g, const DevCtx &c, const int otid, const int nlev,
                                            const int ntop) {
  float4 *const PL = s.P;
  const bool topw = otid < 32;
  const int l_last_up = topw ? 0 : ntop, l_first_down = topw ? 0 : ntop - 1;
#pragma unroll 1
  for (int l = nlev - 1; l >= l_last_up; l--) {
    const int le = s.lev[l + 1];
    if (l == nlev - 1) {
#pragma unroll 1
      for (int i = s.lev[l] + otid; i < le; i += NT) solve_up<false>(i, PL, s);
    } else {
#pragma unroll 1
      for (int i = s.lev[l] + otid; i < le; i += NT) solve_up<true>(i, PL, s);
    }
    OB_FENCE_UP(l)
  }
  __syncthreads();
  float part = 0.f;
#pragma unroll 1
  for (int l = l_first_down; l < nlev; l++) {
    const int le = s.lev[l + 1];
    const bool turn = FUSE && l == nlev - 1 && l >= ntop;   // (a tree that ends inside the top warp turns around there)
#pragma unroll 1
    for (int i = s.lev[l] + otid; i < le; i += NT) part += solve_down<FUSE>(i, PL, s, g, c, turn);
    OB_FENCE_DOWN(l)
  }
  return part;
}

template <int NT, int LPT>
__device__ __noinline__ int pcg_solve(const World *wd, const DevCtx &c, float2 *stage, int *flipp, const int otid,
                                      const bool top_warp, const float bb, const float bz, int *flags) {
  const Sm s = carve(wd);
  const Gm g = wd->g;
  const ob_params &P = c.P;
  const int tid = threadIdx.x, lane = tid & 31;
  const int Np = s.Np, N = wd->N, nlev = wd->nlev, ntop = wd->ntop;
  const bool tree = wd->precond == 2;
  float4 *const PL = s.P;
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
    if (top_lvl < ntop - 1) top_maxc = (int)((__float_as_uint(PL[7 * lane + kCS].w) >> kNcShift) & kNcMask);
  }
  top_maxc = __reduce_max_sync(0xffffffffu, top_maxc);
  int it = 0;
  bool bad = false;
  if (bb == 0.f) {
#pragma unroll
    for (int k = 0; k < LPT; k++) {
      const int i = otid + k * NT;
      if (i < N) PL[7 * i + kXR] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  } else if (!(bb < INFINITY)) {
    bad = true;
  } else {
#pragma unroll
    for (int k = 0; k < LPT; k++) {                 // first product: A x, i.e. p = x
      const int i = otid + k * NT;
      if (i < N) {
        const float4 xr = PL[7 * i + kXR], pd = PL[7 * i + kPD];
        PL[7 * i + kPD] = make_float4(xr.x, xr.y, pd.z, pd.w);
      }
    }
    bool first = true, have_down = false;
    float rz = 0.f, rr = 0.f, pAp_carry = 0.f;
    // stopping rule: |r| <= tol |b| in the 2-norm (cg_norm 0) or in the preconditioned norm (cg_norm 1, precond <= 1)
    const float tol2 = P.cg_tol * P.cg_tol * (P.cg_norm ? bz : bb);
    for (;;) {
      // ---- A p.  The n_top leading levels live in the top warp, lane = link: own record in registers, parents
      //      and children by shuffle, no barrier.  The other levels are swept by the whole CTA, one block
      //      barrier per level; the deepest level turns around at once ----
      float pAp_part = pAp_carry;
      if (!have_down) {
      if (top_warp) {
        const int me = lane < ntopN ? lane : Np;             // idle lanes work on the zero record
        float4 *rec = PL + 7 * me;
        const float4 pd = rec[kPD];
        const Jt j = load_jt(PL, me);
        const int parl = (j.tw & kTrunk) ? lane : (int)(j.tw & kParMask);   // the trunk's "parent" is all zero at level 0
        const float3 sp = f3(j.c2 * pd.x, pd.y, j.s2 * pd.x);
        float3 al = f3(0, 0, 0), a = f3(0, 0, 0);
#pragma unroll 1
        for (int l = 0; l < ntop; l++) {                      // branch-free: every lane computes, level l commits
          float3 alp, ap;
          alp.x = __shfl_sync(0xffffffffu, al.x, parl); alp.y = __shfl_sync(0xffffffffu, al.y, parl);
          alp.z = __shfl_sync(0xffffffffu, al.z, parl);
          ap.x = __shfl_sync(0xffffffffu, a.x, parl); ap.y = __shfl_sync(0xffffffffu, a.y, parl);
          ap.z = __shfl_sync(0xffffffffu, a.z, parl);
          float3 nal, na;
          motion_down(j, alp, ap, nal, na);
          nal = nal + sp;
          const bool mine = top_lvl == l;
          al.x = mine ? nal.x : al.x; al.y = mine ? nal.y : al.y; al.z = mine ? nal.z : al.z;
          a.x = mine ? na.x : a.x; a.y = mine ? na.y : a.y; a.z = mine ? na.z : a.z;
        }
        if (lane < ntopN) {
          rec[kM0] = make_float4(al.x, al.y, al.z, a.x);
          rec[kM1] = make_float4(a.y, a.z, 0.f, 0.f);
        }
      }
      __syncthreads();
#pragma unroll 1
      for (int l = ntop; l < nlev; l++) {
        const int le = s.lev[l + 1];
        const bool deepest = l == nlev - 1;
#pragma unroll 1
        for (int i = s.lev[l] + otid; i < le; i += NT) {
          float4 *rec = PL + 7 * i;
          const float4 pd = rec[kPD];
          const Jt j = load_jt(PL, i);
          float3 al, a;
          mv_down(j, PL, pd, al, a);
          if (deepest) {
            pAp_part += mv_up<false>(j, PL, PL + 7 * Np, i, pd, al, a, s, g, c);
          } else {
            rec[kM0] = make_float4(al.x, al.y, al.z, a.x);
            rec[kM1] = make_float4(a.y, a.z, 0.f, 0.f);
          }
        }
        __syncthreads();
      }
      }                                              // (after a fused solve the top-down pass is done already)
      have_down = false; pAp_carry = 0.f;
#pragma unroll 1
      for (int l = nlev - 2; l >= ntop; l--) {
        const int le = s.lev[l + 1];
#pragma unroll 1
        for (int i = s.lev[l] + otid; i < le; i += NT) {
          const float4 *rec = PL + 7 * i;
          const float4 pd = rec[kPD];
          const Jt j = load_jt(PL, i);
          const float4 u = rec[kM0], v = rec[kM1];
          pAp_part += mv_up<true>(j, PL, PL + 7 * Np, i, pd, f3(u.x, u.y, u.z), f3(u.w, v.x, v.y), s, g, c);
        }
        __syncthreads();
      }
      if (top_warp) {
        const int me = lane < ntopN ? lane : Np;
        float4 *rec = PL + 7 * me;
        const float4 pd = rec[kPD];
        const Jt j = load_jt(PL, me);
        const float4 u = rec[kM0], v = rec[kM1];
        const float3 al = f3(u.x, u.y, u.z), a = f3(u.w, v.x, v.y);
        const int fc = (int)((j.tw >> kChShift) & kParMask), nc = (int)((j.tw >> kNcShift) & kNcMask);
        // own inertia force; the children of the last top level are in shared memory, all others are lanes
        float3 n0, f0;
        own_inertia_force(rec[kIN], al, a, n0, f0);
        if (j.tw & kOffax) {
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
          float3 nun, nuf;
          force_up(j, n, f, nun, nuf);
          const bool mine = top_lvl == l;
          t1 = mine ? nt1 : t1; t2 = mine ? nt2 : t2;
          un.x = mine ? nun.x : un.x; un.y = mine ? nun.y : un.y; un.z = mine ? nun.z : un.z;
          uf.x = mine ? nuf.x : uf.x; uf.y = mine ? nuf.y : uf.y; uf.z = mine ? nuf.z : uf.z;
        }
        if (lane < ntopN) {
          rec[kM1] = make_float4(v.x, v.y, t1, t2);
          pAp_part += pd.x * t1 + pd.y * t2;
        }
      }
      // ---- x, r; z = P^-1 r; p ----
      float rz_p = 0.f, rr_p = 0.f;
      float alpha = 0.f;
      if (first) {
        __syncthreads();                           // A x of the top levels (written by the top warp) is read below
      } else {
        const float pAp = red.sum(pAp_part, 0.f).x;
        alpha = rz / pAp;
      }
      float2 z[LPT], pk[LPT], dtk[LPT];
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = otid + k * NT;
        z[k] = make_float2(0.f, 0.f); pk[k] = make_float2(0.f, 0.f); dtk[k] = make_float2(0.f, 0.f);
        if (i < N) {
          const float4 m1 = PL[7 * i + kM1], pd = PL[7 * i + kPD];
          const float2 ap = make_float2(m1.z, m1.w);
          dtk[k] = make_float2(pd.z, pd.w);
          float4 xr = PL[7 * i + kXR];
          if (first) {                               // r = b - A x
            xr.z -= ap.x; xr.w -= ap.y;
          } else {
            pk[k] = make_float2(pd.x, pd.y);
            xr.x += alpha * pk[k].x; xr.y += alpha * pk[k].y;
            xr.z -= alpha * ap.x; xr.w -= alpha * ap.y;
          }
          PL[7 * i + kXR] = xr;
          rr_p += xr.z * xr.z + xr.w * xr.w;
          if (!tree) {
            const float2 idg = s.IDG[i];
            z[k] = make_float2(xr.z * idg.x, xr.w * idg.y);
            rz_p += xr.z * z[k].x + xr.w * z[k].y;
          }
        }
      }
      float rz_new;
      if (!tree) {
        const float2 t = red.sum(rz_p, rr_p);
        rz_new = t.x; rr = P.cg_norm ? t.x : t.y;
      } else {
        rr = red.sum(rr_p, 0.f).x;
        if (!(rr > tol2)) {                          // converged (or non-finite): no solve
          if (!first) it++;
          break;
        }
        if (first) {                                 // p = z: the solve's top-down pass is the product's as well
          pAp_carry = tree_solve<NT, true>(s, g, c, otid, nlev, ntop);
          have_down = true;
        } else {
          tree_solve<NT, false>(s, g, c, otid, nlev, ntop);
        }
#pragma unroll
        for (int k = 0; k < LPT; k++) {
          const int i = otid + k * NT;
          if (i < N) {
            const float4 zs = have_down ? PL[7 * i + kPD] : PL[7 * i + kM1], xr = PL[7 * i + kXR];
            z[k] = have_down ? make_float2(zs.x, zs.y) : make_float2(zs.z, zs.w);
            rz_p += xr.z * z[k].x + xr.w * z[k].y;
          }
        }
        rz_new = red.sum(rz_p, 0.f).x;
      }
      const float beta = first ? 0.f : rz_new / rz;
      rz = rz_new;
      if (!have_down) {
#pragma unroll
        for (int k = 0; k < LPT; k++) {
          const int i = otid + k * NT;
          if (i < N)
            PL[7 * i + kPD] = make_float4(z[k].x + beta * pk[k].x, z[k].y + beta * pk[k].y, dtk[k].x, dtk[k].y);
        }
      }
      if (!first) it++;
      first = false;
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
    const Sm s = carve(smem, d.Np, d.Ap, d.NFp, d.n_levels);
    const int Np = d.Np, N = d.N;
    const int nlev = d.n_levels, ntop = d.n_top;
    float4 *const PL = s.P;
    Gm g;
    {
      unsigned char *lb = c.link_blk + d.link_blk_off;
      g.q2 = reinterpret_cast<float2 *>(lb); g.w2 = g.q2 + Np;
      g.rstep = reinterpret_cast<int32_t *>(g.w2 + Np);
      g.rupt = lb + kLinkStateFloats * 4 * Np; g.rc = g.rupt + Np;
      const unsigned char *cst = c.link_cst + (size_t)link_const_bytes(1) * d.link_base;
      g.c4 = reinterpret_cast<const float4 *>(cst);
      g.K = reinterpret_cast<const float *>(cst) + 4 * Np;
      g.rz = g.K + Np;
      g.quatd = reinterpret_cast<const double2 *>(c.quatd) + 2 * (size_t)d.link_base;
      g.anchor = c.anchor + 3 * (size_t)d.apple_base;
      g.Mmax = c.Mmax + d.link_base;
      g.hist = c.xprev + d.link_base;
      g.arm = c.arm ? c.arm + 2 * (size_t)d.link_base : nullptr;
      g.topo2 = c.topo2 + d.link_base;
    }
    if (tid == 0) {
      s_world.g = g; s_world.N = N; s_world.A = d.A; s_world.Np = Np; s_world.Ap = d.Ap; s_world.NFp = d.NFp; s_world.nlev = nlev;
      s_world.ntop = ntop; s_world.precond = d.precond;
    }

    // ---- stage the world: the apple block by one TMA bulk copy; topology words, factor slots, level offsets,
    //      wrench slots ----
    if (tid == 0 && d.Ap) {
      fence_proxy_async_all();     // shared (the landing zone was written by generic stores) and global (the acquire above)
      const uint32_t ab = (uint32_t)apple_block_bytes(d.Ap);
      mbar_expect_tx(&s_bar, ab);
      tma_load(s.u, c.apple_blk + d.apple_blk_off, ab, &s_bar);
    }
    {
      const int32_t *src = reinterpret_cast<const int32_t *>(c.wrench + w);
      int32_t *dst = reinterpret_cast<int32_t *>(s.wr);
      for (int k = tid; k < (int)(sizeof(WrenchSlots) / 4); k += NT) dst[k] = __ldg(src + k);
      if (tid < 7) PL[7 * Np + tid] = make_float4(0.f, 0.f, 0.f, 0.f);            // the zero record
      for (int k = tid; k <= nlev; k += NT) s.lev[k] = __ldg(c.level_off + d.level_base + k);
      for (int i = tid; i < N; i += NT) {
        const int4 tp = __ldg(c.topo + d.link_base + i);
        const int4 t2 = __ldg(g.topo2 + i);
        const uint32_t nc = (uint32_t)tp.w, fc = nc ? (uint32_t)tp.y : 0u;
        const uint32_t tw = (tp.x >= 0 ? (uint32_t)tp.x : ((uint32_t)Np | kTrunk)) | (fc << kChShift) | (nc << kNcShift) |
                            ((t2.x >> 16) ? kHasApples : 0u) | (__ldcg(g.rupt + i) ? kRuptured : 0u);
        PL[7 * i + kCS] = make_float4(0.f, 0.f, 0.f, __uint_as_float(tw));
        s.SL[i] = (uint16_t)(t2.y & 0xffff);
      }
    }
    if (d.Ap) {
      mbar_wait(&s_bar, parity);
      parity ^= 1;
    }
    __syncthreads();
    int step0 = __ldcg(&info->step), steps_done = 0, last_iters = 0;
    unsigned long long iters_total = 0;
    for (int sidx = 0; sidx < n_my; sidx++) {
      sweep_kinematics(&s_world, c, NT, step0 + sidx);  // A0, A1
      if (d.precond) sweep_factor(&s_world, c, NT);     // F
      sweep_bias(&s_world, c, NT, step0 + sidx);        // A2, B1: r = b
      float bb_part = 0.f, bz_part = 0.f;
      {                                                 // x = cubic extrapolation of the last four solutions
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
            const float4 xb = PL[7 * i + kXR];
            const float2 b = make_float2(xb.z, xb.w);
            PL[7 * i + kXR] = make_float4(OB_X0(h1[k].x, h2[k].x, h3[k].x, h4[k].x), OB_X0(h1[k].y, h2[k].y, h3[k].y, h4[k].y), b.x, b.y);
            bb_part += b.x * b.x + b.y * b.y;
            if (d.precond == 1) {
              const float2 idg = s.IDG[i];
              bz_part += b.x * b.x * idg.x + b.y * b.y * idg.y;
            } else {
              if (!d.precond) s.IDG[i] = make_float2(1.f, 1.f);
              bz_part += b.x * b.x + b.y * b.y;
            }
          }
        }
      }
      const float2 bbz = red.sum(bb_part, bz_part);
      const float bb = bbz.x, bz = bbz.y;
      // ---- C: PCG, warm-started ----
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
          const float4 x = PL[7 * i + kXR];
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
        const float4 x4 = PL[7 * i + kXR];
        const float2 x = make_float2(x4.x, x4.y);
        g.hist[(step_now & 3) * (size_t)c.sum_np + i] = x;
        float wa = w0.x + x.x, wb = w0.y + x.y;
        if (P.qd_max > 0.f) {
          wa = fminf(fmaxf(wa, -P.qd_max), P.qd_max);
          wb = fminf(fmaxf(wb, -P.qd_max), P.qd_max);
        }
        const float qa = fmaf(P.h, wa, q0.x), qb = fmaf(P.h, wb, q0.y);
        g.w2[i] = make_float2(wa, wb); g.q2[i] = make_float2(qa, qb);
        const uint32_t tw = __float_as_uint(PL[7 * i + kCS].w);
        if (!(tw & kRuptured)) {
          const float Ki = dK[k], Mx = dMx[k];
          const float mu = Ki * sqrtf(qa * qa + qb * qb);                   // Eq. 5
          const int rc0 = drc[k];
          const int rcn = mu > Mx ? rc0 + 1 : 0;
          if (rcn >= P.rupture_frames) {
            g.rupt[i] = 1; g.rc[i] = 0; g.rstep[i] = step_now;
            PL[7 * i + kCS].w = __uint_as_float(tw | kRuptured);
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
        // attached: tether force beyond the rest sag (the sag carries the weight: no gravity term); detached: gravity
        const float3 ft = att ? f3(s.ft[a], s.ft[Ap + a], s.ft[2 * Ap + a]) : f3(0, 0, 0);
        const float3 ga = att ? f3(0, 0, 0) : f3(P.gravity[0], P.gravity[1], P.gravity[2]);
        float3 fu = f3(0, 0, 0);                                            // user force on the apple (wrench slots)
        bool pulled = false;
        for (int k = 0; k < s.wr->n; k++)
          if (s.wr->body[k] == N + a) { fu = fu + f3(s.wr->force[k][0], s.wr->force[k][1], s.wr->force[k][2]); pulled = true; }
        float3 va = f3(s.v[a], s.v[Ap + a], s.v[2 * Ap + a]);
        const float3 v0 = va;                                               // F = -c_v m v on the apple
        const float3 fraw = fu;                                             // the detach predicate counts the pull itself
        if (pulled && P.rail_speed > 0.f) fu = apply_rails(P, ma, v0, fu);                        // an apple is a free body (A36)
        va.x += P.h * (ga.x + (ft.x + fu.x) * inv_m - P.mass_damping * v0.x);
        va.y += P.h * (ga.y + (ft.y + fu.y) * inv_m - P.mass_damping * v0.y);
        va.z += P.h * (ga.z + (ft.z + fu.z) * inv_m - P.mass_damping * v0.z);
        s.v[a] = va.x; s.v[Ap + a] = va.y; s.v[2 * Ap + a] = va.z;
        s.u[a] = fmaf(P.h, va.x, s.u[a]); s.u[Ap + a] = fmaf(P.h, va.y, s.u[Ap + a]);
        s.u[2 * Ap + a] = fmaf(P.h, va.z, s.u[2 * Ap + a]);
        if (att) {
          const float fun = sqrtf(dot(fraw, fraw)), fsn = s.fsn[a], thrB = P.detach_kappa * fdet;
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
        fence_proxy_async_all();   // the bulk store's global writes before the generic-proxy release below
      }
      info->step = step0 + steps_done;
      info->last_iters = last_iters;
      info->status = status;
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
