// ob_step.cu -- k_step, the product kernel (sm_100a): n physics steps of every world in one launch.
//
// One CTA per world in flight (persistent, work queue per size class), several CTAs per SM.  The world's link
// state and apple block are staged into shared memory by two TMA bulk copies (UBLKCP) and written back the same
// way.  A thread owns the same LPT links for the whole launch (link i <-> slot i / NT of thread i % NT) and keeps
// what the PCG loop needs of them in REGISTERS: joint transform E, (c2, s2), effective inertia, diagonal terms
// and the search direction p.  Shared memory carries what crosses threads (the parent <-> child mailboxes of
// the level-synchronous tree sweeps) and the PCG vectors x, r, 1/diag(A), A p.
//
//   A   top-down:  joint transforms (Eq. 3), displacement-form FK, velocities, bias accelerations;
//                  tether forces (Eq. 6 / Eq. 7) and user wrenches -> link bias forces
//   B1  bottom-up: bias torques -> rhs b (Eq. 4 spring-damper terms)
//   B2  bottom-up: composite inertia -> exact diagonal of M for the Jacobi preconditioner, effective link inertia
//   C   matrix-free Jacobi-PCG on (M + M_teth + diag(arm + hD + h^2 K)) dqd = b  (north_star);
//                  M v = acceleration-only inverse dynamics: top-down a_i, bottom-up f_i, project on S_i
//   D   integrate joints and apples; rupture (Eq. 5) and detach predicates
//
// Sweep schedule.  Links are level-ordered and, inside a level, links with children come first, so a warp
// holds either inner links or leaves.  Links 0..31 belong to warp 0: the leading levels that fit there (n_top of
// them) are swept by warp 0 alone with __syncwarp.  A leaf has nothing to wait for on the way up, so it does its
// bottom-up half inside the top-down pass; the bottom-up passes only visit inner links, which find their
// children through an explicit child list (four packed in registers, the rest in global memory).
//
// Scratch planes.  Four float4 planes P0..P3 [Np + 1] plus an overflow of two float4 per inner link.  Column Np
// is never written and stays zero: it stands in for the trunk's parent and for missing children, so the gathers
// of the PCG sweeps need no branches.
//   A    inner link i publishes 24 floats for its children in P0..P3[i], ovf[0..1][inner slot]
//   B1   link i publishes (n, f) for its parent in P0[i], P1[i].xy; writes b_i to P2[i].xy and its diagonal
//        damping / stiffness terms to P3[i].zw
//   B2   link i publishes its composite inertia in P0[i], P1[i], P3[i].xy; writes 1/diag to P2[i].zw
//   C    mailbox (alpha, a) / (n, f) in P0[i], P1[i].xy; A p in P1[i].zw; (r, 1/diag) in P2[i];
//        (p, diagonal terms) in P3[i]
//
// Spatial vectors are [angular; linear at the link origin] in link coordinates.  Link frame: origin at the
// proximal joint, +z along the link.  Joint i: R_rel = Q_i Rx(theta1) Ry(theta2); E_i = R_rel^T maps parent
// coordinates to link coordinates; the joint sits at r = (0,0,L_parent) in the parent frame.
#include <math.h>

#include "ob_device.h"
#include "ob_internal.h"

namespace ob {

// ------------------------------------------------------------------------------------------------------
// shared-memory view of one world
// ------------------------------------------------------------------------------------------------------
struct Sm {
  int Np, Ap, NIp, S;                 // S = Np + 1 columns per scratch plane
  // link state (TMA)
  float2 *q2, *w2, *x2;
  unsigned char *rupt, *rc;
  // apple block (TMA)
  float *u, *v;                       // [3][Ap]
  unsigned char *att, *cA, *cB;
  float *ao, *ak, *am, *ac, *afd;     // ao = [3][Ap]
  float4 *P;                          // scratch planes P[j * S + i]
  float4 *ovf;                        // overflow ovf[j * NIp + inner slot]
  float *ft, *fu, *fsn, *fun;         // tether force [3][Ap], user force [3][Ap], |f_s|, |f_user|
  WrenchSlots *wr;
  unsigned char *snapped;
};

__device__ __forceinline__ Sm carve(unsigned char *base, const WorldDesc &d) {
  Sm s;
  s.Np = d.Np; s.Ap = d.Ap; s.NIp = d.NIp; s.S = d.Np + 1;
  const int Np = d.Np, Ap = d.Ap;
  unsigned char *p = base;
  s.q2 = reinterpret_cast<float2 *>(p); s.w2 = s.q2 + Np; s.x2 = s.w2 + Np;
  s.rupt = p + 24 * Np; s.rc = s.rupt + Np;
  p += link_state_bytes(Np);
  float *f = reinterpret_cast<float *>(p);
  s.u = f; s.v = f + 3 * Ap;
  s.att = p + 24 * Ap; s.cA = s.att + Ap; s.cB = s.cA + Ap;
  f = reinterpret_cast<float *>(p + apple_state_bytes(Ap));
  s.ao = f; s.ak = f + 3 * Ap; s.am = f + 4 * Ap; s.ac = f + 5 * Ap; s.afd = f + 6 * Ap;
  p += apple_block_bytes(Ap);
  s.P = reinterpret_cast<float4 *>(p);
  p += 64 * (Np + 1);
  s.ovf = reinterpret_cast<float4 *>(p);
  p += 32 * d.NIp;
  f = reinterpret_cast<float *>(p);
  s.ft = f; f += 3 * Ap;
  s.fu = f; f += 3 * Ap;
  s.fsn = f; f += Ap;
  s.fun = f; f += Ap;
  s.wr = reinterpret_cast<WrenchSlots *>(f); f += sizeof(WrenchSlots) / 4;
  s.snapped = reinterpret_cast<unsigned char *>(f);
  return s;
}

// read-only per-link data of one world in global memory (L2-resident; consumed into registers once per step)
struct Gm {
  const float4 *c4;       // (m, m c, I about the joint, I_zz)
  const float *K, *rz;    // joint stiffness (Eq. 4), parent length
  const float4 *quat;
  const float *R0;        // [k * Np + i]
  const float *Mmax;
  const float *arm;       // [k * Np + i] or nullptr
  const int4 *topo2;
  const int32_t *child_list;
};

// per-link registers of the owning thread
//   meta = byte offset of the parent's column (16 bits; the zero column for the trunk) | level << 16 (12 bits,
//          0xfff = empty slot) | has children << 28 | more than four children << 29 | trunk << 30
//          | off-axis tether flag << 31
//   ch01, ch23 = byte offsets of the first four children's columns (the zero column where there is none)
struct Slot {
  uint32_t meta, ch01, ch23;
  float E[9];                // parent -> link rotation
  float c2, s2, rz;
  float m, mc, Io, Iz;       // link inertia about the joint + on-axis virtual tether masses (A15)
};
constexpr uint32_t kLvlMask = 0x0fff0000u, kInner = 0x10000000u, kMany = 0x20000000u, kTrunk = 0x40000000u,
                   kOffax = 0x80000000u;
__device__ __forceinline__ bool has_parent(const Slot &L) { return (L.meta & kTrunk) == 0u; }
__device__ __forceinline__ int parent_of(const Slot &L) { return (int)((L.meta & 0xffffu) >> 4); }
__device__ __forceinline__ bool is_inner(const Slot &L) { return (L.meta & kInner) != 0u; }
__device__ __forceinline__ bool is_valid(const Slot &L) { return (L.meta & kLvlMask) != kLvlMask; }
__device__ __forceinline__ bool at_level(const Slot &L, uint32_t lkey) { return (L.meta & kLvlMask) == lkey; }

// children of a link, in ascending index order: four from registers (the zero column where there is none),
// the rest from the global child list.  `ch` is the child's column index.
#define OB_FOR_CHILDREN(L, i, g, BODY)                                              \
  {                                                                                 \
    { const int ch = (int)(((L).ch01 & 0xffffu) >> 4); BODY }                       \
    { const int ch = (int)((L).ch01 >> 20); BODY }                                  \
    { const int ch = (int)(((L).ch23 & 0xffffu) >> 4); BODY }                       \
    { const int ch = (int)((L).ch23 >> 20); BODY }                                  \
    if ((L).meta & kMany) {                                                         \
      const int4 t2_ = __ldg((g).topo2 + (i));                                      \
      for (int cc_ = 4; cc_ < t2_.w; cc_++) { const int ch = __ldg((g).child_list + t2_.z + cc_); BODY } \
    }                                                                               \
  }

// shared-memory accesses of the PCG sweeps by byte offset into the CTA's dynamic shared memory
__device__ __forceinline__ float4 lds4(const unsigned char *sm, int off) { return *reinterpret_cast<const float4 *>(sm + off); }
__device__ __forceinline__ float2 lds2(const unsigned char *sm, int off) { return *reinterpret_cast<const float2 *>(sm + off); }
__device__ __forceinline__ void sts4(unsigned char *sm, int off, float4 v) { *reinterpret_cast<float4 *>(sm + off) = v; }
__device__ __forceinline__ void sts2(unsigned char *sm, int off, float2 v) { *reinterpret_cast<float2 *>(sm + off) = v; }

// one shared copy of the accurate sincosf (its slow path is large); cos - 1 without cancellation
__device__ __noinline__ float2 sincos2(float x) {
  float sn, cs;
  sincosf(x, &sn, &cs);
  return make_float2(sn, cs);
}
__device__ __forceinline__ float cos_minus_one(float sn, float cs) { return cs > 0.f ? -(sn * sn) / (1.f + cs) : cs - 1.f; }

// block-wide sum of two values, result broadcast to every thread; one barrier per call (double-buffered stage)
template <int NT>
struct Reducer {
  float2 *stage;   // [2][32]
  int flip, tid;
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
    const float4 *s4 = reinterpret_cast<const float4 *>(st);
#pragma unroll
    for (int k = 0; k < NT / 64; k++) { const float4 t = s4[k]; sa += t.x + t.z; sb += t.y + t.w; }
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

// kinematic quantities of one link that the bias pass hands from its top-down half to its bottom-up half
struct Kin {
  M3 dR;               // R - R0 (displacement form)
  float3 dp;           // origin - rest origin
  float3 om, vl;       // spatial velocity
  float3 al, aln;      // bias spatial acceleration (gravity as base acceleration)
};

// ------------------------------------------------------------------------------------------------------
// bias force of one link: f = I a + v x* I v - tether reactions - user wrenches (RNEA with qdd = 0)
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void bias_force(const int i, const Kin &k, const unsigned char snapped, const Sm &s,
                                           const Gm &g, const DevCtx &c, float3 &n, float3 &f) {
  const ob_params &P = c.P;
  const int Np = s.Np, Ap = s.Ap;
  const float4 c4 = __ldg(g.c4 + i);
  const float m = c4.x, mc = c4.y, Io = c4.z, Iz = c4.w;
  const float3 om = k.om, vl = k.vl, al = k.al, aln = k.aln;
  // f = I a + v x* I v  (cylinder: com on +z)
  n = f3(Io * al.x - mc * aln.y, Io * al.y + mc * aln.x, Iz * al.z);
  f = f3(m * aln.x + mc * al.y, m * aln.y - mc * al.x, m * aln.z);
  const float3 hn = f3(Io * om.x - mc * vl.y, Io * om.y + mc * vl.x, Iz * om.z);
  const float3 hf = f3(m * vl.x + mc * om.y, m * vl.y - mc * om.x, m * vl.z);
  n = n + cross(om, hn) + cross(vl, hf);
  f = f + cross(om, hf);

  const int4 t2 = __ldg(g.topo2 + i);
  const int ast = t2.x & 0xffff, nap = t2.x >> 16;
  const int nwr = s.wr->n;
  bool wr_here = false;
  for (int q = 0; q < nwr; q++) wr_here |= s.wr->body[q] == i;
  if (nap == 0 && !wr_here) return;

  M3 R;                                                                   // world rotation R0 + dR
#pragma unroll
  for (int q = 0; q < 9; q++) R.a[q] = __ldg(g.R0 + (size_t)q * Np + i) + k.dR.a[q];
  // tethers on this link (Eq. 6, Eq. 7): everything about the hang point is at hand here
  const float eta_h = P.tether_implicit ? P.h : 0.f;
  for (int a = ast; a < ast + nap; a++) {
    if (!s.att[a]) continue;
    const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
    const float3 dh = k.dp + mul(k.dR, o);                                // x_hang - anchor
    const float ks = s.ak[a], cdamp = s.ac[a], ma = s.am[a];
    // x_a - x_hang = u + sag - dh with the rest sag m g / k_s (u is stored relative to the rest position)
    const float gk = ma / ks;
    const float3 st = f3(s.u[a] + (gk * P.gravity[0] - dh.x), s.u[Ap + a] + (gk * P.gravity[1] - dh.y),
                         s.u[2 * Ap + a] + (gk * P.gravity[2] - dh.z));
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
    f = f - fl;
    n = n - cross(o, fl);
  }
  // user wrenches on this link (disabled on snapped sub-trees)
  for (int q = 0; q < nwr; q++) {
    if (s.wr->body[q] != i) continue;
    if (snapped && P.forces_off_on_snapped) continue;
    const float3 fl = mulT(R, f3(s.wr->force[q][0], s.wr->force[q][1], s.wr->force[q][2]));
    const float3 pt = f3(s.wr->point[q][0], s.wr->point[q][1], s.wr->point[q][2]);
    f = f - fl;
    n = n - cross(pt, fl);
  }
}

// project the accumulated bias force on the joint axes -> rhs b (P2[i].xy), the diagonal damping / stiffness
// terms, and publish (n, f) in the parent frame (P0[i], P1[i].xy)
__device__ __forceinline__ void finish_bias(const Slot &L, const int i, float3 n, float3 f, const Sm &s, const Gm &g,
                                            const DevCtx &c) {
  const ob_params &P = c.P;
  const int Np = s.Np, S = s.S;
  const float c2 = L.c2, s2 = L.s2;
  const float tau1 = c2 * n.x + s2 * n.z, tau2 = n.y;
  const float Kt = s.rupt[i] ? 0.f : __ldg(g.K + i), Dt = P.c_d * Kt;
  const float2 th = s.q2[i], w = s.w2[i];
  const float b1 = P.h * (-tau1 - Kt * th.x - (Dt + P.h * Kt) * w.x);
  const float b2 = P.h * (-tau2 - Kt * th.y - (Dt + P.h * Kt) * w.y);
  *reinterpret_cast<float2 *>(s.P + 2 * S + i) = make_float2(b1, b2);
  float dt0 = (P.h * P.c_d + P.h * P.h) * Kt, dt1 = dt0;
  if (g.arm) {
    dt0 += __ldg(g.arm + i);
    dt1 += __ldg(g.arm + Np + i);
  }
  reinterpret_cast<float2 *>(s.P + 3 * S + i)[1] = make_float2(dt0, dt1);    // arm + (h c_d + h^2) K per DoF
  if (has_parent(L)) {
    M3 E;
#pragma unroll
    for (int q = 0; q < 9; q++) E.a[q] = L.E[q];
    const float3 fp = mulT(E, f);
    float3 np = mulT(E, n);
    np.x -= L.rz * fp.y; np.y += L.rz * fp.x;
    s.P[i] = make_float4(np.x, np.y, np.z, fp.x);
    *reinterpret_cast<float2 *>(s.P + S + i) = make_float2(fp.y, fp.z);
  }
}

// ------------------------------------------------------------------------------------------------------
// phase A for one link (top-down); a leaf goes straight on to its phase-B1 half
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void down_bias(Slot &L, const int i, const Sm &s, const Gm &g, const DevCtx &c) {
  const int Np = s.Np, NIp = s.NIp, S = s.S;
  const ob_params &P = c.P;
  const float2 th = s.q2[i], w = s.w2[i];
  const float th1 = th.x, th2 = th.y, w1 = w.x, w2 = w.y;
  const float2 sc1 = sincos2(th1), sc2 = sincos2(th2);
  const float s1 = sc1.x, c1 = sc1.y, s2 = sc2.x, c2 = sc2.y;
  const float vc1 = cos_minus_one(s1, c1), vc2 = cos_minus_one(s2, c2);
  const M3 Q = quat_to_mat(__ldg(g.quat + i));
  M3 XY;                                                           // Rx(th1) Ry(th2)
  XY.a[0] = c2;       XY.a[1] = 0.f; XY.a[2] = s2;
  XY.a[3] = s1 * s2;  XY.a[4] = c1;  XY.a[5] = -s1 * c2;
  XY.a[6] = -c1 * s2; XY.a[7] = s1;  XY.a[8] = c1 * c2;
  const M3 Rrel = mul(Q, XY);
  M3 E;                                                            // E = Rrel^T
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int cc = 0; cc < 3; cc++) E.a[3 * r + cc] = Rrel.a[3 * cc + r];
#pragma unroll
  for (int q = 0; q < 9; q++) L.E[q] = E.a[q];
  L.c2 = c2; L.s2 = s2;
  const int4 t2 = __ldg(g.topo2 + i);

  // parent quantities (world = parent of the trunk: at rest, spatial acceleration (0; -g))
  M3 dRp;
  float3 dpp = f3(0, 0, 0), wp = f3(0, 0, 0), vp = f3(0, 0, 0), alp = f3(0, 0, 0);
  float3 ap = f3(-P.gravity[0], -P.gravity[1], -P.gravity[2]);
  unsigned char snapped_p = 0;
  float rz = 0.f;
#pragma unroll
  for (int q = 0; q < 9; q++) dRp.a[q] = 0.f;
  if (has_parent(L)) {
    const int par = parent_of(L), ps = (int)((uint32_t)t2.y >> 16);
    const float4 t0 = s.P[par], t1 = s.P[S + par], t2v = s.P[2 * S + par], t3 = s.P[3 * S + par],
                 t4 = s.ovf[ps], t5 = s.ovf[NIp + ps];
    dRp.a[0] = t0.x; dRp.a[1] = t0.y; dRp.a[2] = t0.z; dRp.a[3] = t0.w;
    dRp.a[4] = t1.x; dRp.a[5] = t1.y; dRp.a[6] = t1.z; dRp.a[7] = t1.w;
    dRp.a[8] = t2v.x; dpp = f3(t2v.y, t2v.z, t2v.w);
    wp = f3(t3.x, t3.y, t3.z); vp = f3(t3.w, t4.x, t4.y);
    alp = f3(t4.z, t4.w, t5.x); ap = f3(t5.y, t5.z, t5.w);
    snapped_p = s.snapped[par];
    rz = __ldg(g.rz + i);
  }
  L.rz = rz;
  // displacement-form FK: R_i = R0_i + dR_i,  dR_i = dR_p Rrel + R0_i (RxRy - I);  dp_i = dp_p + dR_p (0,0,rz)
  Kin k;
  {
    M3 R0, G = XY;
#pragma unroll
    for (int q = 0; q < 9; q++) R0.a[q] = __ldg(g.R0 + (size_t)q * Np + i);
    G.a[0] = vc2; G.a[4] = vc1; G.a[8] = fmaf(vc1, vc2, vc1 + vc2);
    const M3 t1m = mul(dRp, Rrel), t2m = mul(R0, G);
#pragma unroll
    for (int q = 0; q < 9; q++) k.dR.a[q] = t1m.a[q] + t2m.a[q];
  }
  k.dp = f3(dpp.x + rz * dRp.a[2], dpp.y + rz * dRp.a[5], dpp.z + rz * dRp.a[8]);

  // velocity and (bias) spatial acceleration in link coordinates
  const float3 vJ = f3(c2 * w1, w2, s2 * w1);
  k.om = mul(E, wp) + vJ;
  k.vl = mul(E, f3(vp.x + wp.y * rz, vp.y - wp.x * rz, vp.z));
  const float ww = w1 * w2;
  k.al = mul(E, alp) + f3(-s2 * ww, 0.f, c2 * ww) + cross(k.om, vJ);
  k.aln = mul(E, f3(ap.x + alp.y * rz, ap.y - alp.x * rz, ap.z)) + cross(k.vl, vJ);

  const unsigned char snapped = s.rupt[i] | snapped_p;
  s.snapped[i] = snapped;

  if (is_inner(L)) {
    const int is = t2.y & 0xffff;
    s.P[i] = make_float4(k.dR.a[0], k.dR.a[1], k.dR.a[2], k.dR.a[3]);
    s.P[S + i] = make_float4(k.dR.a[4], k.dR.a[5], k.dR.a[6], k.dR.a[7]);
    s.P[2 * S + i] = make_float4(k.dR.a[8], k.dp.x, k.dp.y, k.dp.z);
    s.P[3 * S + i] = make_float4(k.om.x, k.om.y, k.om.z, k.vl.x);
    s.ovf[is] = make_float4(k.vl.y, k.vl.z, k.al.x, k.al.y);
    s.ovf[NIp + is] = make_float4(k.al.z, k.aln.x, k.aln.y, k.aln.z);
  } else {
    float3 n, f;
    bias_force(i, k, snapped, s, g, c, n, f);
    finish_bias(L, i, n, f, s, g, c);
  }
}

// phase B1 for one inner link: its own bias force (from the kinematics it published on the way down) plus
// what its children sent up
__device__ __forceinline__ void up_bias(Slot &L, const int i, const Sm &s, const Gm &g, const DevCtx &c) {
  const int NIp = s.NIp, S = s.S;
  const int is = __ldg(g.topo2 + i).y & 0xffff;
  Kin k;
  {
    const float4 t0 = s.P[i], t1 = s.P[S + i], t2v = s.P[2 * S + i], t3 = s.P[3 * S + i], t4 = s.ovf[is],
                 t5 = s.ovf[NIp + is];
    k.dR.a[0] = t0.x; k.dR.a[1] = t0.y; k.dR.a[2] = t0.z; k.dR.a[3] = t0.w;
    k.dR.a[4] = t1.x; k.dR.a[5] = t1.y; k.dR.a[6] = t1.z; k.dR.a[7] = t1.w;
    k.dR.a[8] = t2v.x; k.dp = f3(t2v.y, t2v.z, t2v.w);
    k.om = f3(t3.x, t3.y, t3.z); k.vl = f3(t3.w, t4.x, t4.y);
    k.al = f3(t4.z, t4.w, t5.x); k.aln = f3(t5.y, t5.z, t5.w);
  }
  float3 n, f;
  bias_force(i, k, s.snapped[i], s, g, c, n, f);
  OB_FOR_CHILDREN(L, i, g, {
    const float4 u = s.P[ch];
    const float2 v = *reinterpret_cast<const float2 *>(s.P + S + ch);
    n = n + f3(u.x, u.y, u.z);
    f = f + f3(u.w, v.x, v.y);
  })
  finish_bias(L, i, n, f, s, g, c);
}

// ------------------------------------------------------------------------------------------------------
// phase B2 for one link: composite rigid-body inertia about the link origin (mass, first moment h, symmetric
// I) -> exact diagonal of M -> Jacobi factors (P2[i].zw); effective link inertia for A v; publish the composite
// inertia in the parent frame (P0[i], P1[i], P3[i].xy)
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void up_inertia(Slot &L, const int i, const Sm &s, const Gm &g, const DevCtx &c) {
  const int S = s.S, Ap = s.Ap;
  const ob_params &P = c.P;
  const float4 c4 = __ldg(g.c4 + i);
  float cm = c4.x;
  float3 ch3 = f3(0.f, 0.f, c4.y);
  float Ixx = c4.z, Iyy = c4.z, Izz = c4.w, Ixy = 0.f, Ixz = 0.f, Iyz = 0.f;
  L.m = c4.x; L.mc = c4.y; L.Io = c4.z; L.Iz = c4.w;
  L.meta &= ~kOffax;
  if (P.tether_implicit) {
    const int4 t2 = __ldg(g.topo2 + i);
    const int ast = t2.x & 0xffff, nap = t2.x >> 16;
    for (int a = ast; a < ast + nap; a++) {
      if (!s.att[a]) continue;
      const float mv = P.h * P.h * s.ak[a];                     // virtual point mass h^2 k_s at the hang point
      const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
      cm += mv; ch3 = ch3 + mv * o;
      Ixx += mv * (o.y * o.y + o.z * o.z); Iyy += mv * (o.x * o.x + o.z * o.z); Izz += mv * (o.x * o.x + o.y * o.y);
      Ixy -= mv * o.x * o.y; Ixz -= mv * o.x * o.z; Iyz -= mv * o.y * o.z;
      if (o.x == 0.f && o.y == 0.f) { L.m += mv; L.mc += mv * o.z; L.Io += mv * o.z * o.z; }   // stays a body of revolution
      else L.meta |= kOffax;
    }
  }
  if (is_inner(L)) {
    OB_FOR_CHILDREN(L, i, g, {
      const float4 u0 = s.P[ch];
      const float4 u1 = s.P[S + ch];
      const float2 u2 = *reinterpret_cast<const float2 *>(s.P + 3 * S + ch);
      cm += u0.x;
      ch3 = ch3 + f3(u0.y, u0.z, u0.w);
      Ixx += u1.x; Iyy += u1.y; Izz += u1.z; Ixy += u1.w; Ixz += u2.x; Iyz += u2.y;
    })
  }
  const float c2 = L.c2, s2 = L.s2;
  const float2 dt = reinterpret_cast<const float2 *>(s.P + 3 * S + i)[1];
  const float d1 = c2 * c2 * Ixx + 2.f * c2 * s2 * Ixz + s2 * s2 * Izz + dt.x;
  const float d2 = Iyy + dt.y;
  float2 id = make_float2(1.f, 1.f);
  if (P.precond == 1) id = make_float2(1.f / d1, 1.f / d2);
  reinterpret_cast<float2 *>(s.P + 2 * S + i)[1] = id;
  if (has_parent(L)) {
    M3 E;
#pragma unroll
    for (int q = 0; q < 9; q++) E.a[q] = L.E[q];
    const float rz = L.rz;
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
    s.P[i] = make_float4(cm, hp.x, hp.y, hp.z + cm * rz);
    s.P[S + i] = make_float4(Ip.a[0] + sh, Ip.a[4] + sh, Ip.a[8], Ip.a[1]);
    *reinterpret_cast<float2 *>(s.P + 3 * S + i) = make_float2(Ip.a[2] - rz * hp.x, Ip.a[5] - rz * hp.y);
  }
}

// ------------------------------------------------------------------------------------------------------
// phase C: A v for one link.  Shared memory is addressed by byte offset: `own` is the link's column in plane 0,
// PS the plane stride, oP the offset of plane 0; parent and children columns come out of the slot's registers.
// up_mv: f = I a + children, project on S (+ diagonal terms) -> A p (P1[i].zw), publish to the parent; returns
// p . (A p) of this link.  down_mv: accelerations from the parent; a leaf goes straight up.  Mailbox: P0[i] =
// (x, y, z of the angular part, x of the linear part), P1[i].xy = (y, z of the linear part).
// ------------------------------------------------------------------------------------------------------
struct Hot { int oP, PS; };   // world-uniform offsets of the PCG sweeps

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

template <bool INNER>
__device__ __forceinline__ float up_mv(const Slot &L, const int i, const int own, const Hot h, unsigned char *sm,
                                       const float3 al, const float3 a, const float4 pd, const Sm &s, const Gm &g,
                                       const DevCtx &c) {
  float3 n = f3(L.Io * al.x - L.mc * a.y, L.Io * al.y + L.mc * a.x, L.Iz * al.z);
  float3 f = f3(L.m * a.x + L.mc * al.y, L.m * a.y - L.mc * al.x, L.m * a.z);
  if (L.meta & kOffax) {
    const Force6 t = offaxis_tethers(__ldg(g.topo2 + i), al, a, s.att, s.ao, s.ak, s.Ap, c.P.h * c.P.h);
    n = n + t.n; f = f + t.f;
  }
  if (INNER) {
    const int o0 = h.oP + (int)(L.ch01 & 0xffffu), o1 = h.oP + (int)(L.ch01 >> 16);
    const int o2 = h.oP + (int)(L.ch23 & 0xffffu), o3 = h.oP + (int)(L.ch23 >> 16);
    const float4 u0 = lds4(sm, o0), u1 = lds4(sm, o1), u2 = lds4(sm, o2), u3 = lds4(sm, o3);
    const float2 v0 = lds2(sm, o0 + h.PS), v1 = lds2(sm, o1 + h.PS), v2 = lds2(sm, o2 + h.PS), v3 = lds2(sm, o3 + h.PS);
    n = n + f3(u0.x, u0.y, u0.z); f = f + f3(u0.w, v0.x, v0.y);
    n = n + f3(u1.x, u1.y, u1.z); f = f + f3(u1.w, v1.x, v1.y);
    n = n + f3(u2.x, u2.y, u2.z); f = f + f3(u2.w, v2.x, v2.y);
    n = n + f3(u3.x, u3.y, u3.z); f = f + f3(u3.w, v3.x, v3.y);
    if (L.meta & kMany) {
      const int4 t2 = __ldg(g.topo2 + i);
      for (int cc = 4; cc < t2.w; cc++) {
        const int oc = h.oP + 16 * __ldg(g.child_list + t2.z + cc);
        const float4 u = lds4(sm, oc);
        const float2 v = lds2(sm, oc + h.PS);
        n = n + f3(u.x, u.y, u.z); f = f + f3(u.w, v.x, v.y);
      }
    }
  }
  const float t1 = L.c2 * n.x + L.s2 * n.z + pd.z * pd.x;     // pd = (p0, p1, dt0, dt1)
  const float t2 = n.y + pd.w * pd.y;
  M3 E;
#pragma unroll
  for (int q = 0; q < 9; q++) E.a[q] = L.E[q];
  const float3 fp = mulT(E, f);                 // the trunk publishes into its own column, which nobody reads
  float3 np = mulT(E, n);
  np.x -= L.rz * fp.y; np.y += L.rz * fp.x;
  sts4(sm, own, make_float4(np.x, np.y, np.z, fp.x));
  sts4(sm, own + h.PS, make_float4(fp.y, fp.z, t1, t2));
  return pd.x * t1 + pd.y * t2;
}

__device__ __forceinline__ float down_mv(const Slot &L, const int i, const int own, const Hot h, unsigned char *sm,
                                         const Sm &s, const Gm &g, const DevCtx &c) {
  const int po = h.oP + (int)(L.meta & 0xffffu);     // the trunk reads the zero column
  const float4 u = lds4(sm, po);
  const float2 v = lds2(sm, po + h.PS);
  const float4 pd = lds4(sm, own + 3 * h.PS);
  const float3 alp = f3(u.x, u.y, u.z), ap = f3(u.w, v.x, v.y);
  M3 E;
#pragma unroll
  for (int q = 0; q < 9; q++) E.a[q] = L.E[q];
  float3 al = mul(E, alp);
  const float3 a = mul(E, f3(ap.x + alp.y * L.rz, ap.y - alp.x * L.rz, ap.z));
  al = al + f3(L.c2 * pd.x, pd.y, L.s2 * pd.x);
  if (is_inner(L)) {
    sts4(sm, own, make_float4(al.x, al.y, al.z, a.x));
    sts2(sm, own + h.PS, make_float2(a.y, a.z));
    return 0.f;
  }
  return up_mv<false>(L, i, own, h, sm, al, a, pd, s, g, c);
}

__device__ __forceinline__ float up_mv_inner(const Slot &L, const int i, const int own, const Hot h, unsigned char *sm,
                                             const Sm &s, const Gm &g, const DevCtx &c) {
  const float4 u = lds4(sm, own);
  const float2 v = lds2(sm, own + h.PS);
  const float4 pd = lds4(sm, own + 3 * h.PS);
  return up_mv<true>(L, i, own, h, sm, f3(u.x, u.y, u.z), f3(u.w, v.x, v.y), pd, s, g, c);
}

// ------------------------------------------------------------------------------------------------------
// level-synchronous sweeps, slot-major.  A warp's slot k holds 32 consecutive links, i.e. one level (two at a
// level boundary): s_rng[warp][k] = (lowest | highest << 16 level of the slot, the same over its inner links).
// The warp walks its slots in order and catches up on the fences between levels on the way, so every warp
// executes every block barrier exactly once and no warp tests levels it has no links in.  Fence after level l
// on the way down: __syncwarp (warp 0) while level l + 1 is still one of the n_top levels inside warp 0, else
// __syncthreads.  DOWN ends with a block barrier; UP leaves the trunk's level unfenced: what follows is a block
// reduction or an explicit barrier.
// ------------------------------------------------------------------------------------------------------
// The PCG sweeps (OB_SWEEP_*) are unrolled over the slots; the once-per-step sweeps (OB_COLD_*) loop over the
// slots at run time on a copy T of the slot's registers, which keeps their (large) code four times smaller.
#define OB_FENCE_DOWN(l) { if ((l) + 1 < ntop) { if (warp0) __syncwarp(); } else __syncthreads(); }
#define OB_FENCE_UP(l) { if ((l) < ntop) { if (warp0) __syncwarp(); } else __syncthreads(); }
#define OB_SWEEP_DOWN(BODY)                                                      \
  {                                                                              \
    int cur_ = 0;                                                                \
    _Pragma("unroll") for (int k = 0; k < LPT; k++) {                            \
      const uint32_t rg_ = s_rng[wid * LPT + k].x;                               \
      const int lo_ = (int)(rg_ & 0xffffu), hi_ = (int)(rg_ >> 16);              \
      for (int l = lo_; l <= hi_; l++) {                                         \
        while (cur_ < l) { OB_FENCE_DOWN(cur_); cur_++; }                        \
        if (at_level(L[k], (uint32_t)l << 16)) { const int i = k * NT + tid; BODY } \
      }                                                                          \
    }                                                                            \
    while (cur_ < nlev) { OB_FENCE_DOWN(cur_); cur_++; }                         \
  }
#define OB_SWEEP_UP(BODY)                                                        \
  {                                                                              \
    int cur_ = nlev - 2;                                                         \
    _Pragma("unroll") for (int kk = 0; kk < LPT; kk++) {                         \
      const int k = LPT - 1 - kk;                                                \
      const uint32_t rg_ = s_rng[wid * LPT + k].y;                               \
      const int lo_ = (int)(rg_ & 0xffffu), hi_ = (int)(rg_ >> 16);              \
      for (int l = hi_; l >= lo_; l--) {                                         \
        while (cur_ > l) { OB_FENCE_UP(cur_); cur_--; }                          \
        if (at_level(L[k], (uint32_t)l << 16) && is_inner(L[k])) { const int i = k * NT + tid; BODY } \
      }                                                                          \
    }                                                                            \
    while (cur_ > 0) { OB_FENCE_UP(cur_); cur_--; }                              \
  }
#define OB_COLD_DOWN(PUT, BODY)                                                  \
  {                                                                              \
    int cur_ = 0;                                                                \
    _Pragma("unroll 1") for (int k = 0; k < LPT; k++) {                          \
      const uint32_t rg_ = s_rng[wid * LPT + k].x;                               \
      const int lo_ = (int)(rg_ & 0xffffu), hi_ = (int)(rg_ >> 16);              \
      if (lo_ > hi_) continue;                                                   \
      Slot T = slot_get<LPT>(L, k);                                              \
      const int i = k * NT + tid;                                                \
      for (int l = lo_; l <= hi_; l++) {                                         \
        while (cur_ < l) { OB_FENCE_DOWN(cur_); cur_++; }                        \
        if (at_level(T, (uint32_t)l << 16)) { BODY }                             \
      }                                                                          \
      if (PUT) slot_put<LPT>(L, k, T);                                           \
    }                                                                            \
    while (cur_ < nlev) { OB_FENCE_DOWN(cur_); cur_++; }                         \
  }
#define OB_COLD_UP(PUT, BODY)                                                    \
  {                                                                              \
    int cur_ = nlev - 2;                                                         \
    _Pragma("unroll 1") for (int k = LPT - 1; k >= 0; k--) {                     \
      const uint32_t rg_ = s_rng[wid * LPT + k].y;                               \
      const int lo_ = (int)(rg_ & 0xffffu), hi_ = (int)(rg_ >> 16);              \
      if (lo_ > hi_) continue;                                                   \
      Slot T = slot_get<LPT>(L, k);                                              \
      const int i = k * NT + tid;                                                \
      for (int l = hi_; l >= lo_; l--) {                                         \
        while (cur_ > l) { OB_FENCE_UP(cur_); cur_--; }                          \
        if (at_level(T, (uint32_t)l << 16) && is_inner(T)) { BODY }              \
      }                                                                          \
      if (PUT) slot_put<LPT>(L, k, T);                                           \
    }                                                                            \
    while (cur_ > 0) { OB_FENCE_UP(cur_); cur_--; }                              \
  }

// slot k of the register file by run-time index (k is warp-uniform): explicit cases, never a local array
template <int LPT>
__device__ __forceinline__ Slot slot_get(const Slot (&L)[LPT], const int k) {
  static_assert(LPT >= 1 && LPT <= 4, "slot_get / slot_put cover up to four slots");
  switch (k) {
    case 1: return L[LPT > 1 ? 1 : 0];
    case 2: return L[LPT > 2 ? 2 : 0];
    case 3: return L[LPT > 3 ? 3 : 0];
    default: return L[0];
  }
}
template <int LPT>
__device__ __forceinline__ void slot_put(Slot (&L)[LPT], const int k, const Slot &T) {
  switch (k) {
    case 1: L[LPT > 1 ? 1 : 0] = T; break;
    case 2: L[LPT > 2 ? 2 : 0] = T; break;
    case 3: L[LPT > 3 ? 3 : 0] = T; break;
    default: L[0] = T; break;
  }
}

// ------------------------------------------------------------------------------------------------------
// k_step<NT, LPT>
// ------------------------------------------------------------------------------------------------------
template <int NT, int LPT, int MINB>
__global__ void __launch_bounds__(NT, MINB)
k_step(DevCtx c, const int32_t *__restrict__ order, int n_in_class, int32_t *queue, int n_steps) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ __align__(8) uint64_t s_bar;
  __shared__ int s_next;
  __shared__ __align__(16) float2 s_stage[64];
  __shared__ uint2 s_rng[(NT / 32) * LPT];
  const int tid = threadIdx.x, wid = tid >> 5;
  const bool warp0 = tid < 32;
  const ob_params &P = c.P;
  uint32_t parity = 0;
  if (tid == 0) mbar_init(&s_bar, 1);
  __syncthreads();
  Reducer<NT> red;
  red.stage = s_stage;
  red.flip = 0;
  red.tid = tid;
  Slot L[LPT];

  for (;;) {
    if (tid == 0) s_next = atomicAdd(queue, 1);
    __syncthreads();
    const int qi = s_next;
    __syncthreads();
    if (qi >= n_in_class) break;
    const int w = order[qi];
    const WorldDesc d = c.desc[w];
    WorldInfo *info = c.info + w;
    int status = info->status;
    if (status & OB_STATUS_NONFINITE) continue;      // frozen world
    const Sm s = carve(smem, d);
    const int Np = d.Np;
    const int nlev = d.n_levels, ntop = d.n_top;
    Gm g;
    {
      const unsigned char *cst = c.link_blk + d.link_blk_off + link_state_bytes(Np);
      g.c4 = reinterpret_cast<const float4 *>(cst);
      g.K = reinterpret_cast<const float *>(cst) + 4 * Np;
      g.rz = g.K + Np;
      g.quat = c.quat + d.link_base;
      g.R0 = c.R0 + 9 * (size_t)d.link_base;
      g.Mmax = c.Mmax + d.link_base;
      g.arm = c.arm ? c.arm + 2 * (size_t)d.link_base : nullptr;
      g.topo2 = c.topo2 + d.link_base;
      g.child_list = c.child_list + d.link_base;
    }
    // byte offsets of what the PCG loop touches: this thread's columns in planes 0..2 and its x
    Hot h;
    h.oP = (int)(reinterpret_cast<unsigned char *>(s.P) - smem);
    h.PS = 16 * (Np + 1);
    const int own0 = h.oP + 16 * tid;
    const int ox = (int)(reinterpret_cast<unsigned char *>(s.x2) - smem) + 8 * tid;

    // ---- stage the world: two TMA bulk copies (link state, apple block) onto one mbarrier ----
    if (tid == 0) {
      fence_proxy_async();
      const uint32_t lb = (uint32_t)link_state_bytes(Np), ab = (uint32_t)apple_block_bytes(d.Ap);
      mbar_expect_tx(&s_bar, lb + ab);
      tma_load(s.q2, c.link_blk + d.link_blk_off, lb, &s_bar);
      if (ab) tma_load(s.u, c.apple_blk + d.apple_blk_off, ab, &s_bar);
    }
    {
      const int32_t *src = reinterpret_cast<const int32_t *>(c.wrench + w);
      int32_t *dst = reinterpret_cast<int32_t *>(s.wr);
      for (int k = tid; k < (int)(sizeof(WrenchSlots) / 4); k += NT) dst[k] = __ldg(src + k);
      if (tid < 4) s.P[tid * (Np + 1) + Np] = make_float4(0.f, 0.f, 0.f, 0.f);      // the zero column
    }
    const uint32_t zcol = (uint32_t)(16 * Np);
#pragma unroll
    for (int k = 0; k < LPT; k++) {                  // topology of the links this thread owns
      const int i = k * NT + tid;
      L[k].meta = zcol | kLvlMask | kTrunk;
      L[k].ch01 = zcol | (zcol << 16); L[k].ch23 = L[k].ch01;
      uint32_t lmin = 0xffffu, lmax = 0u, imin = 0xffffu, imax = 0u;
      if (i < d.N) {
        const int4 tp = __ldg(c.topo + d.link_base + i);
        const uint32_t lvl = (uint32_t)(tp.w & 0xfff), nch = (uint32_t)((tp.w >> 12) & 7);
        L[k].meta = (tp.x >= 0 ? (uint32_t)(16 * tp.x) : (zcol | kTrunk)) | (lvl << 16) | (nch ? kInner : 0u) |
                    (nch > 4 ? kMany : 0u);
        auto col = [&](uint32_t idx) { return idx == 0xffffu ? zcol : 16u * idx; };
        L[k].ch01 = col((uint32_t)tp.y & 0xffffu) | (col((uint32_t)tp.y >> 16) << 16);
        L[k].ch23 = col((uint32_t)tp.z & 0xffffu) | (col((uint32_t)tp.z >> 16) << 16);
        lmin = lvl; lmax = lvl;
        if (nch) { imin = lvl; imax = lvl; }
      }
      const uint32_t r0 = __reduce_min_sync(0xffffffffu, lmin) | (__reduce_max_sync(0xffffffffu, lmax) << 16);
      const uint32_t r1 = __reduce_min_sync(0xffffffffu, imin) | (__reduce_max_sync(0xffffffffu, imax) << 16);
      if ((tid & 31) == 0) s_rng[wid * LPT + k] = make_uint2(r0, r1);
    }
    mbar_wait(&s_bar, parity);
    parity ^= 1;
    __syncthreads();
    // user forces on apples are constant over the launch
    for (int a = tid; a < d.A; a += NT) {
      float3 fu = f3(0, 0, 0);
      for (int k = 0; k < s.wr->n; k++)
        if (s.wr->body[k] == d.N + a) fu = fu + f3(s.wr->force[k][0], s.wr->force[k][1], s.wr->force[k][2]);
      s.fu[a] = fu.x; s.fu[d.Ap + a] = fu.y; s.fu[2 * d.Ap + a] = fu.z;
      s.fun[a] = sqrtf(dot(fu, fu));
    }
    __syncthreads();

    int step0 = info->step, steps_done = 0, last_iters = 0;
    unsigned long long iters_total = 0;
    for (int sidx = 0; sidx < n_steps; sidx++) {
      // ---- A (+ B1 for leaves): top-down ----
      OB_COLD_DOWN(true, { down_bias(T, i, s, g, c); })
      // ---- B1: bias forces bottom-up over the inner links -> rhs b ----
      OB_COLD_UP(false, { up_bias(T, i, s, g, c); })
      __syncthreads();
      // ---- B2: composite inertia bottom-up -> Jacobi factors, effective inertia (leaves first) ----
#pragma unroll 1
      for (int k = 0; k < LPT; k++) {
        Slot T = slot_get<LPT>(L, k);
        if (is_valid(T) && !is_inner(T)) up_inertia(T, k * NT + tid, s, g, c);
        slot_put<LPT>(L, k, T);
      }
      __syncthreads();
      OB_COLD_UP(true, { up_inertia(T, i, s, g, c); })
      float bb_part = 0.f, bz_part = 0.f;
#pragma unroll
      for (int k = 0; k < LPT; k++)
        if (is_valid(L[k])) {
          const float4 t = lds4(smem, own0 + 2 * h.PS + k * NT * 16);
          bb_part += t.x * t.x + t.y * t.y;
          bz_part += t.x * t.x * t.z + t.y * t.y * t.w;
        }
      const float2 bbz = red.sum(bb_part, bz_part);     // its barrier also closes B2 (planes 0, 1, 3 are free again)
      const float bb = bbz.x, bz = bbz.y;
      // ---- C: PCG, warm-started from the previous dqd (x) ----
      int it = 0;
      bool bad = false;
      if (bb == 0.f) {
#pragma unroll
        for (int k = 0; k < LPT; k++)
          if (is_valid(L[k])) sts2(smem, ox + k * NT * 8, make_float2(0.f, 0.f));
      } else if (!(bb < INFINITY)) {
        bad = true;
      } else {
#pragma unroll
        for (int k = 0; k < LPT; k++)                   // first product: A x, i.e. p = x
          if (is_valid(L[k])) sts2(smem, own0 + 3 * h.PS + k * NT * 16, lds2(smem, ox + k * NT * 8));
        bool first = true;
        float rz = 0.f, rr = 0.f;
        // stopping rule: |r| <= tol |b| in the 2-norm (cg_norm 0) or in the preconditioned norm (cg_norm 1)
        const float tol2 = P.cg_tol * P.cg_tol * (P.cg_norm ? bz : bb);
        for (;;) {
          // ---- A p: top-down (leaves turn around at once), then bottom-up over the inner links ----
          float pAp_part = 0.f;
          OB_SWEEP_DOWN({ pAp_part += down_mv(L[k], i, own0 + k * NT * 16, h, smem, s, g, c); })
          OB_SWEEP_UP({ pAp_part += up_mv_inner(L[k], i, own0 + k * NT * 16, h, smem, s, g, c); })
          float rz_p = 0.f, rr_p = 0.f;
          if (first) {                                 // r = b - A x, z = P^-1 r, p = z
            first = false;
#pragma unroll
            for (int k = 0; k < LPT; k++)
              if (is_valid(L[k])) {
                const int own = own0 + k * NT * 16;
                const float4 rid = lds4(smem, own + 2 * h.PS);
                const float2 ap = lds2(smem, own + h.PS + 8);
                const float ra = rid.x - ap.x, rb = rid.y - ap.y;
                const float za = ra * rid.z, zb = rb * rid.w;
                sts2(smem, own + 2 * h.PS, make_float2(ra, rb));
                sts2(smem, own + 3 * h.PS, make_float2(za, zb));
                rz_p += ra * za + rb * zb; rr_p += ra * ra + rb * rb;
              }
            const float2 t = red.sum(rz_p, rr_p);
            rz = t.x; rr = P.cg_norm ? t.x : t.y;
          } else {
            const float pAp = red.sum(pAp_part, 0.f).x;
            const float alpha = rz / pAp;
            float z0[LPT], z1[LPT], pk0[LPT], pk1[LPT];
#pragma unroll
            for (int k = 0; k < LPT; k++) {
              z0[k] = 0.f; z1[k] = 0.f; pk0[k] = 0.f; pk1[k] = 0.f;
              if (is_valid(L[k])) {
                const int own = own0 + k * NT * 16;
                const float4 rid = lds4(smem, own + 2 * h.PS);
                const float2 ap = lds2(smem, own + h.PS + 8);
                const float2 pk = lds2(smem, own + 3 * h.PS);
                pk0[k] = pk.x; pk1[k] = pk.y;
                float2 x = lds2(smem, ox + k * NT * 8);
                x.x += alpha * pk.x; x.y += alpha * pk.y;
                sts2(smem, ox + k * NT * 8, x);
                const float ra = rid.x - alpha * ap.x, rb = rid.y - alpha * ap.y;
                sts2(smem, own + 2 * h.PS, make_float2(ra, rb));
                z0[k] = ra * rid.z; z1[k] = rb * rid.w;
                rz_p += ra * z0[k] + rb * z1[k]; rr_p += ra * ra + rb * rb;
              }
            }
            const float2 t = red.sum(rz_p, rr_p);
            const float beta = t.x / rz;
            rz = t.x; rr = P.cg_norm ? t.x : t.y;
#pragma unroll
            for (int k = 0; k < LPT; k++)
              if (is_valid(L[k]))
                sts2(smem, own0 + 3 * h.PS + k * NT * 16, make_float2(z0[k] + beta * pk0[k], z1[k] + beta * pk1[k]));
            it++;
          }
          if (!(rr > tol2 && it < P.cg_max_iter)) break;
        }
        if (!(rr <= tol2)) {
          if (rr == rr && rr < INFINITY) status |= OB_STATUS_CG_MAXITER;
          else bad = true;
        }
      }
      // a non-finite solve freezes the world at its last finite state
      int nf = 0;
#pragma unroll
      for (int k = 0; k < LPT; k++)
        if (is_valid(L[k])) {
          const float2 x = lds2(smem, ox + k * NT * 8);
          nf |= !(fabsf(x.x) < INFINITY) || !(fabsf(x.y) < INFINITY);
        }
      if (__syncthreads_or(nf || bad)) { status |= OB_STATUS_NONFINITE; break; }

      // ---- D: integrate, predicates ----
      const int step_now = step0 + sidx;
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        if (!is_valid(L[k])) continue;
        const int i = k * NT + tid;
        const float2 x = s.x2[i], w0 = s.w2[i], q0 = s.q2[i];
        float wa = w0.x + x.x, wb = w0.y + x.y;
        if (P.qd_max > 0.f) {
          wa = fminf(fmaxf(wa, -P.qd_max), P.qd_max);
          wb = fminf(fmaxf(wb, -P.qd_max), P.qd_max);
        }
        const float qa = fmaf(P.h, wa, q0.x), qb = fmaf(P.h, wb, q0.y);
        s.w2[i] = make_float2(wa, wb); s.q2[i] = make_float2(qa, qb);
        if (!s.rupt[i]) {
          const float Ki = __ldg(g.K + i), Mx = __ldg(g.Mmax + i);
          const float mu = Ki * sqrtf(qa * qa + qb * qb);                   // Eq. 5
          const int rcn = mu > Mx ? s.rc[i] + 1 : 0;
          if (rcn >= P.rupture_frames) {
            s.rupt[i] = 1; s.rc[i] = 0;
            push_event(c, w, step_now, 0, __ldg(c.link_ext + d.link_base + i), mu, Mx);
          } else {
            s.rc[i] = (unsigned char)rcn;
          }
        }
      }
      for (int a = tid; a < d.A; a += NT) {
        const int Ap = d.Ap;
        const bool att = s.att[a] != 0;
        const float ma = s.am[a], inv_m = 1.f / ma;
        const float fdet = s.afd[a];
        float3 ft = att ? f3(s.ft[a], s.ft[Ap + a], s.ft[2 * Ap + a]) : f3(0, 0, 0);
        const float3 fu = f3(s.fu[a], s.fu[Ap + a], s.fu[2 * Ap + a]);
        float3 va = f3(s.v[a], s.v[Ap + a], s.v[2 * Ap + a]);
        va.x += P.h * (P.gravity[0] + (ft.x + fu.x) * inv_m);
        va.y += P.h * (P.gravity[1] + (ft.y + fu.y) * inv_m);
        va.z += P.h * (P.gravity[2] + (ft.z + fu.z) * inv_m);
        s.v[a] = va.x; s.v[Ap + a] = va.y; s.v[2 * Ap + a] = va.z;
        s.u[a] = fmaf(P.h, va.x, s.u[a]); s.u[Ap + a] = fmaf(P.h, va.y, s.u[Ap + a]);
        s.u[2 * Ap + a] = fmaf(P.h, va.z, s.u[2 * Ap + a]);
        if (att) {
          const float fun = s.fun[a], fsn = s.fsn[a], thrB = P.detach_kappa * fdet;
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
      steps_done++;
      last_iters = it;
      iters_total += (unsigned long long)it;
      __syncthreads();
    }

    // ---- write the state back: two TMA bulk stores ----
    if (status & OB_STATUS_NONFINITE) {
#pragma unroll
      for (int k = 0; k < LPT; k++)
        if (is_valid(L[k])) s.x2[k * NT + tid] = make_float2(0.f, 0.f);
    }
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
      tma_store(c.link_blk + d.link_blk_off, s.q2, (uint32_t)link_state_bytes(Np));
      if (d.Ap) tma_store(c.apple_blk + d.apple_blk_off, s.u, (uint32_t)apple_state_bytes(d.Ap));
      tma_store_commit_wait();
      info->step = step0 + steps_done;
      info->last_iters = last_iters;
      info->status = status;
      info->steps_taken += steps_done;
      info->cg_iters += iters_total;
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------------
// launchers: one instantiation per size class (ob_internal.h: kStepClasses)
// ------------------------------------------------------------------------------------------------------
#define OB_FOR_CLASS(cls, CALL)                         \
  switch (cls) {                                        \
    case 0: { CALL(128, 2, 6); break; }                 \
    case 1: { CALL(128, 4, 4); break; }                 \
    case 2: { CALL(256, 4, 2); break; }                 \
    case 3: { CALL(512, 3, 1); break; }                 \
    default: return cudaErrorInvalidValue;              \
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
                        int grid, int smem, cudaStream_t s) {
#define OB_LAUNCH(NT, LPT, MINB) k_step<NT, LPT, MINB><<<grid, NT, smem, s>>>(c, order, n_in_class, queue, n_steps);
  OB_FOR_CLASS(cls, OB_LAUNCH)
#undef OB_LAUNCH
  return cudaGetLastError();
}

}  // namespace ob
