// ob_step.cu -- k_step, the product kernel (sm_100a): n physics steps of every world in one launch.
//
// One CTA per world in flight (persistent, work queue per size class), several CTAs per SM.  Everything the
// level-synchronous tree sweeps touch lives in SHARED MEMORY as float4 planes indexed by link, so the sweep code
// exists once, is a few hundred instructions long (it has to stay inside the instruction cache: the first
// versions of this kernel were no_instruction-stalled) and runs over any number of links.  Registers hold what
// only the owner of a link needs: the PCG vectors x, r and the Jacobi factors (link tid + k * NT <-> slot k).
// The apple block is staged by one TMA bulk copy (UBLKCP) and written back the same way; q, qd stay in global
// memory (L2) because only the once-per-step phases A and D touch them.
//
//   A   top-down:  joint transforms (Eq. 3), displacement-form FK, velocities, bias accelerations;
//                  tether forces (Eq. 6 / Eq. 7) and user wrenches -> link bias forces
//   B1  bottom-up: bias torques -> rhs b (Eq. 4 spring-damper terms)
//   B2  bottom-up: composite inertia -> exact diagonal of M for the Jacobi preconditioner, effective link inertia
//   C   matrix-free Jacobi-PCG on (M + M_teth + diag(arm + hD + h^2 K)) dqd = b  (north_star);
//                  M v = acceleration-only inverse dynamics: top-down a_i, bottom-up f_i, project on S_i
//   D   integrate joints and apples; rupture (Eq. 5) and detach predicates
//
// Order.  Links are in plain breadth-first order: levels contiguous, the children of a link contiguous.  The
// leading levels that fit into links 0..31 (n_top of them) are swept by warp 0 with __syncwarp only; every other
// level ends with one block barrier.  In the PCG sweeps only the deepest level turns around inside the top-down
// pass (all of its links are leaves); in the once-per-step sweeps every leaf does.
//
// Planes (S = Np + 1 columns; column Np is never written and stays zero: it stands in for the trunk's parent).
//   M0, M1   A: kinematics an inner link publishes for its children (with PD, C3 and the overflow: 24 floats);
//            B1: (n, f) for the parent; B2: composite inertia for the parent; C: (alpha, a) on the way down,
//            (n, f) on the way up, A p in M1.zw
//   PD       (p, diagonal terms arm + (h c_d + h^2) K); B2 borrows .xy
//   C0..C2   E (parent -> link rotation, row-major), c2, s2, parent length
//   C3       effective link inertia (m, m c, I about the joint, I_zz) incl. on-axis virtual tether masses (A15)
//   G        b after B1, then 1 / diag(A) after B2 (both end up in the owner's registers)
//   T        packed topology word: parent | first child << 11 | children << 22 | flags
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
  int Np, Ap, NIp, S;
  float4 *P;                          // records: P[7 * i + j], j = 0 M0, 1 M1, 2 PD, 3..5 C0..C2, 6 C3
  float2 *G;
  uint32_t *T;
  float4 *ovf;                        // ovf[j * NIp + inner slot], j = 0..2
  int *lev;                           // level offsets [n_levels + 1]
  // apple block (TMA)
  float *u, *v;                       // [3][Ap]
  unsigned char *att, *cA, *cB;
  float *ao, *ak, *am, *ac, *afd;     // ao = [3][Ap]
  float *ft, *fu, *fsn, *fun;         // tether force [3][Ap], user force [3][Ap], |f_s|, |f_user|
  WrenchSlots *wr;
};

__device__ __forceinline__ Sm carve(unsigned char *base, const WorldDesc &d) {
  Sm s;
  s.Np = d.Np; s.Ap = d.Ap; s.NIp = d.NIp; s.S = d.Np + 1;
  const int Np = d.Np, Ap = d.Ap;
  unsigned char *p = base;
  s.P = reinterpret_cast<float4 *>(p); p += step_planes_bytes(Np);
  s.G = reinterpret_cast<float2 *>(p); p += r16(8 * (Np + 1));
  s.T = reinterpret_cast<uint32_t *>(p); p += r16(4 * (Np + 1));
  s.ovf = reinterpret_cast<float4 *>(p); p += 48 * d.NIp;
  s.lev = reinterpret_cast<int *>(p); p += r16(4 * (d.n_levels + 1));
  float *f = reinterpret_cast<float *>(p);
  s.u = f; s.v = f + 3 * Ap;
  s.att = p + 24 * Ap; s.cA = s.att + Ap; s.cB = s.cA + Ap;
  f = reinterpret_cast<float *>(p + apple_state_bytes(Ap));
  s.ao = f; s.ak = f + 3 * Ap; s.am = f + 4 * Ap; s.ac = f + 5 * Ap; s.afd = f + 6 * Ap;
  p += r16(apple_block_bytes(Ap));
  f = reinterpret_cast<float *>(p);
  s.ft = f; f += 3 * Ap;
  s.fu = f; f += 3 * Ap;
  s.fsn = f; f += Ap;
  s.fun = f; f += Ap;
  s.wr = reinterpret_cast<WrenchSlots *>(f);
  return s;
}

// per-link data of one world in global memory (L2-resident; only the once-per-step phases read it)
struct Gm {
  float2 *q2, *w2, *x2;             // state (link block)
  unsigned char *rupt, *rc;
  const float4 *c4;                 // (m, m c, I about the joint, I_zz)
  const float *K, *rz;              // joint stiffness (Eq. 4), parent length
  const float4 *quat;
  const float *R0;                  // [k * Np + i]
  const float *Mmax;
  const float *arm;                 // [k * Np + i] or nullptr
  const int4 *topo2;                // x = first apple | n_apples << 16, y = inner slot | parent's inner slot << 16
};

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

// kinematic quantities of one link that the bias pass hands from its top-down half to its bottom-up half
struct Kin {
  M3 dR;               // R - R0 (displacement form)
  double dpx, dpy, dpz; // origin - rest origin; fp64: the tether stretch is the small difference of two sums
                        // along the chain and k_s times its rounding error is what the thinnest twigs feel
  float3 om, vl;       // spatial velocity
  float3 al, aln;      // bias spatial acceleration (gravity as base acceleration)
};

// ------------------------------------------------------------------------------------------------------
// bias force of one link: f = I a + v x* I v - tether reactions - user wrenches (RNEA with qdd = 0)
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void bias_force(const int i, const Kin &k, const uint32_t tw, const Sm &s, const Gm &g,
                                           const DevCtx &c, float3 &n, float3 &f) {
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

  const int nwr = s.wr->n;
  bool wr_here = false;
  for (int q = 0; q < nwr; q++) wr_here |= s.wr->body[q] == i;
  if (!(tw & kHasApples) && !wr_here) return;

  M3 R;                                                                   // world rotation R0 + dR
#pragma unroll
  for (int q = 0; q < 9; q++) R.a[q] = __ldg(g.R0 + (size_t)q * Np + i) + k.dR.a[q];
  // tethers on this link (Eq. 6, Eq. 7): everything about the hang point is at hand here
  const int4 t2 = __ldg(g.topo2 + i);
  const int ast = t2.x & 0xffff, nap = t2.x >> 16;
  const float eta_h = P.tether_implicit ? P.h : 0.f;
  for (int a = ast; a < ast + nap; a++) {
    if (!s.att[a]) continue;
    const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
    const float3 dro = mul(k.dR, o);
    const double dhx = k.dpx + (double)dro.x, dhy = k.dpy + (double)dro.y, dhz = k.dpz + (double)dro.z;   // x_hang - anchor
    const float ks = s.ak[a], cdamp = s.ac[a], ma = s.am[a];
    // x_a - x_hang = u + sag - dh with the rest sag m g / k_s (u is stored relative to the rest position)
    const float gk = ma / ks;
    const float3 st = f3((float)((double)s.u[a] + ((double)(gk * P.gravity[0]) - dhx)),
                         (float)((double)s.u[Ap + a] + ((double)(gk * P.gravity[1]) - dhy)),
                         (float)((double)s.u[2 * Ap + a] + ((double)(gk * P.gravity[2]) - dhz)));
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
    if ((tw & kSnapped) && P.forces_off_on_snapped) continue;
    const float3 fl = mulT(R, f3(s.wr->force[q][0], s.wr->force[q][1], s.wr->force[q][2]));
    const float3 pt = f3(s.wr->point[q][0], s.wr->point[q][1], s.wr->point[q][2]);
    f = f - fl;
    n = n - cross(pt, fl);
  }
}

// project the accumulated bias force on the joint axes -> rhs b (G[i]), the diagonal damping / stiffness terms
// (PD[i].zw), and publish (n, f) in the parent frame (M0[i], M1[i].xy)
__device__ __forceinline__ void finish_bias(const Jt &j, const int i, const uint32_t tw, float3 n, float3 f,
                                            const Sm &s, const Gm &g, const DevCtx &c) {
  const ob_params &P = c.P;
  const int Np = s.Np, S = s.S;
  const float tau1 = j.c2 * n.x + j.s2 * n.z, tau2 = n.y;
  const float Kt = (tw & kRuptured) ? 0.f : __ldg(g.K + i), Dt = P.c_d * Kt;
  const float2 th = g.q2[i], w = g.w2[i];
  const float b1 = P.h * (-tau1 - Kt * th.x - (Dt + P.h * Kt) * w.x);
  const float b2 = P.h * (-tau2 - Kt * th.y - (Dt + P.h * Kt) * w.y);
  s.G[i] = make_float2(b1, b2);
  float dt0 = (P.h * P.c_d + P.h * P.h) * Kt, dt1 = dt0;
  if (g.arm) {
    dt0 += __ldg(g.arm + i);
    dt1 += __ldg(g.arm + Np + i);
  }
  reinterpret_cast<float2 *>(s.P + 7 * i + 2)[1] = make_float2(dt0, dt1);    // arm + (h c_d + h^2) K per DoF
  if (!(tw & kTrunk)) {
    const float3 fp = mulT(j.E, f);
    float3 np = mulT(j.E, n);
    np.x -= j.rz * fp.y; np.y += j.rz * fp.x;
    s.P[7 * i] = make_float4(np.x, np.y, np.z, fp.x);
    *reinterpret_cast<float2 *>(s.P + 7 * i + 1) = make_float2(fp.y, fp.z);
  }
}

// ------------------------------------------------------------------------------------------------------
// phase A for one link (top-down); a leaf goes straight on to its phase-B1 half
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void down_bias(const int i, const Sm &s, const Gm &g, const DevCtx &c) {
  const int Np = s.Np, NIp = s.NIp, S = s.S;
  const ob_params &P = c.P;
  uint32_t tw = s.T[i];
  const float2 th = g.q2[i], w = g.w2[i];
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
  Jt j;                                                            // E = Rrel^T
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int cc = 0; cc < 3; cc++) j.E.a[3 * r + cc] = Rrel.a[3 * cc + r];
  j.c2 = c2; j.s2 = s2;
  const int4 t2 = __ldg(g.topo2 + i);

  // parent quantities (world = parent of the trunk: at rest, spatial acceleration (0; -g))
  M3 dRp;
  double dppx = 0.0, dppy = 0.0, dppz = 0.0;
  float3 wp = f3(0, 0, 0), vp = f3(0, 0, 0), alp = f3(0, 0, 0);
  float3 ap = f3(-P.gravity[0], -P.gravity[1], -P.gravity[2]);
  uint32_t snapped_p = 0;
  float rz = 0.f;
#pragma unroll
  for (int q = 0; q < 9; q++) dRp.a[q] = 0.f;
  if (!(tw & kTrunk)) {
    const int par = (int)(tw & kParMask), ps = (int)((uint32_t)t2.y >> 16);
    const float4 t0 = s.P[7 * par], t1 = s.P[7 * par + 1], t2v = s.P[7 * par + 2], t3 = s.P[7 * par + 6],
                 t4 = s.ovf[ps], t5 = s.ovf[NIp + ps];
    const double2 d0 = *reinterpret_cast<const double2 *>(s.ovf + 2 * NIp + ps);
    dRp.a[0] = t0.x; dRp.a[1] = t0.y; dRp.a[2] = t0.z; dRp.a[3] = t0.w;
    dRp.a[4] = t1.x; dRp.a[5] = t1.y; dRp.a[6] = t1.z; dRp.a[7] = t1.w;
    dRp.a[8] = t2v.x; wp = f3(t2v.y, t2v.z, t2v.w);
    vp = f3(t3.x, t3.y, t3.z); alp = f3(t3.w, t4.x, t4.y);
    ap = f3(t4.z, t4.w, t5.x);
    dppx = (double)t5.y + (double)t5.z; dppy = d0.x; dppz = d0.y;      // x as a float pair, y and z as doubles
    snapped_p = s.T[par] & kSnapped;
    rz = __ldg(g.rz + i);
  }
  j.rz = rz;
  store_jt(s.P, i, j);
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
  k.dpx = dppx + (double)rz * (double)dRp.a[2];
  k.dpy = dppy + (double)rz * (double)dRp.a[5];
  k.dpz = dppz + (double)rz * (double)dRp.a[8];

  // velocity and (bias) spatial acceleration in link coordinates
  const float3 vJ = f3(c2 * w1, w2, s2 * w1);
  k.om = mul(j.E, wp) + vJ;
  k.vl = mul(j.E, f3(vp.x + wp.y * rz, vp.y - wp.x * rz, vp.z));
  const float ww = w1 * w2;
  k.al = mul(j.E, alp) + f3(-s2 * ww, 0.f, c2 * ww) + cross(k.om, vJ);
  k.aln = mul(j.E, f3(ap.x + alp.y * rz, ap.y - alp.x * rz, ap.z)) + cross(k.vl, vJ);

  tw = (tw & ~kSnapped) | (((tw & kRuptured) || snapped_p) ? kSnapped : 0u);
  s.T[i] = tw;

  if ((tw >> kNcShift) & kNcMask) {
    const int is = t2.y & 0xffff;
    s.P[7 * i] = make_float4(k.dR.a[0], k.dR.a[1], k.dR.a[2], k.dR.a[3]);
    s.P[7 * i + 1] = make_float4(k.dR.a[4], k.dR.a[5], k.dR.a[6], k.dR.a[7]);
    s.P[7 * i + 2] = make_float4(k.dR.a[8], k.om.x, k.om.y, k.om.z);
    s.P[7 * i + 6] = make_float4(k.vl.x, k.vl.y, k.vl.z, k.al.x);
    s.ovf[is] = make_float4(k.al.y, k.al.z, k.aln.x, k.aln.y);
    const float dxh = (float)k.dpx;
    s.ovf[NIp + is] = make_float4(k.aln.z, dxh, (float)(k.dpx - (double)dxh), 0.f);
    *reinterpret_cast<double2 *>(s.ovf + 2 * NIp + is) = make_double2(k.dpy, k.dpz);
  } else {
    float3 n, f;
    bias_force(i, k, tw, s, g, c, n, f);
    finish_bias(j, i, tw, n, f, s, g, c);
  }
}

// phase B1 for one inner link: its own bias force (from the kinematics it published on the way down) plus
// what its children sent up
__device__ __forceinline__ void up_bias(const int i, const uint32_t tw, const Sm &s, const Gm &g, const DevCtx &c) {
  const int NIp = s.NIp, S = s.S;
  const int is = __ldg(g.topo2 + i).y & 0xffff;
  Kin k;
  {
    const float4 t0 = s.P[7 * i], t1 = s.P[7 * i + 1], t2v = s.P[7 * i + 2], t3 = s.P[7 * i + 6], t4 = s.ovf[is],
                 t5 = s.ovf[NIp + is];
    k.dR.a[0] = t0.x; k.dR.a[1] = t0.y; k.dR.a[2] = t0.z; k.dR.a[3] = t0.w;
    k.dR.a[4] = t1.x; k.dR.a[5] = t1.y; k.dR.a[6] = t1.z; k.dR.a[7] = t1.w;
    const double2 d0 = *reinterpret_cast<const double2 *>(s.ovf + 2 * NIp + is);
    k.dR.a[8] = t2v.x; k.om = f3(t2v.y, t2v.z, t2v.w);
    k.vl = f3(t3.x, t3.y, t3.z); k.al = f3(t3.w, t4.x, t4.y);
    k.aln = f3(t4.z, t4.w, t5.x);
    k.dpx = (double)t5.y + (double)t5.z; k.dpy = d0.x; k.dpz = d0.y;
  }
  float3 n, f;
  bias_force(i, k, tw, s, g, c, n, f);
  const int fc = (int)((tw >> kChShift) & kParMask), nc = (int)((tw >> kNcShift) & kNcMask);
  for (int ch = fc; ch < fc + nc; ch++) {
    const float4 u = s.P[7 * ch];
    const float2 v = *reinterpret_cast<const float2 *>(s.P + 7 * ch + 1);
    n = n + f3(u.x, u.y, u.z);
    f = f + f3(u.w, v.x, v.y);
  }
  finish_bias(load_jt(s.P, i), i, tw, n, f, s, g, c);
}

// ------------------------------------------------------------------------------------------------------
// phase B2 for one link: composite rigid-body inertia about the link origin (mass, first moment h, symmetric
// I) -> exact diagonal of M -> Jacobi factors (G[i]); effective link inertia for A v (C3[i]); publish the
// composite inertia in the parent frame (M0[i], M1[i], PD[i].xy)
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void up_inertia(const int i, const Sm &s, const Gm &g, const DevCtx &c) {
  const int S = s.S, Ap = s.Ap;
  const ob_params &P = c.P;
  uint32_t tw = s.T[i];
  const float4 c4 = __ldg(g.c4 + i);
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
  const float d1 = c2 * c2 * Ixx + 2.f * c2 * s2 * Ixz + s2 * s2 * Izz + dt.x;
  const float d2 = Iyy + dt.y;
  float2 id = make_float2(1.f, 1.f);
  if (P.precond == 1) id = make_float2(1.f / d1, 1.f / d2);
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
  // children: the first four with all loads in flight at once (a missing child reads the zero record)
  const float4 *ch = P + 7 * (int)((tw >> kChShift) & kParMask);
  const int nc = (int)((tw >> kNcShift) & kNcMask);
  {
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
  }
#pragma unroll 1
  for (int k = 4; k < nc; k++) {
    const float4 u = ch[7 * k], v = ch[7 * k + 1];
    n = n + f3(u.x, u.y, u.z);
    f = f + f3(u.w, v.x, v.y);
  }
  const float t1 = j.c2 * n.x + j.s2 * n.z + pd.z * pd.x;     // pd = (p0, p1, dt0, dt1)
  const float t2 = n.y + pd.w * pd.y;
  const float3 fp = mulT(j.E, f);                             // the trunk publishes into its own column, which nobody reads
  float3 np = mulT(j.E, n);
  np.x -= j.rz * fp.y; np.y += j.rz * fp.x;
  rec[0] = make_float4(np.x, np.y, np.z, fp.x);
  rec[1] = make_float4(fp.y, fp.z, t1, t2);
  return pd.x * t1 + pd.y * t2;
}

// fence after level l of a top-down sweep / after level l of a bottom-up sweep (see "Order" above)
#define OB_FENCE_DOWN(l) { if ((l) + 1 < ntop) __syncwarp(); else __syncthreads(); }
#define OB_FENCE_UP(l) { if ((l) < ntop) __syncwarp(); else __syncthreads(); }

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
  const int tid = threadIdx.x;
  const ob_params &P = c.P;
  uint32_t parity = 0;
  if (tid == 0) mbar_init(&s_bar, 1);
  __syncthreads();
  Reducer<NT> red;
  red.stage = s_stage;
  red.flip = 0;
  red.tid = tid;

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
    const int Np = d.Np, S = Np + 1, N = d.N;
    const int nlev = d.n_levels, ntop = d.n_top;
    // warps other than warp 0 own no link of the n_top leading levels: they enter a top-down sweep at the level
    // whose fence is the first block barrier and leave a bottom-up sweep after the last one
    const int l_first_down = tid < 32 ? 0 : ntop - 1, l_last_up = tid < 32 ? 0 : ntop;
    float4 *const PL = s.P;
    Gm g;
    {
      unsigned char *lb = c.link_blk + d.link_blk_off;
      g.q2 = reinterpret_cast<float2 *>(lb); g.w2 = g.q2 + Np; g.x2 = g.w2 + Np;
      g.rupt = lb + 24 * Np; g.rc = g.rupt + Np;
      const unsigned char *cst = lb + link_state_bytes(Np);
      g.c4 = reinterpret_cast<const float4 *>(cst);
      g.K = reinterpret_cast<const float *>(cst) + 4 * Np;
      g.rz = g.K + Np;
      g.quat = c.quat + d.link_base;
      g.R0 = c.R0 + 9 * (size_t)d.link_base;
      g.Mmax = c.Mmax + d.link_base;
      g.arm = c.arm ? c.arm + 2 * (size_t)d.link_base : nullptr;
      g.topo2 = c.topo2 + d.link_base;
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
      for (int i = tid; i < S; i += NT) {
        uint32_t tw = (uint32_t)Np | kTrunk;
        if (i < N) {
          const int4 tp = __ldg(c.topo + d.link_base + i);
          const int4 t2 = __ldg(g.topo2 + i);
          const uint32_t nc = (uint32_t)t2.w, fc = nc ? ((uint32_t)tp.y & 0xffffu) : 0u;
          tw = (tp.x >= 0 ? (uint32_t)tp.x : ((uint32_t)Np | kTrunk)) | (fc << kChShift) | (nc << kNcShift) |
               ((t2.x >> 16) ? kHasApples : 0u) | (g.rupt[i] ? kRuptured : 0u);
        }
        s.T[i] = tw;
      }
    }
    float2 x[LPT], r[LPT], idg[LPT];
#pragma unroll
    for (int k = 0; k < LPT; k++) {
      const int i = tid + k * NT;
      x[k] = i < N ? g.x2[i] : make_float2(0.f, 0.f);
      r[k] = make_float2(0.f, 0.f);
      idg[k] = make_float2(0.f, 0.f);
    }
    if (d.Ap) {
      mbar_wait(&s_bar, parity);
      parity ^= 1;
    }
    __syncthreads();
    // lanes of warp 0 <-> links of the n_top leading levels: level of the lane's link, widest child list that
    // stays inside the warp
    const int ntopN = s.lev[ntop];
    int top_lvl = -1, top_maxc = 0;
    if (tid < ntopN) {
      for (int l = 0; l < ntop; l++)
        if (tid >= s.lev[l]) top_lvl = l;
      if (top_lvl < ntop - 1) top_maxc = (int)((s.T[tid] >> kNcShift) & kNcMask);
    }
    top_maxc = __reduce_max_sync(0xffffffffu, top_maxc);
    // user forces on apples are constant over the launch
    for (int a = tid; a < d.A; a += NT) {
      float3 fu = f3(0, 0, 0);
      for (int k = 0; k < s.wr->n; k++)
        if (s.wr->body[k] == N + a) fu = fu + f3(s.wr->force[k][0], s.wr->force[k][1], s.wr->force[k][2]);
      s.fu[a] = fu.x; s.fu[d.Ap + a] = fu.y; s.fu[2 * d.Ap + a] = fu.z;
      s.fun[a] = sqrtf(dot(fu, fu));
    }
    __syncthreads();

    int step0 = info->step, steps_done = 0, last_iters = 0;
    unsigned long long iters_total = 0;
    for (int sidx = 0; sidx < n_steps; sidx++) {
      // ---- A (+ B1 for leaves): top-down ----
#pragma unroll 1
      for (int l = l_first_down; l < nlev; l++) {
        const int le = s.lev[l + 1];
#pragma unroll 1
        for (int i = s.lev[l] + tid; i < le; i += NT) down_bias(i, s, g, c);
        OB_FENCE_DOWN(l)
      }
      // ---- B1: bias forces bottom-up over the inner links -> rhs b ----
#pragma unroll 1
      for (int l = nlev - 2; l >= l_last_up; l--) {
        const int le = s.lev[l + 1];
#pragma unroll 1
        for (int i = s.lev[l] + tid; i < le; i += NT) {
          const uint32_t tw = s.T[i];
          if ((tw >> kNcShift) & kNcMask) up_bias(i, tw, s, g, c);
        }
        OB_FENCE_UP(l)
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = tid + k * NT;
        if (i < N) r[k] = s.G[i];                       // b
      }
      // ---- B2: composite inertia bottom-up -> Jacobi factors, effective inertia (all leaves first) ----
#pragma unroll 1
      for (int i = tid; i < N; i += NT)
        if (((s.T[i] >> kNcShift) & kNcMask) == 0u) up_inertia(i, s, g, c);
      __syncthreads();
#pragma unroll 1
      for (int l = nlev - 2; l >= l_last_up; l--) {
        const int le = s.lev[l + 1];
#pragma unroll 1
        for (int i = s.lev[l] + tid; i < le; i += NT)
          if ((s.T[i] >> kNcShift) & kNcMask) up_inertia(i, s, g, c);
        OB_FENCE_UP(l)
      }
      __syncthreads();
      float bb_part = 0.f, bz_part = 0.f;
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = tid + k * NT;
        if (i < N) {
          idg[k] = s.G[i];
          bb_part += r[k].x * r[k].x + r[k].y * r[k].y;
          bz_part += r[k].x * r[k].x * idg[k].x + r[k].y * r[k].y * idg[k].y;
        }
      }
      const float2 bbz = red.sum(bb_part, bz_part);
      const float bb = bbz.x, bz = bbz.y;
      // ---- C: PCG, warm-started from the previous dqd (x) ----
      int it = 0;
      bool bad = false;
      if (bb == 0.f) {
#pragma unroll
        for (int k = 0; k < LPT; k++) x[k] = make_float2(0.f, 0.f);
      } else if (!(bb < INFINITY)) {
        bad = true;
      } else {
#pragma unroll
        for (int k = 0; k < LPT; k++) {                 // first product: A x, i.e. p = x
          const int i = tid + k * NT;
          if (i < N) *reinterpret_cast<float2 *>(PL + 7 * i + 2) = x[k];
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
          if (tid < 32) {
            const int me = tid < ntopN ? tid : Np;               // idle lanes work on the zero record
            const uint32_t tw = s.T[me];
            float4 *rec = PL + 7 * me;
            const float4 pd = rec[2];
            const Jt j = load_jt(PL, me);
            const int parl = (tw & kTrunk) ? tid : (int)(tw & kParMask);
            float3 al = f3(0, 0, 0), a = f3(0, 0, 0);
#pragma unroll 1
            for (int l = 0; l < ntop; l++) {
              float3 alp, ap;
              alp.x = __shfl_sync(0xffffffffu, al.x, parl); alp.y = __shfl_sync(0xffffffffu, al.y, parl);
              alp.z = __shfl_sync(0xffffffffu, al.z, parl);
              ap.x = __shfl_sync(0xffffffffu, a.x, parl); ap.y = __shfl_sync(0xffffffffu, a.y, parl);
              ap.z = __shfl_sync(0xffffffffu, a.z, parl);
              if (top_lvl == l) {
                if (tw & kTrunk) { alp = f3(0, 0, 0); ap = f3(0, 0, 0); }
                al = mul(j.E, alp) + f3(j.c2 * pd.x, pd.y, j.s2 * pd.x);
                a = mul(j.E, f3(ap.x + alp.y * j.rz, ap.y - alp.x * j.rz, ap.z));
              }
            }
            if (tid < ntopN) {
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
            for (int i = s.lev[l] + tid; i < le; i += NT) {
              const uint32_t tw = s.T[i];
              float4 *rec = PL + 7 * i;
              const float4 pd = rec[2];
              const Jt j = load_jt(PL, i);
              float3 al, a;
              mv_down(j, PL, tw, pd, al, a);
              if (deepest) {
                pAp_part += mv_up(j, PL, PL + 7 * Np, i, tw, pd, al, a, s, g, c);
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
            for (int i = s.lev[l] + tid; i < le; i += NT) {
              const uint32_t tw = s.T[i];
              const float4 *rec = PL + 7 * i;
              const float4 pd = rec[2];
              const Jt j = load_jt(PL, i);
              const float4 u = rec[0], v = rec[1];
              pAp_part += mv_up(j, PL, PL + 7 * Np, i, tw, pd, f3(u.x, u.y, u.z), f3(u.w, v.x, v.y), s, g, c);
            }
            __syncthreads();
          }
          if (tid < 32) {
            const int me = tid < ntopN ? tid : Np;
            const uint32_t tw = s.T[me];
            float4 *rec = PL + 7 * me;
            const float4 pd = rec[2], I = rec[6];
            const Jt j = load_jt(PL, me);
            const float4 u = rec[0], v = rec[1];
            const float3 al = f3(u.x, u.y, u.z), a = f3(u.w, v.x, v.y);
            const int fc = (int)((tw >> kChShift) & kParMask), nc = (int)((tw >> kNcShift) & kNcMask);
            float3 un = f3(0, 0, 0), uf = f3(0, 0, 0);           // (n, f) of this link in its parent's frame
            float t1 = 0.f, t2 = 0.f;
#pragma unroll 1
            for (int l = ntop - 1; l >= 0; l--) {
              const bool mine = top_lvl == l;
              float3 n = f3(I.z * al.x - I.y * a.y, I.z * al.y + I.y * a.x, I.w * al.z);
              float3 f = f3(I.x * a.x + I.y * al.y, I.x * a.y - I.y * al.x, I.x * a.z);
              if (mine && (tw & kOffax)) {
                const Force6 t = offaxis_tethers(__ldg(g.topo2 + me), al, a, s.att, s.ao, s.ak, s.Ap, P.h * P.h);
                n = n + t.n; f = f + t.f;
              }
              if (l == ntop - 1) {                               // children (if any) are in shared memory
                if (mine) {
#pragma unroll 1
                  for (int k = 0; k < nc; k++) {
                    const float4 cu = PL[7 * (fc + k)], cv = PL[7 * (fc + k) + 1];
                    n = n + f3(cu.x, cu.y, cu.z);
                    f = f + f3(cu.w, cv.x, cv.y);
                  }
                }
              } else {                                           // children are lanes fc .. fc + nc - 1
#pragma unroll 1
                for (int k = 0; k < top_maxc; k++) {
                  const int src = min(fc + k, 31);
                  float3 cn, cf;
                  cn.x = __shfl_sync(0xffffffffu, un.x, src); cn.y = __shfl_sync(0xffffffffu, un.y, src);
                  cn.z = __shfl_sync(0xffffffffu, un.z, src);
                  cf.x = __shfl_sync(0xffffffffu, uf.x, src); cf.y = __shfl_sync(0xffffffffu, uf.y, src);
                  cf.z = __shfl_sync(0xffffffffu, uf.z, src);
                  if (k < nc) { n = n + cn; f = f + cf; }
                }
              }
              if (mine) {
                t1 = j.c2 * n.x + j.s2 * n.z + pd.z * pd.x;
                t2 = n.y + pd.w * pd.y;
                uf = mulT(j.E, f);
                un = mulT(j.E, n);
                un.x -= j.rz * uf.y; un.y += j.rz * uf.x;
              }
            }
            if (tid < ntopN) {
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
              const int i = tid + k * NT;
              if (i < N) {
                const float2 ap = reinterpret_cast<const float2 *>(PL + 7 * i + 1)[1];
                r[k].x -= ap.x; r[k].y -= ap.y;
                const float za = r[k].x * idg[k].x, zb = r[k].y * idg[k].y;
                *reinterpret_cast<float2 *>(PL + 7 * i + 2) = make_float2(za, zb);
                rz_p += r[k].x * za + r[k].y * zb; rr_p += r[k].x * r[k].x + r[k].y * r[k].y;
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
              const int i = tid + k * NT;
              z[k] = make_float2(0.f, 0.f); pk[k] = make_float2(0.f, 0.f);
              if (i < N) {
                const float2 ap = reinterpret_cast<const float2 *>(PL + 7 * i + 1)[1];
                pk[k] = *reinterpret_cast<const float2 *>(PL + 7 * i + 2);
                x[k].x += alpha * pk[k].x; x[k].y += alpha * pk[k].y;
                r[k].x -= alpha * ap.x; r[k].y -= alpha * ap.y;
                z[k] = make_float2(r[k].x * idg[k].x, r[k].y * idg[k].y);
                rz_p += r[k].x * z[k].x + r[k].y * z[k].y; rr_p += r[k].x * r[k].x + r[k].y * r[k].y;
              }
            }
            const float2 t = red.sum(rz_p, rr_p);
            const float beta = t.x / rz;
            rz = t.x; rr = P.cg_norm ? t.x : t.y;
#pragma unroll
            for (int k = 0; k < LPT; k++) {
              const int i = tid + k * NT;
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
      // a non-finite solve freezes the world at its last finite state
      int nf = 0;
#pragma unroll
      for (int k = 0; k < LPT; k++) nf |= !(fabsf(x[k].x) < INFINITY) || !(fabsf(x[k].y) < INFINITY);
      if (__syncthreads_or(nf || bad)) { status |= OB_STATUS_NONFINITE; break; }

      // ---- D: integrate, predicates ----
      const int step_now = step0 + sidx;
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = tid + k * NT;
        if (i >= N) continue;
        const float2 w0 = g.w2[i], q0 = g.q2[i];
        float wa = w0.x + x[k].x, wb = w0.y + x[k].y;
        if (P.qd_max > 0.f) {
          wa = fminf(fmaxf(wa, -P.qd_max), P.qd_max);
          wb = fminf(fmaxf(wb, -P.qd_max), P.qd_max);
        }
        const float qa = fmaf(P.h, wa, q0.x), qb = fmaf(P.h, wb, q0.y);
        g.w2[i] = make_float2(wa, wb); g.q2[i] = make_float2(qa, qb);
        const uint32_t tw = s.T[i];
        if (!(tw & kRuptured)) {
          const float Ki = __ldg(g.K + i), Mx = __ldg(g.Mmax + i);
          const float mu = Ki * sqrtf(qa * qa + qb * qb);                   // Eq. 5
          const int rc0 = g.rc[i];
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

    // ---- write the state back: x from the registers, the apple state by one TMA bulk store ----
#pragma unroll
    for (int k = 0; k < LPT; k++) {
      const int i = tid + k * NT;
      if (i < N) g.x2[i] = (status & OB_STATUS_NONFINITE) ? make_float2(0.f, 0.f) : x[k];
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
    case 1: { CALL(256, 2, 3); break; }                 \
    case 2: { CALL(512, 2, 1); break; }                 \
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
