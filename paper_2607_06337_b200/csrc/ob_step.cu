// ob_step.cu -- k_step, the product kernel (sm_100a): n physics steps of every world in one launch.
//
// One CTA per world in flight (persistent, work queue per size class).  The world's link block and apple
// block are staged into shared memory by two TMA bulk copies (UBLKCP) and written back the same way.
// A thread owns the same LPT links for the whole launch (link i <-> slot i / NT of thread i % NT) and keeps
// everything the PCG loop touches in REGISTERS: joint transform E, (c2, s2), effective inertia, diagonal
// terms, Jacobi factors and the vectors x, r, p, A p.  Shared memory carries only what crosses threads:
// the parent -> child and child -> parent mailboxes of the level-synchronous tree sweeps.
//
//   A  top-down:  joint transforms (Eq. 3), displacement-form FK, velocities, bias accelerations,
//                 tether forces (Eq. 6 / Eq. 7), user wrenches -> link bias forces
//   B  bottom-up: bias torques -> rhs b (Eq. 4 spring-damper terms); composite inertia ->
//                 exact diagonal of M for the Jacobi preconditioner
//   C  matrix-free Jacobi-PCG on (M + M_teth + diag(arm + hD + h^2 K)) dqd = b  (north_star);
//                 M v = acceleration-only inverse dynamics: top-down a_i, bottom-up f_i, project on S_i
//   D  integrate joints and apples; rupture (Eq. 5) and detach predicates
//
// Sweep schedule.  Links are level-ordered, so links 0..31 belong to warp 0: the leading levels that fit
// there (n_top of them) are swept by warp 0 alone with __syncwarp.  A leaf link has nothing to wait for on
// the way up, so it does its bottom-up half inside the top-down pass; the bottom-up passes only visit inner
// links.  With levels of 1, 3, 7, 19, 50, 130, 190 links this is 6 block barriers per A v instead of 14.
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
  int N, A, Np, Ap;
  // link block (TMA)
  float *q0, *q1, *w0, *w1, *x0, *x1;
  unsigned char *rupt, *rc;
  float *K, *m, *mc, *Io, *Iz, *rz;
  // apple block (TMA)
  float *u, *v;                       // [3][Ap]
  unsigned char *att, *cA, *cB;
  float *ao, *ak, *am, *ac, *afd;     // ao = [3][Ap]
  // scratch: float4 S[6][Np].  Phase A: parent -> child (dR, dp, omega, v, alpha, a).  Phase B: child -> parent
  // S[0..3] = (n, f, composite inertia).  PCG: S[0] and the head of S[1] = the 6-float mailbox (A, B).
  float4 *S;
  float2 *B;
  float *ft, *fu, *fsn, *fun;         // tether force [3][Ap], user force [3][Ap], |f_s|, |f_user|
  WrenchSlots *wr;
  unsigned char *snapped;
};

__device__ __forceinline__ Sm carve(unsigned char *base, const WorldDesc &d) {
  Sm s;
  s.N = d.N; s.A = d.A; s.Np = d.Np; s.Ap = d.Ap;
  const int Np = d.Np, Ap = d.Ap;
  unsigned char *p = base;
  float *f = reinterpret_cast<float *>(p);
  s.q0 = f; s.q1 = f + Np; s.w0 = f + 2 * Np; s.w1 = f + 3 * Np; s.x0 = f + 4 * Np; s.x1 = f + 5 * Np;
  s.rupt = p + 24 * Np; s.rc = s.rupt + Np;
  f = reinterpret_cast<float *>(p + link_state_bytes(Np));
  s.K = f; s.m = f + Np; s.mc = f + 2 * Np; s.Io = f + 3 * Np; s.Iz = f + 4 * Np; s.rz = f + 5 * Np;
  p += link_block_bytes(Np);
  f = reinterpret_cast<float *>(p);
  s.u = f; s.v = f + 3 * Ap;
  s.att = p + 24 * Ap; s.cA = s.att + Ap; s.cB = s.cA + Ap;
  f = reinterpret_cast<float *>(p + apple_state_bytes(Ap));
  s.ao = f; s.ak = f + 3 * Ap; s.am = f + 4 * Ap; s.ac = f + 5 * Ap; s.afd = f + 6 * Ap;
  p += apple_block_bytes(Ap);
  s.S = reinterpret_cast<float4 *>(p);
  s.B = reinterpret_cast<float2 *>(s.S + Np);
  p += 6 * 16 * Np;
  f = reinterpret_cast<float *>(p);
  s.ft = f; f += 3 * Ap;
  s.fu = f; f += 3 * Ap;
  s.fsn = f; f += Ap;
  s.fun = f; f += Ap;
  s.wr = reinterpret_cast<WrenchSlots *>(f); f += sizeof(WrenchSlots) / 4;
  s.snapped = reinterpret_cast<unsigned char *>(f);
  return s;
}

// per-link registers of the owning thread
struct LinkRegs {
  int i;            // link index, -1 = empty slot
  int lvl;          // level, -1 = empty slot
  int par;          // parent link, -1 = trunk
  int cst, nch;     // children [cst, cst + nch)
  int ast, nap;     // apples [ast, ast + nap)
  int offax;        // an attached apple hangs off the link axis: its virtual mass is applied one by one in A v
  float E[9];       // parent -> link rotation
  float rz, c2, s2;
  float m, mc, Io, Iz;       // link inertia about the joint + on-axis virtual tether masses (A15)
  float dt0, dt1;            // arm + (h c_d + h^2) K per DoF
  float id0, id1;            // Jacobi factors 1 / diag(A)
  float x0, x1, r0, r1, p0, p1, ap0, ap1;
  float3 cn, cf;             // carried between the two halves of a sweep: bias (n, f) or (alpha, a)
};

// block-wide sum of two values, result broadcast to every thread; one barrier per call (double-buffered stage)
template <int NT>
struct Reducer {
  float2 *stage;   // [2][32]
  int flip;
  __device__ __forceinline__ float2 sum(float a, float b) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a += __shfl_xor_sync(0xffffffffu, a, o);
      b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    float2 *st = stage + 32 * flip;
    flip ^= 1;
    if ((threadIdx.x & 31) == 0) st[threadIdx.x >> 5] = make_float2(a, b);
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

// ------------------------------------------------------------------------------------------------------
// phase B for one link: gather the children, rhs b -> (r0, r1), composite inertia -> Jacobi factors,
// effective inertia for A v, and (if the link has a parent) publish (n, f, composite inertia) in the parent frame
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void up_bias(LinkRegs &L, const Sm &s, const DevCtx &c, const WorldDesc &d,
                                        float &bb, float &bz) {
  const int Np = s.Np, Ap = s.Ap, i = L.i;
  const ob_params &P = c.P;
  float3 n = L.cn, f = L.cf;
  // composite rigid-body inertia about the link origin: mass, first moment h, symmetric I (xx,yy,zz,xy,xz,yz)
  const float m0 = s.m[i], mc0 = s.mc[i], Io0 = s.Io[i], Iz0 = s.Iz[i];
  float cm = m0;
  float3 ch = f3(0.f, 0.f, mc0);
  float Ixx = Io0, Iyy = Io0, Izz = Iz0, Ixy = 0.f, Ixz = 0.f, Iyz = 0.f;
  L.m = m0; L.mc = mc0; L.Io = Io0; L.Iz = Iz0; L.offax = 0;
  if (P.tether_implicit) {
    for (int a = L.ast; a < L.ast + L.nap; a++) {
      if (!s.att[a]) continue;
      const float mv = P.h * P.h * s.ak[a];                     // virtual point mass h^2 k_s at the hang point
      const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
      cm += mv; ch = ch + mv * o;
      Ixx += mv * (o.y * o.y + o.z * o.z); Iyy += mv * (o.x * o.x + o.z * o.z); Izz += mv * (o.x * o.x + o.y * o.y);
      Ixy -= mv * o.x * o.y; Ixz -= mv * o.x * o.z; Iyz -= mv * o.y * o.z;
      if (o.x == 0.f && o.y == 0.f) { L.m += mv; L.mc += mv * o.z; L.Io += mv * o.z * o.z; }   // stays a body of revolution
      else L.offax = 1;
    }
  }
  for (int ch_i = L.cst; ch_i < L.cst + L.nch; ch_i++) {
    const float4 u0 = s.S[ch_i], u1 = s.S[Np + ch_i], u2 = s.S[2 * Np + ch_i], u3 = s.S[3 * Np + ch_i];
    n = n + f3(u0.x, u0.y, u0.z);
    f = f + f3(u0.w, u1.x, u1.y);
    cm += u1.z;
    ch = ch + f3(u1.w, u2.x, u2.y);
    Ixx += u2.z; Iyy += u2.w; Izz += u3.x; Ixy += u3.y; Ixz += u3.z; Iyz += u3.w;
  }
  const float c2 = L.c2, s2 = L.s2;
  const float tau1 = c2 * n.x + s2 * n.z, tau2 = n.y;
  const float Kt = s.rupt[i] ? 0.f : s.K[i], Dt = P.c_d * Kt;
  const float b1 = P.h * (-tau1 - Kt * s.q0[i] - (Dt + P.h * Kt) * s.w0[i]);
  const float b2 = P.h * (-tau2 - Kt * s.q1[i] - (Dt + P.h * Kt) * s.w1[i]);
  L.r0 = b1; L.r1 = b2;
  bb += b1 * b1 + b2 * b2;
  float dt0 = (P.h * P.c_d + P.h * P.h) * Kt, dt1 = dt0;
  if (c.arm) {
    dt0 += __ldg(c.arm + 2 * (size_t)d.link_base + i);
    dt1 += __ldg(c.arm + 2 * (size_t)d.link_base + Np + i);
  }
  L.dt0 = dt0; L.dt1 = dt1;
  const float d1 = c2 * c2 * Ixx + 2.f * c2 * s2 * Ixz + s2 * s2 * Izz + dt0;
  const float d2 = Iyy + dt1;
  if (P.precond == 1) { L.id0 = 1.f / d1; L.id1 = 1.f / d2; }
  else { L.id0 = 1.f; L.id1 = 1.f; }
  bz += b1 * b1 * L.id0 + b2 * b2 * L.id1;
  if (L.par >= 0) {
    M3 E;
#pragma unroll
    for (int k = 0; k < 9; k++) E.a[k] = L.E[k];
    const float rz = L.rz;
    const float3 fp = mulT(E, f);
    float3 np = mulT(E, n);
    np.x -= rz * fp.y; np.y += rz * fp.x;
    // composite inertia into the parent frame: rotate by Rrel = E^T, then move the origin by r = (0,0,rz)
    const float3 hp = mulT(E, ch);
    M3 I, T, Ip;
    I.a[0] = Ixx; I.a[1] = Ixy; I.a[2] = Ixz; I.a[3] = Ixy; I.a[4] = Iyy; I.a[5] = Iyz; I.a[6] = Ixz; I.a[7] = Iyz; I.a[8] = Izz;
#pragma unroll
    for (int r = 0; r < 3; r++)
#pragma unroll
      for (int cc = 0; cc < 3; cc++) T.a[3 * r + cc] = E.a[r] * I.a[cc] + E.a[3 + r] * I.a[3 + cc] + E.a[6 + r] * I.a[6 + cc];
    Ip = mul(T, E);
    const float sh = 2.f * rz * hp.z + cm * rz * rz;
    s.S[i] = make_float4(np.x, np.y, np.z, fp.x);
    s.S[Np + i] = make_float4(fp.y, fp.z, cm, hp.x);
    s.S[2 * Np + i] = make_float4(hp.y, hp.z + cm * rz, Ip.a[0] + sh, Ip.a[4] + sh);
    s.S[3 * Np + i] = make_float4(Ip.a[8], Ip.a[1], Ip.a[2] - rz * hp.x, Ip.a[5] - rz * hp.y);
  }
}

// ------------------------------------------------------------------------------------------------------
// phase A for one link (top-down); a leaf goes straight on to its phase-B half
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void down_bias(LinkRegs &L, const Sm &s, const DevCtx &c, const WorldDesc &d,
                                          float &bb, float &bz) {
  const int Np = s.Np, Ap = s.Ap, i = L.i, par = L.par;
  const ob_params &P = c.P;
  const float th1 = s.q0[i], th2 = s.q1[i], w1 = s.w0[i], w2 = s.w1[i];
  float s1, c1, s2, c2;
  sincosf(th1, &s1, &c1);
  sincosf(th2, &s2, &c2);
  const float sh1 = sinf(0.5f * th1), sh2 = sinf(0.5f * th2);
  const float vc1 = -2.f * sh1 * sh1, vc2 = -2.f * sh2 * sh2;      // cos - 1 without cancellation
  const M3 Q = quat_to_mat(__ldg(c.quat + d.link_base + i));
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
  for (int k = 0; k < 9; k++) L.E[k] = E.a[k];
  L.c2 = c2; L.s2 = s2;

  // parent quantities (world = parent of the trunk: at rest, spatial acceleration (0; -g))
  M3 dRp;
  float3 dpp = f3(0, 0, 0), wp = f3(0, 0, 0), vp = f3(0, 0, 0), alp = f3(0, 0, 0);
  float3 ap = f3(-P.gravity[0], -P.gravity[1], -P.gravity[2]);
  unsigned char snapped_p = 0;
  const float rz = L.rz;
#pragma unroll
  for (int k = 0; k < 9; k++) dRp.a[k] = 0.f;
  if (par >= 0) {
    const float4 t0 = s.S[par], t1 = s.S[Np + par], t2 = s.S[2 * Np + par], t3 = s.S[3 * Np + par],
                 t4 = s.S[4 * Np + par], t5 = s.S[5 * Np + par];
    dRp.a[0] = t0.x; dRp.a[1] = t0.y; dRp.a[2] = t0.z; dRp.a[3] = t0.w;
    dRp.a[4] = t1.x; dRp.a[5] = t1.y; dRp.a[6] = t1.z; dRp.a[7] = t1.w;
    dRp.a[8] = t2.x; dpp = f3(t2.y, t2.z, t2.w);
    wp = f3(t3.x, t3.y, t3.z); vp = f3(t3.w, t4.x, t4.y);
    alp = f3(t4.z, t4.w, t5.x); ap = f3(t5.y, t5.z, t5.w);
    snapped_p = s.snapped[par];
  }
  // displacement-form FK: R_i = R0_i + dR_i,  dR_i = dR_p Rrel + R0_i (RxRy - I);  dp_i = dp_p + dR_p (0,0,rz)
  M3 R0, G = XY;
  const float *R0g = c.R0 + 9 * (size_t)d.link_base + i;
#pragma unroll
  for (int k = 0; k < 9; k++) R0.a[k] = __ldg(R0g + (size_t)k * Np);
  G.a[0] = vc2; G.a[4] = vc1; G.a[8] = fmaf(vc1, vc2, vc1 + vc2);
  const M3 t1m = mul(dRp, Rrel), t2m = mul(R0, G);
  M3 dR, R;
#pragma unroll
  for (int k = 0; k < 9; k++) { dR.a[k] = t1m.a[k] + t2m.a[k]; R.a[k] = R0.a[k] + dR.a[k]; }
  const float3 dp = f3(dpp.x + rz * dRp.a[2], dpp.y + rz * dRp.a[5], dpp.z + rz * dRp.a[8]);

  // velocity and (bias) spatial acceleration in link coordinates
  const float3 vJ = f3(c2 * w1, w2, s2 * w1);
  const float3 om = mul(E, wp) + vJ;
  const float3 vl = mul(E, f3(vp.x + wp.y * rz, vp.y - wp.x * rz, vp.z));
  const float ww = w1 * w2;
  const float3 al = mul(E, alp) + f3(-s2 * ww, 0.f, c2 * ww) + cross(om, vJ);
  const float3 aln = mul(E, f3(ap.x + alp.y * rz, ap.y - alp.x * rz, ap.z)) + cross(vl, vJ);

  // f = I a + v x* I v  (cylinder: com on +z)
  const float m = s.m[i], mc = s.mc[i], Io = s.Io[i], Iz = s.Iz[i];
  float3 n = f3(Io * al.x - mc * aln.y, Io * al.y + mc * aln.x, Iz * al.z);
  float3 f = f3(m * aln.x + mc * al.y, m * aln.y - mc * al.x, m * aln.z);
  const float3 hn = f3(Io * om.x - mc * vl.y, Io * om.y + mc * vl.x, Iz * om.z);
  const float3 hf = f3(m * vl.x + mc * om.y, m * vl.y - mc * om.x, m * vl.z);
  n = n + cross(om, hn) + cross(vl, hf);
  f = f + cross(om, hf);

  const unsigned char snapped = s.rupt[i] | snapped_p;
  s.snapped[i] = snapped;

  // tethers on this link (Eq. 6, Eq. 7): everything about the hang point is at hand here
  const float eta_h = P.tether_implicit ? P.h : 0.f;
  for (int a = L.ast; a < L.ast + L.nap; a++) {
    if (!s.att[a]) continue;
    const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
    const float3 dh = dp + mul(dR, o);                                   // x_hang - anchor
    const float k = s.ak[a], cdamp = s.ac[a], ma = s.am[a];
    // x_a - x_hang = u + sag - dh with the rest sag m g / k_s (u is stored relative to the rest position)
    const float gk = ma / k;
    const float3 st = f3(s.u[a] + (gk * P.gravity[0] - dh.x), s.u[Ap + a] + (gk * P.gravity[1] - dh.y),
                         s.u[2 * Ap + a] + (gk * P.gravity[2] - dh.z));
    const float3 vh = mul(R, vl + cross(om, o));                         // world velocity of the hang point
    const float3 fs = (-k) * st;
    const float3 va = f3(s.v[a], s.v[Ap + a], s.v[2 * Ap + a]);
    s.ft[a] = fs.x - cdamp * va.x; s.ft[Ap + a] = fs.y - cdamp * va.y; s.ft[2 * Ap + a] = fs.z - cdamp * va.z;
    s.fsn[a] = sqrtf(dot(fs, fs));
    float3 fr = f3(k * (st.x - eta_h * vh.x) - ma * P.gravity[0], k * (st.y - eta_h * vh.y) - ma * P.gravity[1],
                   k * (st.z - eta_h * vh.z) - ma * P.gravity[2]);
    const float nr = sqrtf(dot(fr, fr));
    if (nr > P.react_max) fr = (P.react_max / nr) * fr;                  // clamp
    const float3 fl = mulT(R, fr);
    f = f - fl;
    n = n - cross(o, fl);
  }
  // user wrenches on this link (disabled on snapped sub-trees)
  const int nwr = s.wr->n;
  for (int k = 0; k < nwr; k++) {
    if (s.wr->body[k] != i) continue;
    if (snapped && P.forces_off_on_snapped) continue;
    const float3 fl = mulT(R, f3(s.wr->force[k][0], s.wr->force[k][1], s.wr->force[k][2]));
    const float3 pt = f3(s.wr->point[k][0], s.wr->point[k][1], s.wr->point[k][2]);
    f = f - fl;
    n = n - cross(pt, fl);
  }
  L.cn = n; L.cf = f;
  if (L.nch) {
    s.S[i] = make_float4(dR.a[0], dR.a[1], dR.a[2], dR.a[3]);
    s.S[Np + i] = make_float4(dR.a[4], dR.a[5], dR.a[6], dR.a[7]);
    s.S[2 * Np + i] = make_float4(dR.a[8], dp.x, dp.y, dp.z);
    s.S[3 * Np + i] = make_float4(om.x, om.y, om.z, vl.x);
    s.S[4 * Np + i] = make_float4(vl.y, vl.z, al.x, al.y);
    s.S[5 * Np + i] = make_float4(al.z, aln.x, aln.y, aln.z);
  } else {
    up_bias(L, s, c, d, bb, bz);
  }
}

// ------------------------------------------------------------------------------------------------------
// phase C: A v for one link.  up_mv: f = I a + children, project on S (+ diagonal terms), publish to the
// parent; returns v . (A v) of this link.  down_mv: accelerations from the parent; a leaf goes straight up.
// Mailbox: A[i] = (x, y, z of the angular part, x of the linear part), B[i] = (y, z of the linear part).
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ float up_mv(LinkRegs &L, const Sm &s, const DevCtx &c) {
  const int Np = s.Np, Ap = s.Ap;
  const float3 al = L.cn, a = L.cf;
  float3 n = f3(L.Io * al.x - L.mc * a.y, L.Io * al.y + L.mc * a.x, L.Iz * al.z);
  float3 f = f3(L.m * a.x + L.mc * al.y, L.m * a.y - L.mc * al.x, L.m * a.z);
  if (L.offax) {
    for (int q = L.ast; q < L.ast + L.nap; q++) {
      if (!s.att[q]) continue;
      const float3 o = f3(s.ao[q], s.ao[Ap + q], s.ao[2 * Ap + q]);
      if (o.x == 0.f && o.y == 0.f) continue;                 // already inside (m, mc, Io)
      const float mv = c.P.h * c.P.h * s.ak[q];
      const float3 fp = mv * (a + cross(al, o));
      f = f + fp;
      n = n + cross(o, fp);
    }
  }
  for (int ch = L.cst; ch < L.cst + L.nch; ch++) {
    const float4 u = s.S[ch];
    const float2 w = s.B[ch];
    n = n + f3(u.x, u.y, u.z);
    f = f + f3(u.w, w.x, w.y);
  }
  const float t1 = L.c2 * n.x + L.s2 * n.z + L.dt0 * L.p0;
  const float t2 = n.y + L.dt1 * L.p1;
  L.ap0 = t1; L.ap1 = t2;
  if (L.par >= 0) {
    M3 E;
#pragma unroll
    for (int k = 0; k < 9; k++) E.a[k] = L.E[k];
    const float3 fp = mulT(E, f);
    float3 np = mulT(E, n);
    np.x -= L.rz * fp.y; np.y += L.rz * fp.x;
    s.S[L.i] = make_float4(np.x, np.y, np.z, fp.x);
    s.B[L.i] = make_float2(fp.y, fp.z);
  }
  return L.p0 * t1 + L.p1 * t2;
}

__device__ __forceinline__ float down_mv(LinkRegs &L, const Sm &s, const DevCtx &c) {
  float3 al = f3(0, 0, 0), a = f3(0, 0, 0);
  if (L.par >= 0) {
    const float4 u = s.S[L.par];
    const float2 w = s.B[L.par];
    const float3 alp = f3(u.x, u.y, u.z), ap = f3(u.w, w.x, w.y);
    M3 E;
#pragma unroll
    for (int k = 0; k < 9; k++) E.a[k] = L.E[k];
    al = mul(E, alp);
    a = mul(E, f3(ap.x + alp.y * L.rz, ap.y - alp.x * L.rz, ap.z));
  }
  al = al + f3(L.c2 * L.p0, L.p1, L.s2 * L.p0);
  L.cn = al; L.cf = a;
  if (L.nch) {
    s.S[L.i] = make_float4(al.x, al.y, al.z, a.x);
    s.B[L.i] = make_float2(a.y, a.z);
    return 0.f;
  }
  return up_mv(L, s, c);
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
  const int tid = threadIdx.x;
  const bool warp0 = tid < 32;
  const ob_params &P = c.P;
  uint32_t parity = 0;
  if (tid == 0) mbar_init(&s_bar, 1);
  __syncthreads();
  Reducer<NT> red;
  red.stage = s_stage;
  red.flip = 0;
  LinkRegs L[LPT];

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
    const int nlev = d.n_levels, ntop = d.n_top;

    // ---- stage the world: two TMA bulk copies (link block, apple block) onto one mbarrier ----
    if (tid == 0) {
      fence_proxy_async();
      const uint32_t lb = (uint32_t)link_block_bytes(d.Np), ab = (uint32_t)apple_block_bytes(d.Ap);
      mbar_expect_tx(&s_bar, lb + ab);
      tma_load(s.q0, c.link_blk + d.link_blk_off, lb, &s_bar);
      if (ab) tma_load(s.u, c.apple_blk + d.apple_blk_off, ab, &s_bar);
    }
    {
      const int32_t *src = reinterpret_cast<const int32_t *>(c.wrench + w);
      int32_t *dst = reinterpret_cast<int32_t *>(s.wr);
      for (int k = tid; k < (int)(sizeof(WrenchSlots) / 4); k += NT) dst[k] = __ldg(src + k);
    }
#pragma unroll
    for (int k = 0; k < LPT; k++) {                  // topology of the links this thread owns
      const int i = k * NT + tid;
      L[k].i = -1; L[k].lvl = -1; L[k].par = -1; L[k].cst = 0; L[k].nch = 0; L[k].ast = 0; L[k].nap = 0; L[k].offax = 0;
      if (i < d.N) {
        const int4 tp = __ldg(c.topo + d.link_base + i);
        L[k].i = i; L[k].par = tp.x; L[k].cst = tp.y; L[k].nch = tp.z & 0xffff; L[k].nap = tp.z >> 16;
        L[k].ast = tp.w & 0xffff; L[k].lvl = tp.w >> 16;
      }
    }
    mbar_wait(&s_bar, parity);
    parity ^= 1;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < LPT; k++) {
      const int i = L[k].i;
      L[k].x0 = i >= 0 ? s.x0[i] : 0.f; L[k].x1 = i >= 0 ? s.x1[i] : 0.f;
      L[k].rz = (i >= 0 && L[k].par >= 0) ? s.rz[i] : 0.f;
      L[k].r0 = L[k].r1 = L[k].p0 = L[k].p1 = L[k].ap0 = L[k].ap1 = 0.f;
    }
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
      // ---- A (+ B for leaves): top-down ----
      float bb_part = 0.f, bz_part = 0.f;
      if (warp0) {
        for (int l = 0; l < ntop; l++) {
          if (L[0].lvl == l) down_bias(L[0], s, c, d, bb_part, bz_part);
          __syncwarp();
        }
      }
      if (ntop < nlev) {
        __syncthreads();
        for (int l = ntop; l < nlev; l++) {
#pragma unroll
          for (int k = 0; k < LPT; k++)
            if (L[k].lvl == l) down_bias(L[k], s, c, d, bb_part, bz_part);
          __syncthreads();
        }
      }
      // ---- B: bottom-up over the inner links ----
      for (int l = nlev - 2; l >= ntop; l--) {
#pragma unroll
        for (int k = 0; k < LPT; k++)
          if (L[k].lvl == l && L[k].nch) up_bias(L[k], s, c, d, bb_part, bz_part);
        __syncthreads();
      }
      if (warp0) {
        for (int l = min(ntop, nlev - 1) - 1; l >= 0; l--) {
          if (L[0].lvl == l && L[0].nch) up_bias(L[0], s, c, d, bb_part, bz_part);
          __syncwarp();
        }
      }
      const float2 bbz = red.sum(bb_part, bz_part);
      const float bb = bbz.x, bz = bbz.y;
      // ---- C: PCG, warm-started from the previous dqd (x) ----
      int it = 0;
      bool bad = false;
      if (bb == 0.f) {
#pragma unroll
        for (int k = 0; k < LPT; k++) { L[k].x0 = 0.f; L[k].x1 = 0.f; }
      } else if (!(bb < INFINITY)) {
        bad = true;
      } else {
#pragma unroll
        for (int k = 0; k < LPT; k++) { L[k].p0 = L[k].x0; L[k].p1 = L[k].x1; }   // first product: A x
        bool first = true;
        float rz = 0.f, rr = 0.f;
        // stopping rule: |r| <= tol |b| in the 2-norm (cg_norm 0) or in the preconditioned norm (cg_norm 1)
        const float tol2 = P.cg_tol * P.cg_tol * (P.cg_norm ? bz : bb);
        for (;;) {
          // ---- A p: top-down (leaves turn around at once), then bottom-up over the inner links ----
          float pAp_part = 0.f;
          if (warp0) {
            for (int l = 0; l < ntop; l++) {
              if (L[0].lvl == l) pAp_part += down_mv(L[0], s, c);
              __syncwarp();
            }
          }
          if (ntop < nlev) {
            __syncthreads();
            for (int l = ntop; l < nlev; l++) {
#pragma unroll
              for (int k = 0; k < LPT; k++)
                if (L[k].lvl == l) pAp_part += down_mv(L[k], s, c);
              __syncthreads();
            }
          }
          for (int l = nlev - 2; l >= ntop; l--) {
#pragma unroll
            for (int k = 0; k < LPT; k++)
              if (L[k].lvl == l && L[k].nch) pAp_part += up_mv(L[k], s, c);
            __syncthreads();
          }
          if (warp0) {
            for (int l = min(ntop, nlev - 1) - 1; l >= 0; l--) {
              if (L[0].lvl == l && L[0].nch) pAp_part += up_mv(L[0], s, c);
              __syncwarp();
            }
          }
          float rz_p = 0.f, rr_p = 0.f;
          if (first) {                                 // r = b - A x, z = P^-1 r, p = z
            first = false;
#pragma unroll
            for (int k = 0; k < LPT; k++) {
              const float ra = L[k].r0 - L[k].ap0, rb = L[k].r1 - L[k].ap1;
              const float za = ra * L[k].id0, zb = rb * L[k].id1;
              L[k].r0 = ra; L[k].r1 = rb; L[k].p0 = za; L[k].p1 = zb;
              rz_p += ra * za + rb * zb; rr_p += ra * ra + rb * rb;
            }
            const float2 t = red.sum(rz_p, rr_p);
            rz = t.x; rr = P.cg_norm ? t.x : t.y;
          } else {
            const float pAp = red.sum(pAp_part, 0.f).x;
            const float alpha = rz / pAp;
#pragma unroll
            for (int k = 0; k < LPT; k++) {
              L[k].x0 += alpha * L[k].p0; L[k].x1 += alpha * L[k].p1;
              const float ra = L[k].r0 - alpha * L[k].ap0, rb = L[k].r1 - alpha * L[k].ap1;
              L[k].r0 = ra; L[k].r1 = rb;
              rz_p += ra * ra * L[k].id0 + rb * rb * L[k].id1; rr_p += ra * ra + rb * rb;
            }
            const float2 t = red.sum(rz_p, rr_p);
            const float beta = t.x / rz;
            rz = t.x; rr = P.cg_norm ? t.x : t.y;
#pragma unroll
            for (int k = 0; k < LPT; k++) {
              L[k].p0 = L[k].r0 * L[k].id0 + beta * L[k].p0;
              L[k].p1 = L[k].r1 * L[k].id1 + beta * L[k].p1;
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
      for (int k = 0; k < LPT; k++) nf |= !(fabsf(L[k].x0) < INFINITY) || !(fabsf(L[k].x1) < INFINITY);
      if (__syncthreads_or(nf || bad)) { status |= OB_STATUS_NONFINITE; break; }

      // ---- D: integrate, predicates ----
      const int step_now = step0 + sidx;
#pragma unroll
      for (int k = 0; k < LPT; k++) {
        const int i = L[k].i;
        if (i < 0) continue;
        float wa = s.w0[i] + L[k].x0, wb = s.w1[i] + L[k].x1;
        if (P.qd_max > 0.f) {
          wa = fminf(fmaxf(wa, -P.qd_max), P.qd_max);
          wb = fminf(fmaxf(wb, -P.qd_max), P.qd_max);
        }
        const float qa = fmaf(P.h, wa, s.q0[i]), qb = fmaf(P.h, wb, s.q1[i]);
        s.w0[i] = wa; s.w1[i] = wb; s.q0[i] = qa; s.q1[i] = qb;
        if (!s.rupt[i]) {
          const float Ki = s.K[i], Mx = __ldg(c.Mmax + d.link_base + i);
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
    const bool frozen = (status & OB_STATUS_NONFINITE) != 0;
#pragma unroll
    for (int k = 0; k < LPT; k++)
      if (L[k].i >= 0) { s.x0[L[k].i] = frozen ? 0.f : L[k].x0; s.x1[L[k].i] = frozen ? 0.f : L[k].x1; }
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
      tma_store(c.link_blk + d.link_blk_off, s.q0, (uint32_t)link_state_bytes(d.Np));
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
    case 0: { CALL(256, 1, 3); break; }                 \
    case 1: { CALL(256, 2, 2); break; }                 \
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
