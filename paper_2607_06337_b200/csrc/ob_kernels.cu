// ob_kernels.cu -- sm_100a kernels of the batched tree-physics step.
//
//   k_rest_pose   rest world rotations R0 (fp64 -> fp32) and apple anchors (fp64), once per ob_create
//   k_randomize   Philox4x32-10 draws, derived constants, state reset (Eq. 4, Eq. 5)
//   k_step        the product: one CTA per world in flight (persistent, work queue), the world's state staged
//                 to shared memory by TMA bulk copies, n steps on chip:
//                   A  top-down sweep: joint transforms, displacement-form FK, velocities, bias accelerations,
//                      tether forces (Eq. 6/7), wrenches -> link forces
//                   B  bottom-up sweep: bias torques -> rhs b; composite inertia -> Jacobi diagonal
//                   C  matrix-free Jacobi-PCG on (M + M_teth + diag(arm + hD + h^2 K)) dqd = b,
//                      M*v = acceleration-only inverse dynamics (top-down a_i, bottom-up f_i, project on S_i)
//                   D  integrate joints and apples; rupture (Eq. 5) and detach predicates
//   k_pose        link poses for ob_get_state(link_pose7)
//
// Spatial vectors are [angular; linear at the link origin] in link coordinates.  Link frame: origin at the
// proximal joint, +z along the link.  Joint i: R_rel = Q_i Rx(theta1) Ry(theta2); E_i = R_rel^T maps parent
// coordinates to link coordinates; the joint sits at r = (0,0,L_parent) in the parent frame.
#include <math.h>

#include "ob_internal.h"

namespace ob {

// ------------------------------------------------------------------------------------------------------
// small vector algebra
// ------------------------------------------------------------------------------------------------------
struct M3 { float a[9]; };  // row-major

__device__ __forceinline__ float3 f3(float x, float y, float z) { return make_float3(x, y, z); }
__device__ __forceinline__ float3 operator+(float3 a, float3 b) { return f3(a.x + b.x, a.y + b.y, a.z + b.z); }
__device__ __forceinline__ float3 operator-(float3 a, float3 b) { return f3(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ float3 operator*(float s, float3 a) { return f3(s * a.x, s * a.y, s * a.z); }
__device__ __forceinline__ float3 cross(float3 a, float3 b) {
  return f3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
__device__ __forceinline__ float dot(float3 a, float3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
__device__ __forceinline__ float3 mul(const M3 &m, float3 v) {
  return f3(m.a[0] * v.x + m.a[1] * v.y + m.a[2] * v.z, m.a[3] * v.x + m.a[4] * v.y + m.a[5] * v.z,
            m.a[6] * v.x + m.a[7] * v.y + m.a[8] * v.z);
}
__device__ __forceinline__ float3 mulT(const M3 &m, float3 v) {
  return f3(m.a[0] * v.x + m.a[3] * v.y + m.a[6] * v.z, m.a[1] * v.x + m.a[4] * v.y + m.a[7] * v.z,
            m.a[2] * v.x + m.a[5] * v.y + m.a[8] * v.z);
}
__device__ __forceinline__ M3 mul(const M3 &A, const M3 &B) {
  M3 C;
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int c = 0; c < 3; c++)
      C.a[3 * r + c] = A.a[3 * r] * B.a[c] + A.a[3 * r + 1] * B.a[3 + c] + A.a[3 * r + 2] * B.a[6 + c];
  return C;
}
__device__ __forceinline__ M3 quat_to_mat(float4 q) {  // q = (w,x,y,z) stored as (x=w, y=x, z=y, w=z)
  float w = q.x, x = q.y, y = q.z, z = q.w;
  M3 R;
  R.a[0] = 1.f - 2.f * (y * y + z * z); R.a[1] = 2.f * (x * y - w * z);       R.a[2] = 2.f * (x * z + w * y);
  R.a[3] = 2.f * (x * y + w * z);       R.a[4] = 1.f - 2.f * (x * x + z * z); R.a[5] = 2.f * (y * z - w * x);
  R.a[6] = 2.f * (x * z - w * y);       R.a[7] = 2.f * (y * z + w * x);       R.a[8] = 1.f - 2.f * (x * x + y * y);
  return R;
}

// ------------------------------------------------------------------------------------------------------
// Philox4x32-10 (counter-based; PAPER.md:167-169 randomization, layout in include/orchard.h)
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; r++) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u;
    k.y += 0xBB67AE85u;
  }
  return c;
}
__device__ __forceinline__ float philox_uniform(uint32_t x, float lo, float hi) {
  float u = (float)(x >> 8) * (1.0f / 16777216.0f);
  return fmaf(u, hi - lo, lo);
}

// ------------------------------------------------------------------------------------------------------
// TMA bulk copies + mbarrier (1-D cp.async.bulk; SASS: UBLKCP)
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void tma_load(void *smem_dst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(smem_dst)),
               "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void tma_store(void *gdst, const void *smem_src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void tma_store_commit_wait() {
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ------------------------------------------------------------------------------------------------------
// k_rest_pose: one CTA per world.  R0_i = Q_0 ... Q_i and anchor_a = p0_b + R0_b o by walking up the
// ancestors in fp64 (create-time only; Eq. 3).
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void quat_to_mat_d(float4 q, double *R) {   // normalises in fp64
  double w = q.x, x = q.y, y = q.z, z = q.w;
  const double n = sqrt(w * w + x * x + y * y + z * z);
  w /= n; x /= n; y /= n; z /= n;
  R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z);     R[2] = 2 * (x * z + w * y);
  R[3] = 2 * (x * y + w * z);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
  R[6] = 2 * (x * z - w * y);     R[7] = 2 * (y * z + w * x);     R[8] = 1 - 2 * (x * x + y * y);
}

__global__ void k_rest_pose(DevCtx c) {
  const WorldDesc d = c.desc[blockIdx.x];
  const int4 *topo = c.topo + d.link_base;
  const float4 *quat = c.quat_raw + d.link_base;   // the caller's quaternions, normalised in fp64 here
  const float *Lown = c.Lown + d.link_base;
  for (int i = threadIdx.x; i < d.N; i += blockDim.x) {
    double R[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    for (int j = i; j >= 0; j = topo[j].x) {
      double Q[9], T[9];
      quat_to_mat_d(quat[j], Q);
      for (int r = 0; r < 3; r++)
        for (int cc = 0; cc < 3; cc++) T[3 * r + cc] = Q[3 * r] * R[cc] + Q[3 * r + 1] * R[3 + cc] + Q[3 * r + 2] * R[6 + cc];
      for (int k = 0; k < 9; k++) R[k] = T[k];
    }
    for (int k = 0; k < 9; k++) c.R0[9 * (size_t)d.link_base + (size_t)k * d.Np + i] = (float)R[k];
  }
  const unsigned char *ab = c.apple_blk + d.apple_blk_off;
  const float *ao = reinterpret_cast<const float *>(ab + apple_state_bytes(d.Ap));
  const int32_t *alink = reinterpret_cast<const int32_t *>(ab + apple_state_bytes(d.Ap) + 7 * 4 * d.Ap);
  for (int a = threadIdx.x; a < d.A; a += blockDim.x) {
    double x[3] = {ao[a], ao[d.Ap + a], ao[2 * d.Ap + a]};
    for (int j = alink[a]; j >= 0; j = topo[j].x) {
      double Q[9];
      quat_to_mat_d(quat[j], Q);
      double y0 = Q[0] * x[0] + Q[1] * x[1] + Q[2] * x[2];
      double y1 = Q[3] * x[0] + Q[4] * x[1] + Q[5] * x[2];
      double y2 = Q[6] * x[0] + Q[7] * x[1] + Q[8] * x[2];
      int pa = topo[j].x;
      x[0] = y0; x[1] = y1; x[2] = y2 + (pa >= 0 ? (double)Lown[pa] : 0.0);
    }
    for (int k = 0; k < 3; k++) c.anchor[3 * (size_t)d.apple_base + (size_t)k * d.Ap + a] = x[k];
  }
}

// ------------------------------------------------------------------------------------------------------
// k_randomize: one CTA per world.  redraw = 0 keeps the current material (used by ob_create).
// ------------------------------------------------------------------------------------------------------
__global__ void k_randomize(DevCtx c, unsigned long long seed, int redraw) {
  const int w = blockIdx.x;
  const WorldDesc d = c.desc[w];
  const ob_params &P = c.P;
  WorldInfo *info = c.info + w;
  const uint2 key = make_uint2((uint32_t)(seed & 0xffffffffull), (uint32_t)(seed >> 32));
  float E = d.E, MOR = d.MOR, rho = d.density;
  if (redraw) {
    uint4 o = philox4x32_10(make_uint4((uint32_t)w, 0u, 0u, 0u), key);
    if (P.range_E[0] != P.range_E[1]) E = philox_uniform(o.x, P.range_E[0], P.range_E[1]);
    if (P.range_MOR[0] != P.range_MOR[1]) MOR = philox_uniform(o.y, P.range_MOR[0], P.range_MOR[1]);
    if (P.range_density[0] != P.range_density[1]) rho = philox_uniform(o.z, P.range_density[0], P.range_density[1]);
  }
  unsigned char *lb = c.link_blk + d.link_blk_off;
  float *st = reinterpret_cast<float *>(lb);
  unsigned char *fl = lb + kLinkStateFloats * 4 * d.Np;
  float *cs = reinterpret_cast<float *>(lb + link_state_bytes(d.Np));
  const float *Lown = c.Lown + d.link_base, *diam = c.diam + d.link_base;
  const int4 *topo = c.topo + d.link_base;
  const double PI = 3.14159265358979323846;
  for (int i = threadIdx.x; i < d.Np; i += blockDim.x) {
    for (int k = 0; k < kLinkStateFloats; k++) st[k * d.Np + i] = 0.f;
    fl[i] = 0; fl[d.Np + i] = 0;
    if (i < d.N) {
      double dd = diam[i], L = Lown[i], r = 0.5 * dd;
      double K = (double)E * PI * dd * dd * dd * dd / (64.0 * L);   // Eq. 4
      double Mx = (double)MOR * PI * dd * dd * dd / 32.0;           // Eq. 5
      double m = (double)rho * PI * r * r * L;                      // solid cylinder
      double Ic = m * (3.0 * r * r + L * L) / 12.0, cz = 0.5 * L;
      int pa = topo[i].x;
      cs[0 * d.Np + i] = (float)K;
      cs[1 * d.Np + i] = (float)m;
      cs[2 * d.Np + i] = (float)(m * cz);
      cs[3 * d.Np + i] = (float)(Ic + m * cz * cz);                  // about the joint
      cs[4 * d.Np + i] = (float)(0.5 * m * r * r);
      cs[5 * d.Np + i] = pa >= 0 ? Lown[pa] : 0.f;
      c.Mmax[d.link_base + i] = (float)Mx;
    } else {
      for (int k = 0; k < kLinkConstFloats; k++) cs[k * d.Np + i] = 0.f;
    }
  }
  unsigned char *ab = c.apple_blk + d.apple_blk_off;
  float *as = reinterpret_cast<float *>(ab);
  unsigned char *af = ab + 6 * 4 * d.Ap;
  float *ac = reinterpret_cast<float *>(ab + apple_state_bytes(d.Ap));   // o[3] k m c fdet
  const float *nom = c.apple_nominal + 2 * (size_t)d.apple_base;
  const int32_t *aext = c.apple_ext + d.apple_base;
  for (int a = threadIdx.x; a < d.Ap; a += blockDim.x) {
    for (int k = 0; k < 6; k++) as[k * d.Ap + a] = 0.f;
    af[a] = a < d.A ? 1 : 0; af[d.Ap + a] = 0; af[2 * d.Ap + a] = 0;
    if (a < d.A) {
      float m, fd;
      if (redraw) {
        // the counter item is the CALLER's apple index (the internal order is a private matter)
        uint4 o = philox4x32_10(make_uint4((uint32_t)w, (uint32_t)aext[a], 1u, 0u), key);
        fd = P.range_detach[0] != P.range_detach[1] ? philox_uniform(o.x, P.range_detach[0], P.range_detach[1])
                                                    : nom[d.Ap + a];
        m = P.range_apple_mass[0] != P.range_apple_mass[1]
                ? philox_uniform(o.y, P.range_apple_mass[0], P.range_apple_mass[1]) : nom[a];
      } else {
        m = ac[4 * d.Ap + a]; fd = ac[6 * d.Ap + a];
      }
      float k = ac[3 * d.Ap + a];
      ac[4 * d.Ap + a] = m;
      ac[5 * d.Ap + a] = d.has_apple_c ? c.apple_c_in[d.apple_base + a]
                                        : (float)(2.0 * (double)P.zeta_s * sqrt((double)k * (double)m));
      ac[6 * d.Ap + a] = fd;
      // u = x - (anchor + m g / k_s) stays 0: the apple starts at its rest sag
    }
  }
  if (threadIdx.x == 0) {
    info->step = 0; info->last_iters = 0; info->status = 0;
    info->E = E; info->MOR = MOR; info->density = rho;
  }
}

// ------------------------------------------------------------------------------------------------------
// k_step
// ------------------------------------------------------------------------------------------------------
struct Sm {            // shared-memory view of one world
  int N, A, Np, Ap, nlev;
  // link block (TMA)
  float *q0, *q1, *w0, *w1, *x0, *x1;
  unsigned char *rupt, *rc;
  float *K, *m, *mc, *Io, *Iz, *rz;
  // apple block (TMA)
  float *u, *v;                       // [3][Ap]
  unsigned char *att, *cA, *cB;
  float *ao, *ak, *am, *ac, *afd;     // ao = [3][Ap]
  int32_t *alink;
  // per-step arrays
  float *E;                           // [9][Np]
  float *c2, *s2;
  float *mb;                          // [6][Np] parent<->child mailbox (acceleration down, force up)
  float *scr;                         // [24][Np]; scr[0..7] alias invd, r, p, Ap
  float *invd0, *invd1, *r0, *r1, *p0, *p1, *Ap0, *Ap1;
  unsigned char *snapped;
  float *ft, *fu, *fsn, *fun;         // tether force [3][Ap], user force [3][Ap], |f_s|, |f_user|
  int32_t *lev;
  WrenchSlots *wr;
};

__device__ __forceinline__ Sm carve(unsigned char *base, const WorldDesc &d) {
  Sm s;
  s.N = d.N; s.A = d.A; s.Np = d.Np; s.Ap = d.Ap; s.nlev = d.n_levels;
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
  s.alink = reinterpret_cast<int32_t *>(f + 7 * Ap);
  p += apple_block_bytes(Ap);
  f = reinterpret_cast<float *>(p);
  s.E = f; f += 9 * Np;
  s.c2 = f; f += Np;
  s.s2 = f; f += Np;
  s.mb = f; f += 6 * Np;
  s.scr = f; f += 24 * Np;
  s.invd0 = s.scr; s.invd1 = s.scr + Np; s.r0 = s.scr + 2 * Np; s.r1 = s.scr + 3 * Np;
  s.p0 = s.scr + 4 * Np; s.p1 = s.scr + 5 * Np; s.Ap0 = s.scr + 6 * Np; s.Ap1 = s.scr + 7 * Np;
  s.ft = f; f += 3 * Ap;
  s.fu = f; f += 3 * Ap;
  s.fsn = f; f += Ap;
  s.fun = f; f += Ap;
  s.lev = reinterpret_cast<int32_t *>(f); f += (d.n_levels + 1 + 3) / 4 * 4;
  s.wr = reinterpret_cast<WrenchSlots *>(f); f += sizeof(WrenchSlots) / 4;
  s.snapped = reinterpret_cast<unsigned char *>(f);
  return s;
}

// block-wide sum of two values, result broadcast to every thread; one barrier per call (double-buffered stage)
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
    const int nw = (blockDim.x + 31) >> 5;
    float sa = 0.f, sb = 0.f;
    for (int k = 0; k < nw; k++) { float2 t = st[k]; sa += t.x; sb += t.y; }
    return make_float2(sa, sb);
  }
};

// -------- phase A: one link of the top-down sweep ------------------------------------------------------
__device__ __forceinline__ void link_topdown_bias(const Sm &s, const DevCtx &c, const WorldDesc &d, int i) {
  const int Np = s.Np, Ap = s.Ap;
  const ob_params &P = c.P;
  const int4 tp = __ldg(c.topo + d.link_base + i);
  const int par = tp.x, nch = tp.z & 0xffff, nap = tp.z >> 16, ast = tp.w;
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
  for (int k = 0; k < 9; k++) s.E[k * Np + i] = E.a[k];
  s.c2[i] = c2; s.s2[i] = s2;

  // parent quantities (world = parent of the trunk: at rest, spatial acceleration (0; -g))
  M3 dRp;
  float3 dpp = f3(0, 0, 0), wp = f3(0, 0, 0), vp = f3(0, 0, 0), alp = f3(0, 0, 0);
  float3 ap = f3(-P.gravity[0], -P.gravity[1], -P.gravity[2]);
  unsigned char snapped_p = 0;
  float rz = 0.f;
#pragma unroll
  for (int k = 0; k < 9; k++) dRp.a[k] = 0.f;
  if (par >= 0) {
    const float *sc = s.scr + par;
#pragma unroll
    for (int k = 0; k < 9; k++) dRp.a[k] = sc[k * Np];
    dpp = f3(sc[9 * Np], sc[10 * Np], sc[11 * Np]);
    wp = f3(sc[12 * Np], sc[13 * Np], sc[14 * Np]);
    vp = f3(sc[15 * Np], sc[16 * Np], sc[17 * Np]);
    alp = f3(sc[18 * Np], sc[19 * Np], sc[20 * Np]);
    ap = f3(sc[21 * Np], sc[22 * Np], sc[23 * Np]);
    snapped_p = s.snapped[par];
    rz = s.rz[i];
  }
  // displacement-form FK: R_i = R0_i + dR_i,  dR_i = dR_p Rrel + R0_i (RxRy - I);  dp_i = dp_p + dR_p (0,0,rz)
  M3 R0, G = XY;
  const float *R0g = c.R0 + 9 * (size_t)d.link_base + i;
#pragma unroll
  for (int k = 0; k < 9; k++) R0.a[k] = __ldg(R0g + (size_t)k * Np);
  G.a[0] = vc2; G.a[4] = vc1; G.a[8] = fmaf(vc1, vc2, vc1 + vc2);
  const M3 t1 = mul(dRp, Rrel), t2 = mul(R0, G);
  M3 dR, R;
#pragma unroll
  for (int k = 0; k < 9; k++) { dR.a[k] = t1.a[k] + t2.a[k]; R.a[k] = R0.a[k] + dR.a[k]; }
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
  for (int a = ast; a < ast + nap; a++) {
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
  float *mb = s.mb + i;
  mb[0] = n.x; mb[Np] = n.y; mb[2 * Np] = n.z; mb[3 * Np] = f.x; mb[4 * Np] = f.y; mb[5 * Np] = f.z;
  if (nch) {
    float *sc = s.scr + i;
#pragma unroll
    for (int k = 0; k < 9; k++) sc[k * Np] = dR.a[k];
    sc[9 * Np] = dp.x; sc[10 * Np] = dp.y; sc[11 * Np] = dp.z;
    sc[12 * Np] = om.x; sc[13 * Np] = om.y; sc[14 * Np] = om.z;
    sc[15 * Np] = vl.x; sc[16 * Np] = vl.y; sc[17 * Np] = vl.z;
    sc[18 * Np] = al.x; sc[19 * Np] = al.y; sc[20 * Np] = al.z;
    sc[21 * Np] = aln.x; sc[22 * Np] = aln.y; sc[23 * Np] = aln.z;
  }
}

// -------- phase B: bottom-up: bias torque -> b (stored in r), composite inertia -> Jacobi diagonal --------
__device__ __forceinline__ float dterm(const Sm &s, const DevCtx &c, const WorldDesc &d, int i, int k) {
  const float Kt = s.rupt[i] ? 0.f : s.K[i];
  float t = (c.P.h * c.P.c_d + c.P.h * c.P.h) * Kt;
  if (c.arm) t += __ldg(c.arm + 2 * (size_t)d.link_base + (size_t)k * s.Np + i);
  return t;
}

__device__ __forceinline__ void link_bottomup_bias(const Sm &s, const DevCtx &c, const WorldDesc &d, int i,
                                                   float &bb) {
  const int Np = s.Np, Ap = s.Ap;
  const ob_params &P = c.P;
  const int4 tp = __ldg(c.topo + d.link_base + i);
  const int par = tp.x, cst = tp.y, nch = tp.z & 0xffff, nap = tp.z >> 16, ast = tp.w;
  float *mb = s.mb + i;
  float3 n = f3(mb[0], mb[Np], mb[2 * Np]), f = f3(mb[3 * Np], mb[4 * Np], mb[5 * Np]);
  // composite rigid-body inertia about the link origin: mass, first moment h, symmetric I (xx,yy,zz,xy,xz,yz)
  float cm = s.m[i];
  float3 ch = f3(0.f, 0.f, s.mc[i]);
  float Ixx = s.Io[i], Iyy = s.Io[i], Izz = s.Iz[i], Ixy = 0.f, Ixz = 0.f, Iyz = 0.f;
  if (P.tether_implicit) {
    for (int a = ast; a < ast + nap; a++) {
      if (!s.att[a]) continue;
      const float mv = P.h * P.h * s.ak[a];                     // virtual point mass h^2 k_s at the hang point
      const float3 o = f3(s.ao[a], s.ao[Ap + a], s.ao[2 * Ap + a]);
      cm += mv; ch = ch + mv * o;
      Ixx += mv * (o.y * o.y + o.z * o.z); Iyy += mv * (o.x * o.x + o.z * o.z); Izz += mv * (o.x * o.x + o.y * o.y);
      Ixy -= mv * o.x * o.y; Ixz -= mv * o.x * o.z; Iyz -= mv * o.y * o.z;
    }
  }
  for (int ch_i = cst; ch_i < cst + nch; ch_i++) {
    const float *cb = s.mb + ch_i;
    n = n + f3(cb[0], cb[Np], cb[2 * Np]);
    f = f + f3(cb[3 * Np], cb[4 * Np], cb[5 * Np]);
    const float *cc = s.scr + 8 * Np + ch_i;
    cm += cc[0];
    ch = ch + f3(cc[Np], cc[2 * Np], cc[3 * Np]);
    Ixx += cc[4 * Np]; Iyy += cc[5 * Np]; Izz += cc[6 * Np]; Ixy += cc[7 * Np]; Ixz += cc[8 * Np]; Iyz += cc[9 * Np];
  }
  const float c2 = s.c2[i], s2 = s.s2[i];
  const float tau1 = c2 * n.x + s2 * n.z, tau2 = n.y;
  const float Kt = s.rupt[i] ? 0.f : s.K[i], Dt = P.c_d * Kt;
  const float b1 = P.h * (-tau1 - Kt * s.q0[i] - (Dt + P.h * Kt) * s.w0[i]);
  const float b2 = P.h * (-tau2 - Kt * s.q1[i] - (Dt + P.h * Kt) * s.w1[i]);
  s.r0[i] = b1; s.r1[i] = b2;
  bb += b1 * b1 + b2 * b2;
  const float d1 = c2 * c2 * Ixx + 2.f * c2 * s2 * Ixz + s2 * s2 * Izz + dterm(s, c, d, i, 0);
  const float d2 = Iyy + dterm(s, c, d, i, 1);
  if (P.precond == 1) { s.invd0[i] = 1.f / d1; s.invd1[i] = 1.f / d2; }
  else { s.invd0[i] = 1.f; s.invd1[i] = 1.f; }
  if (par >= 0) {
    M3 E;
#pragma unroll
    for (int k = 0; k < 9; k++) E.a[k] = s.E[k * Np + i];
    const float rz = s.rz[i];
    const float3 fp = mulT(E, f);
    float3 np = mulT(E, n);
    np.x -= rz * fp.y; np.y += rz * fp.x;
    mb[0] = np.x; mb[Np] = np.y; mb[2 * Np] = np.z; mb[3 * Np] = fp.x; mb[4 * Np] = fp.y; mb[5 * Np] = fp.z;
    // composite inertia into the parent frame: rotate by Rrel = E^T, then move the origin by r = (0,0,rz)
    const float3 hp = mulT(E, ch);
    M3 I, T, Ip;
    I.a[0] = Ixx; I.a[1] = Ixy; I.a[2] = Ixz; I.a[3] = Ixy; I.a[4] = Iyy; I.a[5] = Iyz; I.a[6] = Ixz; I.a[7] = Iyz; I.a[8] = Izz;
    // T = E^T I ; Ip = T E
#pragma unroll
    for (int r = 0; r < 3; r++)
#pragma unroll
      for (int cc = 0; cc < 3; cc++) T.a[3 * r + cc] = E.a[r] * I.a[cc] + E.a[3 + r] * I.a[3 + cc] + E.a[6 + r] * I.a[6 + cc];
    Ip = mul(T, E);
    const float sh = 2.f * rz * hp.z + cm * rz * rz;
    float *cc = s.scr + 8 * Np + i;
    cc[0] = cm;
    cc[Np] = hp.x; cc[2 * Np] = hp.y; cc[3 * Np] = hp.z + cm * rz;
    cc[4 * Np] = Ip.a[0] + sh; cc[5 * Np] = Ip.a[4] + sh; cc[6 * Np] = Ip.a[8];
    cc[7 * Np] = Ip.a[1]; cc[8 * Np] = Ip.a[2] - rz * hp.x; cc[9 * Np] = Ip.a[5] - rz * hp.y;
  }
}

// -------- phase C: A*v.  top-down accelerations, bottom-up forces, projection ---------------------------
__device__ __forceinline__ void link_topdown_mv(const Sm &s, const DevCtx &c, const WorldDesc &d, int i,
                                                const float *v0, const float *v1) {
  const int Np = s.Np;
  const int par = __ldg(c.topo + d.link_base + i).x;
  float3 al = f3(0, 0, 0), a = f3(0, 0, 0);
  if (par >= 0) {
    const float *pb = s.mb + par;
    const float3 alp = f3(pb[0], pb[Np], pb[2 * Np]), ap = f3(pb[3 * Np], pb[4 * Np], pb[5 * Np]);
    const float rz = s.rz[i];
    M3 E;
#pragma unroll
    for (int k = 0; k < 9; k++) E.a[k] = s.E[k * Np + i];
    al = mul(E, alp);
    a = mul(E, f3(ap.x + alp.y * rz, ap.y - alp.x * rz, ap.z));
  }
  const float c2 = s.c2[i], s2 = s.s2[i], x0 = v0[i], x1 = v1[i];
  al = al + f3(c2 * x0, x1, s2 * x0);
  float *mb = s.mb + i;
  mb[0] = al.x; mb[Np] = al.y; mb[2 * Np] = al.z; mb[3 * Np] = a.x; mb[4 * Np] = a.y; mb[5 * Np] = a.z;
}

__device__ __forceinline__ void link_bottomup_mv(const Sm &s, const DevCtx &c, const WorldDesc &d, int i,
                                                 const float *v0, const float *v1, float &vAv) {
  const int Np = s.Np, Ap = s.Ap;
  const ob_params &P = c.P;
  const int4 tp = __ldg(c.topo + d.link_base + i);
  const int par = tp.x, cst = tp.y, nch = tp.z & 0xffff, nap = tp.z >> 16, ast = tp.w;
  float *mb = s.mb + i;
  const float3 al = f3(mb[0], mb[Np], mb[2 * Np]), a = f3(mb[3 * Np], mb[4 * Np], mb[5 * Np]);
  const float m = s.m[i], mc = s.mc[i], Io = s.Io[i], Iz = s.Iz[i];
  float3 n = f3(Io * al.x - mc * a.y, Io * al.y + mc * a.x, Iz * al.z);
  float3 f = f3(m * a.x + mc * al.y, m * a.y - mc * al.x, m * a.z);
  if (P.tether_implicit) {
    for (int q = ast; q < ast + nap; q++) {
      if (!s.att[q]) continue;
      const float mv = P.h * P.h * s.ak[q];
      const float3 o = f3(s.ao[q], s.ao[Ap + q], s.ao[2 * Ap + q]);
      const float3 fp = mv * (a + cross(al, o));
      f = f + fp;
      n = n + cross(o, fp);
    }
  }
  for (int ch = cst; ch < cst + nch; ch++) {
    const float *cb = s.mb + ch;
    n = n + f3(cb[0], cb[Np], cb[2 * Np]);
    f = f + f3(cb[3 * Np], cb[4 * Np], cb[5 * Np]);
  }
  const float c2 = s.c2[i], s2 = s.s2[i], x0 = v0[i], x1 = v1[i];
  const float t1 = c2 * n.x + s2 * n.z + dterm(s, c, d, i, 0) * x0;
  const float t2 = n.y + dterm(s, c, d, i, 1) * x1;
  s.Ap0[i] = t1; s.Ap1[i] = t2;
  vAv += x0 * t1 + x1 * t2;
  if (par >= 0) {
    M3 E;
#pragma unroll
    for (int k = 0; k < 9; k++) E.a[k] = s.E[k * Np + i];
    const float rz = s.rz[i];
    const float3 fp = mulT(E, f);
    float3 np = mulT(E, n);
    np.x -= rz * fp.y; np.y += rz * fp.x;
    mb[0] = np.x; mb[Np] = np.y; mb[2 * Np] = np.z; mb[3 * Np] = fp.x; mb[4 * Np] = fp.y; mb[5 * Np] = fp.z;
  }
}

__device__ __forceinline__ float matvec(const Sm &s, const DevCtx &c, const WorldDesc &d, const float *v0,
                                        const float *v1) {
  const int tid = threadIdx.x, nthr = blockDim.x;
  for (int l = 0; l < s.nlev; l++) {
    const int e = s.lev[l + 1];
    for (int i = s.lev[l] + tid; i < e; i += nthr) link_topdown_mv(s, c, d, i, v0, v1);
    __syncthreads();
  }
  float vAv = 0.f;
  for (int l = s.nlev - 1; l >= 0; l--) {
    const int e = s.lev[l + 1];
    for (int i = s.lev[l] + tid; i < e; i += nthr) link_bottomup_mv(s, c, d, i, v0, v1, vAv);
    __syncthreads();
  }
  return vAv;
}

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

__global__ void __launch_bounds__(256, 2) k_step(DevCtx c, int n_steps) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ __align__(8) uint64_t s_bar;
  __shared__ int s_next;
  __shared__ float2 s_stage[64];
  const int tid = threadIdx.x, nthr = blockDim.x;
  const ob_params &P = c.P;
  uint32_t parity = 0;
  if (tid == 0) mbar_init(&s_bar, 1);
  __syncthreads();
  Reducer red;
  red.stage = s_stage;
  red.flip = 0;

  for (;;) {
    if (tid == 0) s_next = atomicAdd(c.queue, 1);
    __syncthreads();
    const int qi = s_next;
    __syncthreads();
    if (qi >= c.n_worlds) break;
    const int w = c.order[qi];
    const WorldDesc d = c.desc[w];
    WorldInfo *info = c.info + w;
    int status = info->status;
    if (status & OB_STATUS_NONFINITE) continue;      // frozen world
    const Sm s = carve(smem, d);

    // ---- stage the world: two TMA bulk copies (link block, apple block) onto one mbarrier ----
    if (tid == 0) {
      fence_proxy_async();
      const uint32_t lb = (uint32_t)link_block_bytes(d.Np), ab = (uint32_t)apple_block_bytes(d.Ap);
      mbar_expect_tx(&s_bar, lb + ab);
      tma_load(s.q0, c.link_blk + d.link_blk_off, lb, &s_bar);
      if (ab) tma_load(s.u, c.apple_blk + d.apple_blk_off, ab, &s_bar);
    }
    for (int l = tid; l <= d.n_levels; l += nthr) s.lev[l] = __ldg(c.level_off + d.level_base + l);
    {
      const int32_t *src = reinterpret_cast<const int32_t *>(c.wrench + w);
      int32_t *dst = reinterpret_cast<int32_t *>(s.wr);
      for (int k = tid; k < (int)(sizeof(WrenchSlots) / 4); k += nthr) dst[k] = __ldg(src + k);
    }
    mbar_wait(&s_bar, parity);
    parity ^= 1;
    __syncthreads();
    // user forces on apples are constant over the launch
    for (int a = tid; a < d.A; a += nthr) {
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
      // ---- A: top-down ----
      for (int l = 0; l < s.nlev; l++) {
        const int e = s.lev[l + 1];
        for (int i = s.lev[l] + tid; i < e; i += nthr) link_topdown_bias(s, c, d, i);
        __syncthreads();
      }
      // ---- B: bottom-up ----
      float bb_part = 0.f;
      for (int l = s.nlev - 1; l >= 0; l--) {
        const int e = s.lev[l + 1];
        for (int i = s.lev[l] + tid; i < e; i += nthr) link_bottomup_bias(s, c, d, i, bb_part);
        __syncthreads();
      }
      float bz_part = 0.f;
      for (int i = tid; i < d.N; i += nthr)
        bz_part += s.r0[i] * s.r0[i] * s.invd0[i] + s.r1[i] * s.r1[i] * s.invd1[i];
      const float2 bbz = red.sum(bb_part, bz_part);
      const float bb = bbz.x, bz = bbz.y;
      // ---- C: PCG, warm-started from the previous dqd (x) ----
      int it = 0;
      bool bad = false;
      if (bb == 0.f) {
        for (int i = tid; i < d.N; i += nthr) { s.x0[i] = 0.f; s.x1[i] = 0.f; }
      } else if (!(bb < INFINITY)) {
        bad = true;
      } else {
        matvec(s, c, d, s.x0, s.x1);
        float rz_p = 0.f, rr_p = 0.f;
        for (int i = tid; i < d.N; i += nthr) {
          const float ra = s.r0[i] - s.Ap0[i], rb = s.r1[i] - s.Ap1[i];
          const float za = ra * s.invd0[i], zb = rb * s.invd1[i];
          s.r0[i] = ra; s.r1[i] = rb; s.p0[i] = za; s.p1[i] = zb;
          rz_p += ra * za + rb * zb; rr_p += ra * ra + rb * rb;
        }
        float2 t = red.sum(rz_p, rr_p);
        float rz = t.x;
        // stopping rule: |r| <= tol |b| in the 2-norm (cg_norm 0) or in the preconditioned norm (cg_norm 1)
        float rr = P.cg_norm ? rz : t.y;
        const float tol2 = P.cg_tol * P.cg_tol * (P.cg_norm ? bz : bb);
        while (rr > tol2 && it < P.cg_max_iter) {
          const float pAp = red.sum(matvec(s, c, d, s.p0, s.p1), 0.f).x;
          const float alpha = rz / pAp;
          rz_p = 0.f; rr_p = 0.f;
          for (int i = tid; i < d.N; i += nthr) {
            s.x0[i] += alpha * s.p0[i]; s.x1[i] += alpha * s.p1[i];
            const float ra = s.r0[i] - alpha * s.Ap0[i], rb = s.r1[i] - alpha * s.Ap1[i];
            s.r0[i] = ra; s.r1[i] = rb;
            rz_p += ra * ra * s.invd0[i] + rb * rb * s.invd1[i]; rr_p += ra * ra + rb * rb;
          }
          t = red.sum(rz_p, rr_p);
          const float beta = t.x / rz;
          rz = t.x; rr = P.cg_norm ? t.x : t.y;
          for (int i = tid; i < d.N; i += nthr) {
            s.p0[i] = s.r0[i] * s.invd0[i] + beta * s.p0[i];
            s.p1[i] = s.r1[i] * s.invd1[i] + beta * s.p1[i];
          }
          it++;
          // the next matvec's first barrier orders these p writes before any cross-thread read
          __syncthreads();
        }
        if (!(rr <= tol2)) {
          if (rr == rr && rr < INFINITY) status |= OB_STATUS_CG_MAXITER;
          else bad = true;
        }
      }
      // a non-finite solve freezes the world at its last finite state
      int nf = 0;
      for (int i = tid; i < d.N; i += nthr) nf |= !(fabsf(s.x0[i]) < INFINITY) || !(fabsf(s.x1[i]) < INFINITY);
      if (__syncthreads_or(nf || bad)) { status |= OB_STATUS_NONFINITE; break; }

      // ---- D: integrate, predicates ----
      const int step_now = step0 + sidx;
      for (int i = tid; i < d.N; i += nthr) {
        float wa = s.w0[i] + s.x0[i], wb = s.w1[i] + s.x1[i];
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
      for (int a = tid; a < d.A; a += nthr) {
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
// k_pose: link frames of one world (position + quaternion), fp64 ancestor walk from the stored state
// ------------------------------------------------------------------------------------------------------
__global__ void k_pose(DevCtx c, int w) {
  const WorldDesc d = c.desc[w];
  const int4 *topo = c.topo + d.link_base;
  const float4 *quat = c.quat_raw + d.link_base;
  const float *Lown = c.Lown + d.link_base;
  const float *st = reinterpret_cast<const float *>(c.link_blk + d.link_blk_off);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < d.N; i += gridDim.x * blockDim.x) {
    double R[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1}, x[3] = {0, 0, 0};
    for (int j = i; j >= 0; j = topo[j].x) {
      double Q[9], T[9], A[9];
      quat_to_mat_d(quat[j], Q);
      double s1, c1, s2, c2;
      sincos((double)st[j], &s1, &c1);
      sincos((double)st[d.Np + j], &s2, &c2);
      const double XY[9] = {c2, 0, s2, s1 * s2, c1, -s1 * c2, -c1 * s2, s1, c1 * c2};
      for (int r = 0; r < 3; r++)
        for (int cc = 0; cc < 3; cc++) A[3 * r + cc] = Q[3 * r] * XY[cc] + Q[3 * r + 1] * XY[3 + cc] + Q[3 * r + 2] * XY[6 + cc];
      for (int r = 0; r < 3; r++)
        for (int cc = 0; cc < 3; cc++) T[3 * r + cc] = A[3 * r] * R[cc] + A[3 * r + 1] * R[3 + cc] + A[3 * r + 2] * R[6 + cc];
      for (int k = 0; k < 9; k++) R[k] = T[k];
      const double y0 = A[0] * x[0] + A[1] * x[1] + A[2] * x[2];
      const double y1 = A[3] * x[0] + A[4] * x[1] + A[5] * x[2];
      const double y2 = A[6] * x[0] + A[7] * x[1] + A[8] * x[2];
      const int pa = topo[j].x;
      x[0] = y0; x[1] = y1; x[2] = y2 + (pa >= 0 ? (double)Lown[pa] : 0.0);
    }
    // rotation matrix -> quaternion (w,x,y,z)
    double qw, qx, qy, qz;
    const double tr = R[0] + R[4] + R[8];
    if (tr > 0) {
      double S = sqrt(tr + 1.0) * 2; qw = 0.25 * S; qx = (R[7] - R[5]) / S; qy = (R[2] - R[6]) / S; qz = (R[3] - R[1]) / S;
    } else if (R[0] > R[4] && R[0] > R[8]) {
      double S = sqrt(1.0 + R[0] - R[4] - R[8]) * 2; qw = (R[7] - R[5]) / S; qx = 0.25 * S; qy = (R[1] + R[3]) / S; qz = (R[2] + R[6]) / S;
    } else if (R[4] > R[8]) {
      double S = sqrt(1.0 + R[4] - R[0] - R[8]) * 2; qw = (R[2] - R[6]) / S; qx = (R[1] + R[3]) / S; qy = 0.25 * S; qz = (R[5] + R[7]) / S;
    } else {
      double S = sqrt(1.0 + R[8] - R[0] - R[4]) * 2; qw = (R[3] - R[1]) / S; qx = (R[2] + R[6]) / S; qy = (R[5] + R[7]) / S; qz = 0.25 * S;
    }
    float *o = c.pose7 + 7 * i;
    o[0] = (float)x[0]; o[1] = (float)x[1]; o[2] = (float)x[2];
    o[3] = (float)qw; o[4] = (float)qx; o[5] = (float)qy; o[6] = (float)qz;
  }
}

// ------------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------------
cudaError_t launch_rest_pose(const DevCtx &c, int, int, cudaStream_t s) {
  k_rest_pose<<<c.n_worlds, 128, 0, s>>>(c);
  return cudaGetLastError();
}
cudaError_t launch_randomize(const DevCtx &c, unsigned long long seed, int redraw, cudaStream_t s) {
  k_randomize<<<c.n_worlds, 128, 0, s>>>(c, seed, redraw);
  return cudaGetLastError();
}
cudaError_t step_kernel_setup(int smem_bytes, int block, int *max_blocks_per_sm) {
  cudaError_t e = cudaFuncSetAttribute(k_step, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(max_blocks_per_sm, k_step, block, smem_bytes);
}
cudaError_t launch_step(const DevCtx &c, int n_steps, int grid, int block, int smem, cudaStream_t s) {
  k_step<<<grid, block, smem, s>>>(c, n_steps);
  return cudaGetLastError();
}
cudaError_t launch_pose(const DevCtx &c, int world, cudaStream_t s) {
  k_pose<<<4, 128, 0, s>>>(c, world);
  return cudaGetLastError();
}

}  // namespace ob
