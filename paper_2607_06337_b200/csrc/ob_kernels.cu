// ob_kernels.cu -- the small sm_100a kernels around the batched tree-physics step.
//
//   k_rest_pose   rest world rotations R0 (fp64 -> fp32) and apple anchors (fp64), once per ob_create
//   k_randomize   Philox4x32-10 draws, derived constants, state reset (Eq. 4, Eq. 5)
//   (k_step, the product, lives in ob_step.cu)
//   k_pose        link poses for ob_get_state(link_pose7)
//
// Spatial vectors are [angular; linear at the link origin] in link coordinates.  Link frame: origin at the
// proximal joint, +z along the link.  Joint i: R_rel = Q_i Rx(theta1) Ry(theta2); E_i = R_rel^T maps parent
// coordinates to link coordinates; the joint sits at r = (0,0,L_parent) in the parent frame.
#include <math.h>

#include <mutex>

#include "ob_device.h"
#include "ob_internal.h"

#include <curand_philox4x32_x.h>

namespace ob {

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
// k_rest_pose: one CTA per world.  The rest quaternion of every link normalised in fp64 (the FK of k_step starts from
// it); once per ob_create.  k_anchors: anchor_a = p0_b + R0_b o of every apple by walking up the ancestors in fp64 with
// the CURRENT rest quaternions, lengths and attach points (Eq. 3); after ob_create and after
// ob_randomize_geometry.
// ------------------------------------------------------------------------------------------------------
struct Qd4 { double w, x, y, z; };
__device__ __forceinline__ Qd4 qmul4(const Qd4 a, const Qd4 b) {
  Qd4 r;
  r.w = a.w * b.w - a.x * b.x - a.y * b.y - a.z * b.z;
  r.x = a.w * b.x + a.x * b.w + a.y * b.z - a.z * b.y;
  r.y = a.w * b.y - a.x * b.z + a.y * b.w + a.z * b.x;
  r.z = a.w * b.z + a.x * b.y - a.y * b.x + a.z * b.w;
  return r;
}
__device__ __forceinline__ void qrot4(const Qd4 q, const double v[3], double out[3]) {   // R(q) v
  const double tx = 2 * (q.y * v[2] - q.z * v[1]), ty = 2 * (q.z * v[0] - q.x * v[2]), tz = 2 * (q.x * v[1] - q.y * v[0]);
  out[0] = v[0] + q.w * tx + (q.y * tz - q.z * ty);
  out[1] = v[1] + q.w * ty + (q.z * tx - q.x * tz);
  out[2] = v[2] + q.w * tz + (q.x * ty - q.y * tx);
}
__device__ __forceinline__ Qd4 load_q4(const double *quatd, size_t i) {
  Qd4 q;
  q.w = quatd[4 * i]; q.x = quatd[4 * i + 1]; q.y = quatd[4 * i + 2]; q.z = quatd[4 * i + 3];
  return q;
}

__global__ void k_rest_pose(DevCtx c) {
  const WorldDesc d = c.desc[blockIdx.x];
  const float4 *quat = c.quat_raw + d.link_base;   // the caller's quaternions, normalised in fp64 here
  for (int i = threadIdx.x; i < d.N; i += blockDim.x) {
    const float4 q = quat[i];
    const double w = q.x, x = q.y, y = q.z, z = q.w, n = sqrt(w * w + x * x + y * y + z * z);
    double *qd = c.quatd + 4 * ((size_t)d.link_base + i);
    qd[0] = w / n; qd[1] = x / n; qd[2] = y / n; qd[3] = z / n;
  }
}

__global__ void k_anchors(DevCtx c) {
  const WorldDesc d = c.desc[blockIdx.x];
  const int4 *topo = c.topo + d.link_base;
  const float *Lown = c.Lown + d.link_base;
  const unsigned char *ab = c.apple_blk + d.apple_blk_off;
  const float *ao = reinterpret_cast<const float *>(ab + apple_state_bytes(d.Ap));
  const int32_t *alink = reinterpret_cast<const int32_t *>(ab + apple_state_bytes(d.Ap) + 7 * 4 * d.Ap);
  for (int a = threadIdx.x; a < d.A; a += blockDim.x) {
    double x[3] = {ao[a], ao[d.Ap + a], ao[2 * d.Ap + a]};
    for (int j = alink[a]; j >= 0; j = topo[j].x) {
      double y[3];
      qrot4(load_q4(c.quatd, (size_t)d.link_base + j), x, y);
      const int pa = topo[j].x;
      x[0] = y[0]; x[1] = y[1]; x[2] = y[2] + (pa >= 0 ? (double)Lown[pa] : 0.0);
    }
    for (int k = 0; k < 3; k++) c.anchor[3 * (size_t)d.apple_base + (size_t)k * d.Ap + a] = x[k];
  }
}

// ------------------------------------------------------------------------------------------------------
// k_randomize_geometry: ONE THREAD PER WORLD ("an on-device build that perturbs every world's branch
// geometry in a single ... kernel (one thread per world)"): per-world growth habit and dimensions drawn with
// Philox4x32-10 and applied to the base geometry in a top-down re-walk (reading A37 in DESIGN.md;
// the readings are spelled out at ob_randomize_geometry in include/orchard.h).  Quaternion algebra in fp64; the world
// rest quaternion of every link (needed by its children while the droop compounds) is parked in the world's slice of the
// PCG history pool, which the reset that follows clears anyway.
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ Qd4 axis_angle_xy(const double ax, const double ay, const double angle) {   // axis (ax, ay, 0)
  double sn, cs;
  sincos(0.5 * angle, &sn, &cs);
  Qd4 q;
  q.w = cs; q.x = ax * sn; q.y = ay * sn; q.z = 0.0;
  return q;
}

__global__ void k_randomize_geometry(DevCtx c, unsigned long long seed, ob_geometry_ranges G) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= c.n_worlds) return;
  const WorldDesc d = c.desc[w];
  const uint2 key = make_uint2((uint32_t)(seed & 0xffffffffull), (uint32_t)(seed >> 32));
  const uint4 o0 = philox4x32_10(make_uint4((uint32_t)w, 0u, 3u, 0u), key);
  const uint4 o1 = philox4x32_10(make_uint4((uint32_t)w, 1u, 3u, 0u), key);
  const float droop = philox_uniform(o0.x, G.droop[0], G.droop[1]);
  const float lean = philox_uniform(o0.y, G.lean[0], G.lean[1]);
  const float spread = philox_uniform(o0.z, G.spread[0], G.spread[1]);
  const float twist = philox_uniform(o0.w, G.twist[0], G.twist[1]);
  const float phi = philox_uniform(o1.x, 0.0f, 6.2831855f);
  const float sL = philox_uniform(o1.y, G.scale_length[0], G.scale_length[1]);
  const float sD = philox_uniform(o1.z, G.scale_diameter[0], G.scale_diameter[1]);
  const int4 *topo = c.topo + d.link_base;
  const float4 *quat0 = c.quat_raw + d.link_base;
  double *park[4];                                     // world rest quaternion of link i: component k at park[k][i]
  for (int k = 0; k < 4; k++) park[k] = reinterpret_cast<double *>(c.xprev + (size_t)k * c.sum_np + d.link_base);
  for (int i = 0; i < d.N; i++) {
    // dimensions: L = (L0 * scale) * jitter in fp32, the jitter drawn by the CALLER's link index
    const uint4 oi = philox4x32_10(make_uint4((uint32_t)w, (uint32_t)c.link_ext[d.link_base + i], 4u, 0u), key);
    const float jl = philox_uniform(oi.x, G.jitter_length[0], G.jitter_length[1]);
    const float jd = philox_uniform(oi.y, G.jitter_diameter[0], G.jitter_diameter[1]);
    c.Lown[d.link_base + i] = __fmul_rn(__fmul_rn(c.Lown0[d.link_base + i], sL), jl);
    c.diam[d.link_base + i] = __fmul_rn(__fmul_rn(c.diam0[d.link_base + i], sD), jd);
    // rest rotation: spread and twist of a child about its parent's axis, lean of the trunk
    const float4 qf = quat0[i];
    Qd4 q;
    {
      const double nn = sqrt((double)qf.x * qf.x + (double)qf.y * qf.y + (double)qf.z * qf.z + (double)qf.w * qf.w);
      q.w = qf.x / nn; q.x = qf.y / nn; q.y = qf.z / nn; q.z = qf.w / nn;
    }
    const int pa = topo[i].x;
    if (pa >= 0) {
      // direction of the child's axis in the parent frame: R(q) z
      const double dx = 2 * (q.x * q.z + q.w * q.y), dy = 2 * (q.y * q.z - q.w * q.x), dz = 1 - 2 * (q.x * q.x + q.y * q.y);
      const double hn = sqrt(dx * dx + dy * dy);
      if (hn > 1e-12 && spread != 0.f) q = qmul4(axis_angle_xy(-dy / hn, dx / hn, atan2(hn, dz) * (double)spread), q);
      if (twist != 0.f) {
        double sn, cs;
        sincos(0.5 * (double)twist, &sn, &cs);
        Qd4 t;
        t.w = cs; t.x = 0.0; t.y = 0.0; t.z = sn;
        q = qmul4(t, q);
      }
    } else if (lean != 0.f) {
      q = qmul4(axis_angle_xy(cos((double)phi), sin((double)phi), (double)lean), q);
    }
    double *out = c.quatd + 4 * ((size_t)d.link_base + i);
    if (droop == 0.f) {                               // no re-walk: the modified rest rotation is the result, exactly
      out[0] = q.w; out[1] = q.x; out[2] = q.y; out[3] = q.z;
      continue;
    }
    Qd4 qp;
    qp.w = 1.0; qp.x = 0.0; qp.y = 0.0; qp.z = 0.0;
    if (pa >= 0) { qp.w = park[0][pa]; qp.x = park[1][pa]; qp.y = park[2][pa]; qp.z = park[3][pa]; }
    Qd4 qi = qmul4(qp, q);
    {
      const double dx = 2 * (qi.x * qi.z + qi.w * qi.y), dy = 2 * (qi.y * qi.z - qi.w * qi.x);
      const double sn = sqrt(dx * dx + dy * dy);      // sine of the angle to the vertical
      if (sn > 1e-12) qi = qmul4(axis_angle_xy(-dy / sn, dx / sn, (double)droop * sn), qi);   // towards the ground
    }
    park[0][i] = qi.w; park[1][i] = qi.x; park[2][i] = qi.y; park[3][i] = qi.z;
    Qd4 qc;
    qc.w = qp.w; qc.x = -qp.x; qc.y = -qp.y; qc.z = -qp.z;
    const Qd4 qn = qmul4(qc, qi);                      // the new rest rotation in the (turned) parent frame
    out[0] = qn.w; out[1] = qn.x; out[2] = qn.y; out[3] = qn.z;
  }
  // attach points move with their link: x, y by its diameter factor, z by its length factor
  unsigned char *ab = c.apple_blk + d.apple_blk_off;
  float *ao = reinterpret_cast<float *>(ab + apple_state_bytes(d.Ap));
  const int32_t *alink = reinterpret_cast<const int32_t *>(ab + apple_state_bytes(d.Ap) + 7 * 4 * d.Ap);
  const float *ao0 = c.apple_off0 + 3 * (size_t)d.apple_base;
  for (int a = 0; a < d.A; a++) {
    const int b = d.link_base + alink[a];
    const float fl = __fdiv_rn(c.Lown[b], c.Lown0[b]), fd = __fdiv_rn(c.diam[b], c.diam0[b]);
    ao[a] = __fmul_rn(ao0[a], fd); ao[d.Ap + a] = __fmul_rn(ao0[d.Ap + a], fd); ao[2 * d.Ap + a] = __fmul_rn(ao0[2 * d.Ap + a], fl);
  }
}

// ------------------------------------------------------------------------------------------------------
// k_randomize: one CTA per world.  redraw = 0: nominal materials of the specs (ob_create); 1: Philox draws; 2: keep the
// current materials (after ob_randomize_geometry).  Always: derived constants from the current dimensions, full reset.
// ------------------------------------------------------------------------------------------------------
__global__ void k_randomize(DevCtx c, unsigned long long seed, int redraw) {
  const int w = blockIdx.x;
  const WorldDesc d = c.desc[w];
  const ob_params &P = c.P;
  WorldInfo *info = c.info + w;
  const uint2 key = make_uint2((uint32_t)(seed & 0xffffffffull), (uint32_t)(seed >> 32));
  float E = d.E, MOR = d.MOR, rho = d.density;
  if (redraw == 2) {                                   // keep the materials as they are (after ob_randomize_geometry)
    E = info->E; MOR = info->MOR; rho = info->density;
  } else if (redraw) {
    uint4 o = philox4x32_10(make_uint4((uint32_t)w, 0u, 0u, 0u), key);
    if (P.range_E[0] != P.range_E[1]) E = philox_uniform(o.x, P.range_E[0], P.range_E[1]);
    if (P.range_MOR[0] != P.range_MOR[1]) MOR = philox_uniform(o.y, P.range_MOR[0], P.range_MOR[1]);
    if (P.range_density[0] != P.range_density[1]) rho = philox_uniform(o.z, P.range_density[0], P.range_density[1]);
  }
  unsigned char *lb = c.link_blk + d.link_blk_off;
  float *st = reinterpret_cast<float *>(lb);
  unsigned char *fl = lb + kLinkStateFloats * 4 * d.Np;
  float *cs = reinterpret_cast<float *>(c.link_cst + (size_t)link_const_bytes(1) * d.link_base);
  const float *Lown = c.Lown + d.link_base, *diam = c.diam + d.link_base;
  const int4 *topo = c.topo + d.link_base;
  const double PI = 3.14159265358979323846;
  for (int i = threadIdx.x; i < d.Np; i += blockDim.x) {
    for (int k = 0; k < kLinkStateFloats; k++) st[k * d.Np + i] = 0.f;
    fl[i] = 0; fl[d.Np + i] = 0;
    c.xprev[d.link_base + i] = make_float2(0.f, 0.f);              // PCG start-vector history
    c.xprev[c.sum_np + d.link_base + i] = make_float2(0.f, 0.f);
    c.xprev[2 * c.sum_np + d.link_base + i] = make_float2(0.f, 0.f);
    c.xprev[3 * c.sum_np + d.link_base + i] = make_float2(0.f, 0.f);
    if (i < d.N) {
      double dd = diam[i], L = Lown[i], r = 0.5 * dd;
      double K = (double)E * PI * dd * dd * dd * dd / (64.0 * L);   // Eq. 4
      double Mx = (double)MOR * PI * dd * dd * dd / 32.0;           // Eq. 5
      double m = (double)rho * PI * r * r * L;                      // solid cylinder
      double Ic = m * (3.0 * r * r + L * L) / 12.0, cz = 0.5 * L;
      int pa = topo[i].x;
      // c4 = (m, m c, I about the joint, I_zz), then K[Np], rz[Np]  (ob_internal.h)
      reinterpret_cast<float4 *>(cs)[i] =
          make_float4((float)m, (float)(m * cz), (float)(Ic + m * cz * cz), (float)(0.5 * m * r * r));
      cs[4 * d.Np + i] = (float)K;
      cs[5 * d.Np + i] = pa >= 0 ? Lown[pa] : 0.f;
      c.Mmax[d.link_base + i] = (float)Mx;
    } else {
      reinterpret_cast<float4 *>(cs)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      cs[4 * d.Np + i] = 0.f;
      cs[5 * d.Np + i] = 0.f;
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
      if (redraw == 1) {
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
// k_pose: link frames of one world (position + quaternion), fp64 ancestor walk from the stored state
// ------------------------------------------------------------------------------------------------------
__global__ void k_pose(DevCtx c, int w) {
  const WorldDesc d = c.desc[w];
  const int4 *topo = c.topo + d.link_base;
  const float *Lown = c.Lown + d.link_base;
  const float *st = reinterpret_cast<const float *>(c.link_blk + d.link_blk_off);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < d.N; i += gridDim.x * blockDim.x) {
    double R[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1}, x[3] = {0, 0, 0};
    for (int j = i; j >= 0; j = topo[j].x) {
      double Q[9], T[9], A[9];
      {
        const Qd4 q = load_q4(c.quatd, (size_t)d.link_base + j);
        const double w = q.w, x = q.x, y = q.y, z = q.z;
        Q[0] = 1 - 2 * (y * y + z * z); Q[1] = 2 * (x * y - w * z);     Q[2] = 2 * (x * z + w * y);
        Q[3] = 2 * (x * y + w * z);     Q[4] = 1 - 2 * (x * x + z * z); Q[5] = 2 * (y * z - w * x);
        Q[6] = 2 * (x * z - w * y);     Q[7] = 2 * (y * z + w * x);     Q[8] = 1 - 2 * (x * x + y * y);
      }
      double s1, c1, s2, c2;
      sincos((double)st[2 * j], &s1, &c1);
      sincos((double)st[2 * j + 1], &s2, &c2);
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
cudaError_t launch_anchors(const DevCtx &c, cudaStream_t s) {
  k_anchors<<<c.n_worlds, 128, 0, s>>>(c);
  return cudaGetLastError();
}
cudaError_t launch_geometry(const DevCtx &c, unsigned long long seed, const ob_geometry_ranges &r, cudaStream_t s) {
  k_randomize_geometry<<<(c.n_worlds + 63) / 64, 64, 0, s>>>(c, seed, r);
  return cudaGetLastError();
}
cudaError_t launch_randomize(const DevCtx &c, unsigned long long seed, int redraw, cudaStream_t s) {
  k_randomize<<<c.n_worlds, 128, 0, s>>>(c, seed, redraw);
  return cudaGetLastError();
}
// ------------------------------------------------------------------------------------------------------
// k_stats: totals over all worlds for ob_stats (one 32-byte copy instead of every WorldInfo)
// ------------------------------------------------------------------------------------------------------
__global__ void k_stats(DevCtx c) {
  __shared__ unsigned long long sh[3][256];
  unsigned long long it = 0, ws = 0, fl = 0;
  for (int w = threadIdx.x; w < c.n_worlds; w += blockDim.x) {
    const WorldInfo &x = c.info[w];
    it += x.cg_iters; ws += (unsigned long long)x.steps_taken; fl += x.status != 0;
  }
  sh[0][threadIdx.x] = it; sh[1][threadIdx.x] = ws; sh[2][threadIdx.x] = fl;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o)
      for (int k = 0; k < 3; k++) sh[k][threadIdx.x] += sh[k][threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x < 3) c.stats[threadIdx.x] = sh[threadIdx.x][0];
}
cudaError_t launch_stats(const DevCtx &c, cudaStream_t s) {
  k_stats<<<1, 256, 0, s>>>(c);
  return cudaGetLastError();
}
cudaError_t launch_pose(const DevCtx &c, int world, cudaStream_t s) {
  k_pose<<<4, 128, 0, s>>>(c, world);
  return cudaGetLastError();
}

// self-test: the generator above and cuRAND's curand_Philox4x32_10 on the same (counter, key) pairs
__global__ void k_philox_selftest(int n, const uint32_t *__restrict__ in, uint32_t *__restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 ctr = make_uint4(in[6 * i], in[6 * i + 1], in[6 * i + 2], in[6 * i + 3]);
  const uint2 key = make_uint2(in[6 * i + 4], in[6 * i + 5]);
  const uint4 a = philox4x32_10(ctr, key);
  const uint4 b = curand_Philox4x32_10(ctr, key);
  out[8 * i] = a.x; out[8 * i + 1] = a.y; out[8 * i + 2] = a.z; out[8 * i + 3] = a.w;
  out[8 * i + 4] = b.x; out[8 * i + 5] = b.y; out[8 * i + 6] = b.z; out[8 * i + 7] = b.w;
}
cudaError_t launch_philox_selftest(int n, const uint32_t *d_in, uint32_t *d_out, cudaStream_t s) {
  k_philox_selftest<<<(n + 127) / 128, 128, 0, s>>>(n, d_in, d_out);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------
// The same self-test for callers that have no device memory to lend and may not ask the driver for any
// (ob_selftest_philox_static in include/orchard.h).  Its staging area is the file-scope array below: 224 KB that
// every GPU which loads libob.so holds from module load until the process exits.  All calls on one device share
// it and it keeps whatever the previous call left there; the kernel overwrites all 8n output words of a call and
// the inputs are copied in first, so nothing has to start at zero -- but two calls that overlap on the GPU race.
//
// g_selftest_scratch is a device symbol.  In host code that name is only the host-side stand-in of the symbol, not
// an address a kernel can use, so the host asks the runtime for the device address (once per device, with that
// device current) and hands the kernel that pointer.
// ------------------------------------------------------------------------------------------------------
static __device__ __align__(256) uint32_t g_selftest_scratch[14 * OB_SELFTEST_STATIC_MAX];

// layout of the scratch for n pairs: ctr [4n] | key [2n] | library output [4n] | cuRAND output [4n]
__global__ void k_philox_selftest_static(int n, uint32_t *__restrict__ scratch) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t *ctr_in = scratch, *key_in = scratch + 4 * (size_t)n;
  uint32_t *out_lib = scratch + 6 * (size_t)n, *out_cur = scratch + 10 * (size_t)n;
  const uint4 ctr = make_uint4(ctr_in[4 * i], ctr_in[4 * i + 1], ctr_in[4 * i + 2], ctr_in[4 * i + 3]);
  const uint2 key = make_uint2(key_in[2 * i], key_in[2 * i + 1]);
  const uint4 a = philox4x32_10(ctr, key);
  const uint4 b = curand_Philox4x32_10(ctr, key);
  out_lib[4 * i] = a.x; out_lib[4 * i + 1] = a.y; out_lib[4 * i + 2] = a.z; out_lib[4 * i + 3] = a.w;
  out_cur[4 * i] = b.x; out_cur[4 * i + 1] = b.y; out_cur[4 * i + 2] = b.z; out_cur[4 * i + 3] = b.w;
}

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_scratch_mutex;
uint32_t *g_scratch_addr[kMaxDevices];   // device address of g_selftest_scratch on device d, 0 = not looked up yet
}  // namespace

// Device address of the static scratch on the CURRENT device; the first call on a device does the look-up.
static cudaError_t selftest_scratch_address(uint32_t **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_addr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_selftest_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_addr[dev] = static_cast<uint32_t *>(p);
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

// Copies straight from / to the caller's host arrays (no host staging buffer either); synchronises s.
cudaError_t philox_selftest_static(int n, const uint32_t *ctr, const uint32_t *key, uint32_t *out_lib,
                                   uint32_t *out_curand, cudaStream_t s) {
  uint32_t *d = nullptr;
  cudaError_t e = selftest_scratch_address(&d);
  if (e != cudaSuccess) return e;
  const size_t N = (size_t)n;
  e = cudaMemcpyAsync(d, ctr, 16 * N, cudaMemcpyHostToDevice, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d + 4 * N, key, 8 * N, cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return e;
  k_philox_selftest_static<<<(n + 127) / 128, 128, 0, s>>>(n, d);
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(out_lib, d + 6 * N, 16 * N, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(out_curand, d + 10 * N, 16 * N, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  return e;
}

}  // namespace ob
