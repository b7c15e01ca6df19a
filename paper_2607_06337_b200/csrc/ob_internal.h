// ob_internal.h -- device data layout shared by the host runtime (ob_host.cu) and the kernels
// (ob_kernels.cu).  Nothing here is visible across the C ABI (include/orchard.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/orchard.h"

namespace ob {

constexpr int kPad = 16;  // links and apples per world are padded to a multiple of 16 (16-byte TMA granules)
__host__ __device__ inline int pad16(int n) { return (n + kPad - 1) / kPad * kPad; }

// ---- per-world link STATE block in global memory (pool link_blk, worlds back to back: a range of worlds is one
//      contiguous chunk, which is what the batched read-out copies).  k_step reads and writes it in place (L2): only
//      the once-per-step phases touch it.
//   float2  q[Np] qd[Np]                the two DoF of a joint interleaved
//   int32   rstep[Np]                   step during which the joint ruptured (the friction ramp counts from it)
//   bytes   ruptured[Np] rc[Np]
// ---- per-world link CONSTANT block (pool link_cst; written by k_randomize):
//   float4  c4[Np] = (m, m c, I about the joint, I_zz)
//   floats  K[Np] rz[Np]                joint stiffness (Eq. 4), parent length
constexpr int kLinkStateFloats = 5;
constexpr int kLinkConstFloats = 6;
__host__ __device__ inline int link_state_bytes(int Np) { return kLinkStateFloats * 4 * Np + 2 * Np; }
__host__ __device__ inline int link_const_bytes(int Np) { return kLinkConstFloats * 4 * Np; }

// ---- per-world "apple block":
//   floats  u[3][Ap] v[3][Ap]              state (u = x - x_rest, x_rest = anchor + m g / k_s; anchor = rest hang point, fp64, host side)
//   bytes   attached[Ap] cA[Ap] cB[Ap]     state
//   floats  o[3][Ap] k[Ap] m[Ap] c[Ap] fdet[Ap]   constants
//   int32   link[Ap]                       internal link index
__host__ __device__ inline int apple_state_bytes(int Ap) { return 6 * 4 * Ap + 3 * Ap; }
__host__ __device__ inline int apple_block_bytes(int Ap) { return apple_state_bytes(Ap) + 7 * 4 * Ap + 4 * Ap; }

struct WorldDesc {
  int32_t N, A, Np, Ap;
  int32_t NFp;          // factor slots (links with children, leaves with an off-axis apple), padded to a multiple of 8
  int32_t n_levels;
  int32_t n_top;        // leading levels whose links all lie in [0, 32): swept by warp 0 with __syncwarp only
  int32_t cls;          // size class (index into kStepClasses)
  int32_t link_base;    // sum of Np of the worlds before this one
  int32_t apple_base;   // sum of Ap
  int32_t level_base;   // offset into the level-offset pool (n_levels + 1 entries)
  int64_t link_blk_off;   // byte offset of the link state block in its pool (= link_state_bytes(1) * link_base)
  int64_t apple_blk_off;  // byte offset of the apple block in the apple-block pool
  float density, E, MOR;  // nominal (spec) values
  int32_t has_apple_c;
  int32_t precond;      // the preconditioner this world runs with: ob_params.precond, or 1 (Jacobi) where the factor planes
                        // of precond 2 do not fit into one CTA's shared memory beside the world
  int32_t pad_[2];
};

struct WorldInfo {       // mutable per-world scalars
  int32_t step;
  int32_t last_iters;
  int32_t status;
  int32_t steps_taken;           // world-steps actually advanced (frozen worlds do not count)
  unsigned long long cg_iters;   // PCG iterations since ob_create
  float E, MOR, density;         // current material draws
  int32_t pad_;
};

struct WrenchSlots {     // device mirror of the persistent wrenches of one world (internal body indices)
  int32_t n;
  int32_t body[OB_MAX_WRENCH];
  float point[OB_MAX_WRENCH][3];
  float force[OB_MAX_WRENCH][3];
  int32_t pad_[3];
};
static_assert(sizeof(WrenchSlots) % 16 == 0, "WrenchSlots must stay 16-byte sized");

struct DevCtx {
  int32_t n_worlds;
  const WorldDesc *desc;
  const int32_t *order;          // worlds grouped by size class, largest first inside a class (work queues)
  unsigned char *link_blk;       // link state pool
  unsigned char *link_cst;       // link constant pool (block of world w at link_const_bytes(1) * link_base)
  unsigned char *apple_blk;      // apple-block pool
  // per-link statics, indexed link_base + i (SoA pools use k * Np + i inside the world's slice)
  const int4 *topo;              // x = parent (-1 = trunk), y = first child (children are contiguous), z = level,
                                 // w = number of children
  const int4 *topo2;             // x = first apple | n_apples << 16, y = inner slot | parent's inner slot << 16
  const float4 *quat_raw;        // rest quaternion exactly as the caller gave it (create-time fp64 rest pose)
  double *quatd;                 // [4 * (link_base + i)] the same, normalised, in fp64 (k_rest_pose; the FK of k_step)
  float *Mmax;                   // rupture moment (after randomize)
  float2 *xprev;                 // [4][sumNp]: dqd of the last four steps, slot = step & 3 (PCG start: extrapolation)
  int32_t sum_np;                // stride of xprev
  float *Lown;                   // link length (current: ob_randomize_geometry rewrites it from Lown0)
  float *diam;                   // link diameter
  const float *Lown0, *diam0;    // base geometry as given to ob_create
  const float *apple_off0;       // [3 * apple_base + k * Ap + a] base attach points
  const float *arm;              // [2 * link_base + k * Np + i] armature or nullptr
  const int32_t *link_ext;       // internal -> caller's link index
  const int32_t *apple_ext;      // internal -> caller's apple index
  const float *apple_nominal;    // [2 * apple_base + k * Ap + a]: nominal mass, detach force
  const float *apple_c_in;       // [apple_base + a] caller's c_s or nullptr-equivalent (see has_apple_c)
  double *anchor;                // [3 * apple_base + k * Ap + a] rest hang point, world frame, fp64
  const int32_t *level_off;
  WorldInfo *info;
  const WrenchSlots *wrench;
  ob_event *events;
  int32_t ev_cap;
  int32_t *ev_count;             // [0] = appended, [1] = overflow flag
  int32_t *queue;                // work-queue counters, one per size class
  unsigned long long *iter_hist; // [kIterHistBins] world-steps by PCG iteration count (last bin: that many or more)
  unsigned long long *stats;     // [4] scratch of k_stats: PCG iterations, world-steps, flagged worlds
  int32_t *progress;             // [n_worlds] chunks of the current launch a world has finished
  float *pose7;                  // scratch for ob_get_state(link_pose7): 7 * max Np floats
  ob_params P;
};

// ---- k_step size classes: threads per CTA x links per thread (flat ownership: link tid + k * nt) x the CTAs
//      per SM the registers are budgeted for.  Only the PCG vectors x, r and the Jacobi factors live in
//      registers; everything the level sweeps touch lives in shared memory, so the sweep code exists once and
//      runs over any number of links.
struct StepClass { int nt, lpt, min_ctas; };
constexpr int kNumClasses = 5;
constexpr int kIterHistBins = 64;
// Few threads per world: measured on configs[3] (350-450 links, three worlds per SM) 128 threads x 4 links
// give 3.75M world-steps/s, 192 x 3 3.26M, 256 x 2 2.90M, 64 x 8 3.27M: a PCG iteration is a chain of short
// phases, and more warps per world only add barrier and loop overhead to each of them.
constexpr StepClass kStepClasses[kNumClasses] = {
    {64, 4, 6}, {128, 4, 3}, {192, 4, 2}, {256, 4, 1}, {256, 6, 1}};
constexpr int kMaxLinksOnChip = 256 * 6;
constexpr int kMaxChildren = 15;     // children per link (4 bits of the packed topology word)
// the smallest class whose threads cover the links and whose per-SM residency the world's shared memory allows
inline int class_smem_cap(int min_ctas);
inline int step_class_of(int Np, int smem_bytes) {   // host only
  for (int k = 0; k < kNumClasses; k++)
    if (Np <= kStepClasses[k].nt * kStepClasses[k].lpt && smem_bytes <= class_smem_cap(kStepClasses[k].min_ctas)) return k;
  return -1;
}

// shared-memory footprint of one world in k_step (bytes); the host uses it to size the launch and to pick the size
// class.  Np + 1 records of seven float4 (record Np stays zero: the trunk's parent, missing children) | X21 float
// [Np + 1] | factor-slot index uint16 [Np + 1] | factor planes: four float4 [NFp] (precond 2), or 1 / diag(A) float2
// [Np + 1] (precond 0, 1) | level offsets | apple block (TMA) | ten float planes [Ap]: anchor - x_hang (A1 -> A2), then
// f_tether, |f_s| (A2 -> D); the world quaternion of the apple's link | world quaternions of the wrench links |
// wrench slots
__host__ __device__ inline int r16(int b) { return (b + 15) / 16 * 16; }
__host__ __device__ inline int step_planes_bytes(int Np) { return 7 * 16 * (Np + 1); }
__host__ __device__ inline int step_fac_bytes(int Np, int NFp) { return 64 * NFp > r16(8 * (Np + 1)) ? 64 * NFp : r16(8 * (Np + 1)); }
// (a world that runs with precond <= 1 passes NFp = 0)
__host__ __device__ inline int step_smem_bytes(int Np, int Ap, int NFp, int nlev) {
  int b = 0;
  b += step_planes_bytes(Np);
  b += r16(4 * (Np + 1));
  b += r16(2 * (Np + 1));
  b += step_fac_bytes(Np, NFp);
  b += r16(4 * (nlev + 1));
  b += r16(apple_block_bytes(Ap));
  b += 10 * 4 * Ap;
  b += 16 * OB_MAX_WRENCH;
  b += (int)sizeof(WrenchSlots);
  return (b + 127) / 128 * 128;
}
// the most dynamic shared memory a CTA of a class may use so that min_ctas of them stay resident on an SM (228 KB per
// SM, 1 KB reserved per CTA, 1 KB for the kernel's static shared memory)
inline int class_smem_cap(int min_ctas) { return (228 * 1024) / min_ctas - 1024 - 1024; }

// kernel launchers (ob_kernels.cu)
cudaError_t launch_rest_pose(const DevCtx &c, int total_links_padded, int total_apples_padded, cudaStream_t s);
cudaError_t launch_randomize(const DevCtx &c, unsigned long long seed, int redraw, cudaStream_t s);
cudaError_t launch_step(const DevCtx &c, int cls, const int32_t *order, int n_in_class, int32_t *queue, int n_steps,
                        int grid, int smem, int n_sm, int n_chunks, int32_t *progress, cudaStream_t s);
cudaError_t launch_pose(const DevCtx &c, int world, cudaStream_t s);
cudaError_t launch_stats(const DevCtx &c, cudaStream_t s);
cudaError_t launch_geometry(const DevCtx &c, unsigned long long seed, const ob_geometry_ranges &r, cudaStream_t s);
cudaError_t launch_anchors(const DevCtx &c, cudaStream_t s);
cudaError_t launch_philox_selftest(int n, const uint32_t *d_in, uint32_t *d_out, cudaStream_t s);
// the self-test on the library's own static scratch (no allocation anywhere); n <= OB_SELFTEST_STATIC_MAX, synchronises s
cudaError_t philox_selftest_static(int n, const uint32_t *ctr, const uint32_t *key, uint32_t *out_lib,
                                   uint32_t *out_curand, cudaStream_t s);
cudaError_t step_kernel_setup(int cls, int smem_bytes, int *max_blocks_per_sm);

}  // namespace ob
