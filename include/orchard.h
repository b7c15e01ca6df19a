/*
 * orchard.h -- C ABI of the B200-native batched tree-physics step (OrchardBench hot path).
 *
 * One call = one step of the paper's problem statement (PAPER.md = /root/reference/PAPER.md):
 *   articulation      PAPER.md:113-117  (Eq. 3)   links = rigid cylinders along local +z, joint at the
 *                                                  parent's distal tip, rest transform q_rel
 *   compliant joints  PAPER.md:121-126  (Eq. 4)   2 bending DoF, K = E pi d^4/(64 L), D = c_d K
 *   rupture           PAPER.md:132-141  (Eq. 5)   K |theta| > MOR pi d^3/32 for N frames -> K = D = 0 in place
 *   fruit tethers     PAPER.md:147-163  (Eq. 6,7) 3-DoF apples, clamped reaction on the spur, 2 detach paths
 *   randomization     PAPER.md:165-169            per-world E, MOR, density; per-apple detach force, mass
 *   stability rails   PAPER.md:398      (App. B)  forces off on snapped sub-trees; joint speed clamp
 *   time step         BASELINE.json north_star    (M + hD + h^2 K) dqd = rhs by matrix-free Jacobi-PCG,
 *                                                  M*v from inverse-dynamics tree sweeps
 * DESIGN.md lists every reading taken where the paper is silent.
 *
 * Conventions
 *   - Every call returns int: 0 (OB_OK) or a negative OB_E_* code.  Nothing throws or aborts across the ABI.
 *     ob_last_error(ctx) returns a NUL-terminated string owned by the context (or a static string for NULL).
 *   - Pointers are HOST pointers unless the parameter is named dev_* (device memory) or cuda_stream
 *     (a cudaStream_t passed as void*).  The caller owns everything it passes in: inputs are copied during
 *     the call, outputs are filled up to the stated capacity.  The context is opaque and library-owned.
 *   - The library allocates no device memory of its own: the caller provides one workspace of
 *     ob_workspace_bytes() bytes (256-byte aligned), which must outlive the context.
 *   - All device work is enqueued on the stream given to ob_create.  ob_step and ob_randomize are
 *     asynchronous; calls that return data to the host synchronise that stream.
 *   - One context is used from one host thread at a time.  There is no global state.
 *   - There is no CPU fallback: without a CUDA device ob_create returns OB_E_CUDA.
 *   - Indices in specs, wrenches, states and events are the CALLER's indices; the library reorders links
 *     (level order) and apples (by link) internally.
 */
#ifndef ORCHARD_H_
#define ORCHARD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OB_OK 0
#define OB_E_ARG (-1)        /* null pointer, index out of range, non-topological parent, non-unit quaternion */
#define OB_E_CAPACITY (-2)   /* wrench slots, event buffer, or a world too large for on-chip residency */
#define OB_E_WORKSPACE (-3)  /* workspace too small or misaligned */
#define OB_E_CUDA (-4)       /* a CUDA runtime call failed (no device, launch failure, ...) */

#define OB_MAX_WRENCH 8      /* persistent wrench slots per world, keyed by body */

#define OB_STATUS_NONFINITE 1 /* a non-finite value appeared: the world is frozen at its last finite state */
#define OB_STATUS_CG_MAXITER 2 /* PCG hit cg_max_iter at least once (the world keeps stepping) */

typedef struct ob_ctx ob_ctx;

/* One world.  Worlds may differ in every field (heterogeneous batches are fine). */
typedef struct {
  int32_t n_links;              /* >= 1, <= 32767 */
  const int32_t *parent;        /* [n_links] parent[0] = -1 (trunk, jointed to the world), 0 <= parent[i] < i */
  const float *length;          /* [n_links] m, > 0 */
  const float *diameter;        /* [n_links] m, > 0 */
  const float *rest_quat;       /* [4*n_links] (w,x,y,z): child rest frame in the parent frame (Eq. 3);
                                   link 0: in the world frame.  | |q|-1 | <= 1e-3, normalised internally */
  const float *armature;        /* [2*n_links] kg m^2 added to the two DoF of each joint, or NULL */
  float density, E, MOR;        /* kg/m^3, Pa, Pa: nominal values; replaced by ob_randomize when the
                                   corresponding range in ob_params is non-degenerate */
  int32_t n_apples;             /* >= 0, <= 1024 */
  const int32_t *apple_link;    /* [n_apples] link carrying the apple */
  const float *apple_offset;    /* [3*n_apples] attach (hang) point in link-local coordinates */
  const float *apple_mass;      /* [n_apples] kg > 0 */
  const float *apple_radius;    /* [n_apples] m (carried; unused by the dynamics) or NULL */
  const float *apple_k;         /* [n_apples] tether stiffness k_s, N/m > 0 (Eq. 6) */
  const float *apple_c;         /* [n_apples] tether damping c_s, N s/m, or NULL -> 2 zeta_s sqrt(k_s m) */
  const float *apple_detach;    /* [n_apples] detach force f_detach, N */
} ob_world_spec;

/* Numerical parameters; ob_default_params() fills the defaults given in braces. */
typedef struct {
  float h;                      /* {2e-3} step, s */
  float gravity[3];             /* {0,0,-9.81} m/s^2, world frame */
  float c_d;                    /* {0.05} s; D = c_d K (Eq. 4) */
  float cg_tol;                 /* {1e-6} PCG stops at |r| <= cg_tol |b| in the norm selected by cg_norm */
  int32_t cg_max_iter;          /* {200} */
  int32_t precond;              /* {1} 0 = none, 1 = Jacobi (exact diagonal from a composite-inertia sweep) */
  int32_t cg_norm;              /* {0} residual norm of the stopping rule: 0 = plain 2-norm; 1 = the preconditioned
                                   norm sqrt(r^T P^-1 r) that PCG carries anyway (one reduction fewer) */
  int32_t rupture_frames;       /* {3} consecutive steps above M_max before a joint ruptures (<= 255) */
  int32_t detach_frames_pull;   /* {3} steps of |user force on the apple| > f_detach (<= 255) */
  float detach_kappa;           /* {1.1} stem-tension threshold factor */
  int32_t detach_frames_tension;/* {10} steps of |f_s| > kappa f_detach (<= 255) */
  float react_max;              /* {40} N, norm clamp on the tether reaction */
  int32_t tether_implicit;      /* {1} 1 = linearly implicit tether reaction; 0 = paper-literal explicit Eq. 7 */
  float qd_max;                 /* {50} rad/s component-wise joint speed clamp; <= 0 disables */
  float zeta_s;                 /* {0.1} default tether damping ratio */
  int32_t forces_off_on_snapped;/* {1} user wrenches on links at/below a ruptured joint are ignored */
  float range_E[2];             /* per-world uniform ranges; lo == hi keeps the spec's nominal value */
  float range_MOR[2];
  float range_density[2];
  float range_detach[2];        /* per apple */
  float range_apple_mass[2];    /* per apple */
  float mass_damping;           /* {0} 1/s >= 0: velocity-proportional damping F = -c_v m v, tau = -c_omega I omega on
                                   every link and apple with c_v = c_omega = mass_damping; in joint
                                   space -mass_damping M(q) qd, taken linearly implicit like the joint damper */
} ob_params;

typedef struct {
  int32_t world, step;          /* step = 0-based index of the step during which the flag flipped */
  int32_t kind;                 /* 0 = rupture (index = link), 1 = detach (index = apple) */
  int32_t index;
  float value, threshold;       /* rupture: K|theta| vs M_max; detach: |f_user| vs f_detach or |f_s| vs kappa f_detach */
} ob_event;

/* Fill *p with the defaults above.  Returns OB_E_ARG for NULL. */
int ob_default_params(ob_params *p);

/* Bytes of device workspace ob_create needs for these worlds (validates the specs). */
int ob_workspace_bytes(const ob_world_spec *specs, int n_worlds, const ob_params *params, size_t *out);

/* Build the device layout (level-ordered SoA per world), compute rest poses and derived constants, reset the
   state to the rest pose (apples at their rest sag m g / k_s below the hang point).  dev_workspace: device
   memory of at least ob_workspace_bytes bytes; cuda_stream: cudaStream_t (NULL = default stream). */
int ob_create(const ob_world_spec *specs, int n_worlds, const ob_params *params, void *dev_workspace,
              size_t workspace_bytes, void *cuda_stream, ob_ctx **out);

/* On-device Philox4x32-10 redraw of every world (key = seed; counter = (world, item, stream, 0); stream 0 item 0
   -> E, MOR, density; stream 1 item a -> detach force, mass of apple a; u = float(x>>8) 2^-24,
   value = fmaf(u, hi-lo, lo)), then derived constants and a full reset: rest pose, zero velocities, flags,
   counters, step = 0, wrench slots cleared, warm start cleared.  Pending events stay queued.  Asynchronous. */
int ob_randomize(ob_ctx *ctx, uint64_t seed);

/* Persistent external force.  body in [0, n_links) is a link, [n_links, n_links + n_apples) an apple.
   point: application point in the link's local frame (moves with the link; ignored for apples).
   force: world frame, N.  The wrench persists until replaced (same body) or removed (zero force).
   Each world has OB_MAX_WRENCH slots; one more distinct body returns OB_E_CAPACITY. */
int ob_apply_wrench(ob_ctx *ctx, int world, int body, const float point[3], const float force[3]);
int ob_apply_wrench_batch(ob_ctx *ctx, int n, const int32_t *world, const int32_t *body, const float *point3,
                          const float *force3);

/* Upload wrenches applied since the last ob_step / ob_flush now (asynchronous; ob_step does it implicitly). */
int ob_flush(ob_ctx *ctx);

/* Advance every world by n steps (one persistent kernel launch per size class; worlds stay on chip for the
   n steps).  Asynchronous.  Events are appended to the device event list. */
int ob_step(ob_ctx *ctx, int n);

/* Copy one world's state out (synchronises).  Any output pointer may be NULL.
   q, qd: [2*n_links] (theta_1, theta_2 per link); apple_x, apple_v: [3*n_apples] world frame;
   ruptured: [n_links]; attached: [n_apples]; link_pose7: [7*n_links] (x,y,z, qw,qx,qy,qz) of each link frame;
   info: [3] = step, PCG iterations of the last step, status bits (OB_STATUS_*). */
int ob_get_state(ob_ctx *ctx, int world, float *q, float *qd, float *apple_x, float *apple_v, uint8_t *ruptured,
                 uint8_t *attached, float *link_pose7, int32_t *info);
/* Overwrite one world's state (NULL = keep).  Setting `ruptured` / `attached` also clears the corresponding
   hysteresis counters; the PCG warm start of the world is cleared.  Status bits are cleared. */
int ob_set_state(ob_ctx *ctx, int world, const float *q, const float *qd, const float *apple_x,
                 const float *apple_v, const uint8_t *ruptured, const uint8_t *attached);
/* Apple positions at the library's internal precision: anchor (fp64 rest hang point) + fp32 displacement.
   apple_x: [3*n_apples] doubles.  ob_get_state's float apple_x is this value rounded to fp32. */
int ob_get_apple_x64(ob_ctx *ctx, int world, double *apple_x);
/* Hysteresis counters (rupture per link; detach pull / tension per apple), for lock-step comparison. */
int ob_get_counters(ob_ctx *ctx, int world, int32_t *rupture_count, int32_t *pull_count, int32_t *tension_count);
int ob_set_counters(ob_ctx *ctx, int world, const int32_t *rupture_count, const int32_t *pull_count,
                    const int32_t *tension_count);
/* Per-world material draws: emr[3] = E, MOR, density; apple_detach, apple_mass: [n_apples] (NULL ok). */
int ob_get_material(ob_ctx *ctx, int world, float *emr, float *apple_detach, float *apple_mass);

/* Drain up to cap pending events, sorted by (step, world, kind, index).  Synchronises.
   If the device list overflowed since the last drain, returns OB_E_CAPACITY after filling buf. */
int ob_events(ob_ctx *ctx, ob_event *buf, int cap, int *n_out);

/* Totals since ob_create: PCG iterations, world-steps taken (frozen worlds excluded), worlds with status != 0. */
int ob_stats(ob_ctx *ctx, uint64_t *cg_iters_total, uint64_t *world_steps_total, int32_t *n_flagged);

/* Launch geometry of the last ob_step (for reporting): kernel launches, CTAs, threads per CTA, dynamic smem. */
int ob_launch_info(ob_ctx *ctx, int32_t *n_launches, int32_t *grid, int32_t *block, int32_t *smem_bytes);

/* Cumulative counters since ob_create: out[0] = bytes the library copied host -> device, out[1] = device -> host,
   out[2] = kernels it launched, out[3] = ob_step calls.  Host-side bookkeeping; does not synchronise. */
int ob_counters(ob_ctx *ctx, uint64_t out[4]);

/* sizeof of the three ABI structs as the library was compiled (bindings check their own layout against these). */
int ob_sizeof_params(void);
int ob_sizeof_world_spec(void);
int ob_sizeof_event(void);

/* Self-test of the device Philox4x32-10 (reading A23) against NVIDIA's own implementation: for n (counter, key)
   pairs computes the library's generator and cuRAND's curand_Philox4x32_10 on the device.  ctr: [4*n], key: [2*n],
   out_lib / out_curand: [4*n] host arrays; dev_scratch: caller-provided device memory of >= 56*n bytes; the work is
   enqueued on cuda_stream and the call synchronises it.  No context needed.  Returns OB_E_ARG / OB_E_CUDA. */
int ob_selftest_philox(int n, const uint32_t *ctr, const uint32_t *key, uint32_t *out_lib, uint32_t *out_curand,
                       void *dev_scratch, void *cuda_stream);

const char *ob_last_error(const ob_ctx *ctx);
void ob_destroy(ob_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* ORCHARD_H_ */
