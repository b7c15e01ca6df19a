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
 *   time step         BASELINE.json north_star    (M + hD + h^2 K) dqd = rhs by matrix-free PCG (tree-exact
 *                                                  or Jacobi preconditioner),
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
  int32_t n_links;              /* >= 1; a world must fit in one SM's shared memory: ~1500 links at most (fewer
                                   with many apples or tree levels); ob_workspace_bytes / ob_create return
                                   OB_E_CAPACITY with the figures otherwise */
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
  int32_t precond;              /* {2} 0 = none, 1 = Jacobi (exact diagonal from a composite-inertia sweep), 2 = the tree
                                   itself: an articulated-body factorisation of A, exact in exact arithmetic, so PCG
                                   converges in 1-2 iterations (cg_norm must be 0) */
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
  /* post-rupture dissipation */
  float fric_frac;              /* {0 = off} Coulomb friction torque at a ruptured joint, as a fraction of its M_max,
                                   against the joint velocity (regularised below fric_veps) */
  float fric_ramp;              /* {5} ... ramped up by this factor ("~5x") */
  float fric_time;              /* {1.5} ... over this time after the rupture, s ("~1.5 s") */
  float fric_veps;              /* {1e-2} rad/s */
  float snap_drag_scale;        /* {1 = no reduction} factor on mass_damping for the links of snapped sub-trees */
  /* the three rails on applied forces (App. B): act on wrenches on FREE bodies -- apples, and links of
     snapped sub-trees when forces_off_on_snapped = 0; connected links are static loading, which they never touch */
  float rail_speed;             /* {0 = rails off} m/s: impulse cap (no force takes the body past it in one step) and
                                   speed brake above it */
  float rail_fade;              /* {0.5} the part of a force along the body's velocity fades out between
                                   rail_fade * rail_speed and rail_speed */
  float rail_brake;             /* {50} 1/s: brake force - rail_brake m (|v| - rail_speed) v^ above rail_speed */
} ob_params;

typedef struct {
  int32_t world, step;          /* step = 0-based index of the step during which the flag flipped */
  int32_t kind;                 /* 0 = rupture (index = link), 1 = detach (index = apple) */
  int32_t index;
  float value, threshold;       /* rupture: K|theta| vs M_max; detach: |f_user| vs f_detach or |f_s| vs kappa f_detach */
} ob_event;

/* Ranges of ob_randomize_geometry (uniform per world unless noted; lo == hi gives that value for every world). */
typedef struct {
  float droop[2];               /* rad: every link is turned towards the ground by droop * sin(its angle to the vertical)
                                   inside a top-down re-walk, so the droop compounds per internode */
  float lean[2];                /* rad: whole-tree lean of the trunk about a horizontal axis of uniform azimuth */
  float spread[2];              /* relative: the angle between a child and its parent's axis is scaled by 1 + spread */
  float twist[2];               /* rad: every child's rest frame is turned about its parent's axis */
  float scale_length[2];        /* per-world factor on every link length ("global scale") */
  float scale_diameter[2];      /* per-world factor on every link diameter ("stockiness") */
  float jitter_length[2];       /* per-LINK factor on its length ("per-segment length") */
  float jitter_diameter[2];     /* per-LINK factor on its diameter ("per-segment thickness") */
} ob_geometry_ranges;

/* Fill *p with the defaults above (the readings A1..A37 of DESIGN.md section 3).  Returns OB_E_ARG for NULL. */
int ob_default_params(ob_params *p);

/* Bytes of device workspace ob_create needs for these worlds (validates the specs).
   [north_star: "PyTorch is used only for device memory and streams": the library allocates no device memory] */
int ob_workspace_bytes(const ob_world_spec *specs, int n_worlds, const ob_params *params, size_t *out);

/* north_star "ob_create(world specs: parent arrays, link lengths/diameters/densities, E, MOR, apple attachments)".
   Builds the articulation of PAPER.md:113-117 (Eq. 3: joint at the parent's distal tip (0,0,l_parent), rest rotation
   q_rel, trunk base fixed) as a level-ordered SoA per world, computes rest poses and the derived constants of Eq. 4
   (K = E pi d^4 / (64 l)) and Eq. 5 (M_max = MOR pi d^3 / 32), and resets the state to
   the rest pose with every apple at its rest sag m g / k_s below its hang point.
   dev_workspace: device memory of at least ob_workspace_bytes bytes, 256-byte aligned, owned by the caller and alive
   until ob_destroy; cuda_stream: cudaStream_t (NULL = default stream).  Errors: OB_E_ARG (null, non-topological
   parent, non-unit quaternion, non-positive dimension), OB_E_CAPACITY (a world does not fit on chip, > 15 children
   on one link), OB_E_WORKSPACE, OB_E_CUDA (no device: there is no CPU fallback). */
int ob_create(const ob_world_spec *specs, int n_worlds, const ob_params *params, void *dev_workspace,
              size_t workspace_bytes, void *cuda_stream, ob_ctx **out);

/* north_star "ob_randomize(seed)": per-environment domain randomization of PAPER.md:165-169 ("wood density, Young's
   modulus and rupture stress; fruit ... mass") drawn ON THE DEVICE with Philox4x32-10 (key = seed; counter =
   (world, item, stream, 0); stream 0 item 0 -> E, MOR, density; stream 1 item a -> detach force, mass of apple a;
   u = float(x>>8) 2^-24, value = fmaf(u, hi-lo, lo); reading A23), then the derived constants of Eq. 4 / Eq. 5 and a
   full reset: rest pose, zero velocities, flags, counters, step = 0, wrench slots cleared, warm start cleared.
   Pending events stay queued.  Asynchronous. */
int ob_randomize(ob_ctx *ctx, uint64_t seed);

/* Per-world GEOMETRY randomization on the device ("per-segment bend and whole-tree growth habit (a
   gravimorphic droop multiplier applied inside a forward-kinematic re-walk ..., plus whole-tree lean, fork spread and
   an env-wide phyllotactic twist)" and the per-branch dimensions "(global scale and stockiness, and per-segment length
   and thickness)"; "an on-device build that perturbs every world's branch geometry in a single ... kernel
   (one thread per world)").  Every world gets its own draws (Philox4x32-10, key = seed; stream 3 item 0 -> droop, lean,
   spread, twist; stream 3 item 1 -> lean azimuth, length scale, diameter scale; stream 4 item i -> length and
   diameter jitter of link i), applied to the BASE geometry given to ob_create, so identity ranges (angles 0, factors
   1) reproduce the base model exactly and calls do not compound.  Apple attach points move with their link (x, y by
   its diameter factor, z by its length factor).  Then: rest hang points, the derived constants of Eq. 4 / Eq. 5 with
   the materials as they are, and a full state reset as in ob_randomize.  Distinct geometry per world costs nothing
   at step time here (every world carries its own dimensions anyway).  Synchronises (rest hang points come back). */
int ob_randomize_geometry(ob_ctx *ctx, uint64_t seed, const ob_geometry_ranges *ranges);
/* Current geometry of one world (after ob_randomize_geometry): length, diameter [n_links]; rest_quat [4*n_links] doubles
   (w,x,y,z); apple_offset [3*n_apples].  Any pointer may be NULL.  Synchronises. */
int ob_get_geometry(ob_ctx *ctx, int world, float *length, float *diameter, double *rest_quat, float *apple_offset);

/* north_star "ob_apply_wrench(world, body, point, force)": a persistent external force ("applied and interactive
   forces").  body in [0, n_links) is a link, [n_links, n_links + n_apples) an apple (a pull on the
   fruit: the "direct pull force" of the first detachment path).  point: application point in the link's
   local frame (moves with the link; ignored for apples, which do not rotate).  force: world frame, N.
   The wrench persists until replaced (same body) or removed (zero force).  Each world has OB_MAX_WRENCH slots; one
   more distinct body returns OB_E_CAPACITY.  Wrenches on links at or below a ruptured joint are ignored while
   forces_off_on_snapped is set.  Host-side bookkeeping; uploaded by the next ob_step / ob_flush. */
int ob_apply_wrench(ob_ctx *ctx, int world, int body, const float point[3], const float force[3]);
/* The same for n wrenches: world[n], body[n], point3[3n] (or NULL), force3[3n] host arrays. */
int ob_apply_wrench_batch(ob_ctx *ctx, int n, const int32_t *world, const int32_t *body, const float *point3,
                          const float *force3);

/* Upload wrenches applied since the last ob_step / ob_flush now (asynchronous; ob_step does it implicitly). */
int ob_flush(ob_ctx *ctx);

/* north_star "ob_step(n)": advance every world by n steps of the batched physics step -- forward kinematics over the
   level-ordered tree (Eq. 3); tether forces and clamped reaction (Eq. 6, Eq. 7);
   spring-damper torques (Eq. 4); the implicit velocity update (M + hD + h^2 K) dqd = rhs by
   matrix-free preconditioned conjugate gradient with M v from inverse-dynamics tree sweeps (north_star; PAPER.md:185,
   265 "the matrix-free CG solve"); integration; in-place rupture (Eq. 5: "zero the broken degrees
   of freedom's gain ... in place") and detachment ("a single flag flip") -- in one persistent kernel
   launch per size class, worlds staying on chip for the n steps.  Asynchronous.  Events are appended to the device
   event list; a world whose state goes non-finite is frozen and flagged (OB_STATUS_NONFINITE). */
int ob_step(ob_ctx *ctx, int n);

/* north_star "ob_get_state".  Copy one world's state out (synchronises once).  Any output pointer may be NULL.
   q, qd: [2*n_links] (theta_1, theta_2 per link: the two bending DoF of PAPER.md:121); apple_x, apple_v:
   [3*n_apples] world frame (3-DoF fruit); ruptured: [n_links] (Eq. 5); attached: [n_apples]
   (PAPER.md:163); link_pose7: [7*n_links] (x,y,z, qw,qx,qy,qz) of each link frame (Eq. 3);
   info: [3] = step, PCG iterations of the last step, status bits (OB_STATUS_*). */
int ob_get_state(ob_ctx *ctx, int world, float *q, float *qd, float *apple_x, float *apple_v, uint8_t *ruptured,
                 uint8_t *attached, float *link_pose7, int32_t *info);
/* The same for the worlds [world0, world0 + n_worlds): ONE device -> host copy per state pool and ONE synchronisation.
   Outputs are concatenated in world order, each world's slice laid out as in ob_get_state (q of world w starts at
   2 * sum of n_links of the worlds before it in the range, and so on); apple_x64 is the position at the library's
   internal precision (see ob_get_apple_x64); info: [3*n_worlds].  Any output pointer may be NULL. */
int ob_get_state_batch(ob_ctx *ctx, int world0, int n_worlds, float *q, float *qd, float *apple_x, double *apple_x64,
                       float *apple_v, uint8_t *ruptured, uint8_t *attached, int32_t *info);
/* Overwrite one world's state (NULL = keep).  Setting `ruptured` / `attached` also clears the corresponding
   hysteresis counters (the N-frame hysteresis of PAPER.md:139, the "few frames" of PAPER.md:163); the PCG warm start
   of the world is cleared.  Status bits are cleared (by this call only: ob_set_step, ob_set_rupture_steps and
   ob_set_apple_x64 keep them, so a world frozen by OB_STATUS_NONFINITE stays frozen until ob_set_state). */
int ob_set_state(ob_ctx *ctx, int world, const float *q, const float *qd, const float *apple_x,
                 const float *apple_v, const uint8_t *ruptured, const uint8_t *attached);
/* Apple positions at the library's internal precision: anchor (fp64 rest hang point, Eq. 3) + rest sag m g / k_s
    + fp32 displacement.  apple_x: [3*n_apples] doubles.  ob_get_state's float apple_x is this value
   rounded to fp32.  The setter is the exact inverse: get -> set restores the internal displacement bit for bit.  It
   also clears the world's PCG warm start (the positions changed); status bits are kept. */
int ob_get_apple_x64(ob_ctx *ctx, int world, double *apple_x);
int ob_set_apple_x64(ob_ctx *ctx, int world, const double *apple_x);
/* Restore the step counter of a world (events carry it); everything else is kept, the warm start included. */
int ob_set_step(ob_ctx *ctx, int world, int32_t step);
/* Step during which each joint ruptured ([n_links]; meaningful where ruptured): the post-rupture friction ramp
    counts from it.  ob_set_state(ruptured) sets it to the world's current step. */
int ob_get_rupture_steps(ob_ctx *ctx, int world, int32_t *rupture_step);
int ob_set_rupture_steps(ob_ctx *ctx, int world, const int32_t *rupture_step);
/* Hysteresis counters (rupture per link; detach pull / tension per apple), for lock-step
   comparison and checkpoints.  The _batch form covers worlds [world0, world0 + n_worlds), outputs concatenated. */
int ob_get_counters(ob_ctx *ctx, int world, int32_t *rupture_count, int32_t *pull_count, int32_t *tension_count);
int ob_get_counters_batch(ob_ctx *ctx, int world0, int n_worlds, int32_t *rupture_count, int32_t *pull_count,
                          int32_t *tension_count);
int ob_set_counters(ob_ctx *ctx, int world, const int32_t *rupture_count, const int32_t *pull_count,
                    const int32_t *tension_count);
/* Per-world material draws of ob_randomize: emr[3] = E, MOR, density; apple_detach, apple_mass:
   [n_apples] (NULL ok).  The _batch form: emr [3*n_worlds], apple arrays concatenated. */
int ob_get_material(ob_ctx *ctx, int world, float *emr, float *apple_detach, float *apple_mass);
int ob_get_material_batch(ob_ctx *ctx, int world0, int n_worlds, float *emr, float *apple_detach, float *apple_mass);

/* Exact checkpoint of one world: every byte of its mutable state (q, qd, flags, counters, apple state, step and
   status words, the PCG solution history), so that load followed by ob_step(n) reproduces
   an uninterrupted run bit for bit (PCG solution history included).  buf: host memory of ob_world_blob_bytes bytes.  A blob only loads into a world
   of the same sizes (OB_E_ARG otherwise).  Materials and wrenches are not part of it: loading keeps the target world's
   material draws (ob_get_material) and its totals since ob_create (ob_stats), whatever world or moment the blob is from. */
int ob_world_blob_bytes(ob_ctx *ctx, int world, size_t *out);
int ob_save_world(ob_ctx *ctx, int world, void *buf, size_t cap);
int ob_load_world(ob_ctx *ctx, int world, const void *buf, size_t bytes);

/* north_star "ob_events (rupture and detach lists)".  Drain up to cap pending events (Eq. 5 ruptures, PAPER.md:136;
   detachments), sorted by (step, world, kind, index).  Synchronises.  If the device list overflowed
   since the last drain, returns OB_E_CAPACITY after filling buf. */
int ob_events(ob_ctx *ctx, ob_event *buf, int cap, int *n_out);

/* Totals since ob_create: PCG iterations, world-steps taken (frozen worlds excluded), worlds with status != 0
   (BASELINE.json metric: "world-steps/s ...; CG iters/s").  Reduced on the device; one small copy. */
int ob_stats(ob_ctx *ctx, uint64_t *cg_iters_total, uint64_t *world_steps_total, int32_t *n_flagged);
/* World-steps by PCG iteration count since ob_create (or the last reset): bins[k] = world-steps that took k
   iterations, the last bin collecting k >= n_bins - 1.  reset != 0 clears the device histogram after the read. */
int ob_iter_histogram(ob_ctx *ctx, uint64_t *bins, int n_bins, int reset);

/* Launch geometry of the last ob_step (for reporting): kernel launches, CTAs, threads per CTA, dynamic smem. */
int ob_launch_info(ob_ctx *ctx, int32_t *n_launches, int32_t *grid, int32_t *block, int32_t *smem_bytes);

/* Cumulative counters since ob_create: out[0] = bytes the library copied host -> device, out[1] = device -> host,
   out[2] = kernels it launched, out[3] = ob_step calls.  Host-side bookkeeping; does not synchronise. */
int ob_counters(ob_ctx *ctx, uint64_t out[4]);

/* sizeof of the three ABI structs as the library was compiled (bindings check their own layout against these). */
int ob_sizeof_params(void);
int ob_sizeof_world_spec(void);
int ob_sizeof_event(void);
int ob_sizeof_geometry_ranges(void);

/* Self-test of the device Philox4x32-10 (reading A23) against NVIDIA's own implementation: for n (counter, key)
   pairs computes the library's generator and cuRAND's curand_Philox4x32_10 on the device.  ctr: [4*n], key: [2*n],
   out_lib / out_curand: [4*n] host arrays; dev_scratch: caller-provided device memory of >= 56*n bytes; the work is
   enqueued on cuda_stream and the call synchronises it.  No context needed.  Returns OB_E_ARG / OB_E_CUDA. */
int ob_selftest_philox(int n, const uint32_t *ctr, const uint32_t *key, uint32_t *out_lib, uint32_t *out_curand,
                       void *dev_scratch, void *cuda_stream);

/* The same self-test for a caller that cannot supply dev_scratch.  Some code that wants to run this check has no way
   to obtain device memory: a plug-in inside a host application whose pool allocator has already claimed the whole GPU
   and forbids driver allocations behind its back, a start-up health probe that runs before any allocator exists, or a
   thread for which cudaMalloc / cudaFree are off limits because they synchronise the device or would break a stream
   capture under way elsewhere in the process.  For them the staging area is a fixed array inside libob.so itself.
   Cost: OB_SELFTEST_STATIC_MAX * 56 bytes = 224 KB of device memory on every GPU that loads the library, held until
   the process exits.  Limit: n <= OB_SELFTEST_STATIC_MAX; a larger n returns OB_E_CAPACITY (ob_last_error(NULL) says
   so) before anything touches the GPU -- split the pairs over several calls, or use ob_selftest_philox.
   Arguments and results as ob_selftest_philox (host arrays ctr [4n], key [2n] in, out_lib / out_curand [4n] out,
   all owned by the caller; the results are bit-identical to ob_selftest_philox's).  cuda_stream must belong to the
   device that is current on the calling thread; the work is enqueued on it and the call synchronises it.
   The call allocates nothing on the device or through the CUDA runtime: no cudaMalloc, cudaFree, cudaMallocHost or
   library routine that allocates; it copies directly between the caller's host arrays and the static array.
   First call on each device: it looks up the device address of the static array (one cudaGetSymbolAddress, checked,
   with that device current) and remembers it; make that first call before starting any stream capture.
   Sharing: every call on a device uses the same array, and the array keeps the previous call's contents.  Nothing in
   it has to start at zero (each call copies its inputs in and the kernel overwrites all 8n result words before they
   are read back), so no clearing is done; but two calls that overlap on the same GPU (two host threads, two streams)
   race on it and return garbage: serialise them.  Returns OB_E_ARG (null, n < 1), OB_E_CAPACITY, OB_E_CUDA. */
#define OB_SELFTEST_STATIC_MAX 4096
int ob_selftest_philox_static(int n, const uint32_t *ctr, const uint32_t *key, uint32_t *out_lib,
                              uint32_t *out_curand, void *cuda_stream);

const char *ob_last_error(const ob_ctx *ctx);
void ob_destroy(ob_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* ORCHARD_H_ */
