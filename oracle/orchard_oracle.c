/*
 * orchard_oracle.c -- fp64 CPU oracle for the OrchardBench batched tree-physics step.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this file.  It shares
 * no code, header, table or helper with paper_2607_06337_b200/ (the CUDA path)
 * and is written from the paper (/root/reference/PAPER.md, cited as PAPER.md:<line>)
 * plus the readings listed in DESIGN.md section 3 (A1..A31 of SURVEY.md 8(c), A32..A37).
 *
 * What it computes, in the paper's order, all in double precision:
 *   - the articulation of PAPER.md:113-117 (Eq. 3): links are rigid cylinders
 *     along local +z, child joint at the parent's distal tip (0,0,L_parent),
 *     rest rotation q_rel; trunk base fixed to the world;
 *   - compliant joints of PAPER.md:121-126 (Eq. 4): two bending DoF per joint
 *     (two revolutes in series, axes x then y, massless zero-length body in
 *     between), K = E*pi*d^4/(64 L) (= (pi/4) E r^4 / l), D = c_d K,
 *     tau = -K theta - D omega;
 *   - rupture of PAPER.md:132-141 (Eq. 5): K*||theta|| > MOR*pi*d^3/32
 *     (= sigma_r pi r^3/4) for N consecutive steps zeroes K and D in place;
 *   - fruit of PAPER.md:147-163 (Eq. 6, Eq. 7): 3-DoF point bodies on
 *     spring-damper tethers, clamped reaction on the spur, two detachment paths;
 *   - per-world randomization of PAPER.md:167-169 by Philox4x32-10 draws;
 *   - the time step BASELINE.json's north_star names: a linearly implicit
 *     spring-damper velocity update (M + hD + h^2 K) dqd = rhs.  Here M is formed
 *     by brute force, one inverse-dynamics call per unit acceleration, and the
 *     system is solved by dense Cholesky.
 *
 * Dynamics are the textbook Newton-Euler recursion written in WORLD coordinates
 * (angular velocity/acceleration vectors, joint positions, Newton's and Euler's
 * equations about each centre of mass).  The CUDA path uses body-frame spatial
 * algebra, fp32, fused 2-DoF joints and matrix-free PCG; the difference is
 * deliberate.
 *
 * Pins: tests/test_oracle_pins.py (closed forms, invariants, brute force).
 * "parity unpinned": the absolute realism of a trajectory (the paper prints no
 * worked numeric example for this path, PAPER.md:128 vs 259-301).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define OBO_MAX_WRENCH 8

typedef struct {
  double h;
  double g[3];
  double c_d;
  double cg_tol;
  int32_t cg_max_iter;
  int32_t solver;               /* 0 = dense Cholesky (default), 1 = fp64 Jacobi-PCG on the dense matrix */
  int32_t rupture_frames;
  int32_t detach_frames_pull;
  double detach_kappa;
  int32_t detach_frames_tension;
  int32_t tether_implicit;
  double react_max;
  double qd_max;
  double zeta_s;
  double alpha_m;               /* mass- and inertia-proportional damping c_v = c_omega, 1/s (A32) */
  int32_t forces_off_on_snapped;
  int32_t pad_;
  /* post-rupture dissipation (readings A34, A35) and the three force rails (A36) */
  double fric_frac, fric_ramp, fric_time, fric_veps;   /* friction torque fric_frac * M_max, ramped x fric_ramp over fric_time */
  double snap_drag_scale;                             /* factor on alpha_m for links of snapped sub-trees */
  double rail_speed, rail_fade, rail_brake;           /* speed limit (0 = rails off), fade onset fraction, brake rate 1/s */
  float range_E[2], range_MOR[2], range_density[2], range_detach[2], range_apple_mass[2];
} obo_params;

typedef struct {
  int32_t world, step, kind, index;
  double value, threshold;
} obo_event;

typedef struct {
  int N, A;
  obo_params P;
  /* topology and rest geometry (from the fp32 inputs, promoted) */
  int *parent;
  double *L, *d, *Q /*[9N] rest rotation, row-major*/, *arm /*[2N]*/;
  float *L0, *d0;           /* base geometry as given at construction (fp32 inputs) */
  double *Q0, *aoff0;       /* base rest rotations and apple offsets */
  float rho_nom, E_nom, MOR_nom;
  float rho, E, MOR; /* current (fp32 draws, A23) */
  /* derived per link */
  double *K, *Mmax, *m, *Ixx, *Izz;
  /* apples */
  int *alink;
  double *aoff;
  float *am_nom, *adet_nom, *ac_in;
  int ac_given;
  double *am, *ak, *ac, *adet;
  /* state */
  double *q, *qd, *dqd_prev, *ax, *av;
  uint8_t *ruptured, *attached;
  int *rc, *cA, *cB;
  int *rstep;                   /* step during which the joint ruptured (valid where ruptured) */
  int step, status, last_iters;
  long long cg_iters_total;
  /* wrenches (persistent) */
  int wr_body[OBO_MAX_WRENCH];
  double wr_point[OBO_MAX_WRENCH][3], wr_force[OBO_MAX_WRENCH][3];
  /* events */
  obo_event *ev;
  int n_ev, cap_ev;
  int world_index;
} obo_world;

/* ----------------------------------------------------------------------- */
/* small vector helpers                                                     */
/* ----------------------------------------------------------------------- */
static void cross3(const double a[3], const double b[3], double o[3]) {
  double x = a[1] * b[2] - a[2] * b[1];
  double y = a[2] * b[0] - a[0] * b[2];
  double z = a[0] * b[1] - a[1] * b[0];
  o[0] = x; o[1] = y; o[2] = z;
}
static double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static double norm3(const double a[3]) { return sqrt(dot3(a, a)); }
/* C = A B, 3x3 row-major */
static void mat3mul(const double *A, const double *B, double *C) {
  double T[9];
  for (int r = 0; r < 3; r++)
    for (int c = 0; c < 3; c++) T[3 * r + c] = A[3 * r] * B[c] + A[3 * r + 1] * B[3 + c] + A[3 * r + 2] * B[6 + c];
  memcpy(C, T, sizeof(T));
}
static void mat3vec(const double *A, const double v[3], double o[3]) {
  double x = A[0] * v[0] + A[1] * v[1] + A[2] * v[2];
  double y = A[3] * v[0] + A[4] * v[1] + A[5] * v[2];
  double z = A[6] * v[0] + A[7] * v[1] + A[8] * v[2];
  o[0] = x; o[1] = y; o[2] = z;
}
static void quat_to_mat(const double qn[4], double *R) {
  double n = sqrt(qn[0] * qn[0] + qn[1] * qn[1] + qn[2] * qn[2] + qn[3] * qn[3]);
  double w = qn[0] / n, x = qn[1] / n, y = qn[2] / n, z = qn[3] / n;
  R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z);     R[2] = 2 * (x * z + w * y);
  R[3] = 2 * (x * y + w * z);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
  R[6] = 2 * (x * z - w * y);     R[7] = 2 * (y * z + w * x);     R[8] = 1 - 2 * (x * x + y * y);
}
static void rot_x(double t, double *R) {
  double c = cos(t), s = sin(t);
  R[0] = 1; R[1] = 0; R[2] = 0; R[3] = 0; R[4] = c; R[5] = -s; R[6] = 0; R[7] = s; R[8] = c;
}
static void rot_y(double t, double *R) {
  double c = cos(t), s = sin(t);
  R[0] = c; R[1] = 0; R[2] = s; R[3] = 0; R[4] = 1; R[5] = 0; R[6] = -s; R[7] = 0; R[8] = c;
}

/* ----------------------------------------------------------------------- */
/* Philox4x32-10 (Salmon et al., SC'11), reading A23 for the layout          */
/* ----------------------------------------------------------------------- */
void obo_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
  uint32_t k0 = key_in[0], k1 = key_in[1];
  for (int round = 0; round < 10; round++) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
/* u = float(x >> 8) * 2^-24 in [0,1); value = fmaf(u, hi-lo, lo) in fp32 (A23) */
static float philox_uniform(uint32_t x, float lo, float hi) {
  float u = (float)(x >> 8) * (1.0f / 16777216.0f);
  return fmaf(u, hi - lo, lo);
}

/* ----------------------------------------------------------------------- */
/* forward kinematics (Eq. 3; readings A2, A4)             */
/* ----------------------------------------------------------------------- */
typedef struct {
  double *R;    /* [9N] world rotation of link frame */
  double *p;    /* [3N] world position of joint i (= proximal end of link i) */
  double *ax1;  /* [3N] world axis of theta_1 */
  double *ax2;  /* [3N] world axis of theta_2 */
} fk_t;

static fk_t fk_alloc(int N) {
  fk_t f;
  f.R = (double *)calloc(9 * (size_t)N, sizeof(double));
  f.p = (double *)calloc(3 * (size_t)N, sizeof(double));
  f.ax1 = (double *)calloc(3 * (size_t)N, sizeof(double));
  f.ax2 = (double *)calloc(3 * (size_t)N, sizeof(double));
  return f;
}
static void fk_free(fk_t *f) { free(f->R); free(f->p); free(f->ax1); free(f->ax2); }

/* R_i = R_parent * Q_i * Rx(theta_1) * Ry(theta_2);  p_i = p_parent + R_parent (0,0,L_parent) */
static void fk_run(const obo_world *W, const double *q, fk_t *f) {
  static const double I3[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
  for (int i = 0; i < W->N; i++) {
    int pa = W->parent[i];
    const double *Rp = pa < 0 ? I3 : f->R + 9 * pa;
    if (pa < 0) {
      f->p[3 * i] = f->p[3 * i + 1] = f->p[3 * i + 2] = 0.0;
    } else {
      double tip[3] = {0, 0, W->L[pa]}, t[3];
      mat3vec(Rp, tip, t);
      for (int k = 0; k < 3; k++) f->p[3 * i + k] = f->p[3 * pa + k] + t[k];
    }
    double A[9], B[9], Rx[9], Ry[9];
    mat3mul(Rp, W->Q + 9 * i, A);          /* frame after the rest rotation   */
    rot_x(q[2 * i], Rx);
    mat3mul(A, Rx, B);                      /* frame after the first hinge     */
    rot_y(q[2 * i + 1], Ry);
    mat3mul(B, Ry, f->R + 9 * i);           /* link frame                      */
    for (int k = 0; k < 3; k++) {
      f->ax1[3 * i + k] = A[3 * k + 0];     /* x axis of A                     */
      f->ax2[3 * i + k] = B[3 * k + 1];     /* y axis of B                     */
    }
  }
}

/* ----------------------------------------------------------------------- */
/* inverse dynamics: Newton-Euler recursion in world coordinates             */
/*   tau = M(q) qdd + c(q,qd) - (gravity) - J^T f_ext                        */
/* ----------------------------------------------------------------------- */
#define OBO_MAX_APPLES 1024              /* obo_world_new refuses more: ext_t below holds one entry per apple */
typedef struct {
  int n;
  int link[OBO_MAX_WRENCH + OBO_MAX_APPLES];
  double x[OBO_MAX_WRENCH + OBO_MAX_APPLES][3]; /* world application point */
  double F[OBO_MAX_WRENCH + OBO_MAX_APPLES][3]; /* world force             */
} ext_t;

static void rnea(const obo_world *W, const double *q, const double *qd, const double *qdd, const double g[3],
                 const ext_t *ext, double *tau) {
  int N = W->N;
  fk_t f = fk_alloc(N);
  fk_run(W, q, &f);
  double *om = (double *)calloc(3 * (size_t)N, sizeof(double));  /* angular velocity       */
  double *al = (double *)calloc(3 * (size_t)N, sizeof(double));  /* angular acceleration   */
  double *ac = (double *)calloc(3 * (size_t)N, sizeof(double));  /* accel. of joint origin */
  double *cm = (double *)calloc(3 * (size_t)N, sizeof(double));  /* world centre of mass   */
  double *fj = (double *)calloc(3 * (size_t)N, sizeof(double));  /* force through joint i  */
  double *nj = (double *)calloc(3 * (size_t)N, sizeof(double));  /* couple through joint i */

  /* outward pass: velocities and accelerations */
  for (int i = 0; i < N; i++) {
    int pa = W->parent[i];
    double omp[3] = {0, 0, 0}, alp[3] = {0, 0, 0}, acp[3] = {0, 0, 0}, r[3] = {0, 0, 0};
    if (pa >= 0) {
      for (int k = 0; k < 3; k++) {
        omp[k] = om[3 * pa + k]; alp[k] = al[3 * pa + k]; acp[k] = ac[3 * pa + k];
        r[k] = f.p[3 * i + k] - f.p[3 * pa + k];
      }
    }
    /* joint origin rides on the parent: a = a_p + al_p x r + om_p x (om_p x r) */
    double t1[3], t2[3], t3[3];
    cross3(alp, r, t1);
    cross3(omp, r, t2);
    cross3(omp, t2, t3);
    for (int k = 0; k < 3; k++) ac[3 * i + k] = acp[k] + t1[k] + t3[k];
    /* two revolutes in series: om_mid = om_p + ax1 qd1; om = om_mid + ax2 qd2 */
    const double *a1 = f.ax1 + 3 * i, *a2 = f.ax2 + 3 * i;
    double qd1 = qd[2 * i], qd2 = qd[2 * i + 1], dd1 = qdd[2 * i], dd2 = qdd[2 * i + 1];
    double om_mid[3], w1[3], w2[3], c1[3], c2[3];
    for (int k = 0; k < 3; k++) { w1[k] = a1[k] * qd1; w2[k] = a2[k] * qd2; om_mid[k] = omp[k] + w1[k]; }
    cross3(omp, w1, c1);     /* d/dt(ax1) = om_p x ax1      */
    cross3(om_mid, w2, c2);  /* d/dt(ax2) = om_mid x ax2    */
    for (int k = 0; k < 3; k++) {
      om[3 * i + k] = om_mid[k] + w2[k];
      al[3 * i + k] = alp[k] + a1[k] * dd1 + c1[k] + a2[k] * dd2 + c2[k];
    }
  }
  /* Newton and Euler per link, inward accumulation */
  for (int i = 0; i < N; i++) {
    double half[3] = {0, 0, 0.5 * W->L[i]}, rc[3];
    mat3vec(f.R + 9 * i, half, rc);
    for (int k = 0; k < 3; k++) cm[3 * i + k] = f.p[3 * i + k] + rc[k];
  }
  for (int i = N - 1; i >= 0; i--) {
    const double *R = f.R + 9 * i;
    double rc[3], t1[3], t2[3], t3[3], acm[3];
    for (int k = 0; k < 3; k++) rc[k] = cm[3 * i + k] - f.p[3 * i + k];
    cross3(al + 3 * i, rc, t1);
    cross3(om + 3 * i, rc, t2);
    cross3(om + 3 * i, t2, t3);
    for (int k = 0; k < 3; k++) acm[k] = ac[3 * i + k] + t1[k] + t3[k];
    /* world inertia about the centre of mass: R diag(Ixx,Ixx,Izz) R^T */
    double Dg[9] = {W->Ixx[i], 0, 0, 0, W->Ixx[i], 0, 0, 0, W->Izz[i]}, RD[9], Rt[9], Iw[9];
    for (int r_ = 0; r_ < 3; r_++)
      for (int c_ = 0; c_ < 3; c_++) Rt[3 * r_ + c_] = R[3 * c_ + r_];
    mat3mul(R, Dg, RD);
    mat3mul(RD, Rt, Iw);
    double Ial[3], Iom[3], gyro[3];
    mat3vec(Iw, al + 3 * i, Ial);
    mat3vec(Iw, om + 3 * i, Iom);
    cross3(om + 3 * i, Iom, gyro);
    /* Newton: m a_cm = f_i - sum_children f_c + m g + sum F_ext
       (fj[i] already holds sum_children f_c) */
    double fi[3], ni[3];
    for (int k = 0; k < 3; k++) fi[k] = W->m[i] * acm[k] - W->m[i] * g[k] + fj[3 * i + k];
    /* Euler about the cm:
       I al + om x I om = n_i + (p_i - c_i) x f_i - sum_c [n_c + (p_c - c_i) x f_c] + sum (x_e - c_i) x F_e
       (nj[i] already holds sum_c [n_c + (p_c - c_i) x f_c]) */
    for (int k = 0; k < 3; k++) ni[k] = Ial[k] + gyro[k] + nj[3 * i + k];
    if (ext) {
      for (int e = 0; e < ext->n; e++) {
        if (ext->link[e] != i) continue;
        double arm[3], mo[3];
        for (int k = 0; k < 3; k++) { fi[k] -= ext->F[e][k]; arm[k] = ext->x[e][k] - cm[3 * i + k]; }
        cross3(arm, ext->F[e], mo);
        for (int k = 0; k < 3; k++) ni[k] -= mo[k];
      }
    }
    {
      double arm[3], mo[3];
      for (int k = 0; k < 3; k++) arm[k] = f.p[3 * i + k] - cm[3 * i + k];
      cross3(arm, fi, mo);
      for (int k = 0; k < 3; k++) ni[k] -= mo[k];
    }
    for (int k = 0; k < 3; k++) { fj[3 * i + k] = fi[k]; nj[3 * i + k] = ni[k]; }
    tau[2 * i] = dot3(f.ax1 + 3 * i, ni);
    tau[2 * i + 1] = dot3(f.ax2 + 3 * i, ni);
    int pa = W->parent[i];
    if (pa >= 0) {
      double arm[3], mo[3];
      for (int k = 0; k < 3; k++) arm[k] = f.p[3 * i + k] - cm[3 * pa + k];
      cross3(arm, fi, mo);
      for (int k = 0; k < 3; k++) { fj[3 * pa + k] += fi[k]; nj[3 * pa + k] += ni[k] + mo[k]; }
    }
  }
  free(om); free(al); free(ac); free(cm); free(fj); free(nj);
  fk_free(&f);
}

/* ----------------------------------------------------------------------- */
/* mass matrix by brute force: column j = RNEA(q,0,e_j;0,0) - RNEA(q,0,0;0,0) */
/* ----------------------------------------------------------------------- */
static void mass_matrix(const obo_world *W, const double *q, double *M /* n x n row-major */) {
  int n = 2 * W->N;
  double zero3[3] = {0, 0, 0};
  double *z = (double *)calloc((size_t)n, sizeof(double));
  double *e = (double *)calloc((size_t)n, sizeof(double));
  double *t0 = (double *)calloc((size_t)n, sizeof(double));
  double *t1 = (double *)calloc((size_t)n, sizeof(double));
  rnea(W, q, z, z, zero3, NULL, t0);
  for (int j = 0; j < n; j++) {
    e[j] = 1.0;
    rnea(W, q, z, e, zero3, NULL, t1);
    e[j] = 0.0;
    for (int i = 0; i < n; i++) M[(size_t)i * n + j] = t1[i] - t0[i];
  }
  free(z); free(e); free(t0); free(t1);
}

/* dense Cholesky A = L L^T (lower, in place) and solve; returns 0 on success */
static int cholesky_solve(double *A, int n, const double *b, double *x) {
  for (int j = 0; j < n; j++) {
    double s = A[(size_t)j * n + j];
    for (int k = 0; k < j; k++) s -= A[(size_t)j * n + k] * A[(size_t)j * n + k];
    if (!(s > 0.0)) return -1;
    double ljj = sqrt(s);
    A[(size_t)j * n + j] = ljj;
    for (int i = j + 1; i < n; i++) {
      double t = A[(size_t)i * n + j];
      const double *ai = A + (size_t)i * n, *aj = A + (size_t)j * n;
      for (int k = 0; k < j; k++) t -= ai[k] * aj[k];
      A[(size_t)i * n + j] = t / ljj;
    }
  }
  for (int i = 0; i < n; i++) {
    double t = b[i];
    for (int k = 0; k < i; k++) t -= A[(size_t)i * n + k] * x[k];
    x[i] = t / A[(size_t)i * n + i];
  }
  for (int i = n - 1; i >= 0; i--) {
    double t = x[i];
    for (int k = i + 1; k < n; k++) t -= A[(size_t)k * n + i] * x[k];
    x[i] = t / A[(size_t)i * n + i];
  }
  return 0;
}

/* fp64 Jacobi-preconditioned CG on the dense matrix (reading A18); used for pin P13 */
static int pcg_solve(const double *A, int n, const double *b, double *x, double tol, int max_iter) {
  double *r = (double *)malloc(sizeof(double) * n), *z = (double *)malloc(sizeof(double) * n);
  double *p = (double *)malloc(sizeof(double) * n), *Ap = (double *)malloc(sizeof(double) * n);
  double bb = 0;
  for (int i = 0; i < n; i++) bb += b[i] * b[i];
  int it = 0;
  if (bb == 0.0) {
    for (int i = 0; i < n; i++) x[i] = 0.0;
  } else {
    double rz = 0, rr = 0;
    for (int i = 0; i < n; i++) {
      double s = 0;
      for (int j = 0; j < n; j++) s += A[(size_t)i * n + j] * x[j];
      r[i] = b[i] - s; z[i] = r[i] / A[(size_t)i * n + i]; p[i] = z[i];
      rz += r[i] * z[i]; rr += r[i] * r[i];
    }
    while (sqrt(rr) > tol * sqrt(bb) && it < max_iter) {
      double pAp = 0;
      for (int i = 0; i < n; i++) {
        double s = 0;
        for (int j = 0; j < n; j++) s += A[(size_t)i * n + j] * p[j];
        Ap[i] = s; pAp += p[i] * s;
      }
      double alpha = rz / pAp, rz2 = 0;
      rr = 0;
      for (int i = 0; i < n; i++) {
        x[i] += alpha * p[i]; r[i] -= alpha * Ap[i];
        z[i] = r[i] / A[(size_t)i * n + i];
        rz2 += r[i] * z[i]; rr += r[i] * r[i];
      }
      double beta = rz2 / rz;
      rz = rz2;
      for (int i = 0; i < n; i++) p[i] = z[i] + beta * p[i];
      it++;
    }
  }
  free(r); free(z); free(p); free(Ap);
  return it;
}

/* ----------------------------------------------------------------------- */
/* construction, derived constants, randomization                            */
/* ----------------------------------------------------------------------- */
static void derive_constants(obo_world *W) {
  const double PI = 3.14159265358979323846;
  for (int i = 0; i < W->N; i++) {
    double d = W->d[i], L = W->L[i], r = 0.5 * d;
    W->K[i] = (double)W->E * PI * d * d * d * d / (64.0 * L);       /* Eq. 4 */
    W->Mmax[i] = (double)W->MOR * PI * d * d * d / 32.0;            /* Eq. 5 */
    W->m[i] = (double)W->rho * PI * r * r * L;                      /* solid cylinder (A5) */
    W->Ixx[i] = W->m[i] * (3.0 * r * r + L * L) / 12.0;             /* about the cm        */
    W->Izz[i] = 0.5 * W->m[i] * r * r;
  }
  for (int a = 0; a < W->A; a++)
    W->ac[a] = W->ac_given ? (double)W->ac_in[a]
                           : 2.0 * W->P.zeta_s * sqrt(W->ak[a] * W->am[a]);   /* reading A11 */
}

static void reset_state(obo_world *W) {
  int N = W->N, A = W->A;
  memset(W->q, 0, sizeof(double) * 2 * N);
  memset(W->qd, 0, sizeof(double) * 2 * N);
  memset(W->dqd_prev, 0, sizeof(double) * 2 * N);
  memset(W->ruptured, 0, (size_t)N);
  memset(W->rc, 0, sizeof(int) * N);
  memset(W->rstep, 0, sizeof(int) * N);
  memset(W->cA, 0, sizeof(int) * A);
  memset(W->cB, 0, sizeof(int) * A);
  for (int s = 0; s < OBO_MAX_WRENCH; s++) W->wr_body[s] = -1;
  W->step = 0; W->status = 0; W->last_iters = 0;
  /* apples hang at rest: x = x_hang + m g / k_s */
  fk_t f = fk_alloc(N);
  fk_run(W, W->q, &f);
  for (int a = 0; a < A; a++) {
    int b = W->alink[a];
    double o[3];
    mat3vec(f.R + 9 * b, W->aoff + 3 * a, o);
    for (int k = 0; k < 3; k++) {
      W->ax[3 * a + k] = f.p[3 * b + k] + o[k] + W->am[a] * W->P.g[k] / W->ak[a];
      W->av[3 * a + k] = 0.0;
    }
    W->attached[a] = 1;
  }
  fk_free(&f);
}

obo_world *obo_world_new(int world_index, int n_links, const int32_t *parent, const float *length,
                         const float *diameter, const float *rest_quat, const float *armature, float density,
                         float E, float MOR, int n_apples, const int32_t *apple_link, const float *apple_offset,
                         const float *apple_mass, const float *apple_k, const float *apple_c,
                         const float *apple_detach, const obo_params *params) {
  if (n_links < 1 || n_apples < 0 || n_apples > OBO_MAX_APPLES) return NULL;
  for (int i = 0; i < n_links; i++)
    if ((i == 0 && parent[i] != -1) || (i > 0 && (parent[i] < 0 || parent[i] >= i))) return NULL;
  obo_world *W = (obo_world *)calloc(1, sizeof(obo_world));
  int N = n_links, A = n_apples;
  W->N = N; W->A = A; W->P = *params; W->world_index = world_index;
  W->parent = (int *)malloc(sizeof(int) * N);
  W->L = (double *)malloc(sizeof(double) * N);
  W->d = (double *)malloc(sizeof(double) * N);
  W->Q = (double *)malloc(sizeof(double) * 9 * N);
  W->arm = (double *)calloc(2 * (size_t)N, sizeof(double));
  W->L0 = (float *)malloc(sizeof(float) * N);
  W->d0 = (float *)malloc(sizeof(float) * N);
  W->Q0 = (double *)malloc(sizeof(double) * 9 * N);
  W->K = (double *)malloc(sizeof(double) * N);
  W->Mmax = (double *)malloc(sizeof(double) * N);
  W->m = (double *)malloc(sizeof(double) * N);
  W->Ixx = (double *)malloc(sizeof(double) * N);
  W->Izz = (double *)malloc(sizeof(double) * N);
  for (int i = 0; i < N; i++) {
    W->parent[i] = parent[i];
    W->L[i] = (double)length[i];
    W->d[i] = (double)diameter[i];
    double qn[4] = {rest_quat[4 * i], rest_quat[4 * i + 1], rest_quat[4 * i + 2], rest_quat[4 * i + 3]};
    quat_to_mat(qn, W->Q + 9 * i);
    W->L0[i] = length[i]; W->d0[i] = diameter[i];
    memcpy(W->Q0 + 9 * i, W->Q + 9 * i, sizeof(double) * 9);
    if (armature) { W->arm[2 * i] = armature[2 * i]; W->arm[2 * i + 1] = armature[2 * i + 1]; }
  }
  W->rho_nom = W->rho = density; W->E_nom = W->E = E; W->MOR_nom = W->MOR = MOR;
  W->alink = (int *)malloc(sizeof(int) * (A + 1));
  W->aoff = (double *)malloc(sizeof(double) * 3 * (A + 1));
  W->aoff0 = (double *)malloc(sizeof(double) * 3 * (A + 1));
  W->am_nom = (float *)malloc(sizeof(float) * (A + 1));
  W->adet_nom = (float *)malloc(sizeof(float) * (A + 1));
  W->ac_in = (float *)calloc((size_t)A + 1, sizeof(float));
  W->ac_given = apple_c != NULL;
  W->am = (double *)malloc(sizeof(double) * (A + 1));
  W->ak = (double *)malloc(sizeof(double) * (A + 1));
  W->ac = (double *)malloc(sizeof(double) * (A + 1));
  W->adet = (double *)malloc(sizeof(double) * (A + 1));
  for (int a = 0; a < A; a++) {
    W->alink[a] = apple_link[a];
    for (int k = 0; k < 3; k++) W->aoff0[3 * a + k] = W->aoff[3 * a + k] = (double)apple_offset[3 * a + k];
    W->am_nom[a] = apple_mass[a]; W->am[a] = (double)apple_mass[a];
    W->adet_nom[a] = apple_detach[a]; W->adet[a] = (double)apple_detach[a];
    W->ak[a] = (double)apple_k[a];
    if (apple_c) W->ac_in[a] = apple_c[a];
  }
  W->q = (double *)calloc(2 * (size_t)N, sizeof(double));
  W->qd = (double *)calloc(2 * (size_t)N, sizeof(double));
  W->dqd_prev = (double *)calloc(2 * (size_t)N, sizeof(double));
  W->ax = (double *)calloc(3 * (size_t)A + 3, sizeof(double));
  W->av = (double *)calloc(3 * (size_t)A + 3, sizeof(double));
  W->ruptured = (uint8_t *)calloc((size_t)N, 1);
  W->attached = (uint8_t *)calloc((size_t)A + 1, 1);
  W->rc = (int *)calloc((size_t)N, sizeof(int));
  W->rstep = (int *)calloc((size_t)N, sizeof(int));
  W->cA = (int *)calloc((size_t)A + 1, sizeof(int));
  W->cB = (int *)calloc((size_t)A + 1, sizeof(int));
  W->ev = NULL; W->n_ev = 0; W->cap_ev = 0;
  derive_constants(W);
  reset_state(W);
  return W;
}

void obo_world_free(obo_world *W) {
  if (!W) return;
  free(W->parent); free(W->L); free(W->d); free(W->Q); free(W->arm);
  free(W->L0); free(W->d0); free(W->Q0); free(W->aoff0);
  free(W->K); free(W->Mmax); free(W->m); free(W->Ixx); free(W->Izz);
  free(W->alink); free(W->aoff); free(W->am_nom); free(W->adet_nom); free(W->ac_in);
  free(W->am); free(W->ak); free(W->ac); free(W->adet);
  free(W->q); free(W->qd); free(W->dqd_prev); free(W->ax); free(W->av);
  free(W->ruptured); free(W->attached); free(W->rc); free(W->cA); free(W->cB); free(W->rstep);
  free(W->ev);
  free(W);
}

/* PAPER.md:167-169 + reading A23: key = (seed lo, seed hi); counter = (world, item, stream, 0);
   stream 0 item 0 -> (u_E, u_MOR, u_rho, -); stream 1 item a -> (u_det, u_mass, -, -);
   a degenerate range (lo == hi) keeps the spec's nominal value. */
void obo_randomize(obo_world *W, uint64_t seed) {
  uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
  uint32_t ctr[4] = {(uint32_t)W->world_index, 0u, 0u, 0u}, o[4];
  const obo_params *P = &W->P;
  obo_philox4x32_10(ctr, key, o);
  W->E = P->range_E[0] != P->range_E[1] ? philox_uniform(o[0], P->range_E[0], P->range_E[1]) : W->E_nom;
  W->MOR = P->range_MOR[0] != P->range_MOR[1] ? philox_uniform(o[1], P->range_MOR[0], P->range_MOR[1]) : W->MOR_nom;
  W->rho = P->range_density[0] != P->range_density[1]
               ? philox_uniform(o[2], P->range_density[0], P->range_density[1]) : W->rho_nom;
  for (int a = 0; a < W->A; a++) {
    ctr[1] = (uint32_t)a; ctr[2] = 1u;
    obo_philox4x32_10(ctr, key, o);
    float fd = P->range_detach[0] != P->range_detach[1]
                   ? philox_uniform(o[0], P->range_detach[0], P->range_detach[1]) : W->adet_nom[a];
    float fm = P->range_apple_mass[0] != P->range_apple_mass[1]
                   ? philox_uniform(o[1], P->range_apple_mass[0], P->range_apple_mass[1]) : W->am_nom[a];
    W->adet[a] = (double)fd;
    W->am[a] = (double)fm;
  }
  derive_constants(W);
  reset_state(W);
}

/* ----------------------------------------------------------------------- */
/* per-world geometry randomization (reading A37)     */
/* ----------------------------------------------------------------------- */
typedef struct {
  float droop[2], lean[2], spread[2], twist[2];
  float scale_length[2], scale_diameter[2], jitter_length[2], jitter_diameter[2];
} obo_geometry_ranges;

/* rotation by angle t about the unit axis a (Rodrigues) */
static void rot_axis(const double a[3], double t, double *R) {
  double c = cos(t), s = sin(t), v = 1.0 - c;
  R[0] = c + a[0] * a[0] * v;        R[1] = a[0] * a[1] * v - a[2] * s; R[2] = a[0] * a[2] * v + a[1] * s;
  R[3] = a[1] * a[0] * v + a[2] * s; R[4] = c + a[1] * a[1] * v;        R[5] = a[1] * a[2] * v - a[0] * s;
  R[6] = a[2] * a[0] * v - a[1] * s; R[7] = a[2] * a[1] * v + a[0] * s; R[8] = c + a[2] * a[2] * v;
}

/* "we generate one base skeleton and perturb only continuous quantities per world ... per-segment bend and whole-tree
   growth habit (a gravimorphic droop multiplier applied inside a forward-kinematic re-walk so droop compounds per
   internode ..., plus whole-tree lean, fork spread and an env-wide phyllotactic twist)" and the per-branch
   dimensions "(global scale and stockiness, and per-segment length and thickness)".  Always
   starts from the BASE geometry, so zero strength reproduces the base model exactly.  Reading A37:
     draws (A23 layout): stream 3 item 0 -> droop, lean, spread, twist; stream 3 item 1 -> lean azimuth (u * 2 pi),
       length scale, diameter scale; stream 4 item i -> length jitter, diameter jitter of link i; a degenerate range
       gives its lo value;
     dimensions: L_i = (L0_i * scale_length) * jitter_i, d_i likewise, in fp32; apple offsets scale with their link
       (x, y by the diameter factor, z by the length factor);
     twist: every non-trunk rest rotation becomes Rz(twist) Q_i (turned about the parent's axis);
     spread: the swing of Q_i away from the parent's axis (swing-twist decomposition about z) is scaled by 1 + spread;
     lean: the trunk's rest rotation becomes Rot((cos phi, sin phi, 0), lean) Q_0;
     droop: a top-down re-walk in the world frame; with d = R_i z the link direction, s = |d x z_w| the sine of its
       angle to the vertical, the link frame is turned by droop * s about (d x -z_w) / s, i.e. towards the ground;
       children inherit the turned frame (the droop compounds per internode).
   Materials are kept; derived constants are recomputed and the state is reset. */
void obo_randomize_geometry(obo_world *W, uint64_t seed, const obo_geometry_ranges *G) {
  const double PI = 3.14159265358979323846;
  uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
  uint32_t ctr[4] = {(uint32_t)W->world_index, 0u, 3u, 0u}, o[4];
  obo_philox4x32_10(ctr, key, o);
  float droop = philox_uniform(o[0], G->droop[0], G->droop[1]);
  float lean = philox_uniform(o[1], G->lean[0], G->lean[1]);
  float spread = philox_uniform(o[2], G->spread[0], G->spread[1]);
  float twist = philox_uniform(o[3], G->twist[0], G->twist[1]);
  ctr[1] = 1u;
  obo_philox4x32_10(ctr, key, o);
  float phi = philox_uniform(o[0], 0.0f, 6.2831855f);
  float sL = philox_uniform(o[1], G->scale_length[0], G->scale_length[1]);
  float sD = philox_uniform(o[2], G->scale_diameter[0], G->scale_diameter[1]);
  int N = W->N;
  float *fl = (float *)malloc(sizeof(float) * N), *fd = (float *)malloc(sizeof(float) * N);
  for (int i = 0; i < N; i++) {
    ctr[1] = (uint32_t)i; ctr[2] = 4u;
    obo_philox4x32_10(ctr, key, o);
    float jl = philox_uniform(o[0], G->jitter_length[0], G->jitter_length[1]);
    float jd = philox_uniform(o[1], G->jitter_diameter[0], G->jitter_diameter[1]);
    float t = W->L0[i] * sL; float Ln = t * jl;
    float u = W->d0[i] * sD; float dn = u * jd;
    W->L[i] = (double)Ln; W->d[i] = (double)dn;
    fl[i] = Ln / W->L0[i]; fd[i] = dn / W->d0[i];
  }
  for (int a = 0; a < W->A; a++) {
    int b = W->alink[a];
    W->aoff[3 * a] = (double)((float)W->aoff0[3 * a] * fd[b]);
    W->aoff[3 * a + 1] = (double)((float)W->aoff0[3 * a + 1] * fd[b]);
    W->aoff[3 * a + 2] = (double)((float)W->aoff0[3 * a + 2] * fl[b]);
  }
  free(fl); free(fd);
  /* rest rotations: twist, spread, lean, then the droop re-walk */
  double *RW = (double *)malloc(sizeof(double) * 9 * N);   /* world rest rotation of every link, after droop */
  for (int i = 0; i < N; i++) {
    double Qn[9];
    memcpy(Qn, W->Q0 + 9 * i, sizeof(Qn));
    int pa = W->parent[i];
    if (pa >= 0) {
      /* swing-twist decomposition about z: the direction of the child axis in the parent frame is column 2 of Q */
      double dz[3] = {Qn[2], Qn[5], Qn[8]};
      double sw = atan2(sqrt(dz[0] * dz[0] + dz[1] * dz[1]), dz[2]);       /* swing angle away from the parent's axis */
      double hn = sqrt(dz[0] * dz[0] + dz[1] * dz[1]);
      if (hn > 1e-12 && spread != 0.0f) {
        double ax[3] = {-dz[1] / hn, dz[0] / hn, 0.0};                     /* z x dz, the swing axis */
        double Rs[9];
        rot_axis(ax, sw * (double)spread, Rs);                             /* extra swing: sw (1 + spread) in all */
        mat3mul(Rs, Qn, Qn);
      }
      if (twist != 0.0f) {
        double z[3] = {0, 0, 1}, Rt[9];
        rot_axis(z, (double)twist, Rt);
        mat3mul(Rt, Qn, Qn);
      }
    } else if (lean != 0.0f) {
      double ax[3] = {cos((double)phi), sin((double)phi), 0.0}, Rl[9];
      rot_axis(ax, (double)lean, Rl);
      mat3mul(Rl, Qn, Qn);
    }
    if (droop == 0.0f) {                       /* no re-walk: the modified rest rotation is the result, exactly */
      memcpy(W->Q + 9 * i, Qn, sizeof(Qn));
      continue;
    }
    static const double I3[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    const double *Rp = pa < 0 ? I3 : RW + 9 * pa;
    double Ri[9];
    mat3mul(Rp, Qn, Ri);
    double d[3] = {Ri[2], Ri[5], Ri[8]};
    double s = sqrt(d[0] * d[0] + d[1] * d[1]);                            /* |d x z_w| */
    if (s > 1e-12 && droop != 0.0f) {
      double ax[3] = {-d[1] / s, d[0] / s, 0.0}, Rd[9];                    /* (d x -z_w) / s */
      rot_axis(ax, (double)droop * s, Rd);
      mat3mul(Rd, Ri, Ri);
    }
    memcpy(RW + 9 * i, Ri, sizeof(Ri));
    /* new rest rotation in the parent frame: Rp^T Ri */
    double Rpt[9];
    for (int r_ = 0; r_ < 3; r_++)
      for (int c_ = 0; c_ < 3; c_++) Rpt[3 * r_ + c_] = Rp[3 * c_ + r_];
    mat3mul(Rpt, Ri, W->Q + 9 * i);
  }
  free(RW);
  derive_constants(W);
  reset_state(W);
}

int obo_apply_wrench(obo_world *W, int body, const double point[3], const double force[3]) {
  if (body < 0 || body >= W->N + W->A) return -1;
  int zero = force[0] == 0.0 && force[1] == 0.0 && force[2] == 0.0;
  int slot = -1;
  for (int s = 0; s < OBO_MAX_WRENCH; s++)
    if (W->wr_body[s] == body) slot = s;
  if (zero) {
    if (slot >= 0) W->wr_body[slot] = -1;
    return 0;
  }
  if (slot < 0)
    for (int s = 0; s < OBO_MAX_WRENCH && slot < 0; s++)
      if (W->wr_body[s] < 0) slot = s;
  if (slot < 0) return -2;
  W->wr_body[slot] = body;
  for (int k = 0; k < 3; k++) { W->wr_point[slot][k] = point[k]; W->wr_force[slot][k] = force[k]; }
  return 0;
}

static void push_event(obo_world *W, int kind, int index, double value, double threshold) {
  if (W->n_ev == W->cap_ev) {
    W->cap_ev = W->cap_ev ? 2 * W->cap_ev : 16;
    W->ev = (obo_event *)realloc(W->ev, sizeof(obo_event) * W->cap_ev);
  }
  obo_event e = {W->world_index, W->step, kind, index, value, threshold};
  W->ev[W->n_ev++] = e;
}

/* ----------------------------------------------------------------------- */
/* the system of one step (shared by obo_step and the diagnostics)           */
/* ----------------------------------------------------------------------- */
typedef struct {
  double *A, *b;        /* n x n, n */
  double *fteth;        /* [3A] tether force on each apple (Eq. 6)       */
  double *fuser;        /* [3A] user wrench on each apple, after the rails */
  double *fuser_raw;    /* [3A] ... as applied                           */
  double *fs_norm;      /* [A]  |f_s|                                    */
  double *fu_norm;      /* [A]  |f_user|                                 */
} system_t;

static void system_free(system_t *S) { free(S->A); free(S->b); free(S->fteth); free(S->fuser); free(S->fuser_raw); free(S->fs_norm); free(S->fu_norm); }

/* link velocity of a world point x attached to link b:  v = v_joint(b) + om_b x (x - p_b).
   Computed from the joint-rate Jacobian: v = sum_{j in path(b)} (ax_j qd_j) x (x - p_j). */
static void point_velocity(const obo_world *W, const fk_t *f, const double *qd, int b, const double x[3], double v[3]) {
  v[0] = v[1] = v[2] = 0.0;
  for (int j = b; j >= 0; j = W->parent[j]) {
    double r[3], w[3], c[3];
    for (int k = 0; k < 3; k++) {
      r[k] = x[k] - f->p[3 * j + k];
      w[k] = f->ax1[3 * j + k] * qd[2 * j] + f->ax2[3 * j + k] * qd[2 * j + 1];
    }
    cross3(w, r, c);
    for (int k = 0; k < 3; k++) v[k] += c[k];
  }
}

/* Coulomb friction at a ruptured joint ("Coulomb friction is introduced at the break and ramped up ~5x
   over ~1.5 s as the torn fibres seize"), reading A34: torque of magnitude
     T_f(t) = fric_frac * M_max,i * (1 + (fric_ramp - 1) min(t / fric_time, 1)),   t = h (step - step of rupture),
   against the joint velocity (both DoF together, like |theta| in Eq. 5); for the linearly implicit step it is taken as
   the damper D_f = T_f / max(|qd_i|, fric_veps) at the start-of-step speed, which joins D = c_d K in the matrix and
   in the right-hand side.  Returns D_f (0 for an intact joint or fric_frac = 0). */
static double friction_damper(const obo_world *W, int i) {
  const obo_params *P = &W->P;
  if (!W->ruptured[i] || P->fric_frac <= 0.0) return 0.0;
  double t = P->h * (double)(W->step - W->rstep[i]);
  double ramp = P->fric_time > 0.0 ? (t < P->fric_time ? t / P->fric_time : 1.0) : 1.0;
  double Tf = P->fric_frac * W->Mmax[i] * (1.0 + (P->fric_ramp - 1.0) * ramp);
  double w = sqrt(W->qd[2 * i] * W->qd[2 * i] + W->qd[2 * i + 1] * W->qd[2 * i + 1]);
  return Tf / (w > P->fric_veps ? w : P->fric_veps);
}

/* The three rails of PAPER.md:398 (App. B) on an applied force F acting on a FREE body of mass m that moves with
   velocity v at the application point (reading A36; connected links are static loading, which the rails never touch):
     (2) power fade: the part of F along v (if it pushes along v) is scaled by clamp((v_lim - |v|) / (v_lim - v_f), 0, 1),
         v_f = rail_fade v_lim;
     (1) impulse cap: |F| <= m max(v_lim - v . F^, 0) / h -- the force may not take the body past v_lim in one step;
     (3) speed brake: above v_lim an extra force - rail_brake m (|v| - v_lim) v^.
   rail_speed = 0 switches all three off. */
static void apply_rails(const obo_params *P, double m, const double v[3], double F[3]) {
  double vl = P->rail_speed;
  if (!(vl > 0.0)) return;
  double vn = norm3(v);
  if (vn > 0.0) {
    double vh[3] = {v[0] / vn, v[1] / vn, v[2] / vn};
    double Fp = dot3(F, vh);
    if (Fp > 0.0) {
      double vf = P->rail_fade * vl;
      double fade = vn <= vf ? 1.0 : (vn >= vl ? 0.0 : (vl - vn) / (vl - vf));
      for (int k = 0; k < 3; k++) F[k] -= (1.0 - fade) * Fp * vh[k];
    }
  }
  double Fn = norm3(F);
  if (Fn > 0.0) {
    double vF = dot3(v, F) / Fn;
    double cap = m * (vl - vF > 0.0 ? vl - vF : 0.0) / P->h;
    if (Fn > cap) for (int k = 0; k < 3; k++) F[k] *= cap / Fn;
  }
  if (vn > vl) for (int k = 0; k < 3; k++) F[k] -= P->rail_brake * m * (vn - vl) * v[k] / vn;
}

static void build_system(const obo_world *W, system_t *S) {
  int N = W->N, A = W->A, n = 2 * N;
  const obo_params *P = &W->P;
  double h = P->h, eta = P->tether_implicit ? 1.0 : 0.0;
  S->A = (double *)calloc((size_t)n * n, sizeof(double));
  S->b = (double *)calloc((size_t)n, sizeof(double));
  S->fteth = (double *)calloc(3 * (size_t)A + 3, sizeof(double));
  S->fuser = (double *)calloc(3 * (size_t)A + 3, sizeof(double));
  S->fuser_raw = (double *)calloc(3 * (size_t)A + 3, sizeof(double));
  S->fs_norm = (double *)calloc((size_t)A + 1, sizeof(double));
  S->fu_norm = (double *)calloc((size_t)A + 1, sizeof(double));

  /* 1. FK at q; snapped_i = ruptured_i or snapped_parent */
  fk_t f = fk_alloc(N);
  fk_run(W, W->q, &f);
  uint8_t *snapped = (uint8_t *)calloc((size_t)N, 1);
  for (int i = 0; i < N; i++) snapped[i] = W->ruptured[i] || (W->parent[i] >= 0 && snapped[W->parent[i]]);

  ext_t *ext = (ext_t *)calloc(1, sizeof(ext_t));
  /* user wrenches: on apples they are body forces on the apple; on links they enter f_ext */
  for (int s = 0; s < OBO_MAX_WRENCH; s++) {
    int body = W->wr_body[s];
    if (body < 0) continue;
    if (body >= N) {
      int a = body - N;
      double F[3] = {W->wr_force[s][0], W->wr_force[s][1], W->wr_force[s][2]};
      for (int k = 0; k < 3; k++) S->fuser_raw[3 * a + k] += F[k];            /* the detach predicate sees the pull itself */
      apply_rails(P, W->am[a], W->av + 3 * a, F);                           /* an apple is a free body (A36) */
      for (int k = 0; k < 3; k++) S->fuser[3 * a + k] += F[k];
    } else {
      if (P->forces_off_on_snapped && snapped[body]) continue;   /* reading A10 */
      int e = ext->n++;
      double o[3], F[3] = {W->wr_force[s][0], W->wr_force[s][1], W->wr_force[s][2]};
      mat3vec(f.R + 9 * body, W->wr_point[s], o);
      ext->link[e] = body;
      for (int k = 0; k < 3; k++) ext->x[e][k] = f.p[3 * body + k] + o[k];
      if (snapped[body]) {                                       /* a link of a snapped sub-tree is a free body (A36) */
        double vpt[3];
        point_velocity(W, &f, W->qd, body, ext->x[e], vpt);
        apply_rails(P, W->m[body], vpt, F);
      }
      for (int k = 0; k < 3; k++) ext->F[e][k] = F[k];
    }
  }
  /* 2. tethers (Eq. 6, Eq. 7; readings A11-A13, A15) */
  double *xh = (double *)calloc(3 * (size_t)A + 3, sizeof(double));
  for (int a = 0; a < A; a++) {
    S->fu_norm[a] = norm3(S->fuser_raw + 3 * a);
    if (!W->attached[a]) continue;
    int b = W->alink[a];
    double o[3], vh[3], fs[3], fr[3];
    mat3vec(f.R + 9 * b, W->aoff + 3 * a, o);
    for (int k = 0; k < 3; k++) xh[3 * a + k] = f.p[3 * b + k] + o[k];
    point_velocity(W, &f, W->qd, b, xh + 3 * a, vh);
    for (int k = 0; k < 3; k++) {
      double stretch = W->ax[3 * a + k] - xh[3 * a + k];
      fs[k] = -W->ak[a] * stretch;                                   /* f_s, Eq. 7 */
      S->fteth[3 * a + k] = fs[k] - W->ac[a] * W->av[3 * a + k];     /* Eq. 6      */
      /* f_react = -(f_s - m g zhat) with the hang point advanced by eta*h*v_hang (A15);
         -m g_vec equals +m g zhat for g_vec = (0,0,-g) */
      fr[k] = W->ak[a] * (stretch - eta * h * vh[k]) - W->am[a] * P->g[k];
    }
    S->fs_norm[a] = norm3(fs);
    double nr = norm3(fr);
    if (nr > P->react_max) for (int k = 0; k < 3; k++) fr[k] *= P->react_max / nr;   /* clamp */
    int e = ext->n++;
    ext->link[e] = b;
    for (int k = 0; k < 3; k++) { ext->x[e][k] = xh[3 * a + k]; ext->F[e][k] = fr[k]; }
  }
  /* 4. bias and right-hand side */
  double *zero = (double *)calloc((size_t)n, sizeof(double));
  double *bias = (double *)calloc((size_t)n, sizeof(double));
  rnea(W, W->q, W->qd, zero, P->g, ext, bias);
  for (int i = 0; i < N; i++) {
    double Kt = W->ruptured[i] ? 0.0 : W->K[i], Dt = P->c_d * Kt + friction_damper(W, i);
    for (int k = 0; k < 2; k++) {
      int j = 2 * i + k;
      S->b[j] = h * (-bias[j] - Kt * W->q[j] - (Dt + h * Kt) * W->qd[j]);
    }
  }
  /* 5. A = M + eta M_teth + diag(arm + h D + h^2 K) */
  mass_matrix(W, W->q, S->A);
  /* Velocity-proportional damping F = -c_v m v, tau = -c_omega I omega on every link, reading A32:
     c_v = c_omega = alpha_m.  The generalized force of these body forces is -alpha sum_i J_i^T I_i J_i qd =
     -alpha M(q) qd (M = sum J^T I J, the identity pin P2 checks).  Taken at the end-of-step velocity qd + dqd
     (linearly implicit, like the joint damper):  M dqd = h [ ... - alpha M (qd + dqd) ]  ->
     A gets (1 + h alpha) M, b gets - h alpha M qd. */
  if (P->alpha_m != 0.0) {
    /* per link alpha_i = alpha_m, times snap_drag_scale on snapped sub-trees ("a snapped sub-tree's
       linear drag is also reduced"; reading A35).  M is linear in the link inertias, so sum_i alpha_i J_i^T I_i J_i is
       the mass matrix of the same tree with every inertia scaled by alpha_i. */
    obo_world Ws = *W;
    double *ms = (double *)malloc(sizeof(double) * N), *ix = (double *)malloc(sizeof(double) * N), *iz = (double *)malloc(sizeof(double) * N);
    for (int i = 0; i < N; i++) {
      double al = P->alpha_m * (snapped[i] ? P->snap_drag_scale : 1.0);
      ms[i] = al * W->m[i]; ix[i] = al * W->Ixx[i]; iz[i] = al * W->Izz[i];
    }
    Ws.m = ms; Ws.Ixx = ix; Ws.Izz = iz;
    double *Ma = (double *)calloc((size_t)n * n, sizeof(double));
    mass_matrix(&Ws, W->q, Ma);
    for (int r_ = 0; r_ < n; r_++) {
      double mq = 0.0;
      for (int c_ = 0; c_ < n; c_++) mq += Ma[(size_t)r_ * n + c_] * W->qd[c_];
      S->b[r_] -= h * mq;
    }
    for (size_t k = 0; k < (size_t)n * n; k++) S->A[k] += h * Ma[k];
    free(Ma); free(ms); free(ix); free(iz);
  }
  for (int i = 0; i < N; i++) {
    double Kt = W->ruptured[i] ? 0.0 : W->K[i], Dt = P->c_d * Kt + friction_damper(W, i);
    for (int k = 0; k < 2; k++) {
      int j = 2 * i + k;
      S->A[(size_t)j * n + j] += W->arm[j] + h * Dt + h * h * Kt;
    }
  }
  if (eta != 0.0) {
    double *J = (double *)malloc(sizeof(double) * 3 * (size_t)n);
    for (int a = 0; a < A; a++) {
      if (!W->attached[a]) continue;
      memset(J, 0, sizeof(double) * 3 * (size_t)n);
      for (int j = W->alink[a]; j >= 0; j = W->parent[j]) {
        double r[3], c1[3], c2[3];
        for (int k = 0; k < 3; k++) r[k] = xh[3 * a + k] - f.p[3 * j + k];
        cross3(f.ax1 + 3 * j, r, c1);
        cross3(f.ax2 + 3 * j, r, c2);
        for (int k = 0; k < 3; k++) { J[(size_t)k * n + 2 * j] = c1[k]; J[(size_t)k * n + 2 * j + 1] = c2[k]; }
      }
      double s = h * h * W->ak[a];
      for (int r_ = 0; r_ < n; r_++) {
        double j0 = J[r_], j1 = J[n + r_], j2 = J[2 * (size_t)n + r_];
        if (j0 == 0.0 && j1 == 0.0 && j2 == 0.0) continue;
        for (int c_ = 0; c_ < n; c_++)
          S->A[(size_t)r_ * n + c_] += s * (j0 * J[c_] + j1 * J[n + c_] + j2 * J[2 * (size_t)n + c_]);
      }
    }
    free(J);
  }
  free(zero); free(bias); free(xh); free(ext); free(snapped);
  fk_free(&f);
}

/* ----------------------------------------------------------------------- */
/* one step (SURVEY.md 8(c) "One step", items 1-10)                          */
/* ----------------------------------------------------------------------- */
static void step_once(obo_world *W) {
  if (W->status & 1) return; /* frozen after a non-finite state */
  int N = W->N, A = W->A, n = 2 * N;
  const obo_params *P = &W->P;
  double h = P->h;
  system_t S;
  build_system(W, &S);
  double *x = (double *)calloc((size_t)n, sizeof(double));
  if (P->solver == 1) {
    memcpy(x, W->dqd_prev, sizeof(double) * n);
    W->last_iters = pcg_solve(S.A, n, S.b, x, P->cg_tol, P->cg_max_iter);
    W->cg_iters_total += W->last_iters;
  } else {
    if (cholesky_solve(S.A, n, S.b, x) != 0) W->status |= 1;
    W->last_iters = 0;
  }
  int finite = 1;
  for (int j = 0; j < n; j++) if (!isfinite(x[j])) finite = 0;
  if (!finite) W->status |= 1;
  if (W->status & 1) { free(x); system_free(&S); return; }
  memcpy(W->dqd_prev, x, sizeof(double) * n);
  /* 6. integrate joints (semi-implicit Euler), speed clamp (reading A16) */
  for (int j = 0; j < n; j++) {
    double v = W->qd[j] + x[j];
    if (P->qd_max > 0.0) { if (v > P->qd_max) v = P->qd_max; if (v < -P->qd_max) v = -P->qd_max; }
    W->qd[j] = v;
    W->q[j] += h * v;
  }
  /* detach counters use the start-of-step forces (reading A8, A14) */
  for (int a = 0; a < A; a++) {
    if (!W->attached[a]) continue;
    W->cA[a] = S.fu_norm[a] > W->adet[a] ? W->cA[a] + 1 : 0;
    W->cB[a] = S.fs_norm[a] > P->detach_kappa * W->adet[a] ? W->cB[a] + 1 : 0;
  }
  /* 7. apples: 3-DoF point bodies */
  for (int a = 0; a < A; a++) {
    double att = W->attached[a] ? 1.0 : 0.0;
    for (int k = 0; k < 3; k++) {
      /* the apple is a body too: F = -c_v m v, explicit at the start-of-step velocity */
      double acc = P->g[k] + (att * S.fteth[3 * a + k] + S.fuser[3 * a + k]) / W->am[a] - P->alpha_m * W->av[3 * a + k];
      W->av[3 * a + k] += h * acc;
      W->ax[3 * a + k] += h * W->av[3 * a + k];
    }
  }
  /* 8. rupture (Eq. 5) on the new q, N-frame hysteresis (A6, A7) */
  for (int i = 0; i < N; i++) {
    if (W->ruptured[i]) continue;
    double mu = W->K[i] * sqrt(W->q[2 * i] * W->q[2 * i] + W->q[2 * i + 1] * W->q[2 * i + 1]);
    W->rc[i] = mu > W->Mmax[i] ? W->rc[i] + 1 : 0;
    if (W->rc[i] >= P->rupture_frames) {
      W->ruptured[i] = 1;
      W->rstep[i] = W->step;
      push_event(W, 0, i, mu, W->Mmax[i]);
    }
  }
  /* 9. detach (A14): path A = user pull, path B = stem tension */
  for (int a = 0; a < A; a++) {
    if (!W->attached[a]) continue;
    if (W->cA[a] >= P->detach_frames_pull) {
      W->attached[a] = 0;
      push_event(W, 1, a, S.fu_norm[a], W->adet[a]);
    } else if (W->cB[a] >= P->detach_frames_tension) {
      W->attached[a] = 0;
      push_event(W, 1, a, S.fs_norm[a], P->detach_kappa * W->adet[a]);
    }
  }
  for (int j = 0; j < n; j++) if (!isfinite(W->q[j]) || !isfinite(W->qd[j])) W->status |= 1;
  W->step += 1;
  free(x);
  system_free(&S);
}

void obo_step(obo_world *W, int n) { for (int s = 0; s < n; s++) step_once(W); }

/* many independent worlds: OpenMP over worlds (bench cpu_baseline) */
void obo_step_many(obo_world **Ws, int n_worlds, int n) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int w = 0; w < n_worlds; w++) obo_step(Ws[w], n);
}

/* ----------------------------------------------------------------------- */
/* state access                                                              */
/* ----------------------------------------------------------------------- */
void obo_get_state(const obo_world *W, double *q, double *qd, double *ax, double *av, uint8_t *ruptured,
                   uint8_t *attached, int32_t *info /* step, last_iters, status */) {
  if (q) memcpy(q, W->q, sizeof(double) * 2 * W->N);
  if (qd) memcpy(qd, W->qd, sizeof(double) * 2 * W->N);
  if (ax) memcpy(ax, W->ax, sizeof(double) * 3 * W->A);
  if (av) memcpy(av, W->av, sizeof(double) * 3 * W->A);
  if (ruptured) memcpy(ruptured, W->ruptured, (size_t)W->N);
  if (attached) memcpy(attached, W->attached, (size_t)W->A);
  if (info) { info[0] = W->step; info[1] = W->last_iters; info[2] = W->status; }
}
void obo_set_state(obo_world *W, const double *q, const double *qd, const double *ax, const double *av,
                   const uint8_t *ruptured, const uint8_t *attached) {
  if (q) memcpy(W->q, q, sizeof(double) * 2 * W->N);
  if (qd) memcpy(W->qd, qd, sizeof(double) * 2 * W->N);
  if (ax) memcpy(W->ax, ax, sizeof(double) * 3 * W->A);
  if (av) memcpy(W->av, av, sizeof(double) * 3 * W->A);
  if (ruptured) {
    memcpy(W->ruptured, ruptured, (size_t)W->N);
    memset(W->rc, 0, sizeof(int) * W->N);
    for (int i = 0; i < W->N; i++) W->rstep[i] = W->step;      /* friction ramps from the moment the flag was set */
  }
  if (attached) {
    memcpy(W->attached, attached, (size_t)W->A);
    memset(W->cA, 0, sizeof(int) * W->A);
    memset(W->cB, 0, sizeof(int) * W->A);
  }
}
/* predicate counters, for lock-step comparison across a counter window */
void obo_get_counters(const obo_world *W, int32_t *rc, int32_t *cA, int32_t *cB) {
  for (int i = 0; i < W->N; i++) rc[i] = W->rc[i];
  for (int a = 0; a < W->A; a++) { cA[a] = W->cA[a]; cB[a] = W->cB[a]; }
}
void obo_set_counters(obo_world *W, const int32_t *rc, const int32_t *cA, const int32_t *cB) {
  for (int i = 0; i < W->N; i++) W->rc[i] = rc[i];
  for (int a = 0; a < W->A; a++) { W->cA[a] = cA[a]; W->cB[a] = cB[a]; }
}
void obo_set_step(obo_world *W, int step) { W->step = step; }
void obo_get_rupture_steps(const obo_world *W, int32_t *rstep) { for (int i = 0; i < W->N; i++) rstep[i] = W->rstep[i]; }
void obo_set_rupture_steps(obo_world *W, const int32_t *rstep) { for (int i = 0; i < W->N; i++) W->rstep[i] = rstep[i]; }
void obo_set_solver(obo_world *W, int solver, double tol, int max_iter) {
  W->P.solver = solver; W->P.cg_tol = tol; W->P.cg_max_iter = max_iter;
}
int obo_events(obo_world *W, obo_event *buf, int cap) {
  int n = W->n_ev < cap ? W->n_ev : cap;
  if (n <= 0) return 0;                        /* an empty list has ev == NULL: nothing to copy */
  memcpy(buf, W->ev, sizeof(obo_event) * n);
  memmove(W->ev, W->ev + n, sizeof(obo_event) * (W->n_ev - n));
  W->n_ev -= n;
  return n;
}
int obo_n_events(const obo_world *W) { return W->n_ev; }

/* ----------------------------------------------------------------------- */
/* diagnostics for the pins                                                  */
/* ----------------------------------------------------------------------- */
void obo_diag_geometry(const obo_world *W, double *L, double *d, double *Q, double *aoff) {
  if (L) memcpy(L, W->L, sizeof(double) * W->N);
  if (d) memcpy(d, W->d, sizeof(double) * W->N);
  if (Q) memcpy(Q, W->Q, sizeof(double) * 9 * W->N);
  if (aoff) memcpy(aoff, W->aoff, sizeof(double) * 3 * W->A);
}
void obo_diag_material(const obo_world *W, float *E_MOR_rho /*3*/, double *adet, double *am, double *ac) {
  E_MOR_rho[0] = W->E; E_MOR_rho[1] = W->MOR; E_MOR_rho[2] = W->rho;
  for (int a = 0; a < W->A; a++) { if (adet) adet[a] = W->adet[a]; if (am) am[a] = W->am[a]; if (ac) ac[a] = W->ac[a]; }
}
void obo_diag_derived(const obo_world *W, double *K, double *Mmax, double *m, double *Ixx, double *Izz) {
  memcpy(K, W->K, sizeof(double) * W->N); memcpy(Mmax, W->Mmax, sizeof(double) * W->N);
  memcpy(m, W->m, sizeof(double) * W->N); memcpy(Ixx, W->Ixx, sizeof(double) * W->N);
  memcpy(Izz, W->Izz, sizeof(double) * W->N);
}
void obo_diag_fk(const obo_world *W, double *R, double *p, double *ax1, double *ax2) {
  fk_t f = fk_alloc(W->N);
  fk_run(W, W->q, &f);
  if (R) memcpy(R, f.R, sizeof(double) * 9 * W->N);
  if (p) memcpy(p, f.p, sizeof(double) * 3 * W->N);
  if (ax1) memcpy(ax1, f.ax1, sizeof(double) * 3 * W->N);
  if (ax2) memcpy(ax2, f.ax2, sizeof(double) * 3 * W->N);
  fk_free(&f);
}
void obo_diag_mass(const obo_world *W, double *M) { mass_matrix(W, W->q, M); }
/* tau = RNEA(q, qd, qdd; g*use_gravity, no external forces) */
void obo_diag_rnea(const obo_world *W, const double *qdd, int use_gravity, double *tau) {
  double g[3] = {0, 0, 0};
  if (use_gravity) memcpy(g, W->P.g, sizeof(g));
  rnea(W, W->q, W->qd, qdd, g, NULL, tau);
}
/* the linear system of the next step, without stepping */
void obo_diag_system(const obo_world *W, double *A, double *b) {
  system_t S;
  build_system(W, &S);
  int n = 2 * W->N;
  if (A) memcpy(A, S.A, sizeof(double) * (size_t)n * n);
  if (b) memcpy(b, S.b, sizeof(double) * n);
  system_free(&S);
}
/* kinetic energy of the tree 1/2 qd^T M qd, elastic + gravitational potential (no apples) */
void obo_diag_energy(const obo_world *W, double *T, double *V) {
  int N = W->N, n = 2 * N;
  double *M = (double *)malloc(sizeof(double) * (size_t)n * n);
  mass_matrix(W, W->q, M);
  double t = 0;
  for (int i = 0; i < n; i++)
    for (int j = 0; j < n; j++) t += 0.5 * W->qd[i] * M[(size_t)i * n + j] * W->qd[j];
  free(M);
  fk_t f = fk_alloc(N);
  fk_run(W, W->q, &f);
  double v = 0;
  for (int i = 0; i < N; i++) {
    double half[3] = {0, 0, 0.5 * W->L[i]}, rc[3];
    mat3vec(f.R + 9 * i, half, rc);
    for (int k = 0; k < 3; k++) v -= W->m[i] * W->P.g[k] * (f.p[3 * i + k] + rc[k]);
    if (!W->ruptured[i]) v += 0.5 * W->K[i] * (W->q[2 * i] * W->q[2 * i] + W->q[2 * i + 1] * W->q[2 * i + 1]);
  }
  fk_free(&f);
  *T = t; *V = v;
}
int obo_sizeof_params(void) { return (int)sizeof(obo_params); }
int obo_sizeof_event(void) { return (int)sizeof(obo_event); }
