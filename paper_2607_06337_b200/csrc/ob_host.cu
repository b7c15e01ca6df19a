// ob_host.cu -- host runtime behind the C ABI of include/orchard.h: validation, level-order layout,
// workspace carving, wrench staging, launches, state / event copy-out.  No physics here: every step of the
// path runs in the kernels of ob_kernels.cu.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "ob_internal.h"

using namespace ob;

namespace {

constexpr size_t kAlign = 256;
constexpr int kMaxSmem = 227 * 1024 - 1024;   // per-CTA limit minus the kernel's static shared memory (896 B)
const char *kNullCtx = "null context";

struct Pool {
  size_t off = 0, bytes = 0;
};

struct HostWorld {
  std::vector<int32_t> ext2int_link, int2ext_link, ext2int_apple, int2ext_apple;
  std::vector<double> anchor;   // [3*A] caller order, filled after k_rest_pose
};

}  // namespace

struct ob_ctx {
  std::string err;
  int n_worlds = 0;
  cudaStream_t stream = nullptr;
  DevCtx dev{};
  std::vector<WorldDesc> desc;
  std::vector<HostWorld> hw;
  std::vector<size_t> link_prefix, apple_prefix;   // caller-order prefix sums of n_links / n_apples (batched read-out)
  std::vector<WrenchSlots> wrench;       // host mirror (internal body indices)
  int dirty_lo = 0, dirty_hi = -1;
  WrenchSlots *staging[2] = {nullptr, nullptr};
  cudaEvent_t staging_ev[2] = {nullptr, nullptr};
  int staging_next = 0;
  unsigned char *dev_base = nullptr;
  // k_step launch geometry per size class: worlds [cls_off, cls_off + cls_n) of the order list
  int cls_off[kNumClasses] = {}, cls_n[kNumClasses] = {}, cls_grid[kNumClasses] = {}, cls_smem[kNumClasses] = {};
  int main_cls = 0, launches = 0, n_sm = 0;
  int max_Np = 0, max_Ap = 0;
  size_t ev_cap = 0, sum_ap = 0;
  uint64_t h2d_bytes = 0, d2h_bytes = 0, kernel_launches = 0, step_calls = 0;
  // size classes run concurrently: one internal stream per class, forked from and joined to the caller's stream
  cudaStream_t cls_stream[kNumClasses] = {};
  cudaEvent_t ev_fork = nullptr, ev_join[kNumClasses] = {};
  // pinned staging for the read-out calls (grown on demand)
  unsigned char *rd = nullptr;
  size_t rd_cap = 0;
};

namespace {

int fail(ob_ctx *c, int code, const char *fmt, ...) {
  if (c) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    c->err = buf;
  }
  return code;
}

thread_local std::string g_err;   // errors raised before a context exists

// every copy the library issues goes through here, so ob_counters can report the bytes moved
cudaError_t cpy(ob_ctx *c, void *dst, const void *src, size_t n, cudaMemcpyKind kind, cudaStream_t s) {
  if (kind == cudaMemcpyHostToDevice) c->h2d_bytes += n;
  else if (kind == cudaMemcpyDeviceToHost) c->d2h_bytes += n;
  return cudaMemcpyAsync(dst, src, n, kind, s);
}

int fail0(int code, const char *msg) {
  g_err = msg;
  return code;
}

int validate(const ob_world_spec *specs, int n_worlds, const ob_params *P, std::string &why) {
  char b[256];
  if (!specs || !P || n_worlds < 1) { why = "null specs/params or n_worlds < 1"; return OB_E_ARG; }
  if (!(P->h > 0.f) || !(P->cg_tol > 0.f) || P->cg_max_iter < 1 || P->rupture_frames < 1 || P->rupture_frames > 255 ||
      P->detach_frames_pull < 1 || P->detach_frames_pull > 255 || P->detach_frames_tension < 1 ||
      P->detach_frames_tension > 255 || !(P->react_max >= 0.f) || !(P->c_d >= 0.f) || !(P->mass_damping >= 0.f) || P->precond < 0 || P->precond > 2 || P->cg_norm < 0 || P->cg_norm > 1 || (P->precond == 2 && P->cg_norm == 1) ||
      !(P->fric_frac >= 0.f) || !(P->fric_ramp >= 0.f) || !(P->fric_time >= 0.f) || !(P->fric_veps > 0.f) ||
      !(P->snap_drag_scale >= 0.f) || !(P->rail_speed >= 0.f) || !(P->rail_fade >= 0.f) || !(P->rail_fade < 1.f) ||
      !(P->rail_brake >= 0.f)) {
    why = "ob_params out of range";
    return OB_E_ARG;
  }
  for (int w = 0; w < n_worlds; w++) {
    const ob_world_spec &s = specs[w];
    if (s.n_links < 1 || s.n_links > 32767 || !s.parent || !s.length || !s.diameter || !s.rest_quat) {
      snprintf(b, sizeof(b), "world %d: n_links out of range or null link arrays", w); why = b; return OB_E_ARG;
    }
    if (s.n_apples < 0 || s.n_apples > 1024 ||
        (s.n_apples > 0 && (!s.apple_link || !s.apple_offset || !s.apple_mass || !s.apple_k || !s.apple_detach))) {
      snprintf(b, sizeof(b), "world %d: n_apples out of range or null apple arrays", w); why = b; return OB_E_ARG;
    }
    if (!(s.density > 0.f) || !(s.E > 0.f) || !(s.MOR > 0.f)) {
      snprintf(b, sizeof(b), "world %d: density/E/MOR must be positive", w); why = b; return OB_E_ARG;
    }
    for (int i = 0; i < s.n_links; i++) {
      if ((i == 0 && s.parent[0] != -1) || (i > 0 && (s.parent[i] < 0 || s.parent[i] >= i))) {
        snprintf(b, sizeof(b), "world %d: parent[%d] = %d is not topological", w, i, s.parent[i]); why = b; return OB_E_ARG;
      }
      if (!(s.length[i] > 0.f) || !(s.diameter[i] > 0.f) || !std::isfinite(s.length[i]) || !std::isfinite(s.diameter[i])) {
        snprintf(b, sizeof(b), "world %d: link %d has non-positive length or diameter", w, i); why = b; return OB_E_ARG;
      }
      const float *q = s.rest_quat + 4 * i;
      double n = std::sqrt((double)q[0] * q[0] + (double)q[1] * q[1] + (double)q[2] * q[2] + (double)q[3] * q[3]);
      if (!(std::fabs(n - 1.0) <= 1e-3)) {
        snprintf(b, sizeof(b), "world %d: rest_quat[%d] is not a unit quaternion", w, i); why = b; return OB_E_ARG;
      }
      if (s.armature && (!(s.armature[2 * i] >= 0.f) || !(s.armature[2 * i + 1] >= 0.f))) {
        snprintf(b, sizeof(b), "world %d: negative armature on link %d", w, i); why = b; return OB_E_ARG;
      }
    }
    for (int a = 0; a < s.n_apples; a++) {
      if (s.apple_link[a] < 0 || s.apple_link[a] >= s.n_links || !(s.apple_mass[a] > 0.f) || !(s.apple_k[a] > 0.f) ||
          !(s.apple_detach[a] >= 0.f) || (s.apple_c && !(s.apple_c[a] >= 0.f))) {
        snprintf(b, sizeof(b), "world %d: apple %d has a bad link, mass, stiffness, damping or detach force", w, a);
        why = b; return OB_E_ARG;
      }
    }
  }
  return OB_OK;
}

// level order: plain breadth-first order -- parents before children, the links of one level contiguous and the
// children of one link contiguous (k_step gathers them as a range).  Returns the number of links with children.
int level_order(const ob_world_spec &s, std::vector<int32_t> &int2ext, std::vector<int32_t> &level_off) {
  const int N = s.n_links;
  std::vector<std::vector<int32_t>> kids(N);
  for (int i = 1; i < N; i++) kids[s.parent[i]].push_back(i);
  int2ext.clear();
  int2ext.reserve(N);
  level_off.clear();
  level_off.push_back(0);
  int2ext.push_back(0);
  size_t begin = 0;
  int n_inner = 0;
  while (begin < int2ext.size()) {
    size_t end = int2ext.size();
    level_off.push_back((int32_t)end);
    std::vector<int32_t> next;
    for (size_t k = begin; k < end; k++) {
      if (!kids[int2ext[k]].empty()) n_inner++;
      for (int32_t ch : kids[int2ext[k]]) next.push_back(ch);
    }
    int2ext.insert(int2ext.end(), next.begin(), next.end());
    begin = end;
  }
  return n_inner;
}
inline int pad8(int n) { return (n + 7) / 8 * 8; }
int count_factor_slots_raw(const ob_world_spec &s);
// padded number of factor slots a world is laid out with: 0 when it runs without the tree preconditioner, either by
// ob_params.precond or because the factor planes would not fit into one CTA's shared memory (it then runs Jacobi)
int world_factor_slots(const ob_world_spec &s, const ob_params &P, int Np, int Ap, int nlev) {
  if (P.precond != 2) return 0;
  const int NFp = pad8(count_factor_slots_raw(s));
  return step_smem_bytes(Np, Ap, NFp, nlev) <= kMaxSmem ? NFp : 0;
}

// links that need a factor slot for the tree preconditioner: links with children, and leaves that carry an apple off
// their axis (their articulated inertia is not a body of revolution)
int count_factor_slots_raw(const ob_world_spec &s) {
  std::vector<char> need(s.n_links, 0);
  for (int i = 1; i < s.n_links; i++) need[s.parent[i]] = 1;
  for (int a = 0; a < s.n_apples; a++)
    if (s.apple_offset[3 * a] != 0.f || s.apple_offset[3 * a + 1] != 0.f) need[s.apple_link[a]] = 1;
  int n = 0;
  for (char c : need) n += c;
  return n;
}

struct Layout {
  size_t total = 0;
  Pool desc, order, link_blk, link_cst, apple_blk, topo, topo2, quat_raw, quatd, Mmax, xprev, Lown, diam, Lown0, diam0, apple_off0, arm, link_ext, apple_ext, apple_nom,
      apple_c, anchor, level_off, info, wrench, events, ev_count, queue, iter_hist, stats, progress, pose7;
  size_t sumNp = 0, sumAp = 0, sumLev = 0, ev_cap = 0;
  int max_Np = 0, max_Ap = 0, max_smem = 0;
  bool any_arm = false;
};

void take(Layout &L, Pool &p, size_t bytes) {
  L.total = (L.total + kAlign - 1) / kAlign * kAlign;
  p.off = L.total;
  p.bytes = bytes;
  L.total += bytes;
}

int plan(const ob_world_spec *specs, int n_worlds, const ob_params *P, Layout &L, std::string &why) {
  size_t ev = 0;
  for (int w = 0; w < n_worlds; w++) {
    const ob_world_spec &s = specs[w];
    std::vector<int32_t> i2e, lev;
    level_order(s, i2e, lev);
    const int Np = pad16(s.n_links), Ap = pad16(s.n_apples), nlev = (int)lev.size() - 1;
    const int NFp = world_factor_slots(s, *P, Np, Ap, nlev);
    L.sumNp += Np; L.sumAp += Ap; L.sumLev += nlev + 1;
    L.max_Np = std::max(L.max_Np, Np); L.max_Ap = std::max(L.max_Ap, Ap);
    const int sm = step_smem_bytes(Np, Ap, NFp, nlev);
    int max_kids = 0;
    {
      std::vector<int> nk(s.n_links, 0);
      for (int i = 1; i < s.n_links; i++) max_kids = std::max(max_kids, ++nk[s.parent[i]]);
    }
    if (max_kids > kMaxChildren) {
      char b[160];
      snprintf(b, sizeof(b), "world %d: a link has %d children (limit %d)", w, max_kids, kMaxChildren);
      why = b;
      return OB_E_CAPACITY;
    }
    if (sm > kMaxSmem || step_class_of(Np, sm) < 0) {
      char b[200];
      snprintf(b, sizeof(b), "world %d (%d links, %d apples) does not fit on chip: %d B of shared memory (limit %d), "
               "%d links (limit %d)", w, s.n_links, s.n_apples, sm, kMaxSmem, s.n_links, kMaxLinksOnChip);
      why = b;
      return OB_E_CAPACITY;
    }
    L.max_smem = std::max(L.max_smem, sm);
    if (s.armature) L.any_arm = true;
    ev += (size_t)s.n_links + s.n_apples;
  }
  L.ev_cap = std::max<size_t>(ev, 64);
  take(L, L.desc, sizeof(WorldDesc) * n_worlds);
  take(L, L.order, sizeof(int32_t) * n_worlds);
  take(L, L.link_blk, (size_t)link_state_bytes(1) * L.sumNp);
  take(L, L.link_cst, (size_t)link_const_bytes(1) * L.sumNp);
  take(L, L.apple_blk, (size_t)apple_block_bytes(1) * std::max<size_t>(L.sumAp, 16));
  take(L, L.topo, sizeof(int4) * L.sumNp);
  take(L, L.topo2, sizeof(int4) * L.sumNp);
  take(L, L.quat_raw, sizeof(float4) * L.sumNp);
  take(L, L.quatd, sizeof(double) * 4 * L.sumNp);
  take(L, L.Mmax, sizeof(float) * L.sumNp);
  take(L, L.xprev, sizeof(float2) * 4 * L.sumNp);
  take(L, L.Lown, sizeof(float) * L.sumNp);
  take(L, L.diam, sizeof(float) * L.sumNp);
  take(L, L.Lown0, sizeof(float) * L.sumNp);
  take(L, L.diam0, sizeof(float) * L.sumNp);
  take(L, L.apple_off0, sizeof(float) * 3 * std::max<size_t>(L.sumAp, 16));
  take(L, L.arm, L.any_arm ? sizeof(float) * 2 * L.sumNp : 0);
  take(L, L.link_ext, sizeof(int32_t) * L.sumNp);
  take(L, L.apple_ext, sizeof(int32_t) * std::max<size_t>(L.sumAp, 16));
  take(L, L.apple_nom, sizeof(float) * 2 * std::max<size_t>(L.sumAp, 16));
  take(L, L.apple_c, sizeof(float) * std::max<size_t>(L.sumAp, 16));
  take(L, L.anchor, sizeof(double) * 3 * std::max<size_t>(L.sumAp, 16));
  take(L, L.level_off, sizeof(int32_t) * L.sumLev);
  take(L, L.info, sizeof(WorldInfo) * n_worlds);
  take(L, L.wrench, sizeof(WrenchSlots) * n_worlds);
  take(L, L.events, sizeof(ob_event) * L.ev_cap);
  take(L, L.ev_count, sizeof(int32_t) * 4);
  take(L, L.queue, sizeof(int32_t) * 2 * kNumClasses);
  take(L, L.iter_hist, sizeof(unsigned long long) * kIterHistBins);
  take(L, L.stats, sizeof(unsigned long long) * 4);
  take(L, L.progress, sizeof(int32_t) * n_worlds);
  take(L, L.pose7, sizeof(float) * 7 * L.max_Np);
  L.total = (L.total + kAlign - 1) / kAlign * kAlign;
  return OB_OK;
}

#define CU(call)                                                                                  \
  do {                                                                                            \
    cudaError_t e_ = (call);                                                                      \
    if (e_ != cudaSuccess) return fail(ctx, OB_E_CUDA, "%s: %s", #call, cudaGetErrorString(e_));  \
  } while (0)

int flush_wrenches(ob_ctx *ctx) {
  if (ctx->dirty_hi < ctx->dirty_lo) return OB_OK;
  const int lo = ctx->dirty_lo, n = ctx->dirty_hi - ctx->dirty_lo + 1;
  const int sidx = ctx->staging_next;
  ctx->staging_next ^= 1;
  CU(cudaEventSynchronize(ctx->staging_ev[sidx]));
  std::memcpy(ctx->staging[sidx] + lo, ctx->wrench.data() + lo, sizeof(WrenchSlots) * n);
  CU(cpy(ctx, const_cast<WrenchSlots *>(ctx->dev.wrench) + lo, ctx->staging[sidx] + lo, sizeof(WrenchSlots) * n,
                     cudaMemcpyHostToDevice, ctx->stream));
  CU(cudaEventRecord(ctx->staging_ev[sidx], ctx->stream));
  ctx->dirty_lo = 0;
  ctx->dirty_hi = -1;
  return OB_OK;
}

// pinned staging buffer of at least `bytes` bytes for a read-out call
int rd_reserve(ob_ctx *ctx, size_t bytes) {
  if (bytes <= ctx->rd_cap) return OB_OK;
  if (ctx->rd) cudaFreeHost(ctx->rd);
  ctx->rd = nullptr; ctx->rd_cap = 0;
  const size_t cap = (bytes + (1u << 20)) & ~(size_t)((1u << 20) - 1);
  CU(cudaHostAlloc((void **)&ctx->rd, cap, cudaHostAllocDefault));
  ctx->rd_cap = cap;
  return OB_OK;
}

int check_range(ob_ctx *ctx, int world0, int n) {
  if (!ctx) return OB_E_ARG;
  if (world0 < 0 || n < 1 || world0 + n > ctx->n_worlds) return fail(ctx, OB_E_ARG, "world range [%d, %d) out of range", world0, world0 + n);
  return OB_OK;
}

// rest hang points of every apple, device -> host mirror (caller order); synchronises
int fetch_anchors(ob_ctx *ctx) {
  std::vector<double> h_anchor(3 * ctx->sum_ap);
  CU(cpy(ctx, h_anchor.data(), ctx->dev.anchor, sizeof(double) * h_anchor.size(), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  for (int w = 0; w < ctx->n_worlds; w++) {
    const WorldDesc &d = ctx->desc[w];
    HostWorld &H = ctx->hw[w];
    H.anchor.resize(3 * (size_t)d.A);
    for (int a = 0; a < d.A; a++)
      for (int k = 0; k < 3; k++)
        H.anchor[3 * H.int2ext_apple[a] + k] = h_anchor[3 * (size_t)d.apple_base + (size_t)k * d.Ap + a];
  }
  return OB_OK;
}

int check_world(ob_ctx *ctx, int world) {
  if (!ctx) return OB_E_ARG;
  if (world < 0 || world >= ctx->n_worlds) return fail(ctx, OB_E_ARG, "world %d out of range", world);
  return OB_OK;
}

}  // namespace

extern "C" {

int ob_default_params(ob_params *p) {
  if (!p) return OB_E_ARG;
  std::memset(p, 0, sizeof(*p));
  p->h = 2e-3f;
  p->gravity[0] = 0.f; p->gravity[1] = 0.f; p->gravity[2] = -9.81f;
  p->c_d = 0.05f;
  p->cg_tol = 1e-6f;
  p->cg_max_iter = 200;
  p->precond = 2;
  p->rupture_frames = 3;
  p->detach_frames_pull = 3;
  p->detach_kappa = 1.1f;
  p->detach_frames_tension = 10;
  p->react_max = 40.f;
  p->tether_implicit = 1;
  p->qd_max = 50.f;
  p->zeta_s = 0.1f;
  p->forces_off_on_snapped = 1;
  p->mass_damping = 0.f;
  p->fric_frac = 0.f; p->fric_ramp = 5.f; p->fric_time = 1.5f; p->fric_veps = 1e-2f;
  p->snap_drag_scale = 1.f;
  p->rail_speed = 0.f; p->rail_fade = 0.5f; p->rail_brake = 50.f;
  return OB_OK;
}

int ob_workspace_bytes(const ob_world_spec *specs, int n_worlds, const ob_params *params, size_t *out) {
  std::string why;
  if (!out) return fail0(OB_E_ARG, "out is null");
  int rc = validate(specs, n_worlds, params, why);
  if (rc != OB_OK) return fail0(rc, why.c_str());
  Layout L;
  rc = plan(specs, n_worlds, params, L, why);
  if (rc != OB_OK) return fail0(rc, why.c_str());
  *out = L.total;
  return OB_OK;
}

int ob_create(const ob_world_spec *specs, int n_worlds, const ob_params *params, void *dev_workspace,
              size_t workspace_bytes, void *cuda_stream, ob_ctx **out) {
  std::string why;
  if (!out) return fail0(OB_E_ARG, "out is null");
  *out = nullptr;
  int rc = validate(specs, n_worlds, params, why);
  if (rc != OB_OK) return fail0(rc, why.c_str());
  Layout L;
  rc = plan(specs, n_worlds, params, L, why);
  if (rc != OB_OK) return fail0(rc, why.c_str());
  if (!dev_workspace || workspace_bytes < L.total || ((uintptr_t)dev_workspace % kAlign) != 0)
    return fail0(OB_E_WORKSPACE, "workspace null, misaligned (256 B) or smaller than ob_workspace_bytes");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return fail0(OB_E_CUDA, "no CUDA device: there is no CPU fallback");

  ob_ctx *ctx = new ob_ctx();
  ctx->n_worlds = n_worlds;
  ctx->stream = (cudaStream_t)cuda_stream;
  ctx->dev_base = (unsigned char *)dev_workspace;
  ctx->max_Np = L.max_Np; ctx->max_Ap = L.max_Ap;
  ctx->ev_cap = L.ev_cap;
  ctx->desc.resize(n_worlds);
  ctx->hw.resize(n_worlds);
  ctx->wrench.assign(n_worlds, WrenchSlots{});
  ctx->link_prefix.assign(n_worlds + 1, 0);
  ctx->apple_prefix.assign(n_worlds + 1, 0);
  for (int w = 0; w < n_worlds; w++) {
    ctx->link_prefix[w + 1] = ctx->link_prefix[w] + (size_t)specs[w].n_links;
    ctx->apple_prefix[w + 1] = ctx->apple_prefix[w] + (size_t)specs[w].n_apples;
  }
  unsigned char *base = ctx->dev_base;

  // ---- host images of every pool ----
  std::vector<unsigned char> h_link(L.link_blk.bytes, 0), h_apple(L.apple_blk.bytes, 0);
  std::vector<int4> h_topo(L.sumNp, make_int4(-1, 0, 0, 0)), h_topo2(L.sumNp, make_int4(0, -1, 0, 0));
  std::vector<float4> h_quat_raw(L.sumNp, make_float4(1.f, 0.f, 0.f, 0.f));
  std::vector<float> h_Lown(L.sumNp, 1.f), h_diam(L.sumNp, 1.f), h_arm(L.any_arm ? 2 * L.sumNp : 0, 0.f);
  std::vector<int32_t> h_link_ext(L.sumNp, 0), h_apple_ext(std::max<size_t>(L.sumAp, 16), 0), h_lev(L.sumLev, 0);
  std::vector<float> h_nom(2 * std::max<size_t>(L.sumAp, 16), 0.f), h_c(std::max<size_t>(L.sumAp, 16), 0.f);
  std::vector<float> h_off0(3 * std::max<size_t>(L.sumAp, 16), 0.f);
  std::vector<int32_t> h_order(n_worlds);
  size_t link_base = 0, apple_base = 0, lev_base = 0, link_off = 0, apple_off = 0;
  for (int w = 0; w < n_worlds; w++) {
    const ob_world_spec &s = specs[w];
    HostWorld &H = ctx->hw[w];
    std::vector<int32_t> lev;
    level_order(s, H.int2ext_link, lev);
    const int N = s.n_links, A = s.n_apples, Np = pad16(N), Ap = pad16(A), nlev = (int)lev.size() - 1;
    H.ext2int_link.assign(N, 0);
    for (int i = 0; i < N; i++) H.ext2int_link[H.int2ext_link[i]] = i;
    // apples sorted by internal link (stable), so each link's apples are contiguous
    H.int2ext_apple.resize(A);
    for (int a = 0; a < A; a++) H.int2ext_apple[a] = a;
    std::stable_sort(H.int2ext_apple.begin(), H.int2ext_apple.end(), [&](int32_t x, int32_t y) {
      return H.ext2int_link[s.apple_link[x]] < H.ext2int_link[s.apple_link[y]];
    });
    H.ext2int_apple.assign(A, 0);
    for (int a = 0; a < A; a++) H.ext2int_apple[H.int2ext_apple[a]] = a;

    WorldDesc &d = ctx->desc[w];
    d.N = N; d.A = A; d.Np = Np; d.Ap = Ap; d.NFp = world_factor_slots(s, *params, Np, Ap, nlev); d.n_levels = nlev;
    d.precond = params->precond == 2 && d.NFp == 0 && count_factor_slots_raw(s) > 0 ? 1 : params->precond;
    d.n_top = 0;
    while (d.n_top < nlev && lev[d.n_top + 1] <= 32) d.n_top++;
    d.cls = step_class_of(Np, step_smem_bytes(Np, Ap, d.NFp, nlev));
    d.link_base = (int32_t)link_base; d.apple_base = (int32_t)apple_base; d.level_base = (int32_t)lev_base;
    d.link_blk_off = (int64_t)link_off; d.apple_blk_off = (int64_t)apple_off;
    d.density = s.density; d.E = s.E; d.MOR = s.MOR;
    d.has_apple_c = s.apple_c ? 1 : 0;

    std::vector<int32_t> n_child(N, 0), first_apple(N, 0), n_apple(N, 0), islot(N, 0xffff), par(N, -1);
    std::vector<std::vector<int32_t>> kids(N);
    for (int i = 1; i < N; i++) {
      par[i] = H.ext2int_link[s.parent[H.int2ext_link[i]]];
      kids[par[i]].push_back(i);          // ascending internal index: a fixed summation order
    }
    std::vector<char> offax(N, 0);
    for (int a = 0; a < A; a++)
      if (s.apple_offset[3 * a] != 0.f || s.apple_offset[3 * a + 1] != 0.f) offax[H.ext2int_link[s.apple_link[a]]] = 1;
    for (int i = 0, slot = 0; i < N; i++) {
      n_child[i] = (int32_t)kids[i].size();
      if (n_child[i] || offax[i]) islot[i] = slot++;
    }
    for (int a = 0; a < A; a++) {
      const int l = H.ext2int_link[s.apple_link[H.int2ext_apple[a]]];
      if (n_apple[l] == 0) first_apple[l] = a;
      n_apple[l]++;
    }
    std::vector<int32_t> level_of(N, 0);
    for (int l = 0; l < nlev; l++)
      for (int i = lev[l]; i < lev[l + 1]; i++) level_of[i] = l;
    for (int i = 0; i < N; i++) {
      const int e = H.int2ext_link[i];
      const int p = par[i];
      h_topo[link_base + i] = make_int4(p, n_child[i] ? kids[i][0] : 0, level_of[i], n_child[i]);
      h_topo2[link_base + i] = make_int4(first_apple[i] | (n_apple[i] << 16),
                                         islot[i], 0, 0);
      const float *q = s.rest_quat + 4 * e;
      const double n = std::sqrt((double)q[0] * q[0] + (double)q[1] * q[1] + (double)q[2] * q[2] + (double)q[3] * q[3]);
      h_quat_raw[link_base + i] = make_float4(q[0], q[1], q[2], q[3]);
      h_Lown[link_base + i] = s.length[e];
      h_diam[link_base + i] = s.diameter[e];
      h_link_ext[link_base + i] = e;
      if (L.any_arm && s.armature) {
        h_arm[2 * link_base + i] = s.armature[2 * e];
        h_arm[2 * link_base + Np + i] = s.armature[2 * e + 1];
      }
    }
    for (int l = 0; l <= nlev; l++) h_lev[lev_base + l] = lev[l];
    unsigned char *ab = h_apple.data() + apple_off;
    float *aconst = reinterpret_cast<float *>(ab + apple_state_bytes(Ap));
    int32_t *alink = reinterpret_cast<int32_t *>(ab + apple_state_bytes(Ap) + 7 * 4 * Ap);
    for (int a = 0; a < A; a++) {
      const int e = H.int2ext_apple[a];
      for (int k = 0; k < 3; k++) h_off0[3 * apple_base + k * Ap + a] = aconst[k * Ap + a] = s.apple_offset[3 * e + k];
      aconst[3 * Ap + a] = s.apple_k[e];
      aconst[4 * Ap + a] = s.apple_mass[e];
      aconst[6 * Ap + a] = s.apple_detach[e];
      alink[a] = H.ext2int_link[s.apple_link[e]];
      h_apple_ext[apple_base + a] = e;
      h_nom[2 * apple_base + a] = s.apple_mass[e];
      h_nom[2 * apple_base + Ap + a] = s.apple_detach[e];
      h_c[apple_base + a] = s.apple_c ? s.apple_c[e] : 0.f;
    }
    for (int a = A; a < Ap; a++) { aconst[3 * Ap + a] = 1.f; aconst[4 * Ap + a] = 1.f; alink[a] = 0; }
    link_base += Np; apple_base += Ap; lev_base += nlev + 1;
    link_off += link_state_bytes(Np); apple_off += apple_block_bytes(Ap);
    h_order[w] = w;
  }
  // work-queue order: grouped by size class, largest worlds first inside a class (longest-processing-time rule)
  std::stable_sort(h_order.begin(), h_order.end(), [&](int a, int b) {
    if (ctx->desc[a].cls != ctx->desc[b].cls) return ctx->desc[a].cls < ctx->desc[b].cls;
    return ctx->desc[a].N > ctx->desc[b].N;
  });
  for (int k = 0; k < n_worlds; k++) {
    const WorldDesc &d = ctx->desc[h_order[k]];
    if (ctx->cls_n[d.cls]++ == 0) ctx->cls_off[d.cls] = k;
    ctx->cls_smem[d.cls] = std::max(ctx->cls_smem[d.cls], step_smem_bytes(d.Np, d.Ap, d.NFp, d.n_levels));
  }

  DevCtx &D = ctx->dev;
  D.n_worlds = n_worlds;
  D.desc = reinterpret_cast<WorldDesc *>(base + L.desc.off);
  D.order = reinterpret_cast<int32_t *>(base + L.order.off);
  D.link_blk = base + L.link_blk.off;
  D.link_cst = base + L.link_cst.off;
  D.apple_blk = base + L.apple_blk.off;
  D.topo = reinterpret_cast<int4 *>(base + L.topo.off);
  D.topo2 = reinterpret_cast<int4 *>(base + L.topo2.off);
  D.quat_raw = reinterpret_cast<float4 *>(base + L.quat_raw.off);
  D.quatd = reinterpret_cast<double *>(base + L.quatd.off);
  D.Mmax = reinterpret_cast<float *>(base + L.Mmax.off);
  D.xprev = reinterpret_cast<float2 *>(base + L.xprev.off);
  D.sum_np = (int32_t)L.sumNp;
  D.Lown = reinterpret_cast<float *>(base + L.Lown.off);
  D.diam = reinterpret_cast<float *>(base + L.diam.off);
  D.Lown0 = reinterpret_cast<float *>(base + L.Lown0.off);
  D.diam0 = reinterpret_cast<float *>(base + L.diam0.off);
  D.apple_off0 = reinterpret_cast<float *>(base + L.apple_off0.off);
  D.arm = L.any_arm ? reinterpret_cast<float *>(base + L.arm.off) : nullptr;
  D.link_ext = reinterpret_cast<int32_t *>(base + L.link_ext.off);
  D.apple_ext = reinterpret_cast<int32_t *>(base + L.apple_ext.off);
  D.apple_nominal = reinterpret_cast<float *>(base + L.apple_nom.off);
  D.apple_c_in = reinterpret_cast<float *>(base + L.apple_c.off);
  D.anchor = reinterpret_cast<double *>(base + L.anchor.off);
  D.level_off = reinterpret_cast<int32_t *>(base + L.level_off.off);
  D.info = reinterpret_cast<WorldInfo *>(base + L.info.off);
  D.wrench = reinterpret_cast<WrenchSlots *>(base + L.wrench.off);
  D.events = reinterpret_cast<ob_event *>(base + L.events.off);
  D.ev_cap = (int32_t)std::min<size_t>(L.ev_cap, 0x7fffffff);
  D.ev_count = reinterpret_cast<int32_t *>(base + L.ev_count.off);
  D.queue = reinterpret_cast<int32_t *>(base + L.queue.off);
  D.iter_hist = reinterpret_cast<unsigned long long *>(base + L.iter_hist.off);
  D.stats = reinterpret_cast<unsigned long long *>(base + L.stats.off);
  D.progress = reinterpret_cast<int32_t *>(base + L.progress.off);
  D.pose7 = reinterpret_cast<float *>(base + L.pose7.off);
  D.P = *params;

#define UP(pool, vec)                                                                                        \
  do {                                                                                                       \
    if ((pool).bytes && !(vec).empty()) {                                                                    \
      cudaError_t e_ = cpy(ctx, base + (pool).off, (vec).data(),                                      \
                                       std::min((pool).bytes, (vec).size() * sizeof((vec)[0])),              \
                                       cudaMemcpyHostToDevice, ctx->stream);                                 \
      if (e_ != cudaSuccess) { g_err = cudaGetErrorString(e_); delete ctx; return OB_E_CUDA; }               \
    }                                                                                                        \
  } while (0)
  cudaError_t e = cudaMemsetAsync(base, 0, L.total, ctx->stream);
  if (e != cudaSuccess) { g_err = cudaGetErrorString(e); delete ctx; return OB_E_CUDA; }
  UP(L.desc, ctx->desc); UP(L.order, h_order); UP(L.link_blk, h_link); UP(L.apple_blk, h_apple); UP(L.topo, h_topo); UP(L.topo2, h_topo2);
  UP(L.quat_raw, h_quat_raw); UP(L.Lown, h_Lown); UP(L.diam, h_diam); UP(L.Lown0, h_Lown); UP(L.diam0, h_diam); UP(L.apple_off0, h_off0); UP(L.arm, h_arm); UP(L.link_ext, h_link_ext);
  UP(L.apple_ext, h_apple_ext); UP(L.apple_nom, h_nom); UP(L.apple_c, h_c); UP(L.level_off, h_lev);
#undef UP
  e = cudaStreamSynchronize(ctx->stream);   // the host images die at the end of this call
  if (e == cudaSuccess) e = launch_rest_pose(D, 0, 0, ctx->stream);
  if (e == cudaSuccess) e = launch_anchors(D, ctx->stream);
  if (e == cudaSuccess) e = launch_randomize(D, 0ull, 0, ctx->stream);
  ctx->kernel_launches += 3;
  ctx->sum_ap = std::max<size_t>(L.sumAp, 16);
  // launch geometry of k_step
  int n_sm = 0, dev = 0;
  if (e == cudaSuccess) e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  ctx->n_sm = n_sm;
  for (int k = 0; k < kNumClasses && e == cudaSuccess; k++) {
    if (!ctx->cls_n[k]) continue;
    int per_sm = 0;
    e = step_kernel_setup(k, ctx->cls_smem[k], &per_sm);
    if (e == cudaSuccess && per_sm < 1) e = cudaErrorInvalidConfiguration;
    ctx->cls_grid[k] = std::max(1, std::min(ctx->cls_n[k], n_sm * std::max(per_sm, 1)));
    if (ctx->cls_n[k] > ctx->cls_n[ctx->main_cls]) ctx->main_cls = k;
  }
  int n_cls_used = 0;
  for (int k = 0; k < kNumClasses; k++) n_cls_used += ctx->cls_n[k] > 0;
  if (n_cls_used > 1) {          // heterogeneous batch: the size classes run side by side (ob_step forks and joins)
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
    for (int k = 0; k < kNumClasses && e == cudaSuccess; k++) {
      if (!ctx->cls_n[k]) continue;
      e = cudaStreamCreateWithFlags(&ctx->cls_stream[k], cudaStreamNonBlocking);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join[k], cudaEventDisableTiming);
    }
  }
  for (int k = 0; k < 2 && e == cudaSuccess; k++) {
    e = cudaHostAlloc((void **)&ctx->staging[k], sizeof(WrenchSlots) * n_worlds, cudaHostAllocDefault);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->staging_ev[k], cudaEventDisableTiming);
  }
  // the rest hang points come back (they change only with ob_randomize_geometry)
  if (e == cudaSuccess && fetch_anchors(ctx) != OB_OK) e = cudaErrorUnknown;
  if (e != cudaSuccess) {
    g_err = std::string("ob_create: ") + cudaGetErrorString(e);
    ob_destroy(ctx);
    return OB_E_CUDA;
  }
  *out = ctx;
  return OB_OK;
}

int ob_randomize(ob_ctx *ctx, uint64_t seed) {
  if (!ctx) return OB_E_ARG;
  for (auto &wv : ctx->wrench) wv = WrenchSlots{};
  ctx->dirty_lo = 0;
  ctx->dirty_hi = ctx->n_worlds - 1;
  int rc = flush_wrenches(ctx);
  if (rc != OB_OK) return rc;
  CU(launch_randomize(ctx->dev, (unsigned long long)seed, 1, ctx->stream));
  ctx->kernel_launches += 1;
  return OB_OK;
}

int ob_randomize_geometry(ob_ctx *ctx, uint64_t seed, const ob_geometry_ranges *ranges) {
  if (!ctx) return OB_E_ARG;
  if (!ranges) return fail(ctx, OB_E_ARG, "ranges is null");
  const float *f = reinterpret_cast<const float *>(ranges);
  for (int k = 0; k < 16; k++)
    if (!std::isfinite(f[k])) return fail(ctx, OB_E_ARG, "non-finite geometry range");
  for (int k = 8; k < 16; k++)
    if (!(f[k] > 0.f)) return fail(ctx, OB_E_ARG, "dimension factors must be positive");
  for (auto &wv : ctx->wrench) wv = WrenchSlots{};
  ctx->dirty_lo = 0;
  ctx->dirty_hi = ctx->n_worlds - 1;
  int rc = flush_wrenches(ctx);
  if (rc != OB_OK) return rc;
  CU(launch_geometry(ctx->dev, (unsigned long long)seed, *ranges, ctx->stream));
  CU(launch_anchors(ctx->dev, ctx->stream));
  CU(launch_randomize(ctx->dev, 0ull, 2, ctx->stream));       // derived constants, reset; materials kept
  ctx->kernel_launches += 3;
  return fetch_anchors(ctx);
}

int ob_get_geometry(ob_ctx *ctx, int world, float *length, float *diameter, double *rest_quat, float *apple_offset) {
  int rc = check_world(ctx, world);
  if (rc != OB_OK) return rc;
  const WorldDesc &d = ctx->desc[world];
  const HostWorld &H = ctx->hw[world];
  std::vector<float> L(d.Np), dm(d.Np), ao(3 * (size_t)std::max(d.Ap, 1));
  std::vector<double> q(4 * (size_t)d.Np);
  CU(cpy(ctx, L.data(), ctx->dev.Lown + d.link_base, sizeof(float) * d.Np, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cpy(ctx, dm.data(), ctx->dev.diam + d.link_base, sizeof(float) * d.Np, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cpy(ctx, q.data(), ctx->dev.quatd + 4 * (size_t)d.link_base, sizeof(double) * 4 * d.Np, cudaMemcpyDeviceToHost, ctx->stream));
  if (d.Ap)
    CU(cpy(ctx, ao.data(), ctx->dev.apple_blk + d.apple_blk_off + apple_state_bytes(d.Ap), sizeof(float) * 3 * d.Ap,
           cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  for (int i = 0; i < d.N; i++) {
    const int e = H.int2ext_link[i];
    if (length) length[e] = L[i];
    if (diameter) diameter[e] = dm[i];
    if (rest_quat) for (int k = 0; k < 4; k++) rest_quat[4 * e + k] = q[4 * (size_t)i + k];
  }
  if (apple_offset)
    for (int a = 0; a < d.A; a++)
      for (int k = 0; k < 3; k++) apple_offset[3 * H.int2ext_apple[a] + k] = ao[(size_t)k * d.Ap + a];
  return OB_OK;
}

int ob_apply_wrench(ob_ctx *ctx, int world, int body, const float point[3], const float force[3]) {
  int rc = check_world(ctx, world);
  if (rc != OB_OK) return rc;
  if (!force) return fail(ctx, OB_E_ARG, "force is null");
  const WorldDesc &d = ctx->desc[world];
  if (body < 0 || body >= d.N + d.A) return fail(ctx, OB_E_ARG, "world %d: body %d out of range", world, body);
  const HostWorld &H = ctx->hw[world];
  const int ib = body < d.N ? H.ext2int_link[body] : d.N + H.ext2int_apple[body - d.N];
  WrenchSlots &W = ctx->wrench[world];
  int slot = -1;
  for (int k = 0; k < W.n; k++)
    if (W.body[k] == ib) slot = k;
  const bool zero = force[0] == 0.f && force[1] == 0.f && force[2] == 0.f;
  if (zero) {
    if (slot < 0) return OB_OK;
    const int last = W.n - 1;    // keep the active slots dense
    W.body[slot] = W.body[last];
    for (int k = 0; k < 3; k++) { W.point[slot][k] = W.point[last][k]; W.force[slot][k] = W.force[last][k]; }
    W.n = last;
  } else {
    if (slot < 0) {
      if (W.n >= OB_MAX_WRENCH) return fail(ctx, OB_E_CAPACITY, "world %d: all %d wrench slots in use", world, OB_MAX_WRENCH);
      slot = W.n++;
    }
    W.body[slot] = ib;
    for (int k = 0; k < 3; k++) { W.point[slot][k] = point ? point[k] : 0.f; W.force[slot][k] = force[k]; }
  }
  if (ctx->dirty_hi < ctx->dirty_lo) { ctx->dirty_lo = world; ctx->dirty_hi = world; }
  else { ctx->dirty_lo = std::min(ctx->dirty_lo, world); ctx->dirty_hi = std::max(ctx->dirty_hi, world); }
  return OB_OK;
}

int ob_apply_wrench_batch(ob_ctx *ctx, int n, const int32_t *world, const int32_t *body, const float *point3,
                          const float *force3) {
  if (!ctx) return OB_E_ARG;
  if (n < 0 || (n > 0 && (!world || !body || !force3))) return fail(ctx, OB_E_ARG, "null batch arrays");
  for (int k = 0; k < n; k++) {
    int rc = ob_apply_wrench(ctx, world[k], body[k], point3 ? point3 + 3 * k : nullptr, force3 + 3 * k);
    if (rc != OB_OK) return rc;
  }
  return OB_OK;
}

int ob_flush(ob_ctx *ctx) {
  if (!ctx) return OB_E_ARG;
  return flush_wrenches(ctx);
}

int ob_step(ob_ctx *ctx, int n) {
  if (!ctx) return OB_E_ARG;
  if (n < 0) return fail(ctx, OB_E_ARG, "n < 0");
  if (n == 0) return OB_OK;
  int rc = flush_wrenches(ctx);
  if (rc != OB_OK) return rc;
  CU(cudaMemsetAsync(ctx->dev.queue, 0, sizeof(int32_t) * kNumClasses, ctx->stream));
  CU(cudaMemsetAsync(ctx->dev.progress, 0, sizeof(int32_t) * ctx->n_worlds, ctx->stream));
  ctx->launches = 0;
  // A heterogeneous batch has one persistent kernel per size class.  They go to streams of their own, forked from and
  // joined to the caller's stream, so that the CTAs of the next class move in as the CTAs of a class run out of work
  // (back to back on one stream every class would drain to its own tail while the others wait).
  const bool fork = ctx->ev_fork != nullptr;
  if (fork) CU(cudaEventRecord(ctx->ev_fork, ctx->stream));
  for (int k = kNumClasses - 1; k >= 0; k--) {      // the class of the largest worlds first
    if (!ctx->cls_n[k]) continue;
    // Queue items: the n steps of a world are cut into chunks that different CTAs may take.  Long items amortise the
    // staging of a world (25 steps per item measured best on configs[3]: 7.48 M against 7.33 M with 10 and 7.36 M
    // uncut), short ones keep the tail of the launch, where CTAs run out of work, small: at least ~12 items per CTA.
    const int want = (12 * ctx->cls_grid[k] + ctx->cls_n[k] - 1) / ctx->cls_n[k];
    const int n_chunks = std::max(1, std::min(std::min(8, (n + 4) / 5), std::max((n + 24) / 25, want)));
    cudaStream_t st = fork ? ctx->cls_stream[k] : ctx->stream;
    if (fork) CU(cudaStreamWaitEvent(st, ctx->ev_fork, 0));
    CU(launch_step(ctx->dev, k, ctx->dev.order + ctx->cls_off[k], ctx->cls_n[k], ctx->dev.queue + k, n,
                   ctx->cls_grid[k], ctx->cls_smem[k], ctx->n_sm, n_chunks, ctx->dev.progress, st));
    if (fork) {
      CU(cudaEventRecord(ctx->ev_join[k], st));
      CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_join[k], 0));
    }
    ctx->launches += 1;
    ctx->kernel_launches += 1;
  }
  ctx->step_calls += 1;
  return OB_OK;
}

// ------------------------------------------------------------------------------------------------------
// read-out.  The state pools keep the worlds back to back, so a range of worlds is ONE device -> host copy per pool
// (link state, apple blocks, WorldInfo) into pinned staging and ONE stream synchronisation; the host then scatters
// into the caller's order.  The per-world calls are the range calls with n = 1.
// ------------------------------------------------------------------------------------------------------
}  // extern "C"

namespace {

struct RdView {
  const unsigned char *link = nullptr, *apple = nullptr;   // staged copies; index with the world's pool offset - base
  const WorldInfo *info = nullptr;
  const float *pose = nullptr;
  size_t link0 = 0, apple0 = 0;
};

// stage the pools of worlds [w0, w0 + n): async copies + one synchronise
int rd_fetch(ob_ctx *ctx, int w0, int n, bool links, bool apples, bool info, int pose_world, RdView &v) {
  const WorldDesc &a = ctx->desc[w0], &b = ctx->desc[w0 + n - 1];
  const size_t lbytes = links ? (size_t)(b.link_blk_off - a.link_blk_off) + link_state_bytes(b.Np) : 0;
  const size_t abytes = apples ? (size_t)(b.apple_blk_off - a.apple_blk_off) + apple_block_bytes(b.Ap) : 0;
  const size_t ibytes = info ? sizeof(WorldInfo) * (size_t)n : 0;
  const size_t pbytes = pose_world >= 0 ? sizeof(float) * 7 * (size_t)ctx->desc[pose_world].N : 0;
  auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
  int rc = rd_reserve(ctx, up(lbytes) + up(abytes) + up(ibytes) + up(pbytes) + 256);
  if (rc != OB_OK) return rc;
  unsigned char *p = ctx->rd;
  if (pose_world >= 0) {
    CU(launch_pose(ctx->dev, pose_world, ctx->stream));
    ctx->kernel_launches += 1;
  }
  if (lbytes) { CU(cpy(ctx, p, ctx->dev.link_blk + a.link_blk_off, lbytes, cudaMemcpyDeviceToHost, ctx->stream)); v.link = p; p += up(lbytes); }
  if (abytes) { CU(cpy(ctx, p, ctx->dev.apple_blk + a.apple_blk_off, abytes, cudaMemcpyDeviceToHost, ctx->stream)); v.apple = p; p += up(abytes); }
  if (ibytes) { CU(cpy(ctx, p, ctx->dev.info + w0, ibytes, cudaMemcpyDeviceToHost, ctx->stream)); v.info = reinterpret_cast<const WorldInfo *>(p); p += up(ibytes); }
  if (pbytes) { CU(cpy(ctx, p, ctx->dev.pose7, pbytes, cudaMemcpyDeviceToHost, ctx->stream)); v.pose = reinterpret_cast<const float *>(p); p += up(pbytes); }
  CU(cudaStreamSynchronize(ctx->stream));
  v.link0 = (size_t)a.link_blk_off; v.apple0 = (size_t)a.apple_blk_off;
  return OB_OK;
}

// rest sag m g / k_s of one apple in fp64 from the fp32 constants: apple positions cross the ABI as
// anchor + sag + u (the kernel stores u = x - x_rest in fp32)
inline double sag_of(const float *aconst, int Ap, int a, float g) {
  return (double)aconst[4 * Ap + a] * (double)g / (double)aconst[3 * Ap + a];
}

int get_state_impl(ob_ctx *ctx, int w0, int n, float *q, float *qd, float *apple_x, double *apple_x64, float *apple_v,
                   uint8_t *ruptured, uint8_t *attached, int32_t *info, float *link_pose7) {
  int rc = check_range(ctx, w0, n);
  if (rc != OB_OK) return rc;
  RdView v;
  const bool links = q || qd || ruptured, apples = apple_x || apple_x64 || apple_v || attached;
  rc = rd_fetch(ctx, w0, n, links, apples, info != nullptr, link_pose7 ? w0 : -1, v);
  if (rc != OB_OK) return rc;
  const size_t L0 = ctx->link_prefix[w0], A0 = ctx->apple_prefix[w0];
  const float *g = ctx->dev.P.gravity;
#pragma omp parallel for schedule(static) if (n > 64)
  for (int k = 0; k < n; k++) {
    const int w = w0 + k;
    const WorldDesc &d = ctx->desc[w];
    const HostWorld &H = ctx->hw[w];
    const size_t lo = ctx->link_prefix[w] - L0, ao = ctx->apple_prefix[w] - A0;
    if (links) {
      const unsigned char *lb = v.link + ((size_t)d.link_blk_off - v.link0);
      const float *st = reinterpret_cast<const float *>(lb);
      const unsigned char *fl = lb + kLinkStateFloats * 4 * d.Np;
      for (int i = 0; i < d.N; i++) {
        const size_t e = lo + H.int2ext_link[i];
        if (q) { q[2 * e] = st[2 * i]; q[2 * e + 1] = st[2 * i + 1]; }
        if (qd) { qd[2 * e] = st[2 * d.Np + 2 * i]; qd[2 * e + 1] = st[2 * d.Np + 2 * i + 1]; }
        if (ruptured) ruptured[e] = fl[i];
      }
    }
    if (apples && d.A) {
      const unsigned char *ab = v.apple + ((size_t)d.apple_blk_off - v.apple0);
      const float *as = reinterpret_cast<const float *>(ab);
      const unsigned char *af = ab + 6 * 4 * d.Ap;
      const float *ac = reinterpret_cast<const float *>(ab + apple_state_bytes(d.Ap));
      for (int a = 0; a < d.A; a++) {
        const size_t e = ao + H.int2ext_apple[a];
        for (int c = 0; c < 3; c++) {
          if (apple_x || apple_x64) {
            const double x = H.anchor[3 * (size_t)H.int2ext_apple[a] + c] + sag_of(ac, d.Ap, a, g[c]) + (double)as[c * d.Ap + a];
            if (apple_x) apple_x[3 * e + c] = (float)x;
            if (apple_x64) apple_x64[3 * e + c] = x;
          }
          if (apple_v) apple_v[3 * e + c] = as[(3 + c) * d.Ap + a];
        }
        if (attached) attached[e] = af[a];
      }
    }
    if (info) { info[3 * k] = v.info[k].step; info[3 * k + 1] = v.info[k].last_iters; info[3 * k + 2] = v.info[k].status; }
  }
  if (link_pose7) {
    const WorldDesc &d = ctx->desc[w0];
    const HostWorld &H = ctx->hw[w0];
    for (int i = 0; i < d.N; i++) std::memcpy(link_pose7 + 7 * H.int2ext_link[i], v.pose + 7 * i, 7 * sizeof(float));
  }
  return OB_OK;
}

// read-modify-write of one world's state blocks (everything the caller passes as NULL is kept)
int set_state_impl(ob_ctx *ctx, int world, const float *q, const float *qd, const float *apple_x, const double *apple_x64,
                   const float *apple_v, const uint8_t *ruptured, const uint8_t *attached, const int32_t *step,
                   const int32_t *rupture_step = nullptr) {
  int rc = check_world(ctx, world);
  if (rc != OB_OK) return rc;
  const WorldDesc &d = ctx->desc[world];
  const HostWorld &H = ctx->hw[world];
  RdView v;
  rc = rd_fetch(ctx, world, 1, true, d.Ap > 0, true, -1, v);
  if (rc != OB_OK) return rc;
  std::vector<unsigned char> lb(v.link, v.link + link_state_bytes(d.Np));
  std::vector<unsigned char> ab;
  if (d.Ap) ab.assign(v.apple, v.apple + apple_block_bytes(d.Ap));
  WorldInfo wi = v.info[0];
  float *st = reinterpret_cast<float *>(lb.data());
  int32_t *rs = reinterpret_cast<int32_t *>(st + 4 * d.Np);          // step of the rupture per link
  unsigned char *fl = lb.data() + kLinkStateFloats * 4 * d.Np;
  for (int i = 0; i < d.N; i++) {
    const int e = H.int2ext_link[i];
    if (q) { st[2 * i] = q[2 * e]; st[2 * i + 1] = q[2 * e + 1]; }
    if (qd) { st[2 * d.Np + 2 * i] = qd[2 * e]; st[2 * d.Np + 2 * i + 1] = qd[2 * e + 1]; }
    if (ruptured) { fl[i] = ruptured[e] ? 1 : 0; fl[d.Np + i] = 0; rs[i] = step ? *step : wi.step; }
    if (rupture_step) rs[i] = rupture_step[e];
  }
  if (d.Ap) {
    float *as = reinterpret_cast<float *>(ab.data());
    unsigned char *af = ab.data() + 6 * 4 * d.Ap;
    const float *ac = reinterpret_cast<const float *>(ab.data() + apple_state_bytes(d.Ap));
    const float *g = ctx->dev.P.gravity;
    for (int a = 0; a < d.A; a++) {
      const int e = H.int2ext_apple[a];
      for (int c = 0; c < 3; c++) {
        if (apple_x64) as[c * d.Ap + a] = (float)(apple_x64[3 * e + c] - H.anchor[3 * e + c] - sag_of(ac, d.Ap, a, g[c]));
        else if (apple_x) as[c * d.Ap + a] = (float)((double)apple_x[3 * e + c] - H.anchor[3 * e + c] - sag_of(ac, d.Ap, a, g[c]));
        if (apple_v) as[(3 + c) * d.Ap + a] = apple_v[3 * e + c];
      }
      if (attached) { af[a] = attached[e] ? 1 : 0; af[d.Ap + a] = 0; af[2 * d.Ap + a] = 0; }
    }
  }
  // status bits are cleared by ob_set_state only (a new state is a new start); ob_set_step, ob_set_rupture_steps and
  // ob_set_apple_x64 keep them: a frozen world stays frozen
  if (!step && !rupture_step && !apple_x64) wi.status = 0;
  if (step) wi.step = *step;
  if ((!step && !rupture_step) || q || qd || apple_x || apple_x64 || apple_v || ruptured || attached)
    for (int k = 0; k < 4; k++)   // ... and forget the solution history the PCG start vector is extrapolated from
      CU(cudaMemsetAsync(ctx->dev.xprev + (size_t)k * ctx->dev.sum_np + d.link_base, 0, sizeof(float2) * d.Np, ctx->stream));
  CU(cpy(ctx, ctx->dev.link_blk + d.link_blk_off, lb.data(), lb.size(), cudaMemcpyHostToDevice, ctx->stream));
  if (d.Ap)
    CU(cpy(ctx, ctx->dev.apple_blk + d.apple_blk_off, ab.data(), apple_state_bytes(d.Ap), cudaMemcpyHostToDevice, ctx->stream));
  CU(cpy(ctx, ctx->dev.info + world, &wi, sizeof(wi), cudaMemcpyHostToDevice, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  return OB_OK;
}

// exact per-world checkpoint: every byte of mutable state, solver memory included
struct BlobHeader { uint32_t magic; int32_t N, A, Np, Ap; uint32_t bytes; };
constexpr uint32_t kBlobMagic = 0x4f42574cu;   // "OBWL"
size_t blob_bytes(const WorldDesc &d) {
  return sizeof(BlobHeader) + link_state_bytes(d.Np) + apple_state_bytes(d.Ap) + sizeof(WorldInfo) + 4 * sizeof(float2) * (size_t)d.Np;
}

}  // namespace

extern "C" {

int ob_get_state(ob_ctx *ctx, int world, float *q, float *qd, float *apple_x, float *apple_v, uint8_t *ruptured,
                 uint8_t *attached, float *link_pose7, int32_t *info) {
  return get_state_impl(ctx, world, 1, q, qd, apple_x, nullptr, apple_v, ruptured, attached, info, link_pose7);
}

int ob_get_state_batch(ob_ctx *ctx, int world0, int n_worlds, float *q, float *qd, float *apple_x, double *apple_x64,
                       float *apple_v, uint8_t *ruptured, uint8_t *attached, int32_t *info) {
  return get_state_impl(ctx, world0, n_worlds, q, qd, apple_x, apple_x64, apple_v, ruptured, attached, info, nullptr);
}

int ob_get_apple_x64(ob_ctx *ctx, int world, double *apple_x) {
  if (ctx && !apple_x) return fail(ctx, OB_E_ARG, "apple_x is null");
  return get_state_impl(ctx, world, 1, nullptr, nullptr, nullptr, apple_x, nullptr, nullptr, nullptr, nullptr, nullptr);
}

int ob_set_state(ob_ctx *ctx, int world, const float *q, const float *qd, const float *apple_x, const float *apple_v,
                 const uint8_t *ruptured, const uint8_t *attached) {
  return set_state_impl(ctx, world, q, qd, apple_x, nullptr, apple_v, ruptured, attached, nullptr);
}

int ob_set_apple_x64(ob_ctx *ctx, int world, const double *apple_x) {
  if (ctx && !apple_x) return fail(ctx, OB_E_ARG, "apple_x is null");
  return set_state_impl(ctx, world, nullptr, nullptr, nullptr, apple_x, nullptr, nullptr, nullptr, nullptr);
}

int ob_set_step(ob_ctx *ctx, int world, int32_t step) {
  if (ctx && step < 0) return fail(ctx, OB_E_ARG, "step < 0");
  return set_state_impl(ctx, world, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, &step);
}

int ob_get_rupture_steps(ob_ctx *ctx, int world, int32_t *rupture_step) {
  int rc = check_world(ctx, world);
  if (rc != OB_OK) return rc;
  if (!rupture_step) return fail(ctx, OB_E_ARG, "rupture_step is null");
  const WorldDesc &d = ctx->desc[world];
  RdView v;
  rc = rd_fetch(ctx, world, 1, true, false, false, -1, v);
  if (rc != OB_OK) return rc;
  const int32_t *rs = reinterpret_cast<const int32_t *>(v.link) + 4 * d.Np;
  for (int i = 0; i < d.N; i++) rupture_step[ctx->hw[world].int2ext_link[i]] = rs[i];
  return OB_OK;
}

int ob_set_rupture_steps(ob_ctx *ctx, int world, const int32_t *rupture_step) {
  if (ctx && !rupture_step) return fail(ctx, OB_E_ARG, "rupture_step is null");
  return set_state_impl(ctx, world, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, rupture_step);
}

int ob_world_blob_bytes(ob_ctx *ctx, int world, size_t *out) {
  int rc = check_world(ctx, world);
  if (rc != OB_OK) return rc;
  if (!out) return fail(ctx, OB_E_ARG, "out is null");
  *out = blob_bytes(ctx->desc[world]);
  return OB_OK;
}

int ob_save_world(ob_ctx *ctx, int world, void *buf, size_t cap) {
  int rc = check_world(ctx, world);
  if (rc != OB_OK) return rc;
  const WorldDesc &d = ctx->desc[world];
  const size_t need = blob_bytes(d);
  if (!buf || cap < need) return fail(ctx, OB_E_ARG, "checkpoint buffer null or smaller than ob_world_blob_bytes (%zu)", need);
  unsigned char *p = static_cast<unsigned char *>(buf);
  BlobHeader h{kBlobMagic, d.N, d.A, d.Np, d.Ap, (uint32_t)need};
  std::memcpy(p, &h, sizeof(h)); p += sizeof(h);
  CU(cpy(ctx, p, ctx->dev.link_blk + d.link_blk_off, link_state_bytes(d.Np), cudaMemcpyDeviceToHost, ctx->stream)); p += link_state_bytes(d.Np);
  if (d.Ap) CU(cpy(ctx, p, ctx->dev.apple_blk + d.apple_blk_off, apple_state_bytes(d.Ap), cudaMemcpyDeviceToHost, ctx->stream));
  p += apple_state_bytes(d.Ap);
  CU(cpy(ctx, p, ctx->dev.info + world, sizeof(WorldInfo), cudaMemcpyDeviceToHost, ctx->stream)); p += sizeof(WorldInfo);
  for (int k = 0; k < 4; k++) {
    CU(cpy(ctx, p, ctx->dev.xprev + (size_t)k * ctx->dev.sum_np + d.link_base, sizeof(float2) * d.Np, cudaMemcpyDeviceToHost, ctx->stream));
    p += sizeof(float2) * d.Np;
  }
  CU(cudaStreamSynchronize(ctx->stream));
  return OB_OK;
}

int ob_load_world(ob_ctx *ctx, int world, const void *buf, size_t bytes) {
  int rc = check_world(ctx, world);
  if (rc != OB_OK) return rc;
  const WorldDesc &d = ctx->desc[world];
  const size_t need = blob_bytes(d);
  BlobHeader h{};
  if (buf && bytes >= sizeof(h)) std::memcpy(&h, buf, sizeof(h));
  if (!buf || bytes < need || h.magic != kBlobMagic || h.N != d.N || h.A != d.A || h.Np != d.Np || h.Ap != d.Ap || h.bytes != need)
    return fail(ctx, OB_E_ARG, "world %d: not a checkpoint of this world (size or header mismatch)", world);
  const unsigned char *p = static_cast<const unsigned char *>(buf) + sizeof(h);
  CU(cpy(ctx, ctx->dev.link_blk + d.link_blk_off, p, link_state_bytes(d.Np), cudaMemcpyHostToDevice, ctx->stream)); p += link_state_bytes(d.Np);
  if (d.Ap) CU(cpy(ctx, ctx->dev.apple_blk + d.apple_blk_off, p, apple_state_bytes(d.Ap), cudaMemcpyHostToDevice, ctx->stream));
  p += apple_state_bytes(d.Ap);
  // of the WorldInfo in the blob only the mutable words are restored (step, last_iters, status); the target world's
  // material draws (E, MOR, density) and its totals since ob_create (steps_taken, cg_iters) are not part of a checkpoint
  static_assert(offsetof(WorldInfo, steps_taken) == 3 * sizeof(int32_t), "step, last_iters, status lead WorldInfo");
  CU(cpy(ctx, ctx->dev.info + world, p, 3 * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream)); p += sizeof(WorldInfo);
  for (int k = 0; k < 4; k++) {
    CU(cpy(ctx, ctx->dev.xprev + (size_t)k * ctx->dev.sum_np + d.link_base, p, sizeof(float2) * d.Np, cudaMemcpyHostToDevice, ctx->stream));
    p += sizeof(float2) * d.Np;
  }
  CU(cudaStreamSynchronize(ctx->stream));
  return OB_OK;
}

int ob_get_counters_batch(ob_ctx *ctx, int world0, int n_worlds, int32_t *rupture_count, int32_t *pull_count,
                          int32_t *tension_count) {
  int rc = check_range(ctx, world0, n_worlds);
  if (rc != OB_OK) return rc;
  RdView v;
  rc = rd_fetch(ctx, world0, n_worlds, rupture_count != nullptr, pull_count || tension_count, false, -1, v);
  if (rc != OB_OK) return rc;
  const size_t L0 = ctx->link_prefix[world0], A0 = ctx->apple_prefix[world0];
  for (int k = 0; k < n_worlds; k++) {
    const int w = world0 + k;
    const WorldDesc &d = ctx->desc[w];
    const HostWorld &H = ctx->hw[w];
    if (rupture_count) {
      const unsigned char *fl = v.link + ((size_t)d.link_blk_off - v.link0) + kLinkStateFloats * 4 * d.Np;
      for (int i = 0; i < d.N; i++) rupture_count[ctx->link_prefix[w] - L0 + H.int2ext_link[i]] = fl[d.Np + i];
    }
    if ((pull_count || tension_count) && d.A) {
      const unsigned char *af = v.apple + ((size_t)d.apple_blk_off - v.apple0) + 6 * 4 * d.Ap;
      for (int a = 0; a < d.A; a++) {
        const size_t e = ctx->apple_prefix[w] - A0 + H.int2ext_apple[a];
        if (pull_count) pull_count[e] = af[d.Ap + a];
        if (tension_count) tension_count[e] = af[2 * d.Ap + a];
      }
    }
  }
  return OB_OK;
}

int ob_get_counters(ob_ctx *ctx, int world, int32_t *rupture_count, int32_t *pull_count, int32_t *tension_count) {
  return ob_get_counters_batch(ctx, world, 1, rupture_count, pull_count, tension_count);
}

int ob_set_counters(ob_ctx *ctx, int world, const int32_t *rupture_count, const int32_t *pull_count,
                    const int32_t *tension_count) {
  int rc = check_world(ctx, world);
  if (rc != OB_OK) return rc;
  const WorldDesc &d = ctx->desc[world];
  const HostWorld &H = ctx->hw[world];
  RdView v;
  rc = rd_fetch(ctx, world, 1, true, d.Ap > 0, false, -1, v);
  if (rc != OB_OK) return rc;
  std::vector<unsigned char> lf(v.link + kLinkStateFloats * 4 * d.Np, v.link + link_state_bytes(d.Np)), af(std::max(3 * d.Ap, 1));
  if (d.Ap) std::memcpy(af.data(), v.apple + 6 * 4 * d.Ap, 3 * (size_t)d.Ap);
  auto clampc = [](int32_t x) { return (unsigned char)std::min(std::max(x, 0), 255); };
  if (rupture_count)
    for (int i = 0; i < d.N; i++) lf[d.Np + i] = clampc(rupture_count[H.int2ext_link[i]]);
  for (int a = 0; a < d.A; a++) {
    if (pull_count) af[d.Ap + a] = clampc(pull_count[H.int2ext_apple[a]]);
    if (tension_count) af[2 * d.Ap + a] = clampc(tension_count[H.int2ext_apple[a]]);
  }
  CU(cpy(ctx, ctx->dev.link_blk + d.link_blk_off + kLinkStateFloats * 4 * d.Np, lf.data(), lf.size(),
         cudaMemcpyHostToDevice, ctx->stream));
  if (d.Ap)
    CU(cpy(ctx, ctx->dev.apple_blk + d.apple_blk_off + 6 * 4 * d.Ap, af.data(), 3 * d.Ap, cudaMemcpyHostToDevice,
           ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  return OB_OK;
}

int ob_get_material_batch(ob_ctx *ctx, int world0, int n_worlds, float *emr, float *apple_detach, float *apple_mass) {
  int rc = check_range(ctx, world0, n_worlds);
  if (rc != OB_OK) return rc;
  RdView v;
  rc = rd_fetch(ctx, world0, n_worlds, false, apple_detach || apple_mass, emr != nullptr, -1, v);
  if (rc != OB_OK) return rc;
  const size_t A0 = ctx->apple_prefix[world0];
  for (int k = 0; k < n_worlds; k++) {
    const int w = world0 + k;
    const WorldDesc &d = ctx->desc[w];
    const HostWorld &H = ctx->hw[w];
    if (emr) { emr[3 * k] = v.info[k].E; emr[3 * k + 1] = v.info[k].MOR; emr[3 * k + 2] = v.info[k].density; }
    if ((apple_detach || apple_mass) && d.A) {
      const float *ac = reinterpret_cast<const float *>(v.apple + ((size_t)d.apple_blk_off - v.apple0) + apple_state_bytes(d.Ap));
      for (int a = 0; a < d.A; a++) {
        const size_t e = ctx->apple_prefix[w] - A0 + H.int2ext_apple[a];
        if (apple_mass) apple_mass[e] = ac[4 * d.Ap + a];
        if (apple_detach) apple_detach[e] = ac[6 * d.Ap + a];
      }
    }
  }
  return OB_OK;
}

int ob_get_material(ob_ctx *ctx, int world, float *emr, float *apple_detach, float *apple_mass) {
  return ob_get_material_batch(ctx, world, 1, emr, apple_detach, apple_mass);
}

int ob_events(ob_ctx *ctx, ob_event *buf, int cap, int *n_out) {
  if (!ctx) return OB_E_ARG;
  if (!n_out || cap < 0 || (cap > 0 && !buf)) return fail(ctx, OB_E_ARG, "null output");
  int32_t cnt[2] = {0, 0};
  CU(cpy(ctx, cnt, ctx->dev.ev_count, sizeof(cnt), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  const int have = (int)std::min<long long>(cnt[0], (long long)ctx->dev.ev_cap);
  std::vector<ob_event> ev(have);
  if (have) {
    CU(cpy(ctx, ev.data(), ctx->dev.events, sizeof(ob_event) * have, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
  }
  std::sort(ev.begin(), ev.end(), [](const ob_event &a, const ob_event &b) {
    if (a.step != b.step) return a.step < b.step;
    if (a.world != b.world) return a.world < b.world;
    if (a.kind != b.kind) return a.kind < b.kind;
    return a.index < b.index;
  });
  const int n = std::min(have, cap);
  if (n) std::memcpy(buf, ev.data(), sizeof(ob_event) * n);
  *n_out = n;
  // keep what did not fit, in sorted order, at the head of the device list
  const int rest = have - n;
  if (rest) CU(cpy(ctx, ctx->dev.events, ev.data() + n, sizeof(ob_event) * rest, cudaMemcpyHostToDevice, ctx->stream));
  int32_t newcnt[2] = {rest, 0};
  CU(cpy(ctx, ctx->dev.ev_count, newcnt, sizeof(newcnt), cudaMemcpyHostToDevice, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  if (cnt[1] || cnt[0] > ctx->dev.ev_cap) return fail(ctx, OB_E_CAPACITY, "device event list overflowed (capacity %d)", ctx->dev.ev_cap);
  return OB_OK;
}

int ob_stats(ob_ctx *ctx, uint64_t *cg_iters_total, uint64_t *world_steps_total, int32_t *n_flagged) {
  if (!ctx) return OB_E_ARG;
  int rc = rd_reserve(ctx, 256);
  if (rc != OB_OK) return rc;
  CU(launch_stats(ctx->dev, ctx->stream));             // totals reduced on the device: one 24-byte copy
  ctx->kernel_launches += 1;
  unsigned long long *t = reinterpret_cast<unsigned long long *>(ctx->rd);
  CU(cpy(ctx, t, ctx->dev.stats, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  if (cg_iters_total) *cg_iters_total = t[0];
  if (world_steps_total) *world_steps_total = t[1];
  if (n_flagged) *n_flagged = (int32_t)t[2];
  return OB_OK;
}

int ob_iter_histogram(ob_ctx *ctx, uint64_t *bins, int n_bins, int reset) {
  if (!ctx) return OB_E_ARG;
  if (!bins || n_bins < 1) return fail(ctx, OB_E_ARG, "bins is null or n_bins < 1");
  int rc = rd_reserve(ctx, sizeof(unsigned long long) * kIterHistBins);
  if (rc != OB_OK) return rc;
  unsigned long long *t = reinterpret_cast<unsigned long long *>(ctx->rd);
  CU(cpy(ctx, t, ctx->dev.iter_hist, sizeof(unsigned long long) * kIterHistBins, cudaMemcpyDeviceToHost, ctx->stream));
  if (reset) CU(cudaMemsetAsync(ctx->dev.iter_hist, 0, sizeof(unsigned long long) * kIterHistBins, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  for (int k = 0; k < n_bins; k++) bins[k] = 0;
  for (int k = 0; k < kIterHistBins; k++) bins[std::min(k, n_bins - 1)] += t[k];
  return OB_OK;
}

int ob_launch_info(ob_ctx *ctx, int32_t *n_launches, int32_t *grid, int32_t *block, int32_t *smem_bytes) {
  if (!ctx) return OB_E_ARG;
  if (n_launches) *n_launches = ctx->launches;
  if (grid) *grid = ctx->cls_grid[ctx->main_cls];
  if (block) *block = kStepClasses[ctx->main_cls].nt;
  if (smem_bytes) *smem_bytes = ctx->cls_smem[ctx->main_cls];
  return OB_OK;
}

int ob_counters(ob_ctx *ctx, uint64_t out[4]) {
  if (!ctx) return OB_E_ARG;
  if (!out) return fail(ctx, OB_E_ARG, "out is null");
  out[0] = ctx->h2d_bytes; out[1] = ctx->d2h_bytes; out[2] = ctx->kernel_launches; out[3] = ctx->step_calls;
  return OB_OK;
}

int ob_sizeof_params(void) { return (int)sizeof(ob_params); }
int ob_sizeof_world_spec(void) { return (int)sizeof(ob_world_spec); }
int ob_sizeof_event(void) { return (int)sizeof(ob_event); }
int ob_sizeof_geometry_ranges(void) { return (int)sizeof(ob_geometry_ranges); }

int ob_selftest_philox(int n, const uint32_t *ctr, const uint32_t *key, uint32_t *out_lib, uint32_t *out_curand,
                       void *dev_scratch, void *cuda_stream) {
  if (n < 1 || !ctr || !key || !out_lib || !out_curand || !dev_scratch) return fail0(OB_E_ARG, "ob_selftest_philox: null or empty");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::vector<uint32_t> in(6 * (size_t)n), out(8 * (size_t)n);
  for (int i = 0; i < n; i++) {
    for (int k = 0; k < 4; k++) in[6 * (size_t)i + k] = ctr[4 * (size_t)i + k];
    for (int k = 0; k < 2; k++) in[6 * (size_t)i + 4 + k] = key[2 * (size_t)i + k];
  }
  uint32_t *d_in = reinterpret_cast<uint32_t *>(dev_scratch), *d_out = d_in + 6 * (size_t)n;
  cudaError_t e = cudaMemcpyAsync(d_in, in.data(), in.size() * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = launch_philox_selftest(n, d_in, d_out, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(out.data(), d_out, out.size() * 4, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return fail0(OB_E_CUDA, cudaGetErrorString(e));
  for (int i = 0; i < n; i++)
    for (int k = 0; k < 4; k++) {
      out_lib[4 * (size_t)i + k] = out[8 * (size_t)i + k];
      out_curand[4 * (size_t)i + k] = out[8 * (size_t)i + 4 + k];
    }
  return OB_OK;
}

// ob_selftest_philox without any allocation: the staging area is the static device array of ob_kernels.cu, which is
// also where the set-up (cudaGetSymbolAddress, once per device) and the launch live.  Sizes are checked here, before
// the GPU is touched.
int ob_selftest_philox_static(int n, const uint32_t *ctr, const uint32_t *key, uint32_t *out_lib, uint32_t *out_curand,
                              void *cuda_stream) {
  if (n < 1 || !ctr || !key || !out_lib || !out_curand) return fail0(OB_E_ARG, "ob_selftest_philox_static: null or empty");
  if (n > OB_SELFTEST_STATIC_MAX) {
    char b[160];
    snprintf(b, sizeof(b), "ob_selftest_philox_static: n = %d exceeds the static scratch (OB_SELFTEST_STATIC_MAX = %d pairs); "
             "split the call or use ob_selftest_philox", n, OB_SELFTEST_STATIC_MAX);
    return fail0(OB_E_CAPACITY, b);
  }
  cudaError_t e = philox_selftest_static(n, ctr, key, out_lib, out_curand, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return fail0(OB_E_CUDA, cudaGetErrorString(e));
  return OB_OK;
}

const char *ob_last_error(const ob_ctx *ctx) { return ctx ? ctx->err.c_str() : (g_err.empty() ? kNullCtx : g_err.c_str()); }

void ob_destroy(ob_ctx *ctx) {
  if (!ctx) return;
  cudaStreamSynchronize(ctx->stream);
  for (int k = 0; k < 2; k++) {
    if (ctx->staging[k]) cudaFreeHost(ctx->staging[k]);
    if (ctx->staging_ev[k]) cudaEventDestroy(ctx->staging_ev[k]);
  }
  for (int k = 0; k < kNumClasses; k++) {
    if (ctx->cls_stream[k]) { cudaStreamSynchronize(ctx->cls_stream[k]); cudaStreamDestroy(ctx->cls_stream[k]); }
    if (ctx->ev_join[k]) cudaEventDestroy(ctx->ev_join[k]);
  }
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  if (ctx->rd) cudaFreeHost(ctx->rd);
  delete ctx;
}

}  // extern "C"
