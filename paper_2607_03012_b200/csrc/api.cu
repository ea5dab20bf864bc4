// C-ABI glue: size queries, hva_sparse_attention dispatch, hva_forward orchestration (include/hva.h).
// Stage order follows the data flow the paper implies:
// cluster (Alg. 2) -> mask (Eq. 2-3) -> merge (Alg. 1, takes M as input l.134) -> plan/permute (Eq. 1)
// -> attention + inverse permutation (Eq. 4).  Everything is enqueued on one stream, no host sync.
#include "common.cuh"
#include <cmath>
#include <mutex>

namespace {

struct FwdLayout {
  // persistent per-tensor state (index 0 = Q, 1 = K)
  size_t assign[2], mu[2], sums[2], sizes[2], subset[2], state_total;
  // per-call workspace
  size_t lowe, mask, group_of, n_groups, group_mask, plan, qp, kp, vp, scratch, scratch_bytes, ws_total;
  int Nq, Nk, n, BH, m;
  bool fuse_q;
  hva_plan_layout PL;
};

// hva_cluster_qk / hva_forward cluster Q and K on two streams (fork / join by events, legal under stream capture): the second
// persistent assignment kernel fills the SMs as the first one's CTAs drain, and the small finalize launches of one tensor run
// under the other's pass.  One side stream + two events per device, created on first use; a call only enqueues on them.
struct SideStream {
  cudaStream_t st = nullptr;
  cudaEvent_t fork = nullptr, mid = nullptr, join = nullptr;
  bool tried = false, ok = false;
  std::mutex busy;   // held while a call enqueues its fork .. join sequence
  void create() {
    tried = true;
    ok = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) == cudaSuccess &&
         cudaEventCreateWithFlags(&fork, cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&mid, cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&join, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) cudaGetLastError();
  }
};
SideStream* side_stream() {
  static SideStream tab[64];
  static std::mutex table;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
  std::lock_guard<std::mutex> g(table);
  if (!tab[dev].tried) tab[dev].create();
  return tab[dev].ok ? &tab[dev] : nullptr;
}

bool valid_shape(const hva_shape* s) {
  return s && s->B >= 1 && s->heads >= 1 && s->T >= 1 && s->H >= 1 && s->W >= 1 && (s->D == 64 || s->D == 128) &&
         (s->dtype == HVA_F32 || s->dtype == HVA_BF16);
}
bool valid_config(const hva_config* c) {
  if (!c) return false;
  for (int a = 0; a < 3; ++a)
    if (c->cell_q[a] < 1 || c->cell_k[a] < 1 || c->win_q[a] < 1 || c->win_k[a] < 1) return false;
  return c->iters >= 1 && c->tile_q >= 1 && c->tile_k >= 1 && c->top_p > 0.f && c->min_kc >= 0.f && c->min_kc <= 1.f &&
         c->merge_rounds >= 0 && c->max_q_tiles >= 0 && c->subset_frac >= 0.f && c->subset_frac <= 1.f;
}

int make_layout(const hva_shape* s, const hva_config* c, FwdLayout* F) {
  const size_t es = s->dtype == HVA_F32 ? 4 : 2;
  F->n = s->T * s->H * s->W; F->BH = s->B * s->heads;
  F->Nq = hva_num_clusters(s, c->cell_q); F->Nk = hva_num_clusters(s, c->cell_k);
  F->m = (int)std::floor((double)c->subset_frac * (double)F->n + 0.5);   // m = floor(f n + 1/2)  (R-H2)
  const size_t BH = F->BH, n = F->n, D = s->D;
  size_t o = 0;
  auto take = [&](size_t b) { size_t r = o; o += hva_align(b); return r; };
  for (int t = 0; t < 2; ++t) {
    const size_t Nc = t ? F->Nk : F->Nq;
    F->assign[t] = take(BH * n * 4); F->mu[t] = take(BH * Nc * D * 4); F->sums[t] = take(BH * Nc * D * 4);
    F->sizes[t] = take(BH * Nc * 4); F->subset[t] = take(BH * (size_t)(F->m > 0 ? F->m : 1) * 4);
  }
  F->state_total = o;
  const int Nqp = F->Nq > 1 ? F->Nq : 1, Nkp = F->Nk > 1 ? F->Nk : 1;
  HVA_TRY(hva_plan_describe(F->BH, F->n, Nqp, Nkp, c->tile_q, &F->PL));
  o = 0;
  F->lowe = take(BH * n * 4); F->mask = take(BH * (size_t)F->Nq * F->Nk); F->group_of = take(BH * F->Nq * 4);
  F->n_groups = take(BH * 4); F->group_mask = take(BH * (size_t)F->Nq * F->Nk); F->plan = take(F->PL.total);
  // Q' is never materialised on the tensor-pipe path: the attention kernel gathers the Q rows through perm_q (TMA gather4)
  F->fuse_q = s->dtype == HVA_BF16 && s->D == 128 && c->tile_q == 128 && c->tile_k == 128 && !(c->flags & HVA_FLAG_ATTN_SIMT);
  F->qp = take(F->fuse_q ? 0 : BH * n * D * es); F->kp = take(BH * n * D * es); F->vp = take(BH * n * D * es);
  HvaGrid gq = hva_make_grid(s, c->cell_q, c->win_q), gk = hva_make_grid(s, c->cell_k, c->win_k);
  size_t sc = hva_cluster_ws_bytes(gq, F->BH, s->D);
  sc = std::max(sc, hva_cluster_ws_bytes(gk, F->BH, s->D));
  sc = std::max(sc, hva_merge_ws_bytes(F->BH, F->Nq, F->Nk));
  sc = std::max(sc, hva_plan_ws_bytes(F->BH, F->n, F->Nq, F->Nk));
  sc = std::max(sc, hva_hybrid_ws_bytes(F->BH, F->n, std::max(F->Nq, F->Nk), F->m, s->D));
  F->scratch_bytes = sc; F->scratch = take(sc);
  F->ws_total = o;
  return HVA_OK;
}

}  // namespace

extern "C" const char* hva_strerror(int code) {
  switch (code) {
    case HVA_OK: return "ok";
    case HVA_EINVAL: return "invalid argument";
    case HVA_EWORKSPACE: return "workspace / plan / state buffer too small";
    case HVA_EUNSUPPORTED: return "unsupported dtype / tile / size combination";
    case HVA_ECUDA: return "CUDA runtime error";
    case HVA_ELIMIT: return "problem exceeds the built-in scratch of a *_static entry point (use the variant that takes a workspace)";
    default: return "unknown error";
  }
}
extern "C" int hva_version(void) { return 100; }

extern "C" int32_t hva_num_clusters(const hva_shape* s, const int32_t cell[3]) {
  if (!s || !cell || cell[0] < 1 || cell[1] < 1 || cell[2] < 1) return HVA_EINVAL;
  return ((s->T + cell[0] - 1) / cell[0]) * ((s->H + cell[1] - 1) / cell[1]) * ((s->W + cell[2] - 1) / cell[2]);
}

extern "C" size_t hva_workspace_bytes(const hva_shape* s, const hva_config* c) {
  if (!valid_shape(s) || !valid_config(c)) return 0;
  FwdLayout F;
  if (make_layout(s, c, &F) != HVA_OK) return 0;
  // without a caller-provided state buffer the per-tensor arrays also live in the workspace
  return F.ws_total + F.state_total;
}
extern "C" size_t hva_state_bytes(const hva_shape* s, const hva_config* c) {
  if (!valid_shape(s) || !valid_config(c)) return 0;
  FwdLayout F;
  if (make_layout(s, c, &F) != HVA_OK) return 0;
  return F.state_total;
}
extern "C" int hva_state_describe(const hva_shape* s, const hva_config* c, hva_state_layout* out) {
  if (!valid_shape(s) || !valid_config(c) || !out) return HVA_EINVAL;
  FwdLayout F;
  HVA_TRY(make_layout(s, c, &F));
  for (int t = 0; t < 2; ++t) {
    out->assign[t] = F.assign[t]; out->mu[t] = F.mu[t]; out->sums[t] = F.sums[t]; out->sizes[t] = F.sizes[t];
    out->subset[t] = F.subset[t];
  }
  out->n_clusters[0] = F.Nq; out->n_clusters[1] = F.Nk; out->m = F.m; out->total = F.state_total;
  return HVA_OK;
}
extern "C" int hva_workspace_describe(const hva_shape* s, const hva_config* c, hva_workspace_layout* out) {
  if (!valid_shape(s) || !valid_config(c) || !out) return HVA_EINVAL;
  FwdLayout F;
  HVA_TRY(make_layout(s, c, &F));
  out->lowe = F.lowe; out->mask = F.mask; out->group_of = F.group_of; out->n_groups = F.n_groups; out->group_mask = F.group_mask;
  out->plan = F.plan; out->plan_bytes = F.PL.total; out->qp = F.qp; out->kp = F.kp; out->vp = F.vp; out->scratch = F.scratch;
  out->state = F.ws_total; out->total = F.ws_total + F.state_total;
  return HVA_OK;
}
extern "C" size_t hva_plan_workspace_bytes(int32_t BH, int32_t n, int32_t Nq, int32_t Nk) {
  if (BH < 1 || n < 1 || Nq < 1 || Nk < 1) return 0;
  return hva_plan_ws_bytes(BH, n, Nq, Nk);
}

extern "C" int hva_sparse_attention(const hva_shape* s, const hva_config* c, const void* Qp, const void* Kp, const void* Vp,
                                    const void* plan, size_t plan_bytes, int32_t Nq, int32_t Nk, void* O,
                                    int32_t unpermute, void* ws, size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  if (!valid_shape(s) || !valid_config(c) || !Qp || !Kp || !Vp || !plan || !O || Nq < 1 || Nk < 1) return HVA_EINVAL;
  const int n = s->T * s->H * s->W, BH = s->B * s->heads;
  hva_plan_layout L;
  HVA_TRY(hva_plan_describe(BH, n, Nq, Nk, c->tile_q, &L));
  if (plan_bytes < L.total) return HVA_EWORKSPACE;
  const float scale = c->softmax_scale > 0.f ? c->softmax_scale : 1.0f / sqrtf((float)s->D);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const bool tc_ok = s->dtype == HVA_BF16 && s->D == 128 && c->tile_q == 128 && c->tile_k == 128;
  if (tc_ok && !(c->flags & HVA_FLAG_ATTN_SIMT))
    return hva_attention_tc_launch(s, scale, Qp, Kp, Vp, plan, L, Nq, Nk, O, unpermute, (c->flags & HVA_FLAG_Q_UNPERMUTED) != 0, st);
  if (c->flags & HVA_FLAG_Q_UNPERMUTED) return HVA_EUNSUPPORTED;
  return hva_attention_simt_launch(s, scale, Qp, Kp, Vp, plan, L, Nq, Nk, O, unpermute, st, c->tile_q);
}

extern "C" int hva_cluster_qk(const hva_shape* s, const hva_config* c, const void* Q, const void* K, int32_t* assign_q, float* mu_q,
                              int32_t* sizes_q, float* sums_q, int32_t* assign_k, float* mu_k, int32_t* sizes_k, float* sums_k, void* ws_q,
                              size_t ws_q_bytes, void* ws_k, size_t ws_k_bytes, void* stream) {
  if (!valid_shape(s) || !valid_config(c) || !Q || !K || !ws_q || !ws_k) return HVA_EINVAL;
  {   // the two scratch regions must not overlap
    const char *a = (const char*)ws_q, *b = (const char*)ws_k;
    if (a < b + ws_k_bytes && b < a + ws_q_bytes) return HVA_EINVAL;
  }
  if (ws_q_bytes < hva_cluster_workspace_bytes(s, c->cell_q, c->win_q) || ws_k_bytes < hva_cluster_workspace_bytes(s, c->cell_k, c->win_k))
    return HVA_EWORKSPACE;   // before the fork: nothing may fail between fork and join for a reason known up front
  SideStream* side = side_stream();
  if (!side) return HVA_ECUDA;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  std::lock_guard<std::mutex> g(side->busy);
  if (cudaEventRecord(side->fork, st) != cudaSuccess || cudaStreamWaitEvent(side->st, side->fork, 0) != cudaSuccess) return HVA_ECUDA;
  int rc = hva_cluster_ex(s, c->cell_q, c->win_q, c->iters, Q, nullptr, assign_q, mu_q, sizes_q, sums_q, nullptr, c->flags, nullptr, ws_q,
                          ws_q_bytes, stream);
  const int rk = hva_cluster_ex(s, c->cell_k, c->win_k, c->iters, K, nullptr, assign_k, mu_k, sizes_k, sums_k, nullptr, c->flags, nullptr,
                                ws_k, ws_k_bytes, side->st);
  // join even after an error: the side stream must not stay forked (stream capture)
  if (cudaEventRecord(side->join, side->st) != cudaSuccess || cudaStreamWaitEvent(st, side->join, 0) != cudaSuccess) return HVA_ECUDA;
  return rc != HVA_OK ? rc : rk;
}

namespace {
int forward_impl(const hva_shape* s, const hva_config* c, const void* Q, const void* K, const void* V, void* O, int32_t step_kind,
                 void* state, hva_stats* stats_out, void* ws, size_t ws_bytes, void* stream, int bh0) {
  if (!valid_shape(s) || !valid_config(c) || !Q || !K || !V || !O || !ws) return HVA_EINVAL;
  if (step_kind != HVA_ANCHOR && step_kind != HVA_INTERMEDIATE && step_kind != HVA_DENSE) return HVA_EINVAL;
  if (step_kind == HVA_INTERMEDIATE && (!state || c->subset_frac <= 0.f)) return HVA_EINVAL;
  FwdLayout F;
  HVA_TRY(make_layout(s, c, &F));
  if (ws_bytes < F.ws_total + (state ? 0 : F.state_total)) return HVA_EWORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  char* w = reinterpret_cast<char*>(ws);
  char* sb = state ? reinterpret_cast<char*>(state) : w + F.ws_total;
  void* plan = w + F.plan;
  const int BH = F.BH, n = F.n;

  if (step_kind == HVA_DENSE) {   // full attention (warm-up steps / layers, l.324): one group, one key run
    hva_plan_layout L;
    HVA_TRY(hva_plan_describe(BH, n, 1, 1, c->tile_q, &L));
    HVA_TRY(hva_attention_dense_plan(BH, n, c->tile_q, c->tile_k, plan, L, st));
    HVA_TRY(hva_sparse_attention(s, c, Q, K, V, plan, L.total, 1, 1, O, 0, nullptr, 0, stream));
    if (stats_out && cudaMemcpyAsync(stats_out, (char*)plan + L.stats, sizeof(hva_stats) * BH, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
      return HVA_ECUDA;
    return HVA_OK;
  }

  const void* X[2] = {Q, K};
  const int32_t* cell[2] = {c->cell_q, c->cell_k};
  const int32_t* win[2] = {c->win_q, c->win_k};
  const int Nc[2] = {F.Nq, F.Nk};
  const bool hybrid = c->subset_frac > 0.f && state != nullptr && F.m > 0;
  // anchor step without the hybrid subset: Q and K on two streams, K with the (still unused) K' region as its scratch
  const size_t es = s->dtype == HVA_F32 ? 4 : 2;
  const bool two_streams = step_kind == HVA_ANCHOR && !hybrid && (size_t)BH * n * s->D * es >= F.scratch_bytes && side_stream() != nullptr;
  if (two_streams) {
    // caller's stream: cluster Q ................. [wait K clustered] mask, merge, query half of the plan [wait side] attention
    // side stream:     cluster K, key half of the plan (koff, perm_k: they depend on the K clustering alone), K' and V' gathers
    // -- the gathers (HBM-bound) run under mask and merge (ALU / latency-bound).  Scratch on the side stream: the K' region for the
    // clustering, the V' region for the key sort, each before it is written.  Fork / join by events: legal under stream capture.
    SideStream* side = side_stream();
    std::lock_guard<std::mutex> guard(side->busy);
    cudaStream_t ss = side->st;
    const size_t xbytes = (size_t)BH * n * s->D * es;
    if (hva_plan_keys_ws_bytes(BH, n, F.Nk) > xbytes) return HVA_EWORKSPACE;
    if (cudaEventRecord(side->fork, st) != cudaSuccess || cudaStreamWaitEvent(ss, side->fork, 0) != cudaSuccess) return HVA_ECUDA;
    int rc = hva_cluster_ex(s, cell[0], win[0], c->iters, Q, nullptr, (int32_t*)(sb + F.assign[0]), (float*)(sb + F.mu[0]),
                            (int32_t*)(sb + F.sizes[0]), (float*)(sb + F.sums[0]), nullptr, c->flags, nullptr, w + F.scratch, F.scratch_bytes, stream);
    int rs = hva_cluster_ex(s, cell[1], win[1], c->iters, K, nullptr, (int32_t*)(sb + F.assign[1]), (float*)(sb + F.mu[1]),
                            (int32_t*)(sb + F.sizes[1]), (float*)(sb + F.sums[1]), nullptr, c->flags, nullptr, w + F.kp, xbytes, ss);
    if (rs == HVA_OK && cudaEventRecord(side->mid, ss) != cudaSuccess) rs = HVA_ECUDA;
    if (rs == HVA_OK) rs = hva_plan_keys(BH, n, F.Nk, (int32_t*)(sb + F.assign[1]), (int32_t*)(sb + F.sizes[1]), plan, F.PL, w + F.vp, xbytes, ss);
    const char* pbk = reinterpret_cast<const char*>(plan);
    if (rs == HVA_OK) rs = hva_gather_kv(s, K, V, (const int32_t*)(pbk + F.PL.perm_k), w + F.kp, w + F.vp, ss);
    if (rc == HVA_OK && rs == HVA_OK && cudaStreamWaitEvent(st, side->mid, 0) != cudaSuccess) rc = HVA_ECUDA;
    if (rc == HVA_OK && rs == HVA_OK) {
      const float scale2 = c->softmax_scale > 0.f ? c->softmax_scale : 1.0f / sqrtf((float)s->D);
      uint8_t* mask = (uint8_t*)(w + F.mask);
      uint8_t* gmask = (uint8_t*)(w + F.group_mask);
      int32_t* group_of = (int32_t*)(w + F.group_of);
      int32_t* n_groups = (int32_t*)(w + F.n_groups);
      rc = hva_build_mask_ex(BH, F.Nq, F.Nk, s->D, (float*)(sb + F.mu[0]), (float*)(sb + F.mu[1]), (int32_t*)(sb + F.sizes[1]), scale2,
                             c->top_p, c->min_kc, mask, c->flags, w + F.scratch, F.scratch_bytes, stream);
      if (rc == HVA_OK)
        rc = hva_merge_offset(bh0, BH, F.Nq, F.Nk, (int32_t*)(sb + F.sizes[0]), (int32_t*)(sb + F.sizes[1]), mask, c->tile_q, c->tile_k,
                              c->merge_rounds, c->max_q_tiles, c->seed, group_of, n_groups, gmask, c->flags, w + F.scratch, F.scratch_bytes, stream);
      if (rc == HVA_OK)
        rc = hva_plan_queries(BH, n, F.Nq, F.Nk, (int32_t*)(sb + F.assign[0]), (int32_t*)(sb + F.sizes[0]), (int32_t*)(sb + F.sizes[1]), group_of,
                              gmask, c->tile_q, c->tile_k, plan, F.PL, w + F.scratch, F.scratch_bytes, st);
    }
    // join even after an error: the side stream must not stay forked (stream capture)
    if (cudaEventRecord(side->join, ss) != cudaSuccess || cudaStreamWaitEvent(st, side->join, 0) != cudaSuccess) return HVA_ECUDA;
    if (rc != HVA_OK) return rc;
    if (rs != HVA_OK) return rs;
    if (!F.fuse_q) HVA_TRY(hva_permute(s, Q, (const int32_t*)(pbk + F.PL.perm_q), w + F.qp, stream));
    hva_config ca = *c;
    if (F.fuse_q) ca.flags |= HVA_FLAG_Q_UNPERMUTED;
    HVA_TRY(hva_sparse_attention(s, &ca, F.fuse_q ? Q : (const void*)(w + F.qp), w + F.kp, w + F.vp, plan, F.PL.total, F.Nq, F.Nk, O, 1, nullptr, 0,
                                 stream));
    if (stats_out && cudaMemcpyAsync(stats_out, pbk + F.PL.stats, sizeof(hva_stats) * BH, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
      return HVA_ECUDA;
    return HVA_OK;
  }
  for (int t = 0; t < 2 && !two_streams; ++t) {
    int32_t* assign = (int32_t*)(sb + F.assign[t]);
    float* mu = (float*)(sb + F.mu[t]);
    float* sums = (float*)(sb + F.sums[t]);
    int32_t* sizes = (int32_t*)(sb + F.sizes[t]);
    int32_t* subset = (int32_t*)(sb + F.subset[t]);
    if (step_kind == HVA_ANCHOR) {
      float* lowe = hybrid ? (float*)(w + F.lowe) : nullptr;
      HVA_TRY(hva_cluster_ex(s, cell[t], win[t], c->iters, X[t], nullptr, assign, mu, sizes, sums, lowe, c->flags, nullptr,
                             w + F.scratch, F.scratch_bytes, stream));
      if (hybrid) HVA_TRY(hva_select_subset(BH, n, lowe, F.m, subset, w + F.scratch, F.scratch_bytes, stream));
    } else {
      HVA_TRY(hva_cluster_update_ex(s, Nc[t], X[t], subset, F.m, c->hybrid_refresh_all, assign, mu, sums, sizes, c->flags,
                                    w + F.scratch, F.scratch_bytes, stream));
    }
  }
  const float scale = c->softmax_scale > 0.f ? c->softmax_scale : 1.0f / sqrtf((float)s->D);
  uint8_t* mask = (uint8_t*)(w + F.mask);
  uint8_t* gmask = (uint8_t*)(w + F.group_mask);
  int32_t* group_of = (int32_t*)(w + F.group_of);
  int32_t* n_groups = (int32_t*)(w + F.n_groups);
  HVA_TRY(hva_build_mask_ex(BH, F.Nq, F.Nk, s->D, (float*)(sb + F.mu[0]), (float*)(sb + F.mu[1]), (int32_t*)(sb + F.sizes[1]),
                            scale, c->top_p, c->min_kc, mask, c->flags, w + F.scratch, F.scratch_bytes, stream));
  HVA_TRY(hva_merge_offset(bh0, BH, F.Nq, F.Nk, (int32_t*)(sb + F.sizes[0]), (int32_t*)(sb + F.sizes[1]), mask, c->tile_q, c->tile_k,
                    c->merge_rounds, c->max_q_tiles, c->seed, group_of, n_groups, gmask, c->flags, w + F.scratch, F.scratch_bytes, stream));
  HVA_TRY(hva_build_plan(BH, n, F.Nq, F.Nk, (int32_t*)(sb + F.assign[0]), (int32_t*)(sb + F.assign[1]),
                         (int32_t*)(sb + F.sizes[0]), (int32_t*)(sb + F.sizes[1]), group_of, n_groups, gmask, c->tile_q,
                         c->tile_k, plan, F.PL.total, w + F.scratch, F.scratch_bytes, stream));
  const char* pb = reinterpret_cast<const char*>(plan);
  if (!F.fuse_q) HVA_TRY(hva_permute(s, Q, (const int32_t*)(pb + F.PL.perm_q), w + F.qp, stream));
  HVA_TRY(hva_permute(s, K, (const int32_t*)(pb + F.PL.perm_k), w + F.kp, stream));
  HVA_TRY(hva_permute(s, V, (const int32_t*)(pb + F.PL.perm_k), w + F.vp, stream));
  hva_config ca = *c;
  if (F.fuse_q) ca.flags |= HVA_FLAG_Q_UNPERMUTED;
  HVA_TRY(hva_sparse_attention(s, &ca, F.fuse_q ? Q : (const void*)(w + F.qp), w + F.kp, w + F.vp, plan, F.PL.total, F.Nq, F.Nk, O, 1, nullptr, 0,
                               stream));
  if (stats_out && cudaMemcpyAsync(stats_out, pb + F.PL.stats, sizeof(hva_stats) * BH, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
    return HVA_ECUDA;
  return HVA_OK;
}

}  // namespace

extern "C" int hva_forward(const hva_shape* s, const hva_config* c, const void* Q, const void* K, const void* V, void* O,
                           int32_t step_kind, void* state, hva_stats* stats_out, void* ws, size_t ws_bytes, void* stream) {
  return forward_impl(s, c, Q, K, V, O, step_kind, state, stats_out, ws, ws_bytes, stream, 0);
}

namespace {
// Copy streams / events of hva_forward_host: one set per device, created on first use on that device (no device memory
// is allocated).  The table is guarded by a mutex; a call holds its device's set for its whole duration, so concurrent host
// calls on one device are serialised (documented in hva.h).
struct HostPipe {
  cudaStream_t h2d = nullptr, d2h = nullptr, comp[2] = {nullptr, nullptr};   // copy streams; compute streams of the even / odd chunks
  cudaEvent_t in_done[16] = {}, out_ready[16] = {}, start = nullptr;
  bool tried = false, ok = false;
  std::mutex busy;
  void create() {
    tried = true;
    ok = cudaStreamCreateWithFlags(&h2d, cudaStreamNonBlocking) == cudaSuccess &&
         cudaStreamCreateWithFlags(&d2h, cudaStreamNonBlocking) == cudaSuccess &&
         cudaStreamCreateWithFlags(&comp[0], cudaStreamNonBlocking) == cudaSuccess &&
         cudaStreamCreateWithFlags(&comp[1], cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&start, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < 16 && ok; ++i)
      ok = cudaEventCreateWithFlags(&in_done[i], cudaEventDisableTiming) == cudaSuccess &&
           cudaEventCreateWithFlags(&out_ready[i], cudaEventDisableTiming) == cudaSuccess;
  }
};
constexpr int kMaxDevices = 64;
HostPipe* host_pipe() {
  static HostPipe pipes[kMaxDevices];
  static std::mutex table;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
  std::lock_guard<std::mutex> g(table);
  if (!pipes[dev].tried) pipes[dev].create();
  return pipes[dev].ok ? &pipes[dev] : nullptr;
}
}  // namespace

// Heads are independent instances of the whole pipeline, so the host variant runs the call in chunks of heads: the
// host-to-device copy of chunk i+1 and the device-to-host copy of chunk i-1 (two copy streams, both PCIe directions)
// overlap the kernels of chunk i on the caller's stream.  With a hybrid state buffer (per-(b,h) cache) or B > 1 the
// call is not chunked.
extern "C" int hva_forward_host(const hva_shape* s, const hva_config* c, const void* hQ, const void* hK, const void* hV,
                                void* hO, int32_t step_kind, void* state, void* dev_qkvo, void* ws, size_t ws_bytes,
                                void* stream) {
  // everything that can fail on the arguments is checked before anything is enqueued (hva.h: nothing is enqueued on
  // EINVAL / EWORKSPACE): the full-size layout bounds the layout of every chunk
  if (!valid_shape(s) || !valid_config(c) || !hQ || !hK || !hV || !hO || !dev_qkvo || !ws) return HVA_EINVAL;
  if (step_kind != HVA_ANCHOR && step_kind != HVA_INTERMEDIATE && step_kind != HVA_DENSE) return HVA_EINVAL;
  if (step_kind == HVA_INTERMEDIATE && (!state || c->subset_frac <= 0.f)) return HVA_EINVAL;
  {
    FwdLayout F;
    HVA_TRY(make_layout(s, c, &F));
    if (ws_bytes < F.ws_total + (state ? 0 : F.state_total)) return HVA_EWORKSPACE;
  }
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const size_t es = s->dtype == HVA_F32 ? 4 : 2;
  const size_t head_bytes = (size_t)s->T * s->H * s->W * s->D * es;
  const size_t bytes = (size_t)s->B * s->heads * head_bytes;
  char* d = reinterpret_cast<char*>(dev_qkvo);
  HostPipe* pipe = (!state && s->B == 1 && s->heads >= 8) ? host_pipe() : nullptr;
  if (!pipe) {
    int rc = HVA_OK;
    if (cudaMemcpyAsync(d, hQ, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(d + bytes, hK, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(d + 2 * bytes, hV, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
      rc = HVA_ECUDA;
    if (rc == HVA_OK) rc = hva_forward(s, c, d, d + bytes, d + 2 * bytes, d + 3 * bytes, step_kind, state, nullptr, ws, ws_bytes, stream);
    if (rc == HVA_OK && cudaMemcpyAsync(hO, d + 3 * bytes, bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = HVA_ECUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess && rc == HVA_OK) rc = HVA_ECUDA;   // also on error: nothing of ours stays in flight
    return rc;
  }
  std::lock_guard<std::mutex> hold(pipe->busy);
  // Chunk sizes.  The H2D copies run back to back from t = 0; chunk k's kernels can start when its copy has landed and chunk k-1's
  // kernels are done.  With a = copy time and b = r a = kernel time per head, nothing waits iff  c_k <= c_1 + (r - 1) S_{k-1}
  // (S = heads before chunk k): the chunks grow geometrically from a small first one, and the last one is small again because its
  // D2H copy is the one transfer nothing covers.  r is estimated from the problem size (attention ~ n^2 per head, copies ~ n; 0.45
  // of the tile pairs executed, 1.2 PFLOP/s, 55 GB/s); the smallest c_1 whose schedule fits 16 chunks is taken
  // (with the chunks alternating between two compute streams, below, a chunk's fixed costs are hidden, so many chunks are cheap).
  int nchunk = 0;
  int bound[17];
  {
    const double n_tok = (double)s->T * s->H * s->W;
    double r = n_tok * 0.45 * 3.1e-5 * (2.0 / (double)es);
    r = r < 1.05 ? 1.05 : (r > 3.0 ? 3.0 : r);
    for (int c1 = 1; c1 <= s->heads && nchunk == 0; ++c1) {
      int sizes[16], k = 0, S = 0;
      const int last = std::min(c1, s->heads - c1);          // heads >= 8 here
      sizes[k++] = c1; S = c1;
      while (S < s->heads - last && k < 15) {
        int cap = (int)std::floor((double)c1 + (r - 1.0) * (double)S);
        if (cap < 1) cap = 1;
        const int take = std::min(cap, s->heads - last - S);
        sizes[k++] = take; S += take;
      }
      if (S != s->heads - last) continue;                     // does not fit 16 chunks: a larger first chunk
      sizes[k++] = last;
      bound[0] = 0;
      for (int i = 0; i < k; ++i) bound[i + 1] = bound[i] + sizes[i];
      nchunk = k;
    }
    if (nchunk == 0) { nchunk = 1; bound[0] = 0; bound[1] = s->heads; }
  }
  int rc = HVA_OK;
  // Consecutive chunks run on two compute streams with one half of the workspace each, so that the small, latency-bound stages of
  // chunk k+1 (clustering, mask, merge, plan: ~0.5 ms whatever the head count) fill in under the attention kernel of chunk k
  // instead of following it; a stream's order keeps chunk k+2 off the half chunk k still uses.  If a half cannot hold the largest
  // chunk, everything runs on the caller's stream with the whole workspace.
  size_t half = (ws_bytes / 2) & ~(size_t)255, need = 0;
  for (int i = 0; i < nchunk; ++i) {
    hva_shape sc = *s;
    sc.heads = bound[i + 1] - bound[i];
    need = std::max(need, hva_workspace_bytes(&sc, c));
  }
  const bool two = nchunk > 1 && need > 0 && need <= half;
  cudaStream_t cs[2] = {two ? pipe->comp[0] : st, two ? pipe->comp[1] : st};
  // the library's streams start after whatever the caller has queued on `st`
  if (cudaEventRecord(pipe->start, st) != cudaSuccess || cudaStreamWaitEvent(pipe->h2d, pipe->start, 0) != cudaSuccess ||
      cudaStreamWaitEvent(pipe->d2h, pipe->start, 0) != cudaSuccess ||
      (two && (cudaStreamWaitEvent(cs[0], pipe->start, 0) != cudaSuccess || cudaStreamWaitEvent(cs[1], pipe->start, 0) != cudaSuccess)))
    rc = HVA_ECUDA;
  const char* src[3] = {(const char*)hQ, (const char*)hK, (const char*)hV};
  for (int i = 0; i < nchunk && rc == HVA_OK; ++i) {
    const int h0 = bound[i], h1 = bound[i + 1], nh = h1 - h0;
    const size_t off = (size_t)h0 * head_bytes, cb = (size_t)nh * head_bytes;
    cudaStream_t ci = cs[i & 1];
    for (int t = 0; t < 3 && rc == HVA_OK; ++t)
      if (cudaMemcpyAsync(d + t * bytes + off, src[t] + off, cb, cudaMemcpyHostToDevice, pipe->h2d) != cudaSuccess) rc = HVA_ECUDA;
    if (rc == HVA_OK && (cudaEventRecord(pipe->in_done[i], pipe->h2d) != cudaSuccess || cudaStreamWaitEvent(ci, pipe->in_done[i], 0) != cudaSuccess))
      rc = HVA_ECUDA;
    if (rc != HVA_OK) break;
    hva_shape sc = *s;
    sc.heads = nh;
    rc = forward_impl(&sc, c, d + off, d + bytes + off, d + 2 * bytes + off, d + 3 * bytes + off, step_kind, nullptr, nullptr,
                      two ? (char*)ws + (i & 1) * half : (char*)ws, two ? half : ws_bytes, ci, h0);
    if (rc != HVA_OK) break;
    if (cudaEventRecord(pipe->out_ready[i], ci) != cudaSuccess || cudaStreamWaitEvent(pipe->d2h, pipe->out_ready[i], 0) != cudaSuccess ||
        cudaMemcpyAsync((char*)hO + off, d + 3 * bytes + off, cb, cudaMemcpyDeviceToHost, pipe->d2h) != cudaSuccess)
      rc = HVA_ECUDA;
  }
  // drain all three streams, also on error: no copy into or out of the caller's buffers is left in flight
  const bool s0 = cudaStreamSynchronize(pipe->h2d) == cudaSuccess, s1 = cudaStreamSynchronize(st) == cudaSuccess,
             s2 = cudaStreamSynchronize(pipe->d2h) == cudaSuccess, s3 = cudaStreamSynchronize(pipe->comp[0]) == cudaSuccess,
             s4 = cudaStreamSynchronize(pipe->comp[1]) == cudaSuccess;
  if (rc == HVA_OK && !(s0 && s1 && s2 && s3 && s4)) rc = HVA_ECUDA;
  return rc;
}
