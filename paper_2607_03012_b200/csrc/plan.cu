// S7 plan (canonical permutations of PAPER.md Eq. 1 l.37, DESIGN.md R-P1; packed key runs l.109),
// S8 / S10 row gathers (Eq. 1 l.37; Eq. 4 l.56), and the occupancy statistics of Eq. 7-8 / Fig. 5c.
//
// Token sort = stable counting sort by cluster label in three passes over warp tiles of 1024
// consecutive tokens (labels need not be window-local, so hybrid steps work unchanged):
//   A  per-tile label histogram (shared-memory row per warp, __match_any_sync aggregation)
//   B  per-label exclusive scan over tiles, seeded with the cluster's row offset
//   C  per-tile stable scatter: dest = running offset of the label + rank among equal labels
#include "common.cuh"

namespace {

constexpr int kTile = 1024;       // tokens per warp tile
constexpr int kSortWarps = 4;     // warps per CTA in passes A and C

struct PlanPtrs {
  int *perm_q, *inv_perm_q, *perm_k, *koff, *n_groups, *gid, *goff, *kappa, *run_cnt, *work_cnt, *work;
  uint32_t* runs;
  hva_stats* stats;
  int run_stride, work_cap;
};

__host__ PlanPtrs plan_ptrs(void* plan, const hva_plan_layout& L) {
  char* b = reinterpret_cast<char*>(plan);
  PlanPtrs p;
  p.perm_q = (int*)(b + L.perm_q); p.inv_perm_q = (int*)(b + L.inv_perm_q); p.perm_k = (int*)(b + L.perm_k);
  p.koff = (int*)(b + L.koff); p.n_groups = (int*)(b + L.n_groups); p.gid = (int*)(b + L.gid);
  p.goff = (int*)(b + L.goff); p.kappa = (int*)(b + L.kappa); p.run_cnt = (int*)(b + L.run_cnt);
  p.runs = (uint32_t*)(b + L.runs); p.work_cnt = (int*)(b + L.work_cnt); p.work = (int*)(b + L.work);
  p.stats = (hva_stats*)(b + L.stats); p.run_stride = (int)L.run_stride; p.work_cap = (int)L.work_cap;
  return p;
}

// ---- group / cluster bookkeeping: one CTA per (b, head)
__global__ void __launch_bounds__(1024) hva_plan_groups_kernel(int n, int Nq, int Nk, const int* __restrict__ sizes_q,
                                                               const int* __restrict__ sizes_k,
                                                               const int* __restrict__ group_of,
                                                               const uint8_t* __restrict__ group_mask, int tile_q,
                                                               int tile_k, PlanPtrs P, int* __restrict__ qbase) {
  const int bh = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int* sq = sizes_q + (size_t)bh * Nq;
  const int* sk = sizes_k + (size_t)bh * Nk;
  const int* gof = group_of + (size_t)bh * Nq;
  int* koff = P.koff + (size_t)bh * (Nk + 1);
  int* gid = P.gid + (size_t)bh * Nq;
  int* goff = P.goff + (size_t)bh * (Nq + 1);
  int* kappa = P.kappa + (size_t)bh * Nq;
  int* run_cnt = P.run_cnt + (size_t)bh * Nq;
  int* qb = qbase + (size_t)bh * Nq;
  __shared__ int s_ng;
  // the serial parts below are chains of dependent loads: run them on shared-memory copies (global latency made this kernel
  // 0.67 ms at C4)
  extern __shared__ int s_stage[];
  int* s_sq = s_stage;            // [Nq]
  int* s_gof = s_sq + Nq;         // [Nq]
  int* s_sk = s_gof + Nq;         // [Nk]
  int* s_goff = s_sk + Nk;        // [Nq + 1]
  int* s_kap = s_goff + Nq + 1;   // [Nq]
  for (int u = tid; u < Nq; u += blockDim.x) { s_sq[u] = sizes_q[(size_t)bh * Nq + u]; s_gof[u] = group_of[(size_t)bh * Nq + u]; }
  for (int j = tid; j < Nk; j += blockDim.x) s_sk[j] = sizes_k[(size_t)bh * Nk + j];
  __syncthreads();
  sq = s_sq; sk = s_sk; gof = s_gof;
  // Q' row offset of query cluster u: clusters ordered by (gid(u), u)   (R-P1)
  for (int u = tid; u < Nq; u += blockDim.x) {
    int gu = gof[u], off = 0;
    for (int v = 0; v < Nq; ++v) {
      int gv = gof[v];
      if (gv < gu || (gv == gu && v < u)) off += sq[v];
    }
    qb[u] = off;
  }
  if (tid == 0) {  // K' row offsets; active groups in ascending gid
    int a = 0;
    for (int j = 0; j < Nk; ++j) { koff[j] = a; a += sk[j]; }
    koff[Nk] = a;
    int c = 0;
    for (int g = 0; g < Nq; ++g) {
      if (gof[g] != g) continue;
      int s = 0;                      // a leader with an empty group (s^q = 0) is not active
      if (sq[g] > 0) s = 1;
      else for (int v = g + 1; v < Nq && !s; ++v) s = (gof[v] == g && sq[v] > 0);
      if (s) gid[c++] = g;
    }
    s_ng = c; P.n_groups[bh] = c;
  }
  __syncthreads();
  const int ng = s_ng;
  for (int k = tid; k < ng; k += blockDim.x) { const int o = qb[gid[k]]; goff[k] = o; s_goff[k] = o; }   // leader = first cluster of its group
  if (tid == 0) { goff[ng] = n; s_goff[ng] = n; }
  // packed key runs of each group: maximal runs of consecutive selected key clusters (l.109)
  const uint8_t* gm = group_mask + (size_t)bh * Nq * Nk;
  for (int k = warp; k < ng; k += blockDim.x / 32) {
    uint16_t* r16 = reinterpret_cast<uint16_t*>(P.runs + ((size_t)bh * Nq + k) * P.run_stride);
    const uint8_t* grow = gm + (size_t)k * Nk;
    int nstart = 0, nend = 0, kap = 0;
    unsigned carry = 0;                                   // last key of the previous 1024-key block selected?
    for (int jb = 0; jb < Nk; jb += 1024) {
      // pack up to 1024 mask bytes into 32 ballot words (independent loads, one latency), lane l then owns word l
      unsigned mine = 0;
#pragma unroll 8
      for (int w = 0; w < 32; ++w) {
        const int j = jb + 32 * w + lane;
        const int bit = (j < Nk) ? grow[j] : 0;
        const unsigned word = __ballot_sync(0xffffffffu, bit);
        kap += bit ? sk[j] : 0;
        if (w == lane) mine = word;
      }
      const unsigned prev_w = __shfl_up_sync(0xffffffffu, mine, 1), next_w = __shfl_down_sync(0xffffffffu, mine, 1);
      const unsigned prev_bit = lane == 0 ? carry : (prev_w >> 31);
      unsigned next_bit = lane == 31 ? 0u : (next_w & 1u);
      if (lane == 31 && jb + 1024 < Nk) next_bit = grow[jb + 1024] ? 1u : 0u;
      unsigned starts = mine & ~((mine << 1) | prev_bit), ends = mine & ~((mine >> 1) | (next_bit << 31));
      // exclusive prefix of the run counts over the lanes
      int cs = __popc(starts), ce = __popc(ends), ps = cs, pe = ce;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int ys = __shfl_up_sync(0xffffffffu, ps, o), ye = __shfl_up_sync(0xffffffffu, pe, o);
        if (lane >= o) { ps += ys; pe += ye; }
      }
      const int tot_s = __shfl_sync(0xffffffffu, ps, 31), tot_e = __shfl_sync(0xffffffffu, pe, 31);
      int os = nstart + ps - cs, oe = nend + pe - ce;
      while (starts) { const int bpos = __ffs(starts) - 1; starts &= starts - 1; r16[2 * os++] = (uint16_t)(jb + 32 * lane + bpos); }
      while (ends) { const int bpos = __ffs(ends) - 1; ends &= ends - 1; r16[2 * oe++ + 1] = (uint16_t)(jb + 32 * lane + bpos); }
      nstart += tot_s; nend += tot_e;
      carry = __shfl_sync(0xffffffffu, mine, 31) >> 31;
    }
    for (int o = 16; o > 0; o >>= 1) kap += __shfl_xor_sync(0xffffffffu, kap, o);
    if (lane == 0) { run_cnt[k] = nstart; kappa[k] = kap; s_kap[k] = kap; }
  }
  __syncthreads();
  if (tid == 0) {  // work list (group, q-tile) in group order + statistics (Eq. 7-8; Fig. 5c terms)
    int* work = P.work + (size_t)bh * P.work_cap;
    hva_stats s = {};
    int wc = 0;
    for (int k = 0; k < ng; ++k) {
      int rows = s_goff[k + 1] - s_goff[k], kp = s_kap[k];
      int rt = (rows + tile_q - 1) / tile_q, kt = (kp + tile_k - 1) / tile_k;
      for (int t = 0; t < rt; ++t) work[wc++] = k | (t << 16);
      s.q_rows_valid += rows; s.q_rows_padded += (int64_t)rt * tile_q;
      s.k_cols_valid += kp; s.k_cols_padded += (int64_t)kt * tile_k;
      s.tiles_executed += (int64_t)rt * kt; s.pairs_valid += (int64_t)rows * kp;
    }
    s.n_groups = ng; s.q_tiles = wc;
    P.work_cnt[bh] = wc;
    P.stats[bh] = s;
  }
}

// ---- pass A: per-tile histogram
__global__ void __launch_bounds__(kSortWarps * 32) hva_sort_hist_kernel(int n, int Nc, int ntile,
                                                                        const int* __restrict__ assign,
                                                                        int* __restrict__ hist) {
  extern __shared__ int s_h[];  // [kSortWarps][Nc]
  const int bh = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int tile = blockIdx.x * kSortWarps + warp;
  int* h = s_h + warp * Nc;
  for (int c = lane; c < Nc; c += 32) h[c] = 0;
  __syncwarp();
  if (tile < ntile) {
    const int* a = assign + (size_t)bh * n;
    for (int s = 0; s < kTile / 32; ++s) {
      int tok = tile * kTile + s * 32 + lane;
      bool ok = tok < n;
      int lab = ok ? a[tok] : -1 - lane;
      unsigned peers = __match_any_sync(0xffffffffu, lab);
      if (ok && (peers & ((1u << lane) - 1)) == 0) h[lab] += __popc(peers);   // leader lane of each label
      __syncwarp();
    }
    int* out = hist + ((size_t)bh * ntile + tile) * Nc;
    for (int c = lane; c < Nc; c += 32) out[c] = h[c];
  }
}

// ---- pass B: per-label exclusive scan over tiles, seeded with the cluster's row offset
__global__ void hva_sort_scan_kernel(int Nc, int ntile, const int* __restrict__ base, int base_stride,
                                     int* __restrict__ hist) {
  int c = blockIdx.x * blockDim.x + threadIdx.x, bh = blockIdx.y;
  if (c >= Nc) return;
  int run = base[(size_t)bh * base_stride + c];
  int* h = hist + (size_t)bh * ntile * Nc + c;
  for (int t = 0; t < ntile; ++t) { int v = h[(size_t)t * Nc]; h[(size_t)t * Nc] = run; run += v; }
}

// ---- pass C: stable scatter
__global__ void __launch_bounds__(kSortWarps * 32) hva_sort_scatter_kernel(int n, int Nc, int ntile,
                                                                           const int* __restrict__ assign,
                                                                           const int* __restrict__ hist,
                                                                           int* __restrict__ perm,
                                                                           int* __restrict__ inv) {
  extern __shared__ int s_h[];
  const int bh = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int tile = blockIdx.x * kSortWarps + warp;
  if (tile >= ntile) return;
  int* h = s_h + warp * Nc;
  const int* in = hist + ((size_t)bh * ntile + tile) * Nc;
  for (int c = lane; c < Nc; c += 32) h[c] = in[c];
  __syncwarp();
  const int* a = assign + (size_t)bh * n;
  for (int s = 0; s < kTile / 32; ++s) {
    int tok = tile * kTile + s * 32 + lane;
    bool ok = tok < n;
    int lab = ok ? a[tok] : -1 - lane;
    unsigned peers = __match_any_sync(0xffffffffu, lab);
    int rank = __popc(peers & ((1u << lane) - 1));
    int dest = ok ? h[lab] + rank : 0;
    __syncwarp();
    if (ok && rank == 0) h[lab] += __popc(peers);
    __syncwarp();
    if (ok) {
      perm[(size_t)bh * n + dest] = tok;
      if (inv) inv[(size_t)bh * n + tok] = dest;
    }
  }
}

// ---- S8 / S10: row gathers, 16 bytes per lane
__global__ void hva_permute_kernel(size_t rows_total, int n, int row_chunks, const uint4* __restrict__ X,
                                   const int* __restrict__ perm, uint4* __restrict__ Y, int inverse) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  size_t row = i / row_chunks;
  int q = (int)(i % row_chunks);
  if (row >= rows_total) return;
  size_t bh = row / n;
  size_t other = bh * n + (size_t)perm[row];
  if (!inverse) Y[row * row_chunks + q] = __ldg(X + other * row_chunks + q);   // Xp[i] = X[perm[i]]
  else Y[other * row_chunks + q] = __ldg(X + row * row_chunks + q);            // X[perm[i]] = Xp[i]
}

__global__ void hva_dense_plan_kernel(int n, int tile_q, int tile_k, PlanPtrs P) {
  const int bh = blockIdx.x, tid = threadIdx.x;
  for (int i = tid; i < n; i += blockDim.x) {
    P.perm_q[(size_t)bh * n + i] = i; P.inv_perm_q[(size_t)bh * n + i] = i; P.perm_k[(size_t)bh * n + i] = i;
  }
  int rt = (n + tile_q - 1) / tile_q, kt = (n + tile_k - 1) / tile_k;
  int* work = P.work + (size_t)bh * P.work_cap;
  for (int t = tid; t < rt; t += blockDim.x) work[t] = 0 | (t << 16);
  if (tid == 0) {
    P.koff[(size_t)bh * 2] = 0; P.koff[(size_t)bh * 2 + 1] = n;
    P.n_groups[bh] = 1; P.gid[bh] = 0; P.goff[(size_t)bh * 2] = 0; P.goff[(size_t)bh * 2 + 1] = n;
    P.kappa[bh] = n; P.run_cnt[bh] = 1; P.runs[(size_t)bh * P.run_stride] = 0u;
    P.work_cnt[bh] = rt;
    hva_stats s = {};
    s.n_groups = 1; s.q_tiles = rt; s.q_rows_valid = n; s.q_rows_padded = (int64_t)rt * tile_q;
    s.k_cols_valid = n; s.k_cols_padded = (int64_t)kt * tile_k; s.tiles_executed = (int64_t)rt * kt;
    s.pairs_valid = (int64_t)n * n;
    P.stats[bh] = s;
  }
}

}  // namespace

extern "C" int hva_plan_describe(int32_t BH, int32_t n, int32_t Nq, int32_t Nk, int32_t tile_q, hva_plan_layout* L) {
  if (!L || BH < 1 || n < 1 || Nq < 1 || Nk < 1 || tile_q < 1) return HVA_EINVAL;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o += hva_align(bytes); return r; };
  L->run_stride = (size_t)(Nk + 2) / 2;
  L->work_cap = (size_t)(n + tile_q - 1) / tile_q + Nq;
  L->perm_q = take((size_t)BH * n * 4); L->inv_perm_q = take((size_t)BH * n * 4); L->perm_k = take((size_t)BH * n * 4);
  L->koff = take((size_t)BH * (Nk + 1) * 4); L->n_groups = take((size_t)BH * 4); L->gid = take((size_t)BH * Nq * 4);
  L->goff = take((size_t)BH * (Nq + 1) * 4); L->kappa = take((size_t)BH * Nq * 4); L->run_cnt = take((size_t)BH * Nq * 4);
  L->runs = take((size_t)BH * Nq * L->run_stride * 4); L->work_cnt = take((size_t)BH * 4);
  L->work = take((size_t)BH * L->work_cap * 4); L->stats = take((size_t)BH * sizeof(hva_stats));
  L->total = o;
  return HVA_OK;
}

size_t hva_plan_ws_bytes(int BH, int n, int Nq, int Nk) {
  int ntile = (n + kTile - 1) / kTile, Nc = Nq > Nk ? Nq : Nk;
  return hva_align((size_t)BH * ntile * Nc * 4) + hva_align((size_t)BH * Nq * 4);
}

extern "C" int hva_build_plan(int32_t BH, int32_t n, int32_t Nq, int32_t Nk, const int32_t* assign_q,
                              const int32_t* assign_k, const int32_t* sizes_q, const int32_t* sizes_k,
                              const int32_t* group_of_cluster, const int32_t* n_groups, const uint8_t* group_mask,
                              int32_t tile_q, int32_t tile_k, void* plan, size_t plan_bytes, void* ws, size_t ws_bytes,
                              void* stream) {
  (void)n_groups;
  if (!assign_q || !assign_k || !sizes_q || !sizes_k || !group_of_cluster || !group_mask || !plan || !ws) return HVA_EINVAL;
  if (BH < 1 || n < 1 || Nq < 1 || Nk < 1 || tile_q < 1 || tile_k < 1) return HVA_EINVAL;
  if (Nq > 2048 || Nk > 2048 || (n + tile_q - 1) / tile_q > 32767) return HVA_EUNSUPPORTED;
  hva_plan_layout L;
  HVA_TRY(hva_plan_describe(BH, n, Nq, Nk, tile_q, &L));
  if (plan_bytes < L.total) return HVA_EWORKSPACE;
  if (ws_bytes < hva_plan_ws_bytes(BH, n, Nq, Nk)) return HVA_EWORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  PlanPtrs P = plan_ptrs(plan, L);
  const int ntile = (n + kTile - 1) / kTile, Ncmax = Nq > Nk ? Nq : Nk;
  int* hist = reinterpret_cast<int*>(ws);
  int* qbase = reinterpret_cast<int*>(reinterpret_cast<char*>(ws) + hva_align((size_t)BH * ntile * Ncmax * 4));
  const size_t gsmem = sizeof(int) * (4 * (size_t)Nq + Nk + 1);
  if (gsmem > 48 * 1024 && cudaFuncSetAttribute(hva_plan_groups_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gsmem) != cudaSuccess)
    return HVA_EUNSUPPORTED;
  hva_plan_groups_kernel<<<BH, 1024, gsmem, st>>>(n, Nq, Nk, sizes_q, sizes_k, group_of_cluster, group_mask, tile_q, tile_k,
                                              P, qbase);
  HVA_CHECK_LAUNCH();
  dim3 gsort((ntile + kSortWarps - 1) / kSortWarps, BH);
  for (int pass = 0; pass < 2; ++pass) {  // 0: keys (perm_k), 1: queries (perm_q, inv_perm_q)
    const int Nc = pass ? Nq : Nk;
    const int* assign = pass ? assign_q : assign_k;
    size_t smem = (size_t)kSortWarps * Nc * sizeof(int);
    hva_sort_hist_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, Nc, ntile, assign, hist);
    HVA_CHECK_LAUNCH();
    hva_sort_scan_kernel<<<dim3((Nc + 127) / 128, BH), 128, 0, st>>>(Nc, ntile, pass ? qbase : P.koff, pass ? Nq : Nk + 1, hist);
    HVA_CHECK_LAUNCH();
    hva_sort_scatter_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, Nc, ntile, assign, hist, pass ? P.perm_q : P.perm_k,
                                                                 pass ? P.inv_perm_q : nullptr);
    HVA_CHECK_LAUNCH();
  }
  return HVA_OK;
}

static int permute_common(const hva_shape* s, const void* X, const int32_t* perm, void* Y, void* stream, int inverse) {
  if (!s || !X || !perm || !Y) return HVA_EINVAL;
  if (s->D != 64 && s->D != 128) return HVA_EINVAL;
  if (s->dtype != HVA_F32 && s->dtype != HVA_BF16) return HVA_EUNSUPPORTED;
  int n = s->T * s->H * s->W;
  size_t rows = (size_t)s->B * s->heads * n;
  int chunks = s->D * (s->dtype == HVA_F32 ? 4 : 2) / 16;
  size_t total = rows * chunks;
  hva_permute_kernel<<<(unsigned)((total + 255) / 256), 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(
      rows, n, chunks, reinterpret_cast<const uint4*>(X), perm, reinterpret_cast<uint4*>(Y), inverse);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

extern "C" int hva_permute(const hva_shape* s, const void* X, const int32_t* perm, void* Xp, void* stream) {
  return permute_common(s, X, perm, Xp, stream, 0);
}
extern "C" int hva_unpermute(const hva_shape* s, const void* Xp, const int32_t* perm, void* X, void* stream) {
  return permute_common(s, Xp, perm, X, stream, 1);
}

int hva_attention_dense_plan(int BH, int n, int tile_q, int tile_k, void* plan, const hva_plan_layout& L, cudaStream_t st) {
  PlanPtrs P = plan_ptrs(plan, L);
  hva_dense_plan_kernel<<<BH, 256, 0, st>>>(n, tile_q, tile_k, P);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
