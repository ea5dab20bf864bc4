// S7 plan (canonical permutations of PAPER.md Eq. 1 l.37, DESIGN.md R-P1; packed key runs l.109),
// S8 / S10 row gathers (Eq. 1 l.37; Eq. 4 l.56), and the occupancy statistics of Eq. 7-8 / Fig. 5c.
//
// Token sort = stable counting sort by cluster label in three passes over warp tiles of 1024
// consecutive tokens (labels need not be window-local, so hybrid steps work unchanged):
//   A  per-tile label histogram (shared-memory row per warp, __match_any_sync aggregation)
//   B  per-label exclusive scan over tiles, seeded with the cluster's row offset
//   C  per-tile stable scatter: dest = running offset of the label + rank among equal labels
#include "common.cuh"
#include <mutex>

namespace {

constexpr int kTile = 1024;       // tokens per warp tile
constexpr int kSortWarps = 4;     // warps per CTA in passes A and C
constexpr int kGroupSplit = 6;    // CTAs per (b, head) sharing the key-run extraction (24 heads x 6 = 144 CTAs at C4)

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

// block-wide exclusive scan of one int per thread (1024 threads); *total receives the block sum
__device__ __forceinline__ int block_excl_scan(int v, int* s_warp, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
  if (lane == 31) s_warp[warp] = x;
  __syncthreads();
  if (warp == 0) {
    int w = s_warp[lane], t = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, t, o); if (lane >= o) t += y; }
    s_warp[lane] = t - w;
    if (lane == 31) *total = t;
  }
  __syncthreads();
  const int r = s_warp[warp] + x - v;
  __syncthreads();          // s_warp may be reused by the next call
  return r;
}

// ---- group / cluster bookkeeping: one CTA per (b, head), 1024 threads; Nq, Nk <= 2048 (two items per thread).  Every list is
// built by block-wide scans (round 1 ran the prefix sums, the group list and the work list on thread 0: 0.59 ms at C4).
__global__ void __launch_bounds__(1024) hva_plan_groups_kernel(int n, int Nq, int Nk, const int* __restrict__ sizes_q,
                                                               const int* __restrict__ sizes_k,
                                                               const int* __restrict__ group_of,
                                                               const uint8_t* __restrict__ group_mask, int tile_q,
                                                               int tile_k, PlanPtrs P, int* __restrict__ qbase, int write_koff) {
  // blockIdx.y: the key-run extraction (the long part: one pass over the group's mask row per group) is split over the
  // gridDim.y CTAs of a head; the scans are cheap and every CTA does them, CTA 0 of the head writes their results
  const int bh = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool lead = blockIdx.y == 0;
  const bool lead_k = lead && write_koff;     // hva_plan_keys() has written koff already (and K' may be being gathered with it)
  int* koff = P.koff + (size_t)bh * (Nk + 1);
  int* gid = P.gid + (size_t)bh * Nq;
  int* goff = P.goff + (size_t)bh * (Nq + 1);
  int* kappa = P.kappa + (size_t)bh * Nq;
  int* run_cnt = P.run_cnt + (size_t)bh * Nq;
  int* qb = qbase + (size_t)bh * Nq;
  __shared__ int s_warp[32];
  __shared__ int s_tot;
  extern __shared__ int s_stage[];
  int* s_sq = s_stage;            // [Nq] s^q
  int* s_gof = s_sq + Nq;         // [Nq] gid of each query cluster
  int* s_sk = s_gof + Nq;         // [Nk] s^k
  int* s_gsz = s_sk + Nk;         // [Nq] rows of the group led by g (0 if g leads nothing)
  int* s_rank = s_gsz + Nq;       // [Nq] position of group g among the active groups (ascending gid)
  int* s_goff = s_rank + Nq;      // [Nq + 1] Q' row offset of active group k
  for (int u = tid; u < Nq; u += 1024) { s_sq[u] = sizes_q[(size_t)bh * Nq + u]; s_gof[u] = group_of[(size_t)bh * Nq + u]; s_gsz[u] = 0; }
  for (int j = tid; j < Nk; j += 1024) s_sk[j] = sizes_k[(size_t)bh * Nk + j];
  __syncthreads();
  // rows of every group (integer atomics: order-free)
  for (int u = tid; u < Nq; u += 1024) if (s_sq[u] > 0) atomicAdd(&s_gsz[s_gof[u]], s_sq[u]);
  // K' row offsets: exclusive scan of s^k, two consecutive clusters per thread
  {
    const int j0 = 2 * tid, a = j0 < Nk ? s_sk[j0] : 0, b = j0 + 1 < Nk ? s_sk[j0 + 1] : 0;
    const int e = block_excl_scan(a + b, s_warp, &s_tot);
    if (lead_k && j0 < Nk) koff[j0] = e;
    if (lead_k && j0 + 1 < Nk) koff[j0 + 1] = e + a;
    if (lead_k && tid == 0) koff[Nk] = s_tot;
  }
  // active groups in ascending gid (a leader whose group has no rows is not active) and their Q' row offsets
  int ng;
  {
    const int g0 = 2 * tid;
    const int f0 = g0 < Nq && s_gof[g0] == g0 && s_gsz[g0] > 0, f1 = g0 + 1 < Nq && s_gof[g0 + 1] == g0 + 1 && s_gsz[g0 + 1] > 0;
    const int e = block_excl_scan(f0 + f1, s_warp, &s_tot);
    ng = s_tot;
    if (f0) { if (lead) gid[e] = g0; s_rank[g0] = e; }
    if (f1) { if (lead) gid[e + f0] = g0 + 1; s_rank[g0 + 1] = e + f0; }
    const int z0 = f0 ? s_gsz[g0] : 0, z1 = f1 ? s_gsz[g0 + 1] : 0;
    const int o = block_excl_scan(z0 + z1, s_warp, &s_tot);
    if (f0) { if (lead) goff[e] = o; s_goff[e] = o; }
    if (f1) { if (lead) goff[e + f0] = o + z0; s_goff[e + f0] = o + z0; }
    if (tid == 0) { s_goff[ng] = n; if (lead) { goff[ng] = n; P.n_groups[bh] = ng; } }
  }
  __syncthreads();
  // Q' row offset of query cluster u: clusters ordered by (gid(u), u)   (R-P1) = offset of its group + rows of the group's
  // members below u
  for (int u = tid; lead && u < Nq; u += 1024) {
    const int gu = s_gof[u];
    int off = 0;
    for (int v = gu; v < u; ++v) off += (s_gof[v] == gu) ? s_sq[v] : 0;      // members of a group are >= its gid
    qb[u] = (s_sq[u] > 0 ? s_goff[s_rank[gu]] : 0) + off;
  }
  // packed key runs of each group: maximal runs of consecutive selected key clusters (l.109)
  const uint8_t* gm = group_mask + (size_t)bh * Nq * Nk;
  for (int k = warp + 32 * blockIdx.y; k < ng; k += 32 * gridDim.y) {
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
        kap += bit ? s_sk[j] : 0;
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
    if (lane == 0) { run_cnt[k] = nstart; kappa[k] = kap; }
  }
}

// ---- work list (group, q-tile) in group order + statistics (Eq. 7-8; Fig. 5c terms): one CTA per (b, head), two groups per thread
__global__ void __launch_bounds__(1024) hva_plan_work_kernel(int Nq, int tile_q, int tile_k, PlanPtrs P) {
  const int bh = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
  __shared__ int s_warp[32];
  __shared__ int s_tot;
  const int ng = P.n_groups[bh];
  const int* s_goff = P.goff + (size_t)bh * (Nq + 1);
  const int* s_kap = P.kappa + (size_t)bh * Nq;
  {
    int* work = P.work + (size_t)bh * P.work_cap;
    const int k0 = 2 * tid;
    int rt[2] = {0, 0};
    long long st[6] = {0, 0, 0, 0, 0, 0};    // q_rows_valid, q_rows_padded, k_cols_valid, k_cols_padded, tiles_executed, pairs_valid
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int k = k0 + e;
      if (k < ng) {
        const int rows = s_goff[k + 1] - s_goff[k], kp = s_kap[k];
        rt[e] = (rows + tile_q - 1) / tile_q;
        const int kt = (kp + tile_k - 1) / tile_k;
        st[0] += rows; st[1] += (long long)rt[e] * tile_q; st[2] += kp; st[3] += (long long)kt * tile_k;
        st[4] += (long long)rt[e] * kt; st[5] += (long long)rows * kp;
      }
    }
    const int wo = block_excl_scan(rt[0] + rt[1], s_warp, &s_tot);
    const int wc = s_tot;
    for (int t = 0; t < rt[0]; ++t) work[wo + t] = k0 | (t << 16);
    for (int t = 0; t < rt[1]; ++t) work[wo + rt[0] + t] = (k0 + 1) | (t << 16);
    // statistics: warp shuffles, then one 64-bit shared atomic per warp and field (integers: order-free)
    __shared__ unsigned long long s_st[6];
    if (tid < 6) s_st[tid] = 0ull;
    __syncthreads();
#pragma unroll
    for (int f = 0; f < 6; ++f) {
      long long v = st[f];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      if (lane == 0 && v) atomicAdd(&s_st[f], (unsigned long long)v);
    }
    __syncthreads();
    if (tid == 0) {
      hva_stats s = {};
      s.n_groups = ng; s.q_tiles = wc;
      s.q_rows_valid = (int64_t)s_st[0]; s.q_rows_padded = (int64_t)s_st[1]; s.k_cols_valid = (int64_t)s_st[2];
      s.k_cols_padded = (int64_t)s_st[3]; s.tiles_executed = (int64_t)s_st[4]; s.pairs_valid = (int64_t)s_st[5];
      P.work_cnt[bh] = wc;
      P.stats[bh] = s;
    }
  }
}

// ---- pass A: per-tile histogram
// (blockIdx.z selects the tensor: 0 = keys, 1 = queries -- both sorts run in the same three launches)
struct SortPass { int Nc; const int* assign; int* hist; const int* base; int base_stride; int* perm; int* inv; };
struct SortArgs { SortPass p[2]; };

__global__ void __launch_bounds__(kSortWarps * 32) hva_sort_hist_kernel(int n, int ntile, SortArgs A) {
  extern __shared__ int s_h[];  // [kSortWarps][Nc]
  const int Nc = A.p[blockIdx.z].Nc;
  const int* __restrict__ assign = A.p[blockIdx.z].assign;
  int* __restrict__ hist = A.p[blockIdx.z].hist;
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
__global__ void __launch_bounds__(128) hva_sort_scan_kernel(int ntile, SortArgs A) {
  // one warp per label: the lanes take 32 tiles at a time (independent loads), warp scan, running offset carried along
  const int Nc = A.p[blockIdx.z].Nc, base_stride = A.p[blockIdx.z].base_stride;
  const int* __restrict__ base = A.p[blockIdx.z].base;
  int* __restrict__ hist = A.p[blockIdx.z].hist;
  const int lane = threadIdx.x & 31, c = blockIdx.x * 4 + (threadIdx.x >> 5), bh = blockIdx.y;
  if (c >= Nc) return;
  int run = base[(size_t)bh * base_stride + c];
  int* h = hist + (size_t)bh * ntile * Nc + c;
  for (int t0 = 0; t0 < ntile; t0 += 32) {
    const int t = t0 + lane;
    const int v = t < ntile ? h[(size_t)t * Nc] : 0;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (t < ntile) h[(size_t)t * Nc] = run + x - v;
    run += __shfl_sync(0xffffffffu, x, 31);
  }
}

// ---- pass C: stable scatter
__global__ void __launch_bounds__(kSortWarps * 32) hva_sort_scatter_kernel(int n, int ntile, SortArgs A) {
  const int Nc = A.p[blockIdx.z].Nc;
  const int* __restrict__ assign = A.p[blockIdx.z].assign;
  const int* __restrict__ hist = A.p[blockIdx.z].hist;
  int* __restrict__ perm = A.p[blockIdx.z].perm;
  int* __restrict__ inv = A.p[blockIdx.z].inv;
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

// ---- R-H3' (hybrid_refresh_all): every centroid = mean of the CURRENT features of its members.  Tokens are counting-sorted by
// label with the kernels above; the per-label counts (= sizes) and their prefix come from the tile histograms.
// one CTA per (b, head): count[c] = sum over tiles of hist[tile][c] (two labels per thread), block scan -> base[c]
__global__ void __launch_bounds__(1024) hva_label_offsets_kernel(int Nc, int ntile, const int* __restrict__ hist, int* __restrict__ base,
                                                                 int* __restrict__ sizes) {
  const int bh = blockIdx.x, tid = threadIdx.x;
  __shared__ int s_warp[32];
  __shared__ int s_tot;
  const int* h = hist + (size_t)bh * ntile * Nc;
  int cnt[2] = {0, 0};
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    const int c = 2 * tid + e;
    if (c < Nc) for (int t = 0; t < ntile; ++t) cnt[e] += h[(size_t)t * Nc + c];
  }
  const int o = block_excl_scan(cnt[0] + cnt[1], s_warp, &s_tot);
  if (2 * tid < Nc) { base[(size_t)bh * (Nc + 1) + 2 * tid] = o; sizes[(size_t)bh * Nc + 2 * tid] = cnt[0]; }
  if (2 * tid + 1 < Nc) { base[(size_t)bh * (Nc + 1) + 2 * tid + 1] = o + cnt[0]; sizes[(size_t)bh * Nc + 2 * tid + 1] = cnt[1]; }
  if (tid == 0) base[(size_t)bh * (Nc + 1) + Nc] = s_tot;
}

// one CTA per centroid, thread = feature dim: the members' rows are added in ascending token order (the sort is stable), four row
// loads in flight; empty clusters keep mu (Alg. 2 line 23)
template <typename T, int D>
__global__ void __launch_bounds__(D) hva_segment_mean_kernel(int n, int Nc, const T* __restrict__ X, const int* __restrict__ perm,
                                                             const int* __restrict__ base, float* __restrict__ mu,
                                                             float* __restrict__ sums) {
  const int u = blockIdx.x, bh = blockIdx.y, c = threadIdx.x;
  const int b0 = base[(size_t)bh * (Nc + 1) + u], b1 = base[(size_t)bh * (Nc + 1) + u + 1];
  const int* pm = perm + (size_t)bh * n;
  const T* Xb = X + (size_t)bh * n * D;
  float z = 0.f;
  int i = b0;
  for (; i + 4 <= b1; i += 4) {
    const float x0 = HvaElem<T>::ld(Xb + (size_t)pm[i] * D + c), x1 = HvaElem<T>::ld(Xb + (size_t)pm[i + 1] * D + c);
    const float x2 = HvaElem<T>::ld(Xb + (size_t)pm[i + 2] * D + c), x3 = HvaElem<T>::ld(Xb + (size_t)pm[i + 3] * D + c);
    z += x0; z += x1; z += x2; z += x3;
  }
  for (; i < b1; ++i) z += HvaElem<T>::ld(Xb + (size_t)pm[i] * D + c);
  const size_t o = ((size_t)bh * Nc + u) * D + c;
  sums[o] = z;
  if (b1 > b0) mu[o] = __fdiv_rn(z, (float)(b1 - b0));
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
  return 2 * hva_align((size_t)BH * ntile * Nc * 4) + hva_align((size_t)BH * Nq * 4);
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
  int* hist_k = reinterpret_cast<int*>(ws);
  int* hist_q = reinterpret_cast<int*>(reinterpret_cast<char*>(ws) + hva_align((size_t)BH * ntile * Ncmax * 4));
  int* qbase = reinterpret_cast<int*>(reinterpret_cast<char*>(ws) + 2 * hva_align((size_t)BH * ntile * Ncmax * 4));
  const size_t gsmem = sizeof(int) * (5 * (size_t)Nq + Nk + 1);
  if (gsmem > 48 * 1024 && cudaFuncSetAttribute(hva_plan_groups_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gsmem) != cudaSuccess)
    return HVA_EUNSUPPORTED;
  hva_plan_groups_kernel<<<dim3(BH, kGroupSplit), 1024, gsmem, st>>>(n, Nq, Nk, sizes_q, sizes_k, group_of_cluster, group_mask, tile_q,
                                                                 tile_k, P, qbase, 1);
  HVA_CHECK_LAUNCH();
  hva_plan_work_kernel<<<BH, 1024, 0, st>>>(Nq, tile_q, tile_k, P);
  HVA_CHECK_LAUNCH();
  // keys (perm_k) and queries (perm_q, inv_perm_q) in the same three launches
  SortArgs A;
  A.p[0] = SortPass{Nk, assign_k, hist_k, P.koff, Nk + 1, P.perm_k, nullptr};
  A.p[1] = SortPass{Nq, assign_q, hist_q, qbase, Nq, P.perm_q, P.inv_perm_q};
  dim3 gsort((ntile + kSortWarps - 1) / kSortWarps, BH, 2);
  const size_t smem = (size_t)kSortWarps * Ncmax * sizeof(int);
  hva_sort_hist_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, ntile, A);
  HVA_CHECK_LAUNCH();
  hva_sort_scan_kernel<<<dim3((Ncmax + 3) / 4, BH, 2), 128, 0, st>>>(ntile, A);
  HVA_CHECK_LAUNCH();
  hva_sort_scatter_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, ntile, A);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

// ---- hva_build_plan in two halves for hva_forward: the key half (koff, perm_k) depends on the K clustering alone, so it and the
// K', V' gathers run on the side stream while mask, merge and the query half run on the caller's.  Same kernels, same results.
__global__ void __launch_bounds__(1024) hva_koff_kernel(int Nk, const int* __restrict__ sizes_k, int* __restrict__ koff_all) {
  const int bh = blockIdx.x, tid = threadIdx.x;
  __shared__ int s_warp[32];
  __shared__ int s_tot;
  int* koff = koff_all + (size_t)bh * (Nk + 1);
  const int j0 = 2 * tid, a = j0 < Nk ? sizes_k[(size_t)bh * Nk + j0] : 0, b = j0 + 1 < Nk ? sizes_k[(size_t)bh * Nk + j0 + 1] : 0;
  const int e = block_excl_scan(a + b, s_warp, &s_tot);
  if (j0 < Nk) koff[j0] = e;
  if (j0 + 1 < Nk) koff[j0 + 1] = e + a;
  if (tid == 0) koff[Nk] = s_tot;
}

size_t hva_plan_keys_ws_bytes(int BH, int n, int Nk) {
  const int ntile = (n + kTile - 1) / kTile;
  return hva_align((size_t)BH * ntile * Nk * 4);
}

int hva_plan_keys(int BH, int n, int Nk, const int* assign_k, const int* sizes_k, void* plan, const hva_plan_layout& L, void* ws,
                  size_t ws_bytes, cudaStream_t st) {
  if (Nk > 2048) return HVA_EUNSUPPORTED;
  if (ws_bytes < hva_plan_keys_ws_bytes(BH, n, Nk)) return HVA_EWORKSPACE;
  PlanPtrs P = plan_ptrs(plan, L);
  const int ntile = (n + kTile - 1) / kTile;
  hva_koff_kernel<<<BH, 1024, 0, st>>>(Nk, sizes_k, P.koff);
  HVA_CHECK_LAUNCH();
  SortArgs A;
  A.p[0] = SortPass{Nk, assign_k, reinterpret_cast<int*>(ws), P.koff, Nk + 1, P.perm_k, nullptr};
  A.p[1] = A.p[0];
  const dim3 gsort((ntile + kSortWarps - 1) / kSortWarps, BH, 1);
  const size_t smem = (size_t)kSortWarps * Nk * sizeof(int);
  hva_sort_hist_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, ntile, A);
  HVA_CHECK_LAUNCH();
  hva_sort_scan_kernel<<<dim3((Nk + 3) / 4, BH, 1), 128, 0, st>>>(ntile, A);
  HVA_CHECK_LAUNCH();
  hva_sort_scatter_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, ntile, A);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

// the query half: groups, key runs, work list, perm_q / inv_perm_q; koff is left alone.  ws: hva_plan_ws_bytes()
int hva_plan_queries(int BH, int n, int Nq, int Nk, const int* assign_q, const int* sizes_q, const int* sizes_k, const int* group_of_cluster,
                     const uint8_t* group_mask, int tile_q, int tile_k, void* plan, const hva_plan_layout& L, void* ws, size_t ws_bytes,
                     cudaStream_t st) {
  if (Nq > 2048 || Nk > 2048 || (n + tile_q - 1) / tile_q > 32767) return HVA_EUNSUPPORTED;
  if (ws_bytes < hva_plan_ws_bytes(BH, n, Nq, Nk)) return HVA_EWORKSPACE;
  PlanPtrs P = plan_ptrs(plan, L);
  const int ntile = (n + kTile - 1) / kTile;
  int* hist_q = reinterpret_cast<int*>(ws);
  int* qbase = reinterpret_cast<int*>(reinterpret_cast<char*>(ws) + hva_align((size_t)BH * ntile * Nq * 4));
  const size_t gsmem = sizeof(int) * (5 * (size_t)Nq + Nk + 1);
  if (gsmem > 48 * 1024 && cudaFuncSetAttribute(hva_plan_groups_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gsmem) != cudaSuccess)
    return HVA_EUNSUPPORTED;
  hva_plan_groups_kernel<<<dim3(BH, kGroupSplit), 1024, gsmem, st>>>(n, Nq, Nk, sizes_q, sizes_k, group_of_cluster, group_mask, tile_q,
                                                                 tile_k, P, qbase, 0);
  HVA_CHECK_LAUNCH();
  hva_plan_work_kernel<<<BH, 1024, 0, st>>>(Nq, tile_q, tile_k, P);
  HVA_CHECK_LAUNCH();
  SortArgs A;
  A.p[0] = SortPass{Nq, assign_q, hist_q, qbase, Nq, P.perm_q, P.inv_perm_q};
  A.p[1] = A.p[0];
  const dim3 gsort((ntile + kSortWarps - 1) / kSortWarps, BH, 1);
  const size_t smem = (size_t)kSortWarps * Nq * sizeof(int);
  hva_sort_hist_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, ntile, A);
  HVA_CHECK_LAUNCH();
  hva_sort_scan_kernel<<<dim3((Nq + 3) / 4, BH, 1), 128, 0, st>>>(ntile, A);
  HVA_CHECK_LAUNCH();
  hva_sort_scatter_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, ntile, A);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

size_t hva_refresh_ws_bytes(int BH, int n, int Nc) {
  const int ntile = (n + kTile - 1) / kTile;
  return hva_align((size_t)BH * ntile * Nc * 4) + hva_align((size_t)BH * (Nc + 1) * 4) + hva_align((size_t)BH * n * 4);
}

// mu, sums, sizes of every cluster from the current X and labels (R-H3'); deterministic (token order)
int hva_refresh_centroids(int BH, int n, int Nc, int D, int dtype, const void* X, const int* assign, float* mu, float* sums, int* sizes,
                          void* ws, size_t ws_bytes, cudaStream_t st) {
  if (Nc > 2048) return HVA_EUNSUPPORTED;
  if (ws_bytes < hva_refresh_ws_bytes(BH, n, Nc)) return HVA_EWORKSPACE;
  const int ntile = (n + kTile - 1) / kTile;
  char* w = reinterpret_cast<char*>(ws);
  int* hist = reinterpret_cast<int*>(w); w += hva_align((size_t)BH * ntile * Nc * 4);
  int* base = reinterpret_cast<int*>(w); w += hva_align((size_t)BH * (Nc + 1) * 4);
  int* perm = reinterpret_cast<int*>(w);
  SortArgs A;
  A.p[0] = SortPass{Nc, assign, hist, base, Nc + 1, perm, nullptr};
  A.p[1] = A.p[0];
  const dim3 gsort((ntile + kSortWarps - 1) / kSortWarps, BH, 1);
  const size_t smem = (size_t)kSortWarps * Nc * sizeof(int);
  hva_sort_hist_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, ntile, A);
  HVA_CHECK_LAUNCH();
  hva_label_offsets_kernel<<<BH, 1024, 0, st>>>(Nc, ntile, hist, base, sizes);
  HVA_CHECK_LAUNCH();
  hva_sort_scan_kernel<<<dim3((Nc + 3) / 4, BH, 1), 128, 0, st>>>(ntile, A);
  HVA_CHECK_LAUNCH();
  hva_sort_scatter_kernel<<<gsort, kSortWarps * 32, smem, st>>>(n, ntile, A);
  HVA_CHECK_LAUNCH();
  const dim3 g(Nc, BH);
  if (dtype == HVA_F32) {
    if (D == 64) hva_segment_mean_kernel<float, 64><<<g, 64, 0, st>>>(n, Nc, reinterpret_cast<const float*>(X), perm, base, mu, sums);
    else hva_segment_mean_kernel<float, 128><<<g, 128, 0, st>>>(n, Nc, reinterpret_cast<const float*>(X), perm, base, mu, sums);
  } else {
    if (D == 64) hva_segment_mean_kernel<__nv_bfloat16, 64><<<g, 64, 0, st>>>(n, Nc, reinterpret_cast<const __nv_bfloat16*>(X), perm, base, mu, sums);
    else hva_segment_mean_kernel<__nv_bfloat16, 128><<<g, 128, 0, st>>>(n, Nc, reinterpret_cast<const __nv_bfloat16*>(X), perm, base, mu, sums);
  }
  HVA_CHECK_LAUNCH();
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
  if (!s || !X || !perm || !Xp) return HVA_EINVAL;
  if (s->D != 64 && s->D != 128) return HVA_EINVAL;
  if (s->dtype != HVA_F32 && s->dtype != HVA_BF16) return HVA_EUNSUPPORTED;
  if ((size_t)s->B * s->heads * s->T * s->H * s->W >= 0x7fffffffull) return permute_common(s, X, perm, Xp, stream, 0);
  return hva_gather_kv(s, X, nullptr, perm, Xp, nullptr, reinterpret_cast<cudaStream_t>(stream));
}
extern "C" int hva_unpermute(const hva_shape* s, const void* Xp, const int32_t* perm, void* X, void* stream) {
  return permute_common(s, Xp, perm, X, stream, 1);
}

// K' and V' in one background launch for hva_forward's side stream: the same gather as hva_permute (both tensors share perm_k), but as
// two resident CTAs per SM with eight 16-byte loads in flight per thread instead of a grid that fills every thread slot -- it has
// to run UNDER the mask and merge kernels of the caller's stream, which need those slots (a full-occupancy gather just ran before
// them: no overlap).  The perm entries of the next iteration are fetched while the rows of the current one are in flight.
template <int RC, bool kBoth>     // 16-byte chunks per row: 8, 16 or 32; kBoth: K and V (else V, Vp are unused)
__global__ void __launch_bounds__(256) hva_gather_kv_kernel(unsigned rows_total, unsigned n, const uint4* __restrict__ K, const uint4* __restrict__ V,
                                                            const int* __restrict__ perm, uint4* __restrict__ Kp, uint4* __restrict__ Vp) {
  constexpr int RPW = 32 / RC, U = 4;                         // rows per warp instruction, instructions per iteration
  const int lane = threadIdx.x & 31, sub = lane / RC, q = lane % RC;
  const unsigned wg = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
  unsigned src[U], src_next[U];
  auto fetch = [&](unsigned base, unsigned (&out)[U]) {
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const unsigned row = base + u * RPW + sub;
      out[u] = row < rows_total ? (row / n) * n + (unsigned)__ldg(perm + row) : 0xffffffffu;
    }
  };
  unsigned base = wg * (U * RPW);
  const unsigned stride = nw * (U * RPW);
  if (base < rows_total) fetch(base, src_next);
  for (; base < rows_total; base += stride) {
#pragma unroll
    for (int u = 0; u < U; ++u) src[u] = src_next[u];
    uint4 kv[U], vv[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (src[u] != 0xffffffffu) { kv[u] = __ldg(K + (size_t)src[u] * RC + q); if (kBoth) vv[u] = __ldg(V + (size_t)src[u] * RC + q); }
    }
    if (base + stride < rows_total && base + stride > base) fetch(base + stride, src_next);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (src[u] != 0xffffffffu) {
        const size_t row = (size_t)base + u * RPW + sub;
        Kp[row * RC + q] = kv[u]; if (kBoth) Vp[row * RC + q] = vv[u];
      }
    }
  }
}

int hva_gather_kv(const hva_shape* s, const void* K, const void* V, const int32_t* perm, void* Kp, void* Vp, cudaStream_t st) {
  const int n = s->T * s->H * s->W;
  const size_t rows = (size_t)s->B * s->heads * n;
  if (rows >= 0x7fffffffull) return HVA_EUNSUPPORTED;
  const int rc = s->D * (s->dtype == HVA_F32 ? 4 : 2) / 16;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return HVA_ECUDA;
  const dim3 grid(2 * sms);                                   // one tensor alone (hva_permute): four CTAs per SM for the same bytes in flight
  const uint4 *k4 = reinterpret_cast<const uint4*>(K), *v4 = reinterpret_cast<const uint4*>(V);
  uint4 *kp4 = reinterpret_cast<uint4*>(Kp), *vp4 = reinterpret_cast<uint4*>(Vp);
  const unsigned r = (unsigned)rows, nn = (unsigned)n;
  if (V) {
    if (rc == 8) hva_gather_kv_kernel<8, true><<<grid, 256, 0, st>>>(r, nn, k4, v4, perm, kp4, vp4);
    else if (rc == 16) hva_gather_kv_kernel<16, true><<<grid, 256, 0, st>>>(r, nn, k4, v4, perm, kp4, vp4);
    else if (rc == 32) hva_gather_kv_kernel<32, true><<<grid, 256, 0, st>>>(r, nn, k4, v4, perm, kp4, vp4);
    else return HVA_EUNSUPPORTED;
  } else if (rc == 8) hva_gather_kv_kernel<8, false><<<dim3(4 * sms), 256, 0, st>>>(r, nn, k4, v4, perm, kp4, vp4);
  else if (rc == 16) hva_gather_kv_kernel<16, false><<<dim3(4 * sms), 256, 0, st>>>(r, nn, k4, v4, perm, kp4, vp4);
  else if (rc == 32) hva_gather_kv_kernel<32, false><<<dim3(4 * sms), 256, 0, st>>>(r, nn, k4, v4, perm, kp4, vp4);
  else return HVA_EUNSUPPORTED;
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

int hva_attention_dense_plan(int BH, int n, int tile_q, int tile_k, void* plan, const hva_plan_layout& L, cudaStream_t st) {
  PlanPtrs P = plan_ptrs(plan, L);
  hva_dense_plan_kernel<<<BH, 256, 0, st>>>(n, tile_q, tile_k, P);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// hva_build_plan_static: hva_build_plan for callers that cannot allocate (and have no scratch buffer of their own to pass):
// the scratch of the sort / group kernels (per-tile label histograms of Q and K, per-cluster row bases) lives in a file-scope
// device array of HVA_PLAN_STATIC_SCRATCH_BYTES.  Every GPU that loads the library holds the array until the process exits.
// The array's name below is only a host-side stand-in in host code: the kernels get the DEVICE address, which is looked up
// once per device (with that device current) by cudaGetSymbolAddress and kept in a table.  No cudaMalloc / cudaFree / allocating
// library call anywhere on this path.  All calls on a device share the array: two calls that overlap on the GPU (different
// streams, or one stream-captured graph replayed on two streams) race; calls on one stream are ordered and safe.  Nothing in the
// array has to start at zero: the kernels write every word they later read (hva_sort_hist_kernel stores the full histogram row
// of each tile, hva_plan_groups_kernel every row base), so the contents a previous call left behind are never observed.
namespace {
constexpr size_t kPlanStaticBytes = (size_t)HVA_PLAN_STATIC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_plan_static_scratch[kPlanStaticBytes];

struct PlanStaticDev {
  bool tried = false;
  cudaError_t err = cudaSuccess;
  void* ptr = nullptr;
};
constexpr int kPlanStaticMaxDevices = 64;

// device address of the array on the CURRENT device (looked up on first use on that device), or null
void* plan_static_scratch_ptr() {
  static PlanStaticDev tab[kPlanStaticMaxDevices];
  static std::mutex guard;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kPlanStaticMaxDevices) return nullptr;
  std::lock_guard<std::mutex> lock(guard);
  PlanStaticDev& e = tab[dev];
  if (!e.tried) {
    e.tried = true;
    void* p = nullptr;
    e.err = cudaGetSymbolAddress(&p, g_plan_static_scratch);
    if (e.err == cudaSuccess) e.ptr = p;
    else cudaGetLastError();
  }
  return e.err == cudaSuccess ? e.ptr : nullptr;
}
}  // namespace

extern "C" size_t hva_build_plan_static_limit(void) { return kPlanStaticBytes; }

extern "C" int hva_build_plan_static(int32_t BH, int32_t n, int32_t Nq, int32_t Nk, const int32_t* assign_q,
                                     const int32_t* assign_k, const int32_t* sizes_q, const int32_t* sizes_k,
                                     const int32_t* group_of_cluster, const int32_t* n_groups, const uint8_t* group_mask,
                                     int32_t tile_q, int32_t tile_k, void* plan, size_t plan_bytes, void* stream) {
  if (BH < 1 || n < 1 || Nq < 1 || Nk < 1) return HVA_EINVAL;
  if (hva_plan_ws_bytes(BH, n, Nq, Nk) > kPlanStaticBytes) return HVA_ELIMIT;   // before anything is enqueued
  void* scratch = plan_static_scratch_ptr();
  if (!scratch) return HVA_ECUDA;
  return hva_build_plan(BH, n, Nq, Nk, assign_q, assign_k, sizes_q, sizes_k, group_of_cluster, n_groups, group_mask, tile_q, tile_k,
                        plan, plan_bytes, scratch, kPlanStaticBytes, stream);
}
