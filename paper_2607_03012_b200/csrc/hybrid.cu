// S3 / S4: hybrid clustering across denoising steps (section 4.2 l.93-103; A.1 l.322).
//   hva_select_subset : top-m tokens by Lowe ratio (radix select + ordered compaction), ties -> lower index
//   hva_cluster_update: subset tokens re-assigned against ALL centroids (direct form, fp32, first
//                       minimum), then per-centroid deterministic adjustment of sums / sizes / mu
//                       (DESIGN.md R-H3), or a full refresh of every centroid (R-H3').
#include "common.cuh"
#include "cluster_tc.cuh"
#include <cooperative_groups.h>

namespace {

constexpr int kSelThreads = 1024;

// block-wide exclusive scan of a 0/1 flag; returns rank, *total receives the block count
__device__ __forceinline__ int block_rank(bool flag, int* s_warp, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned b = __ballot_sync(0xffffffffu, flag);
  int r = __popc(b & ((1u << lane) - 1));
  if (lane == 0) s_warp[warp] = __popc(b);
  __syncthreads();
  if (warp == 0) {
    int v = s_warp[lane], x = v;
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    s_warp[lane] = x - v;
    if (lane == 31) *total = x;
  }
  __syncthreads();
  r += s_warp[warp];
  return r;   // caller reads *total, then must __syncthreads() before the next call
}

// One thread-block CLUSTER of kSelCtas CTAs per (b, head) (round 1: one CTA per head, 24 CTAs on 148 SMs, 0.31 ms per tensor at C4):
// CTA r owns the contiguous slice r of the tokens; the 256-bin histograms of the MSB-first radix select are merged in CTA 0's shared
// memory through distributed-shared-memory atomics (integers: order-free), the digit decisions and the per-slice counts are read
// back from there, and every CTA compacts its own slice at its own output offset, in index order.
constexpr int kSelCtas = 8;
__global__ void __cluster_dims__(kSelCtas, 1, 1) __launch_bounds__(kSelThreads)
hva_select_subset_kernel(int n, int m, const float* __restrict__ lowe, int* __restrict__ subset) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank(), bh = blockIdx.x / kSelCtas, tid = threadIdx.x;
  const uint32_t* bits = reinterpret_cast<const uint32_t*>(lowe) + (size_t)bh * n;   // rho >= 0: bit order == value order
  const int L = (n + kSelCtas - 1) / kSelCtas, i_lo = rank * L, i_hi = min(n, i_lo + L);
  __shared__ int s_hist[256];            // CTA 0's copy is the cluster-wide histogram
  __shared__ int s_loc[256];
  __shared__ int s_warp[32];
  __shared__ int s_tot;
  __shared__ uint32_t s_prefix;          // (CTA 0) digits decided so far
  __shared__ int s_remain;               // (CTA 0) how many of the m are still to be found among the undecided values
  __shared__ int s_cnt[kSelCtas][2];     // (CTA 0) per slice: values > threshold, values == threshold
  int* g_hist = cluster.map_shared_rank(s_hist, 0);
  if (tid < 256) s_hist[tid] = 0;
  if (tid == 0) { s_prefix = 0; s_remain = m; }
  cluster.sync();
  uint32_t prefix = 0;
  // MSB-first radix select of the m-th largest value
  for (int shift = 24; shift >= 0; shift -= 8) {
    if (tid < 256) s_loc[tid] = 0;
    __syncthreads();
    const uint32_t pmask = shift == 24 ? 0u : (0xffffffffu << (shift + 8));
    for (int i0 = i_lo; i0 < i_hi; i0 += kSelThreads) {   // warp-aggregated: rho values share their top bytes
      const int i = i0 + tid;
      const uint32_t v = i < i_hi ? bits[i] : 0u;
      const int key = (i < i_hi && (v & pmask) == prefix) ? (int)((v >> shift) & 255) : -1;
      const unsigned peers = __match_any_sync(0xffffffffu, key);
      if (key >= 0 && (peers & ((1u << (tid & 31)) - 1)) == 0) atomicAdd(&s_loc[key], __popc(peers));
    }
    __syncthreads();
    if (tid < 256 && s_loc[tid]) atomicAdd(&g_hist[tid], s_loc[tid]);
    cluster.sync();
    if (rank == 0 && tid == 0) {
      int rem = s_remain, d = 255;
      for (; d > 0; --d) { if (s_hist[d] >= rem) break; rem -= s_hist[d]; }
      s_prefix = prefix | ((uint32_t)d << shift);
      s_remain = rem;
    }
    if (rank == 0) {
      __syncthreads();
      if (tid < 256) s_hist[tid] = 0;
    }
    cluster.sync();
    prefix = *cluster.map_shared_rank(&s_prefix, 0);
  }
  const uint32_t thr = prefix;             // m-th largest value
  const int need_eq = *cluster.map_shared_rank(&s_remain, 0);   // how many == thr to take (lowest indices first)
  // per-slice counts -> this slice's output offset and the number of == thr values the earlier slices take
  int gt = 0, eq = 0;
  for (int i = i_lo + tid; i < i_hi; i += kSelThreads) { const uint32_t v = bits[i]; gt += v > thr; eq += v == thr; }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { gt += __shfl_xor_sync(0xffffffffu, gt, o); eq += __shfl_xor_sync(0xffffffffu, eq, o); }
  if ((tid & 31) == 0) { s_warp[tid >> 5] = gt; s_loc[tid >> 5] = eq; }
  __syncthreads();
  if (tid == 0) {
    int a = 0, e = 0;
    for (int w = 0; w < kSelThreads / 32; ++w) { a += s_warp[w]; e += s_loc[w]; }
    int* c = cluster.map_shared_rank(&s_cnt[rank][0], 0);
    c[0] = a; c[1] = e;
  }
  cluster.sync();
  int out = 0, eq_seen = 0;
  {
    const int (*c)[2] = reinterpret_cast<const int (*)[2]>(cluster.map_shared_rank(&s_cnt[0][0], 0));
    for (int r = 0; r < rank; ++r) {
      const int take = max(0, min(c[r][1], need_eq - eq_seen));
      out += c[r][0] + take;
      eq_seen += c[r][1];
    }
  }
  cluster.sync();        // (nobody reads CTA 0's shared memory after this point: it may exit)
  for (int i0 = i_lo; i0 < i_hi; i0 += kSelThreads) {
    const int i = i0 + tid;
    const uint32_t v = i < i_hi ? bits[i] : 0u;
    const bool gtv = i < i_hi && v > thr, eqv = i < i_hi && v == thr;
    const int eq_rank = block_rank(eqv, s_warp, &s_tot);
    const int eq_tot = s_tot;
    __syncthreads();
    const bool take = gtv || (eqv && eq_seen + eq_rank < need_eq);
    const int r = block_rank(take, s_warp, &s_tot);
    const int tot = s_tot;
    __syncthreads();
    if (take) subset[(size_t)bh * m + out + r] = i;
    out += tot; eq_seen += eq_tot;
  }
}

// ---- subset re-assignment against all centroids (thread = subset token, centroid tiles in smem)
constexpr int kUpdThreads = 128, kCTile = 32, kCB2 = 8;

__device__ __forceinline__ void ld8(const float* p, float x[8]) {
  float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
  x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y; x[6] = b.z; x[7] = b.w;
}
__device__ __forceinline__ void ld8(const __nv_bfloat16* p, float x[8]) {
  uint4 r = *reinterpret_cast<const uint4*>(p);
  x[0] = __uint_as_float(r.x << 16); x[1] = __uint_as_float(r.x & 0xffff0000u);
  x[2] = __uint_as_float(r.y << 16); x[3] = __uint_as_float(r.y & 0xffff0000u);
  x[4] = __uint_as_float(r.z << 16); x[5] = __uint_as_float(r.z & 0xffff0000u);
  x[6] = __uint_as_float(r.w << 16); x[7] = __uint_as_float(r.w & 0xffff0000u);
}

template <typename T, int D>
__global__ void __launch_bounds__(kUpdThreads) hva_subset_assign_kernel(int n, int Nc, int m, const T* __restrict__ X,
                                                                        const int* __restrict__ subset,
                                                                        const float* __restrict__ mu,
                                                                        const int* __restrict__ assign,
                                                                        int* __restrict__ oldlab, int* __restrict__ newlab) {
  constexpr int kVec = 16 / sizeof(T), kRow = D + kVec;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* s_mu = reinterpret_cast<float*>(smem_raw);            // [kCTile][D]
  T* s_x = reinterpret_cast<T*>(s_mu + kCTile * D);            // [kUpdThreads][kRow]
  const int bh = blockIdx.y, tid = threadIdx.x, i0 = blockIdx.x * kUpdThreads;
  constexpr int kChunks = D / kVec;
  for (int e = tid; e < kUpdThreads * kChunks; e += kUpdThreads) {
    int li = e / kChunks, q = e % kChunks;
    if (i0 + li < m) {
      size_t tok = (size_t)bh * n + subset[(size_t)bh * m + i0 + li];
      *reinterpret_cast<uint4*>(s_x + (size_t)li * kRow + q * kVec) = __ldg(reinterpret_cast<const uint4*>(X + tok * D) + q);
    }
  }
  float best = __int_as_float(0x7f800000);
  int lab = 0;
  const T* xr = s_x + (size_t)tid * kRow;
  for (int u0 = 0; u0 < Nc; u0 += kCTile) {
    __syncthreads();
    for (int e = tid; e < kCTile * (D / 4); e += kUpdThreads) {
      int v = e / (D / 4), q = e % (D / 4);
      int u = min(u0 + v, Nc - 1);
      reinterpret_cast<float4*>(s_mu)[e] = reinterpret_cast<const float4*>(mu + ((size_t)bh * Nc + u) * D)[q];
    }
    __syncthreads();
    if (i0 + tid < m) {
      for (int v0 = 0; v0 < kCTile; v0 += kCB2) {
        float acc[kCB2];
#pragma unroll
        for (int j = 0; j < kCB2; ++j) acc[j] = 0.f;
        for (int c0 = 0; c0 < D; c0 += 8) {
          float x[8];
          ld8(xr + c0, x);
#pragma unroll
          for (int j = 0; j < kCB2; ++j) {
            float mm[8];
            ld8(s_mu + (size_t)(v0 + j) * D + c0, mm);
#pragma unroll
            for (int e = 0; e < 8; ++e) { float d = x[e] - mm[e]; acc[j] = fmaf(d, d, acc[j]); }
          }
        }
#pragma unroll
        for (int j = 0; j < kCB2; ++j)
          if (u0 + v0 + j < Nc && acc[j] < best) { best = acc[j]; lab = u0 + v0 + j; }   // first minimum
      }
    }
  }
  if (i0 + tid < m) {
    newlab[(size_t)bh * m + i0 + tid] = lab;
    oldlab[(size_t)bh * m + i0 + tid] = assign[(size_t)bh * n + subset[(size_t)bh * m + i0 + tid]];
  }
}

// ---- per-centroid deterministic adjustment (R-H3): moves are applied in subset order.
// The moved subset entries are bucketed by centroid (count / scan / scatter; the scatter order inside a bucket is
// arbitrary), the CTA of centroid u then sorts its few entries by subset position and applies them sequentially,
// thread = feature dim: the result does not depend on the scatter order.
constexpr int kMoveCap = 1024;   // entries of one centroid sorted in shared memory; beyond that the subset is scanned

__global__ void hva_moves_count_kernel(int Nc, int m, const int* __restrict__ oldlab, const int* __restrict__ newlab,
                                       int* __restrict__ cnt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, bh = blockIdx.y;
  if (i >= m) return;
  const int ol = oldlab[(size_t)bh * m + i], nl = newlab[(size_t)bh * m + i];
  if (ol != nl) { atomicAdd(&cnt[(size_t)bh * (Nc + 1) + ol], 1); atomicAdd(&cnt[(size_t)bh * (Nc + 1) + nl], 1); }
}

// cnt[bh][0..Nc) -> exclusive offsets off[bh][0..Nc] (in place) and a copy as scatter cursors
__global__ void __launch_bounds__(1024) hva_moves_scan_kernel(int Nc, int* __restrict__ cnt, int* __restrict__ cursor) {
  const int bh = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  __shared__ int s_warp[32];
  __shared__ int s_carry;
  if (tid == 0) s_carry = 0;
  __syncthreads();
  for (int u0 = 0; u0 <= Nc; u0 += 1024) {
    const int u = u0 + tid;
    const int v = u < Nc ? cnt[(size_t)bh * (Nc + 1) + u] : 0;
    int x = v;
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) s_warp[warp] = x;
    __syncthreads();
    if (warp == 0) {
      int w = s_warp[lane], t = w;
      for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, t, o); if (lane >= o) t += y; }
      s_warp[lane] = t - w;
    }
    __syncthreads();
    const int excl = s_carry + s_warp[warp] + x - v;
    if (u <= Nc) { cnt[(size_t)bh * (Nc + 1) + u] = excl; if (u < Nc) cursor[(size_t)bh * Nc + u] = excl; }
    __syncthreads();
    if (tid == 1023) s_carry = excl + v;
    __syncthreads();
  }
}

__global__ void hva_moves_scatter_kernel(int Nc, int m, const int* __restrict__ oldlab, const int* __restrict__ newlab,
                                         int* __restrict__ cursor, int* __restrict__ entries) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, bh = blockIdx.y;
  if (i >= m) return;
  const int ol = oldlab[(size_t)bh * m + i], nl = newlab[(size_t)bh * m + i];
  if (ol != nl) {
    entries[(size_t)bh * 2 * m + atomicAdd(&cursor[(size_t)bh * Nc + ol], 1)] = i << 1;         // leaves ol
    entries[(size_t)bh * 2 * m + atomicAdd(&cursor[(size_t)bh * Nc + nl], 1)] = (i << 1) | 1;   // joins nl
  }
}

template <typename T, int D>
__global__ void __launch_bounds__(D) hva_subset_apply_kernel(int n, int Nc, int m, const T* __restrict__ X,
                                                             const int* __restrict__ subset, const int* __restrict__ oldlab,
                                                             const int* __restrict__ newlab, const int* __restrict__ off,
                                                             const int* __restrict__ entries, float* __restrict__ mu,
                                                             float* __restrict__ sums, int* __restrict__ sizes) {
  const int u = blockIdx.x, bh = blockIdx.y, c = threadIdx.x, lane = c & 31, warp = c >> 5;
  const int e0 = off[(size_t)bh * (Nc + 1) + u], k = off[(size_t)bh * (Nc + 1) + u + 1] - e0;
  if (k == 0) return;                              // untouched centroid
  const size_t o = ((size_t)bh * Nc + u) * D + c;
  float z = sums[o];
  int cnt = sizes[(size_t)bh * Nc + u];
  if (k <= kMoveCap) {
    __shared__ int s_raw[kMoveCap], s_sorted[kMoveCap];
    for (int e = c; e < k; e += D) s_raw[e] = entries[(size_t)bh * 2 * m + e0 + e];
    __syncthreads();
    for (int e = c; e < k; e += D) {               // keys are distinct: rank = number of smaller keys
      const int key = s_raw[e];
      int rank = 0;
      for (int f = 0; f < k; ++f) rank += s_raw[f] < key;
      s_sorted[rank] = key;
    }
    __syncthreads();
    for (int e = 0; e < k; ++e) {
      const int key = s_sorted[e];
      const float x = HvaElem<T>::ld(X + ((size_t)bh * n + subset[(size_t)bh * m + (key >> 1)]) * D + c);
      if (key & 1) { z += x; ++cnt; } else { z -= x; --cnt; }
    }
  } else {                                         // degenerate: scan the subset in order (one entry per thread, ballot)
    __shared__ unsigned s_bal[D / 32];
    __shared__ int s_tok[D];
    __shared__ int s_dir[D];
    for (int i0 = 0; i0 < m; i0 += D) {
      const int i = i0 + c;
      int ol = -1, nl = -1;
      if (i < m) { ol = oldlab[(size_t)bh * m + i]; nl = newlab[(size_t)bh * m + i]; }
      const bool hit = (ol != nl) && (ol == u || nl == u);
      const unsigned b = __ballot_sync(0xffffffffu, hit);
      if (lane == 0) s_bal[warp] = b;
      if (hit) { s_tok[c] = subset[(size_t)bh * m + i]; s_dir[c] = (ol == u) ? -1 : 1; }
      __syncthreads();
      for (int w = 0; w < D / 32; ++w) {
        unsigned bits = s_bal[w];
        while (bits) {
          int e = w * 32 + __ffs(bits) - 1;
          bits &= bits - 1;
          float x = HvaElem<T>::ld(X + ((size_t)bh * n + s_tok[e]) * D + c);
          if (s_dir[e] < 0) { z -= x; --cnt; } else { z += x; ++cnt; }
        }
      }
      __syncthreads();
    }
  }
  sums[o] = z;
  if (c == 0) sizes[(size_t)bh * Nc + u] = cnt;
  if (cnt > 0) mu[o] = __fdiv_rn(z, (float)cnt);
}

__global__ void hva_subset_commit_kernel(int n, int m, const int* __restrict__ subset, const int* __restrict__ newlab,
                                         int* __restrict__ assign) {
  int i = blockIdx.x * blockDim.x + threadIdx.x, bh = blockIdx.y;
  if (i < m) assign[(size_t)bh * n + subset[(size_t)bh * m + i]] = newlab[(size_t)bh * m + i];
}

template <typename T, int D>
int run_update(int BH, int n, int Nc, int m, const void* X, const int* subset, int refresh_all, int* assign, float* mu,
               float* sums, int* sizes, int* newlab, char* split, int dtype, uint32_t flags, void* rws, size_t rws_bytes, cudaStream_t st) {
  int* oldlab = newlab + (size_t)BH * (m > 0 ? m : 1);
  const T* x = reinterpret_cast<const T*>(X);
  if (m > 0 && hva_subset_tc_supported(D, dtype, Nc) && !(flags & HVA_FLAG_CLUSTER_SIMT)) {
    // tensor-pipe path: split the cached centroids, then the dense m x N_c x D filter with exact refine (hybrid_tc.cu)
    char* hi = split;
    char* lo = hi + hva_align((size_t)BH * Nc * D * 2);
    float* musq = reinterpret_cast<float*>(lo + hva_align((size_t)BH * Nc * D * 2));
    HVA_TRY(hva_mu_split_launch(BH, Nc, D, mu, hi, lo, musq, st));
    HVA_TRY(hva_subset_assign_tc_launch(BH, n, Nc, m, X, subset, mu, hi, lo, musq, assign, oldlab, newlab, st));
  } else if (m > 0) {
    size_t smem = (size_t)kCTile * D * 4 + (size_t)kUpdThreads * (D + 16 / sizeof(T)) * sizeof(T);
    if (cudaFuncSetAttribute(hva_subset_assign_kernel<T, D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
      return HVA_ECUDA;
    hva_subset_assign_kernel<T, D><<<dim3((m + kUpdThreads - 1) / kUpdThreads, BH), kUpdThreads, smem, st>>>(n, Nc, m, x, subset, mu, assign, oldlab, newlab);
    HVA_CHECK_LAUNCH();
  }
  if (!refresh_all && m > 0) {
    int* off = reinterpret_cast<int*>(split + 2 * hva_align((size_t)BH * Nc * D * 2) + hva_align((size_t)BH * Nc * 4));
    int* cursor = off + hva_align((size_t)BH * (Nc + 1) * 4) / 4;
    int* entries = cursor + hva_align((size_t)BH * Nc * 4) / 4;
    if (cudaMemsetAsync(off, 0, (size_t)BH * (Nc + 1) * 4, st) != cudaSuccess) return HVA_ECUDA;
    hva_moves_count_kernel<<<dim3((m + 255) / 256, BH), 256, 0, st>>>(Nc, m, oldlab, newlab, off);
    HVA_CHECK_LAUNCH();
    hva_moves_scan_kernel<<<BH, 1024, 0, st>>>(Nc, off, cursor);
    HVA_CHECK_LAUNCH();
    hva_moves_scatter_kernel<<<dim3((m + 255) / 256, BH), 256, 0, st>>>(Nc, m, oldlab, newlab, cursor, entries);
    HVA_CHECK_LAUNCH();
    hva_subset_apply_kernel<T, D><<<dim3(Nc, BH), D, 0, st>>>(n, Nc, m, x, subset, oldlab, newlab, off, entries, mu, sums, sizes);
    HVA_CHECK_LAUNCH();
  }
  if (m > 0) {
    hva_subset_commit_kernel<<<dim3((m + 255) / 256, BH), 256, 0, st>>>(n, m, subset, newlab, assign);
    HVA_CHECK_LAUNCH();
  }
  if (refresh_all) HVA_TRY(hva_refresh_centroids(BH, n, Nc, D, dtype, X, assign, mu, sums, sizes, rws, rws_bytes, st));
  return HVA_OK;
}

}  // namespace

static size_t hybrid_step_bytes(int BH, int Nc, int m, int D) {
  return hva_align((size_t)BH * (m > 0 ? m : 1) * 8) + 2 * hva_align((size_t)BH * Nc * D * 2) + hva_align((size_t)BH * Nc * 4) +
         hva_align((size_t)BH * (Nc + 1) * 4) + hva_align((size_t)BH * Nc * 4) + hva_align((size_t)BH * 2 * (m > 0 ? m : 1) * 4);
}
size_t hva_hybrid_ws_bytes(int BH, int n, int Nc, int m, int D) {
  return hybrid_step_bytes(BH, Nc, m, D) + hva_refresh_ws_bytes(BH, n, Nc);      // (the refresh of R-H3' sorts the tokens by label)
}

extern "C" size_t hva_cluster_update_workspace_bytes(const hva_shape* s, int32_t Nc, int32_t m) {
  if (!s || Nc < 1 || m < 0 || s->B < 1 || s->heads < 1) return 0;
  return hva_hybrid_ws_bytes(s->B * s->heads, s->T * s->H * s->W, Nc, m, s->D);
}

extern "C" int hva_select_subset(int32_t BH, int32_t n, const float* lowe, int32_t m, int32_t* subset, void* ws,
                                 size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  if (!lowe || !subset || BH < 1 || n < 1 || m < 0 || m > n) return HVA_EINVAL;
  if (m == 0) return HVA_OK;
  hva_select_subset_kernel<<<BH * kSelCtas, kSelThreads, 0, reinterpret_cast<cudaStream_t>(stream)>>>(n, m, lowe, subset);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

extern "C" int hva_cluster_update(const hva_shape* s, int32_t Nc, const void* X, const int32_t* subset, int32_t m,
                                  int32_t refresh_all, int32_t* assign, float* mu, float* sums, int32_t* sizes, void* ws,
                                  size_t ws_bytes, void* stream) {
  return hva_cluster_update_ex(s, Nc, X, subset, m, refresh_all, assign, mu, sums, sizes, 0u, ws, ws_bytes, stream);
}

extern "C" int hva_cluster_update_ex(const hva_shape* s, int32_t Nc, const void* X, const int32_t* subset, int32_t m,
                                     int32_t refresh_all, int32_t* assign, float* mu, float* sums, int32_t* sizes, uint32_t flags,
                                     void* ws, size_t ws_bytes, void* stream) {
  if (!s || !X || !subset || !assign || !mu || !sums || !sizes || !ws) return HVA_EINVAL;
  if (Nc < 1 || m < 0 || (s->D != 64 && s->D != 128)) return HVA_EINVAL;
  if (s->dtype != HVA_F32 && s->dtype != HVA_BF16) return HVA_EUNSUPPORTED;
  const int BH = s->B * s->heads, n = s->T * s->H * s->W;
  if (m > n) return HVA_EINVAL;
  if (ws_bytes < hva_hybrid_ws_bytes(BH, n, Nc, m, s->D)) return HVA_EWORKSPACE;
  if (m == 0 && !refresh_all) return HVA_OK;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  int* newlab = reinterpret_cast<int*>(ws);
  char* split = reinterpret_cast<char*>(ws) + hva_align((size_t)BH * (m > 0 ? m : 1) * 8);
  void* rws = reinterpret_cast<char*>(ws) + hybrid_step_bytes(BH, Nc, m, s->D);
  const size_t rws_bytes = hva_refresh_ws_bytes(BH, n, Nc);
#define HVA_DISPATCH(T, DD) return run_update<T, DD>(BH, n, Nc, m, X, subset, refresh_all, assign, mu, sums, sizes, newlab, split, s->dtype, flags, rws, rws_bytes, st)
  if (s->dtype == HVA_F32) { if (s->D == 64) HVA_DISPATCH(float, 64); HVA_DISPATCH(float, 128); }
  if (s->D == 64) HVA_DISPATCH(__nv_bfloat16, 64);
  HVA_DISPATCH(__nv_bfloat16, 128);
#undef HVA_DISPATCH
}
