// S5: centroid scores, size-weighted softmax and row-wise top-p (Eq. 2-3, l.47-54;
// "Top-p" / "Min-kc" l.332-334).  One CTA per (bh, query cluster) row.  Scores and weights are
// evaluated in fp64 from the fp32 centroids so that the cut decision matches the fp64 oracle
// (DESIGN.md R-K3); each CTA scores kRowsPerCta query clusters per pass over mu^k: w_j = s^k_j exp(S_j - max_j S_j); sort by (w desc, j asc) with an in-smem
// bitonic network; inclusive scan; k = first position with cum >= top_p * Z; keep at least kmin.
#include "common.cuh"

namespace {

constexpr int kMaskThreads = 256;

__device__ __forceinline__ bool before(double wa, int ja, double wb, int jb) {
  return wa > wb || (wa == wb && ja < jb);  // descending weight, ties -> lower j
}

constexpr int kRowsPerCta = 4;   // query clusters per CTA: every mu^k row read from L2 is used for 4 scores

template <int D>
__global__ void __launch_bounds__(kMaskThreads) hva_mask_kernel(int Nq, int Nk, int P, const float* __restrict__ mu_q,
                                                                const float* __restrict__ mu_k,
                                                                const int* __restrict__ sizes_k, double scale,
                                                                double top_p, int all_ones, int kmin,
                                                                uint8_t* __restrict__ mask) {
  const int i0 = blockIdx.x * kRowsPerCta, bh = blockIdx.y, tid = threadIdx.x;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* s_w = reinterpret_cast<double*>(smem_raw);        // [P] weights of the row being sorted
  double* s_sc = s_w + P;                                   // [kRowsPerCta][Nk] scores S_ij
  double* s_q = s_sc + (size_t)kRowsPerCta * Nk;            // [kRowsPerCta][D]
  double* s_red = s_q + kRowsPerCta * D;                    // [kMaskThreads]
  int* s_j = reinterpret_cast<int*>(s_red + kMaskThreads);  // [P]
  __shared__ int s_k;

  const int nrows = min(kRowsPerCta, Nq - i0);
  if (all_ones) {  // top_p >= 1 selects every key cluster (R-K1)
    for (int e = tid; e < nrows * Nk; e += kMaskThreads) mask[((size_t)bh * Nq + i0) * Nk + e] = 1;
    return;
  }
  for (int e = tid; e < kRowsPerCta * D; e += kMaskThreads) {
    int r = e / D;
    s_q[e] = r < nrows ? (double)mu_q[((size_t)bh * Nq + i0 + r) * D + (e % D)] : 0.0;
  }
  __syncthreads();
  // S_ij = <mu^q_i, mu^k_j> * scale   (Eq. 2), fp64 accumulation in ascending feature order
  for (int j = tid; j < Nk; j += kMaskThreads) {
    const float4* kr = reinterpret_cast<const float4*>(mu_k + ((size_t)bh * Nk + j) * D);
    double a[kRowsPerCta];
#pragma unroll
    for (int r = 0; r < kRowsPerCta; ++r) a[r] = 0.0;
#pragma unroll 2
    for (int c = 0; c < D / 4; ++c) {
      float4 v = __ldg(kr + c);
      const double x0 = v.x, x1 = v.y, x2 = v.z, x3 = v.w;
#pragma unroll
      for (int r = 0; r < kRowsPerCta; ++r) {
        const double* q = s_q + r * D + 4 * c;
        a[r] = fma(x0, q[0], a[r]); a[r] = fma(x1, q[1], a[r]); a[r] = fma(x2, q[2], a[r]); a[r] = fma(x3, q[3], a[r]);
      }
    }
#pragma unroll
    for (int r = 0; r < kRowsPerCta; ++r) s_sc[(size_t)r * Nk + j] = a[r] * scale;
  }
  __syncthreads();

  for (int r = 0; r < nrows; ++r) {
    uint8_t* mrow = mask + ((size_t)bh * Nq + i0 + r) * Nk;
    double lmax = -1.0 / 0.0;
    for (int j = tid; j < Nk; j += kMaskThreads) lmax = fmax(lmax, s_sc[(size_t)r * Nk + j]);
    s_red[tid] = lmax;
    __syncthreads();
    for (int o = kMaskThreads / 2; o > 0; o >>= 1) {
      if (tid < o) s_red[tid] = fmax(s_red[tid], s_red[tid + o]);
      __syncthreads();
    }
    const double smax = s_red[0];
    __syncthreads();
    for (int j = tid; j < P; j += kMaskThreads) {   // w_j = s^k_j exp(S_j - max); pads (-1) sort last
      s_w[j] = (j < Nk) ? (double)sizes_k[(size_t)bh * Nk + j] * exp(s_sc[(size_t)r * Nk + j] - smax) : -1.0;
      s_j[j] = j;
    }
    __syncthreads();
    // bitonic sort, order `before`.  Warp w owns the contiguous segment [w seg, (w+1) seg), seg = P / 8: every pass with
    // j < seg stays inside the segment and only needs a warp-level barrier; block barriers around the passes that cross
    // segments (10 instead of 55 for P = 1024).
    const int seg = P / (kMaskThreads / 32), wbase = (tid >> 5) * seg, lane = tid & 31;
    for (int k = 2; k <= P; k <<= 1) {
      for (int j = k >> 1; j > 0; j >>= 1) {
        for (int a = wbase + lane; a < wbase + seg; a += 32) {
          int b = a ^ j;
          if (b > a) {
            double wa = s_w[a], wb = s_w[b];
            int ja = s_j[a], jb = s_j[b];
            bool up = ((a & k) == 0);
            bool swap = up ? before(wb, jb, wa, ja) : before(wa, ja, wb, jb);
            if (swap) { s_w[a] = wb; s_w[b] = wa; s_j[a] = jb; s_j[b] = ja; }
          }
        }
        if (j >= seg || (j == 1 && k >= seg)) __syncthreads(); else __syncwarp();
      }
    }
    // inclusive scan of the sorted weights: per-thread contiguous chunk, then scan of the chunk sums
    const int chunk = P / kMaskThreads;
    const int lo = tid * chunk;
    double run = 0.0;
    for (int x = lo; x < lo + chunk; ++x) run += (x < Nk ? s_w[x] : 0.0);
    s_red[tid] = run;
    __syncthreads();
    if (tid == 0) {  // sequential exclusive scan of the 256 chunk sums (ascending, like a cumulative sum)
      double a = 0.0;
      for (int t = 0; t < kMaskThreads; ++t) { double v = s_red[t]; s_red[t] = a; a += v; }
      s_k = Nk;
    }
    __syncthreads();
    double Z = s_red[kMaskThreads - 1];
    for (int x = (kMaskThreads - 1) * chunk; x < P; ++x) Z += (x < Nk ? s_w[x] : 0.0);
    const double thr = top_p * Z;
    {
      double a = s_red[tid];
      for (int x = lo; x < lo + chunk && x < Nk; ++x) {
        a += s_w[x];
        if (a >= thr) { atomicMin(&s_k, x + 1); break; }   // smallest k with cum_k >= p Z   (Eq. 3)
      }
    }
    __syncthreads();
    const int k = s_k < kmin ? kmin : s_k;
    for (int x = tid; x < Nk; x += kMaskThreads) mrow[s_j[x]] = (x < k) ? 1 : 0;
    __syncthreads();
  }
}

// ---- warp-per-row variant (Nk <= 1024): 8 query clusters per CTA.  The scores of the 8 rows are computed by the block
// (thread = key cluster, every mu^k element read once for 8 fp64 dot products); then warp w owns row w: each lane holds E
// of the row's P = 32 E (weight, j) pairs in registers (position = lane E + i) and the bitonic network runs without shared
// memory or block barriers: distances < E are register-to-register inside a lane, distances >= E are lane-to-lane shuffles.
// One element = ONE 64-bit key: the weight's fp64 bits (w >= 0: bit order == value order) with the low 11 mantissa bits replaced
// by 2047 - j, so that "weight descending, ties -> lower j" is a single unsigned compare and a swap moves two registers (round 1
// sorted (double, int) pairs with two fp64 compares per exchange: 19.5 % fp64 pipe, 1.66 ms at C4).  The weight loses 11 of its 52
// mantissa bits (relative 4.5e-13): the cumulative sums below use the truncated weights, far inside R-K3's 1e-9 Z exemption; two
// DIFFERENT weights that agree in their leading 41 mantissa bits are ordered by index instead of by value (probability ~1e-10 per
// adjacent pair, and it only matters if the cut falls between the two).  Exact ties, empty clusters (w = 0) and pads (key 0,
// j >= N_k) order exactly as the oracle's.
template <int E>
struct WarpSort {
  unsigned long long k[E];
  __device__ __forceinline__ void cex(int a, int b, bool up) {      // positions a < b inside the lane; `up`: larger key first
    const unsigned long long x = k[a], y = k[b];
    const bool sw = up ? (y > x) : (x > y);
    k[a] = sw ? y : x; k[b] = sw ? x : y;
  }
  // descending sort of the lane's own E keys only (the within-lane stages of the network): no shuffles
  __device__ __forceinline__ void sort_lane() {
#pragma unroll
    for (int kk = 2; kk <= E; kk <<= 1) {
#pragma unroll
      for (int d = kk >> 1; d > 0; d >>= 1) {
#pragma unroll
        for (int i = 0; i < E; ++i)
          if ((i & d) == 0) cex(i, i | d, kk < E ? ((i & kk) == 0) : true);
      }
    }
  }
  __device__ __forceinline__ void sort(int lane) {
#pragma unroll
    for (int kk = 2; kk <= 32 * E; kk <<= 1) {
#pragma unroll
      for (int d = kk >> 1; d > 0; d >>= 1) {
        if (d >= E) {                                                 // partner lane, same register index
          const int lm = d / E;
          const bool up = ((lane * E) & kk) == 0, lower = (lane & lm) == 0;
          const bool keep_larger = (lower == up);                     // this position keeps the pair's larger key
#pragma unroll
          for (int i = 0; i < E; ++i) {
            const unsigned long long o = __shfl_xor_sync(0xffffffffu, k[i], lm);
            const bool mine_larger = k[i] > o;
            if (mine_larger != keep_larger) k[i] = o;
          }
        } else {
#pragma unroll
          for (int i = 0; i < E; ++i) {
            if ((i & d) == 0) {
              const bool up = kk < E ? ((i & kk) == 0) : ((((lane * E) | i) & kk) == 0);
              cex(i, i | d, up);
            }
          }
        }
      }
    }
  }
};
__device__ __forceinline__ unsigned long long mask_key(double w, int j) {     // w >= 0
  return ((unsigned long long)__double_as_longlong(w) & ~0x7FFull) | (unsigned long long)(2047 - j);
}
__device__ __forceinline__ double mask_key_w(unsigned long long k) { return __longlong_as_double((long long)(k & ~0x7FFull)); }
__device__ __forceinline__ int mask_key_j(unsigned long long k) { return 2047 - (int)(k & 0x7FFull); }

constexpr int kWarpRows = 8;

// E keys per lane and sorted run, R runs per lane (R = 2: 1024 < N_k <= 2048, two runs of 32: the selection below works on sorted
// runs, so a lane never holds more than 32 keys in registers)
template <int D, int E, int R>
__global__ void __launch_bounds__(256, 2) hva_mask_warp_kernel(int Nq, int Nk, const float* __restrict__ mu_q,
                                                            const float* __restrict__ mu_k, const int* __restrict__ sizes_k,
                                                            double scale, double top_p, int kmin, uint8_t* __restrict__ mask) {
  constexpr int P = 32 * E * R;
  const int i0 = blockIdx.x * kWarpRows, bh = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* s_q = reinterpret_cast<double*>(smem_raw);         // [kWarpRows][D]
  double* s_sc = s_q + kWarpRows * D;                        // [kWarpRows][P] scores S_ij
  const int nrows = min(kWarpRows, Nq - i0);
  for (int e = tid; e < kWarpRows * D; e += 256) {
    const int r = e / D;
    s_q[e] = r < nrows ? (double)mu_q[((size_t)bh * Nq + i0 + r) * D + (e % D)] : 0.0;
  }
  __syncthreads();
  // S_ij = <mu^q_i, mu^k_j> * scale   (Eq. 2) in fp64 on the fp64 tensor path: one mma.m8n8k4 = the CTA's 8 query rows x 8 key
  // clusters x 4 feature dims (256 FMAs per warp instruction, operands in registers; the CUDA-core form spent 6.6 K instructions
  // per row on DFMA + shared-memory operand loads, half of the kernel).  Thread (g = lane / 4, t = lane % 4) holds A[g][t], B[t][g]
  // and C[g][2t, 2t+1].  The k-steps walk the feature dims in the order 16 s + 4 t + e (s = 0 .. D/16 - 1, e = 0 .. 3), so that the
  // thread's four B values of a step group are ONE 16-byte load of its key row; A is laid out to match and is loaded once per warp.
  // The sum over the dims is associated as the tensor unit does it (fixed, deterministic); the products and the accumulation are
  // fp64, so the scores agree with any other fp64 order to ~1e-16 relative (R-K3).
  {
    const int g = lane >> 2, t = lane & 3;
    double aq[D / 4];
#pragma unroll
    for (int s4 = 0; s4 < D / 16; ++s4)
#pragma unroll
      for (int e = 0; e < 4; ++e) aq[4 * s4 + e] = s_q[g * D + 16 * s4 + 4 * t + e];
    const int nblk = (Nk + 7) >> 3;
    for (int blk = warp; blk < nblk; blk += 8) {
      const int n = min(8 * blk + g, Nk - 1);                 // keys past N_k re-read the last row; their columns are not stored
      const float4* kr = reinterpret_cast<const float4*>(mu_k + ((size_t)bh * Nk + n) * D) + t;
      double c0 = 0.0, c1 = 0.0;
#pragma unroll
      for (int s4 = 0; s4 < D / 16; ++s4) {
        const float4 v = __ldg(kr + 4 * s4);
        const double bv[4] = {(double)v.x, (double)v.y, (double)v.z, (double)v.w};
#pragma unroll
        for (int e = 0; e < 4; ++e)
          asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                       : "+d"(c0), "+d"(c1) : "d"(aq[4 * s4 + e]), "d"(bv[e]));
      }
      const int j0 = 8 * blk + 2 * t;
      if (g < nrows) {
        if (j0 < Nk) s_sc[(size_t)g * P + j0] = c0 * scale;
        if (j0 + 1 < Nk) s_sc[(size_t)g * P + j0 + 1] = c1 * scale;
      }
    }
  }
  __syncthreads();
  if (warp >= nrows) return;
  uint8_t* mrow = mask + ((size_t)bh * Nq + i0 + warp) * Nk;
  double* sc = s_sc + (size_t)warp * P;
  double smax = -1.0 / 0.0;
#pragma unroll
  for (int q = 0; q < E * R; ++q) {                          // key j = 32 q + lane (conflict-free, and an interleaved sample of the row)
    const int jj = 32 * q + lane;
    if (jj < Nk) smax = fmax(smax, sc[jj]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
  // Selection instead of a full sort of the row (round 2: 55 bitonic stages, two thirds of the kernel's instructions).  The cut is
  // the LARGEST key c with  sum_{k >= c} w_k >= p Z  and  #{k >= c} >= kmin  (Eq. 3 + min-kc: the same prefix as "sort, then first
  // cum >= p Z"; keys are unique, so "k >= c" is the sorted prefix that ends at c).  Each lane sorts its own keys in runs of E
  // (registers, no shuffles) and parks them in shared memory -- in place: slot 32 q + lane held the score of the key the lane read
  // from it; then a quickselect on the key VALUE: the pivot is the middle key of the longest still-undecided run (a lane's keys
  // are an interleaved sample of the row, so it splits every run about in half), every lane counts its keys >= pivot by binary
  // search and adds the weights of the keys that moved, and the warp decides.  ~12-15 rounds of ~90 instructions.  The sums are
  // associated differently from a sequential cumulative sum (R-K3's 1e-9 Z exemption covers that, as it did the scan's).
  unsigned long long* skey = reinterpret_cast<unsigned long long*>(sc);
  double run = 0.0;
#pragma unroll
  for (int u = 0; u < R; ++u) {
    WarpSort<E> ws;
#pragma unroll
    for (int i = 0; i < E; ++i) {                            // w_j = s^k_j exp(S_j - max); pads get the smallest keys of all (0, j >= N_k)
      const int jj = 32 * (u * E + i) + lane;
      ws.k[i] = jj < Nk ? mask_key((double)sizes_k[(size_t)bh * Nk + jj] * exp(sc[jj] - smax), jj) : (unsigned long long)(2047 - jj);
    }
    ws.sort_lane();
#pragma unroll
    for (int i = 0; i < E; ++i) { run += mask_key_w(ws.k[i]); skey[(u * E + i) * 32 + lane] = ws.k[i]; }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) run += __shfl_xor_sync(0xffffffffu, run, o);   // same bits in every lane (commutative tree)
  const double thr = top_p * run;
  __syncwarp();
  const unsigned long long U0 = (unsigned long long)(2047 - Nk);   // below every real key, at or above every pad: "everything"
  unsigned long long U = U0;                                     // largest key known to satisfy the condition
  int a[R], b[R];                                                // run u: keys [0, a) are >= L (the smallest key known to fail), [a, b) undecided
#pragma unroll
  for (int u = 0; u < R; ++u) {                                  // the run's real keys come first
    a[u] = 0;
    const int first = 32 * u * E + lane;                         // j of the run's first slot
    b[u] = first < Nk ? min(E, (Nk - first + 31) >> 5) : 0;
  }
  double S_hi = 0.0;                                             // sum of the weights of all keys >= L
  int N_hi = 0;
  for (;;) {
    unsigned mine_len = 0;
#pragma unroll
    for (int u = 0; u < R; ++u) mine_len = max(mine_len, ((unsigned)(b[u] - a[u]) << 6) | ((unsigned)u << 5) | (unsigned)lane);
    const unsigned best = __reduce_max_sync(0xffffffffu, mine_len);
    if ((best >> 6) == 0) break;
    const int src = (int)(best & 31u), su = (int)((best >> 5) & 1u);
    unsigned long long mine = 0ull;
#pragma unroll
    for (int u = 0; u < R; ++u)
      if (u == su && b[u] > a[u]) mine = skey[(u * E + ((a[u] + b[u]) >> 1)) * 32 + lane];
    const unsigned long long pv = __shfl_sync(0xffffffffu, mine, src);
    int c[R], moved = 0;
    double sum = 0.0;
#pragma unroll
    for (int u = 0; u < R; ++u) {
      int lo = a[u], hi = b[u];                                  // c = number of this run's keys >= pv
#pragma unroll
      for (int it = 0; it < 6; ++it) {
        if (lo < hi) {
          const int mid = (lo + hi) >> 1;
          if (skey[(u * E + mid) * 32 + lane] >= pv) lo = mid + 1; else hi = mid;
        }
      }
      c[u] = lo;
      for (int idx = a[u]; idx < lo; ++idx) sum += mask_key_w(skey[(u * E + idx) * 32 + lane]);
      moved += lo - a[u];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    const int cn = __reduce_add_sync(0xffffffffu, moved);
    const double S = S_hi + sum;
    const int N = N_hi + cn;
    if (S >= thr && N >= kmin) {     // warp-uniform: S, N are the same bits in every lane
      U = pv;
#pragma unroll
      for (int u = 0; u < R; ++u) b[u] = c[u] - ((lane == src && u == su) ? 1 : 0);   // undecided: the keys above pv
    } else {
#pragma unroll
      for (int u = 0; u < R; ++u) a[u] = c[u];                   // pv fails and becomes L
      S_hi = S; N_hi = N;
    }
  }
#pragma unroll
  for (int q = 0; q < E * R; ++q) {
    const unsigned long long k = skey[q * 32 + lane];
    const int jj = mask_key_j(k);
    if (jj < Nk) mrow[jj] = k >= U ? 1 : 0;
  }
}

template <int D, int E, int R>
int launch_mask_warp(int BH, int Nq, int Nk, const float* mu_q, const float* mu_k, const int* sizes_k, double scale, double top_p,
                     int kmin, uint8_t* mask, cudaStream_t st) {
  const size_t smem = (size_t)kWarpRows * D * 8 + (size_t)kWarpRows * 32 * E * R * 8;
  if (cudaFuncSetAttribute(hva_mask_warp_kernel<D, E, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return HVA_ECUDA;
  hva_mask_warp_kernel<D, E, R><<<dim3((Nq + kWarpRows - 1) / kWarpRows, BH), 256, smem, st>>>(Nq, Nk, mu_q, mu_k, sizes_k, scale, top_p, kmin, mask);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

}  // namespace

extern "C" int hva_build_mask(int32_t BH, int32_t Nq, int32_t Nk, int32_t D, const float* mu_q, const float* mu_k,
                              const int32_t* sizes_k, float scale, float top_p, float min_kc, uint8_t* mask, void* ws,
                              size_t ws_bytes, void* stream) {
  return hva_build_mask_ex(BH, Nq, Nk, D, mu_q, mu_k, sizes_k, scale, top_p, min_kc, mask, 0u, ws, ws_bytes, stream);
}

extern "C" int hva_build_mask_ex(int32_t BH, int32_t Nq, int32_t Nk, int32_t D, const float* mu_q, const float* mu_k,
                                 const int32_t* sizes_k, float scale, float top_p, float min_kc, uint8_t* mask, uint32_t flags,
                                 void* ws, size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  if (!mu_q || !mu_k || !sizes_k || !mask) return HVA_EINVAL;
  if (BH < 1 || Nq < 1 || Nk < 1 || (D != 64 && D != 128)) return HVA_EINVAL;
  if (!(top_p > 0.f) || min_kc < 0.f || min_kc > 1.f) return HVA_EINVAL;
  if (Nk > 2048) return HVA_EUNSUPPORTED;
  int P = kMaskThreads;
  while (P < Nk) P <<= 1;
  int kmin = (int)ceil((double)min_kc * (double)Nk);
  size_t smem = (size_t)P * 12 + (size_t)kRowsPerCta * Nk * 8 + (size_t)kRowsPerCta * D * 8 + kMaskThreads * 8 + 16;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (top_p < 1.f && !(flags & HVA_FLAG_MASK_BLOCKSORT)) {   // warp per row: selection on lane-sorted runs (N_k <= 2048 here)
#define HVA_MASK_WARP(DD)                                                                                                             \
    do {                                                                                                                              \
      if (Nk <= 256) return launch_mask_warp<DD, 8, 1>(BH, Nq, Nk, mu_q, mu_k, sizes_k, (double)scale, (double)top_p, kmin, mask, st);  \
      if (Nk <= 512) return launch_mask_warp<DD, 16, 1>(BH, Nq, Nk, mu_q, mu_k, sizes_k, (double)scale, (double)top_p, kmin, mask, st); \
      if (Nk <= 1024) return launch_mask_warp<DD, 32, 1>(BH, Nq, Nk, mu_q, mu_k, sizes_k, (double)scale, (double)top_p, kmin, mask, st); \
      return launch_mask_warp<DD, 32, 2>(BH, Nq, Nk, mu_q, mu_k, sizes_k, (double)scale, (double)top_p, kmin, mask, st);             \
    } while (0)
    if (D == 64) HVA_MASK_WARP(64);
    HVA_MASK_WARP(128);
#undef HVA_MASK_WARP
  }
  dim3 grid((Nq + kRowsPerCta - 1) / kRowsPerCta, BH);
  if (smem > 48 * 1024) {
    cudaFuncSetAttribute(hva_mask_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(hva_mask_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  if (D == 64)
    hva_mask_kernel<64><<<grid, kMaskThreads, smem, st>>>(Nq, Nk, P, mu_q, mu_k, sizes_k, (double)scale, (double)top_p,
                                                          top_p >= 1.f, kmin, mask);
  else
    hva_mask_kernel<128><<<grid, kMaskThreads, smem, st>>>(Nq, Nk, P, mu_q, mu_k, sizes_k, (double)scale, (double)top_p,
                                                           top_p >= 1.f, kmin, mask);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
