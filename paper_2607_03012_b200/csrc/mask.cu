// S5: centroid scores, size-weighted softmax and row-wise top-p (Eq. 2-3, l.47-54;
// "Top-p" / "Min-kc" l.332-334).  One CTA per (bh, query cluster) row.  Scores and weights are
// evaluated in fp64 from the fp32 centroids so that the cut decision matches the fp64 oracle
// (DESIGN.md R-K3): w_j = s^k_j exp(S_j - max_j S_j); sort by (w desc, j asc) with an in-smem
// bitonic network; inclusive scan; k = first position with cum >= top_p * Z; keep at least kmin.
#include "common.cuh"

namespace {

constexpr int kMaskThreads = 256;

__device__ __forceinline__ bool before(double wa, int ja, double wb, int jb) {
  return wa > wb || (wa == wb && ja < jb);  // descending weight, ties -> lower j
}

template <int D>
__global__ void __launch_bounds__(kMaskThreads) hva_mask_kernel(int Nq, int Nk, int P, const float* __restrict__ mu_q,
                                                                const float* __restrict__ mu_k,
                                                                const int* __restrict__ sizes_k, double scale,
                                                                double top_p, int all_ones, int kmin,
                                                                uint8_t* __restrict__ mask) {
  const int i = blockIdx.x, bh = blockIdx.y, tid = threadIdx.x;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* s_w = reinterpret_cast<double*>(smem_raw);  // [P]
  int* s_j = reinterpret_cast<int*>(s_w + P);         // [P]
  double* s_q = reinterpret_cast<double*>(s_j + P);   // [D]
  double* s_red = s_q + D;                            // [kMaskThreads]
  __shared__ int s_k;

  uint8_t* mrow = mask + ((size_t)bh * Nq + i) * Nk;
  if (all_ones) {  // top_p >= 1 selects every key cluster (R-K1)
    for (int j = tid; j < Nk; j += kMaskThreads) mrow[j] = 1;
    return;
  }
  for (int c = tid; c < D; c += kMaskThreads) s_q[c] = (double)mu_q[((size_t)bh * Nq + i) * D + c];
  __syncthreads();
  // S_ij = <mu^q_i, mu^k_j> * scale   (Eq. 2)
  double lmax = -1.0 / 0.0;
  for (int j = tid; j < P; j += kMaskThreads) {
    double sc = -1.0 / 0.0;
    if (j < Nk) {
      const float4* kr = reinterpret_cast<const float4*>(mu_k + ((size_t)bh * Nk + j) * D);
      double a = 0.0;
#pragma unroll 4
      for (int c = 0; c < D / 4; ++c) {
        float4 v = __ldg(kr + c);
        a = fma((double)v.x, s_q[4 * c + 0], a);
        a = fma((double)v.y, s_q[4 * c + 1], a);
        a = fma((double)v.z, s_q[4 * c + 2], a);
        a = fma((double)v.w, s_q[4 * c + 3], a);
      }
      sc = a * scale;
    }
    s_w[j] = sc;
    s_j[j] = j;
    lmax = fmax(lmax, sc);
  }
  s_red[tid] = lmax;
  __syncthreads();
  for (int o = kMaskThreads / 2; o > 0; o >>= 1) {
    if (tid < o) s_red[tid] = fmax(s_red[tid], s_red[tid + o]);
    __syncthreads();
  }
  const double smax = s_red[0];
  __syncthreads();
  for (int j = tid; j < P; j += kMaskThreads)
    s_w[j] = (j < Nk) ? (double)sizes_k[(size_t)bh * Nk + j] * exp(s_w[j] - smax) : -1.0;  // pads sort last
  __syncthreads();
  // bitonic sort, order `before`
  for (int k = 2; k <= P; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int a = tid; a < P; a += kMaskThreads) {
        int b = a ^ j;
        if (b > a) {
          double wa = s_w[a], wb = s_w[b];
          int ja = s_j[a], jb = s_j[b];
          bool up = ((a & k) == 0);
          bool swap = up ? before(wb, jb, wa, ja) : before(wa, ja, wb, jb);
          if (swap) { s_w[a] = wb; s_w[b] = wa; s_j[a] = jb; s_j[b] = ja; }
        }
      }
      __syncthreads();
    }
  }
  // inclusive scan of the sorted weights: per-thread contiguous chunk, then scan of chunk sums
  const int chunk = P / kMaskThreads > 0 ? P / kMaskThreads : 1;
  const int lo = tid * chunk;
  double run = 0.0;
  if (lo < P)
    for (int r = lo; r < lo + chunk; ++r) run += (r < Nk ? s_w[r] : 0.0);
  s_red[tid] = run;
  __syncthreads();
  if (tid == 0) {  // sequential exclusive scan of <= 256 chunk sums (ascending: mirrors a cumulative sum)
    double a = 0.0;
    for (int t = 0; t < kMaskThreads; ++t) { double v = s_red[t]; s_red[t] = a; a += v; }
    s_k = Nk;
  }
  __syncthreads();
  double Z = s_red[kMaskThreads - 1];
  {  // Z = total = exclusive prefix of last chunk + its sum (recomputed in the same order)
    int l2 = (kMaskThreads - 1) * chunk;
    double a = s_red[kMaskThreads - 1];
    if (l2 < P)
      for (int r = l2; r < l2 + chunk; ++r) a += (r < Nk ? s_w[r] : 0.0);
    Z = a;
  }
  const double thr = top_p * Z;
  if (lo < P) {
    double a = s_red[tid];
    for (int r = lo; r < lo + chunk && r < Nk; ++r) {
      a += s_w[r];
      if (a >= thr) { atomicMin(&s_k, r + 1); break; }   // smallest k with cum_k >= p Z   (Eq. 3)
    }
  }
  __syncthreads();
  int k = s_k < kmin ? kmin : s_k;
  for (int r = tid; r < P; r += kMaskThreads) {
    int j = s_j[r];
    if (r < Nk) mrow[j] = (r < k) ? 1 : 0;
  }
}

}  // namespace

extern "C" int hva_build_mask(int32_t BH, int32_t Nq, int32_t Nk, int32_t D, const float* mu_q, const float* mu_k,
                              const int32_t* sizes_k, float scale, float top_p, float min_kc, uint8_t* mask, void* ws,
                              size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  if (!mu_q || !mu_k || !sizes_k || !mask) return HVA_EINVAL;
  if (BH < 1 || Nq < 1 || Nk < 1 || (D != 64 && D != 128)) return HVA_EINVAL;
  if (!(top_p > 0.f) || min_kc < 0.f || min_kc > 1.f) return HVA_EINVAL;
  if (Nk > 2048) return HVA_EUNSUPPORTED;
  int P = kMaskThreads;
  while (P < Nk) P <<= 1;
  int kmin = (int)ceil((double)min_kc * (double)Nk);
  size_t smem = (size_t)P * 12 + (size_t)D * 8 + kMaskThreads * 8;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  dim3 grid(Nq, BH);
  if (D == 64)
    hva_mask_kernel<64><<<grid, kMaskThreads, smem, st>>>(Nq, Nk, P, mu_q, mu_k, sizes_k, (double)scale, (double)top_p,
                                                          top_p >= 1.f, kmin, mask);
  else
    hva_mask_kernel<128><<<grid, kMaskThreads, smem, st>>>(Nq, Nk, P, mu_q, mu_k, sizes_k, (double)scale, (double)top_p,
                                                           top_p >= 1.f, kmin, mask);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
