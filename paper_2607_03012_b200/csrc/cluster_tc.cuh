// Interface between cluster.cu (iteration driver, centroid update) and cluster_tc.cu (tensor-pipe assignment).
#pragma once
#include "common.cuh"
#include <cuda.h>

struct HvaAssignTc {
  CUtensorMap map_x, map_hi, map_lo;
  int npad, rows_a, csplit, ct;
  int NT, NB, NW, NS;  // token buffers, centroid buffers, scan warpgroups, pipeline slots of the persistent CTA
  int cols;            // TMEM columns per token slot
  size_t smem;
  int one_pass;        // one MMA pass over the stacked [hi; lo] centroid tile
  int coop;            // wide windows (shared memory holds one one-hot tile): the three scan groups share every tile's candidates
  int grid;            // one persistent CTA per SM
  bool probe;          // prepared for the instrumented instantiation (hva_cluster_ex with a probe buffer)
};

// time slices of a cell per CTA tile (<= 128 token rows): a cell of more than 128 tokens is split along t
static inline int hva_assign_tc_slices(const HvaGrid& g) {
  const int per = g.kh * g.kw;
  int ct = per > 0 ? 128 / per : 1;
  if (ct < 1) ct = 1;
  return ct < g.kt ? ct : g.kt;
}
static inline int hva_assign_tc_csplit(const HvaGrid& g) {
  if (g.kh * g.kw > 128) return 1;   // not a tensor-pipe shape: the CUDA-core kernel takes whole cells
  const int ct = hva_assign_tc_slices(g);
  return (g.kt + ct - 1) / ct;
}

// bf16, D = 128, k_h k_w <= 128 (a tile of whole time slices fits 128 rows), window of at most 256 centroids
bool hva_assign_tc_supported(const HvaGrid& g, int D, int dtype);
// X[BH,T,H,W,128] bf16; mu_hi / mu_lo [BH,Kt,Kh,Kw,128] bf16 (two-term split of the fp32 centroids)
int hva_assign_tc_prepare(const HvaGrid& g, int BH, const void* X, const void* mu_hi, const void* mu_lo, bool probe, HvaAssignTc* out);
int hva_assign_tc_launch(const HvaAssignTc& a, const HvaGrid& g, int BH, const float* mu, const float* musq, float* part,
                         int* part_cnt, int* assign, float* lowe, float* xsq, int xsq_mode, int* counter, float* probe, cudaStream_t st);

// Window-less variant for the hybrid subset step (hybrid_tc.cu): subset tokens against ALL centroids.
bool hva_subset_tc_supported(int D, int dtype, int Nc);
int hva_subset_assign_tc_launch(int BH, int n, int Nc, int m, const void* X, const int* subset, const float* mu, const void* mu_hi,
                                const void* mu_lo, const float* musq, const int* assign, int* oldlab, int* newlab, cudaStream_t st);
// two-term bf16 split + |mu|^2 of fp32 centroids [BH, Nc, D] (cluster.cu)
int hva_mu_split_launch(int BH, int Nc, int D, const float* mu, void* mu_hi, void* mu_lo, float* musq, cudaStream_t st);

#ifdef __CUDACC__
namespace hva_tc_dev {
// |tensor-pipe dot - exact dot| <= kEpsDot |x| |mu|: split error 2^-18 plus fp32 accumulation of 256 exact
// products.  Observed on B200 (hva_cluster_ex probe, tests/test_gpu_parity.py): score error 4.6e-6 |x||mu| including the
// rounding of the fp32 direct form it is compared with, against the 2 kEpsDot = 6.1e-5 assumed: 13x head room.
constexpr float kEpsDot = 1.0f / 32768.0f;

// 16-byte chunk q (0..15) of token row r in the swizzled A tile
__device__ __forceinline__ const uint4* x_chunk(const unsigned char* sA, int half_bytes, int r, int q) {
  return reinterpret_cast<const uint4*>(sA + (q >> 3) * half_bytes + r * 128 + (((q & 7) ^ (r & 7)) << 4));
}
__device__ __forceinline__ void unpack8(const uint4& r, float x[8]) {   // bf16 -> fp32 is a 16-bit shift (exact)
  x[0] = __uint_as_float(r.x << 16); x[1] = __uint_as_float(r.x & 0xffff0000u);
  x[2] = __uint_as_float(r.y << 16); x[3] = __uint_as_float(r.y & 0xffff0000u);
  x[4] = __uint_as_float(r.z << 16); x[5] = __uint_as_float(r.z & 0xffff0000u);
  x[6] = __uint_as_float(r.w << 16); x[7] = __uint_as_float(r.w & 0xffff0000u);
}

// The exact direct form sum_c (x_c - mu_c)^2 in fp32 (Eq. 5) with a FIXED summation order shared by every kernel that decides
// a label (this file's users and the CUDA-core kernel of cluster.cu): D/4 partial sums over 4 consecutive dims each
// (p = d0*d0; p = fma(d_k, d_k, p), k = 1..3), combined by the halving tree  p_j += p_{j + o},  o = D/8, D/16, ..., 1.
// One 128-long dependent fma chain cost a refining lane ~6 K clk per candidate (and stalled the whole tile pipeline behind it);
// the D/4 chains are independent.
__device__ __forceinline__ float hva_sq4(float x0, float x1, float x2, float x3, const float4& m) {
  float d = x0 - m.x, p = d * d;
  d = x1 - m.y; p = fmaf(d, d, p);
  d = x2 - m.z; p = fmaf(d, d, p);
  d = x3 - m.w; p = fmaf(d, d, p);
  return p;
}
template <int N>
__device__ __forceinline__ float hva_tree_sum(float (&p)[N]) {
#pragma unroll
  for (int o = N / 2; o >= 1; o >>= 1) {
#pragma unroll
    for (int j = 0; j < o; ++j) p[j] += p[j + o];
  }
  return p[0];
}
__device__ __forceinline__ float direct_dist(const unsigned char* sA, int half_bytes, int r, const float* __restrict__ mu) {
  float pr[32];
#pragma unroll
  for (int q = 0; q < 16; ++q) {
    float x[8];
    unpack8(*x_chunk(sA, half_bytes, r, q), x);
    const float4 m0 = __ldg(reinterpret_cast<const float4*>(mu) + 2 * q);
    const float4 m1 = __ldg(reinterpret_cast<const float4*>(mu) + 2 * q + 1);
    pr[2 * q] = hva_sq4(x[0], x[1], x[2], x[3], m0);
    pr[2 * q + 1] = hva_sq4(x[4], x[5], x[6], x[7], m1);
  }
  return hva_tree_sum(pr);
}

}  // namespace hva_tc_dev
#endif
