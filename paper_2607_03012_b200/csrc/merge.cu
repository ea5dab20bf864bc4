// S6: hardware-aware cluster merging (Eq. 7-10 l.111-125, Alg. 1 l.131-168).
//
// One CTA (32 warps) per (batch, head); all state is integer.  Costs are kept in tile units
// c(S) = ceil(s^q(S)/tau_q) * ceil(kappa(S)/tau_k) (Eq. 8 / (tau_q tau_k)).  Per round:
//   1. side(g) from the counter-based hash of include/hva.h (Alg. 1 line 6),
//   2. warp-parallel pairwise-cost pass: one warp per A in side 1 walks every B in side 0 in
//      ascending gid; lanes split the chi bit-words and add the key sizes of B \ A
//      (kappa(A u B) = kappa(A) + sum_{j in B\A} s^k_j, lines 9-12); only pairs with dC < 0 can be
//      accepted (l.127), so pairs that save no row tile (dC >= 0, DESIGN.md R-M6) or whose lower
//      bound is already >= 0 are pruned exactly; best B by (dC, gid) (line 13),
//   3. per-B conflict resolution with a 64-bit atomicMin on (dC, gid(A)) (line 14; order-free),
//   4. accepted pairs are applied in parallel (lines 15-16): gid = min, s^q = sum, chi = OR.
#include "common.cuh"

namespace {

constexpr int kMergeThreads = 1024;
constexpr unsigned long long kNoProp = ~0ull;

__host__ __device__ __forceinline__ uint32_t hva_side_hash(uint32_t seed, uint32_t bh, uint32_t rnd, uint32_t gid) {
  uint32_t h = (seed * 0x9E3779B1u) ^ (bh * 0x85EBCA77u) ^ (rnd * 0xC2B2AE3Du) ^ (gid * 0x27D4EB2Fu);
  h ^= h >> 16; h *= 0x7FEB352Du; h ^= h >> 15; h *= 0x846CA68Bu; h ^= h >> 16;
  return h >> 31;
}

struct MergeParams {
  int Nq, Nk, Wd;
  const int* sizes_q; const int* sizes_k; const uint8_t* mask;
  int tile_q, tile_k, rounds, max_q_tiles; uint32_t seed;
  int* group_of; int* n_groups; uint8_t* group_mask;
  uint32_t* chi; int* sq; int* kap; int* alive; int* side; int* remap; unsigned long long* best;
};

__device__ __forceinline__ int cdiv(int a, int b) { return (a + b - 1) / b; }

__global__ void __launch_bounds__(kMergeThreads) hva_merge_kernel(MergeParams p) {
  const int bh = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int Nq = p.Nq, Nk = p.Nk, Wd = p.Wd;
  extern __shared__ int s_sk[];  // [Wd*32] key cluster sizes (zero padded)
  uint32_t* chi = p.chi + (size_t)bh * Nq * Wd;
  int* sq = p.sq + (size_t)bh * Nq; int* kap = p.kap + (size_t)bh * Nq; int* alive = p.alive + (size_t)bh * Nq;
  int* side = p.side + (size_t)bh * Nq; int* remap = p.remap + (size_t)bh * Nq;
  unsigned long long* best = p.best + (size_t)bh * Nq;
  int* group_of = p.group_of + (size_t)bh * Nq;
  const uint8_t* mask = p.mask + (size_t)bh * Nq * Nk;

  for (int j = tid; j < Wd * 32; j += kMergeThreads) s_sk[j] = j < Nk ? p.sizes_k[(size_t)bh * Nk + j] : 0;
  __syncthreads();
  // Alg. 1 lines 3-4: singleton groups, chi_j({i}) = m_ij (bit-packed); kappa({i})
  for (int i = warp; i < Nq; i += kMergeThreads / 32) {
    int k = 0;
    for (int w = lane; w < Wd; w += 32) {
      uint32_t bits = 0;
      for (int b = 0; b < 32; ++b) {
        int j = w * 32 + b;
        if (j < Nk && mask[(size_t)i * Nk + j]) { bits |= 1u << b; k += s_sk[j]; }
      }
      chi[(size_t)i * Wd + w] = bits;
    }
    for (int o = 16; o > 0; o >>= 1) k += __shfl_xor_sync(0xffffffffu, k, o);
    if (lane == 0) {
      int s = p.sizes_q[(size_t)bh * Nq + i];
      sq[i] = s; kap[i] = k; alive[i] = s > 0; group_of[i] = i; remap[i] = -1;
    }
  }
  __syncthreads();

  for (int r = 1; r <= p.rounds; ++r) {
    for (int g = tid; g < Nq; g += kMergeThreads) {
      side[g] = alive[g] ? (int)hva_side_hash(p.seed, (uint32_t)bh, (uint32_t)r, (uint32_t)g) : -1;
      best[g] = kNoProp;
    }
    __syncthreads();
    for (int A = warp; A < Nq; A += kMergeThreads / 32) {
      if (side[A] != 1) continue;
      const int sA = sq[A], kA = kap[A], rA = cdiv(sA, p.tile_q), cA = rA * cdiv(kA, p.tile_k);
      uint32_t a0 = lane < Wd ? chi[(size_t)A * Wd + lane] : 0u;
      uint32_t a1 = lane + 32 < Wd ? chi[(size_t)A * Wd + lane + 32] : 0u;
      int best_dc = 0, best_B = -1;
      for (int B = 0; B < Nq; ++B) {
        if (side[B] != 0) continue;
        const int sB = sq[B], kB = kap[B], rB = cdiv(sB, p.tile_q), cB = rB * cdiv(kB, p.tile_k);
        const int rU = cdiv(sA + sB, p.tile_q);
        if (p.max_q_tiles > 0 && rU > p.max_q_tiles) continue;
        if (rU >= rA + rB) continue;                                      // no row tile saved => dC >= 0 (R-M6)
        const int kLow = kA > kB ? kA : kB;
        if (rU * cdiv(kLow, p.tile_k) - cA - cB >= best_dc) continue;     // lower bound cannot beat current best
        int add = 0;
        uint32_t b0 = lane < Wd ? chi[(size_t)B * Wd + lane] & ~a0 : 0u;
        uint32_t b1 = lane + 32 < Wd ? chi[(size_t)B * Wd + lane + 32] & ~a1 : 0u;
        while (b0) { int b = __ffs(b0) - 1; b0 &= b0 - 1; add += s_sk[lane * 32 + b]; }
        while (b1) { int b = __ffs(b1) - 1; b1 &= b1 - 1; add += s_sk[(lane + 32) * 32 + b]; }
        for (int o = 16; o > 0; o >>= 1) add += __shfl_xor_sync(0xffffffffu, add, o);
        const int dc = rU * cdiv(kA + add, p.tile_k) - cA - cB;           // Eq. 10 in tile units
        if (dc < best_dc) { best_dc = dc; best_B = B; }                   // strict: ties -> lower gid(B)
      }
      if (lane == 0 && best_B >= 0) {
        unsigned long long key = ((unsigned long long)(uint32_t)(best_dc + 0x40000000) << 32) | (uint32_t)A;
        atomicMin(&best[best_B], key);                                    // ties -> lower gid(A)
      }
    }
    __syncthreads();
    for (int B = tid; B < Nq; B += kMergeThreads) {
      unsigned long long key = best[B];
      if (key == kNoProp) continue;
      int A = (int)(uint32_t)(key & 0xffffffffu);
      int g = A < B ? A : B, o = A < B ? B : A;
      int k = 0;
      for (int w = 0; w < Wd; ++w) {
        uint32_t bits = chi[(size_t)g * Wd + w] | chi[(size_t)o * Wd + w];
        chi[(size_t)g * Wd + w] = bits;
        while (bits) { int b = __ffs(bits) - 1; bits &= bits - 1; k += s_sk[w * 32 + b]; }
      }
      sq[g] = sq[A] + sq[B]; kap[g] = k; alive[o] = 0; remap[o] = g;
    }
    __syncthreads();
    for (int i = tid; i < Nq; i += kMergeThreads) {
      int m = remap[group_of[i]];
      if (m >= 0) group_of[i] = m;
    }
    __syncthreads();
    for (int i = tid; i < Nq; i += kMergeThreads) remap[i] = -1;
    __syncthreads();
  }
  // outputs: n_groups, chi rows of the active groups in ascending gid order
  __shared__ int s_ng;
  if (tid == 0) {
    int c = 0;
    for (int g = 0; g < Nq; ++g) if (alive[g]) side[c++] = g;   // reuse side[] as the ascending gid list
    s_ng = c; p.n_groups[bh] = c;
  }
  __syncthreads();
  uint8_t* gm = p.group_mask + (size_t)bh * Nq * Nk;
  for (size_t e = tid; e < (size_t)Nq * Nk; e += kMergeThreads) {
    int row = (int)(e / Nk), j = (int)(e % Nk);
    uint8_t v = 0;
    if (row < s_ng) v = (chi[(size_t)side[row] * Wd + (j >> 5)] >> (j & 31)) & 1u;
    gm[e] = v;
  }
}

}  // namespace

size_t hva_merge_ws_bytes(int BH, int Nq, int Nk) {
  size_t Wd = (Nk + 31) / 32;
  return hva_align((size_t)BH * Nq * Wd * 4) + 5 * hva_align((size_t)BH * Nq * 4) + hva_align((size_t)BH * Nq * 8);
}

extern "C" int hva_merge(int32_t BH, int32_t Nq, int32_t Nk, const int32_t* sizes_q, const int32_t* sizes_k,
                         const uint8_t* mask, int32_t tile_q, int32_t tile_k, int32_t rounds, int32_t max_q_tiles,
                         uint32_t seed, int32_t* group_of_cluster, int32_t* n_groups, uint8_t* group_mask, void* ws,
                         size_t ws_bytes, void* stream) {
  if (!sizes_q || !sizes_k || !mask || !group_of_cluster || !n_groups || !group_mask || !ws) return HVA_EINVAL;
  if (BH < 1 || Nq < 1 || Nk < 1 || tile_q < 1 || tile_k < 1 || rounds < 0 || max_q_tiles < 0) return HVA_EINVAL;
  if (Nk > 2048 || Nq > 65535) return HVA_EUNSUPPORTED;
  if (ws_bytes < hva_merge_ws_bytes(BH, Nq, Nk)) return HVA_EWORKSPACE;
  MergeParams p;
  p.Nq = Nq; p.Nk = Nk; p.Wd = (Nk + 31) / 32;
  p.sizes_q = sizes_q; p.sizes_k = sizes_k; p.mask = mask;
  p.tile_q = tile_q; p.tile_k = tile_k; p.rounds = rounds; p.max_q_tiles = max_q_tiles; p.seed = seed;
  p.group_of = group_of_cluster; p.n_groups = n_groups; p.group_mask = group_mask;
  char* w = reinterpret_cast<char*>(ws);
  size_t a4 = hva_align((size_t)BH * Nq * 4);
  p.chi = reinterpret_cast<uint32_t*>(w); w += hva_align((size_t)BH * Nq * p.Wd * 4);
  p.sq = reinterpret_cast<int*>(w); w += a4;
  p.kap = reinterpret_cast<int*>(w); w += a4;
  p.alive = reinterpret_cast<int*>(w); w += a4;
  p.side = reinterpret_cast<int*>(w); w += a4;
  p.remap = reinterpret_cast<int*>(w); w += a4;
  p.best = reinterpret_cast<unsigned long long*>(w);
  hva_merge_kernel<<<BH, kMergeThreads, (size_t)p.Wd * 32 * sizeof(int), reinterpret_cast<cudaStream_t>(stream)>>>(p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
