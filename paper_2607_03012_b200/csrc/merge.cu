// S6: hardware-aware cluster merging (Eq. 7-10 l.111-125, Alg. 1 l.131-168).
//
// All state is integer and lives in the workspace; one launch per phase.  Costs are kept in tile units
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
#include <cstdlib>

namespace {

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
  int bh0;   // index of this call's first (batch, head) in the whole problem: the bipartition hash is keyed by the global bh
  int* group_of; int* n_groups; uint8_t* group_mask;
  uint32_t* chi; int* sq; int* kap; int* alive; int* side; int* remap; unsigned long long* best;
};

__device__ __forceinline__ int cdiv(int a, int b) { return (a + b - 1) / b; }

// Alg. 1 lines 3-4: singleton groups, chi_j({i}) = m_ij (bit-packed by ballot), kappa({i}).  One warp per cluster.
__global__ void __launch_bounds__(256) hva_merge_init_kernel(MergeParams p) {
  const int bh = blockIdx.y, lane = threadIdx.x & 31, i = blockIdx.x * 8 + (threadIdx.x >> 5);
  if (i >= p.Nq) return;
  const uint8_t* mrow = p.mask + ((size_t)bh * p.Nq + i) * p.Nk;
  const int* sk = p.sizes_k + (size_t)bh * p.Nk;
  int k = 0;
  for (int w = 0; w < p.Wd; ++w) {
    int j = w * 32 + lane;
    bool bit = j < p.Nk && mrow[j];
    unsigned bits = __ballot_sync(0xffffffffu, bit);
    if (bit) k += sk[j];
    if (lane == 0) p.chi[((size_t)bh * p.Nq + i) * p.Wd + w] = bits;
  }
  for (int o = 16; o > 0; o >>= 1) k += __shfl_xor_sync(0xffffffffu, k, o);
  if (lane == 0) {
    size_t e = (size_t)bh * p.Nq + i;
    int s = p.sizes_q[e];
    p.sq[e] = s; p.kap[e] = k; p.alive[e] = s > 0; p.group_of[e] = i; p.remap[e] = -1; p.best[e] = kNoProp;
  }
}

// Alg. 1 lines 6-13 for round r: one warp per A in side 1 (warp-parallel pairwise-cost pass).
__global__ void __launch_bounds__(256) hva_merge_propose_kernel(MergeParams p, int r) {
  const int bh = blockIdx.y, tid = threadIdx.x, lane = tid & 31, Nq = p.Nq, Wd = p.Wd;
  extern __shared__ int s_mem[];
  int* s_sk = s_mem;                 // [Wd*32] key cluster sizes, zero padded
  int* s_sq = s_sk + Wd * 32;        // [Nq] s^q(B) for B in side 0, else 0 (0 => skip)
  int* s_kap = s_sq + Nq;            // [Nq]
  const uint32_t* chi = p.chi + (size_t)bh * Nq * Wd;
  const size_t e0 = (size_t)bh * Nq;
  for (int j = tid; j < Wd * 32; j += 256) s_sk[j] = j < p.Nk ? p.sizes_k[(size_t)bh * p.Nk + j] : 0;
  for (int g = tid; g < Nq; g += 256) {
    bool isB = p.alive[e0 + g] && hva_side_hash(p.seed, (uint32_t)(p.bh0 + bh), (uint32_t)r, (uint32_t)g) == 0;
    s_sq[g] = isB ? p.sq[e0 + g] : 0;
    s_kap[g] = p.kap[e0 + g];
  }
  __syncthreads();
  const int A = blockIdx.x * 8 + (tid >> 5);
  if (A >= Nq || !p.alive[e0 + A] || hva_side_hash(p.seed, (uint32_t)(p.bh0 + bh), (uint32_t)r, (uint32_t)A) != 1) return;
  const int sA = p.sq[e0 + A], kA = p.kap[e0 + A], rA = cdiv(sA, p.tile_q), cA = rA * cdiv(kA, p.tile_k);
  const uint32_t a0 = lane < Wd ? ~chi[(size_t)A * Wd + lane] : 0u;
  const uint32_t a1 = lane + 32 < Wd ? ~chi[(size_t)A * Wd + lane + 32] : 0u;
  int best_dc = 0, best_B = -1;
  for (int B = 0; B < Nq; ++B) {
    const int sB = s_sq[B];
    if (sB == 0) continue;
    const int kB = s_kap[B], rB = cdiv(sB, p.tile_q), cB = rB * cdiv(kB, p.tile_k);
    const int rU = cdiv(sA + sB, p.tile_q);
    if (p.max_q_tiles > 0 && rU > p.max_q_tiles) continue;
    if (rU >= rA + rB) continue;                                      // no row tile saved => dC >= 0 (R-M6)
    const int kLow = kA > kB ? kA : kB;
    if (rU * cdiv(kLow, p.tile_k) - cA - cB >= best_dc) continue;     // lower bound cannot beat the current best
    int add = 0;                                                      // sum of s^k over B \ A
    uint32_t b0 = lane < Wd ? chi[(size_t)B * Wd + lane] & a0 : 0u;
    uint32_t b1 = lane + 32 < Wd ? chi[(size_t)B * Wd + lane + 32] & a1 : 0u;
    while (b0) { int b = __ffs(b0) - 1; b0 &= b0 - 1; add += s_sk[lane * 32 + b]; }
    while (b1) { int b = __ffs(b1) - 1; b1 &= b1 - 1; add += s_sk[(lane + 32) * 32 + b]; }
    for (int o = 16; o > 0; o >>= 1) add += __shfl_xor_sync(0xffffffffu, add, o);
    const int dc = rU * cdiv(kA + add, p.tile_k) - cA - cB;           // Eq. 10 in tile units
    if (dc < best_dc) { best_dc = dc; best_B = B; }                   // strict: ties -> lower gid(B)
  }
  if (lane == 0 && best_B >= 0) {
    unsigned long long key = ((unsigned long long)(uint32_t)(best_dc + 0x40000000) << 32) | (uint32_t)A;
    atomicMin(&p.best[e0 + best_B], key);                             // line 14: best A per B, ties -> lower gid(A)
  }
}

// Alg. 1 lines 6-13 for round r with the pairwise overlaps I[A][B] precomputed on the tensor pipe (merge_tc.cu):
// kappa(A u B) = kappa(A) + kappa(B) - I[A][B].  One warp per A in side 1, lanes over B (coalesced row of I); the warp's
// best (dC, gid(B)) is the lexicographic minimum == first minimum in ascending gid(B) with strict '<' (line 13).
// The round's bipartition as two compact lists (Alg. 1 line 6): alive groups of side 1 ascending from the front of list[bh], alive
// groups of side 0 ascending at its end; cnt[bh] = (nA, nB).  One CTA per (b, head), two groups per thread (N_q <= 2048).
__global__ void __launch_bounds__(1024) hva_merge_sides_kernel(MergeParams p, int r, int* __restrict__ list, int* __restrict__ cnt) {
  const int bh = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, Nq = p.Nq;
  const size_t e0 = (size_t)bh * Nq;
  __shared__ int s_a[32], s_b[32];
  int fa[2], fb[2];
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    const int g = 2 * tid + e;
    const bool al = g < Nq && p.alive[e0 + g];
    const uint32_t sd = hva_side_hash(p.seed, (uint32_t)(p.bh0 + bh), (uint32_t)r, (uint32_t)g);
    fa[e] = al && sd == 1; fb[e] = al && sd == 0;
  }
  int ia = fa[0] + fa[1], ib = fb[0] + fb[1];        // inclusive warp scans, then the warps' totals
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int ya = __shfl_up_sync(0xffffffffu, ia, o), yb = __shfl_up_sync(0xffffffffu, ib, o);
    if (lane >= o) { ia += ya; ib += yb; }
  }
  if (lane == 31) { s_a[warp] = ia; s_b[warp] = ib; }
  __syncthreads();
  int oa = 0, ob = 0, ta = 0, tb = 0;
  for (int w = 0; w < 32; ++w) {
    if (w < warp) { oa += s_a[w]; ob += s_b[w]; }
    ta += s_a[w]; tb += s_b[w];
  }
  int pa = oa + ia - (fa[0] + fa[1]), pb = ob + ib - (fb[0] + fb[1]);   // exclusive positions of this thread's first group
  int* la = list + e0;
  int* lb = list + e0 + (Nq - tb);
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    const int g = 2 * tid + e;
    if (fa[e]) la[pa++] = g;
    if (fb[e]) lb[pb++] = g;
  }
  if (tid == 0) { cnt[2 * bh] = ta; cnt[2 * bh + 1] = tb; }
}

__global__ void __launch_bounds__(256) hva_merge_propose_inter_kernel(MergeParams p, int r, const int* __restrict__ inter, int Nqp,
                                                                      const int* __restrict__ list, const int* __restrict__ cnt) {
  const int bh = blockIdx.y, tid = threadIdx.x, lane = tid & 31, Nq = p.Nq;
  const size_t e0 = (size_t)bh * Nq;
  const int nA = cnt[2 * bh], nB = cnt[2 * bh + 1];
  const int i = blockIdx.x * 8 + (tid >> 5);           // i-th group of side 1
  if (i >= nA) return;
  const int A = list[e0 + i];
  const int* listB = list + e0 + (Nq - nB);
  const int sA = p.sq[e0 + A], kA = p.kap[e0 + A], rA = cdiv(sA, p.tile_q), cA = rA * cdiv(kA, p.tile_k);
  const int* row = inter + ((size_t)bh * Nqp + i) * Nqp;
  int best_dc = 0, best_B = 0x7fffffff;
  for (int j = lane; j < nB; j += 32) {
    const int B = listB[j];
    const int sB = p.sq[e0 + B], kB = p.kap[e0 + B], rB = cdiv(sB, p.tile_q), cB = rB * cdiv(kB, p.tile_k);
    const int rU = cdiv(sA + sB, p.tile_q);
    if (p.max_q_tiles > 0 && rU > p.max_q_tiles) continue;
    if (rU >= rA + rB) continue;                                      // no row tile saved => dC >= 0 (R-M6)
    const int dc = rU * cdiv(kA + kB - row[j], p.tile_k) - cA - cB;   // Eq. 10 in tile units
    if (dc < best_dc) { best_dc = dc; best_B = B; }                   // ascending B per lane: strict '<' keeps the lower gid
  }
  for (int o = 16; o > 0; o >>= 1) {
    const int odc = __shfl_xor_sync(0xffffffffu, best_dc, o), oB = __shfl_xor_sync(0xffffffffu, best_B, o);
    if (odc < best_dc || (odc == best_dc && oB < best_B)) { best_dc = odc; best_B = oB; }
  }
  if (lane == 0 && best_dc < 0) {
    unsigned long long key = ((unsigned long long)(uint32_t)(best_dc + 0x40000000) << 32) | (uint32_t)A;
    atomicMin(&p.best[e0 + best_B], key);                             // line 14: best A per B, ties -> lower gid(A)
  }
}

__global__ void __launch_bounds__(1024) hva_merge_apply_kernel(MergeParams p) {
  const int bh = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, Nq = p.Nq, Wd = p.Wd;
  uint32_t* chi = p.chi + (size_t)bh * Nq * Wd;
  const size_t e0 = (size_t)bh * Nq;
  const int* sk = p.sizes_k + (size_t)bh * p.Nk;
  for (int B = warp; B < Nq; B += 32) {
    unsigned long long key = p.best[e0 + B];
    if (key == kNoProp) continue;
    const int A = (int)(uint32_t)(key & 0xffffffffu);
    const int g = A < B ? A : B, o = A < B ? B : A;
    int k = 0;
    for (int w = lane; w < Wd; w += 32) {
      uint32_t bits = chi[(size_t)g * Wd + w] | chi[(size_t)o * Wd + w];
      chi[(size_t)g * Wd + w] = bits;
      while (bits) { int b = __ffs(bits) - 1; bits &= bits - 1; k += sk[w * 32 + b]; }
    }
    for (int x = 16; x > 0; x >>= 1) k += __shfl_xor_sync(0xffffffffu, k, x);
    if (lane == 0) {
      p.sq[e0 + g] = p.sq[e0 + A] + p.sq[e0 + B]; p.kap[e0 + g] = k; p.alive[e0 + o] = 0; p.remap[e0 + o] = g;
    }
  }
  __syncthreads();
  for (int i = tid; i < Nq; i += 1024) {
    int m = p.remap[e0 + p.group_of[e0 + i]];
    if (m >= 0) p.group_of[e0 + i] = m;
  }
  __syncthreads();
  for (int i = tid; i < Nq; i += 1024) { p.remap[e0 + i] = -1; p.best[e0 + i] = kNoProp; }
}

// n_groups and the chi rows of the active groups in ascending gid order.
__global__ void __launch_bounds__(1024) hva_merge_rank_kernel(MergeParams p) {
  const int bh = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, Nq = p.Nq;
  const size_t e0 = (size_t)bh * Nq;
  __shared__ int s_w[32];
  __shared__ int s_base;
  if (tid == 0) s_base = 0;
  __syncthreads();
  for (int g0 = 0; g0 < Nq; g0 += 1024) {
    int g = g0 + tid;
    bool al = g < Nq && p.alive[e0 + g];
    unsigned bal = __ballot_sync(0xffffffffu, al);
    if (lane == 0) s_w[warp] = __popc(bal);
    __syncthreads();
    int off = s_base;
    for (int w = 0; w < warp; ++w) off += s_w[w];
    if (al) p.side[e0 + off + __popc(bal & ((1u << lane) - 1))] = g;     // side[] reused: ascending active gids
    __syncthreads();
    if (tid == 0) { int t = 0; for (int w = 0; w < 32; ++w) t += s_w[w]; s_base += t; }
    __syncthreads();
  }
  if (tid == 0) p.n_groups[bh] = s_base;
}

__global__ void __launch_bounds__(256) hva_merge_out_kernel(MergeParams p) {
  const int bh = blockIdx.y, row = blockIdx.x, Nq = p.Nq, Nk = p.Nk, Wd = p.Wd;
  const int ng = p.n_groups[bh];
  uint8_t* out = p.group_mask + ((size_t)bh * Nq + row) * Nk;
  if (row >= ng) { for (int j = threadIdx.x; j < Nk; j += 256) out[j] = 0; return; }
  const uint32_t* c = p.chi + ((size_t)bh * Nq + p.side[(size_t)bh * Nq + row]) * Wd;
  for (int j = threadIdx.x; j < Nk; j += 256) out[j] = (c[j >> 5] >> (j & 31)) & 1u;
}

}  // namespace

// tensor-pipe overlap matrix (merge_tc.cu)
size_t hva_merge_inter_bytes(int BH, int Nq);
int hva_merge_nterms_launch(int BH, int Nk, const int* sizes_k, int* nterms, cudaStream_t st);
int hva_merge_inter_launch(int BH, int Nq, int Nk, const uint32_t* chi, const int* sizes_k, const int* nterms, int* inter, const int* list,
                           const int* cnt, cudaStream_t st);


size_t hva_merge_ws_bytes(int BH, int Nq, int Nk) {
  size_t Wd = (Nk + 31) / 32;
  return hva_align((size_t)BH * Nq * Wd * 4) + 5 * hva_align((size_t)BH * Nq * 4) + hva_align((size_t)BH * Nq * 8) +
         (Nq <= 2048 ? hva_merge_inter_bytes(BH, Nq) : 0);
}

extern "C" size_t hva_merge_workspace_bytes(int32_t BH, int32_t Nq, int32_t Nk) {
  if (BH < 1 || Nq < 1 || Nk < 1) return 0;
  return hva_merge_ws_bytes(BH, Nq, Nk);
}

int hva_merge_offset(int32_t bh0, int32_t BH, int32_t Nq, int32_t Nk, const int32_t* sizes_q, const int32_t* sizes_k,
                         const uint8_t* mask, int32_t tile_q, int32_t tile_k, int32_t rounds, int32_t max_q_tiles,
                         uint32_t seed, int32_t* group_of_cluster, int32_t* n_groups, uint8_t* group_mask, uint32_t flags, void* ws,
                         size_t ws_bytes, void* stream) {
  if (!sizes_q || !sizes_k || !mask || !group_of_cluster || !n_groups || !group_mask || !ws) return HVA_EINVAL;
  if (BH < 1 || Nq < 1 || Nk < 1 || tile_q < 1 || tile_k < 1 || rounds < 0 || max_q_tiles < 0) return HVA_EINVAL;
  if (Nk > 2048 || Nq > 65535) return HVA_EUNSUPPORTED;
  if (ws_bytes < hva_merge_ws_bytes(BH, Nq, Nk)) return HVA_EWORKSPACE;
  MergeParams p;
  p.Nq = Nq; p.Nk = Nk; p.Wd = (Nk + 31) / 32;
  p.sizes_q = sizes_q; p.sizes_k = sizes_k; p.mask = mask;
  p.tile_q = tile_q; p.tile_k = tile_k; p.rounds = rounds; p.max_q_tiles = max_q_tiles; p.seed = seed; p.bh0 = bh0;
  p.group_of = group_of_cluster; p.n_groups = n_groups; p.group_mask = group_mask;
  char* w = reinterpret_cast<char*>(ws);
  size_t a4 = hva_align((size_t)BH * Nq * 4);
  p.chi = reinterpret_cast<uint32_t*>(w); w += hva_align((size_t)BH * Nq * p.Wd * 4);
  p.sq = reinterpret_cast<int*>(w); w += a4;
  p.kap = reinterpret_cast<int*>(w); w += a4;
  p.alive = reinterpret_cast<int*>(w); w += a4;
  p.side = reinterpret_cast<int*>(w); w += a4;
  p.remap = reinterpret_cast<int*>(w); w += a4;
  p.best = reinterpret_cast<unsigned long long*>(w); w += hva_align((size_t)BH * Nq * 8);
  const bool use_inter = rounds > 0 && Nq <= 2048 && !(flags & HVA_FLAG_MERGE_SIMT);
  const int Nqp = (Nq + 127) / 128 * 128;
  int* inter = reinterpret_cast<int*>(w);
  int* nterms = reinterpret_cast<int*>(w + hva_align((size_t)BH * Nqp * Nqp * 4));
  int* side_cnt = reinterpret_cast<int*>(w + hva_align((size_t)BH * Nqp * Nqp * 4) + hva_align((size_t)BH * 4));
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const dim3 gw((Nq + 7) / 8, BH);
  hva_merge_init_kernel<<<gw, 256, 0, st>>>(p);
  HVA_CHECK_LAUNCH();
  const size_t smem = ((size_t)p.Wd * 32 + 2 * (size_t)Nq) * sizeof(int);
  if (use_inter) HVA_TRY(hva_merge_nterms_launch(BH, Nk, sizes_k, nterms, st));
  for (int r = 1; r <= rounds; ++r) {
    if (use_inter) {
      hva_merge_sides_kernel<<<BH, 1024, 0, st>>>(p, r, p.side, side_cnt);
      HVA_CHECK_LAUNCH();
      HVA_TRY(hva_merge_inter_launch(BH, Nq, Nk, p.chi, sizes_k, nterms, inter, p.side, side_cnt, st));
      hva_merge_propose_inter_kernel<<<gw, 256, 0, st>>>(p, r, inter, Nqp, p.side, side_cnt);
    } else {
      hva_merge_propose_kernel<<<gw, 256, smem, st>>>(p, r);
    }
    HVA_CHECK_LAUNCH();
    hva_merge_apply_kernel<<<BH, 1024, 0, st>>>(p);
    HVA_CHECK_LAUNCH();
  }
  hva_merge_rank_kernel<<<BH, 1024, 0, st>>>(p);
  HVA_CHECK_LAUNCH();
  hva_merge_out_kernel<<<dim3(Nq, BH), 256, 0, st>>>(p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

extern "C" int hva_merge(int32_t BH, int32_t Nq, int32_t Nk, const int32_t* sizes_q, const int32_t* sizes_k,
                         const uint8_t* mask, int32_t tile_q, int32_t tile_k, int32_t rounds, int32_t max_q_tiles,
                         uint32_t seed, int32_t* group_of_cluster, int32_t* n_groups, uint8_t* group_mask, void* ws,
                         size_t ws_bytes, void* stream) {
  return hva_merge_offset(0, BH, Nq, Nk, sizes_q, sizes_k, mask, tile_q, tile_k, rounds, max_q_tiles, seed, group_of_cluster, n_groups,
                          group_mask, 0u, ws, ws_bytes, stream);
}

extern "C" int hva_merge_ex(int32_t BH, int32_t Nq, int32_t Nk, const int32_t* sizes_q, const int32_t* sizes_k,
                            const uint8_t* mask, int32_t tile_q, int32_t tile_k, int32_t rounds, int32_t max_q_tiles,
                            uint32_t seed, int32_t* group_of_cluster, int32_t* n_groups, uint8_t* group_mask, uint32_t flags,
                            void* ws, size_t ws_bytes, void* stream) {
  return hva_merge_offset(0, BH, Nq, Nk, sizes_q, sizes_k, mask, tile_q, tile_k, rounds, max_q_tiles, seed, group_of_cluster, n_groups,
                          group_mask, flags, ws, ws_bytes, stream);
}
