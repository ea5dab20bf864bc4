// S1 on the tensor pipe (bf16 inputs, D = 128): assignment step of 3D local-window k-means
// (Alg. 2 lines 14-21, l.367-381; Eq. 5 l.81; Eq. 6 l.97).
//
// The direct form sum_c (x_c - mu_c)^2 on CUDA cores is ALU-bound (profiles/r1b: 6.5 % of DRAM peak).
// Here the 27.D dot products leave the FP32 pipe:
//   score_v = |mu_v|^2 - 2 x.mu_v  ( = d^2_v - |x|^2 ),   x.mu_v = x.hi_v + x.lo_v
// with mu split into two bf16 terms (hi = RN(mu), lo = RN(mu - hi); |mu - hi - lo| <= 2^-18 |mu|), so
// both products are exact in the MMA and only the fp32 accumulation rounds.  One CTA per home cell:
//   TMA   one 5-D box brings the cell's k_t x k_h x k_w tokens (rows of 256 B) into a 128B-swizzled K-major
//         A tile, one 5-D box per split term brings the window's w_t x w_h x w_w centroids (delta_t-major ==
//         ascending centroid id, Alg. 2 line 18) into the B tiles
//   MMA   tcgen05.mma 128 x NPAD x 16, 8 k-steps x {hi, lo}, fp32 accumulator in TMEM
//   scan  thread = token = TMEM lane: tcgen05.ld of its score row, argmin
// The tensor-pipe score is a FILTER, not the decision: every candidate whose score lies within a rigorous
// error margin of the decisive one is re-evaluated in the exact direct form in fp32 (the arithmetic of the
// CUDA-core kernel), and the first minimum among them wins (strict '<', R-C1).  So labels are those of the
// direct form; with the Lowe ratio requested (Eq. 6) the best and the second best are always exact.
// The centroid update is the same deterministic per-(cell, slot) segmented reduction as in cluster.cu.
#include "common.cuh"
#include "ptx.cuh"
#include "cluster_tc.cuh"

namespace {
using namespace hva_ptx;

constexpr int kD = 128;
constexpr int kThreads = 128;
// |tensor-pipe dot - exact dot| <= kEpsDot |x| |mu|: split error 2^-18 plus fp32 accumulation of 256 exact
// products.  Observed on B200 (HVA_CLUSTER_PROBE, tests/test_gpu_parity.py): score error 4.6e-6 |x||mu| including the
// rounding of the fp32 direct form it is compared with, against the 2 kEpsDot = 6.1e-5 assumed: 13x head room.
constexpr float kEpsDot = 1.0f / 32768.0f;

struct AssignTcParams {
  HvaGrid g;
  const float* mu;     // [BH, Nc, D] fp32 centroids (exact refine)
  const float* musq;   // [BH, Nc] |mu|^2 fp32
  float* part;         // [BH, Nc(cells), nwin, D]
  int* part_cnt;       // [BH, Nc(cells), nwin]
  int* assign;         // [BH, n] or null
  float* lowe;         // [BH, n] or null
  int npad;            // window candidates padded to the MMA N granule (16)
  int rows_a;          // cell tokens padded to the swizzle atom (8 rows)
  uint32_t tmem_cols;
  float* probe;        // debug: max |score_tc - score_exact| / (|x| max|mu|), or null
};

struct __align__(8) AssignTcBars {
  uint64_t full, mma_done;
  uint32_t tmem_base;
};

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

// exact direct form sum_c (x_c - mu_c)^2, fp32, sequential in c (Eq. 5)
__device__ __forceinline__ float direct_dist(const unsigned char* sA, int half_bytes, int r, const float* __restrict__ mu) {
  float acc = 0.f;
#pragma unroll 4
  for (int q = 0; q < 16; ++q) {
    float x[8];
    unpack8(*x_chunk(sA, half_bytes, r, q), x);
    const float4 m0 = __ldg(reinterpret_cast<const float4*>(mu) + 2 * q);
    const float4 m1 = __ldg(reinterpret_cast<const float4*>(mu) + 2 * q + 1);
    float d;
    d = x[0] - m0.x; acc = fmaf(d, d, acc);
    d = x[1] - m0.y; acc = fmaf(d, d, acc);
    d = x[2] - m0.z; acc = fmaf(d, d, acc);
    d = x[3] - m0.w; acc = fmaf(d, d, acc);
    d = x[4] - m1.x; acc = fmaf(d, d, acc);
    d = x[5] - m1.y; acc = fmaf(d, d, acc);
    d = x[6] - m1.z; acc = fmaf(d, d, acc);
    d = x[7] - m1.w; acc = fmaf(d, d, acc);
  }
  return acc;
}

__device__ __noinline__ float direct_dist_probe(const unsigned char* sA, int half_bytes, int r, const float* mu) {
  return direct_dist(sA, half_bytes, r, mu);
}

__global__ void __launch_bounds__(kThreads) hva_assign_tc_kernel(const __grid_constant__ CUtensorMap map_x,
                                                                 const __grid_constant__ CUtensorMap map_hi,
                                                                 const __grid_constant__ CUtensorMap map_lo, AssignTcParams p) {
  const HvaGrid& g = p.g;
  const int cell = blockIdx.x, bh = blockIdx.y, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int ut = cell / (g.Kh * g.Kw), uh = (cell / g.Kw) % g.Kh, uw = cell % g.Kw;
  const int st = hva_win_start(ut, g.wt, g.Kt), sh = hva_win_start(uh, g.wh, g.Kh), sw = hva_win_start(uw, g.ww, g.Kw);
  const int ctok = g.kt * g.kh * g.kw, nwin = g.nwin, npad = p.npad;
  const int half_a = p.rows_a * 128, half_b = npad * 128;

  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  unsigned char* sA = smem;                       // [2 halves][rows_a][128 B]   tokens, K-major SW128
  unsigned char* sBhi = sA + 2 * half_a;          // [2 halves][npad][128 B]     hi term of the window centroids
  unsigned char* sBlo = sBhi + 2 * half_b;        // [2 halves][npad][128 B]     lo term
  float* s_c = reinterpret_cast<float*>(sBlo + 2 * half_b);   // [npad] |mu_v|^2
  int* s_u = reinterpret_cast<int*>(s_c + npad);              // [npad] centroid id of window slot v
  int* s_wcnt = s_u + npad;                                   // [4][npad] per-warp slot counts
  int* s_start = s_wcnt + 4 * npad;                           // [npad + 1]
  int* s_order = s_start + npad + 1;                          // [128]
  AssignTcBars* B = reinterpret_cast<AssignTcBars*>((reinterpret_cast<uintptr_t>(s_order + kThreads) + 7) & ~uintptr_t(7));

  if (tid == 0) {
    mbar_init(&B->full, 1);
    mbar_init(&B->mma_done, 1);
    mbar_fence_init();
  }
  __syncwarp();
  if (warp == 0) tmem_alloc(&B->tmem_base, p.tmem_cols);
  // window slot -> centroid id (ascending == delta_t-major, Alg. 2 line 18), |mu|^2
  for (int v = tid; v < npad; v += kThreads) {
    int u = 0;
    float c = 0.f;
    if (v < nwin) {
      const int dt = v / (g.wh * g.ww), dh = (v / g.ww) % g.wh, dw = v % g.ww;
      u = ((st + dt) * g.Kh + (sh + dh)) * g.Kw + (sw + dw);
      c = __ldg(p.musq + (size_t)bh * g.Nc + u);
    }
    s_u[v] = u; s_c[v] = c;
  }
  for (int i = tid; i < 4 * npad; i += kThreads) s_wcnt[i] = 0;
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = B->tmem_base;

  if (tid == 0) {
    mbar_expect_tx(&B->full, (uint32_t)(2 * ctok * 128 + 4 * nwin * 128));
    tma_load_5d(&map_x, &B->full, sA, 0, uw * g.kw, uh * g.kh, ut * g.kt, bh);
    tma_load_5d(&map_x, &B->full, sA + half_a, 64, uw * g.kw, uh * g.kh, ut * g.kt, bh);
    tma_load_5d(&map_hi, &B->full, sBhi, 0, sw, sh, st, bh);
    tma_load_5d(&map_hi, &B->full, sBhi + half_b, 64, sw, sh, st, bh);
    tma_load_5d(&map_lo, &B->full, sBlo, 0, sw, sh, st, bh);
    tma_load_5d(&map_lo, &B->full, sBlo + half_b, 64, sw, sh, st, bh);
    mbar_wait(&B->full, 0);
    tc_fence_after();
    const uint32_t idesc = umma_idesc_bf16(128, (uint32_t)npad, 0);
    const uint32_t a_addr = smem_u32(sA), hi_addr = smem_u32(sBhi), lo_addr = smem_u32(sBlo);
#pragma unroll
    for (int ks = 0; ks < kD / 16; ++ks) {
      const uint32_t oa = (ks >> 2) * half_a + (ks & 3) * 32, ob = (ks >> 2) * half_b + (ks & 3) * 32;
      mma_ss(tmem, umma_desc(a_addr + oa, 16, 1024), umma_desc(hi_addr + ob, 16, 1024), idesc, ks > 0);
    }
#pragma unroll
    for (int ks = 0; ks < kD / 16; ++ks) {
      const uint32_t oa = (ks >> 2) * half_a + (ks & 3) * 32, ob = (ks >> 2) * half_b + (ks & 3) * 32;
      mma_ss(tmem, umma_desc(a_addr + oa, 16, 1024), umma_desc(lo_addr + ob, 16, 1024), idesc, 1);
    }
    tc_commit(&B->mma_done);
  }
  __syncwarp();

  // ---- token geometry; |x|^2 and the filter margin while the MMAs run
  const int li = tid;
  int lab = -1;
  size_t tok = 0;
  {
    const int dt = li / (g.kh * g.kw), dh = (li / g.kw) % g.kh, dw = li % g.kw;
    const int t = ut * g.kt + dt, h = uh * g.kh + dh, w = uw * g.kw + dw;
    if (li < ctok && t < g.T && h < g.H && w < g.W) { lab = 0; tok = (size_t)(t * g.H + h) * g.W + w; }
  }
  const bool valid = lab == 0;
  float c_max = 0.f;
  for (int v = 0; v < nwin; ++v) c_max = fmaxf(c_max, s_c[v]);
  mbar_wait(&B->full, 0);
  float xsq = 0.f;
  if (valid) {
#pragma unroll 4
    for (int q = 0; q < 16; ++q) {
      float x[8];
      unpack8(*x_chunk(sA, half_a, li, q), x);
#pragma unroll
      for (int i = 0; i < 8; ++i) xsq = fmaf(x[i], x[i], xsq);
    }
  }
  // score error E <= 2 kEpsDot |x| |mu| (+ rounding of |mu|^2 and of the fma: 6e-7 (|mu|^2 + 2|x||mu|)); candidates within
  // 2E of the decisive score are contenders
  const float xm = sqrtf(xsq * c_max);
  const float margin = 2.f * (2.f * kEpsDot * xm + 6e-7f * (c_max + 2.f * xm));

  mbar_wait(&B->mma_done, 0);
  tc_fence_after();
  const float kInf = __int_as_float(0x7f800000);
  float best = kInf, second = kInf;
  const uint32_t trow = tmem + ((uint32_t)(warp * 32) << 16);
  uint32_t sc[32];
  // pass 1: smallest and second smallest filter score
  float s1 = kInf, s2 = kInf;
  int v1 = 0;
  for (int v0 = 0; v0 < nwin; v0 += 32) {
    tmem_ld32(trow + v0, sc);
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      if (v0 + i < nwin) {
        const float s = fmaf(-2.f, __uint_as_float(sc[i]), s_c[v0 + i]);
        if (s < s1) { s2 = s1; s1 = s; v1 = v0 + i; }
        else if (s < s2) s2 = s;
      }
    }
  }
  const bool want2 = p.lowe != nullptr;
  const float thr = (want2 ? s2 : s1) + margin;     // s2 = +inf (single candidate): every candidate is a contender
  const bool refine = valid && (want2 || !(s2 > thr));
  if (valid && !refine) lab = v1;                   // decided by the filter: no other candidate can be the direct-form argmin
  const float* mu_b = p.mu + (size_t)bh * g.Nc * kD;
  if (__any_sync(0xffffffffu, refine)) {            // tcgen05.ld is warp-collective: the chunk loop stays warp-uniform
    // pass 2: exact direct form for the contenders, ascending candidate id, strict '<'  (R-C1)
    for (int v0 = 0; v0 < nwin; v0 += 32) {
      if (nwin > 32) tmem_ld32(trow + v0, sc);
      uint32_t cand = 0;
      if (refine) {
#pragma unroll
        for (int i = 0; i < 32; ++i)
          if (v0 + i < nwin && fmaf(-2.f, __uint_as_float(sc[i]), s_c[v0 + i]) <= thr) cand |= 1u << i;
      }
      while (cand) {
        const int v = v0 + __ffs(cand) - 1;
        cand &= cand - 1;
        const float dd = direct_dist(sA, half_a, li, mu_b + (size_t)s_u[v] * kD);
        if (dd < best) { second = best; best = dd; lab = v; }
        else if (dd < second) second = dd;
      }
    }
  }
  if (valid) {
    if (p.assign) p.assign[(size_t)bh * g.n + tok] = s_u[lab];
    if (p.lowe) {   // rho = d1/d2, unsquared (Eq. 6); single candidate -> 0; d2 == 0 -> 1 (R-H1)
      const float rho = (second == kInf) ? 0.f : (second > 0.f ? sqrtf(best / second) : 1.f);
      p.lowe[(size_t)bh * g.n + tok] = rho;
    }
  }
  if (p.probe) {   // debug: observed filter error against the exact direct form
    float worst = 0.f;
    for (int v0 = 0; v0 < nwin; v0 += 32) {
      tmem_ld32(trow + v0, sc);
      if (valid) {
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          if (v0 + i < nwin) {
            const float s = fmaf(-2.f, __uint_as_float(sc[i]), s_c[v0 + i]);
            const float dd = direct_dist_probe(sA, half_a, li, mu_b + (size_t)s_u[v0 + i] * kD);
            worst = fmaxf(worst, fabsf((dd - xsq) - s) / fmaxf(xm, 1e-30f));
          }
        }
      }
    }
    atomicMax(reinterpret_cast<int*>(p.probe), __float_as_int(worst));
  }
  tc_fence_before();

  // ---- counting sort of the cell's tokens by slot, stable in token order
  {
    const unsigned m = __match_any_sync(0xffffffffu, lab);
    const int rank = __popc(m & ((1u << lane) - 1u));
    if (lab >= 0 && rank == 0) s_wcnt[warp * npad + lab] = __popc(m);
    __syncthreads();
    if (warp == 0) {
      int carry = 0;
      for (int v0 = 0; v0 < nwin; v0 += 32) {
        const int v = v0 + lane;
        const int t = v < nwin ? s_wcnt[v] + s_wcnt[npad + v] + s_wcnt[2 * npad + v] + s_wcnt[3 * npad + v] : 0;
        int inc = t;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int y = __shfl_up_sync(0xffffffffu, inc, o);
          if (lane >= o) inc += y;
        }
        if (v < nwin) s_start[v] = carry + inc - t;
        carry += __shfl_sync(0xffffffffu, inc, 31);
      }
      if (lane == 0) s_start[nwin] = carry;
    }
    __syncthreads();
    if (lab >= 0) {
      int pos = s_start[lab] + rank;
      for (int w2 = 0; w2 < warp; ++w2) pos += s_wcnt[w2 * npad + lab];
      s_order[pos] = li;
    }
    __syncthreads();
  }
  if (warp == 0) { tc_fence_after(); tmem_dealloc(tmem, p.tmem_cols); }

  // ---- segmented per-cell reduction (z_a += x, Alg. 2 line 20): thread = two feature dims, tokens in token order
  const size_t pbase = ((size_t)bh * g.Nc + cell) * nwin;
  for (int v = tid; v < nwin; v += kThreads) p.part_cnt[pbase + v] = s_start[v + 1] - s_start[v];
  const int cp = tid & 63, grp = tid >> 6;          // dims 2cp, 2cp+1; slots grp, grp+2, ...
  const int q = cp >> 2;                             // 16-byte chunk holding the pair
  const unsigned char* colbase = sA + (q >> 3) * half_a + (cp & 3) * 4;
  for (int v = grp; v < nwin; v += 2) {
    const int b = s_start[v], e = s_start[v + 1];
    if (e > b) {
      float a0 = 0.f, a1 = 0.f;
      for (int i = b; i < e; ++i) {
        const int r = s_order[i];
        const uint32_t xx = *reinterpret_cast<const uint32_t*>(colbase + r * 128 + (((q & 7) ^ (r & 7)) << 4));
        a0 += __uint_as_float(xx << 16);
        a1 += __uint_as_float(xx & 0xffff0000u);
      }
      *reinterpret_cast<float2*>(p.part + (pbase + v) * kD + 2 * cp) = make_float2(a0, a1);
    }
  }
}

}  // namespace

bool hva_assign_tc_supported(const HvaGrid& g, int D, int dtype) {
  const int ctok = g.kt * g.kh * g.kw;
  return dtype == HVA_BF16 && D == kD && ctok <= 128 && g.nwin <= 256 && g.kt <= 256 && g.kh <= 256 && g.kw <= 256 &&
         g.wt <= 256 && g.wh <= 256 && g.ww <= 256;
}

namespace {
// 5-D map over Y[BH, d3, d2, d1, 128] bf16, box = 64 dims x b1 x b2 x b3 x 1, 128-byte swizzle; rows past the lattice
// (non-dividing cells, R-C4) read as zero and are never used.
bool make_map5(CUtensorMap* m, const void* base, int BH, int d3, int d2, int d1, int b3, int b2, int b1) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[5] = {(cuuint64_t)kD, (cuuint64_t)d1, (cuuint64_t)d2, (cuuint64_t)d3, (cuuint64_t)BH};
  cuuint64_t strides[4] = {(cuuint64_t)kD * 2, (cuuint64_t)d1 * kD * 2, (cuuint64_t)d2 * d1 * kD * 2, (cuuint64_t)d3 * d2 * d1 * kD * 2};
  cuuint32_t box[5] = {64, (cuuint32_t)b1, (cuuint32_t)b2, (cuuint32_t)b3, 1};
  cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
}  // namespace

int hva_assign_tc_prepare(const HvaGrid& g, int BH, const void* X, const void* mu_hi, const void* mu_lo, HvaAssignTc* a) {
  const int ctok = g.kt * g.kh * g.kw;
  a->npad = (g.nwin + 15) & ~15;
  if (a->npad < 16) a->npad = 16;
  a->rows_a = (ctok + 7) & ~7;
  a->tmem_cols = 32;
  while ((int)a->tmem_cols < ((g.nwin + 31) & ~31)) a->tmem_cols <<= 1;
  // the MMA reads 128 A rows: rows past rows_a alias the B tiles (finite garbage in unused TMEM lanes)
  size_t bytes = 2 * (size_t)a->rows_a * 128 + 4 * (size_t)a->npad * 128;
  const size_t min_a = 128 * 128 + (size_t)a->rows_a * 128;     // second half + 128 rows must stay inside the allocation
  if (bytes < min_a) bytes = min_a;
  bytes += sizeof(int) * (7 * (size_t)a->npad + 1 + kThreads) + sizeof(AssignTcBars) + 8 + 1024;
  a->smem = bytes;
  if (bytes > 227 * 1024) return HVA_EUNSUPPORTED;
  if (!make_map5(&a->map_x, X, BH, g.T, g.H, g.W, g.kt, g.kh, g.kw)) return HVA_ECUDA;
  if (!make_map5(&a->map_hi, mu_hi, BH, g.Kt, g.Kh, g.Kw, g.wt, g.wh, g.ww)) return HVA_ECUDA;
  if (!make_map5(&a->map_lo, mu_lo, BH, g.Kt, g.Kh, g.Kw, g.wt, g.wh, g.ww)) return HVA_ECUDA;
  if (cudaFuncSetAttribute(hva_assign_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess)
    return HVA_ECUDA;
  return HVA_OK;
}

int hva_assign_tc_launch(const HvaAssignTc& a, const HvaGrid& g, int BH, const float* mu, const float* musq, float* part,
                         int* part_cnt, int* assign, float* lowe, float* probe, cudaStream_t st) {
  AssignTcParams p{g, mu, musq, part, part_cnt, assign, lowe, a.npad, a.rows_a, a.tmem_cols, probe};
  hva_assign_tc_kernel<<<dim3(g.Nc, BH), kThreads, a.smem, st>>>(a.map_x, a.map_hi, a.map_lo, p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
