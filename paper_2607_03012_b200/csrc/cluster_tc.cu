// S1 (+ the per-cell part of S2) on the tensor pipe (bf16 inputs, D = 128): assignment step of 3D local-window
// k-means and the per-(cell, slot) partial centroid sums (Alg. 2 lines 14-21, l.367-381; Eq. 5 l.81; Eq. 6 l.97).
//
// The direct form sum_c (x_c - mu_c)^2 on CUDA cores is ALU-bound (profiles/r1b: 6.5 % of DRAM peak).
// Here the 27.D dot products leave the FP32 pipe:
//   score_v = |mu_v|^2 - 2 x.mu_v  ( = d^2_v - |x|^2 ),   x.mu_v = x.hi_v + x.lo_v
// with mu split into two bf16 terms (hi = RN(mu), lo = RN(mu - hi); |mu - hi - lo| <= 2^-18 |mu|), so
// both products are exact in the MMA and only the fp32 accumulation rounds.  One CTA per home cell:
//   TMA   one 5-D box brings the cell's k_t x k_h x k_w tokens (rows of 256 B) into a 128B-swizzled
//         tile, one 5-D box per split term brings the window's w_t x w_h x w_w centroids (delta_t-major ==
//         ascending centroid id, Alg. 2 line 18) into the B tiles
//   MMA 1 scores[token, slot] = X . {hi, lo}^T : tcgen05.mma 128 x NPAD x 16, 8 k-steps x 2 terms, fp32 in TMEM
//   scan  thread = token = TMEM lane: tcgen05.ld of its score row, min / contenders
//   MMA 2 z[slot, :] = P^T X with the one-hot assignment matrix P[token, slot] written to shared memory
//         (line 20: z_a += x); the products 1.0 * x are exact, the fp32 accumulation order is the hardware's,
//         fixed => the result is deterministic (same bits every run)
// The tensor-pipe score is a FILTER, not the decision: every candidate whose score lies within a rigorous
// error margin of the decisive one is re-evaluated in the exact direct form in fp32 (the arithmetic of the
// CUDA-core kernel), and the first minimum among them wins (strict '<', R-C1).  So labels are those of the
// direct form; with the Lowe ratio requested (Eq. 6) the best and the second best are always exact.
#include "common.cuh"
#include "ptx.cuh"
#include "cluster_tc.cuh"
#include <algorithm>

namespace {
using namespace hva_ptx;
using namespace hva_tc_dev;

constexpr int kD = 128;
constexpr int kThreads = 128;
struct AssignTcParams {
  HvaGrid g;
  const float* mu;     // [BH, Nc, D] fp32 centroids (exact refine)
  const float* musq;   // [BH, Nc] |mu|^2 fp32
  float* part;         // [BH, Nc(cells), nwin, D]
  int* part_cnt;       // [BH, Nc(cells), nwin]
  int* assign;         // [BH, n] or null
  float* lowe;         // [BH, n] or null
  int npad;            // window candidates padded to the MMA N granule (16)
  int rows_a;          // tile tokens padded to the MMA K granule (16 rows)
  int csplit, ct;      // a cell of more than 128 tokens is split along t into csplit tiles of ct time slices (one CTA each)
  uint32_t m_khw, m_kw, m_whw, m_ww;   // fast_div multipliers for k_h k_w, k_w, w_h w_w, w_w
  uint32_t tmem_cols;
  float* probe;        // debug: max |score_tc - score_exact| / (|x| max|mu|), or null
};

struct __align__(8) AssignTcBars {
  uint64_t full, mma_done, sum_done;
  uint32_t tmem_base;
};

__device__ __noinline__ float direct_dist_probe(const unsigned char* sA, int half_bytes, int r, const float* mu) {
  return direct_dist(sA, half_bytes, r, mu);
}

#ifdef HVA_ASSIGN_TIMING
#define CMARK(k) do { if (threadIdx.x == 0) { long long _t = clock64(); tacc[k] = (unsigned)(_t - tprev); tprev = _t; } } while (0)
#else
#define CMARK(k) do { } while (0)
#endif

// x / d for 0 <= x, x * d < 2^32 by one multiply-high (m = ceil(2^32 / d); d == 1 is passed as m = 0)
__device__ __forceinline__ int fast_div(int x, uint32_t m) { return m ? (int)__umulhi((uint32_t)x, m) : x; }

// One CTA per home cell: grid = (K_w, K_h, K_t * BH), 128 threads, thread = token row of the cell = TMEM lane.
__global__ void __launch_bounds__(kThreads) hva_assign_tc_kernel(const __grid_constant__ CUtensorMap map_x,
                                                                 const __grid_constant__ CUtensorMap map_hi,
                                                                 const __grid_constant__ CUtensorMap map_lo, AssignTcParams p) {
  const HvaGrid& g = p.g;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int uw = blockIdx.x, uh = blockIdx.y;
  const int chunk = blockIdx.z % p.csplit, zz = blockIdx.z / p.csplit, bh = zz / g.Kt, ut = zz - bh * g.Kt;
  const int dt0 = chunk * p.ct;                        // first time slice of this tile inside the cell
  const int cell = (ut * g.Kh + uh) * g.Kw + uw;
  const int st = hva_win_start(ut, g.wt, g.Kt), sh = hva_win_start(uh, g.wh, g.Kh), sw = hva_win_start(uw, g.ww, g.Kw);
  const int ctok = p.ct * g.kh * g.kw, nwin = g.nwin, npad = p.npad;   // token rows of this tile
  const int half_a = p.rows_a * 128, half_b = npad * 128;
#ifdef HVA_ASSIGN_TIMING
  unsigned tacc[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
  long long tprev = clock64();
#endif

  // Shared memory (offsets from a 1024-byte aligned base, kept as shared-space pointers):
  //   sB  [hi | lo][2 halves][npad][128 B]  window centroids, K-major SW128; after MMA 1 the hi part is reused for
  //       sP [2 halves][npad][128 B], the one-hot tile P^T (rows = slots, K = tokens; B of MMA 2, K-major)
  //   sA  [2 halves][rows_a][128 B]         the cell's tokens (A of MMA 1, K-major; A of MMA 2, MN-major)
  // MMA 1 reads 128 token rows: rows past the tile alias whatever follows inside the allocation and only feed TMEM
  // lanes nobody reads.
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  unsigned char* sBhi = smem;
  unsigned char* sBlo = sBhi + 2 * half_b;
  unsigned char* sP = smem;
  unsigned char* sA = smem + 4 * half_b;
  float* s_c = reinterpret_cast<float*>(sA + 2 * half_a);     // [npad] |mu_v|^2
  int* s_u = reinterpret_cast<int*>(s_c + npad);              // [npad] centroid id of window slot v
  int* s_cnt = s_u + npad;                                    // [npad] tokens of the cell assigned to slot v
  AssignTcBars* B = reinterpret_cast<AssignTcBars*>(s_cnt + npad);

  if (tid == 0) {
    mbar_init(&B->full, 1);
    mbar_init(&B->mma_done, 1);
    mbar_init(&B->sum_done, 1);
    mbar_fence_init();
    // the loads need nothing but the barrier: issue them before any other set-up work
    mbar_expect_tx(&B->full, (uint32_t)(2 * ctok * 128 + 4 * nwin * 128));
    tma_load_5d(&map_x, &B->full, sA, 0, uw * g.kw, uh * g.kh, ut * g.kt + dt0, bh);
    tma_load_5d(&map_x, &B->full, sA + half_a, 64, uw * g.kw, uh * g.kh, ut * g.kt + dt0, bh);
    tma_load_5d(&map_hi, &B->full, sBhi, 0, sw, sh, st, bh);
    tma_load_5d(&map_hi, &B->full, sBhi + half_b, 64, sw, sh, st, bh);
    tma_load_5d(&map_lo, &B->full, sBlo, 0, sw, sh, st, bh);
    tma_load_5d(&map_lo, &B->full, sBlo + half_b, 64, sw, sh, st, bh);
  }
  __syncwarp();
  if (warp == 0) tmem_alloc(&B->tmem_base, p.tmem_cols);
  // window slot -> centroid id (ascending == delta_t-major, Alg. 2 line 18), |mu|^2   (warps 1..3)
  for (int v = tid - 32; v < npad; v += kThreads - 32) {
    if (v < 0) continue;
    int u = 0;
    float c = 0.f;
    if (v < nwin) {
      const int dt = fast_div(v, p.m_whw), r = v - dt * g.wh * g.ww, dh = fast_div(r, p.m_ww), dw = r - dh * g.ww;
      u = ((st + dt) * g.Kh + (sh + dh)) * g.Kw + (sw + dw);
      c = __ldg(p.musq + (size_t)bh * g.Nc + u);
    }
    s_u[v] = u; s_c[v] = c; s_cnt[v] = 0;
  }
  // token rows ctok .. rows_a-1 take part in MMA 2 (K granule 16) with zero weight: they must be finite; TMA never writes them
  for (int i = tid; i < (p.rows_a - ctok) * 16; i += kThreads) {
    const int r = ctok + (i >> 4), q = i & 15;
    *reinterpret_cast<uint4*>(sA + (q >> 3) * half_a + r * 128 + ((q & 7) << 4)) = make_uint4(0, 0, 0, 0);
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  CMARK(0);
  tc_fence_after();
  const uint32_t tmem = B->tmem_base;

  if (warp == 0) {
    // warp-uniform up to the elected lane: descriptors built once in uniform registers, a k-step only adds a constant to the
    // start-address field (a lane-0-only loop spends ~100 clk per MMA on descriptor arithmetic and R2UR moves)
    mbar_wait(&B->full, 0);
    tc_fence_after();
    const uint32_t idesc = umma_idesc_bf16(128, (uint32_t)npad, 0, 0);
    const uint64_t da = umma_desc(smem_u32(sA), 16, 1024), dhi = umma_desc(smem_u32(sBhi), 16, 1024), dlo = umma_desc(smem_u32(sBlo), 16, 1024);
    const uint32_t ha = (uint32_t)half_a >> 4, hb = (uint32_t)half_b >> 4;
    if (elect_one()) {
#pragma unroll
      for (int ks = 0; ks < kD / 16; ++ks)
        mma_ss(tmem, da + ((ks >> 2) * ha + (ks & 3) * 2), dhi + ((ks >> 2) * hb + (ks & 3) * 2), idesc, ks > 0);
#pragma unroll
      for (int ks = 0; ks < kD / 16; ++ks)
        mma_ss(tmem, da + ((ks >> 2) * ha + (ks & 3) * 2), dlo + ((ks >> 2) * hb + (ks & 3) * 2), idesc, 1);
      tc_commit(&B->mma_done);
    }
    __syncwarp();
  }

  // ---- token geometry; an upper bound of |x|^2 and the filter margin while the MMAs run
  const int li = tid;
  int lab = -1;
  size_t tok = 0;
  {
    const int dt = fast_div(li, p.m_khw), r = li - dt * g.kh * g.kw, dh = fast_div(r, p.m_kw), dw = r - dh * g.kw;
    const int t = ut * g.kt + dt0 + dt, h = uh * g.kh + dh, w = uw * g.kw + dw;
    if (li < ctok && dt0 + dt < g.kt && t < g.T && h < g.H && w < g.W) { lab = 0; tok = (size_t)(t * g.H + h) * g.W + w; }
  }
  const bool valid = lab == 0;
  float c_max = 0.f;
  for (int v = 0; v < npad; v += 4) {
    const float4 c4 = *reinterpret_cast<const float4*>(s_c + v);
    c_max = fmaxf(fmaxf(c_max, fmaxf(c4.x, c4.y)), fmaxf(c4.z, c4.w));
  }
  mbar_wait(&B->full, 0);
  CMARK(1);
  // |x|^2 only scales the margin: packed bf16 FMAs (4 x 2 accumulators of 16 non-negative terms each: relative
  // error < 16 * 2^-8), inflated by 1/8 so that it is an upper bound
  float xsq = 0.f;
  if (valid) {
    __nv_bfloat162 acc[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[j] = __floats2bfloat162_rn(0.f, 0.f);
#pragma unroll 8
    for (int q = 0; q < 16; ++q) {
      const uint4 r = *x_chunk(sA, half_a, li, q);
      const __nv_bfloat162 x0 = *reinterpret_cast<const __nv_bfloat162*>(&r.x), x1 = *reinterpret_cast<const __nv_bfloat162*>(&r.y),
                           x2 = *reinterpret_cast<const __nv_bfloat162*>(&r.z), x3 = *reinterpret_cast<const __nv_bfloat162*>(&r.w);
      acc[0] = __hfma2(x0, x0, acc[0]); acc[1] = __hfma2(x1, x1, acc[1]);
      acc[2] = __hfma2(x2, x2, acc[2]); acc[3] = __hfma2(x3, x3, acc[3]);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) xsq += __low2float(acc[j]) + __high2float(acc[j]);
    xsq *= 1.125f;
  }
  // score error E <= 2 kEpsDot |x| |mu| (+ rounding of |mu|^2 and of the fma: 6e-7 (|mu|^2 + 2|x||mu|)); candidates within
  // 2E of the decisive score are contenders
  const float xm = sqrtf(xsq * c_max);
  const float margin = 2.f * (2.f * kEpsDot * xm + 6e-7f * (c_max + 2.f * xm));

  CMARK(2);
  mbar_wait(&B->mma_done, 0);
  CMARK(3);
  tc_fence_after();
  // the B tiles are dead: clear the one-hot tile that aliases the hi part (filled after the labels are known)
  for (int i = tid; i < (2 * half_b) / 16; i += kThreads) reinterpret_cast<uint4*>(sP)[i] = make_uint4(0, 0, 0, 0);

  const float kInf = __int_as_float(0x7f800000);
  const uint32_t trow = tmem + ((uint32_t)(warp * 32) << 16);
  float sv[32];
  // scores of one 32-candidate chunk: sv[j] = |mu_v|^2 - 2 x.mu_v, +inf past the window
  auto load_scores = [&](int v0) {
    uint32_t raw[32];
    tmem_ld32(trow + v0, raw);
#pragma unroll
    for (int j = 0; j < 32; j += 4) {
      const float4 c4 = *reinterpret_cast<const float4*>(s_c + v0 + j);   // npad is a multiple of 16
      sv[j] = v0 + j < nwin ? fmaf(-2.f, __uint_as_float(raw[j]), c4.x) : kInf;
      sv[j + 1] = v0 + j + 1 < nwin ? fmaf(-2.f, __uint_as_float(raw[j + 1]), c4.y) : kInf;
      sv[j + 2] = v0 + j + 2 < nwin ? fmaf(-2.f, __uint_as_float(raw[j + 2]), c4.z) : kInf;
      sv[j + 3] = v0 + j + 3 < nwin ? fmaf(-2.f, __uint_as_float(raw[j + 3]), c4.w) : kInf;
    }
  };
  // pass 1: smallest filter score, and the second smallest when the Lowe ratio is wanted (independent chains, merged);
  // 3-input min keeps the chains short
  const bool want2 = p.lowe != nullptr;
  float s1 = kInf, s2 = kInf, r1 = kInf, r2 = kInf;
  for (int v0 = 0; v0 < nwin; v0 += 32) {
    load_scores(v0);
    if (want2) {
#pragma unroll
      for (int j = 0; j < 32; j += 2) {
        s2 = fminf(s2, fmaxf(s1, sv[j]));
        s1 = fminf(s1, sv[j]);
        r2 = fminf(r2, fmaxf(r1, sv[j + 1]));
        r1 = fminf(r1, sv[j + 1]);
      }
    } else {
#pragma unroll
      for (int j = 0; j < 32; j += 4) {
        s1 = fminf(s1, fminf(sv[j], sv[j + 1]));
        r1 = fminf(r1, fminf(sv[j + 2], sv[j + 3]));
      }
    }
  }
  s2 = fminf(fminf(s2, r2), fmaxf(s1, r1));
  s1 = fminf(s1, r1);
  const float thr = (want2 ? s2 : s1) + margin;     // s2 = +inf (single candidate): every candidate is a contender
  // pass 2: contenders = candidates with score <= thr.  A single contender (without the Lowe ratio) is the direct-form
  // argmin; otherwise the exact direct form decides among them, ascending candidate id, strict '<'  (R-C1)
  float best = kInf, second = kInf;
  const float* mu_b = p.mu + (size_t)bh * g.Nc * kD;
  const bool single_chunk = nwin <= 32;
  int n_cont = 0, first = 0;
  uint32_t cand0 = 0;
  for (int v0 = 0; v0 < nwin; v0 += 32) {
    if (!single_chunk) load_scores(v0);
    uint32_t cand = 0, cand_b = 0;
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
      if (sv[j] <= thr) cand |= 1u << j;
      if (sv[j + 1] <= thr) cand_b |= 2u << j;
    }
    cand |= cand_b;
    if (n_cont == 0 && cand) first = v0 + __ffs(cand) - 1;
    n_cont += __popc(cand);
    if (v0 == 0) cand0 = cand;
  }
  const bool refine = valid && (want2 || n_cont > 1);
  if (valid && !refine) lab = first;
  if (__any_sync(0xffffffffu, refine)) {            // tcgen05.ld is warp-collective: the chunk loop stays warp-uniform
    for (int v0 = 0; v0 < nwin; v0 += 32) {
      uint32_t cand = cand0;
      if (!single_chunk) {
        load_scores(v0);
        cand = 0;
#pragma unroll
        for (int j = 0; j < 32; ++j)
          if (sv[j] <= thr) cand |= 1u << j;
      }
      if (!refine) cand = 0;
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
  CMARK(5);
#ifndef HVA_ASSIGN_TIMING
  if (p.probe) {   // debug: observed filter error against the exact direct form
    float worst = 0.f, xx = 0.f;
    if (valid) {
      for (int q = 0; q < 16; ++q) {
        float x[8];
        unpack8(*x_chunk(sA, half_a, li, q), x);
        for (int i = 0; i < 8; ++i) xx = fmaf(x[i], x[i], xx);
      }
    }
    for (int v0 = 0; v0 < nwin; v0 += 32) {
      load_scores(v0);
      if (valid) {
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          if (v0 + j < nwin) {
            const float dd = direct_dist_probe(sA, half_a, li, mu_b + (size_t)s_u[v0 + j] * kD);
            worst = fmaxf(worst, fabsf((dd - xx) - sv[j]) / fmaxf(sqrtf(xx * c_max), 1e-30f));
          }
        }
      }
    }
    if (xx > xsq) worst = 1.f;   // the packed-bf16 |x|^2 must be an upper bound
    atomicMax(reinterpret_cast<int*>(p.probe), __float_as_int(worst));
  }
#endif
  tc_fence_before();
  __syncthreads();        // one-hot tile cleared, every score read
  CMARK(6);

  // ---- one-hot tile P^T[slot, token] = 1 and the slot counts
  {
    const unsigned m = __match_any_sync(0xffffffffu, lab);
    if (lab >= 0) {
      *reinterpret_cast<__nv_bfloat16*>(sP + (li >> 6) * half_b + lab * 128 + (((((li & 63) >> 3) ^ (lab & 7))) << 4) + (li & 7) * 2) =
          __float2bfloat16_rn(1.0f);
      if ((m & ((1u << lane) - 1u)) == 0) atomicAdd(&s_cnt[lab], __popc(m));
    }
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncthreads();
  CMARK(7);
  tc_fence_after();

  // ---- MMA 2: z^T[dim, slot] = sum_token x[token, dim] P^T[slot, token]   (Alg. 2 line 20): A = the token tile read
  // MN-major (M = 128 feature dims), B = the one-hot tile, D overwrites the score columns; TMEM lane = feature dim
  if (warp == 0) {
    const uint32_t idesc = umma_idesc_bf16(128, (uint32_t)npad, 1, 0);
    const uint64_t dx = umma_desc(smem_u32(sA), half_a, 1024), dp = umma_desc(smem_u32(sP), 16, 1024);
    const uint32_t hb = (uint32_t)half_b >> 4;
    const int ksteps = p.rows_a >> 4;
    if (elect_one()) {
      if (ksteps == 8) {
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) mma_ss(tmem, dx + ks * (2048 >> 4), dp + ((ks >> 2) * hb + (ks & 3) * 2), idesc, ks > 0);
      } else {
        for (int ks = 0; ks < ksteps; ++ks) mma_ss(tmem, dx + ks * (2048 >> 4), dp + ((ks >> 2) * hb + (ks & 3) * 2), idesc, ks > 0);
      }
      tc_commit(&B->sum_done);
    }
    __syncwarp();
  }
  const size_t pbase = (((size_t)bh * g.Nc + cell) * p.csplit + chunk) * nwin;
  for (int v = tid; v < nwin; v += kThreads) p.part_cnt[pbase + v] = s_cnt[v];
  mbar_wait(&B->sum_done, 0);
  CMARK(8);
  tc_fence_after();
  // thread = feature dim: a warp stores 32 consecutive floats of a partial row (coalesced)
  float* prow = p.part + pbase * kD + tid;
  for (int v0 = 0; v0 < nwin; v0 += 32) {
    uint32_t raw[32];
    tmem_ld32(trow + v0, raw);
    // non-empty slots of this chunk as one ballot word: the stores below are then a bit test + STG with an immediate offset
    const unsigned nz = __ballot_sync(0xffffffffu, v0 + lane < nwin && s_cnt[v0 + lane] > 0);
    float* pr = prow + (size_t)v0 * kD;
#pragma unroll
    for (int j = 0; j < 32; ++j)
      if ((nz >> j) & 1u) pr[j * kD] = __uint_as_float(raw[j]);
  }
  CMARK(4);
  tc_fence_before();
  __syncthreads();
  CMARK(9);
#ifdef HVA_ASSIGN_TIMING
  if (threadIdx.x == 0 && p.probe) for (int k = 0; k < 10; ++k) atomicAdd(p.probe + 16 + k, (float)tacc[k]);
#endif
  if (warp == 0) { tc_fence_after(); tmem_dealloc(tmem, p.tmem_cols); }
}

}  // namespace

bool hva_assign_tc_supported(const HvaGrid& g, int D, int dtype) {
  return dtype == HVA_BF16 && D == kD && g.kh * g.kw <= 128 && g.nwin <= 256 && g.kt <= 256 && g.kh <= 256 && g.kw <= 256 &&
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
  a->ct = hva_assign_tc_slices(g);
  a->csplit = (g.kt + a->ct - 1) / a->ct;
  const int ctok = a->ct * g.kh * g.kw;
  a->npad = (g.nwin + 15) & ~15;
  a->rows_a = (ctok + 15) & ~15;
  a->tmem_cols = 32;
  while ((int)a->tmem_cols < a->npad) a->tmem_cols <<= 1;
  const size_t half_a = (size_t)a->rows_a * 128, half_b = (size_t)a->npad * 128;
  size_t bytes = 4 * half_b + 2 * half_a + 3 * sizeof(int) * (size_t)a->npad + sizeof(AssignTcBars) + 16;
  // MMA 1 reads 128 token rows of its A operand: keep the over-read inside the allocation
  bytes = std::max(bytes, 4 * half_b + half_a + 16384);
  bytes += 1024;
  a->smem = bytes;
  if (bytes > 227 * 1024 || (long long)g.Kt * BH * a->csplit > 65535 || g.Kh > 65535) return HVA_EUNSUPPORTED;
  if (!make_map5(&a->map_x, X, BH, g.T, g.H, g.W, a->ct, g.kh, g.kw)) return HVA_ECUDA;
  if (!make_map5(&a->map_hi, mu_hi, BH, g.Kt, g.Kh, g.Kw, g.wt, g.wh, g.ww)) return HVA_ECUDA;
  if (!make_map5(&a->map_lo, mu_lo, BH, g.Kt, g.Kh, g.Kw, g.wt, g.wh, g.ww)) return HVA_ECUDA;
  if (cudaFuncSetAttribute(hva_assign_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess)
    return HVA_ECUDA;
  return HVA_OK;
}

int hva_assign_tc_launch(const HvaAssignTc& a, const HvaGrid& g, int BH, const float* mu, const float* musq, float* part,
                         int* part_cnt, int* assign, float* lowe, float* probe, cudaStream_t st) {
  auto magic = [](int d) -> uint32_t { return d <= 1 ? 0u : (uint32_t)(((1ull << 32) + d - 1) / d); };
  AssignTcParams p{g, mu, musq, part, part_cnt, assign, lowe, a.npad, a.rows_a, a.csplit, a.ct, magic(g.kh * g.kw), magic(g.kw), magic(g.wh * g.ww),
                   magic(g.ww), a.tmem_cols, probe};
  hva_assign_tc_kernel<<<dim3(g.Kw, g.Kh, g.Kt * BH * a.csplit), kThreads, a.smem, st>>>(a.map_x, a.map_hi, a.map_lo, p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
