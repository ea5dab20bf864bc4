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
  int one_pass;        // 2 npad <= 256: one MMA pass over [hi; lo] stacked as 2 npad score columns (the token tile is read once)
  unsigned long long d_khw, d_kw, d_cs, d_kt;   // fast_div64 multipliers of the tile decode: K_h K_w, K_w, csplit, K_t
  int n_items;         // K_w * K_h * K_t * BH * csplit tiles: a CTA starts with tile blockIdx.x and draws the following ones
  int* counter;        // from this device counter (zero at launch), so that the SMs finish together
  float* probe;        // debug: max |score_tc - score_exact| / (|x| max|mu|), or null
};

struct __align__(8) AssignTcBars {
  uint64_t full, mma_done, sum_done;
  uint32_t tmem_base;
  int next;
  uint32_t cmax[4];     // per warp: max |mu_v|^2 over the window slots it set up (bits of a non-negative float)
};

__device__ __noinline__ float direct_dist_probe(const unsigned char* sA, int half_bytes, int r, const float* mu) {
  return direct_dist(sA, half_bytes, r, mu);
}

#ifdef HVA_ASSIGN_TIMING
#define CMARK(k) do { if (threadIdx.x == 0) { long long _t = clock64(); tacc[k] += (unsigned)(_t - tprev); tprev = _t; } } while (0)
#else
#define CMARK(k) do { } while (0)
#endif

// x / d for 0 <= x, x * d < 2^32 by one multiply-high (m = ceil(2^32 / d); d == 1 is passed as m = 0)
__device__ __forceinline__ int fast_div(int x, uint32_t m) { return m ? (int)__umulhi((uint32_t)x, m) : x; }
// x / d for every 0 <= x < 2^31 and d >= 1 by one 64-bit multiply-high (m = ceil(2^64 / d); d == 1 is passed as m = 0):
// m d = 2^64 + e with e < d, so x m / 2^64 = x / d + x e / (d 2^64), and the excess is below 2^-32 < 1 / d
__device__ __forceinline__ int fast_div64(int x, unsigned long long m) { return m ? (int)__umul64hi((unsigned long long)(uint32_t)x, m) : x; }

// Persistent CTAs (as many as fit the SMs, 4 per SM at the 3x5x8 cells) draw the tiles (home cell x time split) in raster
// order from a device counter; 128 threads, thread = token row of the tile = TMEM lane.  Per-CTA set-up (TMEM allocation,
// barriers, the CTA launch itself: ~2.5K clk, during which a kernel that allocates TMEM starts no other CTA on the SM)
// is paid once, and the loads of the next tile are issued as soon as the sums MMA has released the tiles, under the epilogue.
// kProbe = true is the instrumented instantiation behind hva_cluster_ex(probe != NULL) (tests: observed filter error; timing builds:
// per-phase clocks); the product instantiation carries none of that code.
template <bool kProbe>
__global__ void __launch_bounds__(kThreads, 4) hva_assign_tc_kernel(const __grid_constant__ CUtensorMap map_x,
                                                                 const __grid_constant__ CUtensorMap map_hi,
                                                                 const __grid_constant__ CUtensorMap map_lo, AssignTcParams p) {
  const HvaGrid& g = p.g;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int ctok = p.ct * g.kh * g.kw, nwin = g.nwin, npad = p.npad;   // token rows of a tile
  const int half_a = p.rows_a * 128, half_b = npad * 128;
#ifdef HVA_ASSIGN_TIMING
  unsigned tacc[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
  long long tprev = clock64();
#endif

  // Shared memory (offsets from a 1024-byte aligned base, kept as shared-space pointers):
  //   sB  [2 halves][hi | lo][npad][128 B]  window centroids, K-major SW128 (hi and lo rows of a half are contiguous: one
  //       B operand of 2 npad rows); after MMA 1 the first half is reused for
  //       sP [2 halves][npad][128 B], the one-hot tile P^T (rows = slots, K = tokens; B of MMA 2, K-major)
  //   sA  [2 halves][rows_a][128 B]         the tile's tokens (A of MMA 1, K-major; A of MMA 2, MN-major)
  // MMA 1 reads 128 token rows: rows past the tile alias whatever follows inside the allocation and only feed TMEM
  // lanes nobody reads.
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  unsigned char* sBhi = smem;                 // per 64-dim half: [hi rows | lo rows], halves 2 half_b apart
  unsigned char* sBlo = sBhi + half_b;
  unsigned char* sP = smem;
  unsigned char* sA = smem + 4 * half_b;
  float* s_c = reinterpret_cast<float*>(sA + 2 * half_a);     // [npad] |mu_v|^2
  int* s_u = reinterpret_cast<int*>(s_c + npad);              // [npad] centroid id of window slot v
  int* s_cnt = s_u + npad;                                    // [npad] tokens of the tile assigned to slot v
  AssignTcBars* B = reinterpret_cast<AssignTcBars*>(s_cnt + npad);

  // The SM starts the CTAs of a kernel that contains tcgen05.alloc one at a time: the next CTA does not begin before this one
  // has given the allocation permit back (measured: a CTA that never reaches the relinquish keeps the whole SM to itself).
  // So the allocation is the first thing the CTA does, on a warp of its own, while thread 0 sets up the loads.
  if (warp == 1) tmem_alloc(&B->tmem_base, p.tmem_cols);

  // tile -> (cell coordinates, time split, batch*head); thread 0 issues the six boxes of a tile
  struct Tile { int uw, uh, ut, bh, chunk; };
  auto decode = [&](int item) {
    Tile t;
    // (a runtime integer division is ~45 instructions; the decode runs twice per tile and warp: 14 % of the kernel's instructions)
    const int khw = g.Kw * g.Kh, z = fast_div64(item, p.d_khw), r = item - z * khw;
    t.uh = fast_div64(r, p.d_kw); t.uw = r - t.uh * g.Kw;
    const int zz = fast_div64(z, p.d_cs);
    t.chunk = z - zz * p.csplit;
    t.bh = fast_div64(zz, p.d_kt); t.ut = zz - t.bh * g.Kt;
    return t;
  };
  // the six boxes of a tile, two per call: part 0 = tokens, part 1 = hi, part 2 = lo (a 5-D box costs its issuing thread
  // ~150 clk, so the parts go to different warps); the expect-tx may be posted after bytes have landed
  auto issue = [&](const Tile& t, int part) {
    if (part == 0) {
      const int t0 = t.ut * g.kt + t.chunk * p.ct;
      mbar_expect_tx(&B->full, (uint32_t)(2 * ctok * 128 + 4 * nwin * 128));
      tma_load_5d(&map_x, &B->full, sA, 0, t.uw * g.kw, t.uh * g.kh, t0, t.bh);
      tma_load_5d(&map_x, &B->full, sA + half_a, 64, t.uw * g.kw, t.uh * g.kh, t0, t.bh);
    } else {
      const int st = hva_win_start(t.ut, g.wt, g.Kt), sh = hva_win_start(t.uh, g.wh, g.Kh), sw = hva_win_start(t.uw, g.ww, g.Kw);
      const CUtensorMap* m = part == 1 ? &map_hi : &map_lo;
      unsigned char* dst = part == 1 ? sBhi : sBlo;
      tma_load_5d(m, &B->full, dst, 0, sw, sh, st, t.bh);
      tma_load_5d(m, &B->full, dst + 2 * half_b, 64, sw, sh, st, t.bh);
    }
  };
  if (tid == 0) {
    mbar_init(&B->full, 1);
    mbar_init(&B->mma_done, 1);
    mbar_init(&B->sum_done, 1);
    mbar_fence_init();
    if ((int)blockIdx.x < p.n_items) {   // the loads need nothing but the barrier
      const Tile t = decode(blockIdx.x);
      issue(t, 0); issue(t, 1); issue(t, 2);
    }
  }
  // token rows ctok .. rows_a-1 take part in MMA 2 (K granule 16) with zero weight: they must be finite; TMA never writes them
  for (int i = tid; i < (p.rows_a - ctok) * 16; i += kThreads) {
    const int r = ctok + (i >> 4), q = i & 15;
    *reinterpret_cast<uint4*>(sA + (q >> 3) * half_a + r * 128 + ((q & 7) << 4)) = make_uint4(0, 0, 0, 0);
  }
  // rows nwin .. npad-1 of the four centroid tiles (hi | lo per 64-dim half) are never written by TMA: zero them once, so that the
  // pad columns of the score MMA are exactly 0 (the one-hot tile that aliases the first half only ever sets rows < nwin)
  for (int i = tid; i < 4 * (npad - nwin) * 8; i += kThreads) {
    const int k = i / ((npad - nwin) * 8), j = i - k * (npad - nwin) * 8;
    *reinterpret_cast<uint4*>(smem + k * half_b + nwin * 128 + j * 16) = make_uint4(0, 0, 0, 0);
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  // position of this thread's token inside a tile
  const int li = tid;
  const int ldt = fast_div(li, p.m_khw), lr = li - ldt * g.kh * g.kw, ldh = fast_div(lr, p.m_kw), ldw = lr - ldh * g.kw;
  const float kInf = __int_as_float(0x7f800000);
  uint32_t ph = 0;

  for (int item = blockIdx.x, next_item = 0; item < p.n_items; item = next_item, ph ^= 1u) {
  const Tile T = decode(item);
  if (tid == 96) {   // the tile after this one; published by the barrier below (a plain atomicAdd is wrapped in the compiler's
    int got;         // warp-aggregation sequence in all four warps: 28 instructions per warp and tile)
    asm volatile("atom.global.add.u32 %0, [%1], 1;" : "=r"(got) : "l"(p.counter) : "memory");
    B->next = (int)gridDim.x + got;
  }
  const int uw = T.uw, uh = T.uh, ut = T.ut, bh = T.bh, chunk = T.chunk;
  const int dt0 = chunk * p.ct;                        // first time slice of this tile inside the cell
  const int cell = (ut * g.Kh + uh) * g.Kw + uw;
  const int st = hva_win_start(ut, g.wt, g.Kt), sh = hva_win_start(uh, g.wh, g.Kh), sw = hva_win_start(uw, g.ww, g.Kw);
  // window slot -> centroid id (ascending == delta_t-major, Alg. 2 line 18), |mu|^2   (warps 1..3)
  float cm = 0.f;
  for (int v = tid - 32; v < npad; v += kThreads - 32) {
    if (v < 0) continue;
    int u = 0;
    float c = kInf;     // pad slot: its score column is exactly 0 (pad rows of the centroid tiles are zero), so score = +inf
    if (v < nwin) {
      const int dt = fast_div(v, p.m_whw), r = v - dt * g.wh * g.ww, dh = fast_div(r, p.m_ww), dw = r - dh * g.ww;
      u = ((st + dt) * g.Kh + (sh + dh)) * g.Kw + (sw + dw);
      c = __ldg(p.musq + (size_t)bh * g.Nc + u);
    }
    if (v < nwin) cm = fmaxf(cm, c);
    s_u[v] = u; s_c[v] = c; s_cnt[v] = 0;
  }
  {   // max |mu_v|^2 of the window: one redux per warp instead of every thread scanning s_c (|mu|^2 >= 0: uint order == float order)
    const uint32_t m = __reduce_max_sync(0xffffffffu, __float_as_uint(cm));
    if (lane == 0) B->cmax[warp] = m;
  }
  tc_fence_before();
  __syncthreads();
  CMARK(0);
  tc_fence_after();
  const uint32_t tmem = B->tmem_base;
  next_item = B->next;

  if (warp == 0) {
    // warp-uniform up to the elected lane: descriptors built once in uniform registers, a k-step only adds a constant to the
    // start-address field (a lane-0-only loop spends ~100 clk per MMA on descriptor arithmetic and R2UR moves)
    mbar_wait(&B->full, ph);
    tc_fence_after();
    const uint32_t idesc = umma_idesc_bf16(128, (uint32_t)(p.one_pass ? 2 * npad : npad), 0, 0);
    const uint64_t da = umma_desc(smem_u32(sA), 16, 1024), dhi = umma_desc(smem_u32(sBhi), 16, 1024), dlo = umma_desc(smem_u32(sBlo), 16, 1024);
    const uint32_t ha = (uint32_t)half_a >> 4, hb = (uint32_t)(2 * half_b) >> 4;
    if (elect_one()) {
#pragma unroll
      for (int ks = 0; ks < kD / 16; ++ks)
        mma_ss(tmem, da + ((ks >> 2) * ha + (ks & 3) * 2), dhi + ((ks >> 2) * hb + (ks & 3) * 2), idesc, ks > 0);
      if (!p.one_pass) {
#pragma unroll
        for (int ks = 0; ks < kD / 16; ++ks)
          mma_ss(tmem, da + ((ks >> 2) * ha + (ks & 3) * 2), dlo + ((ks >> 2) * hb + (ks & 3) * 2), idesc, 1);
      }
      tc_commit(&B->mma_done);
    }
    __syncwarp();
  }

  // ---- token geometry; an upper bound of |x|^2 and the filter margin while the MMAs run
  int lab = -1;
  size_t tok = 0;
  {
    const int t = ut * g.kt + dt0 + ldt, h = uh * g.kh + ldh, w = uw * g.kw + ldw;
    if (li < ctok && dt0 + ldt < g.kt && t < g.T && h < g.H && w < g.W) { lab = 0; tok = (size_t)(t * g.H + h) * g.W + w; }
  }
  const bool valid = lab == 0;
  // over the window's slots only (the pad slots hold +inf); written before the first barrier of the tile
  const float c_max = fmaxf(fmaxf(__uint_as_float(B->cmax[0]), __uint_as_float(B->cmax[1])),
                            fmaxf(__uint_as_float(B->cmax[2]), __uint_as_float(B->cmax[3])));
  mbar_wait(&B->full, ph);
  CMARK(1);
  // |x|^2 only scales the margin: packed bf16 FMAs (4 x 2 accumulators of 16 non-negative terms each: relative
  // error < 16 * 2^-8), inflated by 1/8 so that it is an upper bound
  float xsq = 0.f;
  if (valid) {
    __nv_bfloat162 acc[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[j] = __floats2bfloat162_rn(0.f, 0.f);
    // chunk q of row li sits at row + (((q & 7) ^ (li & 7)) << 4): the row is 128-byte aligned, so the swizzle is one XOR on
    // (row | (li & 7) << 4); 32-bit shared-space addresses keep the address arithmetic at one instruction per load
    const uint32_t xa0 = smem_u32(sA) + (uint32_t)li * 128u + ((uint32_t)(li & 7) << 4), xa1 = xa0 + (uint32_t)half_a;
#pragma unroll 1
    for (int hh = 0; hh < 2; ++hh) {
    const uint32_t xa = hh ? xa1 : xa0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      uint4 r;
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                   : "r"(xa ^ ((uint32_t)q << 4)));
      const __nv_bfloat162 x0 = *reinterpret_cast<const __nv_bfloat162*>(&r.x), x1 = *reinterpret_cast<const __nv_bfloat162*>(&r.y),
                           x2 = *reinterpret_cast<const __nv_bfloat162*>(&r.z), x3 = *reinterpret_cast<const __nv_bfloat162*>(&r.w);
      acc[0] = __hfma2(x0, x0, acc[0]); acc[1] = __hfma2(x1, x1, acc[1]);
      acc[2] = __hfma2(x2, x2, acc[2]); acc[3] = __hfma2(x3, x3, acc[3]);
    }
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
  mbar_wait(&B->mma_done, ph);
  CMARK(3);
  tc_fence_after();
  // the B tiles are dead: clear the one-hot tile that aliases the hi part (filled after the labels are known)
  for (int i = tid; i < (2 * half_b) / 16; i += kThreads) reinterpret_cast<uint4*>(sP)[i] = make_uint4(0, 0, 0, 0);

  const uint32_t trow = tmem + ((uint32_t)(warp * 32) << 16);
  float sv[32];
  // scores of one 32-candidate chunk: sv[j] = |mu_v|^2 - 2 x.mu_v, +inf past the window
  auto load_scores = [&](int v0) {
#pragma unroll
    for (int h = 0; h < 32; h += 16) {
      uint32_t raw[16], rlo[16];
      if (p.one_pass) {      // x.hi in columns [0, npad), x.lo in [npad, 2 npad)
        tmem_ld16_nowait(trow + v0 + h, raw);
        tmem_ld16_nowait(trow + npad + v0 + h, rlo);
        tmem_ld_wait16(raw);
        tmem_ld_wait16(rlo);
#pragma unroll
        for (int j = 0; j < 16; ++j) raw[j] = __float_as_uint(__uint_as_float(raw[j]) + __uint_as_float(rlo[j]));
      } else {
        tmem_ld16(trow + v0 + h, raw);
      }
      if (v0 + h >= npad) {      // a whole 16-column granule past the padded window (npad is a multiple of 16): warp-uniform
#pragma unroll
        for (int j = 0; j < 16; ++j) sv[h + j] = kInf;
        continue;
      }
#pragma unroll
      for (int j = 0; j < 16; j += 4) {      // pad slots nwin .. npad-1: column 0, |mu|^2 = +inf  =>  +inf without a compare
        const float4 c4 = *reinterpret_cast<const float4*>(s_c + v0 + h + j);
        sv[h + j] = fmaf(-2.f, __uint_as_float(raw[j]), c4.x);
        sv[h + j + 1] = fmaf(-2.f, __uint_as_float(raw[j + 1]), c4.y);
        sv[h + j + 2] = fmaf(-2.f, __uint_as_float(raw[j + 2]), c4.z);
        sv[h + j + 3] = fmaf(-2.f, __uint_as_float(raw[j + 3]), c4.w);
      }
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
    // thr = +inf (single-candidate window with the Lowe ratio: s2 = +inf) would also admit the pad slots, whose score is +inf
    cand &= nwin - v0 >= 32 ? 0xffffffffu : (1u << (nwin - v0)) - 1u;
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
        cand &= nwin - v0 >= 32 ? 0xffffffffu : (1u << (nwin - v0)) - 1u;
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
  if constexpr (kProbe) {   // observed filter error against the exact direct form
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
    if (lab >= 0) {
      *reinterpret_cast<__nv_bfloat16*>(sP + (li >> 6) * half_b + lab * 128 + (((((li & 63) >> 3) ^ (lab & 7))) << 4) + (li & 7) * 2) =
          __float2bfloat16_rn(1.0f);
      atomicAdd(&s_cnt[lab], 1);     // (a warp-wide match.any to combine equal labels first costs more than the conflicts)
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
  mbar_wait(&B->sum_done, ph);
  CMARK(8);
  tc_fence_after();
  // both tiles are dead (every generic read of sA happened before the one-hot barrier, MMA 2 has finished): the next tile's
  // loads run under the epilogue
  if (lane == 0 && warp != 1 && next_item < p.n_items) issue(decode(next_item), warp == 0 ? 0 : warp - 1);
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
  __syncthreads();     // s_cnt and the TMEM columns are free for the next tile
  CMARK(9);
  }   // tiles
#ifdef HVA_ASSIGN_TIMING
  if (kProbe && threadIdx.x == 0) for (int k = 0; k < 10; ++k) atomicAdd(p.probe + 16 + k, (float)tacc[k]);
#endif
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc(B->tmem_base, p.tmem_cols); }
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

int hva_assign_tc_prepare(const HvaGrid& g, int BH, const void* X, const void* mu_hi, const void* mu_lo, bool probe, HvaAssignTc* a) {
  const void* kern = probe ? (const void*)hva_assign_tc_kernel<true> : (const void*)hva_assign_tc_kernel<false>;
  a->probe = probe;
  a->ct = hva_assign_tc_slices(g);
  a->csplit = (g.kt + a->ct - 1) / a->ct;
  const int ctok = a->ct * g.kh * g.kw;
  a->npad = (g.nwin + 15) & ~15;
  a->rows_a = (ctok + 15) & ~15;
  a->one_pass = 2 * a->npad <= 256;
  a->tmem_cols = 32;
  while ((int)a->tmem_cols < (a->one_pass ? 2 : 1) * a->npad) a->tmem_cols <<= 1;
  const size_t half_a = (size_t)a->rows_a * 128, half_b = (size_t)a->npad * 128;
  size_t bytes = 4 * half_b + 2 * half_a + 3 * sizeof(int) * (size_t)a->npad + sizeof(AssignTcBars) + 16;
  // MMA 1 reads 128 token rows of its A operand: keep the over-read inside the allocation
  bytes = std::max(bytes, 4 * half_b + half_a + 16384);
  bytes += 1024;
  a->smem = bytes;
  if (bytes > 227 * 1024 || (long long)g.Kw * g.Kh * g.Kt * BH * a->csplit > 0x7fffffffLL) return HVA_EUNSUPPORTED;
  if (!make_map5(&a->map_x, X, BH, g.T, g.H, g.W, a->ct, g.kh, g.kw)) return HVA_ECUDA;
  if (!make_map5(&a->map_hi, mu_hi, BH, g.Kt, g.Kh, g.Kw, g.wt, g.wh, g.ww)) return HVA_ECUDA;
  if (!make_map5(&a->map_lo, mu_lo, BH, g.Kt, g.Kh, g.Kw, g.wt, g.wh, g.ww)) return HVA_ECUDA;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess)
    return HVA_ECUDA;
  // resident CTAs per SM from the shared-memory, register and TMEM budgets (the runtime's occupancy query answers 1 for a
  // kernel that allocates TMEM, whatever it allocates)
  int dev = 0, sms = 0, smem_sm = 0, smem_res = 0, regs_sm = 0;
  cudaFuncAttributes fa;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&smem_res, cudaDevAttrReservedSharedMemoryPerBlock, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&regs_sm, cudaDevAttrMaxRegistersPerMultiprocessor, dev) != cudaSuccess ||
      cudaFuncGetAttributes(&fa, kern) != cudaSuccess)
    return HVA_ECUDA;
  const int regs_cta = ((fa.numRegs + 7) & ~7) * kThreads;
  int per_sm = std::min({(int)((size_t)smem_sm / (bytes + (size_t)smem_res)), regs_sm / std::max(regs_cta, 1), 512 / (int)a->tmem_cols});
  if (per_sm < 1) return HVA_EUNSUPPORTED;
  a->grid = sms * per_sm;
  return HVA_OK;
}

int hva_assign_tc_launch(const HvaAssignTc& a, const HvaGrid& g, int BH, const float* mu, const float* musq, float* part,
                         int* part_cnt, int* assign, float* lowe, int* counter, float* probe, cudaStream_t st) {
  auto magic = [](int d) -> uint32_t { return d <= 1 ? 0u : (uint32_t)(((1ull << 32) + d - 1) / d); };
  auto magic64 = [](int d) -> unsigned long long { return d <= 1 ? 0ull : ~0ull / (unsigned long long)d + 1ull; };
  AssignTcParams p{g, mu, musq, part, part_cnt, assign, lowe, a.npad, a.rows_a, a.csplit, a.ct, magic(g.kh * g.kw), magic(g.kw), magic(g.wh * g.ww),
                   magic(g.ww), a.tmem_cols, a.one_pass, magic64(g.Kw * g.Kh), magic64(g.Kw), magic64(a.csplit), magic64(g.Kt),
                   g.Kw * g.Kh * g.Kt * BH * a.csplit, counter, probe};
  if (cudaMemsetAsync(counter, 0, sizeof(int), st) != cudaSuccess) return HVA_ECUDA;
  if (a.probe != (probe != nullptr)) return HVA_EINVAL;
  if (probe) hva_assign_tc_kernel<true><<<std::min(a.grid, p.n_items), kThreads, a.smem, st>>>(a.map_x, a.map_hi, a.map_lo, p);
  else hva_assign_tc_kernel<false><<<std::min(a.grid, p.n_items), kThreads, a.smem, st>>>(a.map_x, a.map_hi, a.map_lo, p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
