// S9 (+S10), tensor-core variant for bf16, D = 128, 128x128 tiles (sm_100a only):
// block-sparse FlashAttention over the plan's packed key runs (Eq. 4 l.56; packed key
// blocks l.109; union masks Eq. 8 l.115).
//
// One CTA per (group, q-tile) work item, one CTA per SM, 16 warps in four warpgroups:
//   warps 0-3 / 4-7  two softmax sets (setmaxnreg 200): set b takes the key tiles j = b (mod 2), i.e. always the buffers S_b / P_b;
//                    thread = one full query row (TMEM lane) held in 128 registers; correction and epilogue
//   warps 8, 11      TMA producers of the K ring (64-dim halves 0 / 1; warp 8 also loads the Q tile)
//   warps 10, 12     TMA producers of the V ring (64-dim halves 0 / 1)
//   warp  9          TMEM allocator (512 columns) + tcgen05.mma issuer (one elected lane)
// The producers walk the group's key runs and issue power-of-two-height boxes of a 128B-swizzled 2-D tensor map so that rows
// of different clusters land back to back in the stage buffer (exact packing across cluster boundaries, l.109).
// TMEM: S_0, S_1 (fp32 scores, 128 columns each), O (128), P_0, P_1 (bf16 probabilities, 64 each).
// Per key tile j:  S_b = Q K_j^T (SS MMA, K-major operands, fp32 accumulators in TMEM)
//                  P_b = exp2(S_b*scale*log2e - m_ref) written as bf16 into its own TMEM buffer (tcgen05.st)
//                  O  += P_b V_j (TS MMA: A = P from TMEM, B = V from smem, MN-major)
// with lazy (thresholded) rescaling of O in TMEM, 1/l normalisation and the inverse permutation
// fused into the epilogue's row stores.
#include "common.cuh"
#include "ptx.cuh"

namespace {
using namespace hva_ptx;

constexpr int kBM = 128, kBN = 128, kD = 128;
constexpr int kHalfBytes = 128 * 128;          // one 64-dim half of a 128-row tile: 128 rows x 128 B
constexpr int kTileBytes = 2 * kHalfBytes;     // 32 KB
constexpr int kStagesK = 3, kStagesV = 3;      // K ring and V ring of 128-row tiles (4 + 2 measured the same: the rings are L2-bandwidth bound)
constexpr int kThreadsTC = 512;                // 4 warpgroups: 0-1 softmax (setmaxnreg 200), 2-3 MMA / TMA warps + idle (setmaxnreg 56)                // warps 0-3 / 4-7 softmax of the even / odd key tiles, 9: MMA, TMA: 8 = K dims 0-63 (+Q), 11 = K dims 64-127, 10 = V
constexpr int kNumBoxes = 8;                   // box heights 1,2,4,...,128
constexpr uint32_t kTmemCols = 512;            // S_0, S_1 (fp32 scores), O (fp32), P_0, P_1 (bf16 probabilities)
constexpr uint32_t kColS = 0, kColO = 256, kColP = 384;   // S_b at kColS + 128 b, P_b at kColP + 64 b
constexpr float kRescaleThreshold = 8.0f;      // log2 units
// Share of the exponentials taken off MUFU (16/clk/SM = 1024 clk per 128x128 tile, the MMA time of a tile) by the software
// exp2 below.  It paid while the softmax paced the kernel (1 pair in 4: 96 -> 92 ms); with two softmax sets and the
// tensor pipe as the pace-maker under the power cap the extra FMA work only costs energy: 0 / 1 / 2 of 8 pairs =
// 77.5 / 78.9 / 79.8 ms per call at C4.
constexpr int kPolyPairs = 0;

struct TcMaps {
  CUtensorMap q;        // Q' (permuted) as 128-row boxes, or -- gather mode -- the UNPERMUTED Q as 1-row boxes for tile::gather4
  CUtensorMap k[kNumBoxes];
  CUtensorMap v[kNumBoxes];
};

struct TcParams {
  int n, Nq, Nk, run_stride, work_cap, unpermute, gather_q;
  float scale_log2;
  const int *goff, *koff, *kappa, *run_cnt, *work_cnt, *work, *perm_q;
  const uint32_t* runs;
  __nv_bfloat16* O;
#ifdef HVA_ATTN_TIMING
  unsigned long long* probe;   // per-phase cycle totals (diagnostic build only)
#endif
};
#ifdef HVA_ATTN_TIMING
unsigned long long* g_attn_timing = nullptr;   // diagnostic build only: set through hva_debug_attn_timing()
#endif

// instruction descriptor: D = F32, A = B = BF16, M = 128, N = 128; b_major selects MN-major B
__device__ __forceinline__ uint32_t umma_idesc(uint32_t b_mn_major) {
  return (1u << 4) | (1u << 7) | (1u << 10) | (b_mn_major << 16) | ((uint32_t)(kBN >> 3) << 17) | ((uint32_t)(kBM >> 4) << 24);
}

// 2^x on the FMA pipe for a pair (FlashAttention-4 style software exponential): x = n + f, n = round(x), |f| <= 1/2,
// 2^f by a degree-3 minimax polynomial (max relative error 7.5e-5, far below the bf16 rounding of P), exponent field += n.
__device__ __forceinline__ float2 exp2_poly2(float2 x) {
  x.x = fmaxf(x.x, -125.f); x.y = fmaxf(x.y, -125.f);
  const float2 magic = make_float2(12582912.f, 12582912.f);     // 1.5 * 2^23: the sum's low mantissa bits hold round(x)
  const float2 t = __fadd2_rn(x, magic);
  const float2 r = __fadd2_rn(t, make_float2(-12582912.f, -12582912.f));
  const float2 f = __fadd2_rn(x, make_float2(-r.x, -r.y));
  float2 q = __ffma2_rn(make_float2(0.0551716685f, 0.0551716685f), f, make_float2(0.2426111251f, 0.2426111251f));
  q = __ffma2_rn(q, f, make_float2(0.6932609677f, 0.6932609677f));
  q = __ffma2_rn(q, f, make_float2(0.9999280572f, 0.9999280572f));
  return make_float2(__uint_as_float(__float_as_uint(q.x) + (__float_as_uint(t.x) << 23)),
                     __uint_as_float(__float_as_uint(q.y) + (__float_as_uint(t.y) << 23)));
}

#ifdef HVA_ATTN_TIMING
#define AMARK(k) do { long long _t = clock64(); tacc[k] += (unsigned long long)(_t - tprev); tprev = _t; } while (0)
#else
#define AMARK(k) do { } while (0)
#endif

struct __align__(8) TcBarriers {
  uint64_t q_full, k_full[kStagesK], k_empty[kStagesK], v_full[kStagesV], v_empty[kStagesV], s_full[2], s_free[2], p_ready[2], p_free[2];
  uint32_t tmem_base;
  float xch[2][kBM];          // partial row sums of the two softmax sets
  float mref[kBM];            // reference exponent of each query row (shared by its two softmax threads)
  int seq[kBM];               // number of key tiles whose reference decision has been taken, per row
};

constexpr int kAlignSlack = 512;               // the dynamic window is 1024-byte aligned in practice (checked in the kernel)
constexpr size_t kSmemTC = kAlignSlack + kTileBytes * (1 + kStagesK + kStagesV) + sizeof(TcBarriers);
static_assert(kSmemTC <= 227 * 1024, "attention tile ring exceeds the shared memory of one SM");

// Walks the group's key runs (maximal runs of consecutive selected key clusters, contiguous in K')
// and packs them back to back into 128-row tiles (l.109).
struct RunWalker {
  const uint32_t* runs; const int* koff; int nrun, r, row0, len, used;
  __device__ void load() {
    if (r < nrun) { uint32_t rr = runs[r]; row0 = koff[rr & 0xffff]; len = koff[(rr >> 16) + 1] - row0; }
    else { len = 1 << 30; }   // past the last run: only reached for the finite over-read padding rows
    used = 0;
  }
};

// One segment of `len` consecutive source rows -> `len` consecutive tile rows.  A TMA box costs ~100 clk of the SM's TMA unit
// whatever its height (microbenchmark), and the box count paces the rings: instead of the binary decomposition
// (popcount(len) boxes) a segment takes at most TWO boxes of the largest power of two h <= len, at offsets 0 and len - h;
// the overlap is written twice with the same bytes.  Returns the bytes issued (for the barrier's expect-tx).
__device__ __forceinline__ int emit_boxes(const CUtensorMap* maps, uint64_t* bar, unsigned char* stage, int col, int grow, int dst, int len) {
  const int b = 31 - __clz(len), h = 1 << b;
  if (elect_one()) {
    tma_load_2d(maps + b, bar, stage + dst * 128, col, grow);
    if (len != h) tma_load_2d(maps + b, bar, stage + (dst + len - h) * 128, col, grow + len - h);
  }
  return (len != h ? 2 * h : h) * 128;
}

// the 64-dim half at column `col` of a packed key tile; returns the bytes issued
__device__ __forceinline__ int load_tile(RunWalker& w, const CUtensorMap* maps, uint64_t* bar, unsigned char* stage, int col,
                                         int base_row, int rows_valid, int rows_load) {
  int dst = 0, bytes = 0;
  while (dst < rows_valid) {
    while (w.used == w.len) { ++w.r; w.load(); }
    int seg = min(w.len - w.used, rows_valid - dst);
    bytes += emit_boxes(maps, bar, stage, col, base_row + w.row0 + w.used, dst, seg);
    w.used += seg; dst += seg;
  }
  if (rows_load > rows_valid)   // ragged last tile: round up to the MMA K granule with finite over-read rows
    bytes += emit_boxes(maps, bar, stage, col, base_row + w.row0 + w.used, dst, rows_load - rows_valid);
  return bytes;
}

__global__ void __launch_bounds__(kThreadsTC, 1) hva_attn_tc_kernel(const __grid_constant__ TcMaps maps, TcParams p) {
  const int bh = blockIdx.y;
  if ((int)blockIdx.x >= p.work_cnt[bh]) return;
  const uint32_t wi = (uint32_t)p.work[(size_t)bh * p.work_cap + blockIdx.x];
  const int g = wi & 0xffff, t = wi >> 16;
  const int* goff = p.goff + (size_t)bh * (p.Nq + 1);
  const int row0 = goff[g] + t * kBM, row1 = min(goff[g + 1], row0 + kBM);
  const int kappa = p.kappa[(size_t)bh * p.Nq + g];
  const int jn = (kappa + kBN - 1) / kBN;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int base_row = bh * p.n;

  extern __shared__ __align__(1024) unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  if (smem - smem_raw > kAlignSlack) __trap();
  unsigned char* sQ = smem;
  unsigned char* sK = smem + kTileBytes;
  unsigned char* sV = smem + kTileBytes * (1 + kStagesK);
  TcBarriers* B = reinterpret_cast<TcBarriers*>(smem + kTileBytes * (1 + kStagesK + kStagesV));

  if (jn == 0) {   // no key selected: defined as a zero row
    if (tid < kBM && row0 + tid < row1) {
      size_t orow = (size_t)base_row + (p.unpermute ? p.perm_q[(size_t)base_row + row0 + tid] : row0 + tid);
      uint4 z = make_uint4(0, 0, 0, 0);
      for (int c = 0; c < 16; ++c) reinterpret_cast<uint4*>(p.O + orow * kD)[c] = z;
    }
    return;
  }

  if (tid == 0) {
    mbar_init(&B->q_full, 1);
    for (int s = 0; s < kStagesK; ++s) { mbar_init(&B->k_full[s], 2); mbar_init(&B->k_empty[s], 1); }   // two producers (one per
    for (int s = 0; s < kStagesV; ++s) { mbar_init(&B->v_full[s], 2); mbar_init(&B->v_empty[s], 1); }   // 64-dim half) per ring
    mbar_init(&B->s_full[0], 1); mbar_init(&B->s_full[1], 1);
    mbar_init(&B->p_ready[0], 128); mbar_init(&B->p_ready[1], 128);     // set b = warps 4b..4b+3 owns S_b, P_b
    mbar_init(&B->s_free[0], 128); mbar_init(&B->s_free[1], 128);
    mbar_init(&B->p_free[0], 1); mbar_init(&B->p_free[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 9) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&B->tmem_base)), "r"(kTmemCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid < kBM) { B->mref[tid] = -INFINITY; B->seq[tid] = 0; }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = B->tmem_base;
  // register file: 512 threads x 128 at launch; the two softmax warpgroups hold a 128-column row each and take 200, the rest gives back
  if (warp == 8 || (warp >= 10 && warp <= 12)) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    // ===================================================== TMA producers (warp-uniform, one elected lane issues):
    // the K ring is on the critical path (QK_{j+2} is issued two tiles ahead): one warp per 64-dim half; one warp for the V ring
    const bool is_k = (warp == 8 || warp == 11);   // 8: K dims 0-63 (+Q), 11: K dims 64-127, 10: V dims 0-63, 12: V dims 64-127
    const int half = warp >= 11;
    if (warp == 8 && !p.gather_q && elect_one()) {
      mbar_expect_tx(&B->q_full, kTileBytes);
      tma_load_2d(&maps.q, &B->q_full, sQ, 0, base_row + row0);
      tma_load_2d(&maps.q, &B->q_full, sQ + kHalfBytes, 64, base_row + row0);
    }
    if (warp == 8 && p.gather_q) {
      // Q' = Pi^q Q fused into the load (Eq. 1): the tile's 128 rows are gathered from the unpermuted Q through perm_q, four rows per
      // TMA tile::gather4 instruction (each lands as four consecutive 128-byte rows of the swizzled tile).  Rows past the end of the
      // group repeat its last row (finite, never stored).
      const int* pq = p.perm_q + (size_t)base_row + row0;
      int tok[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) tok[k] = base_row + pq[min(4 * lane + k, row1 - row0 - 1)];
      if (lane == 0) mbar_expect_tx(&B->q_full, kTileBytes);
      for (int i = 0; i < 32; ++i) {
        const int t0 = __shfl_sync(0xffffffffu, tok[0], i), t1 = __shfl_sync(0xffffffffu, tok[1], i);
        const int t2 = __shfl_sync(0xffffffffu, tok[2], i), t3 = __shfl_sync(0xffffffffu, tok[3], i);
        if (lane == 0) {
          tma_gather4_2d(&maps.q, &B->q_full, sQ + i * 512, 0, t0, t1, t2, t3);
          tma_gather4_2d(&maps.q, &B->q_full, sQ + kHalfBytes + i * 512, 64, t0, t1, t2, t3);
        }
      }
      __syncwarp();
    }
    RunWalker w{p.runs + ((size_t)bh * p.Nq + g) * p.run_stride, p.koff + (size_t)bh * (p.Nk + 1),
                p.run_cnt[(size_t)bh * p.Nq + g], 0, 0, 0, 0};
    w.load();
    const CUtensorMap* mp = is_k ? maps.k : maps.v;
    uint64_t* full = is_k ? B->k_full : B->v_full;
    uint64_t* empty = is_k ? B->k_empty : B->v_empty;
    unsigned char* ring = (is_k ? sK : sV) + half * kHalfBytes;
    for (int j = 0; j < jn; ++j) {
      const int ns = is_k ? kStagesK : kStagesV;
      const int s = j % ns, use = j / ns;
      const int rows_valid = min(kBN, kappa - j * kBN);
      const int rows_load = rows_valid == kBN ? kBN : (rows_valid + 15) & ~15;
      if (use > 0) mbar_wait(&empty[s], (use - 1) & 1);
      const int bytes = load_tile(w, mp, &full[s], ring + s * kTileBytes, half * 64, base_row, rows_valid, rows_load);
      if (elect_one()) mbar_expect_tx(&full[s], bytes);   // posted after the boxes: the pending arrival keeps the phase open
      __syncwarp();
    }
  } else if (warp == 9) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    // ===================================================== MMA issuer: the whole warp runs the loop (uniform), one elected lane issues
    // S and P are double buffered and separate: QK_{j+2} is issued as soon as the softmax threads have pulled S_j into
    // registers (s_free), PV_j when P_j is complete (p_ready); the softmax of tile j+2 reuses P_b once PV_j is done (p_free).
    const uint32_t idesc_qk = umma_idesc(0), idesc_pv = umma_idesc(1);
    // descriptors are built once; a k-step / stage only adds a constant to the 14-bit start-address field (no carry out:
    // the tiles end below 256 KB), so each MMA costs one add per operand instead of a shift / mask / or chain
    const uint64_t dq = umma_desc(smem_u32(sQ), 16, 1024), dk = umma_desc(smem_u32(sK), 16, 1024),
                   dv = umma_desc(smem_u32(sV), kHalfBytes, 1024);
#ifdef HVA_ATTN_TIMING
    unsigned long long tacc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long tprev = clock64();
#endif
    auto issue_qk = [&](int j) {
      const int s = j % kStagesK, b = j & 1;
      AMARK(0);
      mbar_wait(&B->k_full[s], (j / kStagesK) & 1);
      AMARK(1);
      tc_fence_after();
      const uint64_t dks = dk + (uint64_t)(s * (kTileBytes >> 4));
      const uint32_t d_s = tmem + kColS + b * 128;
      if (elect_one()) {
#pragma unroll
        for (int ks = 0; ks < kD / 16; ++ks) {
          const uint32_t off = ((ks >> 2) * kHalfBytes + (ks & 3) * 32) >> 4;
          mma_ss(d_s, dq + off, dks + off, idesc_qk, ks > 0);
        }
        tc_commit(&B->s_full[b]);
        tc_commit(&B->k_empty[s]);
      }
      __syncwarp();
    };
    mbar_wait(&B->q_full, 0);
    {
      // rows of the Q tile past the end of the group (the loads over-read / repeat rows there) are cleared: their scores, probabilities
      // and output rows are never used, and under the power cap a zero row costs the tensor pipe less than a live one
      const int nval = row1 - row0;
      if (nval < kBM) {
        for (int e = lane; e < (kBM - nval) * 16; e += 32) {
          const int rr = nval + (e >> 4), q = e & 15;
          *reinterpret_cast<uint4*>(sQ + (q >> 3) * kHalfBytes + rr * 128 + ((q & 7) << 4)) = make_uint4(0u, 0u, 0u, 0u);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
      }
    }
    issue_qk(0);
    if (jn > 1) issue_qk(1);
    for (int j = 0; j < jn; ++j) {
      const int s = j % kStagesV, b = j & 1;
      if (j + 2 < jn) {
        AMARK(0);
        mbar_wait(&B->s_free[b], (j >> 1) & 1);
        AMARK(2);
        issue_qk(j + 2);
      }
      AMARK(0);
      mbar_wait(&B->p_ready[b], (j >> 1) & 1);
      AMARK(3);
      mbar_wait(&B->v_full[s], (j / kStagesV) & 1);
      AMARK(4);
      tc_fence_after();
      const int rows_valid = min(kBN, kappa - j * kBN);
      const int ksteps = (rows_valid + 15) >> 4;
      const uint64_t dvs = dv + (uint64_t)(s * (kTileBytes >> 4));
      const uint32_t a_p = tmem + kColP + b * 64;
      if (elect_one()) {
        if (ksteps == 8) {
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) mma_ts(tmem + kColO, a_p + ks * 8, dvs + ks * (2048 >> 4), idesc_pv, (j > 0 || ks > 0));
        } else {
          for (int ks = 0; ks < ksteps; ++ks) mma_ts(tmem + kColO, a_p + ks * 8, dvs + ks * (2048 >> 4), idesc_pv, (j > 0 || ks > 0));
        }
        tc_commit(&B->v_empty[s]);
        tc_commit(&B->p_free[b]);
      }
      __syncwarp();
    }
#ifdef HVA_ATTN_TIMING
    AMARK(0);
    if (p.probe && lane == 0) for (int k = 0; k < 8; ++k) atomicAdd(p.probe + k, tacc[k]);
#endif
  } else if (warp < 8) {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 200;");
    // ===================================================== softmax / correction / epilogue
    // Two sets of 128 threads alternate over the key tiles: set b = warp >> 2 takes the tiles j = b (mod 2), i.e. always
    // the buffers S_b / P_b; thread = one full query row (TMEM lane 32 (warp & 3) + lane) held in 128 registers.  While one
    // set loads and reduces its tile the other one is in the MUFU-bound exponentials.  The two threads of a row share the
    // row's reference exponent through shared memory: decisions are taken in tile order (seq[r] = tiles decided), each
    // thread keeps its own partial row sum relative to the reference it last saw.
    const int b = warp >> 2, r = (warp & 3) * 32 + lane;
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t s_addr = tmem + lane_base + kColS + b * 128, p_addr = tmem + lane_base + kColP + b * 64;
    const float sl2 = p.scale_log2;
    const float2 sl2x2 = make_float2(sl2, sl2);
    const bool row_ok = row0 + r < row1;
    float m_seen = -INFINITY;         // reference (log2 units) the partial sum l2 is relative to: P = 2^(s*scale*log2e - m_ref)
    float2 l2 = make_float2(0.f, 0.f);
    uint32_t v0[32], v1[32], v2[32], v3[32];
    volatile int* seq = B->seq;
    volatile float* mref = B->mref;
#ifdef HVA_ATTN_TIMING
    unsigned long long tacc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long tprev = clock64();
#endif
    // A warp whose 32 rows all lie past the end of the group (the padding of the group's last q-tile: 12 % of all rows at C4) has
    // nothing to compute: its rows of P stay zero (written once per buffer, here, while both are free), and per key tile it only
    // keeps the barrier phases in step.  The kernel runs at the board's power cap, so the exponentials it does not compute and the
    // zero rows the PV MMA multiplies are clock for the valid rows.
    const bool warp_dead = !__any_sync(0xffffffffu, row_ok);
    if (warp_dead) {
      uint32_t z[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) z[i] = 0u;
#pragma unroll
      for (int c = 0; c < 4; ++c) tmem_st16(p_addr + c * 16, z);     // this set's P_b (64 columns); ordered before PV by the set's p_ready arrivals
      tmem_st_wait();
      tc_fence_before();
    }
    for (int j = b; j < jn; j += 2) {
      const int rows_valid = min(kBN, kappa - j * kBN);
      AMARK(0);
      mbar_wait(&B->s_full[b], (j >> 1) & 1);
      AMARK(1);
      if (warp_dead) {
        mbar_arrive(&B->s_free[b]);
        if (j >= 2) mbar_wait(&B->p_free[b], ((j - 2) >> 1) & 1);
        mbar_arrive(&B->p_ready[b]);
        continue;
      }
      tc_fence_after();
      tmem_ld32_nowait(s_addr, v0);
      tmem_ld32_nowait(s_addr + 32, v1);
      tmem_ld32_nowait(s_addr + 64, v2);
      tmem_ld32_nowait(s_addr + 96, v3);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(&B->s_free[b]);          // the row is in registers: the MMA warp may overwrite S_b with QK_{j+2}
      if (rows_valid != kBN) {
#pragma unroll
        for (int i = 0; i < 32; ++i) {     // -inf: key columns past the packed list
          if (i >= rows_valid) v0[i] = 0xff800000u;
          if (32 + i >= rows_valid) v1[i] = 0xff800000u;
          if (64 + i >= rows_valid) v2[i] = 0xff800000u;
          if (96 + i >= rows_valid) v3[i] = 0xff800000u;
        }
      }
      float mx0 = fmaxf(__uint_as_float(v0[0]), __uint_as_float(v0[1])), mx1 = fmaxf(__uint_as_float(v1[0]), __uint_as_float(v1[1]));
      float mx2 = fmaxf(__uint_as_float(v2[0]), __uint_as_float(v2[1])), mx3 = fmaxf(__uint_as_float(v3[0]), __uint_as_float(v3[1]));
#pragma unroll
      for (int i = 2; i < 32; i += 2) {
        mx0 = fmaxf(mx0, fmaxf(__uint_as_float(v0[i]), __uint_as_float(v0[i + 1])));
        mx1 = fmaxf(mx1, fmaxf(__uint_as_float(v1[i]), __uint_as_float(v1[i + 1])));
        mx2 = fmaxf(mx2, fmaxf(__uint_as_float(v2[i]), __uint_as_float(v2[i + 1])));
        mx3 = fmaxf(mx3, fmaxf(__uint_as_float(v3[i]), __uint_as_float(v3[i + 1])));
      }
      const float m_c = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * sl2;
      AMARK(2);
      // reference decisions are sequential in j: wait for the partner's decision on tile j-1 (normally long taken)
      while (seq[r] != j) { }
      __threadfence_block();
      float m_ref = mref[r];
      AMARK(3);
      if (m_ref != m_seen) { const float f0 = ex2(m_seen - m_ref); l2.x *= f0; l2.y *= f0; m_seen = m_ref; }   // m_seen = -inf: l2 = 0
      // the reference only moves when a score exceeds it by > 2^8 (lazy rescale); then O (complete up to PV_{j-1}) is rescaled
      // (rows past the end of the group -- the Q tile over-reads its neighbours -- do not vote: they are never stored, and the
      // bits of the valid rows must not depend on them)
      if (__any_sync(0xffffffffu, row_ok && m_c - m_ref > kRescaleThreshold)) {
        const float m_new = fmaxf(m_ref, m_c);
        const float f = (m_new == m_ref) ? 1.f : ex2(m_ref - m_new);
        l2.x *= f; l2.y *= f;
        if (j > 0) {
          mbar_wait(&B->p_free[b ^ 1], ((j - 1) >> 1) & 1);   // PV_{j-1} complete
          tc_fence_after();
          uint32_t o[16];
#pragma unroll 1
          for (int cc = 0; cc < 8; ++cc) {
            tmem_ld16(tmem + lane_base + kColO + cc * 16, o);
#pragma unroll
            for (int i = 0; i < 16; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
            tmem_st16(tmem + lane_base + kColO + cc * 16, o);
          }
          tmem_st_wait();
          tc_fence_before();
        }
        m_ref = m_new; m_seen = m_new;
        mref[r] = m_new;
      }
      __threadfence_block();
      seq[r] = j + 1;
      AMARK(4);
      if (j >= 2) { mbar_wait(&B->p_free[b], ((j - 2) >> 1) & 1); tc_fence_after(); }   // PV_{j-2} has read P_b
      AMARK(5);
      const float2 nm = make_float2(-m_ref, -m_ref);
      auto exp_chunk = [&](const uint32_t (&vv)[32], int c) {
        uint32_t pk[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const float2 x = __ffma2_rn(make_float2(__uint_as_float(vv[2 * i]), __uint_as_float(vv[2 * i + 1])), sl2x2, nm);
          float2 e;
          if (kPolyPairs > 0 && (i & 7) < kPolyPairs) {
            e = exp2_poly2(x);            // software exponential on the FMA pipe for kPolyPairs of every 8 pairs
          } else {
            e.x = ex2(x.x); e.y = ex2(x.y);
          }
          l2 = __fadd2_rn(l2, e);
          pk[i] = pack_bf16(e.x, e.y);
        }
        tmem_st16(p_addr + c * 16, pk);
      };
      exp_chunk(v0, 0); exp_chunk(v1, 1); exp_chunk(v2, 2); exp_chunk(v3, 3);
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(&B->p_ready[b]);
      AMARK(6);
    }
#ifdef HVA_ATTN_TIMING
    if (p.probe && tid == 0) for (int k = 0; k < 8; ++k) atomicAdd(p.probe + 8 + k, tacc[k]);
#endif
    // final reference of the row, partial sums of the two sets
    if (!warp_dead) while (seq[r] != jn) { }
    __threadfence_block();
    {
      const float m_fin = mref[r];
      if (m_fin != m_seen) { const float f0 = ex2(m_seen - m_fin); l2.x *= f0; l2.y *= f0; }
    }
    B->xch[b][r] = l2.x + l2.y;
    asm volatile("bar.sync 1, 256;" ::: "memory");
    const float l = B->xch[0][r] + B->xch[1][r];
    // epilogue: O / l, bf16, row store with the inverse permutation fused (Eq. 4: O = Pi^{q-1} O'); set b stores columns [64b, 64b+64)
    mbar_wait(&B->p_free[(jn - 1) & 1], ((jn - 1) >> 1) & 1);   // last PV complete
    tc_fence_after();
    const float inv = 1.f / l;
    const int row = row0 + r;
    const bool ok = row < row1;
    size_t orow = 0;
    if (ok) orow = (size_t)base_row + (p.unpermute ? p.perm_q[(size_t)base_row + row] : row);
#pragma unroll 1
    for (int c = 0; c < 2; ++c) {
      uint32_t o[32];
      tmem_ld32(tmem + lane_base + kColO + b * 64 + c * 32, o);
      if (ok) {
        uint4* dst = reinterpret_cast<uint4*>(p.O + orow * kD + b * 64 + c * 32);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          uint4 w;
          w.x = pack_bf16(__uint_as_float(o[8 * q + 0]) * inv, __uint_as_float(o[8 * q + 1]) * inv);
          w.y = pack_bf16(__uint_as_float(o[8 * q + 2]) * inv, __uint_as_float(o[8 * q + 3]) * inv);
          w.z = pack_bf16(__uint_as_float(o[8 * q + 4]) * inv, __uint_as_float(o[8 * q + 5]) * inv);
          w.w = pack_bf16(__uint_as_float(o[8 * q + 6]) * inv, __uint_as_float(o[8 * q + 7]) * inv);
          dst[q] = w;
        }
      }
    }
  } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");   // idle warps of the last warpgroup
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 9) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTmemCols) : "memory");
  }
}

// 2-D map over X[rows, 128] bf16, box = 64 dims x box_rows rows, 128-byte swizzle, OOB rows read as zero.
bool make_map(CUtensorMap* m, const void* base, uint64_t rows, uint32_t box_rows) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[2] = {(cuuint64_t)kD, rows};
  cuuint64_t strides[1] = {(cuuint64_t)kD * 2};
  cuuint32_t box[2] = {64, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

#ifdef HVA_ATTN_TIMING
extern "C" void hva_debug_attn_timing(unsigned long long* dev16) { g_attn_timing = dev16; }
#endif

int hva_attention_tc_launch(const hva_shape* s, float scale, const void* Qp, const void* Kp, const void* Vp,
                            const void* plan, const hva_plan_layout& L, int Nq, int Nk, void* O, int unpermute, int gather_q,
                            cudaStream_t st) {
  if (s->D != kD || s->dtype != HVA_BF16) return HVA_EUNSUPPORTED;
  const int n = s->T * s->H * s->W, BH = s->B * s->heads;
  const uint64_t rows = (uint64_t)BH * n;
  if (rows >= (1ull << 31)) return HVA_EUNSUPPORTED;
  TcMaps maps;
  if (!make_map(&maps.q, Qp, rows, gather_q ? 1 : kBM)) return HVA_ECUDA;
  for (int b = 0; b < kNumBoxes; ++b) {
    if (!make_map(&maps.k[b], Kp, rows, 1u << b)) return HVA_ECUDA;
    if (!make_map(&maps.v[b], Vp, rows, 1u << b)) return HVA_ECUDA;
  }
  const char* b = reinterpret_cast<const char*>(plan);
  TcParams p;
  p.n = n; p.Nq = Nq; p.Nk = Nk; p.run_stride = (int)L.run_stride; p.work_cap = (int)L.work_cap; p.unpermute = unpermute; p.gather_q = gather_q;
  p.scale_log2 = scale * 1.4426950408889634f;
  p.goff = (const int*)(b + L.goff); p.koff = (const int*)(b + L.koff); p.kappa = (const int*)(b + L.kappa);
  p.run_cnt = (const int*)(b + L.run_cnt); p.work_cnt = (const int*)(b + L.work_cnt); p.work = (const int*)(b + L.work);
  p.perm_q = (const int*)(b + L.perm_q); p.runs = (const uint32_t*)(b + L.runs);
  p.O = reinterpret_cast<__nv_bfloat16*>(O);
#ifdef HVA_ATTN_TIMING
  p.probe = g_attn_timing;
#endif
  // the attribute is per device: set on every call (cheap) rather than behind a process-wide flag
  if (cudaFuncSetAttribute(hva_attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemTC) != cudaSuccess)
    return HVA_ECUDA;
  dim3 grid((unsigned)L.work_cap, BH);
  hva_attn_tc_kernel<<<grid, kThreadsTC, kSmemTC, st>>>(maps, p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
