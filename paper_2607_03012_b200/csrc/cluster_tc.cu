// S1 (+ the per-cell part of S2) on the tensor pipe (bf16 inputs, D = 128): assignment step of 3D local-window
// k-means and the per-(cell, slot) partial centroid sums (Alg. 2 lines 14-21, l.367-381; Eq. 5 l.81; Eq. 6 l.97).
//
// The direct form sum_c (x_c - mu_c)^2 on CUDA cores is ALU-bound (round 1, first ncu capture: 6.5 % of DRAM peak).
// Here the 27.D dot products leave the FP32 pipe:
//   score_v = |mu_v|^2 - 2 x.mu_v  ( = d^2_v - |x|^2 ),   x.mu_v = x.hi_v + x.lo_v
// with mu split into two bf16 terms (hi = RN(mu), lo = RN(mu - hi); |mu - hi - lo| <= 2^-18 |mu|), so
// both products are exact in the MMA and only the fp32 accumulation rounds.  Per tile (a home cell, or a t-slab of it):
//   TMA   one 5-D box brings the tile's k_t x k_h x k_w tokens (rows of 256 B) into a 128B-swizzled
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
//
// Round 2 organisation: ONE persistent CTA per SM (640 threads) that keeps NT tiles in flight in a ring of token slots
// (5 x 30 KB at the 3x5x8 cells), each with its own TMEM score columns, slot table and mbarriers; CTA b takes the tiles
// b, b + gridDim.x, ...  Roles (nothing but mbarriers between them, no block barrier in the steady state):
//   warps 0-11   NW = 3 scan warpgroups, tile q goes to group q mod NW: thread = token row = TMEM lane: scan / refine /
//                label store / one-hot write into the group's own one-hot tile
//   warps 12-15  epilogue warpgroup, every tile in order: thread = feature dim = TMEM lane: partial-row stores
//   warp  16     loader: draws the tiles, waits for a free token slot and centroid buffer, issues the six TMA boxes
//   warp  17     MMA 1 when the tile's boxes have landed
//   warp  18     MMA 2 when the tile's one-hot arrivals are in
//   warp  19     slot tables (centroid ids, |mu|^2, zeroed counts) of the tile
// (a single warp runs dependent integer code at one instruction per 4-8 clk: every role loop keeps its slot index and barrier
// parity incrementally -- a runtime q % NT is ~40 instructions -- and no role does two long-latency things per tile)
// Round 1's kernel ran these steps in line in four independent 128-thread CTAs per SM (9.5 K clk per tile, of which the
// scan threads waited for TMA / MMA round trips and block barriers more than half; now: profiles/r2_assign_phases.md): the same four tiles
// per SM were in flight, but a warp that waits now has another tile to work on.
#include "common.cuh"
#include "ptx.cuh"
#include "cluster_tc.cuh"
#include <algorithm>

namespace {
using namespace hva_ptx;
using namespace hva_tc_dev;

constexpr int kD = 128;
constexpr int kMaxNW = 3;                         // scan warpgroups
constexpr int kMaxNT = 8;                         // pipeline slots / token buffers
constexpr int kEpiWarp0 = 4 * kMaxNW;             // first warp of the epilogue warpgroup
constexpr int kLoadWarp = kEpiWarp0 + 4, kMma1Warp = kLoadWarp + 1, kMma2Warp = kLoadWarp + 2, kTableWarp = kLoadWarp + 3;
constexpr int kThreads = 32 * (kTableWarp + 1);   // 640
constexpr uint32_t kTmemCols = 512;               // one CTA per SM: all of it

struct AssignTcParams {
  HvaGrid g;
  const float* mu;     // [BH, Nc, D] fp32 centroids (exact refine)
  const float* musq;   // [BH, Nc] |mu|^2 fp32
  float* part;         // [BH, Nc(cells), nwin, D]
  int* part_cnt;       // [BH, Nc(cells), nwin]
  int* assign;         // [BH, n] or null
  float* lowe;         // [BH, n] or null
  float* xsq;          // [BH, n] upper bound of |x|^2 (only scales the filter margin): written when xsq_mode == 1, read when 2
  int xsq_mode;        // 0 compute, 1 compute + store, 2 load (the bound is the same in every iteration of a call)
  int npad;            // window candidates padded to the MMA N granule (16)
  int rows_a;          // tile tokens padded to the MMA K granule (16 rows)
  int csplit, ct;      // a cell of more than 128 tokens is split along t into csplit tiles of ct time slices
  uint32_t m_khw, m_kw, m_whw, m_ww;   // fast_div multipliers for k_h k_w, k_w, w_h w_w, w_w
  int NT, NB, NW;      // token buffers, centroid buffers, scan warpgroups (= one-hot tiles)
  int NS;              // pipeline slots (TMEM columns, slot tables, barriers) >= NT: a token buffer is free once MMA 2 has read it, its
                       // TMEM columns and tables only after the epilogue
  int cols;            // TMEM columns per token slot
  int one_pass;        // 2 npad <= 256: one MMA pass over [hi; lo] stacked as 2 npad score columns (the token tile is read once)
  int coop;            // cooperative scan: every tile is scanned by all three groups, each taking a share of the window's 32-candidate chunks
  unsigned long long d_khw, d_kw, d_cs, d_kt;   // fast_div64 multipliers of the tile decode: K_h K_w, K_w, csplit, K_t
  int n_items;         // K_w * K_h * K_t * BH * csplit tiles: CTA b takes tiles b, b + gridDim.x, ...
  float* probe;        // instrumented instantiation: max |score_tc - score_exact| / (|x| max|mu|)
};

// per token slot: the tile's header (written by the loader / the table warp) and the slot's barriers
struct __align__(8) TileSlot {
  uint64_t hdr_ready;    // loader -> table warp, MMA 1 warp: header written                       (1 arrival)
  uint64_t table_ready;  // table warp -> scan group, epilogue group, MMA 2 warp: tables written   (32 arrivals)
  uint64_t full;         // TMA: tokens and centroids landed                                       (expect-tx)
  uint64_t mma_done;     // MMA 1 complete -> scan group; centroid buffer free -> loader           (commit)
  uint64_t onehot;       // scan group -> MMA 2 warp: scores read, one-hot written                 (128 arrivals)
  uint64_t sum_done;     // MMA 2 complete -> epilogue group; one-hot tile free -> scan group      (commit)
  uint64_t free_;        // epilogue group -> loader: the slot (tokens, TMEM columns, tables) is free (128 arrivals)
  int item;              // tile id, or -1: no more work
  int uw, uh, ut, bh, chunk;
  uint32_t cmax;         // max |mu_v|^2 over the window (bits of a non-negative float)
  int pad_;
};

struct __align__(8) AssignTcShared {
  TileSlot slot[kMaxNT];
  uint32_t tmem_base;
};

__device__ __noinline__ float direct_dist_probe(const unsigned char* sA, int half_bytes, int r, const float* mu) {
  return direct_dist(sA, half_bytes, r, mu);
}

// Diagnostic build (-DHVA_ASSIGN_TIMING, instrumented instantiation only): lane 0 of the first warp of every role adds its clocks
// per phase to probe[16 + 8 role + phase]  (bench.py --report assign-phases); roles: 0 scan group 0, 1 epilogue, 2 loader, 3 MMA 1, 4 MMA 2
#ifdef HVA_ASSIGN_TIMING
#define CMARK(k) do { if (kProbe && tmark) { long long _t = clock64(); tacc[k] += (unsigned)(_t - tprev); tprev = _t; } } while (0)
#define CFLUSH(role) do { if (kProbe && tmark) for (int _k = 0; _k < 8; ++_k) atomicAdd(p.probe + 16 + 8 * (role) + _k, (float)tacc[_k]); } while (0)
// event trace of CTA 0 (-DHVA_ASSIGN_TRACE as well): probe[64 + 16 q + ev] = clocks since the CTA's start (first 48 tiles)
#ifdef HVA_ASSIGN_TRACE
#define TRACE(ev, q) do { if (kProbe && blockIdx.x == 0 && (lane == 0) && ((warp & 3) == 0 || warp >= kLoadWarp) && (q) < 48) p.probe[64 + 16 * (q) + (ev)] = (float)(clock64() - tstart); } while (0)
#else
#define TRACE(ev, q) do { } while (0)
#endif
#else
#define TRACE(ev, q) do { } while (0)
#define CMARK(k) do { } while (0)
#define CFLUSH(role) do { } while (0)
#endif

// x / d for 0 <= x, x * d < 2^32 by one multiply-high (m = ceil(2^32 / d); d == 1 is passed as m = 0)
__device__ __forceinline__ int fast_div(int x, uint32_t m) { return m ? (int)__umulhi((uint32_t)x, m) : x; }
// x / d for every 0 <= x < 2^31 and d >= 1 by one 64-bit multiply-high (m = ceil(2^64 / d); d == 1 is passed as m = 0):
// m d = 2^64 + e with e < d, so x m / 2^64 = x / d + x e / (d 2^64), and the excess is below 2^-32 < 1 / d
__device__ __forceinline__ int fast_div64(int x, unsigned long long m) { return m ? (int)__umul64hi((unsigned long long)(uint32_t)x, m) : x; }

__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void named_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// kProbe = true is the instrumented instantiation behind hva_cluster_ex(probe != NULL) (tests: observed filter error);
// the product instantiation carries none of that code.
// kVar selects a specialisation of the scan code: 0 = everything decided at run time (and the only one that carries the
// cooperative wide-window scan); 1 = windows of at most 32 candidates, one MMA pass, labels only; 2 = the same with the Lowe
// ratio.  The instrumented instantiation is generic.  (The 27-candidate path is sensitive to what is compiled next to it: a
// score more instructions on its rare refine branch cost 7 %.)
template <bool kProbe, int kVar>
__global__ void __launch_bounds__(kThreads, 1) hva_assign_tc_kernel(const __grid_constant__ CUtensorMap map_x,
                                                                 const __grid_constant__ CUtensorMap map_hi,
                                                                 const __grid_constant__ CUtensorMap map_lo, AssignTcParams p) {
  const HvaGrid& g = p.g;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int ctok = p.ct * g.kh * g.kw, nwin = g.nwin, npad = p.npad;   // token rows of a tile
  const int half_a = p.rows_a * 128, half_b = npad * 128;
  const int NT = p.NT, NB = p.NB, NW = p.NW, NS = p.NS;
  const bool one_pass = kVar ? true : (bool)p.one_pass;

  // Shared memory (offsets from a 1024-byte aligned base):
  //   sA  [NT][2 halves][rows_a][128 B]           token slots (A of MMA 1, K-major SW128; A of MMA 2, MN-major)
  //   sB  [NB][2 halves][hi | lo][npad][128 B]    window centroids, K-major SW128 (hi and lo rows of a half are contiguous:
  //                                               one B operand of 2 npad rows)
  //   sP  [NW][2 halves][npad][128 B]             one one-hot tile P^T per scan group (rows = slots, K = tokens; B of MMA 2).
  //       Zero except for one element per token row; a thread clears the element it set for its previous tile and sets the new one
  //   per token slot: |mu_v|^2 [npad] f32, token count per slot [npad] i32, centroid id of window slot [npad] u16; slots
  // MMA 1 reads 128 token rows: rows past the tile alias whatever follows inside the allocation and only feed TMEM
  // lanes nobody reads.
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  unsigned char* sA_all = smem;
  unsigned char* sB_all = sA_all + (size_t)NT * 2 * half_a;
  unsigned char* sP_all = sB_all + (size_t)NB * 4 * half_b;
  float* s_c_all = reinterpret_cast<float*>(sP_all + (size_t)NW * 2 * half_b);
  int* s_cnt_all = reinterpret_cast<int*>(s_c_all + NS * npad);
  uint16_t* s_u_all = reinterpret_cast<uint16_t*>(s_cnt_all + NS * npad);
  AssignTcShared* SH = reinterpret_cast<AssignTcShared*>(reinterpret_cast<unsigned char*>(s_u_all + NS * npad) + ((8 - ((NS * npad * 2) & 7)) & 7));

  // cooperative scan only: (s1, s2) of every group and row, two parities; contender word of every chunk and row
  float2* coop_ex = reinterpret_cast<float2*>(reinterpret_cast<unsigned char*>(SH + 1) + ((16 - (sizeof(AssignTcShared) & 15)) & 15));
  uint32_t* coop_m = reinterpret_cast<uint32_t*>(coop_ex + 2 * 3 * 128);

  if (warp == kLoadWarp) tmem_alloc(&SH->tmem_base, kTmemCols);

  // tile -> (cell coordinates, time split, batch*head)
  struct Tile { int uw, uh, ut, bh, chunk; };
  auto decode = [&](int item) {
    Tile t;
    const int khw = g.Kw * g.Kh, z = fast_div64(item, p.d_khw), r = item - z * khw;
    t.uh = fast_div64(r, p.d_kw); t.uw = r - t.uh * g.Kw;
    const int zz = fast_div64(z, p.d_cs);
    t.chunk = z - zz * p.csplit;
    t.bh = fast_div64(zz, p.d_kt); t.ut = zz - t.bh * g.Kt;
    return t;
  };
  if (tid == 0) {
    for (int i = 0; i < NS; ++i) {
      TileSlot* S = &SH->slot[i];
      mbar_init(&S->hdr_ready, 1); mbar_init(&S->table_ready, 32); mbar_init(&S->full, 1); mbar_init(&S->mma_done, 1);
      mbar_init(&S->onehot, 128); mbar_init(&S->sum_done, 1); mbar_init(&S->free_, 128);
    }
    mbar_fence_init();
  }
  // token rows ctok .. rows_a-1 of every slot take part in MMA 2 (K granule 16) with zero weight: they must be finite; TMA never
  // writes them
  for (int i = tid; i < NT * (p.rows_a - ctok) * 16; i += kThreads) {
    const int s = i / ((p.rows_a - ctok) * 16), j = i - s * (p.rows_a - ctok) * 16;
    const int r = ctok + (j >> 4), q = j & 15;
    *reinterpret_cast<uint4*>(sA_all + (size_t)s * 2 * half_a + (q >> 3) * half_a + r * 128 + ((q & 7) << 4)) = make_uint4(0, 0, 0, 0);
  }
  // rows nwin .. npad-1 of the four centroid tiles (hi | lo per 64-dim half) of every buffer are never written by TMA: zero them
  // once, so that the pad columns of the score MMA are exactly 0
  for (int i = tid; i < NB * 4 * (npad - nwin) * 8; i += kThreads) {
    const int k = i / ((npad - nwin) * 8), j = i - k * (npad - nwin) * 8;     // k = buffer * 4 + quarter
    *reinterpret_cast<uint4*>(sB_all + (size_t)k * half_b + nwin * 128 + j * 16) = make_uint4(0, 0, 0, 0);
  }
  for (int i = tid; i < NW * (2 * half_b) / 16; i += kThreads) reinterpret_cast<uint4*>(sP_all)[i] = make_uint4(0, 0, 0, 0);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = SH->tmem_base;
  const float kInf = __int_as_float(0x7f800000);
#ifdef HVA_ASSIGN_TIMING
  unsigned tacc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  long long tprev = clock64();
  const bool tmark = lane == 0 && (warp == 0 || warp == kEpiWarp0 || warp >= kLoadWarp);
  const long long tstart = tprev;
  int tq = 0;
#endif

  // register file: the CTA gets 640 x 96 at launch; setmaxnreg only moves registers inside that pool: the controller warpgroup
  // gives back 128 x (96 - 48), the epilogue group 128 x (96 - 56), the three scan groups take 384 x (120 - 96) of those 11264
  if (warp >= kLoadWarp) asm volatile("setmaxnreg.dec.sync.aligned.u32 48;");   // the four controller warps form one warpgroup
  if (warp == kLoadWarp) {
    // ================================================================ loader
    const uint32_t tile_bytes = (uint32_t)(2 * ctok * 128 + 4 * nwin * 128);
    // the tokens stream through L2 once per pass (evict first); the centroids and the partial rows are what should stay there
    const uint64_t pol_x = l2_policy_evict_first(), pol_mu = l2_policy_evict_last();
    int item = blockIdx.x;                   // (the grid never exceeds n_items)
    int n_term = 0;
    int i = 0, jb = 0, ib = 0, ia = 0, ix = 0;   // slot / centroid buffer / token buffer of tile q; slots of tiles q - NB, q - NT
    uint32_t par = 0, parb = 0, parx = 0;        // parity of the slot's barriers for tile q / q - NB / q - NT
    for (int q = 0; n_term < NW; ++q) {
      TileSlot* S = &SH->slot[i];
      CMARK(0);
      if (q >= NS) mbar_wait(&S->free_, par ^ 1u);          // the slot's previous tile has left the pipeline
      CMARK(1);
      TRACE(0, q);
      Tile t{0, 0, 0, 0, 0};
      if (item >= 0) t = decode(item);
      if (lane == 0) { S->item = item; S->uw = t.uw; S->uh = t.uh; S->ut = t.ut; S->bh = t.bh; S->chunk = t.chunk; mbar_arrive(&S->hdr_ready); }
      if (item >= 0) {
        if (q >= NB) {                       // the centroid buffer is free once MMA 1 of the tile NB tiles back has read it
          CMARK(2);
          mbar_wait(&SH->slot[ib].mma_done, parb);
          CMARK(3);
          if (++ib == NS) { ib = 0; parb ^= 1u; }
        }
        if (q >= NT) {                       // the token buffer is free once MMA 2 of the tile NT tiles back has read it
          mbar_wait(&SH->slot[ix].sum_done, parx);
          if (++ix == NS) { ix = 0; parx ^= 1u; }
        }
        unsigned char* sA = sA_all + (size_t)ia * 2 * half_a;
        unsigned char* sBhi = sB_all + (size_t)jb * 4 * half_b;
        unsigned char* sBlo = sBhi + half_b;
        const int st = hva_win_start(t.ut, g.wt, g.Kt), sh = hva_win_start(t.uh, g.wh, g.Kh), sw = hva_win_start(t.uw, g.ww, g.Kw);
        const int t0 = t.ut * g.kt + t.chunk * p.ct;
        if (elect_one()) {
          mbar_expect_tx(&S->full, tile_bytes);
          tma_load_5d_hint(&map_hi, &S->full, sBhi, 0, sw, sh, st, t.bh, pol_mu);
          tma_load_5d_hint(&map_hi, &S->full, sBhi + 2 * half_b, 64, sw, sh, st, t.bh, pol_mu);
          tma_load_5d_hint(&map_lo, &S->full, sBlo, 0, sw, sh, st, t.bh, pol_mu);
          tma_load_5d_hint(&map_lo, &S->full, sBlo + 2 * half_b, 64, sw, sh, st, t.bh, pol_mu);
          tma_load_5d_hint(&map_x, &S->full, sA, 0, t.uw * g.kw, t.uh * g.kh, t0, t.bh, pol_x);
          tma_load_5d_hint(&map_x, &S->full, sA + half_a, 64, t.uw * g.kw, t.uh * g.kh, t0, t.bh, pol_x);
        }
        __syncwarp();
        CMARK(4);
        TRACE(1, q);
        // static round robin: every tile costs the same within ~1 %, so a device counter buys nothing here -- and ptxas turns a
        // uniform-address atom into a warp-aggregated sequence whose shuffle waits for the round trip right behind it (1 K clk per tile)
        item += (int)gridDim.x;
        if (item >= p.n_items) item = -1;
        CMARK(5);
      } else {
        ++n_term;                            // one terminator header per scan group
      }
      if (++i == NS) { i = 0; par ^= 1u; }
      if (++jb == NB) jb = 0;
      if (++ia == NT) ia = 0;
    }
    CFLUSH(2);
  } else if (warp == kMma1Warp) {
    // ================================================================ MMA 1 (scores) as soon as a tile's boxes have landed
    const uint32_t idesc1 = umma_idesc_bf16(128, (uint32_t)(one_pass ? 2 * npad : npad), 0, 0);
    const uint32_t ha = (uint32_t)half_a >> 4, hb2 = (uint32_t)(2 * half_b) >> 4;
    int i = 0, jb = 0, ia = 0;
    uint32_t par = 0;
    for (;;) {
      TileSlot* S = &SH->slot[i];
      CMARK(0);
      mbar_wait(&S->hdr_ready, par);
      CMARK(1);
      if (S->item < 0) break;
      mbar_wait(&S->full, par);
      CMARK(3);
      TRACE(2, tq);
      tc_fence_after();
      // descriptors in uniform registers; a k-step only adds a constant to the start-address field
      const uint64_t da = umma_desc(smem_u32(sA_all + (size_t)ia * 2 * half_a), 16, 1024);
      const uint64_t dhi = umma_desc(smem_u32(sB_all + (size_t)jb * 4 * half_b), 16, 1024), dlo = dhi + ((uint32_t)half_b >> 4);
      const uint32_t d_t = tmem + (uint32_t)(i * p.cols);
      if (elect_one()) {
#pragma unroll
        for (int ks = 0; ks < kD / 16; ++ks)
          mma_ss(d_t, da + ((ks >> 2) * ha + (ks & 3) * 2), dhi + ((ks >> 2) * hb2 + (ks & 3) * 2), idesc1, ks > 0);
        if (!one_pass) {
#pragma unroll
          for (int ks = 0; ks < kD / 16; ++ks)
            mma_ss(d_t, da + ((ks >> 2) * ha + (ks & 3) * 2), dlo + ((ks >> 2) * hb2 + (ks & 3) * 2), idesc1, 1);
        }
        tc_commit(&S->mma_done);
      }
      __syncwarp();
      CMARK(4);
      TRACE(3, tq);
#ifdef HVA_ASSIGN_TIMING
      ++tq;
#endif
      if (++i == NS) { i = 0; par ^= 1u; }
      if (++jb == NB) jb = 0;
      if (++ia == NT) ia = 0;
    }
    CFLUSH(3);
  } else if (warp == kTableWarp) {
    // ================================================================ slot tables of every tile (lane = window slot); forwards the terminators
    int i = 0, n_term = 0;
    uint32_t par = 0;
    while (n_term < NW) {
      TileSlot* S = &SH->slot[i];
      mbar_wait(&S->hdr_ready, par);
      if (S->item < 0) {
        ++n_term;
      } else {
        float* s_c = s_c_all + i * npad; uint16_t* s_u = s_u_all + i * npad; int* s_cnt = s_cnt_all + i * npad;
        const int ut = S->ut, uh = S->uh, uw = S->uw, bh = S->bh;
        const int st = hva_win_start(ut, g.wt, g.Kt), sh = hva_win_start(uh, g.wh, g.Kh), sw = hva_win_start(uw, g.ww, g.Kw);
        float cm = 0.f;
        for (int v = lane; v < npad; v += 32) {
          int u = 0;
          float c = kInf;     // pad slot: its score column is exactly 0 (pad rows of the centroid tiles are zero), so score = +inf
          if (v < nwin) {
            const int dt = fast_div(v, p.m_whw), r = v - dt * g.wh * g.ww, dh = fast_div(r, p.m_ww), dw = r - dh * g.ww;
            u = ((st + dt) * g.Kh + (sh + dh)) * g.Kw + (sw + dw);
            c = __ldg(p.musq + (size_t)bh * g.Nc + u);
            cm = fmaxf(cm, c);
          }
          s_u[v] = (uint16_t)u; s_c[v] = c; s_cnt[v] = 0;
        }
        const uint32_t m = __reduce_max_sync(0xffffffffu, __float_as_uint(cm));   // |mu|^2 >= 0: uint order == float order
        if (lane == 0) S->cmax = m;
      }
      mbar_arrive(&S->table_ready);
      if (++i == NS) { i = 0; par ^= 1u; }
    }
  } else if (warp == kMma2Warp) {
    // ================================================================ MMA 2: z^T[dim, slot] = sum_token x[token, dim] P^T[slot, token]
    // (Alg. 2 line 20): A = the token tile read MN-major (M = 128 feature dims), B = the one-hot tile of the tile's scan group,
    // D overwrites the tile's score columns; TMEM lane = feature dim
    const uint32_t idesc2 = umma_idesc_bf16(128, (uint32_t)npad, 1, 0);
    const uint32_t hb = (uint32_t)half_b >> 4;
    const int ksteps2 = p.rows_a >> 4;
    int i = 0, jw = 0, ia = 0;
    uint32_t par = 0;
    for (;;) {
      TileSlot* S = &SH->slot[i];
      CMARK(0);
      mbar_wait(&S->table_ready, par);
      CMARK(1);
      if (S->item < 0) break;
      mbar_wait(&S->onehot, par);          // every score read, every one-hot element (and its proxy fence) written
      CMARK(2);
      TRACE(10, tq);
      tc_fence_after();
      const uint64_t dx = umma_desc(smem_u32(sA_all + (size_t)ia * 2 * half_a), half_a, 1024);
      const uint64_t dp = umma_desc(smem_u32(sP_all + (size_t)jw * 2 * half_b), 16, 1024);
      const uint32_t d_t = tmem + (uint32_t)(i * p.cols);
      if (elect_one()) {
        if (ksteps2 == 8) {
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) mma_ss(d_t, dx + ks * (2048 >> 4), dp + ((ks >> 2) * hb + (ks & 3) * 2), idesc2, ks > 0);
        } else {
          for (int ks = 0; ks < ksteps2; ++ks) mma_ss(d_t, dx + ks * (2048 >> 4), dp + ((ks >> 2) * hb + (ks & 3) * 2), idesc2, ks > 0);
        }
        tc_commit(&S->sum_done);
      }
      __syncwarp();
      CMARK(3);
      TRACE(11, tq);
#ifdef HVA_ASSIGN_TIMING
      ++tq;
#endif
      if (++i == NS) { i = 0; par ^= 1u; }
      if (++jw == NW) jw = 0;
      if (++ia == NT) ia = 0;
    }
    CFLUSH(4);
  } else if (warp >= kEpiWarp0) {
    // ================================================================ epilogue group: thread = feature dim; a warp stores 32 consecutive
    // floats of a partial row (coalesced)
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    const int dim = tid - kEpiWarp0 * 32;
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    int i = 0;
    uint32_t par = 0;
    for (;;) {
      TileSlot* S = &SH->slot[i];
      CMARK(0);
      mbar_wait(&S->table_ready, par);
      CMARK(1);
      if (S->item < 0) break;
      const int* s_cnt = s_cnt_all + i * npad;
      const int cell = (S->ut * g.Kh + S->uh) * g.Kw + S->uw;
      const size_t pbase = (((size_t)S->bh * g.Nc + cell) * p.csplit + S->chunk) * nwin;
      mbar_wait(&S->sum_done, par);        // all 128 one-hot arrivals are in, MMA 2 has finished
      CMARK(2);
      TRACE(12, tq);
      tc_fence_after();
      for (int v = dim; v < nwin; v += 128) p.part_cnt[pbase + v] = s_cnt[v];
      float* prow = p.part + pbase * kD + dim;
      const uint32_t trow = tmem + lane_base + (uint32_t)(i * p.cols);
      for (int v0 = 0; v0 < nwin; v0 += 32) {
        // non-empty slots of this chunk as one ballot word: the stores below are then a bit test + STG with an immediate offset
        const unsigned nz = __ballot_sync(0xffffffffu, v0 + lane < nwin && s_cnt[v0 + lane] > 0);
        float* pr = prow + (size_t)v0 * kD;
        if (kVar == 0 && __popc(nz) <= 16) {
          // wide windows: most of a chunk's slots are empty, and TMEM reads (64 B per clock and SM) are what the kernel runs out of:
          // only the non-empty columns are read, four single-column loads in flight
          unsigned m = nz;
          while (m) {
            uint32_t val[4] = {0u, 0u, 0u, 0u};
            int js[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              js[k] = m ? __ffs(m) - 1 : -1;
              m &= m - 1;                    // 0 stays 0
              if (js[k] >= 0) tmem_ld1_nowait(trow + v0 + js[k], val[k]);
            }
            tmem_ld_wait4(val);
#pragma unroll
            for (int k = 0; k < 4; ++k)
              if (js[k] >= 0) pr[js[k] * kD] = __uint_as_float(val[k]);
          }
          continue;
        }
        uint32_t raw[32];
        tmem_ld32(trow + v0, raw);
#pragma unroll
        for (int j = 0; j < 32; ++j)
          if ((nz >> j) & 1u) pr[j * kD] = __uint_as_float(raw[j]);
      }
      tc_fence_before();     // the TMEM reads are complete (wait::ld): the slot may be reused
      mbar_arrive(&S->free_);
      CMARK(3);
      TRACE(13, tq);
#ifdef HVA_ASSIGN_TIMING
      ++tq;
#endif
      if (++i == NS) { i = 0; par ^= 1u; }
    }
    CFLUSH(1);
  } else {
    // ================================================================ scan groups: thread = token row of the tile == TMEM lane
    asm volatile("setmaxnreg.inc.sync.aligned.u32 120;");
    // Cooperative scan (wide windows: shared memory holds ONE one-hot tile, so one tile at a time is in the scan stage): all three
    // groups work on every tile, group w on its share of the window's 32-candidate chunks; they exchange their two smallest scores,
    // mark the contenders of their chunks against the common threshold, and group 0 decides, stores and writes the one-hot tile.
    const bool coop = kVar == 0 && p.coop != 0;
    if (warp < 4 * NW || coop) {
    const int w = warp >> 2;                 // group: tiles q = w, w + NW, ... (cooperative: every tile)
    const int step = coop ? 1 : NW;
    const int nchunk = (nwin + 31) >> 5;
    int c_lo = 0, c_hi = nchunk;             // chunks of this group
    if (coop) {                              // group 0 also runs the decision part of every tile: the smallest share
      const int n0 = max(1, nchunk >> 2), n1 = (nchunk - n0) >> 1;
      c_lo = w == 0 ? 0 : (w == 1 ? n0 : n0 + n1);
      c_hi = w == 0 ? n0 : (w == 1 ? n0 + n1 : nchunk);
    }
    const int v_lo = 32 * c_lo, v_hi = min(nwin, 32 * c_hi);
    uint32_t tpar = 0;                       // parity of the exchange buffer (cooperative scan)
    const int li = tid & 127;
    const int ldt = fast_div(li, p.m_khw), lr = li - ldt * g.kh * g.kw, ldh = fast_div(lr, p.m_kw), ldw = lr - ldh * g.kw;
    const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
    const bool want2 = kVar ? kVar == 2 : p.lowe != nullptr;
    const bool single_chunk = kVar ? true : nwin <= 32;
    unsigned char* sP = sP_all + (size_t)(coop ? 0 : w) * 2 * half_b;
    uint32_t prev_p = 0;      // shared-space address of the one-hot element set for the group's previous tile (0: none)
    int i = coop ? 0 : w, pi = 0, ia = i;    // slot of the group's tile / of its previous tile, token buffer (NW < NT <= NS)
    uint32_t par = 0, ppar = 0;
    for (bool first_tile = true;; first_tile = false) {
      TileSlot* S = &SH->slot[i];
      CMARK(0);
      mbar_wait(&S->table_ready, par);
      CMARK(1);
#ifdef HVA_ASSIGN_TIMING
      if (first_tile) tq = w;
#endif
      TRACE(4, tq);
      if (S->item < 0) break;
      struct { uint32_t cmax; } T{S->cmax};
      const float* s_c = s_c_all + i * npad; const uint16_t* s_u = s_u_all + i * npad; int* s_cnt = s_cnt_all + i * npad;
      const unsigned char* sA = sA_all + (size_t)ia * 2 * half_a;
      const uint32_t trow = tmem + lane_base + (uint32_t)(i * p.cols);
      const int uw = S->uw, uh = S->uh, ut = S->ut, bh = S->bh, chunk = S->chunk;
      const int dt0 = chunk * p.ct;                        // first time slice of this tile inside the cell
      // ---- token geometry; an upper bound of |x|^2 and the filter margin
      int lab = -1;
      size_t tok = 0;
      {
        const int t = ut * g.kt + dt0 + ldt, h = uh * g.kh + ldh, w = uw * g.kw + ldw;
        if (li < ctok && dt0 + ldt < g.kt && t < g.T && h < g.H && w < g.W) { lab = 0; tok = (size_t)bh * g.n + (size_t)(t * g.H + h) * g.W + w; }
      }
      const bool valid = lab == 0;
      const float c_max = __uint_as_float(T.cmax);
      float xsq = 0.f;
      if (p.xsq_mode == 2) {
        if (valid) xsq = __ldg(p.xsq + tok);     // in flight while the tile lands
        mbar_wait(&S->full, par);
      } else {
        mbar_wait(&S->full, par);
        // |x|^2 only scales the margin: packed bf16 FMAs (4 x 2 accumulators of 16 non-negative terms each: relative
        // error < 16 * 2^-8), inflated by 1/8 so that it is an upper bound
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
          if (p.xsq_mode == 1 && (!coop || w == 0)) p.xsq[tok] = xsq;
        }
      }
      CMARK(2);
      TRACE(5, tq);
      mbar_wait(&S->mma_done, par);
      CMARK(3);
      TRACE(6, tq);
      tc_fence_after();
      // score error E <= 2 kEpsDot |x| |mu| (+ rounding of |mu|^2 and of the fma: 6e-7 (|mu|^2 + 2|x||mu|)); candidates within
      // 2E of the decisive score are contenders
      const float xm = sqrtf(xsq * c_max);
      const float margin = 2.f * (2.f * kEpsDot * xm + 6e-7f * (c_max + 2.f * xm));

      float sv[32];
      // scores of one 32-candidate chunk: sv[j] = |mu_v|^2 - 2 x.mu_v, +inf past the window
      auto load_scores = [&](int v0) {
#pragma unroll
        for (int h = 0; h < 32; h += 16) {
          uint32_t raw[16], rlo[16];
          if (one_pass) {      // x.hi in columns [0, npad), x.lo in [npad, 2 npad)
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
      float s1 = kInf, s2 = kInf, r1 = kInf, r2 = kInf;
      for (int v0 = v_lo; v0 < v_hi; v0 += 32) {
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
      if (coop) {       // the two smallest scores of the whole window from the three groups' shares
        float2* ex = coop_ex + tpar * (3 * 128);
        ex[w * 128 + li] = make_float2(s1, s2);
        named_bar_sync(1, 384);
#pragma unroll
        for (int k = 1; k < 3; ++k) {
          const float2 o = ex[(w + k >= 3 ? w + k - 3 : w + k) * 128 + li];
          s2 = fminf(fminf(s2, o.y), fmaxf(s1, o.x));
          s1 = fminf(s1, o.x);
        }
      }
      const float thr = (want2 ? s2 : s1) + margin;     // s2 = +inf (single candidate): every candidate is a contender
      // pass 2: contenders = candidates with score <= thr.  A single contender (without the Lowe ratio) is the direct-form
      // argmin; otherwise the exact direct form decides among them, ascending candidate id, strict '<'  (R-C1)
      float best = kInf, second = kInf;
      const float* mu_b = p.mu + (size_t)bh * g.Nc * kD;
      int n_cont = 0, first = 0;
      uint32_t cand0 = 0;
      for (int v0 = v_lo; v0 < v_hi; v0 += 32) {
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
        if (coop) coop_m[(v0 >> 5) * 128 + li] = cand;
      }
      if (coop) {
        tc_fence_before();                  // this group's score reads are complete (MMA 2 overwrites the columns after group 0's arrival)
        __threadfence_block();
        if (w != 0) {                       // groups 1 and 2 are done with the tile
          named_bar_arrive(2, 384);
          i += 1; if (i >= NS) { i = 0; par ^= 1u; }
          ia += 1; if (ia >= NT) ia = 0;
          tpar ^= 1u;
          continue;
        }
        named_bar_sync(2, 384);
        n_cont = 0; first = 0;
        for (int c = 0; c < nchunk; ++c) {
          const uint32_t m = coop_m[c * 128 + li];
          if (n_cont == 0 && m) first = 32 * c + __ffs(m) - 1;
          n_cont += __popc(m);
        }
      }
      const bool refine = valid && (want2 || n_cont > 1);
      if (valid && !refine) lab = first;
      if (__any_sync(0xffffffffu, refine)) {            // tcgen05.ld is warp-collective: the chunk loop stays warp-uniform
        for (int v0 = 0; v0 < nwin; v0 += 32) {
          uint32_t cand = cand0;
          if (coop) {
            cand = coop_m[(v0 >> 5) * 128 + li];
          } else if (!single_chunk) {
            load_scores(v0);
            cand = 0;
#pragma unroll
            for (int j = 0; j < 32; ++j)
              if (sv[j] <= thr) cand |= 1u << j;
            cand &= nwin - v0 >= 32 ? 0xffffffffu : (1u << (nwin - v0)) - 1u;
          }
          if (!refine) cand = 0;
          if (want2) {
            // every lane refines (Lowe ratio): each evaluates its own contenders, fully unrolled tree form; this code runs for
            // every tile of such a pass and stays in the instruction cache
            while (cand) {
              const int v = v0 + __ffs(cand) - 1;
              cand &= cand - 1;
              const float dd = direct_dist(sA, half_a, li, mu_b + (size_t)s_u[v] * kD);
              if (dd < best) { second = best; best = dd; lab = v; }
              else if (dd < second) second = dd;
            }
          } else {
            // rare (a near tie in one lane of ~1 warp in 20): the WARP evaluates the lane's contenders, lane j holding partial sum j
            // of the tree form and the halving tree running as an xor butterfly -- the same bits as direct_dist() in ~60 rolled
            // instructions.  (The unrolled per-lane form is ~1 K instructions that are never in the instruction cache when a lone
            // lane needs them: 14 K clk per occurrence, during which the in-order tile pipeline behind the tile stands still.)
            uint32_t need = __ballot_sync(0xffffffffu, cand != 0);
            while (need) {
              const int src = __ffs(need) - 1;
              need &= need - 1;
              uint32_t cm = __shfl_sync(0xffffffffu, cand, src);
              const int row = (li & ~31) | src, qc = lane >> 1;
              const uint2 xr = *reinterpret_cast<const uint2*>(sA + (qc >> 3) * half_a + row * 128 + (((qc & 7) ^ (row & 7)) << 4) + (lane & 1) * 8);
              const float x0 = __uint_as_float(xr.x << 16), x1 = __uint_as_float(xr.x & 0xffff0000u);
              const float x2 = __uint_as_float(xr.y << 16), x3 = __uint_as_float(xr.y & 0xffff0000u);
#pragma unroll 1
              while (cm) {
                const int v = v0 + __ffs(cm) - 1;
                cm &= cm - 1;
                const float4 m = __ldg(reinterpret_cast<const float4*>(mu_b + (size_t)s_u[v] * kD) + lane);
                float pp = hva_sq4(x0, x1, x2, x3, m);
#pragma unroll
                for (int o = 16; o >= 1; o >>= 1) pp += __shfl_xor_sync(0xffffffffu, pp, o);
                if (lane == src) {
                  if (pp < best) { second = best; best = pp; lab = v; }
                  else if (pp < second) second = pp;
                }
              }
            }
          }
        }
      }
      if (valid) {
        if (p.assign) p.assign[tok] = s_u[lab];
        if (p.lowe) {   // rho = d1/d2, unsquared (Eq. 6); single candidate -> 0; d2 == 0 -> 1 (R-H1)
          const float rho = (second == kInf) ? 0.f : (second > 0.f ? sqrtf(best / second) : 1.f);
          p.lowe[tok] = rho;
        }
      }
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
      // ---- one-hot tile P^T[slot, token] = 1 and the slot counts.  The group's one-hot tile is free once MMA 2 of the group's
      // previous tile has read it; the element set for that tile goes back to zero first.
      CMARK(4);
      TRACE(7, tq);
      if (!first_tile) mbar_wait(&SH->slot[pi].sum_done, ppar);
      CMARK(5);
      TRACE(8, tq);
      if (prev_p) asm volatile("st.shared.u16 [%0], %1;" ::"r"(prev_p), "h"((unsigned short)0) : "memory");
      prev_p = 0;
      if (lab >= 0) {
        prev_p = smem_u32(sP) + (uint32_t)((li >> 6) * half_b + lab * 128 + (((((li & 63) >> 3) ^ (lab & 7))) << 4) + (li & 7) * 2);
        asm volatile("st.shared.u16 [%0], %1;" ::"r"(prev_p), "h"((unsigned short)0x3f80) : "memory");   // bf16 1.0
        atomicAdd(&s_cnt[lab], 1);     // (a warp-wide match.any to combine equal labels first costs more than the conflicts)
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      tc_fence_before();
      mbar_arrive(&S->onehot);
      CMARK(6);
      TRACE(9, tq);
#ifdef HVA_ASSIGN_TIMING
#ifdef HVA_ASSIGN_TRACE
      if (kProbe && blockIdx.x == 0 && lane == 0 && (warp & 3) != 0 && tq < 48) p.probe[64 + 16 * 48 + 4 * tq + (warp & 3)] = (float)(clock64() - tstart);
      { const int _nr = __popc(__ballot_sync(0xffffffffu, refine)) * 100 + __reduce_max_sync(0xffffffffu, n_cont);
        if (kProbe && blockIdx.x == 0 && lane == 0 && (warp & 3) != 0 && tq < 48) p.probe[64 + 16 * 48 + 4 * 48 + 4 * tq + (warp & 3)] = (float)_nr; }
#endif
      tq += NW;
#endif
      pi = i; ppar = par;
      i += step;
      if (i >= NS) { i -= NS; par ^= 1u; }
      ia += step;
      if (ia >= NT) ia -= NT;
      tpar ^= 1u;
    }
    CFLUSH(0);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kLoadWarp) { tc_fence_after(); tmem_dealloc(tmem, kTmemCols); }
}

// shared memory of a configuration (NT token slots, NB centroid buffers, NW one-hot tiles)
// exchange area of the cooperative scan: [2 parities][3 groups][128 rows] (s1, s2) + [8 chunks][128 rows] contender words
constexpr size_t kCoopBytes = 2 * 3 * 128 * 8 + 8 * 128 * 4;
size_t assign_tc_smem(int npad, int rows_a, int NT, int NB, int NW, int NS, int coop = 0) {
  const size_t half_a = (size_t)rows_a * 128, half_b = (size_t)npad * 128;
  size_t bytes = (size_t)NT * 2 * half_a + (size_t)NB * 4 * half_b + (size_t)NW * 2 * half_b;
  // MMA 1 reads 128 token rows of its A operand: keep the over-read of the last slot inside the allocation
  bytes = std::max(bytes, (size_t)(NT - 1) * 2 * half_a + half_a + 16384);
  bytes += (size_t)NS * npad * (sizeof(float) + sizeof(int) + sizeof(uint16_t)) + 8 + sizeof(AssignTcShared) + 16;
  if (coop) bytes += kCoopBytes + 16;
  return bytes + 1024;
}

// the largest pipeline that fits 227 KB of shared memory and 512 TMEM columns: three scan groups if possible
bool assign_tc_config(int npad, int rows_a, int cols, int* NT, int* NB, int* NW, int* NS, int* coop) {
  const int ns = std::min(kMaxNT, (int)kTmemCols / cols);      // pipeline slots: as many as TMEM holds
  for (int nw = kMaxNW; nw >= 1; --nw)
    for (int nb = 2; nb >= 1; --nb)
      for (int nt = ns; nt >= nw + 1; --nt) {
        if (nt <= nb) continue;
        // one scan group only (wide windows): the two idle groups join in, if the exchange area fits as well
        const int co = nw == 1 && npad > 32 && assign_tc_smem(npad, rows_a, nt, nb, nw, ns, 1) <= 227 * 1024;
        if (assign_tc_smem(npad, rows_a, nt, nb, nw, ns, co) <= 227 * 1024) { *NT = nt; *NB = nb; *NW = nw; *NS = ns; *coop = co; return true; }
      }
  return false;
}

}  // namespace

bool hva_assign_tc_supported(const HvaGrid& g, int D, int dtype) {
  if (!(dtype == HVA_BF16 && D == kD && g.kh * g.kw <= 128 && g.nwin <= 256 && g.Nc < 65536 && g.kt <= 256 && g.kh <= 256 &&
        g.kw <= 256 && g.wt <= 256 && g.wh <= 256 && g.ww <= 256))
    return false;
  const int ctok = hva_assign_tc_slices(g) * g.kh * g.kw, npad = (g.nwin + 15) & ~15;
  int NT, NB, NW, NS, coop;
  return assign_tc_config(npad, (ctok + 15) & ~15, 2 * npad <= 256 ? 2 * npad : npad, &NT, &NB, &NW, &NS, &coop);
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
  a->probe = probe;
  a->ct = hva_assign_tc_slices(g);
  a->csplit = (g.kt + a->ct - 1) / a->ct;
  const int ctok = a->ct * g.kh * g.kw;
  a->npad = (g.nwin + 15) & ~15;
  a->rows_a = (ctok + 15) & ~15;
  a->one_pass = 2 * a->npad <= 256;
  a->cols = a->one_pass ? 2 * a->npad : a->npad;
  if (!assign_tc_config(a->npad, a->rows_a, a->cols, &a->NT, &a->NB, &a->NW, &a->NS, &a->coop)) return HVA_EUNSUPPORTED;
  a->smem = assign_tc_smem(a->npad, a->rows_a, a->NT, a->NB, a->NW, a->NS, a->coop);
  if ((long long)g.Kw * g.Kh * g.Kt * BH * a->csplit > 0x7fffffffLL) return HVA_EUNSUPPORTED;
  if (!make_map5(&a->map_x, X, BH, g.T, g.H, g.W, a->ct, g.kh, g.kw)) return HVA_ECUDA;
  if (!make_map5(&a->map_hi, mu_hi, BH, g.Kt, g.Kh, g.Kw, g.wt, g.wh, g.ww)) return HVA_ECUDA;
  if (!make_map5(&a->map_lo, mu_lo, BH, g.Kt, g.Kh, g.Kw, g.wt, g.wh, g.ww)) return HVA_ECUDA;
  const void* kerns[4] = {(const void*)hva_assign_tc_kernel<true, 0>, (const void*)hva_assign_tc_kernel<false, 0>,
                          (const void*)hva_assign_tc_kernel<false, 1>, (const void*)hva_assign_tc_kernel<false, 2>};
  for (int k = probe ? 0 : 1; k < (probe ? 1 : 4); ++k)
    if (cudaFuncSetAttribute(kerns[k], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)a->smem) != cudaSuccess) return HVA_ECUDA;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return HVA_ECUDA;
  a->grid = sms;         // one persistent CTA per SM
  return HVA_OK;
}

int hva_assign_tc_launch(const HvaAssignTc& a, const HvaGrid& g, int BH, const float* mu, const float* musq, float* part,
                         int* part_cnt, int* assign, float* lowe, float* xsq, int xsq_mode, int* counter, float* probe, cudaStream_t st) {
  auto magic = [](int d) -> uint32_t { return d <= 1 ? 0u : (uint32_t)(((1ull << 32) + d - 1) / d); };
  auto magic64 = [](int d) -> unsigned long long { return d <= 1 ? 0ull : ~0ull / (unsigned long long)d + 1ull; };
  AssignTcParams p{g, mu, musq, part, part_cnt, assign, lowe, xsq, xsq ? xsq_mode : 0, a.npad, a.rows_a, a.csplit, a.ct, magic(g.kh * g.kw),
                   magic(g.kw), magic(g.wh * g.ww), magic(g.ww), a.NT, a.NB, a.NW, a.NS, a.cols, a.one_pass, a.coop, magic64(g.Kw * g.Kh), magic64(g.Kw),
                   magic64(a.csplit), magic64(g.Kt), g.Kw * g.Kh * g.Kt * BH * a.csplit, probe};
  (void)counter;
  if (a.probe != (probe != nullptr)) return HVA_EINVAL;
  const int grid = std::min(a.grid, p.n_items);
  const bool special = a.one_pass && g.nwin <= 32;
  if (probe) hva_assign_tc_kernel<true, 0><<<grid, kThreads, a.smem, st>>>(a.map_x, a.map_hi, a.map_lo, p);
  else if (!special) hva_assign_tc_kernel<false, 0><<<grid, kThreads, a.smem, st>>>(a.map_x, a.map_hi, a.map_lo, p);
  else if (!lowe) hva_assign_tc_kernel<false, 1><<<grid, kThreads, a.smem, st>>>(a.map_x, a.map_hi, a.map_lo, p);
  else hva_assign_tc_kernel<false, 2><<<grid, kThreads, a.smem, st>>>(a.map_x, a.map_hi, a.map_lo, p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
