// S9 (+S10), tensor-core variant for bf16, D = 128, 128x128 tiles (sm_100a only):
// block-sparse FlashAttention over the plan's packed key runs (Eq. 4 l.56; packed key
// blocks l.109; union masks Eq. 8 l.115).
//
// One CTA per (group, q-tile) work item.  Warp roles:
//   warps 0-3  softmax / correction / epilogue: thread i owns query row i == TMEM lane i
//   warp  4    TMA producer: Q tile once, then per packed key tile the K and V rows of the group's
//              key runs, as power-of-two-height boxes of a 128B-swizzled 2-D tensor map, packed
//              back to back in the stage buffer (exact packing across cluster boundaries)
//   warp  5    TMEM allocator + single-thread tcgen05.mma issuer
// Two CTAs are resident per SM (96 KB smem, 256 TMEM columns each): one CTA's softmax overlaps the other's MMAs.
// Per key tile j:  S_j = Q K_j^T (SS MMA, K-major operands, fp32 accumulators in TMEM)
//                  P_j = exp2(S_j*scale*log2e - m) written back over S_j as bf16 (tcgen05.st)
//                  O  += P_j V_j (TS MMA: A = P from TMEM, B = V from smem, MN-major)
// with lazy (thresholded) rescaling of O in TMEM, 1/l normalisation and the inverse permutation
// fused into the epilogue's row stores.
#include "common.cuh"
#include "ptx.cuh"
#include <cstdlib>

namespace {
using namespace hva_ptx;

constexpr int kBM = 128, kBN = 128, kD = 128;
constexpr int kHalfBytes = 128 * 128;          // one 64-dim half of a 128-row tile: 128 rows x 128 B
constexpr int kTileBytes = 2 * kHalfBytes;     // 32 KB
constexpr int kStages = 1;                     // one K and one V buffer per CTA: two CTAs share an SM
constexpr int kThreadsTC = 192;
constexpr int kNumBoxes = 8;                   // box heights 1,2,4,...,128
constexpr uint32_t kTmemCols = 256;            // S (P aliased over it) + O; two CTAs fit the SM's 512 columns
constexpr uint32_t kColS = 0, kColO = 128;
constexpr float kRescaleThreshold = 8.0f;      // log2 units

struct TcMaps {
  CUtensorMap q;
  CUtensorMap k[kNumBoxes];
  CUtensorMap v[kNumBoxes];
};

struct TcParams {
  int n, Nq, Nk, run_stride, work_cap, unpermute;
  float scale_log2;
  const int *goff, *koff, *kappa, *run_cnt, *work_cnt, *work, *perm_q;
  const uint32_t* runs;
  __nv_bfloat16* O;
};

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

struct __align__(8) TcBarriers {
  uint64_t q_full, k_full[kStages], k_empty[kStages], v_full[kStages], v_empty[kStages], s_full, p_ready, o_done;
  uint32_t tmem_base;
};

constexpr size_t kSmemTC = 1024 + kTileBytes * (1 + 2 * kStages) + sizeof(TcBarriers);

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

__device__ __forceinline__ void emit_boxes(const CUtensorMap* maps, uint64_t* bar, unsigned char* stage, int grow, int dst, int len) {
#pragma unroll 1
  for (int b = kNumBoxes - 1; b >= 0; --b) {
    const int h = 1 << b;
    if (len & h) {
      tma_load_2d(maps + b, bar, stage + dst * 128, 0, grow);
      tma_load_2d(maps + b, bar, stage + kHalfBytes + dst * 128, 64, grow);
      grow += h; dst += h;
    }
  }
}

__device__ __forceinline__ void load_tile(RunWalker& w, const CUtensorMap* maps, uint64_t* bar, unsigned char* stage,
                                          int base_row, int rows_valid, int rows_load) {
  int dst = 0;
  while (dst < rows_valid) {
    while (w.used == w.len) { ++w.r; w.load(); }
    int seg = min(w.len - w.used, rows_valid - dst);
    emit_boxes(maps, bar, stage, base_row + w.row0 + w.used, dst, seg);
    w.used += seg; dst += seg;
  }
  if (rows_load > rows_valid)   // ragged last tile: round up to the MMA K granule with finite over-read rows
    emit_boxes(maps, bar, stage, base_row + w.row0 + w.used, dst, rows_load - rows_valid);
}

__global__ void __launch_bounds__(kThreadsTC, 2) hva_attn_tc_kernel(const __grid_constant__ TcMaps maps, TcParams p) {
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

  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  unsigned char* sQ = smem;
  unsigned char* sK = smem + kTileBytes;
  unsigned char* sV = smem + kTileBytes * (1 + kStages);
  TcBarriers* B = reinterpret_cast<TcBarriers*>(smem + kTileBytes * (1 + 2 * kStages));

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
    for (int s = 0; s < kStages; ++s) {
      mbar_init(&B->k_full[s], 1); mbar_init(&B->k_empty[s], 1);
      mbar_init(&B->v_full[s], 1); mbar_init(&B->v_empty[s], 1);
    }
    mbar_init(&B->s_full, 1); mbar_init(&B->p_ready, 128);
    mbar_init(&B->o_done, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 5) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&B->tmem_base)), "r"(kTmemCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = B->tmem_base;

  if (warp == 4) {
    // ===================================================== TMA producer
    if (lane == 0) {
      mbar_expect_tx(&B->q_full, kTileBytes);
      tma_load_2d(&maps.q, &B->q_full, sQ, 0, base_row + row0);
      tma_load_2d(&maps.q, &B->q_full, sQ + kHalfBytes, 64, base_row + row0);
      RunWalker wk{p.runs + ((size_t)bh * p.Nq + g) * p.run_stride, p.koff + (size_t)bh * (p.Nk + 1),
                   p.run_cnt[(size_t)bh * p.Nq + g], 0, 0, 0, 0};
      wk.load();
      RunWalker wv = wk;
      for (int j = 0; j < jn; ++j) {
        const int s = j % kStages, use = j / kStages;
        const int rows_valid = min(kBN, kappa - j * kBN);
        const int rows_load = rows_valid == kBN ? kBN : (rows_valid + 15) & ~15;
        if (use > 0) mbar_wait(&B->k_empty[s], (use - 1) & 1);
        mbar_expect_tx(&B->k_full[s], rows_load * 256);
        load_tile(wk, maps.k, &B->k_full[s], sK + s * kTileBytes, base_row, rows_valid, rows_load);
        if (use > 0) mbar_wait(&B->v_empty[s], (use - 1) & 1);
        mbar_expect_tx(&B->v_full[s], rows_load * 256);
        load_tile(wv, maps.v, &B->v_full[s], sV + s * kTileBytes, base_row, rows_valid, rows_load);
      }
    }
  } else if (warp == 5) {
    // ===================================================== MMA issuer (one thread)
    if (lane == 0) {
      const uint32_t idesc_qk = umma_idesc(0), idesc_pv = umma_idesc(1);
      const uint32_t q_addr = smem_u32(sQ), k_addr = smem_u32(sK), v_addr = smem_u32(sV);
      auto issue_qk = [&](int j) {
        const int s = j % kStages;
        mbar_wait(&B->k_full[s], (j / kStages) & 1);
        tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < kD / 16; ++ks) {
          const uint32_t off = (ks >> 2) * kHalfBytes + (ks & 3) * 32;
          mma_ss(tmem + kColS, umma_desc(q_addr + off, 16, 1024), umma_desc(k_addr + s * kTileBytes + off, 16, 1024), idesc_qk, ks > 0);
        }
        tc_commit(&B->s_full);
        tc_commit(&B->k_empty[s]);
      };
      mbar_wait(&B->q_full, 0);
      issue_qk(0);
      for (int j = 0; j < jn; ++j) {
        const int s = j % kStages;
        mbar_wait(&B->p_ready, j & 1);
        mbar_wait(&B->v_full[s], (j / kStages) & 1);
        tc_fence_after();
        const int rows_valid = min(kBN, kappa - j * kBN);
        const int ksteps = (rows_valid + 15) >> 4;
        for (int ks = 0; ks < ksteps; ++ks)
          mma_ts(tmem + kColO, tmem + kColS + ks * 8, umma_desc(v_addr + s * kTileBytes + ks * 2048, kHalfBytes, 1024), idesc_pv,
                 (j > 0 || ks > 0));
        tc_commit(&B->v_empty[s]);
        tc_commit(&B->o_done);
        if (j + 1 < jn) issue_qk(j + 1);   // S is aliased by P_j: issue order after PV(j) keeps the tensor pipe in order
      }
    }
  } else {
    // ===================================================== softmax / correction / epilogue (thread = row)
    const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
    const float sl2 = p.scale_log2;
    const float2 sl2x2 = make_float2(sl2, sl2);
    float m_ref = -INFINITY;          // reference exponent (log2 units) of the row: P = 2^(s*scale*log2e - m_ref)
    float2 l2 = make_float2(0.f, 0.f);
    uint32_t v[32];
    for (int j = 0; j < jn; ++j) {
      const uint32_t s_addr = tmem + lane_base + kColS;
      const int rows_valid = min(kBN, kappa - j * kBN);
      mbar_wait(&B->s_full, j & 1);
      tc_fence_after();
      // One pass over S, 32 columns at a time: chunk max -> (rarely) move the reference -> exponentials -> P over S.
      // The reference only moves when a score exceeds it by > 2^8 (lazy rescale); then l, the P chunks of this tile already
      // written and O (complete: the commit of S_j covers PV_{j-1}) are rescaled.
#pragma unroll 1
      for (int c = 0; c < 4; ++c) {
        tmem_ld32(s_addr + c * 32, v);
        if (rows_valid != kBN) {
#pragma unroll
          for (int i = 0; i < 32; ++i)
            if (c * 32 + i >= rows_valid) v[i] = 0xff800000u;   // -inf: key columns past the packed list
        }
        float mx0 = fmaxf(__uint_as_float(v[0]), __uint_as_float(v[1])), mx1 = fmaxf(__uint_as_float(v[2]), __uint_as_float(v[3]));
#pragma unroll
        for (int i = 4; i < 32; i += 4) {
          mx0 = fmaxf(mx0, fmaxf(__uint_as_float(v[i]), __uint_as_float(v[i + 1])));
          mx1 = fmaxf(mx1, fmaxf(__uint_as_float(v[i + 2]), __uint_as_float(v[i + 3])));
        }
        const float m_c = fmaxf(mx0, mx1) * sl2;
        if (__any_sync(0xffffffffu, m_c - m_ref > kRescaleThreshold)) {   // warp-uniform
          const float m_new = fmaxf(m_ref, m_c);
          const float f = (m_new == m_ref) ? 1.f : ex2(m_ref - m_new);
          l2.x *= f; l2.y *= f;
          tmem_st_wait();
          for (int cc = 0; cc < c; ++cc) {          // P chunks of this tile written against the old reference
            uint32_t pk[16];
            tmem_ld16(s_addr + cc * 16, pk);
#pragma unroll
            for (int i = 0; i < 16; ++i)
              pk[i] = pack_bf16(__uint_as_float(pk[i] << 16) * f, __uint_as_float(pk[i] & 0xffff0000u) * f);
            tmem_st16(s_addr + cc * 16, pk);
          }
          if (j > 0) {
            mbar_wait(&B->o_done, (j - 1) & 1);
            tc_fence_after();
            uint32_t o[32];
#pragma unroll 1
            for (int cc = 0; cc < 4; ++cc) {
              tmem_ld32(tmem + lane_base + kColO + cc * 32, o);
#pragma unroll
              for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
              tmem_st32(tmem + lane_base + kColO + cc * 32, o);
            }
          }
          m_ref = m_new;
        }
        const float2 nm = make_float2(-m_ref, -m_ref);
        uint32_t pk[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const float2 x = __ffma2_rn(make_float2(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1])), sl2x2, nm);
          float2 e;
          if ((i & 3) == 3) {
            e = exp2_poly2(x);            // 1 pair in 4 on the FMA pipe: the MUFU rate (16/clk/SM) equals the MMA time of a tile
          } else {
            e.x = ex2(x.x); e.y = ex2(x.y);
          }
          l2 = __fadd2_rn(l2, e);
          pk[i] = pack_bf16(e.x, e.y);
        }
        tmem_st16(s_addr + c * 16, pk);
      }
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(&B->p_ready);
    }
    const float l = l2.x + l2.y;
    // epilogue: O / l, bf16, row store with the inverse permutation fused (Eq. 4: O = Pi^{q-1} O')
    mbar_wait(&B->o_done, (jn - 1) & 1);
    tc_fence_after();
    const float inv = 1.f / l;
    const int row = row0 + tid;
    const bool ok = row < row1;
    size_t orow = 0;
    if (ok) orow = (size_t)base_row + (p.unpermute ? p.perm_q[(size_t)base_row + row] : row);
#pragma unroll 1
    for (int c = 0; c < 4; ++c) {
      tmem_ld32(tmem + lane_base + kColO + c * 32, v);
      if (ok) {
        uint4* dst = reinterpret_cast<uint4*>(p.O + orow * kD + c * 32);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          uint4 o;
          o.x = pack_bf16(__uint_as_float(v[8 * q + 0]) * inv, __uint_as_float(v[8 * q + 1]) * inv);
          o.y = pack_bf16(__uint_as_float(v[8 * q + 2]) * inv, __uint_as_float(v[8 * q + 3]) * inv);
          o.z = pack_bf16(__uint_as_float(v[8 * q + 4]) * inv, __uint_as_float(v[8 * q + 5]) * inv);
          o.w = pack_bf16(__uint_as_float(v[8 * q + 6]) * inv, __uint_as_float(v[8 * q + 7]) * inv);
          dst[q] = o;
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 5) {
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

int hva_attention_tc_launch(const hva_shape* s, float scale, const void* Qp, const void* Kp, const void* Vp,
                            const void* plan, const hva_plan_layout& L, int Nq, int Nk, void* O, int unpermute,
                            cudaStream_t st) {
  if (s->D != kD || s->dtype != HVA_BF16) return HVA_EUNSUPPORTED;
  const int n = s->T * s->H * s->W, BH = s->B * s->heads;
  const uint64_t rows = (uint64_t)BH * n;
  if (rows >= (1ull << 31)) return HVA_EUNSUPPORTED;
  TcMaps maps;
  if (!make_map(&maps.q, Qp, rows, kBM)) return HVA_ECUDA;
  for (int b = 0; b < kNumBoxes; ++b) {
    if (!make_map(&maps.k[b], Kp, rows, 1u << b)) return HVA_ECUDA;
    if (!make_map(&maps.v[b], Vp, rows, 1u << b)) return HVA_ECUDA;
  }
  const char* b = reinterpret_cast<const char*>(plan);
  TcParams p;
  p.n = n; p.Nq = Nq; p.Nk = Nk; p.run_stride = (int)L.run_stride; p.work_cap = (int)L.work_cap; p.unpermute = unpermute;
  p.scale_log2 = scale * 1.4426950408889634f;
  p.goff = (const int*)(b + L.goff); p.koff = (const int*)(b + L.koff); p.kappa = (const int*)(b + L.kappa);
  p.run_cnt = (const int*)(b + L.run_cnt); p.work_cnt = (const int*)(b + L.work_cnt); p.work = (const int*)(b + L.work);
  p.perm_q = (const int*)(b + L.perm_q); p.runs = (const uint32_t*)(b + L.runs);
  p.O = reinterpret_cast<__nv_bfloat16*>(O);
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(hva_attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemTC) != cudaSuccess)
      return HVA_ECUDA;
    attr_set = true;
  }
  dim3 grid((unsigned)L.work_cap, BH);
  hva_attn_tc_kernel<<<grid, kThreadsTC, kSmemTC, st>>>(maps, p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
