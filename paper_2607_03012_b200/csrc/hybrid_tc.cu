// S4 on the tensor pipe (bf16, D = 128): subset tokens re-assigned against ALL N_c centroids of the cached state
// (DESIGN.md R-H3): a dense m x N_c x D contraction, the one clustering step that is GEMM-shaped.
//
// Same filter-and-refine scheme as cluster_tc.cu: score_v = |mu_v|^2 - 2 x.(hi_v + lo_v) from tcgen05 MMAs with the
// two-term bf16 split of mu; the decision is taken in the exact fp32 direct form among the candidates whose score lies
// within the rigorous error margin of the best one, first minimum in ascending centroid id (R-C1).
//   CTA = 128 subset tokens of one (batch, head): rows gathered into a 128B-swizzled A tile (16-byte coalesced loads)
//   warp 8  TMA producer: centroid tiles of 128 candidates (hi + lo, 64 KB) through a 2-stage ring
//   warp 9  MMA issuer: 16 MMAs per candidate tile into one of two 128-column TMEM score buffers
//   warps 0-7  scan: thread = (token row, half of the tile's columns) keeps the three smallest scores (two with their
//              ids); the halves are merged through shared memory and part 0 decides / refines
#include "common.cuh"
#include "ptx.cuh"
#include "cluster_tc.cuh"

namespace {
using namespace hva_ptx;
using namespace hva_tc_dev;

constexpr int kD = 128, kTok = 128, kCand = 128;
constexpr int kHalf = 128 * 128;                 // one 64-dim half of a 128-row tile
constexpr int kTile = 2 * kHalf;                 // 32 KB
constexpr int kStageBytes = 2 * kTile;           // hi + lo
constexpr int kThreadsS = 320;

struct SubsetTcParams {
  int n, Nc, m, ntiles;
  const __nv_bfloat16* X;
  const int* subset;
  const float* mu;
  const float* musq;
  const int* assign;
  int *oldlab, *newlab;
};

struct __align__(8) SubsetBars {
  uint64_t full[2], smem_empty[2], score_full[2], tmem_free[2];
  uint32_t tmem_base;
  int cmax_bits;
};

struct Top3 {
  float s1, s2, s3;
  int i1, i2;
  // candidates arrive in ascending id: strict '<' keeps the lower id among equal scores
  __device__ __forceinline__ void push(float s, int v) {
    const bool lt1 = s < s1, lt2 = s < s2;
    s3 = fminf(s3, fmaxf(s2, s));
    i2 = lt1 ? i1 : (lt2 ? v : i2);
    s2 = fminf(s2, fmaxf(s1, s));
    i1 = lt1 ? v : i1;
    s1 = fminf(s1, s);
  }
};

__global__ void __launch_bounds__(kThreadsS, 1) hva_subset_assign_tc_kernel(const __grid_constant__ CUtensorMap map_hi,
                                                                            const __grid_constant__ CUtensorMap map_lo,
                                                                            SubsetTcParams p) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int bh = blockIdx.y, i0 = blockIdx.x * kTok;
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  unsigned char* sA = smem;                                  // [2 halves][128 tokens][128 B]
  unsigned char* sB = smem + kTile;                          // [2 stages][hi | lo][2 halves][128 candidates][128 B]
  float* s_c = reinterpret_cast<float*>(sB + 2 * kStageBytes);   // [ntiles * 128] |mu_v|^2, +inf past N_c
  float* s_x = s_c + p.ntiles * kCand;                       // [5][128] part-1 results handed to part 0
  SubsetBars* B = reinterpret_cast<SubsetBars*>(s_x + 5 * kTok);

  if (tid == 0) {
    for (int s = 0; s < 2; ++s) {
      mbar_init(&B->full[s], 1); mbar_init(&B->smem_empty[s], 1);
      mbar_init(&B->score_full[s], 1); mbar_init(&B->tmem_free[s], 256);
    }
    B->cmax_bits = 0;
    mbar_fence_init();
  }
  __syncwarp();
  if (warp == 9) tmem_alloc(&B->tmem_base, 256);
  __syncthreads();
  // gather the subset rows: 16 lanes per row, 16 bytes each (two rows = 512 contiguous-per-row bytes per warp instruction)
  for (int e = tid; e < kTok * 16; e += kThreadsS) {
    const int row = e >> 4, q = e & 15;
    uint4 v = make_uint4(0, 0, 0, 0);
    if (i0 + row < p.m) {
      const size_t tok = (size_t)bh * p.n + p.subset[(size_t)bh * p.m + i0 + row];
      v = __ldg(reinterpret_cast<const uint4*>(p.X + tok * kD) + q);
    }
    *reinterpret_cast<uint4*>(sA + (q >> 3) * kHalf + row * 128 + (((q & 7) ^ (row & 7)) << 4)) = v;
  }
  {
    float cm = 0.f;
    for (int v = tid; v < p.ntiles * kCand; v += kThreadsS) {
      const float c = v < p.Nc ? __ldg(p.musq + (size_t)bh * p.Nc + v) : __int_as_float(0x7f800000);
      s_c[v] = c;
      if (v < p.Nc) cm = fmaxf(cm, c);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cm = fmaxf(cm, __shfl_xor_sync(0xffffffffu, cm, o));
    if (lane == 0) atomicMax(&B->cmax_bits, __float_as_int(cm));     // c >= 0: integer order == float order
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = B->tmem_base;
  const int nt = p.ntiles;

  if (warp == 8) {
    // ===================================================== TMA producer (warp-uniform, one elected lane issues)
    for (int t = 0; t < nt; ++t) {
      const int s = t & 1;
      if (t >= 2) mbar_wait(&B->smem_empty[s], ((t >> 1) - 1) & 1);
      if (elect_one()) {
        unsigned char* dst = sB + s * kStageBytes;
        const int row = bh * p.Nc + t * kCand;     // rows past N_c belong to the next head (masked by s_c = +inf) or read as zero
        mbar_expect_tx(&B->full[s], kStageBytes);
        tma_load_2d(&map_hi, &B->full[s], dst, 0, row);
        tma_load_2d(&map_hi, &B->full[s], dst + kHalf, 64, row);
        tma_load_2d(&map_lo, &B->full[s], dst + kTile, 0, row);
        tma_load_2d(&map_lo, &B->full[s], dst + kTile + kHalf, 64, row);
      }
      __syncwarp();
    }
  } else if (warp == 9) {
    // ===================================================== MMA issuer
    const uint32_t idesc = umma_idesc_bf16(128, 128, 0, 0);
    const uint64_t da = umma_desc(smem_u32(sA), 16, 1024), db = umma_desc(smem_u32(sB), 16, 1024);
    for (int t = 0; t < nt; ++t) {
      const int s = t & 1;
      mbar_wait(&B->full[s], (t >> 1) & 1);
      if (t >= 2) mbar_wait(&B->tmem_free[s], ((t >> 1) - 1) & 1);
      tc_fence_after();
      if (elect_one()) {
        const uint64_t dbs = db + (uint64_t)(s * (kStageBytes >> 4));
#pragma unroll
        for (int ks = 0; ks < kD / 16; ++ks) {
          const uint32_t off = ((ks >> 2) * kHalf + (ks & 3) * 32) >> 4;
          mma_ss(tmem + s * 128, da + off, dbs + off, idesc, ks > 0);
        }
#pragma unroll
        for (int ks = 0; ks < kD / 16; ++ks) {
          const uint32_t off = ((ks >> 2) * kHalf + (ks & 3) * 32) >> 4;
          mma_ss(tmem + s * 128, da + off, dbs + (kTile >> 4) + off, idesc, 1);
        }
        tc_commit(&B->score_full[s]);
        tc_commit(&B->smem_empty[s]);
      }
      __syncwarp();
    }
  } else {
    // ===================================================== scan: thread = (token row r, part h of the tile's columns)
    const int h = warp >> 2, r = (warp & 3) * 32 + lane;
    const uint32_t trow = tmem + ((uint32_t)((warp & 3) * 32) << 16) + h * 64;
    const float kInf = __int_as_float(0x7f800000);
    Top3 top{kInf, kInf, kInf, 0, 0};
    for (int t = 0; t < nt; ++t) {
      const int s = t & 1;
      mbar_wait(&B->score_full[s], (t >> 1) & 1);
      tc_fence_after();
#pragma unroll 1
      for (int c = 0; c < 2; ++c) {
        uint32_t raw[32];
        tmem_ld32(trow + s * 128 + c * 32, raw);
        const int v0 = t * kCand + h * 64 + c * 32;
#pragma unroll
        for (int j = 0; j < 32; j += 4) {
          const float4 c4 = *reinterpret_cast<const float4*>(s_c + v0 + j);
          top.push(fmaf(-2.f, __uint_as_float(raw[j]), c4.x), v0 + j);
          top.push(fmaf(-2.f, __uint_as_float(raw[j + 1]), c4.y), v0 + j + 1);
          top.push(fmaf(-2.f, __uint_as_float(raw[j + 2]), c4.z), v0 + j + 2);
          top.push(fmaf(-2.f, __uint_as_float(raw[j + 3]), c4.w), v0 + j + 3);
        }
      }
      tc_fence_before();
      mbar_arrive(&B->tmem_free[s]);
    }
    // merge the two column halves of a row (part 1 -> part 0); ids of part 0 are not ordered against part 1's, so the
    // merged list only serves as a contender set: the exact comparison below goes by ascending id
    if (h == 1) {
      s_x[r] = top.s1; s_x[kTok + r] = top.s2; s_x[2 * kTok + r] = top.s3;
      s_x[3 * kTok + r] = __int_as_float(top.i1); s_x[4 * kTok + r] = __int_as_float(top.i2);
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (h == 0) {                                 // warp-uniform: warps 0-3 decide for their 32 rows
      const bool valid = i0 + r < p.m;
      const float* mu_b = p.mu + (size_t)bh * p.Nc * kD;
      int lab = 0;
      bool full_scan = false;
      if (valid) {
        const float a1 = s_x[r], a2 = s_x[kTok + r], a3 = s_x[2 * kTok + r];
        const int j1 = __float_as_int(s_x[3 * kTok + r]), j2 = __float_as_int(s_x[4 * kTok + r]);
        top.push(a1, j1); top.push(a2, j2);
        top.s3 = fminf(top.s3, a3);   // a3 >= a2 >= merged s2: it can only displace the third value
        // filter margin (cluster_tc.cu): E <= 2 kEpsDot |x| |mu|max + rounding of |mu|^2 and of the fma
        float xsq = 0.f;
        __nv_bfloat162 acc[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[j] = __floats2bfloat162_rn(0.f, 0.f);
#pragma unroll 8
        for (int q = 0; q < 16; ++q) {
          const uint4 w = *x_chunk(sA, kHalf, r, q);
          const __nv_bfloat162 x0 = *reinterpret_cast<const __nv_bfloat162*>(&w.x), x1 = *reinterpret_cast<const __nv_bfloat162*>(&w.y),
                               x2 = *reinterpret_cast<const __nv_bfloat162*>(&w.z), x3 = *reinterpret_cast<const __nv_bfloat162*>(&w.w);
          acc[0] = __hfma2(x0, x0, acc[0]); acc[1] = __hfma2(x1, x1, acc[1]);
          acc[2] = __hfma2(x2, x2, acc[2]); acc[3] = __hfma2(x3, x3, acc[3]);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) xsq += __low2float(acc[j]) + __high2float(acc[j]);
        xsq *= 1.125f;
        const float c_max = __int_as_float(B->cmax_bits);
        const float xm = sqrtf(xsq * c_max);
        const float margin = 2.f * (2.f * kEpsDot * xm + 6e-7f * (c_max + 2.f * xm));
        lab = top.i1;
        if (!(top.s2 > top.s1 + margin)) {
          if (top.s3 > top.s1 + margin) {       // exactly two contenders: exact direct form, lower id first, strict '<'
            const int lo = min(top.i1, top.i2), hi = max(top.i1, top.i2);
            const float dlo = direct_dist(sA, kHalf, r, mu_b + (size_t)lo * kD), dhi = direct_dist(sA, kHalf, r, mu_b + (size_t)hi * kD);
            lab = dhi < dlo ? hi : lo;
          } else {
            full_scan = true;                   // three or more within the margin (rare)
          }
        }
      }
      // exact scan of every centroid for such a token, shared by the warp: lane = candidates v = lane, lane + 32, ...
      unsigned need = __ballot_sync(0xffffffffu, full_scan);
      while (need) {
        const int src = __ffs(need) - 1;
        need &= need - 1;
        const int rr = __shfl_sync(0xffffffffu, r, src);
        float best = kInf;
        int bi = 0x7fffffff;
        for (int v = lane; v < p.Nc; v += 32) {
          const float dd = direct_dist(sA, kHalf, rr, mu_b + (size_t)v * kD);
          if (dd < best) { best = dd; bi = v; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {      // (distance, id) lexicographic minimum == first minimum in ascending id
          const float ob = __shfl_xor_sync(0xffffffffu, best, o);
          const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
          if (ob < best || (ob == best && oi < bi)) { best = ob; bi = oi; }
        }
        if (lane == src) lab = bi;
      }
      if (valid) {
        const size_t o = (size_t)bh * p.m + i0 + r;
        p.newlab[o] = lab;
        p.oldlab[o] = p.assign[(size_t)bh * p.n + p.subset[o]];
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 9) { tc_fence_after(); tmem_dealloc(tmem, 256); }
}

bool make_map2(CUtensorMap* m, const void* base, uint64_t rows) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[2] = {(cuuint64_t)kD, rows};
  cuuint64_t strides[1] = {(cuuint64_t)kD * 2};
  cuuint32_t box[2] = {64, (cuuint32_t)kCand};
  cuuint32_t estr[2] = {1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

bool hva_subset_tc_supported(int D, int dtype, int Nc) { return dtype == HVA_BF16 && D == kD && Nc <= 4096; }

int hva_subset_assign_tc_launch(int BH, int n, int Nc, int m, const void* X, const int* subset, const float* mu, const void* mu_hi,
                                const void* mu_lo, const float* musq, const int* assign, int* oldlab, int* newlab, cudaStream_t st) {
  CUtensorMap map_hi, map_lo;
  if (!make_map2(&map_hi, mu_hi, (uint64_t)BH * Nc) || !make_map2(&map_lo, mu_lo, (uint64_t)BH * Nc)) return HVA_ECUDA;
  SubsetTcParams p{n, Nc, m, (Nc + kCand - 1) / kCand, reinterpret_cast<const __nv_bfloat16*>(X), subset, mu, musq, assign, oldlab, newlab};
  const size_t smem = 1024 + kTile + 2 * kStageBytes + sizeof(float) * ((size_t)p.ntiles * kCand + 5 * kTok) + sizeof(SubsetBars) + 16;
  if (smem > 227 * 1024) return HVA_EUNSUPPORTED;
  if (cudaFuncSetAttribute(hva_subset_assign_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return HVA_ECUDA;
  hva_subset_assign_tc_kernel<<<dim3((m + kTok - 1) / kTok, BH), kThreadsS, smem, st>>>(map_hi, map_lo, p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
