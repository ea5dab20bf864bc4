// S6 on the tensor pipe: the pairwise key-overlap of Alg. 1 lines 9-12 for ALL pairs of groups at once.
//   kappa(A u B) = kappa(A) + kappa(B) - I[A][B],   I[A][B] = sum_j chi_j(A) chi_j(B) s^k_j        (Eq. 8 l.115-117)
// I = X Y^T with X = chi (0/1) and Y = chi . diag(s^k): a dense N_q x N_q x N_k contraction.  The operands are exact in bf16
// (0/1; s^k split in base 256: s = t_0 + 256 t_1 + 65536 t_2, every digit < 256 has 8 significant bits), every product and
// every fp32 partial sum is an integer < 2^24, so the MMA result is the exact integer -- the merge plan stays bit-exact.
// CTA = 128 groups A x up to 512 groups B of one (batch, head): per 64-key chunk the threads expand the bit-packed chi
// rows into 128B-swizzled K-major tiles, one thread issues tcgen05.mma 128x128x16 (4 k-steps per chunk and column block
// and digit), accumulators in TMEM; the epilogue adds the digits and stores int32.
#include "common.cuh"
#include "ptx.cuh"

namespace {
using namespace hva_ptx;

constexpr int kTileB = 128 * 128;      // one 128-row x 64-key bf16 tile (128 B per row)
constexpr int kThreadsG = 256;

struct InterParams {
  int Nq, Nk, Wd, Nqp;               // Nqp = N_q rounded up to 128 (row pitch of I)
  const uint32_t* chi;               // [BH, Nq, Wd] bit-packed key sets
  const int* sizes_k;                // [BH, Nk]
  const int* nterms;                 // [BH] base-256 digits needed for max_j s^k_j (1..3)
  int* inter;                        // [BH, Nqp, Nqp]: I[i][j] for the i-th group of side 1 (rows) and the j-th group of side 0 (columns)
  const int* list;                   // [BH, Nq]: the round's alive groups of side 1 ascending from the front, of side 0 ascending at the end
  const int* cnt;                    // [BH, 2]: how many of each
};

// 8 key bits -> 8 bf16 values (bit ? v[i] : 0) as one 16-byte chunk; v4 = the 8 bf16 values packed in four words
// (a 256-entry shared-memory mask table was measured slower: bank conflicts)
// Two bits select the two bf16 halves of a word with ONE byte permute: selector = 16 bits of a constant picked by the bit pair
// (00 -> 0x4444: both halves from the zero operand, 01 -> 0x4410, 10 -> 0x3244, 11 -> 0x3210): 4 instructions per word where the
// multiply-by-0xFFFF masks took 9 (the expansion is what this kernel's threads spend their time on)
__device__ __forceinline__ uint32_t pick2(uint32_t v, uint32_t bits, int i) {
  const unsigned long long sel = 0x3210324444104444ull;
  return __byte_perm(v, 0u, (uint32_t)(sel >> (((bits >> (2 * i)) & 3u) << 4)));
}
__device__ __forceinline__ uint4 expand8(uint32_t bits, const uint4& v4) {
  return make_uint4(pick2(v4.x, bits, 0), pick2(v4.y, bits, 1), pick2(v4.z, bits, 2), pick2(v4.w, bits, 3));
}

constexpr int kColBlocks = 2;          // 128-group column blocks per CTA: 256 TMEM columns and 48 KB of tiles, so that TWO CTAs share an SM and
                                       // one expands its tiles while the other's MMAs run (4 blocks / one CTA per SM: 0.31 ms per round at C4)
constexpr int kRowsPerThread = ((1 + kColBlocks) * 128 + 255) / 256;      // (1 + kColBlocks) tiles x 128 rows over 256 threads

__global__ void __launch_bounds__(kThreadsG, 2) hva_merge_inter_kernel(InterParams p) {
  const int bh = blockIdx.z, mb = blockIdx.x, cg = blockIdx.y;          // rows [128 mb, +128), column blocks kColBlocks cg ...
  const int tid = threadIdx.x, warp = tid >> 5;
  // Alg. 1 only pairs a group A of side 1 with a group B of side 0 (line 6): rows = the nA alive groups of side 1, columns = the nB
  // of side 0, both compacted -- a quarter of the N_q x N_q pairs in the first round, fewer later.  The grid is sized for the worst
  // case; CTAs past the counts leave at once.
  const int nA = p.cnt[2 * bh], nB = p.cnt[2 * bh + 1];
  if (128 * mb >= nA || 128 * kColBlocks * cg >= nB) return;
  const int* listA = p.list + (size_t)bh * p.Nq;
  const int* listB = listA + (p.Nq - nB);
  const int ncb = min(kColBlocks, (nB + 127) / 128 - kColBlocks * cg);  // column blocks of this CTA
  const int nt = p.nterms[bh];
  extern __shared__ unsigned char raw[];
  unsigned char* smem = raw + ((1024u - (smem_u32(raw) & 1023u)) & 1023u);
  unsigned char* sA = smem;                                             // [128][128 B]   chi(A) as 1.0 / 0
  unsigned char* sB = smem + kTileB;                                    // [kColBlocks][128][128 B]  chi(B) . digit_t(s^k)
  uint4* s_v = reinterpret_cast<uint4*>(sB + kColBlocks * kTileB);      // [8] the chunk's 64 bf16 digits of s^k, 8 per entry
  __shared__ uint64_t bar;
  __shared__ uint32_t tbase;
  if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  if (warp == 0) tmem_alloc(&tbase, 128 * kColBlocks);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tbase;
  const uint32_t* chi = p.chi + (size_t)bh * p.Nq * p.Wd;
  const int nchunk = (p.Nk + 63) / 64;
  const uint4 ones = make_uint4(0x3F803F80u, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u);
  // this thread expands the rows tid, tid + 256, tid + 512 of the (1 + ncb) x 128 tile rows; their two chi words of the
  // next chunk are fetched while the MMAs of the current one run
  int grp[kRowsPerThread];
  unsigned char* dst[kRowsPerThread];
  uint32_t w0[kRowsPerThread], w1[kRowsPerThread];
#pragma unroll
  for (int k = 0; k < kRowsPerThread; ++k) {
    const int e = tid + 256 * k, tile = e >> 7, r = e & 127;
    grp[k] = -1; dst[k] = sA;
    if (tile < 1 + ncb) {
      const int gg = tile == 0 ? 128 * mb + r : 128 * (kColBlocks * cg + tile - 1) + r;
      grp[k] = tile == 0 ? (gg < nA ? listA[gg] : -2) : (gg < nB ? listB[gg] : -2);   // -2: row of zeros
      dst[k] = (tile == 0 ? sA : sB + (size_t)(tile - 1) * kTileB) + r * 128;
    }
  }
  auto fetch = [&](int c) {
#pragma unroll
    for (int k = 0; k < kRowsPerThread; ++k) {
      w0[k] = w1[k] = 0;
      if (grp[k] >= 0) {
        if (2 * c < p.Wd) w0[k] = __ldg(chi + (size_t)grp[k] * p.Wd + 2 * c);
        if (2 * c + 1 < p.Wd) w1[k] = __ldg(chi + (size_t)grp[k] * p.Wd + 2 * c + 1);
      }
    }
  };
  // TMEM: column block cb accumulates at columns 128 cb.  One pass over the key chunks per base-256 digit t of s^k
  // (Y_t = chi . digit_t); the epilogue of pass t adds 256^t D to I.  C4 needs one digit (sizes < 256).
  for (int t = 0; t < nt; ++t) {
    fetch(0);
    for (int c = 0; c < nchunk; ++c) {
      if (c > 0 || t > 0) mbar_wait(&bar, (uint32_t)((t * nchunk + c - 1) & 1));   // MMAs of the previous chunk have read the tiles
      if (tid < 32) {                                                  // 64 digits of the chunk, two per thread
        uint32_t pk = 0;
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          const int j = 64 * c + 2 * tid + hh;
          const int sj = j < p.Nk ? p.sizes_k[(size_t)bh * p.Nk + j] : 0;
          pk |= (__float_as_uint((float)((sj >> (8 * t)) & 255)) >> 16) << (16 * hh);   // exact: < 256 has 8 significant bits
        }
        reinterpret_cast<uint32_t*>(s_v)[tid] = pk;
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < kRowsPerThread; ++k) {
        if (grp[k] != -1) {
          const int r = (tid + 256 * k) & 127;
          const bool is_a = (tid + 256 * k) < 128;
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const uint32_t bits = ((q < 4 ? w0[k] : w1[k]) >> (8 * (q & 3))) & 255u;
            *reinterpret_cast<uint4*>(dst[k] + ((q ^ (r & 7)) << 4)) = expand8(bits, is_a ? ones : s_v[q]);
          }
        }
      }
      if (c + 1 < nchunk) fetch(c + 1);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncthreads();
      if (warp == 0) {
        const uint32_t idesc = umma_idesc_bf16(128, 128, 0, 0);
        const uint64_t da = umma_desc(smem_u32(sA), 16, 1024), db = umma_desc(smem_u32(sB), 16, 1024);
        if (elect_one()) {
          for (int cb = 0; cb < ncb; ++cb) {
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)
              mma_ss(tmem + cb * 128, da + ks * 2, db + cb * (kTileB >> 4) + ks * 2, idesc, (c > 0 || ks > 0) ? 1u : 0u);
          }
          tc_commit(&bar);
        }
        __syncwarp();
      }
    }
    // epilogue of digit t: I (+)= 256^t * D
    mbar_wait(&bar, (uint32_t)((t * nchunk + nchunk - 1) & 1));
    tc_fence_after();
    if (warp < 4) {
      const int r = 128 * mb + warp * 32 + (tid & 31);
      for (int cb = 0; cb < ncb; ++cb) {
#pragma unroll 1
        for (int cc = 0; cc < 4; ++cc) {
          uint32_t v[32];
          tmem_ld32(tmem + ((uint32_t)(warp * 32) << 16) + cb * 128 + cc * 32, v);
          if (r < nA) {
            int* out = p.inter + ((size_t)bh * p.Nqp + r) * p.Nqp + 128 * (kColBlocks * cg + cb) + cc * 32;
#pragma unroll
            for (int i = 0; i < 32; i += 4) {
              int4 o = make_int4((int)__uint_as_float(v[i]) << (8 * t), (int)__uint_as_float(v[i + 1]) << (8 * t),
                                 (int)__uint_as_float(v[i + 2]) << (8 * t), (int)__uint_as_float(v[i + 3]) << (8 * t));
              if (t > 0) { const int4 old = *reinterpret_cast<const int4*>(out + i); o.x += old.x; o.y += old.y; o.z += old.z; o.w += old.w; }
              *reinterpret_cast<int4*>(out + i) = o;
            }
          }
        }
      }
    }
    tc_fence_before();
    __syncthreads();     // TMEM read before the next digit overwrites it (accumulate flag restarts at c == 0)
    tc_fence_after();
  }
  if (warp == 0) tmem_dealloc(tmem, 128 * kColBlocks);
}

__global__ void hva_merge_nterms_kernel(int Nk, const int* __restrict__ sizes_k, int* __restrict__ nterms) {
  const int bh = blockIdx.x;
  int mx = 0;
  for (int j = threadIdx.x; j < Nk; j += blockDim.x) mx = max(mx, sizes_k[(size_t)bh * Nk + j]);
  for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  __shared__ int s_m[32];
  if ((threadIdx.x & 31) == 0) s_m[threadIdx.x >> 5] = mx;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) mx = max(mx, s_m[w]);
    nterms[bh] = mx < 256 ? 1 : (mx < 65536 ? 2 : 3);
  }
}

}  // namespace

size_t hva_merge_inter_bytes(int BH, int Nq) {
  const size_t Nqp = ((size_t)Nq + 127) / 128 * 128;
  return hva_align((size_t)BH * Nqp * Nqp * 4) + hva_align((size_t)BH * 4) + hva_align((size_t)BH * 2 * 4);   // I, digits, side counts
}

int hva_merge_nterms_launch(int BH, int Nk, const int* sizes_k, int* nterms, cudaStream_t st) {
  hva_merge_nterms_kernel<<<BH, 256, 0, st>>>(Nk, sizes_k, nterms);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

int hva_merge_inter_launch(int BH, int Nq, int Nk, const uint32_t* chi, const int* sizes_k, const int* nterms, int* inter, const int* list,
                           const int* cnt, cudaStream_t st) {
  InterParams p{Nq, Nk, (Nk + 31) / 32, (Nq + 127) / 128 * 128, chi, sizes_k, nterms, inter, list, cnt};
  const size_t smem = 1024 + (1 + kColBlocks) * (size_t)kTileB + 8 * 16 + 64;
  // (per device and cheap: set on every call rather than behind a process-wide flag)
  if (cudaFuncSetAttribute(hva_merge_inter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return HVA_ECUDA;
  const int nrb = p.Nqp / 128;
  hva_merge_inter_kernel<<<dim3(nrb, (nrb + kColBlocks - 1) / kColBlocks, BH), kThreadsG, smem, st>>>(p);
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
