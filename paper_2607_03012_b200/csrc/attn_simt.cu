// S9 (+S10), CUDA-core variant: block-sparse attention over the plan's packed key runs in fp32
// (Eq. 4 l.56; union masks Eq. 8 l.115).  Used for dtype f32 (config C1, where the 1e-4
// tolerance rules out bf16/tf32 tensor-core products) and as an on-device cross-check of the
// tcgen05 kernel.  One CTA per (group, q-tile) work item, one warp per query row, lanes over D;
// online softmax with max-subtraction, fp32 accumulation.
#include "common.cuh"

namespace {

template <typename T, int D>
__global__ void __launch_bounds__(128) hva_attn_simt_kernel(int n, int Nq, int Nk, int tile_q, float scale_log2,
                                                            const T* __restrict__ Qp, const T* __restrict__ Kp,
                                                            const T* __restrict__ Vp, const int* __restrict__ goff_,
                                                            const int* __restrict__ koff_, const int* __restrict__ run_cnt_,
                                                            const uint32_t* __restrict__ runs_, int run_stride,
                                                            const int* __restrict__ work_cnt, const int* __restrict__ work_,
                                                            int work_cap, const int* __restrict__ perm_q, T* __restrict__ O) {
  constexpr int E = D / 32;
  const int bh = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if ((int)blockIdx.x >= work_cnt[bh]) return;
  const uint32_t wi = (uint32_t)work_[(size_t)bh * work_cap + blockIdx.x];
  const int g = wi & 0xffff, t = wi >> 16;
  const int* goff = goff_ + (size_t)bh * (Nq + 1);
  const int* koff = koff_ + (size_t)bh * (Nk + 1);
  const int nrun = run_cnt_[(size_t)bh * Nq + g];
  const uint32_t* runs = runs_ + ((size_t)bh * Nq + g) * run_stride;
  const int row0 = goff[g] + t * tile_q, row1 = min(goff[g + 1], row0 + tile_q);
  const size_t base = (size_t)bh * n;
  for (int row = row0 + warp; row < row1; row += 4) {
    float q[E], o[E];
#pragma unroll
    for (int e = 0; e < E; ++e) { q[e] = HvaElem<T>::ld(Qp + (base + row) * D + e * 32 + lane); o[e] = 0.f; }
    float m = -INFINITY, l = 0.f;
    for (int r = 0; r < nrun; ++r) {
      const uint32_t rr = runs[r];
      const int k0 = koff[rr & 0xffff], k1 = koff[(rr >> 16) + 1];
      for (int k = k0; k < k1; ++k) {
        float s = 0.f;
#pragma unroll
        for (int e = 0; e < E; ++e) s = fmaf(q[e], HvaElem<T>::ld(Kp + (base + k) * D + e * 32 + lane), s);
#pragma unroll
        for (int x = 16; x > 0; x >>= 1) s += __shfl_xor_sync(0xffffffffu, s, x);
        s *= scale_log2;
        float mn = fmaxf(m, s);
        float corr = exp2f(m - mn), pw = exp2f(s - mn);
        l = l * corr + pw;
#pragma unroll
        for (int e = 0; e < E; ++e) o[e] = fmaf(pw, HvaElem<T>::ld(Vp + (base + k) * D + e * 32 + lane), o[e] * corr);
        m = mn;
      }
    }
    const float inv = l > 0.f ? 1.f / l : 0.f;
    const size_t orow = perm_q ? base + perm_q[base + row] : base + row;   // fused O = Pi^{q-1} O'  (Eq. 4)
#pragma unroll
    for (int e = 0; e < E; ++e) HvaElem<T>::st(O + orow * D + e * 32 + lane, o[e] * inv);
  }
}

}  // namespace

int hva_attention_simt_launch(const hva_shape* s, float scale, const void* Qp, const void* Kp, const void* Vp,
                              const void* plan, const hva_plan_layout& L, int Nq, int Nk, void* O, int unpermute,
                              cudaStream_t st, int tile_q) {
  const char* b = reinterpret_cast<const char*>(plan);
  const int n = s->T * s->H * s->W, BH = s->B * s->heads;
  dim3 grid((unsigned)L.work_cap, BH);
  const float sl2 = scale * 1.4426950408889634f;
#define HVA_ARGS(T)                                                                                                  \
  n, Nq, Nk, tile_q, sl2, (const T*)Qp, (const T*)Kp, (const T*)Vp, (const int*)(b + L.goff), (const int*)(b + L.koff), \
      (const int*)(b + L.run_cnt), (const uint32_t*)(b + L.runs), (int)L.run_stride, (const int*)(b + L.work_cnt),      \
      (const int*)(b + L.work), (int)L.work_cap, unpermute ? (const int*)(b + L.perm_q) : nullptr, (T*)O
  if (s->dtype == HVA_F32) {
    if (s->D == 64) hva_attn_simt_kernel<float, 64><<<grid, 128, 0, st>>>(HVA_ARGS(float));
    else hva_attn_simt_kernel<float, 128><<<grid, 128, 0, st>>>(HVA_ARGS(float));
  } else {
    if (s->D == 64) hva_attn_simt_kernel<__nv_bfloat16, 64><<<grid, 128, 0, st>>>(HVA_ARGS(__nv_bfloat16));
    else hva_attn_simt_kernel<__nv_bfloat16, 128><<<grid, 128, 0, st>>>(HVA_ARGS(__nv_bfloat16));
  }
#undef HVA_ARGS
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}
