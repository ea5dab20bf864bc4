// Shared device/host helpers of the hva CUDA path (sm_100a).  Not used by the oracle.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/hva.h"

#define HVA_CHECK_LAUNCH()                                \
  do {                                                    \
    if (cudaGetLastError() != cudaSuccess) return HVA_ECUDA; \
  } while (0)

#define HVA_TRY(expr)                 \
  do {                                \
    int _rc = (expr);                 \
    if (_rc != HVA_OK) return _rc;    \
  } while (0)

static inline int64_t hva_cdiv64(int64_t a, int64_t b) { return (a + b - 1) / b; }
static inline size_t hva_align(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Grid geometry of 3D local-window clustering (Alg. 2 lines 3-6, l.352-356).
struct HvaGrid {
  int T, H, W;        // lattice
  int kt, kh, kw;     // cell size
  int Kt, Kh, Kw;     // K_* = ceil(dim / k_*)
  int wt, wh, ww;     // window, clipped to K_* (line 4)
  int Nc, nwin, n;
};

static inline HvaGrid hva_make_grid(const hva_shape* s, const int32_t cell[3], const int32_t win[3]) {
  HvaGrid g;
  g.T = s->T; g.H = s->H; g.W = s->W;
  g.kt = cell[0]; g.kh = cell[1]; g.kw = cell[2];
  g.Kt = (g.T + g.kt - 1) / g.kt; g.Kh = (g.H + g.kh - 1) / g.kh; g.Kw = (g.W + g.kw - 1) / g.kw;
  g.wt = win[0] < g.Kt ? win[0] : g.Kt; g.wh = win[1] < g.Kh ? win[1] : g.Kh; g.ww = win[2] < g.Kw ? win[2] : g.Kw;
  g.Nc = g.Kt * g.Kh * g.Kw; g.nwin = g.wt * g.wh * g.ww; g.n = g.T * g.H * g.W;
  return g;
}

// window start  u_bar = clip(u - floor(w/2), 0, K - w)   (Alg. 2 lines 15-17, l.369-373)
__host__ __device__ __forceinline__ int hva_win_start(int u, int w, int K) {
  int s = u - w / 2;
  s = s < 0 ? 0 : s;
  return s > K - w ? K - w : s;
}

template <typename T> struct HvaElem;
template <> struct HvaElem<float> {
  static __device__ __forceinline__ float ld(const float* p) { return *p; }
  static __device__ __forceinline__ void st(float* p, float v) { *p = v; }
};
template <> struct HvaElem<__nv_bfloat16> {
  static __device__ __forceinline__ float ld(const __nv_bfloat16* p) { return __bfloat162float(*p); }
  static __device__ __forceinline__ void st(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }
};

// Entry points implemented across translation units (internal linkage to the library).
int hva_attention_tc_launch(const hva_shape* s, float scale, const void* Qp, const void* Kp, const void* Vp,
                            const void* plan, const hva_plan_layout& L, int Nq, int Nk, void* O, int unpermute, int gather_q,
                            cudaStream_t st);
int hva_attention_simt_launch(const hva_shape* s, float scale, const void* Qp, const void* Kp, const void* Vp,
                              const void* plan, const hva_plan_layout& L, int Nq, int Nk, void* O, int unpermute,
                              cudaStream_t st, int tile_q);
int hva_attention_dense_plan(int BH, int n, int tile_q, int tile_k, void* plan, const hva_plan_layout& L, cudaStream_t st);

// hva_merge for the (batch, head) pairs bh0 .. bh0 + BH - 1 of a larger problem (chunked host path)
int hva_merge_offset(int32_t bh0, int32_t BH, int32_t Nq, int32_t Nk, const int32_t* sizes_q, const int32_t* sizes_k, const uint8_t* mask,
                     int32_t tile_q, int32_t tile_k, int32_t rounds, int32_t max_q_tiles, uint32_t seed, int32_t* group_of_cluster,
                     int32_t* n_groups, uint8_t* group_mask, uint32_t flags, void* ws, size_t ws_bytes, void* stream);

struct HvaGrid;
size_t hva_cluster_ws_bytes(const HvaGrid& g, int BH, int D);
size_t hva_merge_ws_bytes(int BH, int Nq, int Nk);
size_t hva_plan_ws_bytes(int BH, int n, int Nq, int Nk);
// hva_build_plan in two halves (plan.cu): keys (koff, perm_k) from the K clustering alone; queries (everything else)
int hva_gather_kv(const hva_shape* s, const void* K, const void* V, const int32_t* perm, void* Kp, void* Vp, cudaStream_t st);
size_t hva_plan_keys_ws_bytes(int BH, int n, int Nk);
int hva_plan_keys(int BH, int n, int Nk, const int* assign_k, const int* sizes_k, void* plan, const hva_plan_layout& L, void* ws,
                  size_t ws_bytes, cudaStream_t st);
int hva_plan_queries(int BH, int n, int Nq, int Nk, const int* assign_q, const int* sizes_q, const int* sizes_k, const int* group_of_cluster,
                     const uint8_t* group_mask, int tile_q, int tile_k, void* plan, const hva_plan_layout& L, void* ws, size_t ws_bytes,
                     cudaStream_t st);
size_t hva_hybrid_ws_bytes(int BH, int n, int Nc, int m, int D);
size_t hva_refresh_ws_bytes(int BH, int n, int Nc);
// R-H3': mu, sums, sizes of every cluster recomputed from the current X and labels (plan.cu: label sort + segment means)
int hva_refresh_centroids(int BH, int n, int Nc, int D, int dtype, const void* X, const int* assign, float* mu, float* sums, int* sizes,
                          void* ws, size_t ws_bytes, cudaStream_t st);
