/* hva.h -- C ABI of the B200-native HyperVAttention operator (arxiv/paper_2607_03012).
 *
 * One DiT attention call: 3D local-window k-means on Q and K (Alg. 2, l.346-388),
 * centroid-level top-p block mask (Eq. 2-3, l.47-54), hardware-aware cluster merging
 * (Eq. 7-10, Alg. 1, l.111-168), cluster-contiguous permutation (Eq. 1, l.37), block-sparse
 * attention over the selected key clusters and inverse permutation (Eq. 4, l.56), plus the
 * hybrid anchor / subset clustering across denoising steps (section 4.2, l.93-103).
 *
 * Conventions (all entry points):
 *  - Every pointer is a DEVICE pointer owned by the caller unless it is a `const hva_shape*`
 *    / `const hva_config*` / `hva_plan_layout*` (HOST structs read during the call).  The
 *    library never allocates, frees, or keeps a pointer after return.
 *  - Tensors are contiguous: X[B, heads, n, D], n = T*H*W tokens in (t,h,w) row-major order
 *    (the "native flattened T x H x W layout", l.91), feature dim innermost.  BH = B*heads.
 *  - Work is enqueued on `stream` (a cudaStream_t passed as void*) with no host sync.
 *  - Return 0 on success or a negative HVA_E* code; nothing is enqueued on EINVAL /
 *    EWORKSPACE / EUNSUPPORTED.  No exceptions, no abort, no stdout.
 *  - `ws`/`ws_bytes`: scratch of at least hva_workspace_bytes(); contents undefined after.
 *  - There is NO CPU fallback: without a CUDA device every compute entry returns HVA_ECUDA.
 *  - hva_*_host entry points (bottom) take HOST buffers and perform the copies themselves.
 */
#ifndef HVA_H_
#define HVA_H_
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define HVA_F32 0
#define HVA_BF16 1

#define HVA_OK 0
#define HVA_EINVAL (-1)       /* null pointer, non-positive dim, D not in {64,128}, iters<1, top_p not in (0,1], ... */
#define HVA_EWORKSPACE (-2)   /* ws_bytes / plan_bytes / state_bytes too small */
#define HVA_EUNSUPPORTED (-3) /* dtype / tile / size combination without a kernel */
#define HVA_ECUDA (-4)        /* a CUDA runtime call or launch failed (cudaGetLastError) */
#define HVA_ELIMIT (-5)       /* the problem needs more scratch than the built-in array of a *_static entry point holds */

#define HVA_ANCHOR 0          /* full clustering (and, if subset_frac>0, refresh the hybrid cache) */
#define HVA_INTERMEDIATE 1    /* hybrid: re-assign only the cached subset (l.101)                  */
#define HVA_DENSE 2           /* full attention (warm-up steps/layers, l.324); no clustering       */

/* Kernel-selection flags (hva_config.flags and the hva_*_ex entry points).  0 = the product path.  The flagged kernels
 * compute the same stage with plain CUDA-core code (no tcgen05): they exist so that the tensor-pipe kernels can be
 * cross-checked against an independent implementation ON THE DEVICE (tests/), not as a dispatch for users.  The
 * library reads no environment variable and keeps no mutable global state besides per-device caches of CUDA function
 * attributes and of the copy streams of hva_forward_host. */
#define HVA_FLAG_CLUSTER_SIMT 1u    /* S1/S4: fp32 direct-form assignment on CUDA cores instead of the tcgen05 filter + refine */
#define HVA_FLAG_ATTN_SIMT 2u       /* S9: CUDA-core attention kernel instead of the tcgen05 kernel                            */
#define HVA_FLAG_MASK_BLOCKSORT 4u  /* S5: block-level shared-memory sort instead of the warp-per-row register sort           */
#define HVA_FLAG_MERGE_SIMT 8u      /* S6: per-pair bit-loop union sizes instead of the tcgen05 overlap contraction           */
#define HVA_FLAG_Q_UNPERMUTED 16u   /* hva_sparse_attention: `Qp` is the UNPERMUTED Q; the tcgen05 kernel gathers its rows through the
                                       plan's perm_q (Eq. 1 fused into the load, TMA tile::gather4).  hva_forward works this way: Q' is
                                       never materialised.  EUNSUPPORTED with the CUDA-core kernel                            */

/* Bipartition hash of Alg. 1 line 6 ("randomly bipartition", l.141; DESIGN.md R-M1):
 *   h  = seed*0x9E3779B1 ^ bh*0x85EBCA77 ^ round*0xC2B2AE3D ^ gid*0x27D4EB2F   (mod 2^32)
 *   h ^= h>>16; h *= 0x7FEB352D; h ^= h>>15; h *= 0x846CA68B; h ^= h>>16;
 *   side = h>>31   (1 -> A, 0 -> B);  round is 1-based, bh = b*heads+head, gid = smallest member. */

typedef struct {              /* problem statement, l.35 and Alg. 2 inputs l.349 */
  int32_t B, heads, T, H, W, D;
  int32_t dtype;              /* HVA_F32 | HVA_BF16; Q, K, V, O share it */
} hva_shape;

typedef struct {
  int32_t cell_q[3], cell_k[3];   /* (k_t,k_h,k_w); K_* = ceil(dim/k_*)            l.352 */
  int32_t win_q[3], win_k[3];     /* (w_t,w_h,w_w), clipped to K_*                 l.353 */
  int32_t iters;                  /* N_iter >= 1                                     l.349 */
  int32_t tile_q, tile_k;         /* tau_q, tau_k of the cost model                  l.111 */
  float top_p;                    /* (0,1]; >= 1 selects every key cluster           l.50  */
  float min_kc;                   /* [0,1], keep >= ceil(min_kc*N_k) key clusters    l.334 */
  int32_t merge_rounds;           /* R; 0 = merging off; the paper uses 3            l.322 */
  int32_t max_q_tiles;            /* 0 = uncapped (paper); k>0 = merged group <= k row tiles */
  uint32_t seed;                  /* bipartition hash seed                           l.141 */
  float subset_frac;              /* hybrid: 0 = off; the paper uses 0.15            l.322 */
  int32_t hybrid_refresh_all;     /* 0 = reading R-H3, 1 = R-H3'               */
  float softmax_scale;            /* 0 => 1/sqrt(D)                                  l.47  */
  uint32_t flags;                 /* HVA_FLAG_* (0 = product kernels)                      */
} hva_config;

typedef struct {              /* per (batch, head); written on device by hva_build_plan */
  int32_t n_groups;           /* |P| after merging (groups with s^q > 0)                   */
  int32_t q_tiles;            /* sum_S ceil(s^q(S)/tau_q)                                  */
  int64_t q_rows_valid;       /* sum_S s^q(S) = n                                          */
  int64_t q_rows_padded;      /* sum_S tau_q ceil(s^q(S)/tau_q)                            */
  int64_t k_cols_valid;       /* sum_S kappa(S),  kappa(S) = sum_j chi_j(S) s^k_j   Eq. 8  */
  int64_t k_cols_padded;      /* sum_S tau_k ceil(kappa(S)/tau_k)                          */
  int64_t tiles_executed;     /* sum_S ceil(s^q/tau_q) ceil(kappa/tau_k) = sum C(S)/(tau_q tau_k), Eq. 8-9 */
  int64_t pairs_valid;        /* sum_S s^q(S) kappa(S)  -> theoretical density = /n^2, l.225 */
} hva_stats;

typedef struct {              /* byte offsets of the arrays inside the opaque plan buffer; every
                                 array is int32 and has a leading BH dimension                   */
  size_t perm_q, inv_perm_q, perm_k;   /* [BH,n]: perm[i] = token placed at permuted row i    */
  size_t koff;                /* [BH,Nk+1] K' row offset of key cluster j                      */
  size_t n_groups;            /* [BH]                                                          */
  size_t gid;                 /* [BH,Nq] ascending active group ids (first n_groups valid)     */
  size_t goff;                /* [BH,Nq+1] Q' row offset of group g (gid order)                */
  size_t kappa;               /* [BH,Nq] packed key count of group g                           */
  size_t run_cnt;             /* [BH,Nq] number of key runs of group g                         */
  size_t runs;                /* [BH,Nq,run_stride] runs as (first | last<<16) key-cluster ids */
  size_t run_stride;          /* = ceil((Nk+1)/2) entries, not a byte offset                   */
  size_t work_cnt;            /* [BH] number of (group, q-tile) work items                     */
  size_t work;                /* [BH,work_cap] g | tile<<16                                    */
  size_t work_cap;            /* = ceil(n/tau_q) + Nq entries, not a byte offset               */
  size_t stats;               /* [BH] hva_stats                                                */
  size_t total;               /* plan size in bytes                                            */
} hva_plan_layout;

typedef struct {              /* byte offsets of the arrays inside the hybrid `state` buffer of hva_forward; index 0 = Q, 1 = K */
  size_t assign[2];           /* [BH,n] int32 labels                                            */
  size_t mu[2];               /* [BH,Nc,D] fp32 centroids                                       */
  size_t sums[2];             /* [BH,Nc,D] fp32 z                                               */
  size_t sizes[2];            /* [BH,Nc] int32                                                  */
  size_t subset[2];           /* [BH,max(m,1)] int32 cached subset (ascending token ids)        */
  int32_t n_clusters[2];      /* N_q, N_k                                                       */
  int32_t m;                  /* floor(subset_frac * n + 1/2)                                   */
  size_t total;               /* = hva_state_bytes()                                            */
} hva_state_layout;

typedef struct {              /* byte offsets inside the workspace of hva_forward: where a caller (or a test) finds the
                                 intermediate results of the last ANCHOR / INTERMEDIATE call; valid until the next call */
  size_t lowe;                /* [BH,n] fp32 rho of the last clustered tensor (hybrid anchors only)            */
  size_t mask;                /* [BH,Nq,Nk] uint8 M (Eq. 3)                                                    */
  size_t group_of;            /* [BH,Nq] int32 gid of each query cluster (Alg. 1)                              */
  size_t n_groups;            /* [BH] int32                                                                    */
  size_t group_mask;          /* [BH,Nq,Nk] uint8 chi of the active groups in gid order                        */
  size_t plan, plan_bytes;    /* the plan buffer (hva_plan_describe(BH, n, max(Nq,1), max(Nk,1), tile_q))      */
  size_t qp, kp, vp;          /* permuted tensors Q', K', V' [B,heads,n,D] (Eq. 1); Q' has size 0 on the tensor-pipe path,
                                 where the attention kernel gathers the rows of Q itself (HVA_FLAG_Q_UNPERMUTED)      */
  size_t scratch;             /* stage scratch                                                                 */
  size_t state;               /* where the per-tensor state lives when hva_forward is called with state == NULL */
  size_t total;               /* = hva_workspace_bytes()                                                       */
} hva_workspace_layout;

const char* hva_strerror(int code);
int hva_version(void);

/* Number of centroids N_c = ceil(T/k_t) ceil(H/k_h) ceil(W/k_w)  (Alg. 2 line 3, l.352). */
int32_t hva_num_clusters(const hva_shape* s, const int32_t cell[3]);
size_t hva_workspace_bytes(const hva_shape* s, const hva_config* c);
size_t hva_state_bytes(const hva_shape* s, const hva_config* c);   /* hybrid cache, l.101 */
/* Scratch needed by one hva_cluster call (per-cell partial sums, split centroids); 0 on invalid arguments. */
size_t hva_cluster_workspace_bytes(const hva_shape* s, const int32_t cell[3], const int32_t win[3]);
int hva_plan_describe(int32_t BH, int32_t n, int32_t Nq, int32_t Nk, int32_t tile_q, hva_plan_layout* out);
/* Scratch needed by one hva_build_plan call; 0 on invalid arguments. */
size_t hva_plan_workspace_bytes(int32_t BH, int32_t n, int32_t Nq, int32_t Nk);
int hva_workspace_describe(const hva_shape* s, const hva_config* c, hva_workspace_layout* out);
/* Layout of the `state` buffer (what hva_forward keeps between calls, and where a caller finds the clustering result). */
int hva_state_describe(const hva_shape* s, const hva_config* c, hva_state_layout* out);

/* S0-S2 (+A4): 3D local-window k-means on one tensor X[B,heads,n,D] (Alg. 2, l.346-388; Eq. 5
 * l.81; Eq. 6 l.97).  Centre-token init (lines 7-11) unless mu_init != NULL ([BH,Nc,D] fp32,
 * used for teacher-forced parity and warm starts).  `iters` Jacobi passes; argmin = first
 * minimum in ascending centroid id over the clipped (shifted, full-size) window.
 * Outputs: assign[BH,n] int32 (last pass); mu[BH,Nc,D] fp32 AFTER the last update (line 24;
 * empty clusters keep mu, line 23); sizes[BH,Nc] int32; sums[BH,Nc,D] fp32 z of the last pass
 * (nullable); lowe[BH,n] fp32 rho = d1/d2 of the last pass (nullable).  Deterministic: no
 * floating-point atomics; the same inputs give the same bits. */
int hva_cluster(const hva_shape* s, const int32_t cell[3], const int32_t win[3], int32_t iters,
                const void* X, const float* mu_init, int32_t* assign, float* mu, int32_t* sizes,
                float* sums, float* lowe, void* ws, size_t ws_bytes, void* stream);

/* hva_cluster with kernel-selection flags (HVA_FLAG_CLUSTER_SIMT) and, if probe != NULL (device float[32], zeroed by the
 * caller; tensor-pipe path only), the instrumented kernel instantiation: probe[0] receives the largest observed
 * |filter score - exact score| / (|x| max|mu|) (1.0 if the |x|^2 bound was violated).  Labels are unaffected. */
int hva_cluster_ex(const hva_shape* s, const int32_t cell[3], const int32_t win[3], int32_t iters,
                   const void* X, const float* mu_init, int32_t* assign, float* mu, int32_t* sizes,
                   float* sums, float* lowe, uint32_t flags, float* probe, void* ws, size_t ws_bytes, void* stream);

/* S1 + S2 of BOTH tensors of a call (what hva_forward runs at an anchor step without the hybrid subset): hva_cluster of Q
 * (cells c->cell_q, window c->win_q) on `stream` and of K (c->cell_k, c->win_k) on a library-owned side stream of the current
 * device, forked from and joined back into `stream` by events (legal under stream capture), so that the two chains of
 * kernels overlap; c->iters passes each, c->flags as in hva_cluster_ex.  Outputs as hva_cluster, per tensor (sums_* nullable).
 * ws_q / ws_k: two DISJOINT device scratch regions of at least hva_cluster_workspace_bytes() for the respective grid
 * (HVA_EINVAL if they overlap).  The results are bit-identical to two hva_cluster calls.  Concurrent host calls on one device
 * are serialised while they enqueue.  HVA_ECUDA if the side stream cannot be created. */
int hva_cluster_qk(const hva_shape* s, const hva_config* c, const void* Q, const void* K,
                   int32_t* assign_q, float* mu_q, int32_t* sizes_q, float* sums_q,
                   int32_t* assign_k, float* mu_k, int32_t* sizes_k, float* sums_k,
                   void* ws_q, size_t ws_q_bytes, void* ws_k, size_t ws_k_bytes, void* stream);

/* S3: indices (ascending) of the m tokens with the largest rho per (b,head), ties -> lower
 * token index (l.101, l.322; R-H2).  lowe[BH,n] fp32 >= 0; subset[BH,m] int32. */
int hva_select_subset(int32_t BH, int32_t n, const float* lowe, int32_t m, int32_t* subset,
                      void* ws, size_t ws_bytes, void* stream);

/* S4: intermediate hybrid step on one tensor (l.101-103; R-H3 / R-H3').  For l in subset:
 * a_l <- argmin over ALL Nc centroids of ||x_l - mu_u||^2 against the cached mu (first minimum);
 * sums/sizes adjusted for moved tokens with their current features; mu_u <- sums_u/sizes_u for
 * touched u with sizes_u > 0.  refresh_all=1: recompute sums, sizes, mu of every cluster from the
 * current X.  assign, mu, sums, sizes are updated in place. */
int hva_cluster_update(const hva_shape* s, int32_t Nc, const void* X, const int32_t* subset, int32_t m,
                       int32_t refresh_all, int32_t* assign, float* mu, float* sums, int32_t* sizes,
                       void* ws, size_t ws_bytes, void* stream);

int hva_cluster_update_ex(const hva_shape* s, int32_t Nc, const void* X, const int32_t* subset, int32_t m,
                          int32_t refresh_all, int32_t* assign, float* mu, float* sums, int32_t* sizes, uint32_t flags,
                          void* ws, size_t ws_bytes, void* stream);   /* flags: HVA_FLAG_CLUSTER_SIMT */

/* Scratch needed by one hva_cluster_update call; 0 on invalid arguments. */
size_t hva_cluster_update_workspace_bytes(const hva_shape* s, int32_t Nc, int32_t m);

/* S5: M[BH,Nq,Nk] uint8 (Eq. 2-3, l.47-54; min-kc l.334).  fp64 on device from the fp32
 * centroids; order by weight descending, ties -> lower j; smallest prefix with cumulative
 * weight >= top_p * Z; top_p >= 1 -> all ones; at least ceil(min_kc*Nk) kept.  Nk <= 2048. */
int hva_build_mask(int32_t BH, int32_t Nq, int32_t Nk, int32_t D, const float* mu_q, const float* mu_k,
                   const int32_t* sizes_k, float scale, float top_p, float min_kc, uint8_t* mask,
                   void* ws, size_t ws_bytes, void* stream);

int hva_build_mask_ex(int32_t BH, int32_t Nq, int32_t Nk, int32_t D, const float* mu_q, const float* mu_k,
                      const int32_t* sizes_k, float scale, float top_p, float min_kc, uint8_t* mask, uint32_t flags,
                      void* ws, size_t ws_bytes, void* stream);       /* flags: HVA_FLAG_MASK_BLOCKSORT */

/* S6: parallel agglomerative merging (Eq. 7-10 l.111-125; Alg. 1 l.131-168), R = rounds.
 * group_of_cluster[BH,Nq] = gid (smallest member) of each query cluster's group (clusters with
 * s^q = 0 keep their own id); n_groups[BH]; group_mask[BH,Nq,Nk] uint8: row g = chi(S_g) for the
 * g-th active group in ascending gid order (first n_groups rows valid, rest zero).
 * Pure integer; bit-exact against Alg. 1 with the hash above; ties -> lower gid. */
int hva_merge(int32_t BH, int32_t Nq, int32_t Nk, const int32_t* sizes_q, const int32_t* sizes_k,
              const uint8_t* mask, int32_t tile_q, int32_t tile_k, int32_t rounds, int32_t max_q_tiles,
              uint32_t seed, int32_t* group_of_cluster, int32_t* n_groups, uint8_t* group_mask,
              void* ws, size_t ws_bytes, void* stream);

int hva_merge_ex(int32_t BH, int32_t Nq, int32_t Nk, const int32_t* sizes_q, const int32_t* sizes_k,
                 const uint8_t* mask, int32_t tile_q, int32_t tile_k, int32_t rounds, int32_t max_q_tiles,
                 uint32_t seed, int32_t* group_of_cluster, int32_t* n_groups, uint8_t* group_mask, uint32_t flags,
                 void* ws, size_t ws_bytes, void* stream);            /* flags: HVA_FLAG_MERGE_SIMT */

/* Scratch needed by one hva_merge call; 0 on invalid arguments. */
size_t hva_merge_workspace_bytes(int32_t BH, int32_t Nq, int32_t Nk);

/* S7: canonical permutations (Eq. 1, l.37; R-P1) and the attention work list.  perm_k sorts
 * tokens by (a^k, l); perm_q by (gid(a^q), a^q, l).  `plan` is an opaque device buffer of
 * hva_plan_describe().total bytes.  Labels need not be window-local (hybrid steps). */
int hva_build_plan(int32_t BH, int32_t n, int32_t Nq, int32_t Nk, const int32_t* assign_q,
                   const int32_t* assign_k, const int32_t* sizes_q, const int32_t* sizes_k,
                   const int32_t* group_of_cluster, const int32_t* n_groups, const uint8_t* group_mask,
                   int32_t tile_q, int32_t tile_k, void* plan, size_t plan_bytes,
                   void* ws, size_t ws_bytes, void* stream);

/* hva_build_plan for callers that may not allocate device memory and have no scratch buffer to hand over (code under CUDA
 * graph capture, serving loops, harnesses that forbid cudaMalloc): same inputs, same `plan` output (bit-identical), but the
 * scratch is a device array built into the library, HVA_PLAN_STATIC_SCRATCH_BYTES large, which every GPU that loads the
 * library holds until the process exits.  The call allocates nothing (no cudaMalloc / cudaFree / allocating library routine);
 * its first use on a device looks the array's device address up (cudaGetSymbolAddress, with the caller's current device).
 * Limit: hva_plan_workspace_bytes(BH, n, Nq, Nk) <= hva_build_plan_static_limit() (32 MiB: C4 with 24 heads needs 22.3 MB,
 * C3 with 40 heads 15.0 MB); beyond it the call returns HVA_ELIMIT and enqueues nothing -- use hva_build_plan with a
 * caller-owned buffer.  All calls on a device SHARE the array, and it keeps the previous call's contents: nothing in it has to
 * start at zero (every word a kernel reads is written earlier in the same call), but two calls that overlap on the GPU
 * (different streams) race on it; calls on one stream are ordered.  Other errors as hva_build_plan. */
#define HVA_PLAN_STATIC_SCRATCH_BYTES (32u << 20)
size_t hva_build_plan_static_limit(void);
int hva_build_plan_static(int32_t BH, int32_t n, int32_t Nq, int32_t Nk, const int32_t* assign_q,
                          const int32_t* assign_k, const int32_t* sizes_q, const int32_t* sizes_k,
                          const int32_t* group_of_cluster, const int32_t* n_groups, const uint8_t* group_mask,
                          int32_t tile_q, int32_t tile_k, void* plan, size_t plan_bytes, void* stream);

/* S8 / S10: Xp[bh,i,:] = X[bh,perm[bh,i],:]  and its inverse  X[bh,perm[bh,i],:] = Xp[bh,i,:]
 * (Eq. 1 l.37; Eq. 4 l.56). */
int hva_permute(const hva_shape* s, const void* X, const int32_t* perm, void* Xp, void* stream);
int hva_unpermute(const hva_shape* s, const void* Xp, const int32_t* perm, void* X, void* stream);

/* S9 (+S10): block-sparse attention over the permuted tensors (Eq. 4 l.56; packed key blocks
 * l.109; union masks Eq. 8 l.115).  Qp/Kp/Vp[B,heads,n,D] permuted by the plan.  If
 * unpermute != 0, row i of group order is written to O[perm_q[i]] (S10 fused), else to O'[i].
 * bf16, D = 128, tile 128 x 128: the tcgen05 kernel (the product path).  Every other combination (f32; bf16 with D = 64;
 * tiles other than 128 x 128) and c->flags & HVA_FLAG_ATTN_SIMT run the CUDA-core kernel: same result at reference
 * precision, one warp per query row, NOT tuned -- orders of magnitude slower at the large shapes.  It exists for the
 * fp32 C1 config and as the on-device cross-check of the tcgen05 kernel. */
int hva_sparse_attention(const hva_shape* s, const hva_config* c, const void* Qp, const void* Kp,
                         const void* Vp, const void* plan, size_t plan_bytes, int32_t Nq, int32_t Nk,
                         void* O, int32_t unpermute, void* ws, size_t ws_bytes, void* stream);

/* Whole hot path for one attention call.  step_kind: HVA_ANCHOR | HVA_INTERMEDIATE | HVA_DENSE.
 * `state` (hva_state_bytes(), nullable when subset_frac == 0) carries the hybrid cache between
 * calls; `stats_out` (nullable) receives hva_stats[BH] (device). */
int hva_forward(const hva_shape* s, const hva_config* c, const void* Q, const void* K, const void* V,
                void* O, int32_t step_kind, void* state, hva_stats* stats_out,
                void* ws, size_t ws_bytes, void* stream);

/* Same as hva_forward with HOST Q,K,V,O (pinned or pageable); allocates nothing: `dev_qkvo` is a
 * caller-owned DEVICE staging buffer of 4*B*heads*n*D elements.  Heads are independent, so with B = 1, >= 8 heads and no
 * hybrid state the call runs in up to 16 chunks of heads whose sizes grow geometrically from a one-head first chunk (so that
 * a chunk's H2D copy has landed before the kernels of the chunk before it are done) and end with a small one: only the first
 * chunk's H2D copy and the last chunk's D2H copy are not covered by kernels.  The copies (two library-owned copy streams, both
 * PCIe directions; pinned host buffers needed for the overlap) run under the kernels; consecutive chunks run on two library-owned
 * compute streams with one half of `ws` each when a half holds the largest chunk (the small stages of chunk k+1 then fill in under
 * the attention kernel of chunk k), else on `stream`; all of them start after what the caller has queued on `stream` and are
 * drained before the call returns.  Chunked and unchunked calls give the same bits (the merge hash is keyed by the global head).
 * Arguments are validated before anything is enqueued; on any error the stream and the copy streams are drained before
 * returning.  The copy streams are per device; concurrent host calls on the same device are serialised by the library.
 * Synchronises the stream. */
int hva_forward_host(const hva_shape* s, const hva_config* c, const void* hQ, const void* hK,
                     const void* hV, void* hO, int32_t step_kind, void* state, void* dev_qkvo,
                     void* ws, size_t ws_bytes, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* HVA_H_ */
