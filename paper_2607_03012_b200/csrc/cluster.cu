// S0-S2 (+A4): 3D local-window k-means (Alg. 2, l.346-388; Eq. 5 l.81; Eq. 6 l.97).
//
// v1 layout: one CTA per home cell.  The cell's window centroids (fp32) and the cell's tokens are
// staged in shared memory; one thread per token evaluates the direct form sum_c (x_c - mu_c)^2 in
// fp32 for every window candidate (ascending centroid id, strict '<' => first minimum, R-C1) and
// keeps the best / second best (Eq. 6).  Tokens are then counting-sorted by target slot and each
// thread (= one feature dim) adds its column in token order: a deterministic segmented per-cell
// reduction with no atomics.  The per-(cell, slot) partial sums are combined per centroid, in a
// fixed cell order, by hva_finalize_kernel (Alg. 2 line 23: mu <- z/n, empty keeps mu).
#include "common.cuh"
#include "cluster_tc.cuh"
#include <algorithm>

namespace {

constexpr int kThreads = 128;

__device__ __forceinline__ void load8(const float* p, float x[8]) {
  float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
  x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y; x[6] = b.z; x[7] = b.w;
}
__device__ __forceinline__ void load8(const __nv_bfloat16* p, float x[8]) {
  uint4 r = *reinterpret_cast<const uint4*>(p);  // bf16 -> fp32 is a 16-bit shift (exact)
  x[0] = __uint_as_float(r.x << 16); x[1] = __uint_as_float(r.x & 0xffff0000u);
  x[2] = __uint_as_float(r.y << 16); x[3] = __uint_as_float(r.y & 0xffff0000u);
  x[4] = __uint_as_float(r.z << 16); x[5] = __uint_as_float(r.z & 0xffff0000u);
  x[6] = __uint_as_float(r.w << 16); x[7] = __uint_as_float(r.w & 0xffff0000u);
}

struct ClusterParams {
  HvaGrid g;
  int BH;
  const void* X;       // [BH, n, D]
  const float* mu;     // [BH, Nc, D]
  float* part;         // [BH, Nc(cells), nwin, D]
  int* part_cnt;       // [BH, Nc(cells), nwin]
  int* assign;         // [BH, n] or null
  float* lowe;         // [BH, n] or null
};

// Operands of the tensor-pipe assignment (cluster_tc.cu): two-term bf16 split hi + lo of the fp32 centroid and
// |mu|^2 in fp32 (fixed shuffle-tree order => deterministic).  Block = D threads, thread c owns mu_c.
struct MuSplit {
  __nv_bfloat16 *hi, *lo;   // [BH, Nc, D] or null
  float* musq;              // [BH, Nc]
};
template <int D>
__device__ __forceinline__ void mu_split_store(const MuSplit& sp, size_t row, int c, float m) {
  if (!sp.hi) return;
  const __nv_bfloat16 h = __float2bfloat16_rn(m);
  sp.hi[row * D + c] = h;
  sp.lo[row * D + c] = __float2bfloat16_rn(m - __bfloat162float(h));
  __shared__ float s_red[D / 32];
  float q = m * m;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
  if ((c & 31) == 0) s_red[c >> 5] = q;
  __syncthreads();
  if (c == 0) {
    float t = s_red[0];
#pragma unroll
    for (int w = 1; w < D / 32; ++w) t += s_red[w];
    sp.musq[row] = t;
  }
}

template <int D>
__global__ void __launch_bounds__(D) hva_mu_split_kernel(int Nc, const float* __restrict__ mu, MuSplit sp) {
  const size_t row = (size_t)blockIdx.y * Nc + blockIdx.x;
  mu_split_store<D>(sp, row, threadIdx.x, mu[row * D + threadIdx.x]);
}

// Alg. 2 lines 7-11 and the operands of the first tensor-pipe pass in one launch: warp = centroid, lane = D/32 consecutive dims
// (one launch of Nc*BH/8 CTAs instead of two of Nc*BH: both were bound by the CTA launch rate, 23 + 16 us at C4)
constexpr int kInitWarps = 8;
template <typename T, int D>
__global__ void __launch_bounds__(32 * kInitWarps) hva_init_centroids_kernel(HvaGrid g, const T* __restrict__ X,
                                                                             float* __restrict__ mu, MuSplit sp) {
  // mu_u <- X[c_t, c_h, c_w, :],  c = min(u*k + floor(k/2), dim-1)
  constexpr int E = D / 32;
  const int u = blockIdx.x * kInitWarps + (threadIdx.x >> 5), bh = blockIdx.y, lane = threadIdx.x & 31;
  if (u >= g.Nc) return;
  const int ut = u / (g.Kh * g.Kw), uh = (u / g.Kw) % g.Kh, uw = u % g.Kw;
  const int ct = min(ut * g.kt + g.kt / 2, g.T - 1), ch = min(uh * g.kh + g.kh / 2, g.H - 1),
            cw = min(uw * g.kw + g.kw / 2, g.W - 1);
  const size_t tok = (size_t)(ct * g.H + ch) * g.W + cw, row = (size_t)bh * g.Nc + u;
  float q = 0.f;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int c = lane * E + e;
    const float m = HvaElem<T>::ld(X + ((size_t)bh * g.n + tok) * D + c);
    mu[row * D + c] = m;
    if (sp.hi) {
      const __nv_bfloat16 h = __float2bfloat16_rn(m);
      sp.hi[row * D + c] = h;
      sp.lo[row * D + c] = __float2bfloat16_rn(m - __bfloat162float(h));
      q = fmaf(m, m, q);
    }
  }
  if (sp.hi) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
    if (lane == 0) sp.musq[row] = q;
  }
}

template <typename T, int D>
__global__ void __launch_bounds__(kThreads) hva_assign_kernel(ClusterParams p) {
  constexpr int kVec = 16 / sizeof(T);          // elements per 16-byte chunk
  constexpr int kRowStride = D + kVec;          // padded row (elements): conflict-free 16 B row reads
  const HvaGrid& g = p.g;
  const int cell = blockIdx.x, bh = blockIdx.y, tid = threadIdx.x;
  const int ut = cell / (g.Kh * g.Kw), uh = (cell / g.Kw) % g.Kh, uw = cell % g.Kw;
  const int st = hva_win_start(ut, g.wt, g.Kt), sh = hva_win_start(uh, g.wh, g.Kh), sw = hva_win_start(uw, g.ww, g.Kw);
  const int ctok = g.kt * g.kh * g.kw;          // token slots of a cell (border cells: some invalid)

  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* s_mu = reinterpret_cast<float*>(smem_raw);                 // [nwin][D]
  T* s_x = reinterpret_cast<T*>(s_mu + (size_t)g.nwin * D);         // [ctok][kRowStride]
  int* s_lab = reinterpret_cast<int*>(s_x + (size_t)ctok * kRowStride);  // [ctok] slot or -1
  int* s_cnt = s_lab + ctok;                                        // [nwin]
  int* s_start = s_cnt + g.nwin;                                    // [nwin+1]
  int* s_order = s_start + g.nwin + 1;                              // [ctok]

  // ---- stage window centroids (ascending centroid id == delta_t-major, Alg. 2 line 18)
  const float* mu_b = p.mu + (size_t)bh * g.Nc * D;
  for (int i = tid; i < g.nwin * (D / 4); i += kThreads) {
    int v = i / (D / 4), q = i % (D / 4);
    int dt = v / (g.wh * g.ww), dh = (v / g.ww) % g.wh, dw = v % g.ww;
    int u = ((st + dt) * g.Kh + (sh + dh)) * g.Kw + (sw + dw);
    reinterpret_cast<float4*>(s_mu)[i] = reinterpret_cast<const float4*>(mu_b + (size_t)u * D)[q];
  }
  // ---- stage the cell's tokens (16-byte coalesced loads; runs of k_w consecutive tokens)
  const T* X_b = reinterpret_cast<const T*>(p.X) + (size_t)bh * g.n * D;
  constexpr int kChunks = D / kVec;
  for (int i = tid; i < ctok * kChunks; i += kThreads) {
    int li = i / kChunks, q = i % kChunks;
    int dt = li / (g.kh * g.kw), dh = (li / g.kw) % g.kh, dw = li % g.kw;
    int t = ut * g.kt + dt, h = uh * g.kh + dh, w = uw * g.kw + dw;
    if (t < g.T && h < g.H && w < g.W) {
      size_t tok = (size_t)(t * g.H + h) * g.W + w;
      *reinterpret_cast<uint4*>(s_x + (size_t)li * kRowStride + q * kVec) =
          __ldg(reinterpret_cast<const uint4*>(X_b + tok * D) + q);
    }
  }
  __syncthreads();

  // ---- one thread per token: distances to every window candidate (Eq. 5), best and second best
  for (int li = tid; li < ctok; li += kThreads) {
    int dt = li / (g.kh * g.kw), dh = (li / g.kw) % g.kh, dw = li % g.kw;
    int t = ut * g.kt + dt, h = uh * g.kh + dh, w = uw * g.kw + dw;
    bool valid = (t < g.T && h < g.H && w < g.W);
    int lab = valid ? 0 : -1;
    if (valid) {
      float best = __int_as_float(0x7f800000), second = __int_as_float(0x7f800000);
      const T* xr = s_x + (size_t)li * kRowStride;
      // the direct form in the summation order of cluster_tc.cuh (D/4 partial sums of 4 dims, halving tree): the labels and the
      // Lowe ratio of the tensor-pipe kernel are those of this kernel bit for bit
      for (int v = 0; v < g.nwin; ++v) {
        float pr[D / 4];
#pragma unroll
        for (int c0 = 0; c0 < D; c0 += 8) {
          float x[8];
          load8(xr + c0, x);
          const float4 m0 = *reinterpret_cast<const float4*>(s_mu + (size_t)v * D + c0);
          const float4 m1 = *reinterpret_cast<const float4*>(s_mu + (size_t)v * D + c0 + 4);
          pr[c0 / 4] = hva_tc_dev::hva_sq4(x[0], x[1], x[2], x[3], m0);
          pr[c0 / 4 + 1] = hva_tc_dev::hva_sq4(x[4], x[5], x[6], x[7], m1);
        }
        const float dd = hva_tc_dev::hva_tree_sum(pr);
        if (dd < best) { second = best; best = dd; lab = v; }
        else if (dd < second) second = dd;
      }
      size_t tok = (size_t)(t * g.H + h) * g.W + w;
      if (p.assign) {
        int dtv = lab / (g.wh * g.ww), dhv = (lab / g.ww) % g.wh, dwv = lab % g.ww;
        p.assign[(size_t)bh * g.n + tok] = ((st + dtv) * g.Kh + (sh + dhv)) * g.Kw + (sw + dwv);
      }
      if (p.lowe) {  // rho = d1/d2, unsquared (Eq. 6); single candidate -> 0; d2 == 0 -> 1 (R-H1)
        float rho = (second == __int_as_float(0x7f800000)) ? 0.f : (second > 0.f ? sqrtf(best / second) : 1.f);
        p.lowe[(size_t)bh * g.n + tok] = rho;
      }
    }
    s_lab[li] = lab;
  }
  __syncthreads();

  // ---- counting sort of the cell's tokens by slot (stable in token order)
  for (int v = tid; v < g.nwin; v += kThreads) {
    int c = 0;
    for (int li = 0; li < ctok; ++li) c += (s_lab[li] == v);
    s_cnt[v] = c;
  }
  __syncthreads();
  if (tid == 0) {
    int a = 0;
    for (int v = 0; v < g.nwin; ++v) { s_start[v] = a; a += s_cnt[v]; }
    s_start[g.nwin] = a;
  }
  __syncthreads();
  for (int v = tid; v < g.nwin; v += kThreads) {
    int pos = s_start[v];
    for (int li = 0; li < ctok; ++li)
      if (s_lab[li] == v) s_order[pos++] = li;
  }
  __syncthreads();

  // ---- segmented per-cell reduction: thread = feature dim, tokens added in token order (z_a += x)
  const size_t pbase = ((size_t)bh * g.Nc + cell) * g.nwin;
  constexpr int kGroups = kThreads / D;  // 1 for D=128, 2 for D=64
  const int c = tid % D, grp = tid / D;
  for (int v = grp; v < g.nwin; v += kGroups) {
    int b = s_start[v], e = s_start[v + 1];
    if (c == 0) p.part_cnt[pbase + v] = e - b;
    if (e > b) {
      float acc = 0.f;
      for (int i = b; i < e; ++i) acc += HvaElem<T>::ld(s_x + (size_t)s_order[i] * kRowStride + c);
      p.part[(pbase + v) * D + c] = acc;
    }
  }
}

// Home cells g (one axis) whose clipped window [start(g), start(g)+w) contains centroid coordinate u: a contiguous range.
__device__ __forceinline__ void axis_cells(int u, int w, int K, int& lo, int& cnt) {
  lo = 0; cnt = 0;
  for (int gc = max(0, u - w); gc <= min(K - 1, u + w); ++gc) {
    const int s0 = hva_win_start(gc, w, K);
    if (u >= s0 && u < s0 + w) { if (cnt == 0) lo = gc; ++cnt; }
  }
}

// mu_u <- z_u / n_u if n_u > 0 else mu_u   (Alg. 2 lines 22-23).  z_u = sum over the home cells g whose
// window contains u of part[g][slot(u in g)], in ascending cell order (fixed => deterministic).  One warp per centroid,
// four centroids per block, no shared memory and no block barrier: the lanes read the counts of up to 32 (cell, slot)
// partials at once, the non-empty ones are then walked in order (ballot bits), four row loads in flight, each lane adding
// its D/32 feature dims.
constexpr int kFinWarps = 4;
template <int D>
__global__ void __launch_bounds__(32 * kFinWarps) hva_finalize_kernel(HvaGrid g, const float* __restrict__ part,
                                                                      const int* __restrict__ part_cnt, float* __restrict__ mu,
                                                                      int* __restrict__ sizes, float* __restrict__ sums, MuSplit sp,
                                                                      int csplit) {
  constexpr int V = D / 32;
  const int lane = threadIdx.x & 31, u = blockIdx.x * kFinWarps + (threadIdx.x >> 5), bh = blockIdx.y;
  if (u >= g.Nc) return;
  const int ut = u / (g.Kh * g.Kw), uh = (u / g.Kw) % g.Kh, uw = u % g.Kw;
  int lt, nt, lh, nh, lw, nw;
  axis_cells(ut, g.wt, g.Kt, lt, nt);
  axis_cells(uh, g.wh, g.Kh, lh, nh);
  axis_cells(uw, g.ww, g.Kw, lw, nw);
  const int total = nt * nh * nw * csplit;      // (home cell, t-tile of the cell) partials, ascending cell then tile
  float z[V];
#pragma unroll
  for (int i = 0; i < V; ++i) z[i] = 0.f;
  int n = 0;
  auto row = [&](unsigned id, float (&r)[V]) {
    const float* q = part + (size_t)id * D + lane * V;
    if constexpr (V == 4) { const float4 t = *reinterpret_cast<const float4*>(q); r[0] = t.x; r[1] = t.y; r[2] = t.z; r[3] = t.w; }
    else { const float2 t = *reinterpret_cast<const float2*>(q); r[0] = t.x; r[1] = t.y; }
  };
  for (int e0 = 0; e0 < total; e0 += 32) {
    const int e = e0 + lane;
    int k = 0;
    unsigned idx = 0;
    if (e < total) {
      const int ce = e / csplit, chunk = e - ce * csplit;
      const int gt = lt + ce / (nh * nw), gh = lh + (ce / nw) % nh, gw = lw + ce % nw;
      const int cell = (gt * g.Kh + gh) * g.Kw + gw;
      const int slot = ((ut - hva_win_start(gt, g.wt, g.Kt)) * g.wh + (uh - hva_win_start(gh, g.wh, g.Kh))) * g.ww +
                       (uw - hva_win_start(gw, g.ww, g.Kw));
      idx = (unsigned)((((size_t)bh * g.Nc + cell) * csplit + chunk) * g.nwin + slot);
      k = part_cnt[idx];
    }
    unsigned bal = __ballot_sync(0xffffffffu, k > 0);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) k += __shfl_xor_sync(0xffffffffu, k, o);
    n += k;
    while (bal) {      // ascending partial order, up to four rows in flight
      unsigned id[4];
      int cnt = 0;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int b = bal ? __ffs(bal) - 1 : 0;
        id[j] = __shfl_sync(0xffffffffu, idx, b);
        if (bal) { ++cnt; bal &= bal - 1; }
      }
      float r[4][V];
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (j < cnt) row(id[j], r[j]);
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (j < cnt) {
#pragma unroll
          for (int i = 0; i < V; ++i) z[i] += r[j][i];
        }
    }
  }
  const size_t o = ((size_t)bh * g.Nc + u) * D + lane * V;
  float m[V];
  float q = 0.f;
  auto ld = [&](const float* a, float (&r)[V]) {
    if constexpr (V == 4) { const float4 t = *reinterpret_cast<const float4*>(a); r[0] = t.x; r[1] = t.y; r[2] = t.z; r[3] = t.w; }
    else { const float2 t = *reinterpret_cast<const float2*>(a); r[0] = t.x; r[1] = t.y; }
  };
  auto stv = [&](float* a, const float (&r)[V]) {
    if constexpr (V == 4) *reinterpret_cast<float4*>(a) = make_float4(r[0], r[1], r[2], r[3]);
    else *reinterpret_cast<float2*>(a) = make_float2(r[0], r[1]);
  };
  if (n > 0) {
#pragma unroll
    for (int i = 0; i < V; ++i) m[i] = __fdiv_rn(z[i], (float)n);
    stv(mu + o, m);
  } else {
    ld(mu + o, m);
  }
  if (sums) stv(sums + o, z);
#pragma unroll
  for (int i = 0; i < V; ++i) q = fmaf(m[i], m[i], q);
  if (lane == 0) sizes[(size_t)bh * g.Nc + u] = n;
  if (sp.hi) {
    __nv_bfloat162 h2[V / 2], l2[V / 2];
#pragma unroll
    for (int i = 0; i < V; i += 2) {
      const __nv_bfloat16 h0 = __float2bfloat16_rn(m[i]), h1 = __float2bfloat16_rn(m[i + 1]);
      h2[i / 2] = __nv_bfloat162(h0, h1);
      l2[i / 2] = __nv_bfloat162(__float2bfloat16_rn(m[i] - __bfloat162float(h0)), __float2bfloat16_rn(m[i + 1] - __bfloat162float(h1)));
    }
    if constexpr (V == 4) {
      *reinterpret_cast<uint2*>(sp.hi + o) = *reinterpret_cast<const uint2*>(h2);
      *reinterpret_cast<uint2*>(sp.lo + o) = *reinterpret_cast<const uint2*>(l2);
    } else {
      *reinterpret_cast<__nv_bfloat162*>(sp.hi + o) = h2[0];
      *reinterpret_cast<__nv_bfloat162*>(sp.lo + o) = l2[0];
    }
#pragma unroll
    for (int s2 = 16; s2 > 0; s2 >>= 1) q += __shfl_xor_sync(0xffffffffu, q, s2);
    if (lane == 0) sp.musq[(size_t)bh * g.Nc + u] = q;
  }
}

size_t assign_smem_bytes(const HvaGrid& g, int D, int esize) {
  int ctok = g.kt * g.kh * g.kw;
  int rowstride = D + 16 / esize;
  return (size_t)g.nwin * D * 4 + (size_t)ctok * rowstride * esize + sizeof(int) * (ctok + g.nwin + g.nwin + 1 + ctok) + 16;
}

struct ClusterWs {
  float* part; int* part_cnt; __nv_bfloat16 *hi, *lo; float* musq; int* counter; float* xsq;
};

template <typename T, int D>
int run_cluster(const HvaGrid& g, int BH, int iters, const void* X, const float* mu_init, int* assign, float* mu,
                int* sizes, float* sums, float* lowe, const ClusterWs& ws, int dtype, uint32_t flags, float* probe, cudaStream_t st) {
  dim3 grid(g.Nc, BH);
  const bool tc = hva_assign_tc_supported(g, D, dtype) && !(flags & HVA_FLAG_CLUSTER_SIMT);
  if (!tc) probe = nullptr;
  HvaAssignTc atc;
  size_t smem = 0;
  if (tc) {
    HVA_TRY(hva_assign_tc_prepare(g, BH, X, ws.hi, ws.lo, probe != nullptr, &atc));
  } else {
    smem = assign_smem_bytes(g, D, sizeof(T));
    if (smem > 227 * 1024) return HVA_EUNSUPPORTED;
    if (cudaFuncSetAttribute(hva_assign_kernel<T, D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
      return HVA_ECUDA;
  }
  const MuSplit sp{tc ? ws.hi : nullptr, tc ? ws.lo : nullptr, ws.musq}, none{nullptr, nullptr, nullptr};
  if (mu_init) {
    if (mu_init != mu &&
        cudaMemcpyAsync(mu, mu_init, (size_t)BH * g.Nc * D * sizeof(float), cudaMemcpyDeviceToDevice, st) != cudaSuccess)
      return HVA_ECUDA;
  } else {
    hva_init_centroids_kernel<T, D><<<dim3((g.Nc + kInitWarps - 1) / kInitWarps, BH), 32 * kInitWarps, 0, st>>>(
        g, reinterpret_cast<const T*>(X), mu, tc ? sp : none);
    HVA_CHECK_LAUNCH();
  }
  if (tc && mu_init) {
    hva_mu_split_kernel<D><<<grid, D, 0, st>>>(g.Nc, mu, sp);
    HVA_CHECK_LAUNCH();
  }
  for (int it = 0; it < iters; ++it) {
    bool last = (it == iters - 1);
    if (tc) {
      // the |x|^2 bound of the filter margin is the same in every pass: written by the first, read by the others
      HVA_TRY(hva_assign_tc_launch(atc, g, BH, mu, ws.musq, ws.part, ws.part_cnt, last ? assign : nullptr, last ? lowe : nullptr,
                                   ws.xsq, iters == 1 ? 0 : (it == 0 ? 1 : 2), ws.counter, probe, st));
    } else {
      ClusterParams p{g, BH, X, mu, ws.part, ws.part_cnt, last ? assign : nullptr, last ? lowe : nullptr};
      hva_assign_kernel<T, D><<<grid, kThreads, smem, st>>>(p);
      HVA_CHECK_LAUNCH();
    }
    hva_finalize_kernel<D><<<dim3((g.Nc + kFinWarps - 1) / kFinWarps, BH), 32 * kFinWarps, 0, st>>>(g, ws.part, ws.part_cnt, mu, sizes, last ? sums : nullptr, last ? none : sp, tc ? atc.csplit : 1);
    HVA_CHECK_LAUNCH();
  }
  return HVA_OK;
}

}  // namespace

size_t hva_cluster_ws_bytes(const HvaGrid& g, int BH, int D) {
  const size_t cs = (size_t)hva_assign_tc_csplit(g);
  return hva_align((size_t)BH * g.Nc * cs * g.nwin * D * sizeof(float)) + hva_align((size_t)BH * g.Nc * cs * g.nwin * sizeof(int)) +
         2 * hva_align((size_t)BH * g.Nc * D * sizeof(__nv_bfloat16)) + hva_align((size_t)BH * g.Nc * sizeof(float)) + hva_align(sizeof(int)) +
         hva_align((size_t)BH * g.n * sizeof(float));
}

int hva_mu_split_launch(int BH, int Nc, int D, const float* mu, void* mu_hi, void* mu_lo, float* musq, cudaStream_t st) {
  const MuSplit sp{reinterpret_cast<__nv_bfloat16*>(mu_hi), reinterpret_cast<__nv_bfloat16*>(mu_lo), musq};
  if (D == 128) hva_mu_split_kernel<128><<<dim3(Nc, BH), 128, 0, st>>>(Nc, mu, sp);
  else if (D == 64) hva_mu_split_kernel<64><<<dim3(Nc, BH), 64, 0, st>>>(Nc, mu, sp);
  else return HVA_EINVAL;
  HVA_CHECK_LAUNCH();
  return HVA_OK;
}

extern "C" size_t hva_cluster_workspace_bytes(const hva_shape* s, const int32_t cell[3], const int32_t win[3]) {
  if (!s || !cell || !win || s->B < 1 || s->heads < 1 || s->T < 1 || s->H < 1 || s->W < 1) return 0;
  for (int a = 0; a < 3; ++a)
    if (cell[a] < 1 || win[a] < 1) return 0;
  return hva_cluster_ws_bytes(hva_make_grid(s, cell, win), s->B * s->heads, s->D);
}

extern "C" int hva_cluster(const hva_shape* s, const int32_t cell[3], const int32_t win[3], int32_t iters, const void* X,
                           const float* mu_init, int32_t* assign, float* mu, int32_t* sizes, float* sums, float* lowe,
                           void* ws, size_t ws_bytes, void* stream) {
  return hva_cluster_ex(s, cell, win, iters, X, mu_init, assign, mu, sizes, sums, lowe, 0u, nullptr, ws, ws_bytes, stream);
}

extern "C" int hva_cluster_ex(const hva_shape* s, const int32_t cell[3], const int32_t win[3], int32_t iters, const void* X,
                              const float* mu_init, int32_t* assign, float* mu, int32_t* sizes, float* sums, float* lowe,
                              uint32_t flags, float* probe, void* ws, size_t ws_bytes, void* stream) {
  if (!s || !cell || !win || !X || !assign || !mu || !sizes || !ws) return HVA_EINVAL;
  if (s->B < 1 || s->heads < 1 || s->T < 1 || s->H < 1 || s->W < 1 || iters < 1) return HVA_EINVAL;
  if (s->D != 64 && s->D != 128) return HVA_EINVAL;
  for (int a = 0; a < 3; ++a)
    if (cell[a] < 1 || win[a] < 1) return HVA_EINVAL;
  if (s->dtype != HVA_F32 && s->dtype != HVA_BF16) return HVA_EUNSUPPORTED;
  HvaGrid g = hva_make_grid(s, cell, win);
  int BH = s->B * s->heads;
  if ((size_t)g.nwin * hva_assign_tc_csplit(g) > 1024 || (size_t)BH * g.Nc * g.nwin * hva_assign_tc_csplit(g) >= (1ull << 32)) return HVA_EUNSUPPORTED;
  if (ws_bytes < hva_cluster_ws_bytes(g, BH, s->D)) return HVA_EWORKSPACE;
  ClusterWs cw;
  {
    char* w = reinterpret_cast<char*>(ws);
    const size_t cs = (size_t)hva_assign_tc_csplit(g);
    cw.part = reinterpret_cast<float*>(w); w += hva_align((size_t)BH * g.Nc * cs * g.nwin * s->D * sizeof(float));
    cw.part_cnt = reinterpret_cast<int*>(w); w += hva_align((size_t)BH * g.Nc * cs * g.nwin * sizeof(int));
    cw.hi = reinterpret_cast<__nv_bfloat16*>(w); w += hva_align((size_t)BH * g.Nc * s->D * sizeof(__nv_bfloat16));
    cw.lo = reinterpret_cast<__nv_bfloat16*>(w); w += hva_align((size_t)BH * g.Nc * s->D * sizeof(__nv_bfloat16));
    cw.musq = reinterpret_cast<float*>(w); w += hva_align((size_t)BH * g.Nc * sizeof(float));
    cw.counter = reinterpret_cast<int*>(w); w += hva_align(sizeof(int));
    cw.xsq = reinterpret_cast<float*>(w);
  }
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
#define HVA_DISPATCH(T, DD) return run_cluster<T, DD>(g, BH, iters, X, mu_init, assign, mu, sizes, sums, lowe, cw, s->dtype, flags, probe, st)
  if (s->dtype == HVA_F32) {
    if (s->D == 64) HVA_DISPATCH(float, 64);
    HVA_DISPATCH(float, 128);
  } else {
    if (s->D == 64) HVA_DISPATCH(__nv_bfloat16, 64);
    HVA_DISPATCH(__nv_bfloat16, 128);
  }
#undef HVA_DISPATCH
}
