// Interface between cluster.cu (iteration driver, centroid update) and cluster_tc.cu (tensor-pipe assignment).
#pragma once
#include "common.cuh"
#include <cuda.h>

struct HvaAssignTc {
  CUtensorMap map_x, map_hi, map_lo;
  int npad, rows_a;
  uint32_t tmem_cols;
  size_t smem;
};

// bf16, D = 128, cell of at most 128 tokens, window of at most 256 centroids
bool hva_assign_tc_supported(const HvaGrid& g, int D, int dtype);
// X[BH,T,H,W,128] bf16; mu_hi / mu_lo [BH,Kt,Kh,Kw,128] bf16 (two-term split of the fp32 centroids)
int hva_assign_tc_prepare(const HvaGrid& g, int BH, const void* X, const void* mu_hi, const void* mu_lo, HvaAssignTc* out);
int hva_assign_tc_launch(const HvaAssignTc& a, const HvaGrid& g, int BH, const float* mu, const float* musq, float* part,
                         int* part_cnt, int* assign, float* lowe, float* probe, cudaStream_t st);
