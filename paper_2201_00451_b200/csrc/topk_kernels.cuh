// H8: per-template top-k over bins (PAPER.md:214 max over the band, :307 GPU-side retention).
// Order: descending 2F, ties -> lower bin first (S15).
#pragma once
#include "fstat_common.cuh"

#define TOPK_THREADS 256
#define TOPK_SLICE 8192          // bins per block in the first stage

// "a is better than b"
__device__ __forceinline__ bool topk_better(float va, int ia, float vb, int ib) {
    return (va > vb) || (va == vb && ia < ib);
}

// Block-wide arg-best by warp shuffles; result valid in every thread.
__device__ __forceinline__ void block_argbest(float &v, int &i, float *s_v, int *s_i) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(0xffffffffu, v, o);
        const int oi = __shfl_xor_sync(0xffffffffu, i, o);
        if (topk_better(ov, oi, v, i)) { v = ov; i = oi; }
    }
    const int wid = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { s_v[wid] = v; s_i[wid] = i; }
    __syncthreads();
    v = s_v[0]; i = s_i[0];
#pragma unroll
    for (int w = 1; w < TOPK_THREADS / 32; ++w)
        if (topk_better(s_v[w], s_i[w], v, i)) { v = s_v[w]; i = s_i[w]; }
    __syncthreads();
}

// Stage 1: grid = (ceil(n_bins / TOPK_SLICE), n_rows).  Each block selects the k best of its
// slice by k rounds of block-wide arg-best over a shared-memory copy, removing the winner.
// NaN rows (D <= 0) compare false everywhere and come out as (-inf, -1).
__global__ void __launch_bounds__(TOPK_THREADS)
topk_stage1_kernel(const float *__restrict__ twoF, int64_t row_stride, int64_t n_bins, int k,
                   float *__restrict__ cand_v, int *__restrict__ cand_i /* [n_rows][gridDim.x][k] */) {
    __shared__ float s_val[TOPK_SLICE];
    __shared__ float s_v[TOPK_THREADS / 32];
    __shared__ int s_i[TOPK_THREADS / 32];
    const float *row = twoF + (int64_t)blockIdx.y * row_stride;
    const int64_t q0 = (int64_t)blockIdx.x * TOPK_SLICE;
    const int n = (int)min((int64_t)TOPK_SLICE, n_bins - q0);
    const float NEG = __int_as_float(0xff800000);
    for (int t = threadIdx.x; t < TOPK_SLICE; t += TOPK_THREADS) s_val[t] = (t < n) ? __ldcs(row + q0 + t) : NEG;
    __syncthreads();
    float *ov = cand_v + ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * k;
    int *oi = cand_i + ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * k;
    for (int round = 0; round < k; ++round) {
        float v = NEG; int i = 0x7fffffff;
        for (int t = threadIdx.x; t < TOPK_SLICE; t += TOPK_THREADS) {
            const float x = s_val[t];
            if (topk_better(x, t, v, i)) { v = x; i = t; }
        }
        block_argbest(v, i, s_v, s_i);
        if (threadIdx.x == 0) {
            const bool ok = (i != 0x7fffffff) && (v > NEG);
            ov[round] = ok ? v : NEG;
            oi[round] = ok ? (int)(q0 + i) : -1;
            if (ok) s_val[i] = NEG;
        }
        __syncthreads();
    }
}

// Stage 2: one block per row merges the n_cand candidates into the final sorted top-k.
__global__ void __launch_bounds__(TOPK_THREADS)
topk_stage2_kernel(float *__restrict__ cand_v, int *__restrict__ cand_i, int n_cand, int k,
                   float *__restrict__ out_v, int *__restrict__ out_i) {
    __shared__ float s_v[TOPK_THREADS / 32];
    __shared__ int s_i[TOPK_THREADS / 32];
    float *cv = cand_v + (int64_t)blockIdx.x * n_cand;
    int *ci = cand_i + (int64_t)blockIdx.x * n_cand;
    const float NEG = __int_as_float(0xff800000);
    for (int round = 0; round < k; ++round) {
        float v = NEG; int i = 0x7fffffff; int pos = -1;
        for (int t = threadIdx.x; t < n_cand; t += TOPK_THREADS) {
            const float x = cv[t]; const int b = ci[t];
            if (b >= 0 && topk_better(x, b, v, i)) { v = x; i = b; pos = t; }
        }
        const float myv = v; const int myi = i;
        block_argbest(v, i, s_v, s_i);
        if (pos >= 0 && myi == i && myv == v) ci[pos] = -1;      // winner removes itself (bins are unique)
        if (threadIdx.x == 0) {
            const bool ok = (i != 0x7fffffff);
            out_v[(int64_t)blockIdx.x * k + round] = ok ? v : NEG;
            out_i[(int64_t)blockIdx.x * k + round] = ok ? i : -1;
        }
        __syncthreads();
    }
}
