// H8: per-template top-k over bins (PAPER.md:214 max over the band, :307 GPU-side retention).
// Order: descending 2F, ties -> lower bin first (S15).
#pragma once
#include "fstat_common.cuh"

#define TOPK_THREADS 256
#define TOPK_MAX_GROUPS ((1 << 24) / 512)     // groups of 512 bins per row at the largest n_fft

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

// How FFT pass 2 lays one warp's 32 x elems outputs ("group") over the bins of a row: element e (0..15) of
// lane l of warp wp of tile x is bin q (fft_kernels.cuh, pass-2 epilogue).
struct TopkGeom {
    int elems;       // register elements per thread of pass 2 (16 or 32): a group is 32 * elems bins
    int nt;          // threads per pass-2 CTA
    int log_w;       // log2(rows per tile)
    int log_rl;      // log2(last radix)
    int pl;          // product of the earlier radices
    int log_other;   // log2(N1)
    int n_groups;    // groups per row = tiles per template * warps per CTA
    int linear;      // != 0: rows not written by pass 2 (fstat_select_*): group g is bins [512 g, 512 g + 512), maxima from group_max_kernel
};
__device__ __forceinline__ int64_t topk_group_bin(const TopkGeom &tg, int group, int lane, int e) {
    if (tg.linear) return (int64_t)group * 512 + e * 32 + lane;
    const int warps = tg.nt >> 5;
    const int x = group / warps, wp = group - x * warps;
    const int rl = 1 << tg.log_rl;
    const int bb = e >> tg.log_rl, r = e & (rl - 1);
    const int g = wp * 32 + lane + bb * tg.nt;
    const int w = g & ((1 << tg.log_w) - 1), i = g >> tg.log_w;
    const int k = i & (tg.pl - 1);
    const int oi = ((i - k) << tg.log_rl) + k + r * tg.pl;
    return ((int64_t)oi << tg.log_other) + ((int64_t)x << tg.log_w) + w;
}

#define TOPK_HOT_CAP 512
#define TOPK_CAND_CAP 2048

// One block per row.  FFT pass 2 has left, next to the 2F row, the maximum of every group of 512 bins
// (as topk_key).  The k-th largest group maximum L is a lower bound of the k-th largest bin (k groups
// hold a value >= L), so only groups whose maximum is >= L ("hot": k of them, plus ties) can hold
// one of the k loudest bins: they are re-read, their values >= L collected, and the k best picked
// with the tie rule.  Exact.  Degenerate rows (more ties than the caps, NaN rows) take a slow exact
// path that scans the whole row once per output.
__global__ void __launch_bounds__(TOPK_THREADS)
topk_select_kernel(const float *__restrict__ twoF, int64_t row_stride, int64_t n_bins, int k,
                   const uint32_t *__restrict__ gmax, const __grid_constant__ TopkGeom tg,
                   float *__restrict__ out_v, int *__restrict__ out_i,
                   float thr, int *__restrict__ out_count) {
    extern __shared__ uint32_t s_g[];                 // [n_groups] keys
    __shared__ int s_hist[256];
    __shared__ uint32_t s_prefix;
    __shared__ int s_remaining, s_nhot, s_ncand;
    __shared__ int s_hot[TOPK_HOT_CAP];
    __shared__ float s_cv[TOPK_CAND_CAP];
    __shared__ int s_ci[TOPK_CAND_CAP];
    __shared__ float s_v[TOPK_THREADS / 32];
    __shared__ int s_i[TOPK_THREADS / 32];
    const float *row = twoF + (int64_t)blockIdx.x * row_stride;
    const uint32_t *gm = gmax + (int64_t)blockIdx.x * tg.n_groups;
    float *ov = out_v + (int64_t)blockIdx.x * k;
    int *oi = out_i + (int64_t)blockIdx.x * k;
    const float NEG = __int_as_float(0xff800000);
    const int G = tg.n_groups;
    for (int g = threadIdx.x; g < G; g += TOPK_THREADS) s_g[g] = gm[g];
    __shared__ int s_count;
    if (threadIdx.x == 0) { s_prefix = 0u; s_remaining = k; s_nhot = 0; s_ncand = 0; s_count = 0; }
    __syncthreads();
    // threshold mode (out_count != null): only bins with 2F > thr are reported, and their exact number
    // is counted by re-reading the groups whose maximum exceeds thr
    const bool thr_mode = (out_count != nullptr);
    if (thr_mode) {
        const uint32_t kt = topk_key(thr);
        const int lane = threadIdx.x & 31;
        for (int g0 = (threadIdx.x >> 5); g0 < G; g0 += TOPK_THREADS / 32) {
            if (s_g[g0] <= kt) continue;                      // uniform per warp
            int c = 0;
#pragma unroll 4
            for (int e = 0; e < tg.elems; ++e) {
                const int64_t q = topk_group_bin(tg, g0, lane, e);
                if (q < n_bins && row[q] > thr) ++c;
            }
            c = __reduce_add_sync(0xffffffffu, c);
            if (lane == 0 && c) atomicAdd(&s_count, c);
        }
        __syncthreads();
        if (threadIdx.x == 0) out_count[blockIdx.x] = s_count;
    }
    bool slow = (G < k);
    uint32_t L = 0u;
    if (!slow) {
        // radix select (4 x 8 bits) of the k-th largest key
        uint32_t mask = 0u;
        for (int shift = 24; shift >= 0; shift -= 8) {
            s_hist[threadIdx.x] = 0;
            __syncthreads();
            const uint32_t prefix = s_prefix;
            for (int g = threadIdx.x; g < G; g += TOPK_THREADS) {
                const uint32_t key = s_g[g];
                if ((key & mask) == prefix) atomicAdd(&s_hist[(key >> shift) & 255u], 1);
            }
            __syncthreads();
            if (threadIdx.x == 0) {
                int rem = s_remaining, d = 255;
                for (; d > 0; --d) {
                    const int c = s_hist[d];
                    if (c >= rem) break;
                    rem -= c;
                }
                s_remaining = rem;
                s_prefix = prefix | ((uint32_t)d << shift);
            }
            mask |= 0xffu << shift;
            __syncthreads();
        }
        L = s_prefix;
        // hot groups
        for (int g = threadIdx.x; g < G; g += TOPK_THREADS)
            if (s_g[g] >= L) {
                const int pos = atomicAdd(&s_nhot, 1);
                if (pos < TOPK_HOT_CAP) s_hot[pos] = g;
            }
        __syncthreads();
        slow = (s_nhot > TOPK_HOT_CAP) || (L <= topk_key(NEG));
    }
    if (!slow) {
        const int nhot = s_nhot, lane = threadIdx.x & 31;
        for (int h = threadIdx.x >> 5; h < nhot; h += TOPK_THREADS / 32) {
            const int g = s_hot[h];
#pragma unroll 4
            for (int e = 0; e < tg.elems; ++e) {
                const int64_t q = topk_group_bin(tg, g, lane, e);
                if (q < n_bins) {
                    const float v = row[q];
                    if (topk_key(v) >= L) {
                        const int pos = atomicAdd(&s_ncand, 1);
                        if (pos < TOPK_CAND_CAP) { s_cv[pos] = v; s_ci[pos] = (int)q; }
                    }
                }
            }
        }
        __syncthreads();
        slow = s_ncand > TOPK_CAND_CAP;
    }
    if (!slow) {
        const int nc = s_ncand;
        for (int round = 0; round < k; ++round) {
            float v = NEG; int i = 0x7fffffff; int pos = -1;
            for (int t = threadIdx.x; t < nc; t += TOPK_THREADS) {
                const float x = s_cv[t]; const int b = s_ci[t];
                if (b >= 0 && topk_better(x, b, v, i)) { v = x; i = b; pos = t; }
            }
            const float myv = v; const int myi = i;
            block_argbest(v, i, s_v, s_i);
            if (pos >= 0 && myi == i && myv == v) s_ci[pos] = -1;    // winner removes itself (bins are unique)
            if (threadIdx.x == 0) {
                const bool ok = (i != 0x7fffffff) && (!thr_mode || v > thr);
                ov[round] = ok ? v : NEG;
                oi[round] = ok ? i : -1;
            }
            __syncthreads();
        }
        return;
    }
    // slow exact path: output r is the best bin that is worse than output r-1 in the (2F desc, bin asc) order
    float pv = __int_as_float(0x7f800000); int pi = -1;
    for (int round = 0; round < k; ++round) {
        float v = NEG; int i = 0x7fffffff;
        for (int64_t q = threadIdx.x; q < n_bins; q += TOPK_THREADS) {
            const float x = row[q];
            const bool after_prev = (x < pv) || (x == pv && (int)q > pi);
            if (after_prev && x > NEG && topk_better(x, (int)q, v, i)) { v = x; i = (int)q; }
        }
        block_argbest(v, i, s_v, s_i);
        const bool ok = (i != 0x7fffffff) && (!thr_mode || v > thr);
        if (threadIdx.x == 0) { ov[round] = ok ? v : NEG; oi[round] = ok ? i : -1; }
        if (!ok) {
            for (int r2 = round + 1 + threadIdx.x; r2 < k; r2 += TOPK_THREADS) { ov[r2] = NEG; oi[r2] = -1; }
            return;
        }
        pv = v; pi = i;
    }
}


// Per-group maxima (as topk_key) of rows that did not come out of FFT pass 2 in this call -- e.g. the sum of 2F over the
// segments of a semi-coherent search -- in the linear group layout: one warp per group of 512 bins.
// grid = (ceil(n_groups / 8), n_rows), 256 threads.
__global__ void __launch_bounds__(TOPK_THREADS)
group_max_kernel(const float *__restrict__ rows, int64_t row_stride, int64_t n_bins, int n_groups, uint32_t *__restrict__ gmax) {
    const int g = blockIdx.x * (TOPK_THREADS / 32) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (g >= n_groups) return;
    const float *row = rows + (int64_t)blockIdx.y * row_stride;
    uint32_t key = 0u;
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const int64_t q = (int64_t)g * 512 + e * 32 + lane;
        if (q < n_bins) key = max(key, topk_key(row[q]));
    }
    key = __reduce_max_sync(0xffffffffu, key);
    if (lane == 0) gmax[(int64_t)blockIdx.y * n_groups + g] = key;
}
