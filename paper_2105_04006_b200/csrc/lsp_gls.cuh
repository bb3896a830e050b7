// lsp_gls.cuh -- generalised Lomb-Scargle periodogram (floating mean + per-point errors; Zechmeister &
// Kuerster 2009) on top of the standard path's contraction kernels.
//
// With w_j = sigma_j^-2 / sum sigma^-2, ybar = sum w y and theta = 2 pi f t, the chi^2 reduction of the weighted fit of
// a cos + b sin + c relative to the constant model is (ZK09 Eq. 4-5, hatted sums)
//     P = (SS YC^2 + CC YS^2 - 2 CS YC YS) / (YY D),   D = CC SS - CS^2,
//     YC = sum w (y - ybar) cos,  YS = sum w (y - ybar) sin,  YY = sum w (y - ybar)^2,
//     CC = 1/2 (1 + c2) - C^2,  SS = 1/2 (1 - c2) - S^2,  CS = 1/2 s2 - C S,
//     C + i S = sum w e^{i theta},   c2 + i s2 = sum w e^{2 i theta}.
// The standard kernels evaluate two slots per frequency, Z = sum x e^{i theta} and W = sum e^{2 i theta}.  With the W slot
// carrying the weights (the kernels' WGT variants: W = sum w e^{2 i theta}) two passes in their partial-sum form give all six sums:
//     pass 1: x = w (y - ybar), W weighted   -> (YC, YS) and (c2, s2)
//     pass 2: x = w                           -> (C, S)    (the tensor path skips the W contraction and reuses pass 1's table)
// and lsp_gls_combine_kernel finishes.  Cost: 2x the standard periodogram on the FMA-pipe kernels, ~1.5x on the tensor path
// (the paper's own implementation: 2.06-2.14x, L419).
#pragma once
#include "lsp_direct.cuh"

namespace lsp {

// One CTA per object: weights, weighted mean, chi0^2; writes x_A = w (y - ybar) and x_B = w in the plan's dtype.
template <typename T>
__global__ void __launch_bounds__(256)
lsp_gls_prep_kernel(const int64_t* __restrict__ offsets, const T* __restrict__ y, const T* __restrict__ sigma,
                    T* __restrict__ xa, T* __restrict__ xb, double* __restrict__ yy)
{
    __shared__ double red[8];
    __shared__ double bcast;
    const int64_t obj = blockIdx.x;
    const int64_t lo = offsets[obj], n = offsets[obj + 1] - lo;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    auto block_sum = [&](double v) {
        for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
        __syncthreads();
        if (lane == 0) red[wid] = v;
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = 0.0;
            for (int i = 0; i < 8; ++i) s += red[i];
            bcast = s;
        }
        __syncthreads();
        return bcast;
    };
    double acc = 0.0;
    for (int64_t j = threadIdx.x; j < n; j += blockDim.x) {
        const double s = (double)sigma[lo + j];
        acc += 1.0 / (s * s);
    }
    const double wsum = block_sum(acc);
    acc = 0.0;
    for (int64_t j = threadIdx.x; j < n; j += blockDim.x) {
        const double s = (double)sigma[lo + j];
        acc += (1.0 / (s * s) / wsum) * (double)y[lo + j];
    }
    const double ybar = block_sum(acc);
    acc = 0.0;
    for (int64_t j = threadIdx.x; j < n; j += blockDim.x) {
        const double s = (double)sigma[lo + j];
        const double w = 1.0 / (s * s) / wsum, d = (double)y[lo + j] - ybar;
        acc += w * d * d;
        xa[lo + j] = (T)(w * d);
        xb[lo + j] = (T)w;
    }
    const double chi0 = block_sum(acc);
    if (threadIdx.x == 0) yy[obj] = (n > 0) ? chi0 : 0.0;
}

// Combine the two passes' partial sums (fixed split order: deterministic) and evaluate P; same launch geometry and
// argmax partials as lsp_combine_kernel.
template <typename T>
__global__ void __launch_bounds__(kCombineThreads)
lsp_gls_combine_kernel(GridParams gp, const double* __restrict__ yy, const typename Vec4<T>::type* __restrict__ sa,
                       const typename Vec4<T>::type* __restrict__ sb,
                       T* __restrict__ out_power, Best* __restrict__ partials, int n_parts, int64_t n_obj_launch)
{
    __shared__ Best sbest[kCombineThreads / 32];
    const int64_t obj_local = blockIdx.x / n_parts;
    const int part = (int)(blockIdx.x % n_parts);
    const double chi0 = yy[obj_local + gp.obj_base];
    const double d_eps = sizeof(T) == 4 ? 1e-5 : 1e-12;
    Best mine;
    mine.p = -1.0;
    mine.k = INT64_MAX;
#pragma unroll
    for (int r = 0; r < kCombinePerThread; ++r) {
        const int64_t k = ((int64_t)part * kCombinePerThread + r) * kCombineThreads + threadIdx.x;
        if (k >= gp.n_freq) continue;
        double YC = 0, YS = 0, C = 0, S = 0, c2 = 0, s2 = 0;
        for (int s = 0; s < gp.n_split; ++s) {
            const int64_t at = ((int64_t)s * n_obj_launch + obj_local) * gp.n_freq + k;
            const typename Vec4<T>::type a = sa[at], b = sb[at];
            YC += (double)a.x; YS += (double)a.y;
            c2 += (double)a.z; s2 += (double)a.w;
            C += (double)b.x;  S += (double)b.y;
        }
        const double CC = 0.5 * (1.0 + c2) - C * C, SS = 0.5 * (1.0 - c2) - S * S, CS = 0.5 * s2 - C * S;
        const double D = CC * SS - CS * CS;
        double p = 0.0;
        if (chi0 > 0.0) {
            if (D > d_eps) p = (SS * YC * YC + CC * YS * YS - 2.0 * CS * YC * YS) / (chi0 * D);
            else if (CC > d_eps) p = YC * YC / (CC * chi0);        // aliased design matrix: the vanishing direction is dropped
            else if (SS > d_eps) p = YS * YS / (SS * chi0);
        }
        if (out_power) out_power[obj_local * gp.n_freq + k] = (T)p;
        Best b;
        b.p = (p == p) ? (double)(T)p : -1.0;
        b.k = k;
        mine = best_of(mine, b);
    }
    if (partials) {
        const Best b = block_best(mine, sbest);
        if (threadIdx.x == 0) partials[obj_local * n_parts + part] = b;
    }
}

}  // namespace lsp
