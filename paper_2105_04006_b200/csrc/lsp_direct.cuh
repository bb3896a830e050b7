// lsp_direct.cuh -- the "direct" periodogram kernel family: one sincos per (t, f) pair, thread = frequency.
//
// This is the paper's own kernel shape (Listing 1: thread tid owns frequency tid and loops
// over the N_t observations; shared-memory tiling of the observations; batch mode: one
// object per block), re-cut for B200:
//   * work item = (object, frequency tile, observation split) instead of one block per object, so a single
//     object with few frequencies still fills 148 SMs (PAPER.md:L373, L396 note the under-filled GPU);
//   * each thread owns R frequencies strided by the block size, so the staged (t_j, y_j) are reused R times
//     from registers and the periodogram stores stay coalesced;
//   * FP32: the phase f_k*t_j is formed as a two-float product reduced to (-1/2, 1/2] cycles BEFORE the
//     sincos (BASELINE.json north_star "range-reduced phase frac(f t)"), then either MUFU.SIN/COS
//     (fast_math, the paper's __sincosf question) or sincospif;
//   * FP64: exact-product phase (fma) + sincospi: no Payne-Hanek slow path;
//   * four accumulators instead of Listing 1's five: ss = n - cc;
//   * the epilogue is the tau-free closed form (lsp_common.cuh) instead of atan2 + a second sincos;
//   * optional fused argmax writing one (power, index) partial per CTA.
// It is the comparison kernel for the fast-vs-accurate sincos question and the fallback for problems too
// small for the factored kernel; the flagship is lsp_factored.cuh.
#pragma once
#include "lsp_common.cuh"

namespace lsp {

template <typename T> struct Vec4;
template <> struct Vec4<float>  { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

template <typename T>
__device__ __forceinline__ typename Vec4<T>::type make_vec4(T a, T b, T c, T d);
template <> __device__ __forceinline__ float4 make_vec4<float>(float a, float b, float c, float d) { return make_float4(a, b, c, d); }
template <> __device__ __forceinline__ double4 make_vec4<double>(double a, double b, double c, double d) { return make_double4(a, b, c, d); }

// Frequency representation of one thread-owned frequency.
template <typename T> struct Freq;
template <> struct Freq<float> {
    float hi, lo;   // f = hi + lo to ~2^-48 relative
    __device__ __forceinline__ void set(double f) { hi = (float)f; lo = (float)(f - (double)hi); }
    // phase in cycles, reduced: f*t = ph + pe exactly for the hi part; the lo part only needs FP32.
    __device__ __forceinline__ float phase(float t) const
    {
        const float ph = hi * t;
        const float pe = fmaf(hi, t, -ph);
        const float q = ph - rintf(ph);
        return q + fmaf(lo, t, pe);
    }
};
template <> struct Freq<double> {
    double f;
    __device__ __forceinline__ void set(double v) { f = v; }
    __device__ __forceinline__ double phase(double t) const { return phase_cycles_exact(f, t); }
};

constexpr int kDirectThreads = 256;

// Work decode shared by both kernel families: blockIdx.x -> (object, tile, split).
struct WorkItem {
    int64_t obj_local;
    int tile, split;
};
__device__ __forceinline__ WorkItem decode_item(const GridParams& gp)
{
    WorkItem w;
    const int64_t item = blockIdx.x;
    w.split = (int)(item % gp.n_split);
    const int64_t r = item / gp.n_split;
    w.tile = (int)(r % gp.n_tiles);
    w.obj_local = r / gp.n_tiles;
    return w;
}

// WGT (generalised mode only, partial-sum output): the doubled-angle sums carry the weights, c2 + i s2 = sum w e^{2 i theta}.
template <typename T, bool FAST, int R, bool WGT = false>
__global__ void __launch_bounds__(kDirectThreads)
lsp_direct_kernel(GridParams gp, const int64_t* __restrict__ offsets, const T* __restrict__ t,
                  const T* __restrict__ y, const ObjStats* __restrict__ stats,
                  T* __restrict__ out_power, Best* __restrict__ partials,
                  typename Vec4<T>::type* __restrict__ sums, int64_t n_obj_launch, const T* __restrict__ wgt = nullptr)
{
    constexpr int TPB = kDirectThreads;
    constexpr int JC = 512;                       // observations staged per pass (tile = block)
    __shared__ T st[JC];
    __shared__ T sy[JC];
    __shared__ T sw[WGT ? JC : 1];
    T w_sum = T(0);
    __shared__ Best sbest[TPB / 32];

    const WorkItem wi = decode_item(gp);
    const int64_t obj = wi.obj_local + gp.obj_base;
    const int64_t lo = offsets[obj];
    const int64_t n_t = offsets[obj + 1] - lo;
    const int64_t j0 = (n_t * wi.split) / gp.n_split;
    const int64_t j1 = (n_t * (wi.split + 1)) / gp.n_split;
    const T mean = stats ? (T)stats[obj].mean : T(0);
    const int tid = threadIdx.x;

    Freq<T> fr[R];
    T xc[R], xs[R], cc[R], cs[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int64_t k = (int64_t)wi.tile * (TPB * R) + r * TPB + tid;
        fr[r].set(gp.f_min + (double)k * gp.df);               // PAPER.md:L53, Listing 1
        xc[r] = xs[r] = cc[r] = cs[r] = T(0);
    }

    for (int64_t jb = j0; jb < j1; jb += JC) {
        const int cnt = (int)min((int64_t)JC, j1 - jb);
        __syncthreads();
        for (int i = tid; i < cnt; i += TPB) {                 // step 2: coalesced staging
            st[i] = t[lo + jb + i];
            sy[i] = y[lo + jb + i] - mean;
            if (WGT) sw[i] = wgt[lo + jb + i];
        }
        __syncthreads();
#pragma unroll 4
        for (int j = 0; j < cnt; ++j) {                        // step 4: the per-pair hot loop
            const T tj = st[j], yj = sy[j];
            const T wj = WGT ? sw[j] : T(1);
            if (WGT) w_sum += wj;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                T s, c;
                const T ph = fr[r].phase(tj);
                sincos_cycles<FAST>(ph, &s, &c);
                xc[r] = fma(yj, c, xc[r]);
                xs[r] = fma(yj, s, xs[r]);
                if (WGT) {
                    const T wc = wj * c;
                    cc[r] = fma(wc, c, cc[r]);
                    cs[r] = fma(wc, s, cs[r]);
                } else {
                    cc[r] = fma(c, c, cc[r]);
                    cs[r] = fma(c, s, cs[r]);
                }
            }
        }
    }

    const T n_part = WGT ? w_sum : (T)(j1 - j0);   // sum of the weights of this item's observations
    Best mine;
    mine.p = -1.0;
    mine.k = INT64_MAX;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int64_t k = (int64_t)wi.tile * (TPB * R) + r * TPB + tid;
        if (k >= gp.n_freq) continue;
        const T c2 = T(2) * cc[r] - n_part, s2 = T(2) * cs[r];   // sum cos 2wt, sum sin 2wt
        if (sums) {      // split-N_t (or the generalised mode): partial sums, not powers
            sums[((int64_t)wi.split * n_obj_launch + wi.obj_local) * gp.n_freq + k] = make_vec4<T>(xc[r], xs[r], c2, s2);
        } else {
            const T scale = stats ? (T)stats[obj].scale : T(1);
            const T p = power_from_sums<T>(xc[r], xs[r], c2, s2, (T)n_t, scale);
            if (out_power) out_power[wi.obj_local * gp.n_freq + k] = p;
            Best b;
            b.p = (p == p) ? (double)p : -1.0;
            b.k = k;
            mine = best_of(mine, b);
        }
    }
    if (partials && !sums) {
        const Best b = block_best(mine, sbest);
        if (tid == 0) partials[wi.obj_local * gp.n_tiles + wi.tile] = b;
    }
}

// Split-N_t combine (n_split > 1): adds the partial sums of the splits in a FIXED order (so results do not
// depend on scheduling), then runs step 5 and, optionally, the argmax partial.  One thread per frequency,
// 1024 frequencies per CTA.
constexpr int kCombineThreads = 256;
constexpr int kCombinePerThread = 4;
template <typename T>
__global__ void __launch_bounds__(kCombineThreads)
lsp_combine_kernel(GridParams gp, const int64_t* __restrict__ offsets, const ObjStats* __restrict__ stats,
                   const typename Vec4<T>::type* __restrict__ sums, T* __restrict__ out_power,
                   Best* __restrict__ partials, int n_parts, int64_t n_obj_launch)
{
    __shared__ Best sbest[kCombineThreads / 32];
    const int64_t obj_local = blockIdx.x / n_parts;
    const int part = (int)(blockIdx.x % n_parts);
    const int64_t obj = obj_local + gp.obj_base;
    const T n_t = (T)(offsets[obj + 1] - offsets[obj]);
    const T scale = stats ? (T)stats[obj].scale : T(1);
    Best mine;
    mine.p = -1.0;
    mine.k = INT64_MAX;
#pragma unroll
    for (int r = 0; r < kCombinePerThread; ++r) {
        const int64_t k = ((int64_t)part * kCombinePerThread + r) * kCombineThreads + threadIdx.x;
        if (k >= gp.n_freq) continue;
        T xc = 0, xs = 0, c2 = 0, s2 = 0;
        for (int s = 0; s < gp.n_split; ++s) {
            const typename Vec4<T>::type v = sums[((int64_t)s * n_obj_launch + obj_local) * gp.n_freq + k];
            xc += v.x; xs += v.y; c2 += v.z; s2 += v.w;
        }
        const T p = power_from_sums<T>(xc, xs, c2, s2, n_t, scale);
        if (out_power) out_power[obj_local * gp.n_freq + k] = p;
        Best b;
        b.p = (p == p) ? (double)p : -1.0;
        b.k = k;
        mine = best_of(mine, b);
    }
    if (partials) {
        const Best b = block_best(mine, sbest);
        if (threadIdx.x == 0) partials[obj_local * n_parts + part] = b;
    }
}

// Step 6' finalize: one warp per object reduces the per-CTA partials and writes (period, power, index).
// period = 1/f_k* (PAPER.md:L87 in cyclic-frequency form, reading a1); N_t = 0 -> index -1, NaN period.
template <typename T>
__global__ void lsp_finalize_best_kernel(GridParams gp, const int64_t* __restrict__ offsets,
                                         const Best* __restrict__ partials, int n_parts, int64_t n_obj,
                                         T* __restrict__ best_period, T* __restrict__ best_power,
                                         int64_t* __restrict__ best_index)
{
    const int64_t obj_local = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (obj_local >= n_obj) return;
    const int64_t obj = obj_local + gp.obj_base;
    const int lane = threadIdx.x & 31;
    Best v;
    v.p = -2.0;
    v.k = INT64_MAX;
    for (int i = lane; i < n_parts; i += 32) v = best_of(v, partials[obj_local * n_parts + i]);
    v = warp_best(v);
    if (lane == 0) {
        const bool empty = (offsets[obj + 1] - offsets[obj]) <= 0 || v.p < 0.0 || v.k >= gp.n_freq;
        best_index[obj] = empty ? -1 : v.k;
        best_power[obj] = empty ? T(0) : (T)v.p;
        best_period[obj] = empty ? (T)NAN : (T)(1.0 / (gp.f_min + (double)v.k * gp.df));
    }
}

// Step 6' across frequency shards: merges, per object, the fused-argmax results of n_parts runs that each
// covered a contiguous slice of ONE global grid.  part_index holds GLOBAL grid indices (-1 = the slice had no valid frequency).
// Same rule as everywhere: largest power, lowest index on exact ties, NaN / -1 never win; period = 1/f_k on the global grid.
template <typename T>
__global__ void lsp_merge_best_kernel(GridParams gp, const T* __restrict__ part_power, const int64_t* __restrict__ part_index,
                                      int n_parts, int64_t n_obj, T* __restrict__ best_period, T* __restrict__ best_power,
                                      int64_t* __restrict__ best_index)
{
    const int64_t obj = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (obj >= n_obj) return;
    Best v;
    v.p = -2.0;
    v.k = INT64_MAX;
    for (int i = 0; i < n_parts; ++i) {
        const T pw = part_power[(int64_t)i * n_obj + obj];
        const int64_t k = part_index[(int64_t)i * n_obj + obj];
        if (k < 0 || k >= gp.n_freq || !(pw == pw)) continue;
        Best b;
        b.p = (double)pw;
        b.k = k;
        v = best_of(v, b);
    }
    const bool empty = v.k == INT64_MAX;
    best_index[obj] = empty ? -1 : v.k;
    best_power[obj] = empty ? T(0) : (T)v.p;
    best_period[obj] = empty ? (T)NAN : (T)(1.0 / (gp.f_min + (double)v.k * gp.df));
}

// Step 1 pre-pass (only when center=1 or normalize=1): per-object mean and 1/(0.5 sum (y-mean)^2).
template <typename T>
__global__ void lsp_object_stats_kernel(const int64_t* __restrict__ offsets, const T* __restrict__ y,
                                        ObjStats* __restrict__ stats, int center, int normalize)
{
    __shared__ double red[2][4];
    const int64_t obj = blockIdx.x;
    const int64_t lo = offsets[obj], n = offsets[obj + 1] - lo;
    double s = 0.0, q = 0.0;
    for (int64_t j = threadIdx.x; j < n; j += blockDim.x) {
        const double v = (double)y[lo + j];
        s += v;
        q += v * v;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        s += __shfl_xor_sync(0xffffffffu, s, d);
        q += __shfl_xor_sync(0xffffffffu, q, d);
    }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = s; red[1][threadIdx.x >> 5] = q; }
    __syncthreads();
    if (threadIdx.x == 0) {
        s = red[0][0] + red[0][1] + red[0][2] + red[0][3];
        q = red[1][0] + red[1][1] + red[1][2] + red[1][3];
        const double mean = (center && n > 0) ? s / (double)n : 0.0;
        const double ssq = q - 2.0 * mean * s + (double)n * mean * mean;   // sum (y - mean)^2
        ObjStats o;
        o.mean = mean;
        o.scale = normalize ? (ssq > 0.0 ? 2.0 / ssq : 0.0) : 1.0;
        stats[obj] = o;
    }
}

}  // namespace lsp
