// lsp_common.cuh -- shared device helpers of the CUDA path: phase reduction, the per-(object, frequency)
// epilogue (hot-path step 5), and the (power, index) argmax reduction (step 6').
// Nothing here is shared with oracle/ (the CPU oracle is a separate C file with its own arithmetic).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>

namespace lsp {

constexpr double kTwoPi = 6.283185307179586476925286766559;

// Per-call constants every kernel needs; passed by value (fits the 4 KB parameter space easily).
struct GridParams {
    double f_min;       // cycles per unit of t
    double df;          // (f_max - f_min) / n_freq
    int    n_freq;      // N_f
    int    n_tiles;     // frequency tiles per object
    int    n_split;     // observation splits per (object, tile); 1 = epilogue fused in the main kernel
    int    obj_base;    // first object of this launch (host-output chunks)
};

// Per-object pre-pass results (step 1): mean to subtract (0 unless center=1) and the output scale
// (1, or 1/(0.5*sum y^2) when normalize=1).
struct ObjStats {
    double mean;
    double scale;
};

// A (power, index) candidate of the fused argmax.  Lowest index wins exact ties; NaN never wins
// (reading a7): NaN powers are mapped to -1 before they get here (P >= 0 otherwise).
struct Best {
    double  p;
    int64_t k;
};

__device__ __forceinline__ Best best_of(Best a, Best b)
{
    return (b.p > a.p || (b.p == a.p && b.k < a.k)) ? b : a;
}

__device__ __forceinline__ Best warp_best(Best v)
{
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        Best o;
        o.p = __shfl_xor_sync(0xffffffffu, v.p, s);
        o.k = __shfl_xor_sync(0xffffffffu, v.k, s);
        v = best_of(v, o);
    }
    return v;
}

// CTA-wide argmax; result valid in thread 0.  `scratch` holds >= blockDim.x/32 entries.
__device__ __forceinline__ Best block_best(Best v, Best* scratch)
{
    v = warp_best(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) scratch[wid] = v;
    __syncthreads();
    if (wid == 0) {
        Best w;
        w.p = -2.0;
        w.k = INT64_MAX;
        if (lane < nw) w = scratch[lane];
        v = warp_best(w);
    }
    return v;
}

// ---------------------------------------------------------------------------------------------------
// Step 5: power from the four un-rotated sums of one (object, frequency):
//   xc = sum y cos(wt), xs = sum y sin(wt), c2 = sum cos(2wt), s2 = sum sin(2wt), n = N_t.
// Eq. 1's tau diagonalises M = [[CC, CS], [CS, SS]] with CC = (n + c2)/2, SS = (n - c2)/2, CS = s2/2, and
// Eq. 2 is 1/2 b^T M^-1 b with b = (xc, xs) (the paper's own single-scan epilogue,
// Listing 1, evaluates the same quantity through atan2 + a second sincos).  Written out:
//   P = [ n (xc^2 + xs^2) - c2 (xc^2 - xs^2) - 2 s2 xc xs ] / (n^2 - c2^2 - s2^2)
// One division, no atan2/sincos.  When the smaller eigenvalue (n - |w|)/2 of M vanishes (all 2wt_j equal
// mod 2pi: N_t = 1, exact aliasing) its term is dropped, as the oracle does (reading a6):
//   P -> (xc^2 + xs^2) / (n + |w|).
// Every product and sum below is an explicit round-to-nearest intrinsic, so the compiler cannot contract them
// differently in different kernels or code paths: the same sums give the same bits everywhere.
__device__ __forceinline__ float  mul_rn(float a, float b)   { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float  add_rn(float a, float b)   { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float  div_rn(float a, float b)   { return __fdividef(a, b); }   // MUFU.RCP + FMUL, <= 2 ulp: the
                                                                                          // FP32 tolerance is 1e-3 max P
__device__ __forceinline__ double div_rn(double a, double b) { return __ddiv_rn(a, b); }

template <typename T>
__device__ __forceinline__ T power_from_sums(T xc, T xs, T c2, T s2, T n, T scale)
{
    const T eps = sizeof(T) == 4 ? T(2e-6) : T(4e-12);
    const T a = mul_rn(xc, xc), b = mul_rn(xs, xs);
    const T w2 = fma(c2, c2, mul_rn(s2, s2));
    const T nn = mul_rn(n, n);
    const T den = add_rn(nn, -w2);
    T p;
    if (den > mul_rn(eps, nn)) {
        // n (a + b) - c2 (a - b) - 2 s2 xc xs
        const T num = fma(-mul_rn(T(2), s2), mul_rn(xc, xs), fma(-c2, add_rn(a, -b), mul_rn(n, add_rn(a, b))));
        p = div_rn(num, den);
    } else if (n > T(0)) {
        p = div_rn(add_rn(a, b), add_rn(n, sqrt(w2)));
    } else {
        p = T(0);
    }
    return mul_rn(p, scale);
}

// frac(x) to (-1/2, 1/2] by the round-to-nearest magic constant (x >= 0 and < 2^51 here): two DADDs on the
// FP64 pipe instead of FRND.F64.
__device__ __forceinline__ double frac_cycles(double p)
{
    const double magic = 6755399441055744.0;   // 1.5 * 2^52
    const double r = (p + magic) - magic;
    return p - r;
}

// Exact-product phase: f*t = p + e exactly (fma), reduced to cycles in (-1/2, 1/2].
__device__ __forceinline__ double phase_cycles_exact(double f, double t)
{
    const double p = f * t;
    const double e = fma(f, t, -p);
    return frac_cycles(p) + e;
}

// sin/cos of 2*pi*r for r in about [-1, 1] cycles.
//   FAST (FP32): MUFU.SIN / MUFU.COS through __sinf/__cosf (the paper's "__sincosf").
//   accurate FP32: CUDA's sincospif (polynomial on the FMA pipe, <= 2 ulp).
template <bool FAST>
__device__ __forceinline__ void sincos_cycles(float r, float* s, float* c)
{
    if (FAST) {
        const float a = r * 6.283185307179586f;
        *s = __sinf(a);
        *c = __cosf(a);
    } else {
        sincospif(2.0f * r, s, c);
    }
}
template <bool FAST>
__device__ __forceinline__ void sincos_cycles(double r, double* s, double* c)
{
    sincospi(2.0 * r, s, c);   // FAST has no FP64 meaning (rejected at plan creation)
}

// sin/cos of 2*pi*r in FP64 for an ALREADY REDUCED r in about [-1/2 - 2^-20, 1/2 + 2^-20] cycles: 21 FP64-pipe instructions
// and a handful of integer ones, against ~36 + ~75 for the library sincospi (which redoes the range reduction, handles
// Inf/NaN and moves 64-bit halves around).  k = round(4 r) picks the octant pair, s = r - k/4 is exact (fma), and
// sin 2 pi s, cos 2 pi s are Taylor series in z = s^2 on |2 pi s| <= pi/4 + 2^-17: truncation error <= (pi/4)^17/17! = 5e-17
// (sin) and (pi/4)^18/18! = 2e-18 (cos), i.e. below one ulp of 1.  The quadrant is applied with selects and a sign flip.
__device__ __forceinline__ void sincos_cycles_reduced(double r, double* sn, double* cs)
{
    const double magic = 6755399441055744.0;              // 1.5 * 2^52: the low word of (x + magic) is round(x)
    const double tq = fma(r, 4.0, magic);
    const int k = __double2loint(tq);
    const double kf = tq - magic;
    const double s = fma(kf, -0.25, r);
    const double z = s * s;
    double ps = -0.71812230177850051223;
    ps = fma(ps, z, 3.8199525848482821277);
    ps = fma(ps, z, -15.094642576822990392);
    ps = fma(ps, z, 42.058693944897653145);
    ps = fma(ps, z, -76.705859753061385842);
    ps = fma(ps, z, 81.605249276075054203);
    ps = fma(ps, z, -41.341702240399760234);
    ps = fma(ps, z, 6.2831853071795864769);
    const double S = ps * s;
    double pc = 0.28200596845579121507;
    pc = fma(pc, z, -1.7143907110886720654);
    pc = fma(pc, z, 7.9035363713184688042);
    pc = fma(pc, z, -26.426256783374397453);
    pc = fma(pc, z, 60.244641371876660363);
    pc = fma(pc, z, -85.456817206693727736);
    pc = fma(pc, z, 64.939394022668291491);
    pc = fma(pc, z, -19.739208802178717238);
    const double C = fma(pc, z, 1.0);
    // k mod 4 = 0: (S, C); 1: (C, -S); 2: (-S, -C); 3: (-C, S)
    const bool swap = (k & 1) != 0;
    const double a = swap ? C : S, b = swap ? S : C;
    const int sa = (int)(((unsigned)k & 2u) << 30);        // sign bit of sin: quadrants 2, 3
    const int sb = (int)(((unsigned)(k + 1) & 2u) << 30);  // sign bit of cos: quadrants 1, 2
    *sn = __hiloint2double(__double2hiint(a) ^ sa, __double2loint(a));
    *cs = __hiloint2double(__double2hiint(b) ^ sb, __double2loint(b));
}

// FP32 version for a reduced r in about [-1/2, 1/2] cycles: k = round(4 r) by the magic-constant add, s = r - k/4 exact, Taylor
// series on |2 pi s| <= pi/4 (truncation 1.8e-9 for sin, 2.5e-8 for cos: below half an ulp of 1), quadrant by selects and
// sign flips: ~22 FMA/ALU-pipe instructions and no XU instruction (sincospif: ~40 with FRND / F2I).
__device__ __forceinline__ void sincos_cycles_reduced(float r, float* sn, float* cs)
{
    const float magic = 12582912.0f;                       // 1.5 * 2^23: the low mantissa bits of (x + magic) are round(x)
    const float tq = fmaf(r, 4.0f, magic);
    const unsigned k = __float_as_uint(tq);                // 0x4B400000 + round(4 r): the two low bits are the quadrant
    const float kf = tq - magic;
    const float s = fmaf(kf, -0.25f, r);
    const float z = s * s;
    float ps = 42.058693944897653f;
    ps = fmaf(ps, z, -76.705859753061386f);
    ps = fmaf(ps, z, 81.605249276075054f);
    ps = fmaf(ps, z, -41.341702240399760f);
    ps = fmaf(ps, z, 6.2831853071795865f);
    const float S = ps * s;
    float pc = 60.244641371876660f;
    pc = fmaf(pc, z, -85.456817206693728f);
    pc = fmaf(pc, z, 64.939394022668291f);
    pc = fmaf(pc, z, -19.739208802178717f);
    const float C = fmaf(pc, z, 1.0f);
    const bool swap = (k & 1u) != 0;
    const float a = swap ? C : S, b = swap ? S : C;
    *sn = __uint_as_float(__float_as_uint(a) ^ ((k & 2u) << 30));
    *cs = __uint_as_float(__float_as_uint(b) ^ (((k + 1u) & 2u) << 30));
}

// A frequency prepared for phase evaluation against observation times of type T, and the phasor e^{2 pi i f t}.
//   float : f = hi + lo (two floats); f t = p + e exactly (fma), p reduced by rintf, low terms added after the reduction:
//           about 2^-48 relative to f t, no FP64 instruction.
//   double: exact-product phase (phase_cycles_exact) and the reduced-argument sincos above.
template <typename T> struct PhaseFreq;
template <> struct PhaseFreq<float> {
    float hi, lo;
    __device__ __forceinline__ void set(double f) { hi = (float)f; lo = (float)(f - (double)hi); }
    __device__ __forceinline__ float cycles(float t) const
    {
        const float p = hi * t;
        const float e = fmaf(hi, t, -p);
        return (p - rintf(p)) + fmaf(lo, t, e);
    }
    template <bool FAST> __device__ __forceinline__ void phasor(float t, float* s, float* c) const
    {
        sincos_cycles<FAST>(cycles(t), s, c);
    }
};
template <> struct PhaseFreq<double> {
    double f;
    __device__ __forceinline__ void set(double f_) { f = f_; }
    __device__ __forceinline__ double cycles(double t) const { return phase_cycles_exact(f, t); }
    template <bool FAST> __device__ __forceinline__ void phasor(double t, double* s, double* c) const
    {
        sincos_cycles_reduced(cycles(t), s, c);
    }
};

}  // namespace lsp
