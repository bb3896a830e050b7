// lsp_factored.cuh -- the flagship periodogram kernel: NO sincos in the O(N_t N_f) loop, 4 FMA per (t, f) pair.
//
// Idea (angle addition, BASELINE.json north_star "tau-dependent sums obtained by angle-addition identities").
// The four sums every frequency needs (PAPER.md:L172-185 accumulates the same information as xc, xs, cc, ss, cs):
//     Z(k) = sum_j y_j e^{i theta_kj}   = xc + i xs         theta_kj = 2 pi f_k t_j
//     W(k) = sum_j     e^{2 i theta_kj} = (cc - ss) + 2 i cs
// A frequency tile is cut into G groups of L = 2*NL consecutive grid points.  Group g is addressed from its
// (half-integer) centre c_g = K0 + g L + NL - 1/2 as k = c_g +/- (m + 1/2), m = 0..NL-1.  Since the grid is
// linear in frequency,
//     theta_kj = alpha_gj +/- beta_mj,   alpha_gj = 2 pi f(c_g) t_j,   beta_mj = 2 pi (m + 1/2) df t_j
// and with a = y_j e^{i alpha} (per group, observation), b = e^{i beta} (per m, observation; the SAME for
// every group, tile and object sharing t_j):
//     Z(c_g + m + 1/2) = sum_j a b       = (Srr - Sii) + i (Sri + Sir)
//     Z(c_g - m - 1/2) = sum_j a conj(b) = (Srr + Sii) + i (Sir - Sri)
// where Srr = sum ar br, Sri = sum ar bi, Sir = sum ai br, Sii = sum ai bi.  Four real FMAs per observation
// produce BOTH frequencies' complex sum, i.e. 2 FMA per pair per complex sum; W(k) is the same contraction with
// the doubled angles.  Total: 4 FMA per (t, f) pair -- one per real output sum, the floor for an FMA
// formulation -- against 1 sincos + 5 FMA in Listing 1.  The sincos work drops to (G + NL) evaluations per
// observation per tile (G*L frequencies), done once per observation chunk by the whole CTA into shared memory.
//
// B200 mapping.  The contraction is a small real GEMM per (object, tile) held in registers.  Warps 0-3 of the
// CTA contract Z, warps 4-7 contract W (same instruction stream, different operand arrays); each thread owns
// TH groups x TM values of m = 64 accumulator registers.  FP32 uses the packed FFMA2 (fma.rn.f32x2, sm_100+)
// with the broadcast-scalar operand form: (Srr, Sri) += ar * (br, bi) is ONE instruction, so the inner loop is
// 32 FFMA2 + 4 LDS.128 per observation per thread: issue slots are not the limit, the FMA pipe is.  FP64 uses
// DFMA (32 DFMA + 6 LDS.128).  Shared-memory operand reads are the second resource: on B200 a warp-wide
// LDS.128 costs 2 data-pipe cycles only if every aligned group of 4 lanes touches at most 2 distinct
// addresses, else 4 (measured; profiles/).  The lane -> (group, m) map below is built for that rule: lane bit 0
// selects the group index, lane bit 1 the m index, and operands are stored so that a warp's distinct 16-byte
// chunks are contiguous (no bank conflicts).
// Operands a, b are generated into a double-buffered shared-memory chunk (JC observations) by all threads
// (phase in FP64 -> range-reduced -> MUFU or accurate sincos) while the previous chunk is being contracted.
// This file is the FMA-pipe / FP64-pipe form of the contraction; lsp_tensor.cuh runs the same contraction on tcgen05 (FP32 mode).
//
// Work item = (object, frequency tile, observation split) as in the direct kernel; n_split > 1 writes the
// four sums per frequency for lsp_combine_kernel (split-N_t path for large-N_t / small-N_f problems).
#pragma once
#include "lsp_direct.cuh"

namespace lsp {

constexpr int kFacThreads = 256;
constexpr int kFacGroups = 64;                                   // G

template <typename T> struct FactoredCfg;
template <> struct FactoredCfg<float> {
    static constexpr int TH = 4;               // groups per thread
    static constexpr int TM = 4;               // m values per thread
    static constexpr int NL = 32;              // half-width of a group
    static constexpr int JC = 16;              // observations per smem chunk
    static constexpr int EPC = 2;              // complex elements per 16-byte chunk
    static constexpr int TILE = kFacGroups * 2 * NL;   // 4096 frequencies per CTA
    using V2 = float2;
};
template <> struct FactoredCfg<double> {
    static constexpr int TH = 2;
    static constexpr int TM = 4;
    static constexpr int NL = 16;
    static constexpr int JC = 8;
    static constexpr int EPC = 1;
    static constexpr int TILE = kFacGroups * 2 * NL;   // 2048
    using V2 = double2;
};

template <typename T> constexpr int fac_tile() { return FactoredCfg<T>::TILE; }   // host-side helpers
template <typename T> constexpr size_t fac_smem_bytes()
{
    // operand buffers: per observation G + G + NL + NL complex values, two buffers;
    // epilogue: TILE (c2, s2) pairs + TILE powers.  The larger of the two.
    const size_t ops = 2 * (size_t)FactoredCfg<T>::JC * (2 * kFacGroups + 2 * FactoredCfg<T>::NL) * 2 * sizeof(T);
    const size_t epi = (size_t)FactoredCfg<T>::TILE * 3 * sizeof(T);
    return ops > epi ? ops : epi;
}

// Storage position (in complex elements) of logical index x = xi*PER + a inside one observation's operand row,
// when a thread owns PER consecutive indices and NI thread-indices exist: the 16-byte chunks that one LDS.128 of
// a warp touches are contiguous.
template <int PER, int NI, int EPC>
__device__ __forceinline__ int operand_pos(int x)
{
    const int xi = x / PER, a = x % PER;
    return ((a / EPC) * NI + xi) * EPC + (a % EPC);
}

// acc_r += ar * b, acc_i += ai * b  (b = (br, bi))
__device__ __forceinline__ void cmac(float2& acc_r, float2& acc_i, float ar, float ai, float2 b)
{
    acc_r = __ffma2_rn(make_float2(ar, ar), b, acc_r);   // FFMA2 Rd, Ra.F32 (broadcast), Rb.F32x2, Rd
    acc_i = __ffma2_rn(make_float2(ai, ai), b, acc_i);
}
__device__ __forceinline__ void cmac(double2& acc_r, double2& acc_i, double ar, double ai, double2 b)
{
#ifdef LSP_DFMA_ASM
    asm("fma.rn.f64 %0, %1, %2, %0;" : "+d"(acc_r.x) : "d"(ar), "d"(b.x));
    asm("fma.rn.f64 %0, %1, %2, %0;" : "+d"(acc_r.y) : "d"(ar), "d"(b.y));
    asm("fma.rn.f64 %0, %1, %2, %0;" : "+d"(acc_i.x) : "d"(ai), "d"(b.x));
    asm("fma.rn.f64 %0, %1, %2, %0;" : "+d"(acc_i.y) : "d"(ai), "d"(b.y));
    return;
#endif
    acc_r.x = fma(ar, b.x, acc_r.x);
    acc_r.y = fma(ar, b.y, acc_r.y);
    acc_i.x = fma(ai, b.x, acc_i.x);
    acc_i.y = fma(ai, b.y, acc_i.y);
}

template <typename T> __device__ __forceinline__ T phase_for(double f, T t);
template <> __device__ __forceinline__ float phase_for<float>(double f, float t)
{
    return (float)frac_cycles(f * (double)t);      // FP64 product: 2e-11 cycles at f t = 1.8e5, far below FP32 needs
}
template <> __device__ __forceinline__ double phase_for<double>(double f, double t)
{
    return phase_cycles_exact(f, t);
}

template <typename T, bool FAST>
__global__ void __launch_bounds__(kFacThreads, 2)
lsp_factored_kernel(GridParams gp, const int64_t* __restrict__ offsets, const T* __restrict__ t,
                    const T* __restrict__ y, const ObjStats* __restrict__ stats,
                    T* __restrict__ out_power, Best* __restrict__ partials,
                    typename Vec4<T>::type* __restrict__ sums, int64_t n_obj_launch)
{
    using C = FactoredCfg<T>;
    using V2 = typename C::V2;
    constexpr int G = kFacGroups, TH = C::TH, TM = C::TM, NL = C::NL, L = 2 * NL, TILE = C::TILE, JC = C::JC, EPC = C::EPC;
    constexpr int TPB = kFacThreads;
    constexpr int NGI = G / TH, NMI = NL / TM;            // thread-index extents: 16 x 8 (FP32), 32 x 4 (FP64)
    static_assert(NGI * NMI == TPB / 2, "Z and W halves of the CTA each cover the G x NL tile once");
    static_assert(NMI == 8 || NMI == 4, "lane map below");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    // operand layout: [2 buffers][JC][G] a, [2][JC][G] a2, [2][JC][NL] b, [2][JC][NL] b2   (complex V2 each)
    V2* sA1 = reinterpret_cast<V2*>(smem_raw);
    V2* sA2 = sA1 + 2 * JC * G;
    V2* sB1 = sA2 + 2 * JC * G;
    V2* sB2 = sB1 + 2 * JC * NL;
    __shared__ Best sbest[TPB / 32];

    const WorkItem wi = decode_item(gp);
    const int64_t obj = wi.obj_local + gp.obj_base;
    const int64_t lo = offsets[obj];
    const int64_t n_t = offsets[obj + 1] - lo;
    const int64_t j0 = (n_t * wi.split) / gp.n_split;
    const int64_t j1 = (n_t * (wi.split + 1)) / gp.n_split;
    const T mean = stats ? (T)stats[obj].mean : T(0);
    const int tid = threadIdx.x;
    const int64_t K0 = (int64_t)wi.tile * TILE;

    // ---- contraction coordinates: lane bit 0 -> group index, lane bit 1 -> m index (the LDS rule above) -------
    const int lane = tid & 31, wq = (tid >> 5) & 3;
    const bool is_w = tid >= TPB / 2;                     // warps 4-7 contract W (doubled angles)
    int gi, mi;
    if (NMI == 8) {      // FP32: mi = (b1, b3, b4), gi = (b0, b2, warp)
        mi = ((lane >> 1) & 1) | (((lane >> 3) & 3) << 1);
        gi = (lane & 1) | (((lane >> 2) & 1) << 1) | (wq << 2);
    } else {             // FP64: mi = (b1, b3), gi = (b0, b2, b4, warp)
        mi = ((lane >> 1) & 1) | (((lane >> 3) & 1) << 1);
        gi = (lane & 1) | (((lane >> 2) & 1) << 1) | (((lane >> 4) & 1) << 2) | (wq << 3);
    }
    const V2* opA = is_w ? sA2 : sA1;
    const V2* opB = is_w ? sB2 : sB1;

    // ---- generator coordinates of this thread (fixed for the whole kernel) -----------------------------------
    const int gen_g = tid & (G - 1);
    const int gen_m = tid & (NL - 1);
    const int gen_pos_a = operand_pos<TH, NGI, EPC>(gen_g);
    const int gen_pos_b = operand_pos<TM, NMI, EPC>(gen_m);
    const double f_centre = gp.f_min + ((double)(K0 + (int64_t)gen_g * L + NL) - 0.5) * gp.df;   // f(c_g)
    const double f_beta = ((double)gen_m + 0.5) * gp.df;                                         // (m + 1/2) df

    V2 acc_r[TH][TM], acc_i[TH][TM];        // (Srr, Sri) and (Sir, Sii) of this thread's (group, m) pairs
#pragma unroll
    for (int a = 0; a < TH; ++a)
#pragma unroll
        for (int c = 0; c < TM; ++c) {
            acc_r[a][c].x = acc_r[a][c].y = T(0);
            acc_i[a][c].x = acc_i[a][c].y = T(0);
        }

    // ---- operand generation for the chunk starting at jb into buffer `buf` (steps 2-3) -------------------
    auto generate = [&](int64_t jb, int buf) {
#pragma unroll
        for (int it = 0; it < (G * JC) / TPB; ++it) {
            const int jj = (tid + it * TPB) / G;             // gen_g = tid % G is the same for every `it`
            const int64_t j = jb + jj;
            V2 a1, a2;
            a1.x = a1.y = a2.x = a2.y = T(0);
            if (j < j1) {
                const T tj = t[lo + j];
                const T yj = y[lo + j] - mean;
                T s, c;
                sincos_cycles<FAST>(phase_for<T>(f_centre, tj), &s, &c);
                a1.x = yj * c;                 // a  = y e^{i alpha}
                a1.y = yj * s;
                a2.x = fma(c, c, -s * s);      // a2 = e^{2 i alpha}
                a2.y = T(2) * c * s;
            }
            sA1[(buf * JC + jj) * G + gen_pos_a] = a1;
            sA2[(buf * JC + jj) * G + gen_pos_a] = a2;
        }
#pragma unroll
        for (int it = 0; it < (NL * JC + TPB - 1) / TPB; ++it) {
            const int e = tid + it * TPB;
            if ((NL * JC) % TPB != 0 && e >= NL * JC) break;
            const int jj = e / NL;                           // gen_m = tid % NL likewise
            const int64_t j = jb + jj;
            const T tj = (j < j1) ? t[lo + j] : T(0);
            T s, c;
            sincos_cycles<FAST>(phase_for<T>(f_beta, tj), &s, &c);
            V2 b1, b2;
            b1.x = c;                          // b  = e^{i beta}
            b1.y = s;
            b2.x = fma(c, c, -s * s);          // b2 = e^{2 i beta}
            b2.y = T(2) * c * s;
            sB1[(buf * JC + jj) * NL + gen_pos_b] = b1;
            sB2[(buf * JC + jj) * NL + gen_pos_b] = b2;
        }
    };

    // ---- the contraction over one chunk (step 4): 32 FFMA2 + 4 LDS.128 (32 DFMA + 6 LDS.128) per observation ----
    auto contract = [&](int buf) {
        const V2* A = opA + buf * JC * G;
        const V2* B = opB + buf * JC * NL;
#pragma unroll 4
        for (int jj = 0; jj < JC; ++jj) {       // 4: more spills the 64 accumulators at the 128-register cap
            V2 av[TH], bv[TM];
            if constexpr (EPC == 2) {           // one LDS.128 = two complex operands
#pragma unroll
                for (int q = 0; q < TH / 2; ++q) {
                    const float4 ch = reinterpret_cast<const float4*>(A + jj * G)[q * NGI + gi];
                    av[2 * q].x = ch.x; av[2 * q].y = ch.y; av[2 * q + 1].x = ch.z; av[2 * q + 1].y = ch.w;
                }
#pragma unroll
                for (int q = 0; q < TM / 2; ++q) {
                    const float4 ch = reinterpret_cast<const float4*>(B + jj * NL)[q * NMI + mi];
                    bv[2 * q].x = ch.x; bv[2 * q].y = ch.y; bv[2 * q + 1].x = ch.z; bv[2 * q + 1].y = ch.w;
                }
            } else {                            // one LDS.128 = one complex operand
#pragma unroll
                for (int a = 0; a < TH; ++a) av[a] = A[jj * G + a * NGI + gi];
#pragma unroll
                for (int c = 0; c < TM; ++c) bv[c] = B[jj * NL + c * NMI + mi];
            }
#pragma unroll
            for (int a = 0; a < TH; ++a)
#pragma unroll
                for (int c = 0; c < TM; ++c) cmac(acc_r[a][c], acc_i[a][c], av[a].x, av[a].y, bv[c]);
        }
    };

    if (j0 < j1) {
        generate(j0, 0);
        __syncthreads();
        int buf = 0;
        for (int64_t jb = j0; jb < j1; jb += JC) {
            if (jb + JC < j1) generate(jb + JC, buf ^ 1);
            contract(buf);
            __syncthreads();
            buf ^= 1;
        }
    }

    // ---- epilogue (step 5) + outputs (steps 6 / 6') ----------------------------------------------------------
    // W warps publish (c2, s2) per frequency through shared memory; Z warps combine them with (xc, xs).
    V2* sW = reinterpret_cast<V2*>(smem_raw);                               // [TILE] (c2, s2)
    T* sP = reinterpret_cast<T*>(smem_raw + (size_t)TILE * 2 * sizeof(T));   // [TILE] powers, for coalesced stores
    if (is_w) {
#pragma unroll
        for (int a = 0; a < TH; ++a)
#pragma unroll
            for (int c = 0; c < TM; ++c) {
                const int kg = (gi * TH + a) * L, m = mi * TM + c;
                V2 up, dn;
                up.x = acc_r[a][c].x - acc_i[a][c].y;    // Srr - Sii
                up.y = acc_r[a][c].y + acc_i[a][c].x;    // Sri + Sir
                dn.x = acc_r[a][c].x + acc_i[a][c].y;    // Srr + Sii
                dn.y = acc_i[a][c].x - acc_r[a][c].y;    // Sir - Sri
                sW[kg + NL + m] = up;
                sW[kg + NL - 1 - m] = dn;
            }
    }
    __syncthreads();
    Best mine;
    mine.p = -1.0;
    mine.k = INT64_MAX;
    const bool stage = !sums && (out_power != nullptr);
    if (!is_w) {
        const T scale = stats ? (T)stats[obj].scale : T(1);
#pragma unroll
        for (int a = 0; a < TH; ++a)
#pragma unroll
            for (int c = 0; c < TM; ++c) {
                const int kg = (gi * TH + a) * L, m = mi * TM + c;
#pragma unroll
                for (int up = 0; up < 2; ++up) {
                    const int kl = up ? (kg + NL + m) : (kg + NL - 1 - m);
                    const int64_t k = K0 + kl;
                    const V2 w = sW[kl];
                    T xc, xs;
                    if (up) {
                        xc = acc_r[a][c].x - acc_i[a][c].y;
                        xs = acc_r[a][c].y + acc_i[a][c].x;
                    } else {
                        xc = acc_r[a][c].x + acc_i[a][c].y;
                        xs = acc_i[a][c].x - acc_r[a][c].y;
                    }
                    if (sums) {
                        if (k < gp.n_freq)
                            sums[((int64_t)wi.split * n_obj_launch + wi.obj_local) * gp.n_freq + k] = make_vec4<T>(xc, xs, w.x, w.y);
                    } else {
                        const T p = power_from_sums<T>(xc, xs, w.x, w.y, (T)n_t, scale);
                        if (stage) sP[kl] = p;
                        if (k < gp.n_freq) {
                            Best b;
                            b.p = (p == p) ? (double)p : -1.0;
                            b.k = k;
                            mine = best_of(mine, b);
                        }
                    }
                }
            }
    }
    if (stage) {
        __syncthreads();
        T* dst = out_power + wi.obj_local * gp.n_freq + K0;
        const int n_valid = (int)min((int64_t)TILE, (int64_t)gp.n_freq - K0);
        for (int i = tid; i < n_valid; i += TPB) dst[i] = sP[i];
    }
    if (partials && !sums) {
        const Best b = block_best(mine, sbest);
        if (tid == 0) partials[wi.obj_local * gp.n_tiles + wi.tile] = b;
    }
}

}  // namespace lsp
