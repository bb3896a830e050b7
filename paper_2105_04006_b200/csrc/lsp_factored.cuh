// lsp_factored.cuh -- the factored formulation shared by the FMA-pipe kernel (lsp_factored_ws.cuh) and the tensor-core
// kernel (lsp_tensor.cuh): NO sincos in the O(N_t N_f) loop, 4 FMA per (t, f) pair.  Mathematics, tile geometry, operand layout.
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
// The kernel itself (persistent, warp-specialised producers and consumers) is in lsp_factored_ws.cuh; lsp_tensor.cuh runs the
// same contraction on tcgen05 (FP32 mode).
//
// Work item = (object, frequency tile, observation split) as in the direct kernel; n_split > 1 writes the
// four sums per frequency for lsp_combine_kernel (split-N_t path for large-N_t / small-N_f problems).
#pragma once
#include "lsp_direct.cuh"

namespace lsp {

constexpr int kFacGroups = 64;                                   // G

template <typename T> struct FactoredCfg;
template <> struct FactoredCfg<float> {
    static constexpr int TH = 4;               // groups per thread
    static constexpr int TM = 4;               // m values per thread
    static constexpr int NL = 32;              // half-width of a group
    static constexpr int EPC = 2;              // complex elements per 16-byte chunk
    static constexpr int TILE = kFacGroups * 2 * NL;   // 4096 frequencies per CTA
    using V2 = float2;
};
template <> struct FactoredCfg<double> {
    // 4 x 4 register tile (64 DFMA per 8 LDS.128 and observation; 128 accumulator registers, see the setmaxnreg split in
    // lsp_factored_ws.cuh) and groups twice as wide as in round 1 (NL = 32): every non-DFMA instruction displaces a DFMA
    // on this pipe, and both the operand loads and the producers' work per pair halve.
    static constexpr int TH = 4;
    static constexpr int TM = 4;
    static constexpr int NL = 32;
    static constexpr int EPC = 1;
    static constexpr int TILE = kFacGroups * 2 * NL;   // 4096
    using V2 = double2;
};

template <typename T> constexpr int fac_tile() { return FactoredCfg<T>::TILE; }   // host-side helpers
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

}  // namespace lsp
