// lsp_tensor.cuh -- the FP32-mode periodogram contraction on the 5th-generation tensor cores (tcgen05 + TMEM).
//
// The factored formulation (lsp_factored.cuh: theta_kj = alpha_gj +/- beta_mj, a = y e^{i alpha}, b = e^{i beta})
// makes step 4 of the hot path a dense real contraction over the observations j of one object:
//
//     D_Z[128 x 2NL] = A_Z[128 x N_t] * B_Z[N_t x 2NL]        A_Z rows: Re a_g / Im a_g of 64 frequency groups
//     D_W[128 x 2NL] = A_W[128 x N_t] * B_W[N_t x 2NL]        B_Z cols: Re b_m (m < NL) | Im b_m;  W: doubled angles
//
// D holds, per (group g, offset m), Srr, Sri (row "Re a_g") and Sir, Sii (row "Im a_g"), from which
//     Z(c_g + m + 1/2) = (Srr - Sii) + i (Sri + Sir),   Z(c_g - m - 1/2) = (Srr + Sii) + i (Sir - Sri)
// and the same for W: one 128 x 2NL tile pair covers 64 * 2NL <= 14336 grid frequencies of one object, and the four
// real sums of Eq. 2's closed form (lsp_common.cuh) for every one of them.  This is a GEMM, so it runs as one:
// tcgen05.mma kind::f16, M = 128, N = 2NL <= 224, K = 16, FP32 accumulators in TMEM.
//
// Where the operands live (round 2: the shared-memory pipe was the ceiling of the SS-mode kernel -- 12 KB of operand reads
// per 128-cycle MMA plus the generators' operand stores plus the TMA fills):
//   A operands (tile dependent, generated on the fly) are written by the generator warps STRAIGHT INTO TENSOR MEMORY
//               (tcgen05.st) and the MMAs read them from there (A-from-TMEM form of tcgen05.mma): no shared-memory store,
//               no shared-memory read, no proxy fence.  TMEM columns (MNL = the instantiation's largest NL, 112 or 104): Z
//               accumulators [0, 2NL), W accumulators [2 MNL, 2 MNL + 2NL), A ring [4 MNL, 512) in stages of 2 planes x 8
//               columns (4 planes with three products).
//   B operands  e^{i beta}, e^{2 i beta} depend on (object, observation, m) only -- not on the tile -- so one pre-pass launch
//               (lsp_tensor_prepass_kernel) writes them once per object into a table already laid out as shared-memory
//               stages; warp 0 streams the stages in with 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx).
//               Each table stage also carries an "aux" block (t_j, y_j, w_j and the tile-independent phasors v of its 16
//               observations), so the generators never touch global memory.
//
// Precision: the tabulated operand b is an FP16 pair b_hi + b_lo (22 significand bits, the same class
// as FP32's 24); the generated operand a is one FP16 (two products a_hi b_hi + a_hi b_lo per multiply-accumulate: the default)
// or a pair as well (three products, + a_lo b_hi; a_lo b_lo < 2^-22 is dropped), with y pre-scaled by a power of two per object
// so FP16 never overflows or loses the low part.  fast_math = 1 keeps only a_hi b_hi (one MMA, ~2^-11 per operand) and
// evaluates sincos with MUFU: the "fast vs accurate" comparison of PAPER.md:L423-433 carried over to this formulation.
// Phases are range-reduced before any FP32 trigonometry.
//
// Roles of one CTA (persistent, one per SM, static round-robin over (object, tile, split) work items):
//   warp 0      TMA producer of the B ring          warp 1   MMA issuer (one elected lane)        warp 2   TMEM allocator
//   warps 4..   epilogue: tcgen05.ld the accumulators, pair rows with a shuffle, closed-form power (step 5), vector
//               stores of the periodogram (step 6) or the fused argmax partial (step 6'); for split-N_t items the
//               partial sums go to global memory in the epilogue's own order (coalesced) and lsp_tensor_fix_kernel adds
//               them in split order and finishes the tiles
//   then NG generator groups of 4 warps, each taking every NG-th stage: one sincos per thread (the tile's phasors u),
//               then row r = (group g, Re/Im) of the stage's A operand for its 16 observations in registers -> TMEM.
#pragma once
#include <cuda_fp16.h>

#include <type_traits>

#include "lsp_factored_ws.cuh"

namespace lsp {

constexpr int kTcGroups = 64;                  // frequency groups per tile (128 MMA rows)
constexpr int kTcKB = 16;                      // observations per MMA / ring stage (kind::f16: K = 16)
#ifndef LSP_TC_MAX_NL
#define LSP_TC_MAX_NL 112
#endif
constexpr int kTcMaxNL = LSP_TC_MAX_NL;        // N = 2 NL <= 224: leaves 64 TMEM columns for the A ring
#ifndef LSP_TC_PAIR_MAX_NL
#define LSP_TC_PAIR_MAX_NL 112
#endif
constexpr int kTcPairMaxNL = LSP_TC_PAIR_MAX_NL;   // largest NL of the pair-mode kernel (104 would leave 96 columns = a 6-stage A ring)
constexpr int kTcPreThreads = 128;             // threads of a pre-pass block
constexpr int kTcMaxSB = 12;                   // deepest B ring (barrier arrays are sized for it)
#ifndef LSP_TC_PAIR_NG
#define LSP_TC_PAIR_NG 4
#endif
constexpr int kTcPairNG = LSP_TC_PAIR_NG;      // generator groups of the pair-mode kernel
// aux block of a table stage (floats): t[16], y[16], w[16], then 16 phasor rows of 16 complex values (+ 4 floats of padding
// per row: 144-byte rows keep the LDS.128 of lanes that read different rows conflict-free).  Rows 0-7: v_g1 = e^{2 pi i (8 g1 L df) t_j};
// rows 8-15: v_g1 e^{-i pi/4}, the version the "Im a" rows use (see the generators).  Inside a row the 16 phasors are stored
// per observation PAIR as (cos_2h, cos_2h+1, sin_2h, sin_2h+1): one LDS.128 yields two register-aligned float2 operands
// of the packed FP32x2 instructions.
constexpr int kTcVRow = 36;
constexpr int kTcAuxFloats = 48 + 16 * kTcVRow;
constexpr int kTcAuxBytes = kTcAuxFloats * 4;  // 2496
constexpr float kTcUnitScale = 256.0f;         // scale of the unit-modulus A_W operands (keeps the FP16 low part normal)
constexpr float kTcPhasorScale = 16.0f;        // sqrt of it: carried by the phasors u

// Warp roles of one CTA: 4 control warps, EW epilogue warps, NG generator groups of 4 warps.  Two shapes are built:
//   (EW, NG) = (8, 3): short items (batches of short light curves): the per-item epilogue is on the critical path
//   (EW, NG) = (4, 4): long items (hundreds of stages): the generators are, the epilogue is rare
// Both have 768 threads (80 registers at launch).  Registers are re-split with setmaxnreg: short-item shape control 40,
// generators 72, epilogue 112; long-item shape (single CTAs and CTA pairs) control 32, generators 88, epilogue 96.
template <int EW, int NG> struct TcRoles {
    static constexpr int kThreads = (4 + EW + 4 * NG) * 32;
    static constexpr int kEpiThreads = EW * 32;
    static constexpr int kGenGroupThreads = 128;
    static constexpr int kLaunchRegs = (65536 / kThreads) / 8 * 8;
    // long-item shape: the generators are the critical role (they keep a stage's tile-independent phasors in registers while
    // the tile's own are still being evaluated); its epilogue runs once per few hundred stages
    static constexpr int kCtrlRegs = NG >= 4 ? 32 : 40, kGenRegs = NG == 4 ? 88 : 72;
    static constexpr int kEpiRegs = ((kLaunchRegs * kThreads - 128 * kCtrlRegs - 4 * NG * 32 * kGenRegs) / kEpiThreads) / 8 * 8;
    static_assert(EW % 4 == 0 && kThreads <= 1024 && kCtrlRegs <= kLaunchRegs && kEpiRegs >= 96 && kEpiRegs <= 255 &&
                  128 * kCtrlRegs + 4 * NG * 32 * kGenRegs + kEpiThreads * kEpiRegs <= kLaunchRegs * kThreads, "role split");
};

struct TensorParams {
    int nl;             // NL: half-width of a frequency group (multiple of 8, <= 112); group width L = 2 NL = MMA N
    int tile;           // frequencies per tile = 64 * 2 NL
    int n_ops;          // FP16 planes of a B stage: 4 (hi and lo of the Z- and W-operands) or 2 (fast_math: hi only)
    int stages_b;       // B-operand ring depth (TMA -> MMA)
    int long_items;     // 1: many stages per item -> the (4 epilogue warps, 4 generator groups) shape; 0: (8, 3)
    int b_plane_bytes;  // bytes of one FP16 plane of a B stage in a CTA's shared memory: 2 NL * 32 (pair mode: NL * 32, the CTA's half)
    int b_stage_bytes;  // bytes of one stage of the TABLE: n_ops * 2 NL * 32 + kTcAuxBytes
    int smem_stage_bytes;   // bytes of one B stage in a CTA's ring: n_ops * b_plane_bytes + kTcAuxBytes
    int pair;           // 1: CTA pairs (2-CTA clusters, tcgen05 cta_group::2): an item is (object, PAIR of tiles, split), CTA rank r
                        // takes tile 2 q + r and holds columns [r NL, (r + 1) NL) of every B plane (the "Re b" / "Im b" half);
                        // the table stage is laid out [half 0][half 1][aux]
    int fixup;          // n_split > 1: 1 = partial slots in the epilogue's own order, finished by lsp_tensor_fix_kernel;
                        // 0 = partial sums per grid frequency (generalised mode)
    int weighted;       // generalised mode: the W operand carries the weights w_j (aux.w) instead of 1
    int z_only;         // generalised mode, second pass: only the Z contraction is wanted
    int y_is_w;         // generalised mode, second pass: the Z operand carries the weights (aux.w, scale wscale) instead of y
    int gls;            // generalised mode fused into the epilogue (n_split = 1): 1 = this launch writes (C, S) = sum w e^{i theta}
                        // per element in the epilogue's own order (float2); 2 = this launch (weighted W) reads them back and
                        // evaluates ZK09's power in place of step 5
};

// Generalised Lomb-Scargle power from the six weighted sums (Zechmeister & Kuerster 2009 Eq. 4-5; lsp_gls.cuh has the notation),
// FP32 arithmetic for the fused epilogue: weights are normalised (sum w = 1), so CC, SS, CS are O(1).
__device__ __forceinline__ float gls_power_f32(float YC, float YS, float C, float S, float c2, float s2, float inv_chi0)
{
    const float CC = fmaf(-C, C, 0.5f * (1.0f + c2)), SS = fmaf(-S, S, 0.5f * (1.0f - c2)), CS = fmaf(-C, S, 0.5f * s2);
    const float D = fmaf(CC, SS, -CS * CS);
    float p = 0.0f;
    if (D > 1e-5f) p = (SS * YC * YC + CC * YS * YS - 2.0f * CS * YC * YS) / D;
    else if (CC > 1e-5f) p = YC * YC / CC;                // aliased design matrix: the vanishing direction is dropped
    else if (SS > 1e-5f) p = YS * YS / SS;
    return p * inv_chi0;
}

// Per-object pre-pass results of the tensor path.
struct TensorObj {
    double  mean;       // subtracted from y (0 unless center = 1)
    float   yscale;     // power of two: max |y - mean| * yscale in [256, 512)
    float   pscale;     // output scale: nrm * 256 / yscale^2
    float   zinv;       // 1 / yscale (partial sums are written un-scaled)
    float   nrm;        // normalize ? 2 / sum (y-mean)^2 : 1
    float   wscale;     // weighted mode: power of two, max w * wscale in [256, 512); else 256
    float   winv;       // 1 / wscale
};

__host__ __device__ inline int tc_n_kb(int64_t n_t) { return (int)((n_t + kTcKB - 1) / kTcKB); }
// First table block of launch-local object o: floor(offset / 16) + o.  It needs no scan over the objects and leaves every
// object at least ceil(N_t / 16) blocks (the table is sized total_obs / 16 + n_obj blocks; a few blocks stay unused).
__device__ __forceinline__ int64_t tc_kb_off(const int64_t* __restrict__ offsets, int64_t obj_base, int64_t o)
{
    return (offsets[obj_base + o] - offsets[obj_base]) / kTcKB + o;
}

// Programmatic dependent launch (the tensor path's launches are chained: pre-pass -> main -> fix): a kernel lets its dependent
// start launching early (`pdl_trigger`), the dependent waits for the prerequisite grid to have completed and flushed its
// memory before touching its results (`pdl_wait`).  Hides the launch latency between the launches; both are no-ops when the
// kernel was launched without the attribute.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ void split_half2(float x0, float x1, __half2* hi, __half2* lo)
{
    const __half2 h = __floats2half2_rn(x0, x1);
    const float2 b = __half22float2(h);
    *hi = h;
    *lo = __floats2half2_rn(x0 - b.x, x1 - b.y);
}

// ---- the pre-pass: ONE launch ----------------------------------------------------------------------------------------
// Blocks [0, n_table_blocks): one block per (object, 16-observation block) of the B-operand table; thread m < NL owns offset m.
//   Stage layout (FP16), identical to one shared-memory B stage:  [plane: b_hi, b2_hi, (b_lo, b2_lo)] [k chunk c = 0,1]
//   [column n] [k%8] with column n = m (Re) or NL + m (Im) and observation 16 kb + 8 c + k%8, then the aux block (FP32).
//   Observations past N_t are zero everywhere (v = 0 makes the generated A operand vanish too).
// Blocks [n_table_blocks, n_table_blocks + n_obj): per-object statistics (mean, power-of-two scales).
template <bool FAST>
__global__ void __launch_bounds__(kTcPreThreads)
lsp_tensor_prepass_kernel(GridParams gp, TensorParams tp, const int64_t* __restrict__ offsets, const float* __restrict__ t,
                          const float* __restrict__ y, const float* __restrict__ wgt, TensorObj* __restrict__ objs, int n_obj,
                          long long n_table_blocks, int center, int normalize, unsigned char* __restrict__ table)
{
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    pdl_trigger();
    if ((long long)blockIdx.x >= n_table_blocks) {
        // ---------------- statistics of object o ----------------
        __shared__ double red[4][4];
        const int o = (int)((long long)blockIdx.x - n_table_blocks);
        const int64_t lo = offsets[gp.obj_base + o], n = offsets[gp.obj_base + o + 1] - lo;
        double s = 0.0;
        if (center) {
            for (int64_t j = tid; j < n; j += kTcPreThreads) s += (double)y[lo + j];
            for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
            if (lane == 0) red[0][wid] = s;
            __syncthreads();
            s = red[0][0] + red[0][1] + red[0][2] + red[0][3];
        }
        const double mean = (center && n > 0) ? s / (double)n : 0.0;
        double q = 0.0, mx = 0.0, mw = 0.0;
        for (int64_t j = tid; j < n; j += kTcPreThreads) {
            const double v = (double)y[lo + j] - mean;
            q += v * v;
            mx = fmax(mx, fabs(v));
            if (wgt) mw = fmax(mw, fabs((double)wgt[lo + j]));
        }
        for (int d = 16; d > 0; d >>= 1) {
            q += __shfl_xor_sync(0xffffffffu, q, d);
            mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
            mw = fmax(mw, __shfl_xor_sync(0xffffffffu, mw, d));
        }
        if (lane == 0) { red[1][wid] = q; red[2][wid] = mx; red[3][wid] = mw; }
        __syncthreads();
        if (tid == 0) {
            q = red[1][0] + red[1][1] + red[1][2] + red[1][3];
            mx = fmax(fmax(red[2][0], red[2][1]), fmax(red[2][2], red[2][3]));
            mw = fmax(fmax(red[3][0], red[3][1]), fmax(red[3][2], red[3][3]));
            auto pow2_scale = [](double m) {       // 2^e with m * 2^e in [256, 512); 1 for m = 0 / non-finite
                int e = 0;
                if (!(m > 0.0) || !isfinite(m)) return 1.0;
                frexp(m, &e);                      // m = f * 2^e, f in [0.5, 1)
                return ldexp(1.0, max(-100, min(100, 9 - e)));
            };
            TensorObj ob;
            ob.mean = mean;
            const double ys = pow2_scale(mx);
            ob.yscale = (float)ys;
            ob.zinv = (float)(1.0 / ys);
            const double nrm = normalize ? (q > 0.0 ? 2.0 / q : 0.0) : 1.0;
            ob.nrm = (float)nrm;
            ob.pscale = (float)(nrm * (double)kTcUnitScale / (ys * ys));
            const double ws = wgt ? pow2_scale(mw) : (double)kTcUnitScale;
            ob.wscale = (float)ws;
            ob.winv = (float)(1.0 / ws);
            objs[o] = ob;
        }
        return;
    }
    // ---------------- one stage of the B-operand table ----------------
    const int64_t blk = blockIdx.x;
    int lo_o = 0, hi_o = n_obj - 1;                 // largest o with kb_off(o) <= blk (kb_off is strictly increasing)
    while (lo_o < hi_o) {
        const int mid = (lo_o + hi_o + 1) >> 1;
        if (tc_kb_off(offsets, gp.obj_base, mid) <= blk) lo_o = mid; else hi_o = mid - 1;
    }
    const int o = lo_o;
    const int64_t base = offsets[gp.obj_base + o], n_t = offsets[gp.obj_base + o + 1] - base;
    const int kb = (int)(blk - tc_kb_off(offsets, gp.obj_base, o));
    if (kb >= tc_n_kb(n_t)) return;                 // slack block between two objects
    unsigned char* stage = table + (size_t)blk * (size_t)tp.b_stage_bytes;
    const int L = 2 * tp.nl;
    const int full_plane_bytes = L * kTcKB * 2;                     // one FP16 plane of all 2 NL columns
    {   // aux: t, y, w of the 16 observations and the tile-independent phasors v (two versions)
        float* aux = reinterpret_cast<float*>(stage + (size_t)tp.n_ops * full_plane_bytes);
        const int j16 = tid & 15, g1 = tid >> 4;
        const int64_t j = (int64_t)kb * kTcKB + j16;
        const bool live = j < n_t;
        const float tj = live ? t[base + j] : 0.f;
        if (tid < 16) {
            aux[tid] = tj;
            aux[16 + tid] = live ? y[base + j] : 0.f;
            aux[32 + tid] = live ? (wgt ? wgt[base + j] : 1.f) : 0.f;
        }
        float sn = 0.f, cs = 0.f;
        if (live) {
            const float r = (float)frac_cycles((double)(8 * g1) * (double)L * gp.df * (double)tj);
            if (FAST) sincos_cycles<true>(r, &sn, &cs); else sincos_cycles_reduced(r, &sn, &cs);
        }
        const float h = 0.70710678118654752f;
        const int pos = 4 * (j16 >> 1) + (j16 & 1);                // pair-planar: (c0, c1, s0, s1)
        aux[48 + g1 * kTcVRow + pos] = cs;
        aux[48 + g1 * kTcVRow + pos + 2] = sn;
        aux[48 + (8 + g1) * kTcVRow + pos] = (cs + sn) * h;
        aux[48 + (8 + g1) * kTcVRow + pos + 2] = (sn - cs) * h;
    }
    const int m = tid;
    if (m >= tp.nl) return;
    const double f_beta = ((double)m + 0.5) * gp.df;
    // unpaired: [plane][k chunk c][column n < 2 NL][8];  pair mode: [half r][plane][k chunk c][column n' < NL][8], half 0 = the
    // "Re b" columns, half 1 = the "Im b" columns (what CTA rank r of a pair holds)
    const int n_cols = tp.pair ? tp.nl : L;                         // columns of one plane as stored
    const int plane = n_cols * kTcKB;                               // halfs per stored plane
    const size_t im_base = tp.pair ? (size_t)tp.n_ops * plane : (size_t)tp.nl * 8;     // where the "Im b" columns start
    __half* dst = reinterpret_cast<__half*>(stage);
    float c1[kTcKB], s1[kTcKB];
#pragma unroll
    for (int k = 0; k < kTcKB; ++k) {
        const int64_t j = (int64_t)kb * kTcKB + k;
        float sn = 0.f, cs = 0.f;
        if (j < n_t) {
            const float r = (float)frac_cycles(f_beta * (double)t[base + j]);
            if (FAST) sincos_cycles<true>(r, &sn, &cs); else sincos_cycles_reduced(r, &sn, &cs);
        }
        c1[k] = cs;
        s1[k] = sn;
    }
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        __half2 re_h[4], re_l[4], im_h[4], im_l[4], re2_h[4], re2_l[4], im2_h[4], im2_l[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const int k = c * 8 + 2 * p;
            split_half2(c1[k], c1[k + 1], &re_h[p], &re_l[p]);
            split_half2(s1[k], s1[k + 1], &im_h[p], &im_l[p]);
            const float cc0 = fmaf(c1[k], c1[k], -s1[k] * s1[k]), ss0 = 2.f * c1[k] * s1[k];
            const float cc1 = fmaf(c1[k + 1], c1[k + 1], -s1[k + 1] * s1[k + 1]), ss1 = 2.f * c1[k + 1] * s1[k + 1];
            split_half2(cc0, cc1, &re2_h[p], &re2_l[p]);
            split_half2(ss0, ss1, &im2_h[p], &im2_l[p]);
        }
        const size_t off_re = (size_t)c * (n_cols * 8) + (size_t)m * 8;            // [c][n/8][n%8][8] == [c][n][8]
        const size_t off_im = off_re + im_base;
        auto put = [&](int pl, size_t off, const __half2* v) {
            uint4 u;
            u.x = *reinterpret_cast<const unsigned*>(&v[0]);
            u.y = *reinterpret_cast<const unsigned*>(&v[1]);
            u.z = *reinterpret_cast<const unsigned*>(&v[2]);
            u.w = *reinterpret_cast<const unsigned*>(&v[3]);
            *reinterpret_cast<uint4*>(dst + (size_t)pl * plane + off) = u;
        };
        put(0, off_re, re_h);  put(0, off_im, im_h);
        put(1, off_re, re2_h); put(1, off_im, im2_h);
        if (!FAST) {
            put(2, off_re, re_l);  put(2, off_im, im_l);
            put(3, off_re, re2_l); put(3, off_im, im2_l);
        }
    }
}

// ---- tcgen05 / TMA wrappers ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t tc_smem_desc(unsigned saddr, unsigned lbo_bytes, unsigned sbo_bytes)
{
    // no-swizzle K-major canonical layout: ((8, n), 2) : ((16 B, SBO), LBO); version 1 (sm_100)
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
// D[tmem] (+)= A[tmem] * B[smem]: the A operand (128 rows x 16 FP16 = 8 columns, row = lane, k even in the low half-word)
// is read from tensor memory, B through a shared-memory descriptor.
__device__ __forceinline__ void tc_mma_f16_ts(unsigned d_tmem, unsigned a_tmem, uint64_t b_desc, unsigned idesc, unsigned accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tc_commit(unsigned long long* bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// ---- CTA pairs (2-CTA clusters, cta_group::2): the leader (cluster rank 0) issues every MMA for both CTAs; M = 256 = the 128
// A rows each CTA generated into its own tensor memory, N = the two CTAs' halves of B side by side; each CTA accumulates its
// own 128 x N tile in its own tensor memory.
__device__ __forceinline__ unsigned cluster_ctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of the same variable in CTA `rank` of the cluster
__device__ __forceinline__ unsigned cluster_map(unsigned saddr, unsigned rank)
{
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(unsigned cluster_addr)
{
    // default semantics (release at CTA scope), as a local arrive: what crosses the pair is tensor-memory / async-proxy state,
    // ordered by the tcgen05 fences around it; a cluster-scope release would cost a MEMBAR.ALL.GPU per arrival
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void tc_mma_f16_ts2(unsigned d_tmem, unsigned a_tmem, uint64_t b_desc, unsigned idesc, unsigned accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// arrives (once the MMAs issued so far have completed) on the barrier at this shared-memory offset in BOTH CTAs of the pair
__device__ __forceinline__ void tc_commit2(unsigned long long* bar)
{
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(smem_u32(bar)), "h"((unsigned short)3) : "memory");
}
// mbarrier wait for roles whose waits are long when they are not the bottleneck (generators on a full ring, epilogue on
// unfinished accumulators): back off between polls so the spinning warps do not take issue slots from the working ones.
__device__ __forceinline__ void mbar_wait_backoff(unsigned long long* bar, unsigned parity, unsigned ns = 40u)
{
    unsigned done;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    while (!done) {
        __nanosleep(ns);
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ bool elect_one()
{
    unsigned pred;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_ld16(unsigned taddr, float* v)
{
    unsigned r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tc_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// 8 consecutive TMEM columns of this thread's lane <- 8 registers (one A-operand plane of a stage: 16 FP16 of one row)
__device__ __forceinline__ void tc_st8(unsigned taddr, const unsigned (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
}
__device__ __forceinline__ void tc_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ float4 lds128(unsigned saddr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(saddr));
    return v;
}
__device__ __forceinline__ float lds32(unsigned saddr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(saddr));
    return v;
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void* smem_dst, const void* gmem_src, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

struct TcItem {
    int64_t obj_local, obj, n_t, K0;
    int tile, split, kb0, kb1;
    bool tile_ok;       // false: the phantom second tile of the last pair of an odd tile count (pair mode): computed, never stored
};
__device__ __forceinline__ TcItem tc_decode(const GridParams& gp, const TensorParams& tp, long long item,
                                            const int64_t* __restrict__ offsets, int rank = 0)
{
    TcItem w;
    // (the host launches at most 2^31 - 1 items: 32-bit divisions; every role decodes every item of its CTA)
    const unsigned it32 = (unsigned)item, ns = (unsigned)gp.n_split;
    const unsigned r = ns == 1 ? it32 : it32 / ns;
    w.split = (int)(it32 - r * ns);
    if (tp.pair) {
        const unsigned n_tp = (unsigned)(gp.n_tiles + 1) >> 1, o = r / n_tp;
        w.tile = 2 * (int)(r - o * n_tp) + rank;
        w.obj_local = o;
    } else {
        const unsigned o = r / (unsigned)gp.n_tiles;
        w.tile = (int)(r - o * (unsigned)gp.n_tiles);
        w.obj_local = o;
    }
    w.tile_ok = w.tile < gp.n_tiles;
    w.obj = w.obj_local + gp.obj_base;
    w.n_t = offsets[w.obj + 1] - offsets[w.obj];
    const int nkb = tc_n_kb(w.n_t);
    if (ns == 1) {
        w.kb0 = 0;
        w.kb1 = nkb;
    } else {
        w.kb0 = (int)(((long long)nkb * w.split) / gp.n_split);
        w.kb1 = (int)(((long long)nkb * (w.split + 1)) / gp.n_split);
    }
    w.K0 = (int64_t)w.tile * tp.tile;
    return w;
}

// static shared memory of the kernel (generator scratch etc.), for the ring sizing here and on the host
constexpr int tc_static_smem_of(int ew, int ng) { return ng * 2 * (8 * kTcVRow + 32) * 4 + ew * 16 + 256; }
// B stages of the largest tile (NL = mnl) that fit beside it: dynamic = 1 KB alignment slack + ring + 384 B of barriers
__host__ __device__ constexpr int tc_b_fit(int pm, int ew, int ng, bool pair, int mnl)
{
    const int stage = (pm == 1 ? 2 : 4) * (pair ? 1 : 2) * mnl * 32 + kTcAuxBytes;
    const int fit = (232448 - tc_static_smem_of(ew, ng) - 1024 - 384 - 512) / stage;
    return fit < kTcMaxSB ? fit : kTcMaxSB;
}
// Depth D of the A ring (operand stages in flight between the generators and the MMA warp).  A slot is recycled only after
// the MMAs that read it have COMPLETED and the news has travelled commit -> generator -> tcgen05.st -> arrive -> MMA warp
// (measured ~1500 cycles on a CTA pair), so the kernel sustains at most D stages per (that + the stage's MMA time): the ring is
// made as deep as the tensor-memory columns left of the accumulators allow (512 - 4 mnl columns; a stage is 16 columns, 32 with
// three products); narrower tiles would buy a deeper ring, but the generators redo their work per tile (measured: NL <= 104 and
// a 6-deep ring is 8 % slower than NL <= 112 and 4).  The generators
// wait on the B ring's "full" barriers out of step with the MMA warp, and their parity waits stay within one phase of the
// barrier only if the B ring is at least NG + D stages deep: D is capped by what fits in shared memory at NL = mnl.
__host__ __device__ constexpr int tc_a_depth(int pm, int ew, int ng, bool pair, int mnl)
{
    int d = (512 - 4 * mnl) / (pm == 0 ? 32 : 16);
    if (d > 8) d = 8;
    const int room = tc_b_fit(pm, ew, ng, pair, mnl) - ng;
    return d < room ? d : room;
}
// ---- split-N_t fix-up (n_split > 1) ----------------------------------------------------------------------------------
// The n_split partial slots of a tile (lane-oriented un-scaled sums in the epilogue's own element order: element (i, row r)
// at i * 128 + r, see the epilogue) are added in SPLIT ORDER -- results do not depend on scheduling -- and steps 5, 6, 6'
// run on the totals.  One CTA per (object, tile, part): part p of kTcFixParts takes every kTcFixParts-th unit; a unit is
// (row, four consecutive m); consecutive threads take consecutive rows, so every load is fully coalesced.  A kernel of its
// own because it needs the whole GPU's memory parallelism: the same sums inside the main kernel's epilogue warps (a few
// hundred threads per tile) are bound by the latency of their few loads in flight.
constexpr int kTcFixThreads = 256;
#ifndef LSP_TC_FIX_PARTS
#define LSP_TC_FIX_PARTS 16
#endif
constexpr int kTcFixParts = LSP_TC_FIX_PARTS;
template <typename T>
__global__ void __launch_bounds__(kTcFixThreads)
lsp_tensor_fix_kernel(GridParams gp, TensorParams tp, const int64_t* __restrict__ offsets, const TensorObj* __restrict__ objs,
                      const float4* __restrict__ sums, T* __restrict__ out_power, Best* __restrict__ partials, int64_t n_obj_launch)
{
    __shared__ Best sbest[kTcFixThreads / 32];
    pdl_wait();            // the main kernel's partial slots are complete and visible
    const int part = (int)(blockIdx.x % kTcFixParts);
    const long long r0 = blockIdx.x / kTcFixParts;
    const int tile = (int)(r0 % gp.n_tiles);
    const int64_t obj_local = r0 / gp.n_tiles, obj = obj_local + gp.obj_base;
    const int NL = tp.nl, L = 2 * NL;
    const int n_quads = (NL + 3) >> 2;
    const int64_t K0 = (int64_t)tile * tp.tile;
    const int n_valid = (int)min((int64_t)tp.tile, (int64_t)gp.n_freq - K0);
    const bool ragged = n_valid < tp.tile;
    const bool vec_ok = (gp.n_freq % 4 == 0) && ((reinterpret_cast<uintptr_t>(out_power) & 15) == 0);
    const float n_t = (float)(offsets[obj + 1] - offsets[obj]);
    const float nrm = objs[obj_local].nrm;
    const int64_t tile_elems = (int64_t)((NL + 15) >> 4) * 16 * 128;
    const float4* slot0 = sums + (obj_local * gp.n_tiles + tile) * tile_elems;
    const int64_t sstride = n_obj_launch * (int64_t)gp.n_tiles * tile_elems;
    T* otile = out_power ? out_power + obj_local * (int64_t)gp.n_freq + K0 : nullptr;
    float bp = -1.0f;
    int bk = 0x7fffffff;
    for (int u = part * kTcFixThreads + threadIdx.x; u < 128 * n_quads; u += kTcFixParts * kTcFixThreads) {
        const int r = u & 127, i0 = (u >> 7) * 4;
        const bool is_im = (r & 16) != 0;
        const int g = 16 * (r >> 5) + (r & 15);
        const int kc = g * L + NL;
        const float4* src = slot0 + (int64_t)i0 * 128 + r;
        float4 acc[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[e] = make_float4(0.f, 0.f, 0.f, 0.f);
        int sp = 0;
        for (; sp + 4 <= gp.n_split; sp += 4) {                    // fixed order: split 0, 1, 2, ...; 16 loads in flight (many-split
            float4 v[4][4];                                        // launches are latency-bound here: few CTAs, long dependent chains)
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
                for (int e = 0; e < 4; ++e) v[q][e] = src[(int64_t)(sp + q) * sstride + e * 128];
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    acc[e].x += v[q][e].x;  acc[e].y += v[q][e].y;  acc[e].z += v[q][e].z;  acc[e].w += v[q][e].w;
                }
        }
        for (; sp + 2 <= gp.n_split; sp += 2) {                    // 8 loads in flight
            float4 v0[4], v1[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                v0[e] = src[(int64_t)sp * sstride + e * 128];
                v1[e] = src[(int64_t)(sp + 1) * sstride + e * 128];
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                acc[e].x = (acc[e].x + v0[e].x) + v1[e].x;  acc[e].y = (acc[e].y + v0[e].y) + v1[e].y;
                acc[e].z = (acc[e].z + v0[e].z) + v1[e].z;  acc[e].w = (acc[e].w + v0[e].w) + v1[e].w;
            }
        }
        if (sp < gp.n_split) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const float4 v = src[(int64_t)sp * sstride + e * 128];
                acc[e].x += v.x;  acc[e].y += v.y;  acc[e].z += v.z;  acc[e].w += v.w;
            }
        }
        // Re rows: (x, y, z, w) = (xc, xs, c2, s2) of k = kc + i;  Im rows: (xs, xc, s2, c2) of k = kc - 1 - i
        float pw[4];
#pragma unroll
        for (int e = 0; e < 4; ++e)
            pw[e] = power_from_sums<float>(is_im ? acc[e].y : acc[e].x, is_im ? acc[e].x : acc[e].y, is_im ? acc[e].w : acc[e].z,
                                           is_im ? acc[e].z : acc[e].w, n_t, nrm);
        const int klv = is_im ? (kc - i0 - 4) : (kc + i0);         // first of the four consecutive grid points
        float o4[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) o4[e] = is_im ? pw[3 - e] : pw[e];      // ascending frequency
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int k = klv + e;
            if (k < n_valid && o4[e] == o4[e] && (o4[e] > bp || (o4[e] == bp && k < bk))) { bp = o4[e]; bk = k; }
        }
        if (otile) {
            if (!ragged && vec_ok) {
                *reinterpret_cast<float4*>(otile + klv) = make_float4(o4[0], o4[1], o4[2], o4[3]);
            } else {
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    if (klv + e < n_valid) otile[klv + e] = (T)o4[e];
            }
        }
    }
    if (partials) {
        Best mine;
        mine.p = (double)bp;
        mine.k = (bk == 0x7fffffff) ? INT64_MAX : K0 + (int64_t)bk;
        const Best b = block_best(mine, sbest);
        if (threadIdx.x == 0) partials[(obj_local * gp.n_tiles + tile) * kTcFixParts + part] = b;
    }
}

constexpr size_t tc_smem_bytes(int stages_b, int b_stage)
{
    return 1024 /* alignment slack */ + (size_t)stages_b * (size_t)b_stage + 384 /* barriers */;
}
template <int EW, int NG> constexpr int tc_static_smem() { return tc_static_smem_of(EW, NG); }

// GM (generalised mode): 0 = standard; 1 = the W slot carries the weights (partial-sum output); 2 = 1 + ZK09's power fused into
// the epilogue (n_split = 1).  A template parameter so that the standard kernel carries none of it.
// PM (precision mode): 0 = three products a_hi b_hi + a_hi b_lo + a_lo b_hi; 2 = two products a_hi (b_hi + b_lo) -- the A
// operand is one FP16 (the generators skip the low part, the A ring is twice as deep), the B table is the same;
// 1 = fast_math: one product and MUFU sincos.
// PAIR: CTA pairs (2-CTA clusters; the launch carries the cluster dimension): see TensorParams::pair.
// MNL: the largest NL the instantiation accepts; fixes the tensor-memory layout: Z accumulators [0, 2 NL), W accumulators
// [2 MNL, 2 MNL + 2 NL), A ring [4 MNL, 512).
template <typename T, int PM, int EW, int NG, int GM, bool PAIR = false, int MNL = kTcMaxNL>
__global__ void __launch_bounds__((TcRoles<EW, NG>::kThreads), 1)
lsp_tensor_kernel(GridParams gp, TensorParams tp, const int64_t* __restrict__ offsets, const TensorObj* __restrict__ objs,
                  const unsigned char* __restrict__ table, T* __restrict__ out_power, Best* __restrict__ partials,
                  float4* __restrict__ sums, int64_t n_obj_launch, long long total_items, const double* __restrict__ gls_yy)
{
    using R = TcRoles<EW, NG>;
    constexpr bool WGT = GM != 0, FUSED = GM == 2;
    constexpr int kEpiWarps = EW, kEpiThreads = R::kEpiThreads;
    constexpr bool FAST = PM == 1;                            // MUFU sincos, B table without low planes
    constexpr bool A_LO = PM == 0;                            // the A operand carries a low part
    constexpr int NOPS = FAST ? 2 : 4;                        // FP16 planes of a B stage
    constexpr int A_STAGE_COLS = (A_LO ? 4 : 2) * 8;          // TMEM columns of one A stage
    constexpr int WCOL = 2 * MNL, ACOL = 4 * MNL;             // first TMEM column of the W accumulators / of the A ring
    constexpr int AS = (512 - ACOL) / A_STAGE_COLS;           // A stages that fit in the ring's columns
    // Hand-off protocol of the A ring.  Stage s (numbered per CTA across items) is built by generator group s % NG into TMEM
    // slot s % D (tc_a_depth).  full_a[slot]: the generators' arrivals, waited on by the MMA warp only, in order.  "Slot free" is
    // the commit that follows the MMAs of a stage.  mbarrier waits are parity waits, so a waiter must never be two phases away
    // from its barrier (in either direction); which barrier carries the signal therefore depends on the shape:
    //   D >= NG: one barrier per SLOT.  Use u of a slot (stage u D + q) waits for the slot's u-th arrival.  Arrival u + 1 needs use
    //            u built, whose builder has consumed arrival u; and the builder of stage s has already waited for MMA(s - NG - D),
    //            which completes after MMA(s - 2 D) (NG <= D), i.e. arrival u - 1 has happened when it starts to wait.
    //   D <  NG: one barrier per GROUP: the commit after the MMAs of stage j arrives on the barrier of group (j + D) % NG, which
    //            will write stage j + D into that slot.  A group sees exactly one arrival per stage it builds (none for its first
    //            if that is one of the CTA's first D), waits for them strictly in order, and arrival i + 1 cannot precede its
    //            consumption of arrival i (it needs MMA(s + NG - D), issued after MMA(s), which needs this group's stage s).
    constexpr int D = tc_a_depth(PM, EW, NG, PAIR, MNL);
    static_assert(D >= 1 && D <= AS && D <= 8 && NG <= 8 && MNL % 8 == 0 && MNL <= 112, "A ring depth");
    constexpr bool PER_SLOT = D >= NG;
    constexpr int NFREE = PER_SLOT ? D : NG;                  // "slot free" barriers in use
    static_assert(!PAIR || GM == 0, "pair mode is built for the standard periodogram only");
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem_b = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
    const int SB = tp.stages_b;
    const unsigned b_bytes = (unsigned)tp.smem_stage_bytes;       // one B stage in this CTA's ring
    const unsigned rank = PAIR ? cluster_ctarank() : 0u;         // pair mode: 0 = leader (issues the MMAs of both CTAs)
    // this CTA's item sequence: items first, first + stride, ... (pair mode: both CTAs of a cluster walk the same sequence)
    const long long first = PAIR ? (long long)(blockIdx.x >> 1) : (long long)blockIdx.x;
    const long long stride = PAIR ? (long long)(gridDim.x >> 1) : (long long)gridDim.x;
    const int aux_off = NOPS * tp.b_plane_bytes;              // byte offset of the aux block inside a B stage
    unsigned long long* full_b = reinterpret_cast<unsigned long long*>(smem_b + (size_t)SB * b_bytes);
    unsigned long long* empty_b = full_b + kTcMaxSB;
    unsigned long long* full_a = empty_b + kTcMaxSB;
    unsigned long long* free_s = full_a + 8;
    unsigned long long* tmem_full = free_s + 8;
    unsigned long long* tmem_empty = tmem_full + 1;
    __shared__ unsigned tmem_base_s;
    __shared__ Best sbest[kEpiWarps];
    // generator scratch: [group][buffer]: 8 rows (g0) of the tile's phasors u * 16, pair-planar like the aux rows, then the
    // stage's scaled magnitudes for the "Re a" rows (16) and the "Im a" rows (16)
    __shared__ __align__(16) float s_u[NG][2][8 * kTcVRow + 32];

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);      // broadcast: the compiler may treat the role as warp-uniform
    if (tid == 0) {
        for (int s = 0; s < SB; ++s) {
            mbar_init(&full_b[s], 1);
            mbar_init(&empty_b[s], 1);
        }
        // one arrival per generator warp of the stage's group; pair mode: of both CTAs, on the leader's barrier
        for (int s = 0; s < D; ++s) mbar_init(&full_a[s], PAIR ? 8 : 4);
        for (int s = 0; s < NFREE; ++s) mbar_init(&free_s[s], 1);
        mbar_init(tmem_full, 1);
        mbar_init(tmem_empty, PAIR ? 2 * kEpiThreads : kEpiThreads);      // pair mode: both CTAs' epilogues sign off with the leader
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        if (PAIR) {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&tmem_base_s)));
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
        } else {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&tmem_base_s)));
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
        }
    }
    tc_fence_before();
    if (PAIR) cluster_sync_all(); else __syncthreads();          // pair mode: the peer's barriers exist before anything arrives on them
    tc_fence_after();
    // where the generators / the epilogue arrive: the local barrier, or (pair mode) the leader's copy of it
    const unsigned full_a_addr0 = PAIR ? cluster_map(smem_u32(&full_a[0]), 0) : smem_u32(&full_a[0]);
    const unsigned tmem_empty_addr = PAIR ? cluster_map(smem_u32(tmem_empty), 0) : smem_u32(tmem_empty);
    auto arrive_tmem_empty = [&]() {
        if (PAIR) mbar_arrive_cluster(tmem_empty_addr); else mbar_arrive(tmem_empty);
    };
    const unsigned tmem = tmem_base_s;
    pdl_trigger();
    pdl_wait();            // the pre-pass's table and statistics are complete and visible from here on

    if (warp < 4) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R::kCtrlRegs));
    if (warp == 0) {
        // =============================== TMA producer: B stages (+ aux) from the per-object table ================
        if (lane == 0) {
            int st = 0;
            unsigned ph = 1;                                      // parity of the "empty" phase to wait for
            const unsigned t_bytes = (unsigned)tp.b_stage_bytes;      // one stage of the table
            const unsigned half_bytes = (unsigned)(NOPS * tp.b_plane_bytes);      // pair mode: this CTA's half of the planes
            for (long long item = first; item < total_items; item += stride) {
                const TcItem w = tc_decode(gp, tp, item, offsets, (int)rank);
                const unsigned char* src = table + (size_t)(tc_kb_off(offsets, gp.obj_base, w.obj_local) + w.kb0) * (size_t)t_bytes;
                for (int kb = w.kb0; kb < w.kb1; ++kb) {
                    mbar_wait(&empty_b[st], ph);
                    mbar_arrive_expect_tx(&full_b[st], b_bytes);
                    if (PAIR) {                                   // table stage = [half 0][half 1][aux]: this CTA's half, then the aux block
                        tma_bulk_g2s(smem_b + (size_t)st * b_bytes, src + (size_t)rank * half_bytes, half_bytes, &full_b[st]);
                        tma_bulk_g2s(smem_b + (size_t)st * b_bytes + half_bytes, src + 2 * (size_t)half_bytes, (unsigned)kTcAuxBytes, &full_b[st]);
                    } else {
                        tma_bulk_g2s(smem_b + (size_t)st * b_bytes, src, b_bytes, &full_b[st]);
                    }
                    src += t_bytes;
                    if (++st == SB) { st = 0; ph ^= 1; }
                }
            }
        }
    } else if (warp == 1 && rank == 0) {
        // =============================== MMA issuer (pair mode: the leader CTA's, for both CTAs) ====================
        // The whole warp runs the loop with warp-uniform values (item ranges are broadcast from lane 0), so descriptors
        // and barrier addresses live in uniform registers; one elected lane issues the MMAs and commits.
        const unsigned idesc = (1u << 4) | ((unsigned)((2 * tp.nl) >> 3) << 17) | ((unsigned)((PAIR ? 256 : 128) >> 4) << 24);
        // bytes between the two k chunks of a plane = columns stored per plane x 16 (pair mode: the CTA's NL columns)
        const unsigned b_lbo = (unsigned)((PAIR ? tp.nl : 2 * tp.nl) / 8) * 128, sbo = 128;
        // Descriptors of B stage 0; stage s adds s * stage_bytes / 16 to the 14-bit start-address field (the whole ring
        // lies below 256 KB, so the field never carries into the LBO bits).
        const unsigned sb0 = smem_u32(smem_b);
        const uint64_t b_zh0 = tc_smem_desc(sb0, b_lbo, sbo), b_wh0 = tc_smem_desc(sb0 + tp.b_plane_bytes, b_lbo, sbo);
        const uint64_t b_zl0 = tc_smem_desc(sb0 + 2 * tp.b_plane_bytes, b_lbo, sbo), b_wl0 = tc_smem_desc(sb0 + 3 * tp.b_plane_bytes, b_lbo, sbo);
        const uint64_t stage_inc_b = (uint64_t)(b_bytes >> 4);
        const unsigned d_z = tmem, d_w = tmem + WCOL, a0 = tmem + ACOL;
        const bool do_w = tp.z_only == 0;
        int sa = 0, stb = 0, gsel = D % NG;                      // A slot, B slot, (D < NG) group that reuses the A slot next
        unsigned pha = 0, phb = 0, n_acc = 0;
        uint64_t sob = 0;                                         // stb * stage_inc_b
        auto mma = [&](unsigned d, unsigned a, uint64_t b, unsigned acc_) {
            if (PAIR) tc_mma_f16_ts2(d, a, b, idesc, acc_); else tc_mma_f16_ts(d, a, b, idesc, acc_);
        };
        auto commit = [&](unsigned long long* bar) {
            if (PAIR) tc_commit2(bar); else tc_commit(bar);
        };
        for (long long item = first; item < total_items; item += stride) {
            const TcItem w = tc_decode(gp, tp, item, offsets);
            const int kb0 = __shfl_sync(0xffffffffu, w.kb0, 0), kb1 = __shfl_sync(0xffffffffu, w.kb1, 0);
            if (kb1 <= kb0) continue;
            // the epilogue (pair mode: of both CTAs) has drained the previous accumulators
            mbar_wait(tmem_empty, (n_acc & 1) ^ 1);
            tc_fence_after();
            unsigned acc = 0;
            for (int kb = kb0; kb < kb1; ++kb) {
                // pair mode: full_a counts the generator warps of both CTAs, and the peer's generators arrive only after the
                // peer's B stage has landed (they read its aux block), so the two waits cover all four operands
                mbar_wait(&full_b[stb], phb);
                mbar_wait(&full_a[sa], pha);
                tc_fence_after();
                if (elect_one()) {
                    // planes (A in TMEM and B in shared memory alike): 0 = Z-operand hi, 1 = W-operand hi, 2 = Z lo, 3 = W lo
                    const unsigned a = a0 + (unsigned)(sa * A_STAGE_COLS);
                    if (PM == 2) {
                        mma(d_z, a, b_zl0 + sob, acc);
                        mma(d_z, a, b_zh0 + sob, 1u);
                        if (do_w) {
                            mma(d_w, a + 8, b_wl0 + sob, acc);
                            mma(d_w, a + 8, b_wh0 + sob, 1u);
                        }
                    } else if (!FAST) {
                        mma(d_z, a + 16, b_zh0 + sob, acc);
                        mma(d_z, a, b_zl0 + sob, 1u);
                        mma(d_z, a, b_zh0 + sob, 1u);
                        if (do_w) {
                            mma(d_w, a + 24, b_wh0 + sob, acc);
                            mma(d_w, a + 8, b_wl0 + sob, 1u);
                            mma(d_w, a + 8, b_wh0 + sob, 1u);
                        }
                    } else {
                        mma(d_z, a, b_zh0 + sob, acc);
                        if (do_w) mma(d_w, a + 8, b_wh0 + sob, acc);
                    }
                    commit(&free_s[PER_SLOT ? sa : gsel]);       // both stages are free once these MMAs have read them
                    commit(&empty_b[stb]);
                }
                __syncwarp();
                acc = 1u;
                sob += stage_inc_b;
                if (++sa == D) { sa = 0; pha ^= 1; }
                if (++gsel == NG) gsel = 0;
                if (++stb == SB) { stb = 0; phb ^= 1; sob = 0; }
            }
            if (elect_one()) commit(tmem_full);                  // accumulators complete
            __syncwarp();
            ++n_acc;
        }
    } else if (warp >= 4 && warp < 4 + kEpiWarps) {
        // =============================== epilogue (steps 5, 6, 6') ================================================
        // Lane l of quadrant q holds row 32 q + l: lanes 0-15 the "Re a" rows (Srr, Sri) of groups 16 q + l, lanes 16-31
        // the "Im a" rows (Sir, Sii) of the same groups.  One shuffle per accumulator pairs them; the Re lane then owns
        // the frequency above the group centre (k = c + m), the Im lane the one below (k = c - 1 - m), so all 32 lanes
        // produce distinct powers.  Indices are tile-local 32-bit integers; the argmax runs in FP32 + int and is widened
        // once per item; bounds are only checked on the grid's ragged last tile.
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(R::kEpiRegs));
        const int ew = warp - 4;
        const int q = warp & 3;                                   // TMEM lane quadrant this warp may access
        const int half_sel = ew >> 2;                             // which part of the m range (EW / 4 parts)
        constexpr int kParts = EW / 4;
        const int etid = tid - 128;
        const bool is_im = lane >= 16;
        const int g = 16 * q + (lane & 15);
        const int NL = tp.nl, L = 2 * NL;
        const int n_chunks = (NL + 15) >> 4;                      // 16-column chunks over m (NL is a multiple of 8)
        const int ch0 = (n_chunks * half_sel) / kParts, ch1 = (n_chunks * (half_sel + 1)) / kParts;
        const bool vec_ok = (gp.n_freq % 4 == 0) && ((reinterpret_cast<uintptr_t>(out_power) & 15) == 0);
        const int kc = g * L + NL;                                // tile-local index of the first frequency above the centre
        const bool do_w = tp.z_only == 0;
        unsigned n_acc = 0;
        for (long long item = first; item < total_items; item += stride) {
            const TcItem w = tc_decode(gp, tp, item, offsets, (int)rank);
            const TensorObj ob = objs[w.obj_local];
            const bool have = w.kb1 > w.kb0;
            if (FUSED) {
                // generalised mode, fused: pull this warp's (C, S) lines of the tile into L2 while the item's MMAs still run
                const float2* base = reinterpret_cast<const float2*>(sums) + (w.obj_local * gp.n_tiles + w.tile) * ((int64_t)n_chunks * 16 * 128) + 32 * q;
                for (int ch = ch0; ch < ch1; ++ch) {
                    const float2* ptr = base + (int64_t)(16 * ch + (lane >> 1)) * 128 + (lane & 1) * 16;      // 32 lines of 128 bytes per chunk
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr));
                }
            }
            if (have) {
                mbar_wait_backoff(tmem_full, n_acc & 1, EW == 4 ? 400u : 100u);     // long items: the wait lasts a whole item
                tc_fence_after();
            }
            float bp = -1.0f;                                     // running maximum (P >= 0; NaN never compares greater)
            int bi = -1;                                          // its position m = 16 ch + i in this lane's sequence
            const float n_hat = kTcUnitScale * (float)w.n_t;
            const float nn = n_hat * n_hat, nn_eps = 2e-6f * nn;
            const int n_valid = (int)min((int64_t)tp.tile, (int64_t)gp.n_freq - w.K0);     // frequencies of this tile on the grid
            const bool ragged = n_valid < tp.tile;
            T* otile = out_power ? out_power + w.obj_local * (int64_t)gp.n_freq + w.K0 : nullptr;
            const unsigned ta = tmem + ((unsigned)(32 * q) << 16);
            bool released = false;
            // generalised mode, fused (tp.gls == 2): this tile's (C, S) of the earlier launch, and 1 / chi0^2 of the object
            const float2* gls_cs = FUSED ? reinterpret_cast<const float2*>(sums) +
                                                              (w.obj_local * gp.n_tiles + w.tile) * ((int64_t)n_chunks * 16 * 128) + 32 * q + lane
                                                        : nullptr;
            float inv_chi0 = 0.f;
            if (FUSED) {
                const double c0 = gls_yy[w.obj];
                inv_chi0 = c0 > 0.0 ? (float)(1.0 / c0) : 0.f;
            }
            // one chunk = 16 accumulator columns of each of the four TMEM regions; RAG = the tile overhangs the grid
            auto chunk = [&](int ch, auto rag_tag) {
                constexpr bool RAG = decltype(rag_tag)::value;
                const int m0 = ch * 16;
                float zr[16], zi[16], wr[16], wi[16];
                float2 csv[FUSED ? 16 : 1];
                if (FUSED) {                                      // the chunk's (C, S): all 16 loads in flight before anything waits
#pragma unroll
                    for (int i = 0; i < 16; ++i) csv[i] = __ldcg(gls_cs + (int64_t)(m0 + i) * 128);
                }
                if (have) {
                    tc_ld16(ta + m0, zr);
                    tc_ld16(ta + NL + m0, zi);
                    tc_ld16(ta + WCOL + m0, wr);
                    tc_ld16(ta + WCOL + NL + m0, wi);
                    tc_ld_wait();
                    if (ch == ch1 - 1) {                          // last TMEM read of this warp: the MMA warp may overwrite
                        tc_fence_before();
                        arrive_tmem_empty();
                        released = true;
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < 16; ++i) zr[i] = zi[i] = wr[i] = wi[i] = 0.f;
                }
                const int i_lim = min(16, NL - m0);               // 16, or 8 in the last chunk when NL % 16 == 8
                // tile-local index of element i: up lanes kc + m0 + i, down lanes kc - 1 - m0 - i
                const int kl0 = is_im ? (kc - 1 - m0) : (kc + m0);
#pragma unroll
                for (int v4 = 0; v4 < 4; ++v4) {
                    if (4 * v4 >= i_lim) break;
                    float za[4], zb[4], wa[4], wb[4], pw[4];
                    bool bad = false;
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int i = 4 * v4 + e;
                        // partner lane (xor 16) holds the other row of the same group
                        const float p0 = __shfl_xor_sync(0xffffffffu, zr[i], 16), p1 = __shfl_xor_sync(0xffffffffu, zi[i], 16);
                        const float q0 = __shfl_xor_sync(0xffffffffu, wr[i], 16), q1 = __shfl_xor_sync(0xffffffffu, wi[i], 16);
                        // Re lane: (zr, zi) = (Srr, Sri), (p0, p1) = (Sir, Sii): up   Z = (Srr - Sii) + i (Sri + Sir) = za + i zb
                        // Im lane: (zr, zi) = (Sir, Sii), (p0, p1) = (Srr, Sri): down Z = (Srr + Sii) + i (Sir - Sri) = zb + i za
                        za[e] = zr[i] - p1;  zb[e] = zi[i] + p0;
                        wa[e] = wr[i] - q1;  wb[e] = wi[i] + q0;
                        // Step 5 (lsp_common.cuh power_from_sums) written on (za, zb): swapping xc <-> xs only flips the sign
                        // of the c2 term, so with (c, s) = (wa, wb) on Re lanes and (-wb, wa) on Im lanes
                        //   P = [ n (A + B) - c (A - B) - 2 s za zb ] / (n^2 - wa^2 - wb^2),  A = za^2, B = zb^2.
                        const float cc = is_im ? -wb[e] : wa[e], ss = is_im ? wa[e] : wb[e];
                        // (the epilogue is issue-bound on short items: A + B and A - B as two FMAs on B, the denominator as two)
                        const float B = __fmul_rn(zb[e], zb[e]);
                        const float ApB = fmaf(za[e], za[e], B), AmB = fmaf(za[e], za[e], -B);
                        const float den = fmaf(-wa[e], wa[e], fmaf(-wb[e], wb[e], nn));
                        const float num = fmaf(-2.0f * ss, __fmul_rn(za[e], zb[e]), fmaf(-cc, AmB, __fmul_rn(n_hat, ApB)));
                        bad = bad || !(den > nn_eps);
                        // den > nn_eps > 0 here or the value is replaced below: the bare reciprocal (MUFU.RCP + FMUL), without
                        // __fdividef's range scaling
                        pw[e] = __fmul_rn(num, rcp_approx(den)) * ob.pscale;
                    }
                    if (bad) {                                    // vanishing denominator (reading a6): the full epilogue, rarely
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            pw[e] = power_from_sums<float>(is_im ? zb[e] : za[e], is_im ? za[e] : zb[e], is_im ? wb[e] : wa[e],
                                                           is_im ? wa[e] : wb[e], n_hat, ob.pscale);
                    }
                    if (FUSED) {                                  // generalised mode: ZK09's power instead (lsp_gls.cuh)
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const float2 cs = csv[FUSED ? 4 * v4 + e : 0];                              // lane-oriented, like (za, zb)
                            const float ya = za[e] * ob.zinv, yb = zb[e] * ob.zinv, ua = wa[e] * ob.winv, ub = wb[e] * ob.winv;
                            pw[e] = gls_power_f32(is_im ? yb : ya, is_im ? ya : yb, is_im ? cs.y : cs.x, is_im ? cs.x : cs.y,
                                                  is_im ? ub : ua, is_im ? ua : ub, inv_chi0);
                        }
                    }
                    if (partials) {
                        // up lanes meet their frequencies in ascending, down lanes in descending order: "lowest index wins
                        // ties" is "first wins" for the former and "last wins" for the latter
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const int i = 4 * v4 + e;
                            bool take = (pw[e] > bp) || (is_im && pw[e] == bp);
                            if (RAG) take = take && ((is_im ? kl0 - i : kl0 + i) < n_valid);
                            bi = take ? (m0 + i) : bi;
                            bp = take ? pw[e] : bp;
                        }
                    }
                    if (otile) {
                        // element e of the 4-vector in ascending frequency: up -> pw[e], down -> pw[3 - e]
                        const int klv = is_im ? (kl0 - 4 * v4 - 3) : (kl0 + 4 * v4);
                        const float e0 = is_im ? pw[3] : pw[0], e1 = is_im ? pw[2] : pw[1];
                        const float e2 = is_im ? pw[1] : pw[2], e3 = is_im ? pw[0] : pw[3];
                        if (!RAG && vec_ok) {
                            *reinterpret_cast<float4*>(otile + klv) = make_float4(e0, e1, e2, e3);
                        } else {
                            if (klv < n_valid) otile[klv] = (T)e0;
                            if (klv + 1 < n_valid) otile[klv + 1] = (T)e1;
                            if (klv + 2 < n_valid) otile[klv + 2] = (T)e2;
                            if (klv + 3 < n_valid) otile[klv + 3] = (T)e3;
                        }
                    }
                }
            };
            // Partial sums instead of powers, un-scaled.
            //   split-N_t (tp.fixup): the lane-oriented sums (za, zb, wa, wb) of element (ch, i) of thread (q, lane) go to
            //     ((16 ch + i) * 128 + 32 q + lane) of this split's slot of the tile -- the epilogue's own order, every store a
            //     fully coalesced 512-byte warp access; lsp_tensor_fix_kernel adds the slots in split order and finishes;
            //   generalised mode: (xc, xs, c2, s2) per grid frequency, for lsp_gls_combine_kernel.
            const int64_t tile_elems = (int64_t)n_chunks * 16 * 128;
            float4* nat = (sums && tp.fixup) ? sums + (((int64_t)w.split * n_obj_launch + w.obj_local) * gp.n_tiles + w.tile) * tile_elems +
                                                   32 * q + lane : nullptr;
            float4* stile = (sums && !tp.fixup && !tp.gls) ? sums + ((int64_t)w.split * n_obj_launch + w.obj_local) * gp.n_freq + w.K0 : nullptr;
            float2* nat2 = (sums && tp.gls == 1) ? reinterpret_cast<float2*>(sums) + (w.obj_local * gp.n_tiles + w.tile) * tile_elems +
                                                       32 * q + lane : nullptr;
            const float zinv = tp.y_is_w ? ob.winv : ob.zinv;
            auto chunk_sums = [&](int ch) {
                const int m0 = ch * 16;
                float zr[16], zi[16], wr[16], wi[16];
                if (have) {
                    tc_ld16(ta + m0, zr);
                    tc_ld16(ta + NL + m0, zi);
                    if (do_w) {
                        tc_ld16(ta + WCOL + m0, wr);
                        tc_ld16(ta + WCOL + NL + m0, wi);
                    }
                    tc_ld_wait();
                    if (ch == ch1 - 1) {
                        tc_fence_before();
                        arrive_tmem_empty();
                        released = true;
                    }
                }
                if (!have || !do_w) {
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        wr[i] = wi[i] = 0.f;
                        if (!have) zr[i] = zi[i] = 0.f;
                    }
                }
                const int i_lim = min(16, NL - m0);
                const int kl0 = is_im ? (kc - 1 - m0) : (kc + m0);
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const float p0 = __shfl_xor_sync(0xffffffffu, zr[i], 16), p1 = __shfl_xor_sync(0xffffffffu, zi[i], 16);
                    const float q0 = __shfl_xor_sync(0xffffffffu, wr[i], 16), q1 = __shfl_xor_sync(0xffffffffu, wi[i], 16);
                    const float za = (zr[i] - p1) * zinv, zb = (zi[i] + p0) * zinv;
                    const float wa = (wr[i] - q1) * ob.winv, wb = (wi[i] + q0) * ob.winv;
                    if (nat) {
                        nat[(int64_t)(m0 + i) * 128] = make_float4(za, zb, wa, wb);
                    } else if (nat2) {
                        nat2[(int64_t)(m0 + i) * 128] = make_float2(za, zb);
                    } else {
                        const int kl = is_im ? kl0 - i : kl0 + i;
                        if (i < i_lim && kl < n_valid)
                            stile[kl] = make_float4(is_im ? zb : za, is_im ? za : zb, is_im ? wb : wa, is_im ? wa : wb);
                    }
                }
            };
            if (!w.tile_ok) {
                // phantom tile of an odd tile count (pair mode): nothing to store
            } else if (sums && !FUSED) {
                for (int ch = ch0; ch < ch1; ++ch) chunk_sums(ch);
            } else if (ragged) {
                for (int ch = ch0; ch < ch1; ++ch) chunk(ch, std::true_type{});
            } else {
                for (int ch = ch0; ch < ch1; ++ch) chunk(ch, std::false_type{});
            }
            const int bk = (bi < 0) ? 0x7fffffff : (is_im ? kc - 1 - bi : kc + bi);
            if (have) {
                if (!released) {                                  // a warp without chunks (NL <= 16, phantom tile) still signs off
                    tc_fence_before();
                    arrive_tmem_empty();
                }
                ++n_acc;
            }
            if (partials && (!sums || FUSED) && w.tile_ok) {
                Best mine;
                mine.p = (double)bp;
                mine.k = (bk == 0x7fffffff) ? INT64_MAX : w.K0 + (int64_t)bk;
                mine = warp_best(mine);
                if (lane == 0) sbest[ew] = mine;
                named_bar_sync(3, kEpiThreads);
                if (etid < 32) {
                    Best v;
                    v.p = -2.0;
                    v.k = INT64_MAX;
                    if (lane < kEpiWarps) v = sbest[lane];
                    v = warp_best(v);
                    if (lane == 0) partials[w.obj_local * gp.n_tiles + w.tile] = v;
                }
                named_bar_sync(3, kEpiThreads);
            }
        }
    } else if (warp >= 4 + kEpiWarps) {
        // =============================== A-operand generators (steps 2-3) ==========================================
        // a_gj = y_j e^{i alpha_gj}, alpha_gj = 2 pi f(c_g) t_j, g = 8 g1 + g0.  Since f(c_g) = f(c_g0) + g1 (8 L df),
        //     e^{i alpha_gj} = u_{g0 j} v_{g1 j},   u = e^{2 pi i f(c_g0) t_j},   v = e^{2 pi i (8 g1 L df) t_j}.
        // v does not depend on the tile: it arrives with the B stage (aux block).  Phase 1: the 128 threads of a group each
        // evaluate ONE phasor u (g0, j) of the stage (two-float FP32 phase, reduced before the low terms are added) into a
        // small scratch.  Phase 2: thread = A row r = 32 q + l (q = the warp's TMEM lane quadrant): lanes 0-15 the "Re a"
        // rows of groups 16 q + l, lanes 16-31 the "Im a" rows.  With (p, q) = u v' for the 16 observations of the stage,
        //     Re rows (v' = v):              a_Z = y p,             a_W = p^2 - q^2 = cos 2 alpha
        //     Im rows (v' = v e^{-i pi/4}):  a_Z = y (p + q)/sqrt2, a_W = p^2 - q^2 = sin 2 alpha
        // -- the same instruction stream for both halves of the warp (the lane's v row, a 0/1 factor and its y scale are
        // the only differences).  The row's 16 values per plane are split into FP16 hi / lo, packed, and stored with
        // tcgen05.st into the stage's TMEM columns; the MMAs read them from there.
        if (R::kGenRegs > R::kLaunchRegs) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(R::kGenRegs));
        else asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R::kGenRegs));
        const int gw = warp - (4 + kEpiWarps);                    // 0 .. 4 NG - 1
        const int grp = gw >> 2;                                  // generator group: stages with (stage number mod NG) == grp
        const int q = warp & 3;                                   // TMEM lane quadrant (= gw & 3)
        const int gtid = (gw & 3) * 32 + lane;                    // 0..127 inside the group
        // phase 1 role: phasor u of (g0 = gtid & 7, observation j = gtid >> 3)
        const int g0p = gtid & 7, jp = gtid >> 3;
        // phase 2 role
        const bool is_im = lane >= 16;
        const int g = 16 * q + (lane & 15);
        const int g0 = g & 7, g1 = g >> 3;
        const int NL = tp.nl, L = 2 * NL;
        const float2 gam2 = is_im ? make_float2(1.f, 1.f) : make_float2(0.f, 0.f);
        const bool do_w = PAIR ? true : tp.z_only == 0;           // (pair mode runs the standard periodogram only)
        const bool y_is_w = PAIR ? false : tp.y_is_w != 0;
        const unsigned trow = tmem + ((unsigned)(32 * q) << 16) + ACOL;
        const unsigned smem_b_u32 = smem_u32(smem_b);
        const int v_row = is_im ? 8 + g1 : g1;
        const int pos1 = g0p * kTcVRow + 4 * (jp >> 1) + (jp & 1);   // phase 1: where u (g0p, jp) goes (pair-planar)

        // A cursor walks the CTA's stage sequence (items in round-robin order, 16-observation blocks inside an item).
        long long item = first;
        int left = 0;                                             // stages of `item` not yet consumed by this group's cursor
        float f_hi = 0.f, f_lo = 0.f, mean = 0.f, ysc = 0.f, wsc = 0.f;
        auto load_item = [&]() {                                  // `item` is set; returns its number of stages
            const TcItem w = tc_decode(gp, tp, item, offsets, (int)rank);
            const double fd = gp.f_min + ((double)(w.K0 + (int64_t)g0p * L + NL) - 0.5) * gp.df;
            f_hi = (float)fd;
            f_lo = (float)(fd - (double)f_hi);
            const TensorObj ob = objs[w.obj_local];
            mean = y_is_w ? 0.f : (float)ob.mean;
            ysc = (y_is_w ? ob.wscale : ob.yscale) * (1.0f / kTcPhasorScale);
            wsc = ob.wscale * (1.0f / kTcUnitScale);
            return w.kb1 - w.kb0;
        };
        auto seek = [&]() {                                       // first item at or after `item` that has stages
            while (item < total_items && (left = load_item()) <= 0) item += stride;
        };
        auto advance = [&](int n) {                               // move the cursor n stages ahead
            if (left > n) { left -= n; return; }                  // (almost always: the item has more stages)
            while (n > 0 && item < total_items) {
                if (left > n) { left -= n; n = 0; }
                else { n -= left; item += stride; seek(); }
            }
        };
        seek();
        advance(grp);
        // Stage s of the CTA (this group builds s = grp, grp + NG, ...) goes into A slot s % D as that slot's use number s / D.
        // PER_SLOT: use u waits for the slot's u-th "free" arrival (parity (u - 1) & 1); else the group's n-th wait is for the
        // n-th arrival on its own barrier (see the protocol notes at the top of the kernel).
        int sb = grp % SB, sa = grp % D;                          // ring slots of this group's current stage
        unsigned phb = (unsigned)((grp / SB) & 1);
        unsigned it = 0, use = (unsigned)(grp / D), n_wait = 0;   // stages built; use number of slot sa; (per group) arrivals consumed
        while (item < total_items) {
            float* su = &s_u[grp][it & 1][0];
            const unsigned aux = smem_b_u32 + (unsigned)sb * b_bytes + (unsigned)aux_off;     // shared-space address of the aux block
            mbar_wait_backoff(&full_b[sb], phb);                  // the stage's table block (and its aux) has landed
            // this row's tile-independent phasors v' (in the aux block): loaded now, in flight while phase 1 runs
            // (register budget permitting: the long-item shape) -- (c0, c1, s0, s1) of observations 2 h, 2 h + 1
            constexpr bool EARLY_V = R::kGenRegs >= 88;
            const unsigned vp = aux + 4 * (48 + v_row * kTcVRow);
            float4 vq[2][4];
            if (EARLY_V) {
#pragma unroll
                for (int e = 0; e < 4; ++e) vq[0][e] = lds128(vp + 16 * e);
            }
            // ---- phase 1: u (g0p, jp), scaled by 16; threads with g0p = 0 also scale the stage's magnitudes
            {
                const float tv = lds32(aux + 4 * jp);
                const float p = f_hi * tv;
                const float e = fmaf(f_hi, tv, -p);
                const float r = (p - rintf(p)) + fmaf(f_lo, tv, e);
                float sn, cs;
                // two products: the operand is rounded to 11 bits right after, MUFU's 2^-21 is far below that
                if (FAST || PM == 2) sincos_cycles<true>(r, &sn, &cs); else sincos_cycles_reduced(r, &sn, &cs);
                su[pos1] = cs * kTcPhasorScale;
                su[pos1 + 2] = sn * kTcPhasorScale;
                if (g0p == 0) {
                    const float ys = (lds32(aux + (y_is_w ? 128 : 64) + 4 * jp) - mean) * ysc;
                    su[8 * kTcVRow + jp] = ys;                                  // "Re a" rows: y p
                    su[8 * kTcVRow + 16 + jp] = ys * 0.70710678118654752f;      // "Im a" rows: y (p + q) / sqrt 2
                }
            }
            named_bar_sync(4 + grp, R::kGenGroupThreads);
            // ---- phase 2: this row's 16 operand values per plane; the tile's phasors u in two batches of four loads
            const unsigned up = smem_u32(su + g0 * kTcVRow);
            const unsigned yp = smem_u32(su + 8 * kTcVRow + (is_im ? 16 : 0));
            unsigned zh[8], zl[8], wh[8], wl[8];
            float4 y4 = make_float4(0.f, 0.f, 0.f, 0.f), w4 = y4;
#pragma unroll
            for (int hb = 0; hb < 8; hb += 4) {
                float4 uq[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) uq[e] = lds128(up + 16 * (hb + e));
                const float4 y4a = lds128(yp + 16 * (hb >> 1)), y4b = lds128(yp + 16 * (hb >> 1) + 16);
                if (EARLY_V ? hb == 0 : true) {                    // v' of the other batch (EARLY_V) / of this batch
#pragma unroll
                    for (int e = 0; e < 4; ++e) vq[EARLY_V ? 1 : hb >> 2][e] = lds128(vp + 16 * ((EARLY_V ? 4 : hb) + e));
                }
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int h = hb + e;                              // observations 2 h, 2 h + 1
                    const float4 uu = uq[e];
                    const float2 uc = make_float2(uu.x, uu.y), us = make_float2(uu.z, uu.w);
                    const float4 vv = vq[hb >> 2][e];
                    const float2 vc = make_float2(vv.x, vv.y), vs = make_float2(vv.z, vv.w);
                    y4 = (e & 2) ? y4b : y4a;
                    const float2 ys2 = (h & 1) ? make_float2(y4.z, y4.w) : make_float2(y4.x, y4.y);
                    const float2 pp = __ffma2_rn(uc, vc, __fmul2_rn(make_float2(-us.x, -us.y), vs));     // uc vc - us vs
                    const float2 qq = __ffma2_rn(uc, vs, __fmul2_rn(us, vc));                            // uc vs + us vc
                    const float2 az = __fmul2_rn(__ffma2_rn(qq, gam2, pp), ys2);
                    auto pack = [&](const float2 x, unsigned& hi, unsigned& lo) {
                        const __half2 hh = __floats2half2_rn(x.x, x.y);
                        hi = *reinterpret_cast<const unsigned*>(&hh);
                        if (A_LO) {
                            const float2 r = __ffma2_rn(__half22float2(hh), make_float2(-1.f, -1.f), x);     // one packed op
                            const __half2 ll = __floats2half2_rn(r.x, r.y);
                            lo = *reinterpret_cast<const unsigned*>(&ll);
                        }
                    };
                    pack(az, zh[h], zl[h]);
                    if (do_w) {
                        float2 aw = __ffma2_rn(make_float2(-qq.x, -qq.y), qq, __fmul2_rn(pp, pp));       // p^2 - q^2 (x 256)
                        if (WGT) {
                            if ((h & 1) == 0) w4 = lds128(aux + 128 + 16 * (h >> 1));
                            const float2 ww = (h & 1) ? make_float2(w4.z, w4.w) : make_float2(w4.x, w4.y);
                            aw = __fmul2_rn(aw, __fmul2_rn(ww, make_float2(wsc, wsc)));
                        }
                        pack(aw, wh[h], wl[h]);
                    }
                }
            }
            // ---- into the stage's TMEM columns once the MMAs that read its previous contents have completed
            if (use > 0) {                                        // not one of the CTA's first D stages; on the critical path: no sleep
                if (PER_SLOT) mbar_wait(&free_s[sa], (use - 1) & 1);
                else { mbar_wait(&free_s[grp], n_wait & 1); ++n_wait; }
            }
            tc_fence_after();
            const unsigned ta = trow + (unsigned)(sa * A_STAGE_COLS);
            tc_st8(ta, zh);
            if (do_w) tc_st8(ta + 8, wh);
            if (A_LO) {
                tc_st8(ta + 16, zl);
                if (do_w) tc_st8(ta + 24, wl);
            }
            tc_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if (PAIR) mbar_arrive_cluster(full_a_addr0 + 8u * (unsigned)sa); else mbar_arrive(&full_a[sa]);
            }
            // ---- next stage of this group
            advance(NG);
            sb += NG;
            if (sb >= SB) { sb -= SB; phb ^= 1; }                // NG <= SB
            sa += NG;
            while (sa >= D) { sa -= D; ++use; }
            ++it;
            asm volatile("" : "+r"(sb), "+r"(phb), "+r"(sa), "+r"(use), "+r"(it));
        }
    }
    // teardown: everyone is done with TMEM before it is freed
    tc_fence_before();
    if (PAIR) {
        cluster_sync_all();           // the peer has stopped arriving on this CTA's barriers and reading its shared memory
        if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem));
    } else {
        __syncthreads();
        if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem));
    }
}

}  // namespace lsp
