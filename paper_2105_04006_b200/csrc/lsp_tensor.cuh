// lsp_tensor.cuh -- the FP32-mode periodogram contraction on the 5th-generation tensor cores (tcgen05 + TMEM).
//
// The factored formulation (lsp_factored.cuh: theta_kj = alpha_gj +/- beta_mj, a = y e^{i alpha}, b = e^{i beta})
// makes steps 4 of the hot path a dense real contraction over the observations j of one object:
//
//     D_Z[128 x 2NL] = A_Z[128 x N_t] * B_Z[N_t x 2NL]        A_Z rows: Re a_g / Im a_g of 64 frequency groups
//     D_W[128 x 2NL] = A_W[128 x N_t] * B_W[N_t x 2NL]        B_Z cols: Re b_m (m < NL) | Im b_m;  W: doubled angles
//
// D holds, per (group g, offset m), Srr, Sri (row "Re a_g") and Sir, Sii (row "Im a_g"), from which
//     Z(c_g + m + 1/2) = (Srr - Sii) + i (Sri + Sir),   Z(c_g - m - 1/2) = (Srr + Sii) + i (Sir - Sri)
// and the same for W: one 128 x 2NL tile pair covers 64 * 2NL <= 16384 grid frequencies of one object, and the four
// real sums of Eq. 2's closed form (lsp_common.cuh) for every one of them.  This is a GEMM, so it runs as one:
// tcgen05.mma kind::f16 (M = 128, N = 2NL <= 256, K = 16), FP32 accumulators in TMEM (Z in columns [0,256),
// W in [256,512): the whole 256 KB), operands in shared memory in the no-swizzle K-major core-matrix layout.
//
// Precision: operands are FP16 pairs x = x_hi + x_lo (22 significand bits, the same class as
// FP32's 24) and the product is a_hi b_hi + a_hi b_lo + a_lo b_hi (three MMAs; a_lo b_lo < 2^-24 is dropped), with y
// pre-scaled by a power of two per object so FP16 never overflows or loses the low part.  fast_math = 1 keeps only
// a_hi b_hi (one MMA, ~2^-11 per operand) and evaluates sincos with MUFU: the "fast vs accurate" comparison of
// PAPER.md:L423-433 carried over to this formulation.  Phases are formed in FP64 and range-reduced before any FP32
// trigonometry, as everywhere in the library.
//
// Data flow per CTA (persistent, one per SM, static round-robin over (object, tile, split) work items):
//   B operands  e^{i beta}, e^{2 i beta} depend on (object, observation, m) only -- not on the tile -- so a pre-pass
//               (lsp_tensor_table_kernel) writes them once per object into a table already laid out as shared-memory
//               stages; warp 0 streams the stages in with 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx).
//   A operands  depend on the tile: warps 12-19 generate them straight into the stage ring (st.shared +
//               fence.proxy.async): one sincos per thread per stage (two-float FP32 phase), then the 64 x 16 operands as
//               phasor products e^{i alpha_g} = u_{g mod 8} v_{g div 8} on the FMA pipe, scaled by y, split into FP16 hi/lo.
//   warp 1      one thread issues the MMAs of a stage when its mbarrier completes, and tcgen05.commit releases the
//               stage / publishes the finished accumulators.
//   warps 4-11  epilogue: tcgen05.ld the accumulators, combine rows with a shuffle, closed-form power (step 5),
//               vector stores of the periodogram (step 6) or the fused argmax partial (step 6').
#pragma once
#include <cuda_fp16.h>

#include <type_traits>

#include "lsp_factored_ws.cuh"

namespace lsp {

constexpr int kTcGroups = 64;                  // frequency groups per tile (128 MMA rows)
constexpr int kTcKB = 16;                      // observations per MMA / ring stage (kind::f16: K = 16)
constexpr int kTcMaxNL = 128;                  // N = 2 NL <= 256
// Generator scratch (floats): three planes (cos, sin, -sin) of [observation quad j/4][phasor q][j%4]; a quad row is 16 x 4
// floats + 16 floats of padding so that the two quads a quarter-warp reads fall into different banks (conflict-free LDS.128).
constexpr int kTcScratchQuad = 16 * 4 + 16;
constexpr int kTcScratchPlane = 4 * kTcScratchQuad;
constexpr int kTcGenGroupThreads = 256;                               // threads that build one ring stage
// Warp roles of one CTA: 4 control warps, EW epilogue warps, NG generator groups of 8 warps.  Two shapes are built:
//   (EW, NG) = (8, 2): 896 threads -- short items (batches of short light curves): the per-item epilogue is on the critical path
//   (EW, NG) = (4, 3): 1024 threads -- long items (hundreds of stages): the generators are, the epilogue is rare
// Registers are re-split with setmaxnreg (per 4-warp group): control 40, generators 56, epilogue what is left
// (120 resp. 136): 128 x 40 + 256 x 120 + 512 x 56 = 64512 = 896 x 72;  128 x 40 + 128 x 136 + 768 x 56 = 65536 = 1024 x 64.
template <int EW, int NG> struct TcRoles {
    static constexpr int kThreads = (4 + EW + 8 * NG) * 32;
    static constexpr int kEpiThreads = EW * 32;
    static constexpr int kLaunchRegs = (65536 / kThreads) / 8 * 8;
    static constexpr int kCtrlRegs = 40, kGenRegs = 56;
    static constexpr int kEpiRegs = ((kLaunchRegs * kThreads - 128 * kCtrlRegs - 8 * NG * 32 * kGenRegs) / kEpiThreads) / 8 * 8;
    static_assert(EW % 4 == 0 && kThreads <= 1024 && kEpiRegs >= 96 && kEpiRegs <= 255, "role split");
};
// static shared memory of the kernel (generator scratch etc.) + alignment slack, for the host's ring sizing
template <int NG> constexpr int tc_static_smem() { return NG * 2 * (3 * kTcScratchPlane + kTcKB) * 4 + 1024; }
constexpr float kTcUnitScale = 256.0f;         // scale of the unit-modulus A_W operands (keeps the FP16 low part normal)

struct TensorParams {
    int nl;             // NL: half-width of a frequency group (multiple of 8, <= 128); group width L = 2 NL = MMA N
    int tile;           // frequencies per tile = 64 * 2 NL
    int n_ops;          // FP16 operand planes per stage side: 4 (accurate: hi and lo of Z- and W-operands) or 2 (fast)
    int stages;         // A-operand ring depth (generators -> MMA)
    int stages_b;       // B-operand ring depth (TMA -> MMA): shallower, the copies are fast and B stages are twice as large
    int long_items;     // 1: many stages per item -> the (4 epilogue warps, 3 generator groups) shape; 0: (8, 2)
    int b_stage_bytes;  // n_ops * 2 NL * 32
    int a_stage_bytes;  // n_ops * 128 * 32
};

// Per-object pre-pass results of the tensor path.
struct TensorObj {
    double  mean;       // subtracted from y (0 unless center = 1)
    float   yscale;     // power of two: max |y - mean| * yscale in [256, 512)
    float   pscale;     // output scale: (normalize ? 2 / sum (y-mean)^2 : 1) * 256 / yscale^2
    float   zinv;       // 1 / yscale (split-N_t path: sums are written un-scaled)
    int     pad;
    int64_t kb_off;     // first table block of this object
};

__host__ __device__ inline int tc_n_kb(int64_t n_t) { return (int)((n_t + kTcKB - 1) / kTcKB); }

// ---- pre-pass 1: per-object statistics (one CTA per object) -----------------------------------------------------
template <typename T>
__global__ void lsp_tensor_stats_kernel(const int64_t* __restrict__ offsets, const T* __restrict__ y, TensorObj* __restrict__ objs,
                                        int obj_base, int center, int normalize)
{
    __shared__ double red[3][32];
    const int64_t obj = (int64_t)blockIdx.x + obj_base;
    const int64_t lo = offsets[obj], n = offsets[obj + 1] - lo;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    double s = 0.0;
    if (center) {
        for (int64_t j = threadIdx.x; j < n; j += blockDim.x) s += (double)y[lo + j];
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (lane == 0) red[0][wid] = s;
        __syncthreads();
        s = 0.0;
        for (int w = 0; w < nw; ++w) s += red[0][w];
        __syncthreads();
    }
    const double mean = (center && n > 0) ? s / (double)n : 0.0;
    double q = 0.0, mx = 0.0;
    for (int64_t j = threadIdx.x; j < n; j += blockDim.x) {
        const double v = (double)y[lo + j] - mean;
        q += v * v;
        mx = fmax(mx, fabs(v));
    }
    for (int d = 16; d > 0; d >>= 1) {
        q += __shfl_xor_sync(0xffffffffu, q, d);
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
    }
    if (lane == 0) { red[1][wid] = q; red[2][wid] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        q = 0.0; mx = 0.0;
        for (int w = 0; w < nw; ++w) { q += red[1][w]; mx = fmax(mx, red[2][w]); }
        TensorObj* o = &objs[blockIdx.x];     // kb_off is written by the scan kernel
        o->mean = mean;
        int e = 0;
        if (mx > 0.0 && isfinite(mx)) frexp(mx, &e);          // mx = f * 2^e, f in [0.5, 1)  ->  mx * 2^(9-e) in [256, 512)
        e = max(-100, min(100, 9 - e));
        const double ys = (mx > 0.0 && isfinite(mx)) ? ldexp(1.0, e) : 1.0;
        o->yscale = (float)ys;
        o->zinv = (float)(1.0 / ys);
        const double nrm = normalize ? (q > 0.0 ? 2.0 / q : 0.0) : 1.0;
        o->pscale = (float)(nrm * (double)kTcUnitScale / (ys * ys));
        o->pad = 0;
    }
}

// ---- pre-pass 2: exclusive scan of ceil(N_t / 16) over the launch's objects (single CTA) -----------------------
__global__ void lsp_tensor_scan_kernel(const int64_t* __restrict__ offsets, TensorObj* __restrict__ objs, int obj_base, int n_obj)
{
    __shared__ int64_t wsum[32];
    const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, wid = tid >> 5;
    const int per = (n_obj + nt - 1) / nt;
    const int o0 = min(n_obj, tid * per), o1 = min(n_obj, o0 + per);
    int64_t s = 0;
    for (int o = o0; o < o1; ++o) s += tc_n_kb(offsets[obj_base + o + 1] - offsets[obj_base + o]);
    // block-wide exclusive scan of the per-thread totals: warp shuffles, then the warp totals
    int64_t inc = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int64_t v = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += v;
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int64_t w = (lane < (nt >> 5)) ? wsum[lane] : 0, winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int64_t v = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += v;
        }
        wsum[lane] = winc - w;                     // exclusive offset of each warp
        if (lane == 31) objs[n_obj].kb_off = winc; // total number of table blocks
    }
    __syncthreads();
    int64_t run = wsum[wid] + inc - s;              // exclusive prefix of this thread's first object
    for (int o = o0; o < o1; ++o) {
        objs[o].kb_off = run;
        run += tc_n_kb(offsets[obj_base + o + 1] - offsets[obj_base + o]);
    }
}

__device__ __forceinline__ void split_half2(float x0, float x1, __half2* hi, __half2* lo)
{
    const __half2 h = __floats2half2_rn(x0, x1);
    const float2 b = __half22float2(h);
    *hi = h;
    *lo = __floats2half2_rn(x0 - b.x, x1 - b.y);
}

// ---- pre-pass 3: the B-operand table ---------------------------------------------------------------------------------
// One CTA per (object, 16-observation block); thread m < NL owns offset m.  Block layout (FP16), identical to one
// shared-memory B stage:  [plane: b_hi, b2_hi, (b_lo, b2_lo)] [k chunk c = 0,1] [column group n/8] [n%8] [k%8]
// with column n = m (Re) or NL + m (Im) and observation 16 kb + 8 c + k%8.  Observations past N_t are zero.
template <typename T, bool FAST>
__global__ void __launch_bounds__(kTcMaxNL)
lsp_tensor_table_kernel(GridParams gp, TensorParams tp, const int64_t* __restrict__ offsets, const T* __restrict__ t,
                        const TensorObj* __restrict__ objs, int n_obj, __half* __restrict__ table)
{
    // locate the object of this block: binary search on kb_off (exclusive scan, non-decreasing)
    const int64_t blk = blockIdx.x;
    if (blk >= objs[n_obj].kb_off) return;     // the grid is an upper bound
    int lo_o = 0, hi_o = n_obj - 1;
    while (lo_o < hi_o) {
        const int mid = (lo_o + hi_o + 1) >> 1;
        if (objs[mid].kb_off <= blk) lo_o = mid; else hi_o = mid - 1;
    }
    // objects with zero blocks share kb_off with their successor: the search lands on the last of them, which is the one
    // that owns the block as long as it has blocks; step forward is never needed because equal offsets mean empty objects.
    const int o = lo_o;
    const int64_t obj = (int64_t)o + gp.obj_base;
    const int64_t base = offsets[obj], n_t = offsets[obj + 1] - base;
    const int kb = (int)(blk - objs[o].kb_off);
    const int m = threadIdx.x;
    if (m >= tp.nl) return;
    const double f_beta = ((double)m + 0.5) * gp.df;
    const int n_cols = 2 * tp.nl;
    const int plane = n_cols * kTcKB;                           // halfs per plane
    __half* dst = table + (size_t)blk * (size_t)(tp.n_ops * plane);
    float c1[kTcKB], s1[kTcKB];
#pragma unroll
    for (int k = 0; k < kTcKB; ++k) {
        const int64_t j = (int64_t)kb * kTcKB + k;
        float sn = 0.f, cs = 0.f;
        if (j < n_t) {
            const float r = (float)frac_cycles(f_beta * (double)t[base + j]);
            sincos_cycles<FAST>(r, &sn, &cs);
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
        const size_t off_im = (size_t)c * (n_cols * 8) + (size_t)(tp.nl + m) * 8;
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
__device__ __forceinline__ void tc_mma_f16(unsigned d_tmem, uint64_t a_desc, uint64_t b_desc, unsigned idesc, unsigned accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tc_commit(unsigned long long* bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// mbarrier wait for roles whose waits are long when they are not the bottleneck (generators on a full ring, epilogue on
// unfinished accumulators): back off between polls so the spinning warps do not take issue slots from the working ones.
__device__ __forceinline__ void mbar_wait_backoff(unsigned long long* bar, unsigned parity)
{
    unsigned done;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    while (!done) {
        __nanosleep(40);
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
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void* smem_dst, const void* gmem_src, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

struct TcItem {
    int64_t obj_local, obj, lo, n_t, K0;
    int tile, split, kb0, kb1;
};
__device__ __forceinline__ TcItem tc_decode(const GridParams& gp, const TensorParams& tp, long long item,
                                            const int64_t* __restrict__ offsets)
{
    TcItem w;
    w.split = (int)(item % gp.n_split);
    const long long r = item / gp.n_split;
    w.tile = (int)(r % gp.n_tiles);
    w.obj_local = r / gp.n_tiles;
    w.obj = w.obj_local + gp.obj_base;
    w.lo = offsets[w.obj];
    w.n_t = offsets[w.obj + 1] - w.lo;
    const int nkb = tc_n_kb(w.n_t);
    w.kb0 = (int)(((long long)nkb * w.split) / gp.n_split);
    w.kb1 = (int)(((long long)nkb * (w.split + 1)) / gp.n_split);
    w.K0 = (int64_t)w.tile * tp.tile;
    return w;
}

constexpr size_t tc_smem_bytes(int stages_a, int stages_b, int a_stage, int b_stage)
{
    return 1024 /* alignment slack */ + (size_t)stages_a * (size_t)a_stage + (size_t)stages_b * (size_t)b_stage + 512;
}

template <typename T, bool FAST, int EW, int NG>
__global__ void __launch_bounds__((TcRoles<EW, NG>::kThreads), 1)
lsp_tensor_kernel(GridParams gp, TensorParams tp, const int64_t* __restrict__ offsets, const T* __restrict__ t,
                  const T* __restrict__ y, const TensorObj* __restrict__ objs, const __half* __restrict__ table,
                  T* __restrict__ out_power, Best* __restrict__ partials, float4* __restrict__ sums,
                  int64_t n_obj_launch, long long total_items)
{
    using R = TcRoles<EW, NG>;
    constexpr int kTcEpiWarps = EW, kTcEpiThreads = R::kEpiThreads;
    constexpr int NOPS = FAST ? 2 : 4;
    constexpr int A_PLANE = 128 * kTcKB * 2;                  // bytes of one A plane: 128 rows x 16 x FP16
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
    // Two rings: A stages (16 KB, written by the generators) and B stages (up to 32 KB, filled by TMA).  The A ring is the
    // deep one: while the epilogue of a short item holds TMEM, the generators keep building the next item's stages.
    const int S = tp.stages, SB = tp.stages_b;
    const int stage_bytes = tp.a_stage_bytes;                 // A ring stride
    const int b_plane = 2 * tp.nl * kTcKB * 2;                // bytes of one B plane
    unsigned char* smem_b = smem + (size_t)S * tp.a_stage_bytes;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(smem_b + (size_t)SB * tp.b_stage_bytes);   // A ring
    unsigned long long* empty = full + 8;
    unsigned long long* full_b = empty + 8;                   // B ring
    unsigned long long* empty_b = full_b + 8;
    unsigned long long* tmem_full = empty_b + 8;
    unsigned long long* tmem_empty = tmem_full + 1;
    __shared__ unsigned tmem_base_s;
    __shared__ Best sbest[kTcEpiWarps];
    __shared__ __align__(16) float s_uv[NG][2][3 * kTcScratchPlane]; // generator scratch: [group][buffer][plane][j/4][phasor q][j%4]
    __shared__ __align__(16) float s_yv[NG][2][kTcKB];               // scaled, centred y of the stage

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);      // broadcast: the compiler may treat the role as warp-uniform
    if (tid == 0) {
        for (int s = 0; s < S; ++s) {
            mbar_init(&full[s], kTcGenGroupThreads);
            mbar_init(&empty[s], 1);
        }
        for (int s = 0; s < SB; ++s) {
            mbar_init(&full_b[s], 1);
            mbar_init(&empty_b[s], 1);
        }
        mbar_init(tmem_full, 1);
        mbar_init(tmem_empty, kTcEpiThreads);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&tmem_base_s)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem = tmem_base_s;

    if (warp < 4) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R::kCtrlRegs));
    if (warp == 0) {
        // =============================== TMA producer: B stages from the per-object table ========================
        if (lane == 0) {
            int st = 0;
            unsigned ph = 1;                                      // parity of the "empty" phase to wait for
            const unsigned b_bytes = (unsigned)tp.b_stage_bytes;
            for (long long item = blockIdx.x; item < total_items; item += gridDim.x) {
                const TcItem w = tc_decode(gp, tp, item, offsets);
                const unsigned char* src = reinterpret_cast<const unsigned char*>(table) +
                                           (size_t)(objs[w.obj_local].kb_off + w.kb0) * (size_t)b_bytes;
                for (int kb = w.kb0; kb < w.kb1; ++kb) {
                    mbar_wait(&empty_b[st], ph);
                    mbar_arrive_expect_tx(&full_b[st], b_bytes);
                    tma_bulk_g2s(smem_b + (size_t)st * b_bytes, src, b_bytes, &full_b[st]);
                    src += b_bytes;
                    if (++st == SB) { st = 0; ph ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // =============================== MMA issuer ===============================================================
        // The whole warp runs the loop with warp-uniform values (item ranges are broadcast from lane 0), so descriptors
        // and barrier addresses live in uniform registers; one elected lane issues the MMAs and commits.
        {
            const unsigned idesc = (1u << 4) | ((unsigned)((2 * tp.nl) >> 3) << 17) | ((unsigned)(128 >> 4) << 24);
            const unsigned a_lbo = 16 * 128, b_lbo = (unsigned)(2 * tp.nl / 8) * 128, sbo = 128;
            // Descriptors of stage 0; stage s adds s * stage_bytes / 16 to the 14-bit start-address field (the whole ring
            // lies below 256 KB, so the field never carries into the LBO bits).
            const unsigned sa0 = smem_u32(smem), sb0 = smem_u32(smem_b);
            const uint64_t a_zh0 = tc_smem_desc(sa0, a_lbo, sbo), a_wh0 = tc_smem_desc(sa0 + A_PLANE, a_lbo, sbo);
            const uint64_t a_zl0 = tc_smem_desc(sa0 + 2 * A_PLANE, a_lbo, sbo), a_wl0 = tc_smem_desc(sa0 + 3 * A_PLANE, a_lbo, sbo);
            const uint64_t b_zh0 = tc_smem_desc(sb0, b_lbo, sbo), b_wh0 = tc_smem_desc(sb0 + b_plane, b_lbo, sbo);
            const uint64_t b_zl0 = tc_smem_desc(sb0 + 2 * b_plane, b_lbo, sbo), b_wl0 = tc_smem_desc(sb0 + 3 * b_plane, b_lbo, sbo);
            const uint64_t stage_inc = (uint64_t)(tp.a_stage_bytes >> 4), stage_inc_b = (uint64_t)(tp.b_stage_bytes >> 4);
            int st = 0, stb = 0;
            unsigned ph = 0, phb = 0, n_acc = 0;
            uint64_t so = 0, sob = 0;                             // st * stage_inc, stb * stage_inc_b
            for (long long item = blockIdx.x; item < total_items; item += gridDim.x) {
                const TcItem w = tc_decode(gp, tp, item, offsets);
                const int kb0 = __shfl_sync(0xffffffffu, w.kb0, 0), kb1 = __shfl_sync(0xffffffffu, w.kb1, 0);
                if (kb1 <= kb0) continue;
                mbar_wait(tmem_empty, (n_acc & 1) ^ 1);          // the epilogue has drained the previous accumulators
                tc_fence_after();
                unsigned acc = 0;
                for (int kb = kb0; kb < kb1; ++kb) {
                    mbar_wait(&full_b[stb], phb);
                    mbar_wait(&full[st], ph);
                    tc_fence_after();
                    if (elect_one()) {
                        // planes: 0 = Z-operand hi, 1 = W-operand hi, 2 = Z lo, 3 = W lo
                        if (!FAST) {
                            tc_mma_f16(tmem, a_zl0 + so, b_zh0 + sob, idesc, acc);
                            tc_mma_f16(tmem, a_zh0 + so, b_zl0 + sob, idesc, 1u);
                            tc_mma_f16(tmem, a_zh0 + so, b_zh0 + sob, idesc, 1u);
                            tc_mma_f16(tmem + 256, a_wl0 + so, b_wh0 + sob, idesc, acc);
                            tc_mma_f16(tmem + 256, a_wh0 + so, b_wl0 + sob, idesc, 1u);
                            tc_mma_f16(tmem + 256, a_wh0 + so, b_wh0 + sob, idesc, 1u);
                        } else {
                            tc_mma_f16(tmem, a_zh0 + so, b_zh0 + sob, idesc, acc);
                            tc_mma_f16(tmem + 256, a_wh0 + so, b_wh0 + sob, idesc, acc);
                        }
                        tc_commit(&empty[st]);                   // both stages are free once these MMAs have read them
                        tc_commit(&empty_b[stb]);
                    }
                    __syncwarp();
                    acc = 1u;
                    so += stage_inc;
                    sob += stage_inc_b;
                    if (++st == S) { st = 0; ph ^= 1; so = 0; }
                    if (++stb == SB) { stb = 0; phb ^= 1; sob = 0; }
                }
                if (elect_one()) tc_commit(tmem_full);           // accumulators complete
                __syncwarp();
                ++n_acc;
            }
        }
    } else if (warp >= 4 && warp < 4 + kTcEpiWarps) {
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
        unsigned n_acc = 0;
        for (long long item = blockIdx.x; item < total_items; item += gridDim.x) {
            const TcItem w = tc_decode(gp, tp, item, offsets);
            const TensorObj ob = objs[w.obj_local];
            const bool have = w.kb1 > w.kb0;
            if (have) {
                mbar_wait_backoff(tmem_full, n_acc & 1);
                tc_fence_after();
            }
            float bp = -1.0f;                                     // running maximum (P >= 0; NaN never compares greater)
            int bi = -1;                                          // its position m = 16 ch + i in this lane's sequence
            const float n_hat = kTcUnitScale * (float)w.n_t;
            const float nn = n_hat * n_hat, nn_eps = 2e-6f * nn;
            const int n_valid = (int)min((int64_t)tp.tile, (int64_t)gp.n_freq - w.K0);     // frequencies of this tile on the grid
            const bool ragged = n_valid < tp.tile;
            T* otile = out_power ? out_power + w.obj_local * (int64_t)gp.n_freq + w.K0 : nullptr;
            float4* stile = sums ? sums + ((int64_t)w.split * n_obj_launch + w.obj_local) * gp.n_freq + w.K0 : nullptr;
            const unsigned ta = tmem + ((unsigned)(32 * q) << 16);
            bool released = false;
            // one chunk = 16 accumulator columns of each of the four TMEM regions; RAG = the tile overhangs the grid
            auto chunk = [&](int ch, auto rag_tag) {
                constexpr bool RAG = decltype(rag_tag)::value;
                const int m0 = ch * 16;
                float zr[16], zi[16], wr[16], wi[16];
                if (have) {
                    tc_ld16(ta + m0, zr);
                    tc_ld16(ta + NL + m0, zi);
                    tc_ld16(ta + 256 + m0, wr);
                    tc_ld16(ta + 256 + NL + m0, wi);
                    tc_ld_wait();
                    if (ch == ch1 - 1) {                          // last TMEM read of this warp: the MMA warp may overwrite
                        tc_fence_before();
                        mbar_arrive(tmem_empty);
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
                        const float A = __fmul_rn(za[e], za[e]), B = __fmul_rn(zb[e], zb[e]);
                        const float den = nn - fmaf(wa[e], wa[e], __fmul_rn(wb[e], wb[e]));
                        const float num = fmaf(-2.0f * ss, __fmul_rn(za[e], zb[e]), fmaf(-cc, A - B, __fmul_rn(n_hat, A + B)));
                        bad = bad || !(den > nn_eps);
                        pw[e] = __fdividef(num, den) * ob.pscale;
                    }
                    if (bad) {                                    // vanishing denominator (reading a6): the full epilogue, rarely
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            pw[e] = power_from_sums<float>(is_im ? zb[e] : za[e], is_im ? za[e] : zb[e], is_im ? wb[e] : wa[e],
                                                           is_im ? wa[e] : wb[e], n_hat, ob.pscale);
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
            // split-N_t: un-scaled partial sums (xc, xs, c2, s2) per frequency for lsp_combine_kernel
            auto chunk_sums = [&](int ch) {
                const int m0 = ch * 16;
                float zr[16], zi[16], wr[16], wi[16];
                if (have) {
                    tc_ld16(ta + m0, zr);
                    tc_ld16(ta + NL + m0, zi);
                    tc_ld16(ta + 256 + m0, wr);
                    tc_ld16(ta + 256 + NL + m0, wi);
                    tc_ld_wait();
                    if (ch == ch1 - 1) {
                        tc_fence_before();
                        mbar_arrive(tmem_empty);
                        released = true;
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < 16; ++i) zr[i] = zi[i] = wr[i] = wi[i] = 0.f;
                }
                const int i_lim = min(16, NL - m0);
                const int kl0 = is_im ? (kc - 1 - m0) : (kc + m0);
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const float p0 = __shfl_xor_sync(0xffffffffu, zr[i], 16), p1 = __shfl_xor_sync(0xffffffffu, zi[i], 16);
                    const float q0 = __shfl_xor_sync(0xffffffffu, wr[i], 16), q1 = __shfl_xor_sync(0xffffffffu, wi[i], 16);
                    const float za = zr[i] - p1, zb = zi[i] + p0, wa = wr[i] - q1, wb = wi[i] + q0;
                    const float xc = is_im ? zb : za, xs = is_im ? za : zb;
                    const float c2 = is_im ? wb : wa, s2 = is_im ? wa : wb;
                    const int kl = is_im ? kl0 - i : kl0 + i;
                    if (i < i_lim && kl < n_valid)
                        stile[kl] = make_float4(xc * ob.zinv, xs * ob.zinv, c2 * (1.0f / kTcUnitScale), s2 * (1.0f / kTcUnitScale));
                }
            };
            if (stile) {
                for (int ch = ch0; ch < ch1; ++ch) chunk_sums(ch);
            } else if (ragged) {
                for (int ch = ch0; ch < ch1; ++ch) chunk(ch, std::true_type{});
            } else {
                for (int ch = ch0; ch < ch1; ++ch) chunk(ch, std::false_type{});
            }
            const int bk = (bi < 0) ? 0x7fffffff : (is_im ? kc - 1 - bi : kc + bi);
            if (have) {
                if (!released) {                                  // a warp without chunks (NL <= 16) still signs off
                    tc_fence_before();
                    mbar_arrive(tmem_empty);
                }
                ++n_acc;
            }
            if (partials && !stile) {
                Best mine;
                mine.p = (double)bp;
                mine.k = (bk == 0x7fffffff) ? INT64_MAX : w.K0 + (int64_t)bk;
                mine = warp_best(mine);
                if (lane == 0) sbest[ew] = mine;
                named_bar_sync(3, kTcEpiThreads);
                if (etid < 32) {
                    Best v;
                    v.p = -2.0;
                    v.k = INT64_MAX;
                    if (lane < kTcEpiWarps) v = sbest[lane];
                    v = warp_best(v);
                    if (lane == 0) partials[w.obj_local * gp.n_tiles + w.tile] = v;
                }
                named_bar_sync(3, kTcEpiThreads);
            }
        }
    } else if (warp >= 4 + kTcEpiWarps) {
        // =============================== A-operand generators (steps 2-3) ==========================================
        // a_gj = y_j e^{i alpha_gj}, alpha_gj = 2 pi f(c_g) t_j, g = 8 g1 + g0.  Since f(c_g) = f(c_g0) + g1 (8 L df),
        //     e^{i alpha_gj} = u_{g0 j} v_{g1 j},   u = e^{2 pi i f(c_g0) t_j},   v = e^{2 pi i (8 g1 L df) t_j}
        // so a stage (16 observations) needs 16 x 16 sincos -- ONE per thread of a generator group (phase 1, into a
        // small shared-memory scratch) -- instead of 64 x 16; phase 2 forms the 64 x 16 products on the FMA pipe, splits
        // them into FP16 hi/lo and writes the UMMA operand planes.  Phases are FP32 two-float products (f = f_hi + f_lo,
        // exact f_hi t through fma, reduced to (-1/2, 1/2] cycles before the low terms are added): no FP64 in the loop.
        // Two groups of 8 warps take alternate ring stages, so one group's latencies (sincos chain, group barrier,
        // LDS, mbarrier wait, proxy fence) are covered by the other group's instructions on the same schedulers.
        // t / y of a group's NEXT stage (of this or a later work item) are loaded before its current stage is processed.
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R::kGenRegs));
        const int gw = warp - (4 + kTcEpiWarps);                  // 0 .. 8 NG - 1
        const int grp = gw >> 3;                                  // generator group: stages with (stage number mod NG) == grp
        const int gw8 = gw & 7;
        const int gtid = (tid - (4 + kTcEpiWarps) * 32) & (kTcGenGroupThreads - 1);      // 0..255 inside the group
        // phase 1 role: phasor q (0-7: u_g0, 8-15: v_g1) of observation j1 of the stage
        const int q1 = gtid >> 4, j1 = gtid & 15;
        const int sc_w = (j1 >> 2) * kTcScratchQuad + q1 * 4 + (j1 & 3);
        // phase 2 role: 16-group row block qb, k chunk c, group g, observations 4 hsel .. 4 hsel + 3 of the chunk
        const int qb = gw8 & 3, c = gw8 >> 2;
        const int g = 16 * qb + (lane >> 1);
        const int hsel = lane & 1;
        const int row_re = 32 * qb + (lane >> 1), row_im = row_re + 16;
        const int off_re = c * (16 * 128) + (row_re >> 3) * 128 + (row_re & 7) * 16 + hsel * 8;
        const int off_im = c * (16 * 128) + (row_im >> 3) * 128 + (row_im & 7) * 16 + hsel * 8;
        const int sc_u = (2 * c + hsel) * kTcScratchQuad + (g & 7) * 4;
        const int sc_v = (2 * c + hsel) * kTcScratchQuad + (8 + (g >> 3)) * 4;
        const int NL = tp.nl, L = 2 * NL;
        const double fv = (q1 >= 8) ? (double)(8 * (q1 - 8)) * (double)L * gp.df : 0.0;      // v: the same for every item

        // A cursor walks the CTA's stage sequence (items in round-robin order, 16-observation blocks inside an item).
        struct Cursor {
            long long item;
            int64_t lo;           // first observation of the object
            int n_t, kb, kb1;
            float f_hi, f_lo, mean, yscale;
        };
        auto load_item = [&](Cursor& cu) {        // cu.item is set; fills the rest; returns false if the item has no stages
            const TcItem w = tc_decode(gp, tp, cu.item, offsets);
            cu.lo = w.lo;
            cu.n_t = (int)w.n_t;
            cu.kb = w.kb0;
            cu.kb1 = w.kb1;
            const double fd = (q1 < 8) ? gp.f_min + ((double)(w.K0 + (int64_t)q1 * L + NL) - 0.5) * gp.df : fv;
            cu.f_hi = (float)fd;
            cu.f_lo = (float)(fd - (double)cu.f_hi);
            cu.mean = (float)objs[w.obj_local].mean;
            cu.yscale = objs[w.obj_local].yscale;
            return w.kb1 > w.kb0;
        };
        auto seek = [&](Cursor& cu) {             // first item at or after cu.item that has stages
            while (cu.item < total_items && !load_item(cu)) cu.item += gridDim.x;
        };
        auto step = [&](Cursor& cu) {
            if (++cu.kb >= cu.kb1) {
                cu.item += gridDim.x;
                seek(cu);
            }
        };
        // cur = the group's stage being built (its t, y already in registers); its successor's (t, y) are loaded before
        // the current stage is processed.
        Cursor p1;
        p1.item = blockIdx.x;
        seek(p1);
        for (int i = 0; i < grp; ++i)
            if (p1.item < total_items) step(p1);
        int st = grp;                                             // ring slot of the stage phase 2 writes
        unsigned eph = 1;                                         // parity of the "empty" phase to wait for
        while (st >= S) { st -= S; eph ^= 1; }
        unsigned it = 0;
        float* s_uvg = &s_uv[grp][0][0];
        float* s_yvg = &s_yv[grp][0][0];
        auto fetch = [&](const Cursor& cu, float& tv, float& yv_) {
            tv = 0.f;
            yv_ = 0.f;
            if (cu.item < total_items) {
                const int j = cu.kb * kTcKB + j1;
                if (j < cu.n_t) { tv = (float)t[cu.lo + j]; yv_ = (float)y[cu.lo + j]; }
            }
        };
        auto phase1 = [&](const Cursor& cu, float tv, float yv_, int buf) {
            float* suv = s_uvg + buf * (3 * kTcScratchPlane);
            const bool live = (cu.kb * kTcKB + j1) < cu.n_t;
            const float p = cu.f_hi * tv;
            const float e = fmaf(cu.f_hi, tv, -p);
            const float r = (p - rintf(p)) + fmaf(cu.f_lo, tv, e);
            float sn, cs;
            if (FAST) sincos_cycles<true>(r, &sn, &cs); else sincos_cycles_reduced(r, &sn, &cs);
            cs = live ? cs : 0.f;
            sn = live ? sn : 0.f;
            suv[sc_w] = cs;
            suv[kTcScratchPlane + sc_w] = sn;
            if (q1 < 8) suv[2 * kTcScratchPlane + sc_w] = -sn;
            if (q1 == 0) s_yvg[buf * kTcKB + j1] = live ? (yv_ - cu.mean) * cu.yscale : 0.f;
        };
        float t_p1, y_p1;
        fetch(p1, t_p1, y_p1);
        while (p1.item < total_items) {
            const int buf = it & 1;
            const float* suv = s_uvg + buf * (3 * kTcScratchPlane);
            const float* syv = s_yvg + buf * kTcKB;
            // ---- phase 1 of this stage, then the loads of the group's next stage (two ring stages ahead)
            phase1(p1, t_p1, y_p1, buf);
#pragma unroll
            for (int i = 0; i < NG; ++i)
                if (p1.item < total_items) step(p1);
            float t_pf, y_pf;
            fetch(p1, t_pf, y_pf);
            named_bar_sync(4 + grp, kTcGenGroupThreads);
            const float4 ucv = *reinterpret_cast<const float4*>(&suv[sc_u]);
            const float4 usv = *reinterpret_cast<const float4*>(&suv[kTcScratchPlane + sc_u]);
            const float4 unv = *reinterpret_cast<const float4*>(&suv[2 * kTcScratchPlane + sc_u]);
            const float4 vcv = *reinterpret_cast<const float4*>(&suv[sc_v]);
            const float4 vsv = *reinterpret_cast<const float4*>(&suv[kTcScratchPlane + sc_v]);
            const float4 yv = *reinterpret_cast<const float4*>(&syv[8 * c + 4 * hsel]);
            // ---- phase 2: products (packed FP32x2), FP16 split, operand stores
            float2 ar[2], ai[2], a2r[2], a2i[2];
            {
                const float2 k256 = make_float2(kTcUnitScale, kTcUnitScale), km256 = make_float2(-kTcUnitScale, -kTcUnitScale);
                const float2 k512 = make_float2(2.f * kTcUnitScale, 2.f * kTcUnitScale);
                const float2 uc[2] = {make_float2(ucv.x, ucv.y), make_float2(ucv.z, ucv.w)};
                const float2 us[2] = {make_float2(usv.x, usv.y), make_float2(usv.z, usv.w)};
                const float2 un[2] = {make_float2(unv.x, unv.y), make_float2(unv.z, unv.w)};
                const float2 vc[2] = {make_float2(vcv.x, vcv.y), make_float2(vcv.z, vcv.w)};
                const float2 vs[2] = {make_float2(vsv.x, vsv.y), make_float2(vsv.z, vsv.w)};
                const float2 yy[2] = {make_float2(yv.x, yv.y), make_float2(yv.z, yv.w)};
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const float2 ec = __ffma2_rn(uc[h], vc[h], __fmul2_rn(un[h], vs[h]));      // uc vc - us vs
                    const float2 es = __ffma2_rn(uc[h], vs[h], __fmul2_rn(us[h], vc[h]));      // uc vs + us vc
                    ar[h] = __fmul2_rn(yy[h], ec);
                    ai[h] = __fmul2_rn(yy[h], es);
                    const float2 e256 = __fmul2_rn(ec, k256), n256 = __fmul2_rn(es, km256);
                    a2r[h] = __ffma2_rn(e256, ec, __fmul2_rn(n256, es));                       // 256 (ec^2 - es^2)
                    a2i[h] = __fmul2_rn(__fmul2_rn(ec, k512), es);                             // 512 ec es
                }
            }
            mbar_wait_backoff(&empty[st], eph);
            const unsigned sa = smem_u32(smem) + (unsigned)st * (unsigned)stage_bytes;
            // hi = fp16x2(x), lo = fp16x2(x - hi): one packed convert, two unpacks, one FFMA2, one packed convert per pair
            auto put = [&](int plane_hi, int plane_lo, int off, const float2 (&x)[2]) {
                const float2 m1 = make_float2(-1.f, -1.f);
                const __half2 h0 = __floats2half2_rn(x[0].x, x[0].y), h1 = __floats2half2_rn(x[1].x, x[1].y);
                asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(sa + plane_hi * A_PLANE + off),
                             "r"(*reinterpret_cast<const unsigned*>(&h0)), "r"(*reinterpret_cast<const unsigned*>(&h1)) : "memory");
                if (!FAST) {
                    const float2 r0 = __ffma2_rn(__half22float2(h0), m1, x[0]), r1 = __ffma2_rn(__half22float2(h1), m1, x[1]);
                    const __half2 l0 = __floats2half2_rn(r0.x, r0.y), l1 = __floats2half2_rn(r1.x, r1.y);
                    asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(sa + plane_lo * A_PLANE + off),
                                 "r"(*reinterpret_cast<const unsigned*>(&l0)), "r"(*reinterpret_cast<const unsigned*>(&l1)) : "memory");
                }
            };
            put(0, 2, off_re, ar);
            put(0, 2, off_im, ai);
            put(1, NOPS - 1, off_re, a2r);
            put(1, NOPS - 1, off_im, a2i);
            fence_proxy_async();            // generic-proxy stores -> visible to the tensor core's async proxy
            mbar_arrive(&full[st]);
            st += NG;
            while (st >= S) { st -= S; eph ^= 1; }
            ++it;
            t_p1 = t_pf;
            y_p1 = y_pf;
        }
    }
    // teardown: everyone is done with TMEM before it is freed
    tc_fence_before();
    __syncthreads();
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem));
}

}  // namespace lsp
