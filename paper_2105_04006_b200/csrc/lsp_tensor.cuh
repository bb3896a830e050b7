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
//   A operands  depend on the tile: warps 12-19 generate them (FP64 phase -> sincos -> scale by y -> FP16 hi/lo) straight
//               into the stage ring (st.shared + fence.proxy.async).
//   warp 1      one thread issues the MMAs of a stage when its mbarrier completes, and tcgen05.commit releases the
//               stage / publishes the finished accumulators.
//   warps 4-11  epilogue: tcgen05.ld the accumulators, combine rows with a shuffle, closed-form power (step 5),
//               vector stores of the periodogram (step 6) or the fused argmax partial (step 6').
#pragma once
#include <cuda_fp16.h>

#include "lsp_factored_ws.cuh"

namespace lsp {

constexpr int kTcGroups = 64;                  // frequency groups per tile (128 MMA rows)
constexpr int kTcKB = 16;                      // observations per MMA / ring stage (kind::f16: K = 16)
constexpr int kTcMaxNL = 128;                  // N = 2 NL <= 256
constexpr int kTcGenWarps = 8, kTcEpiWarps = 8;
constexpr int kTcThreads = (4 + kTcEpiWarps + kTcGenWarps) * 32;      // 640
constexpr int kTcGenThreads = kTcGenWarps * 32;
constexpr int kTcEpiThreads = kTcEpiWarps * 32;
constexpr float kTcUnitScale = 256.0f;         // scale of the unit-modulus A_W operands (keeps the FP16 low part normal)

struct TensorParams {
    int nl;             // NL: half-width of a frequency group (multiple of 8, <= 128); group width L = 2 NL = MMA N
    int tile;           // frequencies per tile = 64 * 2 NL
    int n_ops;          // FP16 operand planes per stage side: 4 (accurate: hi and lo of Z- and W-operands) or 2 (fast)
    int stages;         // ring depth
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
    __shared__ double red[3][8];
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
    __shared__ int64_t part[1024];
    const int tid = threadIdx.x, nt = blockDim.x;
    const int per = (n_obj + nt - 1) / nt;
    const int o0 = min(n_obj, tid * per), o1 = min(n_obj, o0 + per);
    int64_t s = 0;
    for (int o = o0; o < o1; ++o) s += tc_n_kb(offsets[obj_base + o + 1] - offsets[obj_base + o]);
    part[tid] = s;
    __syncthreads();
    if (tid == 0) {
        int64_t run = 0;
        for (int i = 0; i < nt; ++i) { const int64_t v = part[i]; part[i] = run; run += v; }
        objs[n_obj].kb_off = run;              // total number of table blocks
    }
    __syncthreads();
    int64_t run = part[tid];
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

constexpr size_t tc_smem_bytes(int stages, int a_stage, int b_stage)
{
    return 1024 /* alignment slack */ + (size_t)stages * (size_t)(a_stage + b_stage) + 256;
}

template <typename T, bool FAST>
__global__ void __launch_bounds__(kTcThreads, 1)
lsp_tensor_kernel(GridParams gp, TensorParams tp, const int64_t* __restrict__ offsets, const T* __restrict__ t,
                  const T* __restrict__ y, const TensorObj* __restrict__ objs, const __half* __restrict__ table,
                  T* __restrict__ out_power, Best* __restrict__ partials, float4* __restrict__ sums,
                  int64_t n_obj_launch, long long total_items)
{
    constexpr int NOPS = FAST ? 2 : 4;
    constexpr int A_PLANE = 128 * kTcKB * 2;                  // bytes of one A plane: 128 rows x 16 x FP16
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
    const int S = tp.stages;
    const int stage_bytes = tp.a_stage_bytes + tp.b_stage_bytes;
    const int b_plane = 2 * tp.nl * kTcKB * 2;                // bytes of one B plane
    unsigned long long* full = reinterpret_cast<unsigned long long*>(smem + (size_t)S * stage_bytes);
    unsigned long long* empty = full + 8;
    unsigned long long* tmem_full = empty + 8;
    unsigned long long* tmem_empty = tmem_full + 1;
    __shared__ unsigned tmem_base_s;
    __shared__ Best sbest[kTcEpiWarps];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < S; ++s) {
            mbar_init(&full[s], kTcGenThreads + 1);
            mbar_init(&empty[s], 1);
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

    if (warp == 0) {
        // =============================== TMA producer: B stages from the per-object table ========================
        if (lane == 0) {
            unsigned c = 0;
            for (long long item = blockIdx.x; item < total_items; item += gridDim.x) {
                const TcItem w = tc_decode(gp, tp, item, offsets);
                const __half* src = table + (size_t)(objs[w.obj_local].kb_off + w.kb0) * (size_t)(tp.b_stage_bytes / 2);
                for (int kb = w.kb0; kb < w.kb1; ++kb, ++c) {
                    const int s = c % S;
                    mbar_wait(&empty[s], ((c / S) & 1) ^ 1);
                    mbar_arrive_expect_tx(&full[s], (unsigned)tp.b_stage_bytes);
                    tma_bulk_g2s(smem + (size_t)s * stage_bytes + tp.a_stage_bytes, src, (unsigned)tp.b_stage_bytes, &full[s]);
                    src += tp.b_stage_bytes / 2;
                }
            }
        }
    } else if (warp == 1) {
        // =============================== MMA issuer ===============================================================
        if (lane == 0) {
            const unsigned idesc = (1u << 4) | ((unsigned)((2 * tp.nl) >> 3) << 17) | ((unsigned)(128 >> 4) << 24);
            const unsigned a_lbo = 16 * 128, b_lbo = (unsigned)(2 * tp.nl / 8) * 128, sbo = 128;
            unsigned c = 0, n_acc = 0;
            for (long long item = blockIdx.x; item < total_items; item += gridDim.x) {
                const TcItem w = tc_decode(gp, tp, item, offsets);
                if (w.kb1 <= w.kb0) continue;
                mbar_wait(tmem_empty, (n_acc & 1) ^ 1);          // the epilogue has drained the previous accumulators
                tc_fence_after();
                for (int kb = w.kb0; kb < w.kb1; ++kb, ++c) {
                    const int s = c % S;
                    mbar_wait(&full[s], (c / S) & 1);
                    tc_fence_after();
                    const unsigned sa = smem_u32(smem + (size_t)s * stage_bytes);
                    const unsigned sb = sa + tp.a_stage_bytes;
                    const unsigned acc = kb > w.kb0;
                    // planes: 0 = Z-operand hi, 1 = W-operand hi, 2 = Z lo, 3 = W lo
                    const uint64_t a_zh = tc_smem_desc(sa, a_lbo, sbo), a_wh = tc_smem_desc(sa + A_PLANE, a_lbo, sbo);
                    const uint64_t b_zh = tc_smem_desc(sb, b_lbo, sbo), b_wh = tc_smem_desc(sb + b_plane, b_lbo, sbo);
                    if (!FAST) {
                        const uint64_t a_zl = tc_smem_desc(sa + 2 * A_PLANE, a_lbo, sbo), a_wl = tc_smem_desc(sa + 3 * A_PLANE, a_lbo, sbo);
                        const uint64_t b_zl = tc_smem_desc(sb + 2 * b_plane, b_lbo, sbo), b_wl = tc_smem_desc(sb + 3 * b_plane, b_lbo, sbo);
                        tc_mma_f16(tmem, a_zl, b_zh, idesc, acc);
                        tc_mma_f16(tmem, a_zh, b_zl, idesc, 1u);
                        tc_mma_f16(tmem, a_zh, b_zh, idesc, 1u);
                        tc_mma_f16(tmem + 256, a_wl, b_wh, idesc, acc);
                        tc_mma_f16(tmem + 256, a_wh, b_wl, idesc, 1u);
                        tc_mma_f16(tmem + 256, a_wh, b_wh, idesc, 1u);
                    } else {
                        tc_mma_f16(tmem, a_zh, b_zh, idesc, acc);
                        tc_mma_f16(tmem + 256, a_wh, b_wh, idesc, acc);
                    }
                    tc_commit(&empty[s]);                        // stage s is free once these MMAs have read it
                }
                tc_commit(tmem_full);                            // accumulators complete
                ++n_acc;
            }
        }
    } else if (warp >= 4 && warp < 4 + kTcEpiWarps) {
        // =============================== epilogue (steps 5, 6, 6') ================================================
        const int ew = warp - 4;
        const int q = warp & 3;                                   // TMEM lane quadrant this warp may access
        const int half_sel = ew >> 2;                             // which half of the m range
        const int etid = tid - 128;
        const bool is_im = lane >= 16;
        const int g = 16 * q + (lane & 15);
        const int NL = tp.nl, L = 2 * NL;
        const int n_chunks = NL / 16 + ((NL % 16) ? 1 : 0);       // 16-column chunks over m (NL is a multiple of 8)
        const int ch0 = (n_chunks * half_sel) / 2, ch1 = (n_chunks * (half_sel + 1)) / 2;
        const bool vec_ok = (gp.n_freq % 4 == 0) && ((reinterpret_cast<uintptr_t>(out_power) & 15) == 0);
        unsigned n_acc = 0;
        for (long long item = blockIdx.x; item < total_items; item += gridDim.x) {
            const TcItem w = tc_decode(gp, tp, item, offsets);
            const TensorObj ob = objs[w.obj_local];
            const bool have = w.kb1 > w.kb0;
            if (have) {
                mbar_wait(tmem_full, n_acc & 1);
                tc_fence_after();
            }
            Best mine;
            mine.p = -1.0;
            mine.k = INT64_MAX;
            const float n_hat = kTcUnitScale * (float)w.n_t;
            T* orow = out_power ? out_power + w.obj_local * (int64_t)gp.n_freq : nullptr;
            for (int ch = ch0; ch < ch1; ++ch) {
                const int m0 = ch * 16;
                float zr[16], zi[16], wr[16], wi[16];
                if (have) {
                    const unsigned ta = tmem + ((unsigned)(32 * q) << 16);
                    tc_ld16(ta + m0, zr);
                    tc_ld16(ta + NL + m0, zi);
                    tc_ld16(ta + 256 + m0, wr);
                    tc_ld16(ta + 256 + NL + m0, wi);
                    tc_ld_wait();
                } else {
#pragma unroll
                    for (int i = 0; i < 16; ++i) zr[i] = zi[i] = wr[i] = wi[i] = 0.f;
                }
                float pw[16];
                const int m_lim = NL - m0;                               // valid i < m_lim (last chunk when NL % 16 == 8)
                const int64_t kbase = w.K0 + (int64_t)g * L + NL;
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    // rows "Re a": (Srr, Sri); rows "Im a": (Sir, Sii); partner lane (xor 16) holds the other row
                    const float p0 = __shfl_xor_sync(0xffffffffu, zr[i], 16), p1 = __shfl_xor_sync(0xffffffffu, zi[i], 16);
                    const float q0 = __shfl_xor_sync(0xffffffffu, wr[i], 16), q1 = __shfl_xor_sync(0xffffffffu, wi[i], 16);
                    const float dz = is_im ? (p0 + zi[i]) : (zr[i] - p1);      // down: Srr + Sii ; up: Srr - Sii
                    const float ez = is_im ? (zr[i] - p1) : (zi[i] + p0);      // down: Sir - Sri ; up: Sri + Sir
                    const float dw = is_im ? (q0 + wi[i]) : (wr[i] - q1);
                    const float ew2 = is_im ? (wr[i] - q1) : (wi[i] + q0);
                    // up lanes own k = c + m (ascending in i), down lanes k = c - 1 - m (descending in i)
                    if (gp.n_split > 1) {       // split-N_t: un-scaled partial sums for lsp_combine_kernel
                        const int64_t k = is_im ? (kbase - 1 - (m0 + i)) : (kbase + m0 + i);
                        if (i < m_lim && k < gp.n_freq)
                            sums[((int64_t)w.split * n_obj_launch + w.obj_local) * gp.n_freq + k] =
                                make_float4(dz * ob.zinv, ez * ob.zinv, dw * (1.0f / kTcUnitScale), ew2 * (1.0f / kTcUnitScale));
                    } else {
                        pw[i] = power_from_sums<float>(dz, ez, dw, ew2, n_hat, ob.pscale);
                    }
                }
                if (gp.n_split > 1) continue;
#pragma unroll
                for (int v4 = 0; v4 < 4; ++v4) {
                    if (v4 * 4 >= m_lim) break;
                    // element e of this vector: up -> i = 4 v4 + e ; down -> i = 4 v4 + 3 - e
                    const int64_t k0 = is_im ? (kbase - 1 - (m0 + 4 * v4 + 3)) : (kbase + m0 + 4 * v4);
                    {
                        const float e0 = is_im ? pw[4 * v4 + 3] : pw[4 * v4], e1 = is_im ? pw[4 * v4 + 2] : pw[4 * v4 + 1];
                        const float e2 = is_im ? pw[4 * v4 + 1] : pw[4 * v4 + 2], e3 = is_im ? pw[4 * v4] : pw[4 * v4 + 3];
                        if (orow) {
                            if (vec_ok && k0 + 3 < gp.n_freq) {
                                *reinterpret_cast<float4*>(orow + k0) = make_float4(e0, e1, e2, e3);
                            } else {
                                if (k0 < gp.n_freq) orow[k0] = (T)e0;
                                if (k0 + 1 < gp.n_freq) orow[k0 + 1] = (T)e1;
                                if (k0 + 2 < gp.n_freq) orow[k0 + 2] = (T)e2;
                                if (k0 + 3 < gp.n_freq) orow[k0 + 3] = (T)e3;
                            }
                        }
                        if (partials) {
                            const float ev[4] = {e0, e1, e2, e3};
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                if (k0 + e < gp.n_freq) {
                                    Best b;
                                    b.p = (ev[e] == ev[e]) ? (double)ev[e] : -1.0;
                                    b.k = k0 + e;
                                    mine = best_of(mine, b);
                                }
                            }
                        }
                    }
                }
            }
            if (have) {
                tc_fence_before();
                mbar_arrive(tmem_empty);                          // 256 arrivals: TMEM may be overwritten
                ++n_acc;
            }
            if (partials && gp.n_split == 1) {
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
        const int gw = warp - 4 - kTcEpiWarps;                    // 0..7
        const int qb = gw & 3, c = gw >> 2;                       // row block (16 groups) and k chunk of this warp
        const int g = 16 * qb + (lane >> 1);
        const int hsel = lane & 1;                                // observations 4 hsel .. 4 hsel + 3 of the chunk
        const int row_re = 32 * qb + (lane >> 1), row_im = row_re + 16;
        // byte offset of this thread's 8-byte slot inside an A plane: chunk c, row r, k%8 = 4 hsel
        const int off_re = c * (16 * 128) + (row_re >> 3) * 128 + (row_re & 7) * 16 + hsel * 8;
        const int off_im = c * (16 * 128) + (row_im >> 3) * 128 + (row_im & 7) * 16 + hsel * 8;
        const int NL = tp.nl, L = 2 * NL;
        unsigned cnt = 0;
        for (long long item = blockIdx.x; item < total_items; item += gridDim.x) {
            const TcItem w = tc_decode(gp, tp, item, offsets);
            const TensorObj ob = objs[w.obj_local];
            const float mean = (float)ob.mean;
            const double f_centre = gp.f_min + ((double)(w.K0 + (int64_t)g * L + NL) - 0.5) * gp.df;
            for (int kb = w.kb0; kb < w.kb1; ++kb, ++cnt) {
                const int64_t jb = (int64_t)kb * kTcKB + 8 * c + 4 * hsel;
                float tj[4], yj[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const bool live = (jb + i) < w.n_t;
                    tj[i] = live ? (float)t[w.lo + jb + i] : 0.f;
                    yj[i] = live ? ((float)y[w.lo + jb + i] - mean) * ob.yscale : 0.f;
                }
                float ar[4], ai[4], a2r[4], a2i[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const bool live = (jb + i) < w.n_t;
                    float sn, cs;
                    sincos_cycles<FAST>((float)frac_cycles(f_centre * (double)tj[i]), &sn, &cs);
                    ar[i] = yj[i] * cs;
                    ai[i] = yj[i] * sn;
                    const float u = live ? kTcUnitScale : 0.f;
                    a2r[i] = u * fmaf(cs, cs, -sn * sn);
                    a2i[i] = u * (2.f * cs * sn);
                }
                const int s = cnt % S;
                mbar_wait(&empty[s], ((cnt / S) & 1) ^ 1);
                unsigned char* sa = smem + (size_t)s * stage_bytes;
                auto put = [&](int plane, int off, __half2 v0, __half2 v1) {
                    uint2 u;
                    u.x = *reinterpret_cast<unsigned*>(&v0);
                    u.y = *reinterpret_cast<unsigned*>(&v1);
                    *reinterpret_cast<uint2*>(sa + plane * A_PLANE + off) = u;
                };
                __half2 h0, h1, l0, l1;
                split_half2(ar[0], ar[1], &h0, &l0);  split_half2(ar[2], ar[3], &h1, &l1);
                put(0, off_re, h0, h1);  if (!FAST) put(2, off_re, l0, l1);
                split_half2(ai[0], ai[1], &h0, &l0);  split_half2(ai[2], ai[3], &h1, &l1);
                put(0, off_im, h0, h1);  if (!FAST) put(2, off_im, l0, l1);
                split_half2(a2r[0], a2r[1], &h0, &l0);  split_half2(a2r[2], a2r[3], &h1, &l1);
                put(1, off_re, h0, h1);  if (!FAST) put(NOPS - 1, off_re, l0, l1);
                split_half2(a2i[0], a2i[1], &h0, &l0);  split_half2(a2i[2], a2i[3], &h1, &l1);
                put(1, off_im, h0, h1);  if (!FAST) put(NOPS - 1, off_im, l0, l1);
                fence_proxy_async();            // generic-proxy stores -> visible to the tensor core's async proxy
                mbar_arrive(&full[s]);
            }
        }
    }
    // teardown: everyone is done with TMEM before it is freed
    tc_fence_before();
    __syncthreads();
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem));
}

}  // namespace lsp
