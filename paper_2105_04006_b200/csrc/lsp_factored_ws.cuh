// lsp_factored_ws.cuh -- persistent, warp-specialised version of the factored kernel (see lsp_factored.cuh for
// the mathematics: angle addition + conjugate symmetry, 4 FMA per (t, f) pair, no sincos in the O(N_t N_f) loop).
//
// One CTA per SM, 12 warps:
//   warps 0-3   consumers, contract Z(k) = sum y e^{i theta}        } 32 FFMA2 + 4 LDS.128 (FP32) or
//   warps 4-7   consumers, contract W(k) = sum e^{2 i theta}        } 32 DFMA  + 6 LDS.128 (FP64) per observation
//   warps 8-11  producers: stage (t_j, y_j), form the range-reduced phases in FP64, evaluate sincos (MUFU or
//               accurate) and write the operands a = y e^{i alpha}, a2, b = e^{i beta}, b2 of one observation
//               chunk into a shared-memory ring (hot-path steps 2-3)
// Producers and consumers meet only through mbarriers (full[s] / empty[s] per ring stage), so the FMA pipe is
// fed by warps that never wait on a sincos dependency chain or a CTA-wide barrier, while the XU / FP64 pipes
// work for the producers.  The CTA is persistent: it pulls (object, frequency tile, observation split) work
// items from a global counter (step 1: dynamic scheduling absorbs the 10x spread of N_t across objects), and the
// producers run ahead into the next item while the consumers finish the epilogue of the previous one.
//
// Epilogue (step 5, 6, 6'): Z and W warps exchange half of their sums through shared memory so that all eight
// consumer warps evaluate powers; powers are staged and stored coalesced; the per-CTA argmax partial is fused.
#pragma once
#include "lsp_factored.cuh"

namespace lsp {

constexpr int kWsConsumers = 256;
constexpr int kWsProducers = 128;
constexpr int kWsThreads = kWsConsumers + kWsProducers;
constexpr int kWsProducerRegs = 88, kWsConsumerRegs = 208;      // 128 x 88 + 256 x 208 = 64512 = 384 x 168

#ifndef LSP_WS_JC_F32
#define LSP_WS_JC_F32 16
#endif
#ifndef LSP_WS_JC_F64
#define LSP_WS_JC_F64 16      // FP64: 16-observation stages x 2 (48 KB each with NL = 32)
#endif
#ifndef LSP_WS_STAGES_F32
#define LSP_WS_STAGES_F32 4
#endif
#ifndef LSP_WS_STAGES_F64
#define LSP_WS_STAGES_F64 2
#endif
// An a-operand row (one observation, G = 64 groups) is stored in operand_pos order: the TH elements of a thread land in TH
// (FP32: TH / 2) sub-rows, and consecutive producer lanes alternate between the sub-rows, i.e. between addresses a
// multiple of 128 bytes apart: without a swizzle every quarter-warp store is a 2- or 4-way bank conflict (r01: 87.7 M
// conflicts per FP64 launch).  Inside sub-row r element i therefore sits at i ^ (r * SWZ): a 64-byte (FP32: 2 sub-rows of 32)
// or 32-byte (FP64: 4 sub-rows of 16) XOR swizzle.  No padding: the rings already fill shared memory.
template <typename T> struct WsCfg;
template <> struct WsCfg<float> {
    static constexpr int JC = LSP_WS_JC_F32;         // observations per ring stage
    static constexpr int STAGES = LSP_WS_STAGES_F32;
    static constexpr int SUB = 32, SWZ = 8;          // sub-rows of 32 float2; XOR 8 float2 = 64 bytes per sub-row index
    static constexpr int GP = kFacGroups;            // a-row length
    static constexpr int STAGE_ELEMS = JC * (2 * GP + 2 * FactoredCfg<float>::NL);   // complex elements per stage
};
template <> struct WsCfg<double> {
    static constexpr int JC = LSP_WS_JC_F64;
    static constexpr int STAGES = LSP_WS_STAGES_F64;
    static constexpr int SUB = 16, SWZ = 2;          // sub-rows of 16 double2; XOR 2 double2 = 32 bytes per sub-row index
    static constexpr int GP = kFacGroups;
    static constexpr int STAGE_ELEMS = JC * (2 * GP + 2 * FactoredCfg<double>::NL);
};

struct WsMeta {          // one per ring stage, written by producer thread 0
    long long item;      // work item id, -1 = no more work
    int last;            // 1 = last chunk of the item: consumers run the epilogue after it
    int pad;
};

// producer scratch per buffer (complex elements): u [JC][8], v [JC][8], then JC reals (y) and JC reals (w) = JC complex slots
template <typename T> __host__ __device__ constexpr int ws_scratch_elems() { return WsCfg<T>::JC * 16 + WsCfg<T>::JC; }
template <typename T> constexpr size_t ws_smem_bytes()
{
    return (size_t)WsCfg<T>::STAGES * WsCfg<T>::STAGE_ELEMS * 2 * sizeof(T)      // operand ring
           + (size_t)FactoredCfg<T>::TILE * 3 * sizeof(T)              // epilogue exchange + staged powers
           + (size_t)2 * ws_scratch_elems<T>() * 2 * sizeof(T)         // producer scratch, double-buffered
           + WsCfg<T>::STAGES * (2 * sizeof(unsigned long long) + sizeof(WsMeta)) + 64;
}

// ---- mbarrier helpers (CTA scope) ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    unsigned done;
    do {       // try_wait suspends the thread in hardware for a bounded time; loop until the phase completes
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
// The same wait with a back-off between polls, for the role that is NOT the bottleneck (its waits are long): a spinning warp
// takes issue slots from the working warps of its scheduler, and in FP64 every such slot displaces a DFMA.
__device__ __forceinline__ void mbar_wait_sleep(unsigned long long* bar, unsigned parity, unsigned ns)
{
    unsigned done;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    while (!done) {
        __nanosleep(ns);      // measured: the actual sleep is a fraction of `ns`; every poll costs the working warps issue slots
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ void named_bar_sync(int id, int n_threads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n_threads) : "memory");
}

struct WsItem {
    int64_t obj_local, obj, lo, n_t, j0, j1, K0;
    int tile, split;
};
template <int TILE>
__device__ __forceinline__ WsItem ws_decode(const GridParams& gp, long long item, const int64_t* __restrict__ offsets)
{
    WsItem w;
    w.split = (int)(item % gp.n_split);
    const long long r = item / gp.n_split;
    w.tile = (int)(r % gp.n_tiles);
    w.obj_local = r / gp.n_tiles;
    w.obj = w.obj_local + gp.obj_base;
    w.lo = offsets[w.obj];
    w.n_t = offsets[w.obj + 1] - w.lo;
    w.j0 = (w.n_t * w.split) / gp.n_split;
    w.j1 = (w.n_t * (w.split + 1)) / gp.n_split;
    w.K0 = (int64_t)w.tile * TILE;
    return w;
}

// ---- pre-pass: the tile-independent phasors of every observation --------------------------------------------------
// v_{g1 j} = e^{2 pi i (8 g1 L df) t_j} (g1 < 8), b_mj = e^{2 pi i (m + 1/2) df t_j} and b2 = b^2 (m < NL) depend on the
// observation only, not on the frequency tile, so they are evaluated once per call instead of once per (tile, observation)
// by the producers.  Three planes indexed by the GLOBAL observation number (CSR position), each padded by JC zero rows so a
// chunk that runs past an object's end still reads finite values (they meet a = 0):
//   V  [n_obs + JC][8]     complex
//   B1 [n_obs + JC][NL]    complex, columns already in the consumers' operand order (operand_pos)
//   B2 [n_obs + JC][NL]
template <typename T> constexpr size_t ws_table_row_elems() { return 8 + 2 * (size_t)FactoredCfg<T>::NL; }
template <typename T> constexpr size_t ws_table_bytes(int64_t n_obs)
{
    return (size_t)(n_obs + WsCfg<T>::JC) * ws_table_row_elems<T>() * 2 * sizeof(T);
}
template <typename T, bool FAST>
__global__ void __launch_bounds__(256)
lsp_ws_table_kernel(GridParams gp, const T* __restrict__ t, int64_t n_obs, typename FactoredCfg<T>::V2* __restrict__ tabV,
                    typename FactoredCfg<T>::V2* __restrict__ tabB1, typename FactoredCfg<T>::V2* __restrict__ tabB2)
{
    using C = FactoredCfg<T>;
    using V2 = typename C::V2;
    constexpr int NL = C::NL, L = 2 * NL, ROW = 8 + NL;            // phasors evaluated per observation
    constexpr int NMI = NL / C::TM;
    const int64_t rows = n_obs + WsCfg<T>::JC;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < rows * ROW; idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t j = idx / ROW;
        const int e = (int)(idx - j * ROW);
        V2 z;
        z.x = z.y = T(0);
        PhaseFreq<T> f;
        if (e < 8) {
            if (j < n_obs) {
                f.set((double)(8 * e) * (double)L * gp.df);
                T sn, cs;
                f.template phasor<FAST>(t[j], &sn, &cs);
                z.x = cs;
                z.y = sn;
            }
            tabV[j * 8 + e] = z;
        } else {
            const int m = e - 8;
            V2 z2 = z;
            if (j < n_obs) {
                f.set(((double)m + 0.5) * gp.df);
                T sn, cs;
                f.template phasor<FAST>(t[j], &sn, &cs);
                z.x = cs;
                z.y = sn;
                z2.x = fma(cs, cs, -sn * sn);
                z2.y = T(2) * cs * sn;
            }
            const int pos = operand_pos<C::TM, NMI, C::EPC>(m);
            tabB1[j * NL + pos] = z;
            tabB2[j * NL + pos] = z2;
        }
    }
}

// 1-D TMA (bulk async copy) global -> shared, completion on an mbarrier's transaction count
__device__ __forceinline__ void ws_mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void ws_bulk_g2s(void* smem_dst, const void* gmem_src, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// WGT (generalised mode only): the W operands carry the weights, a2 = w e^{2 i alpha}, so W(k) = sum w e^{2 i theta}.
template <typename T, bool FAST, bool WGT = false>
__global__ void __launch_bounds__(kWsThreads, 1)
lsp_factored_ws_kernel(GridParams gp, const int64_t* __restrict__ offsets, const T* __restrict__ t,
                       const T* __restrict__ y, const ObjStats* __restrict__ stats,
                       T* __restrict__ out_power, Best* __restrict__ partials,
                       typename Vec4<T>::type* __restrict__ sums, int64_t n_obj_launch,
                       long long total_items, unsigned long long* __restrict__ work_counter,
                       const typename FactoredCfg<T>::V2* __restrict__ tabV, const typename FactoredCfg<T>::V2* __restrict__ tabB1,
                       const typename FactoredCfg<T>::V2* __restrict__ tabB2, const T* __restrict__ wgt = nullptr)
{
    using C = FactoredCfg<T>;
    using V2 = typename C::V2;
    constexpr int G = kFacGroups, TH = C::TH, TM = C::TM, NL = C::NL, L = 2 * NL, TILE = C::TILE, EPC = C::EPC;
    constexpr int JC = WsCfg<T>::JC, S = WsCfg<T>::STAGES, GP = WsCfg<T>::GP, SUB = WsCfg<T>::SUB, SWZ = WsCfg<T>::SWZ;
    constexpr int NGI = G / TH, NMI = NL / TM;
    constexpr int STAGE = WsCfg<T>::STAGE_ELEMS;             // V2 elements per stage: [JC][GP] a, [JC][GP] a2, [JC][NL] b, [JC][NL] b2
    static_assert(NGI * NMI == kWsConsumers / 2, "Z and W halves each cover the G x NL tile once");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    V2* ring = reinterpret_cast<V2*>(smem_raw);
    V2* sX = ring + (size_t)S * STAGE;                         // [TILE] exchanged sums
    T* sP = reinterpret_cast<T*>(sX + TILE);                   // [TILE] staged powers
    constexpr int SCR = ws_scratch_elems<T>();
    V2* scratch = reinterpret_cast<V2*>(sP + TILE);            // [2][SCR] producer phasor scratch
    unsigned long long* full = reinterpret_cast<unsigned long long*>(scratch + 2 * SCR);
    unsigned long long* empty = full + S;
    WsMeta* meta = reinterpret_cast<WsMeta*>(empty + S);
    __shared__ Best sbest[kWsConsumers / 32];
    __shared__ long long s_next_item;

    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s = 0; s < S; ++s) {
            mbar_init(&full[s], kWsProducers + 1);     // + the expect_tx arrival of the B-operand bulk copies
            mbar_init(&empty[s], kWsConsumers / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // Register split (384 threads x 168 at launch): the consumers hold TH x TM x 4 accumulators (FP64: 128 registers) plus their
    // operands, the producers need little.
    if (tid >= kWsConsumers) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kWsProducerRegs));
        // =========================================== producers ===============================================
        // a_gj = y_j e^{i alpha_gj} with alpha_gj = 2 pi f(c_g) t_j and g = 8 g1 + g0.  f(c_g) = f(c_g0) + g1 (8 L df), so
        //     e^{i alpha_gj} = u_{g0 j} v_{g1 j},   u = e^{2 pi i f(c_g0) t_j},   v = e^{2 pi i (8 g1 L df) t_j}.
        // Only u depends on the frequency tile: v, b and b2 come from the per-call table (lsp_ws_table_kernel).  Per stage a
        // producer thread evaluates JC/16 phasors u (reduced-argument sincos, lsp_common.cuh) and copies as many v into a small
        // scratch (phase 1), then forms G JC / 128 complex products a = y u v, a2 = (u v)^2 (phase 2); the b / b2 rows of the
        // stage are two bulk copies (TMA) from the table straight into the ring, completing on the stage's full barrier.
        const int ptid = tid - kWsConsumers;
        const int gen_g = ptid & (G - 1);
        const int gen_pos_raw = operand_pos<TH, NGI, EPC>(gen_g);
        const int gen_pos_a = gen_pos_raw ^ ((gen_pos_raw / SUB) * SWZ);        // XOR swizzle inside the sub-row
        const int p_q = ptid & 7, p_j = ptid >> 3;                                 // phase 1: phasor index, observation
        static_assert(JC % 16 == 0 && kWsProducers == 128 && G == 64, "producer work split");
        constexpr int NP = JC / 16;                                                // u phasors per thread per chunk
        PhaseFreq<T> f_u;
        constexpr int NA = (G * JC) / kWsProducers;                                // a-elements per thread per chunk
        constexpr unsigned B_BYTES = (unsigned)(JC * NL * sizeof(V2));             // one of the two B planes of a stage
        long long item = blockIdx.x;      // first item is static; the rest come from the global counter
        unsigned c = 0;
        while (true) {
            if (item >= total_items) {
                const int s = c % S;
                mbar_wait(&empty[s], ((c / S) & 1) ^ 1);
                if (ptid == 0) { meta[s].item = -1; meta[s].last = 1; mbar_arrive(&full[s]); }      // stands in for the expect_tx arrival
                mbar_arrive(&full[s]);
                break;
            }
            const WsItem w = ws_decode<TILE>(gp, item, offsets);
            const T mean = stats ? (T)stats[w.obj].mean : T(0);
            f_u.set(gp.f_min + ((double)(w.K0 + (int64_t)p_q * L + NL) - 0.5) * gp.df);      // f(c_{g0 = p_q})
            if (ptid == 0) s_next_item = (long long)gridDim.x + (long long)atomicAdd(work_counter, 1ULL);
            int64_t jb = w.j0;
            do {      // at least one chunk per item, so empty objects still reach the epilogue
                // loads first, so their latency overlaps the phase-1 arithmetic and the wait for a free stage
                T t1[NP], y1[NP], w1[NP];
                V2 v1[NP];
#pragma unroll
                for (int h = 0; h < NP; ++h) {
                    const int64_t j = jb + p_j + 16 * h;
                    const bool live1 = j < w.j1;
                    t1[h] = live1 ? t[w.lo + j] : T(0);
                    y1[h] = (live1 && p_q == 0) ? y[w.lo + j] - mean : T(0);
                    w1[h] = (WGT && live1 && p_q == 0) ? wgt[w.lo + j] : T(0);
                    v1[h] = tabV[(w.lo + j) * 8 + p_q];                              // padded table: always in range, finite
                }
                // ---- phase 1: u of (p_q, p_j + 16 h) (zero beyond the item's range) and v into the scratch
                V2* sU = scratch + (size_t)(c & 1) * SCR;                            // [JC][8]
                V2* sV = sU + JC * 8;                                                // [JC][8]
                T* sY = reinterpret_cast<T*>(sV + JC * 8);                           // [JC]
                T* sW = sY + JC;                                                     // [JC] (WGT only)
#pragma unroll
                for (int h = 0; h < NP; ++h) {
                    const bool live1 = (jb + p_j + 16 * h) < w.j1;
                    T sn, cs;
                    V2 u;
                    f_u.template phasor<FAST>(t1[h], &sn, &cs);
                    u.x = live1 ? cs : T(0);
                    u.y = live1 ? sn : T(0);
                    sU[(p_j + 16 * h) * 8 + p_q] = u;
                    sV[(p_j + 16 * h) * 8 + p_q] = v1[h];
                    if (p_q == 0) sY[p_j + 16 * h] = y1[h];
                    if (WGT && p_q == 0) sW[p_j + 16 * h] = w1[h];
                }
                named_bar_sync(1, kWsProducers);
                const int s = c % S;
                mbar_wait_sleep(&empty[s], ((c / S) & 1) ^ 1, 1500);
                V2* sA1 = ring + (size_t)s * STAGE;
                V2* sA2 = sA1 + JC * GP;
                V2* sB1 = sA2 + JC * GP;
                V2* sB2 = sB1 + JC * NL;
                if (ptid == 0) {          // b, b2 rows of observations [jb, jb + JC) of this object: table -> ring (async proxy)
                    ws_mbar_arrive_expect_tx(&full[s], 2 * B_BYTES);
                    ws_bulk_g2s(sB1, tabB1 + (w.lo + jb) * NL, B_BYTES, &full[s]);
                    ws_bulk_g2s(sB2, tabB2 + (w.lo + jb) * NL, B_BYTES, &full[s]);
                }
                // ---- phase 2: a = y u v, a2 = (u v)^2 for this thread's group and NA observations
#pragma unroll
                for (int it = 0; it < NA; ++it) {
                    const int jj = (ptid + it * kWsProducers) / G;                  // 2 it + (ptid >> 6)
                    const V2 u = sU[jj * 8 + (gen_g & 7)];
                    const V2 v = sV[jj * 8 + (gen_g >> 3)];
                    const T yj = sY[jj];
                    const T ec = fma(u.x, v.x, -u.y * v.y);
                    const T es = fma(u.x, v.y, u.y * v.x);
                    V2 a1, a2;
                    a1.x = yj * ec;                  // a  = y e^{i alpha}   (u = 0, y = 0 beyond the item's range)
                    a1.y = yj * es;
                    a2.x = fma(ec, ec, -es * es);    // a2 = e^{2 i alpha}
                    a2.y = T(2) * ec * es;
                    if (WGT) {                       // ... times w_j
                        const T wj = sW[jj];
                        a2.x *= wj;
                        a2.y *= wj;
                    }
                    sA1[jj * GP + gen_pos_a] = a1;
                    sA2[jj * GP + gen_pos_a] = a2;
                }
                jb += JC;
                if (ptid == 0) { meta[s].item = item; meta[s].last = (jb >= w.j1) ? 1 : 0; }
                mbar_arrive(&full[s]);      // release: the stores above are visible to the waiting consumers
                ++c;
            } while (jb < w.j1);
            named_bar_sync(1, kWsProducers);         // s_next_item written (and everyone done with this item's decode)
            item = s_next_item;
            named_bar_sync(1, kWsProducers);         // everyone has read it before thread 0 overwrites it
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kWsConsumerRegs));
        // =========================================== consumers ===============================================
        const int lane = tid & 31, wq = (tid >> 5) & 3;
        const bool is_w = tid >= kWsConsumers / 2;             // warps 4-7 contract W (doubled angles)
        int gi, mi;
        if (NMI == 8) {      // FP32: mi = (b1, b3, b4), gi = (b0, b2, warp)
            mi = ((lane >> 1) & 1) | (((lane >> 3) & 3) << 1);
            gi = (lane & 1) | (((lane >> 2) & 1) << 1) | (wq << 2);
        } else {             // FP64: mi = (b1, b3), gi = (b0, b2, b4, warp)
            mi = ((lane >> 1) & 1) | (((lane >> 3) & 1) << 1);
            gi = (lane & 1) | (((lane >> 2) & 1) << 1) | (((lane >> 4) & 1) << 2) | (wq << 3);
        }
        const int offA = is_w ? JC * GP : 0;
        const int offB = 2 * JC * GP + (is_w ? JC * NL : 0);
        // element offsets of this thread's operands inside one observation's rows (the XOR swizzle is folded in here, once):
        // the inner loop's loads then differ by compile-time multiples of the row lengths only (immediate offsets)
        int oa[EPC == 2 ? TH / 2 : TH], ob[EPC == 2 ? TM / 2 : TM];
        if constexpr (EPC == 2) {          // float4 units (two complex operands per load)
            static_assert(EPC == 1 || (TH / 2 * NGI * 2 == G && NGI * 2 == SUB), "one float4 index step of NGI = one sub-row");
#pragma unroll
            for (int q = 0; q < TH / 2; ++q) oa[q] = q * NGI + (gi ^ (q * (SWZ / 2)));
#pragma unroll
            for (int q = 0; q < TM / 2; ++q) ob[q] = q * NMI + mi;
        } else {
            static_assert(EPC == 2 || NGI == SUB, "one index step of NGI = one sub-row");
#pragma unroll
            for (int a = 0; a < TH; ++a) oa[a] = a * NGI + (gi ^ (a * SWZ));
#pragma unroll
            for (int cc = 0; cc < TM; ++cc) ob[cc] = cc * NMI + mi;
        }

        V2 acc_r[TH][TM], acc_i[TH][TM];        // (Srr, Sri) and (Sir, Sii) of this thread's (group, m) pairs
#pragma unroll
        for (int a = 0; a < TH; ++a)
#pragma unroll
            for (int cc = 0; cc < TM; ++cc) {
                acc_r[a][cc].x = acc_r[a][cc].y = T(0);
                acc_i[a][cc].x = acc_i[a][cc].y = T(0);
            }
        unsigned c = 0;
        // One ring stage: JC observations into this thread's accumulators (step 4).
        auto contract_stage = [&](int s) {
            const V2* A = ring + (size_t)s * STAGE + offA;
            const V2* B = ring + (size_t)s * STAGE + offB;
#pragma unroll
            for (int jj = 0; jj < JC; ++jj) {
                V2 av[TH], bv[TM];
                if constexpr (EPC == 2) {           // one LDS.128 = two complex operands
#pragma unroll
                    for (int q = 0; q < TH / 2; ++q) {
                        const float4 ch = reinterpret_cast<const float4*>(A)[jj * (GP / 2) + oa[q]];
                        av[2 * q].x = ch.x; av[2 * q].y = ch.y; av[2 * q + 1].x = ch.z; av[2 * q + 1].y = ch.w;
                    }
#pragma unroll
                    for (int q = 0; q < TM / 2; ++q) {
                        const float4 ch = reinterpret_cast<const float4*>(B)[jj * (NL / 2) + ob[q]];
                        bv[2 * q].x = ch.x; bv[2 * q].y = ch.y; bv[2 * q + 1].x = ch.z; bv[2 * q + 1].y = ch.w;
                    }
                } else {                            // one LDS.128 = one complex operand
#pragma unroll
                    for (int a = 0; a < TH; ++a) av[a] = A[jj * GP + oa[a]];
#pragma unroll
                    for (int cc = 0; cc < TM; ++cc) bv[cc] = B[jj * NL + ob[cc]];
                }
#pragma unroll
                for (int a = 0; a < TH; ++a)
#pragma unroll
                    for (int cc = 0; cc < TM; ++cc) cmac(acc_r[a][cc], acc_i[a][cc], av[a].x, av[a].y, bv[cc]);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        };
        while (true) {
            // The stages of one item, TWO per trip of the loop.  ptxas renames the 64 accumulators through the unrolled stage body
            // and restores the loop-carried assignment with ~250 moves at the back edge (0.47 other instructions per DFMA; a DFMA
            // holds its scheduler for two cycles, so every one of them displaces half a DFMA).  The renaming is an involution: a
            // second copy of the body brings the accumulators home and the moves disappear (0.14 per DFMA).
            long long item;
            int last;
            bool fin = false;
            do {
                {
                    const int s = c % S;
                    mbar_wait(&full[s], (c / S) & 1);
                    item = meta[s].item;
                    last = meta[s].last;
                    if (item < 0) { fin = true; break; }
                    contract_stage(s);
                    ++c;
                }
                if (last) break;
                {
                    const int s = c % S;
                    mbar_wait(&full[s], (c / S) & 1);
                    item = meta[s].item;
                    last = meta[s].last;
                    if (item < 0) { fin = true; break; }
                    contract_stage(s);
                    ++c;
                }
            } while (!last);
            if (fin) break;

            // ---- epilogue of `item` (steps 5, 6, 6') -------------------------------------------------------------
            const WsItem w = ws_decode<TILE>(gp, item, offsets);
            const T scale = stats ? (T)stats[w.obj].scale : T(1);
            // Each thread keeps the sums of its "own" half of its (group, m) pairs and publishes the other half:
            // Z threads own cc < TM/2, W threads own cc >= TM/2.
            // (register arrays are indexed with compile-time constants only; the role picks by select)
            constexpr int HM = TM / 2;
#pragma unroll
            for (int a = 0; a < TH; ++a)
#pragma unroll
                for (int h = 0; h < HM; ++h) {
                    const V2 pr = is_w ? acc_r[a][h] : acc_r[a][HM + h];
                    const V2 pi = is_w ? acc_i[a][h] : acc_i[a][HM + h];
                    const int kg = (gi * TH + a) * L, m = mi * TM + (is_w ? h : HM + h);
                    V2 up, dn;
                    up.x = pr.x - pi.y;    // Srr - Sii
                    up.y = pr.y + pi.x;    // Sri + Sir
                    dn.x = pr.x + pi.y;    // Srr + Sii
                    dn.y = pi.x - pr.y;    // Sir - Sri
                    sX[kg + NL + m] = up;
                    sX[kg + NL - 1 - m] = dn;
                }
            named_bar_sync(2, kWsConsumers);
            Best mine;
            mine.p = -1.0;
            mine.k = INT64_MAX;
            const bool stage_out = !sums && (out_power != nullptr);
#pragma unroll
            for (int a = 0; a < TH; ++a)
#pragma unroll
                for (int h = 0; h < HM; ++h) {
                    const V2 orr = is_w ? acc_r[a][HM + h] : acc_r[a][h];
                    const V2 oi = is_w ? acc_i[a][HM + h] : acc_i[a][h];
                    const int kg = (gi * TH + a) * L, m = mi * TM + (is_w ? HM + h : h);
#pragma unroll
                    for (int up = 0; up < 2; ++up) {
                        const int kl = up ? (kg + NL + m) : (kg + NL - 1 - m);
                        const int64_t k = w.K0 + kl;
                        const V2 other = sX[kl];
                        V2 me;
                        if (up) {
                            me.x = orr.x - oi.y;
                            me.y = orr.y + oi.x;
                        } else {
                            me.x = orr.x + oi.y;
                            me.y = oi.x - orr.y;
                        }
                        const V2 z = is_w ? other : me;      // (xc, xs)
                        const V2 ww = is_w ? me : other;     // (c2, s2)
                        if (sums) {
                            if (k < gp.n_freq)
                                sums[((int64_t)w.split * n_obj_launch + w.obj_local) * gp.n_freq + k] = make_vec4<T>(z.x, z.y, ww.x, ww.y);
                        } else {
                            const T p = power_from_sums<T>(z.x, z.y, ww.x, ww.y, (T)w.n_t, scale);
                            if (stage_out) sP[kl] = p;
                            if (k < gp.n_freq) {
                                Best b;
                                b.p = (p == p) ? (double)p : -1.0;
                                b.k = k;
                                mine = best_of(mine, b);
                            }
                        }
                    }
                }
            if (stage_out) {
                named_bar_sync(2, kWsConsumers);
                T* dst = out_power + w.obj_local * gp.n_freq + w.K0;
                const int n_valid = (int)min((int64_t)TILE, (int64_t)gp.n_freq - w.K0);
                for (int i = tid; i < n_valid; i += kWsConsumers) dst[i] = sP[i];
            }
            if (partials && !sums) {
                mine = warp_best(mine);
                if (lane == 0) sbest[tid >> 5] = mine;
                named_bar_sync(2, kWsConsumers);
                if (tid < 32) {
                    Best v;
                    v.p = -2.0;
                    v.k = INT64_MAX;
                    if (lane < kWsConsumers / 32) v = sbest[lane];
                    v = warp_best(v);
                    if (lane == 0) partials[w.obj_local * gp.n_tiles + w.tile] = v;
                }
            }
            named_bar_sync(2, kWsConsumers);      // sX / sP / sbest are free again before the next item's epilogue
#pragma unroll
            for (int a = 0; a < TH; ++a)
#pragma unroll
                for (int cc = 0; cc < TM; ++cc) {
                    acc_r[a][cc].x = acc_r[a][cc].y = T(0);
                    acc_i[a][cc].x = acc_i[a][cc].y = T(0);
                }
        }
    }
}

}  // namespace lsp
