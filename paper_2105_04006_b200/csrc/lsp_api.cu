// lsp_api.cu -- the C ABI of include/lsp.h: plan object, argument validation, scheduling (hot-path step 1),
// kernel launches (steps 2-6') and the pinned-host multi-stream D2H pipeline (step 7).
// There is no CPU fallback in this file or anywhere in the library.
#include "../../include/lsp.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <utility>
#include <type_traits>
#include <vector>

#include "lsp_factored_ws.cuh"
#include "lsp_tensor.cuh"
#include "lsp_gls.cuh"

using namespace lsp;

namespace {

thread_local std::string g_create_error;

struct DeviceBuffer {
    void*  ptr = nullptr;
    size_t bytes = 0;
};

}  // namespace

struct lsp_plan {
    lsp_config cfg{};
    int sm_count = 0;
    int smem_optin = 0;           // max dynamic shared memory per CTA
    std::string error;

    std::vector<cudaStream_t> copy_streams;
    std::vector<cudaEvent_t> slot_ready, slot_free;
    std::vector<char> slot_used;
    DeviceBuffer ring;            // n_slots * slot_bytes
    void*  stage_host = nullptr;  // pinned staging ring for a PAGEABLE host destination (n_slots * slot_bytes)
    size_t stage_host_bytes = 0;
    struct HostCopy { void* dst; const void* src; size_t bytes; };
    std::vector<HostCopy> host_copies;           // arguments of the per-chunk host memcpy callbacks (stable during a call)
    int pageable_mode = 1;        // 1 = plain cudaMemcpyAsync to a pageable destination (default: faster on the measured host),
                                  // 0 = staged (pinned ring + host-side copies; LSP_FLAG_PAGEABLE_STAGED)
    DeviceBuffer partials;        // Best[n_obj * n_parts]
    DeviceBuffer sums;            // Vec4<T>[n_split * n_obj_launch * n_freq]
    DeviceBuffer stats;           // ObjStats[n_obj]
    DeviceBuffer counter;         // work counter of the persistent kernel
    DeviceBuffer ws_table;        // tile-independent phasors V, B1, B2 of every observation (factored WS path pre-pass)
    DeviceBuffer tc_objs;         // TensorObj[n_obj_launch]   (tensor path pre-pass)
    DeviceBuffer tc_table;        // B-operand table of the launch's objects (tensor path)
    size_t tc_table_budget = (size_t)12 << 30;    // objects per launch are capped so the table stays below this
    int tc_stages_b = 0;          // B-operand ring depth of the tensor kernel; 0 = as many as fit (cfg.tensor_b_stages)
    int tc_products = 3;          // FP16 products per MAC of the accurate tensor mode: 3 (default) or 2 (cfg.tensor_products)
    int tc_pair = 0;              // CTA pairs on the tensor path: 0 = when items are long, 1 = never, 2 = whenever there are >= 2 tiles (cfg.tensor_pair)
    int tc_roles = 0;             // 0 = by item length, 1 = force the short-item role shape, 2 = force the long-item one (cfg.tensor_roles)
    DeviceBuffer in_off, in_t, in_y, in_sigma, out_best;   // device copies of host inputs / best-period outputs (lsp_periodogram_batched_host)
    int64_t ws_table_obs = 0;     // observations the table was built for (this call)
    DeviceBuffer gls_x, gls_yy, gls_sums;        // generalised mode: x_A / x_B arrays, chi0^2 per object, 3 passes of partial sums
    int64_t* h_offsets_pinned = nullptr;
    size_t   h_offsets_cap = 0;
    // Dynamic shared memory opted in per kernel function on THIS plan's device (the attribute is per device, and a plan is
    // bound to one device): (function, bytes) pairs.
    std::vector<std::pair<const void*, size_t>> smem_optins;

    // last-call bookkeeping
    int64_t n_launches = 0, n_pairs = 0, n_chunks = 0;
    int32_t kernel_used = 0, n_split = 1;
    int32_t tensor_shape = 0;     // role shape of the last tensor-kernel launch: 0 = none, 1 = short-item, 2 = long-item
    int32_t tensor_products = 0;  // FP16 products per MAC of the last tensor-kernel launch (0 = none)
    bool timing = false;
    std::vector<cudaEvent_t> t_start, t_stop;
    size_t t_used = 0;
};

namespace {

lsp_status fail(lsp_plan* p, lsp_status st, const char* fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (p) p->error = buf; else g_create_error = buf;
    return st;
}

#define LSP_CUDA(p, call)                                                                              \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess)                                                                         \
            return fail((p), e_ == cudaErrorMemoryAllocation ? LSP_ERR_OOM : LSP_ERR_CUDA, "%s: %s",  \
                        #call, cudaGetErrorString(e_));                                                \
    } while (0)

lsp_status ensure(lsp_plan* p, DeviceBuffer& b, size_t bytes)
{
    if (bytes <= b.bytes) return LSP_OK;
    if (b.ptr) {
        LSP_CUDA(p, cudaFree(b.ptr));
        b.ptr = nullptr;
        b.bytes = 0;
    }
    LSP_CUDA(p, cudaMalloc(&b.ptr, bytes));
    b.bytes = bytes;
    return LSP_OK;
}

size_t elem_size(const lsp_config& c) { return c.dtype == LSP_F32 ? 4 : 8; }

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute: remembered per plan (one device), never per process.
template <typename K>
cudaError_t optin_smem(lsp_plan* p, K kern, size_t bytes)
{
    const void* key = reinterpret_cast<const void*>(kern);
    for (auto& e : p->smem_optins)
        if (e.first == key) {
            if (e.second >= bytes) return cudaSuccess;
            const cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
            if (err == cudaSuccess) e.second = bytes;
            return err;
        }
    const cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (err == cudaSuccess) p->smem_optins.emplace_back(key, bytes);
    return err;
}

// Launch with programmatic stream serialisation: the kernel may start while its predecessor on the stream drains; it must
// execute griddepcontrol.wait (pdl_wait in lsp_tensor.cuh) before reading what the predecessor wrote.
// `cluster` > 1 launches thread-block clusters of that many CTAs (the tensor kernel's CTA pairs).
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st, int cluster, Args... args)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.numAttrs = 1;
    if (cluster > 1) {
        attr[1].id = cudaLaunchAttributeClusterDimension;
        attr[1].val.clusterDim.x = (unsigned)cluster;
        attr[1].val.clusterDim.y = 1;
        attr[1].val.clusterDim.z = 1;
        cfg.numAttrs = 2;
    }
    cfg.attrs = attr;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// The grid and per-object conventions one launch sequence runs with.  The standard calls use the plan's own; the generalised
// mode passes derived ones (doubled grid, no centring) BY VALUE -- the plan's public configuration is never scratch space.
struct GridSpec {
    double f_min, f_max;
    int center, normalize;
};
GridSpec plan_grid(const lsp_config& c) { return GridSpec{c.f_min, c.f_max, c.center, c.normalize}; }

// ---- step 1: scheduling ------------------------------------------------------------------------------------
struct Schedule {
    int kernel;      // LSP_KERNEL_DIRECT / LSP_KERNEL_FACTORED
    int direct_r;    // frequencies per thread of the direct kernel (1 or 4)
    int tile;        // frequencies per CTA
    int n_tiles;
    int n_split;
    int products;      // tensor path: FP16 products per MAC (1 = fast_math, 2, 3)
    TensorParams tp;   // tensor path only
};

// Two-product tensor mode (lsp_config.tensor_products = 2, an explicit opt-in; the default is three): the generated operand
// a = y e^{i alpha} is a single FP16, i.e. every term of a sum carries a relative error of up to 2^-12.  What that does to P is set
// by the conditioning of step 5's 2 x 2 system (n^2 - c2^2 - s2^2), not by N_t: a few 1e-5 of max P when a signal dominates,
// <= 4.5e-4 on pure-noise objects observed over a year, but several 1e-3 -- over the FP32 tolerance -- on noise-only objects
// taken on a handful of nights inside a short nightly window (tests/test_gpu_parity.py, few-night cadences).
// The caller who opts in vouches for the cadence.  One guard stays: objects of a handful of observations are close to singular
// at many grid frequencies whatever the cadence, so a CALL that holds an object shorter than this runs with three products.
// The decision is per call -- never per launch -- so chunks and table-budget sub-ranges of one call all run the same mode.
constexpr int64_t kTcMinNtTwoProducts = 32;

// Smallest N_t > 0 among objects [o0, o0 + no) (INT64_MAX if all are empty); `ho` = host copy of the CSR offsets.
int64_t range_min_nt(const int64_t* ho, int64_t o0, int64_t no)
{
    int64_t m = INT64_MAX;
    for (int64_t o = o0; o < o0 + no; ++o) {
        const int64_t n = ho[o + 1] - ho[o];
        if (n > 0 && n < m) m = n;
    }
    return m;
}

Schedule make_schedule(const lsp_plan* p, int64_t n_obj, int64_t total_obs, int kernel_override = -1, int64_t min_nt = INT64_MAX,
                       bool allow_pair = true)
{
    const lsp_config& c = p->cfg;
    Schedule s{};
    int k = kernel_override >= 0 ? kernel_override : c.kernel;
    if (k == LSP_KERNEL_AUTO)
        k = (c.n_freq < 1024) ? LSP_KERNEL_DIRECT : (c.dtype == LSP_F32 ? LSP_KERNEL_TENSOR : LSP_KERNEL_FACTORED);
    s.kernel = k;
    int64_t slots;                                                // resident CTAs on the whole GPU
    // tensor path: tiles of 64 groups x 2 NL frequencies, NL the smallest multiple of 8 that covers N_f with `nt` tiles
    int64_t max_nl = kTcMaxNL;
    int64_t max_tile = (int64_t)kTcGroups * 2 * max_nl;
    auto tensor_tiles = [&](int64_t nt) {
        int64_t nl = (c.n_freq + nt * 2 * kTcGroups - 1) / (nt * 2 * kTcGroups);
        nl = std::min<int64_t>(max_nl, std::max<int64_t>(8, (nl + 7) / 8 * 8));
        s.tp.nl = (int)nl;
        s.tp.tile = (int)(kTcGroups * 2 * nl);
        s.tile = s.tp.tile;
        s.n_tiles = (int)((c.n_freq + s.tile - 1) / s.tile);
    };
    if (k == LSP_KERNEL_TENSOR) {
        tensor_tiles((c.n_freq + max_tile - 1) / max_tile);
        s.tp.n_ops = c.fast_math ? 2 : 4;
        s.products = c.fast_math ? 1 : ((p->tc_products != 2 || min_nt < kTcMinNtTwoProducts) ? 3 : 2);
        s.direct_r = 0;
        slots = p->sm_count;
    } else if (k == LSP_KERNEL_FACTORED) {
        s.tile = c.dtype == LSP_F32 ? fac_tile<float>() : fac_tile<double>();
        s.direct_r = 0;
        slots = (int64_t)p->sm_count;                             // one persistent CTA per SM
    } else {
        const int64_t tiles4 = (c.n_freq + 4 * kDirectThreads - 1) / (4 * kDirectThreads);
        s.direct_r = (n_obj * tiles4 >= (int64_t)p->sm_count * 8) ? 4 : 1;
        s.tile = s.direct_r * kDirectThreads;
        slots = (int64_t)p->sm_count * (s.direct_r == 4 ? (c.dtype == LSP_F32 ? 4 : 3) : 8);
    }
    if (k != LSP_KERNEL_TENSOR) s.n_tiles = (int)((c.n_freq + s.tile - 1) / s.tile);
    // Split the observations of every object when (object, tile) items alone cannot fill the GPU for a few
    // waves (large-N_t / small-N_f problems; PAPER.md:L373, L396 describe the under-filled GPU).  Among the
    // admissible split counts pick the one whose last wave is fullest (wave quantisation), then the smallest.
    const int64_t avg_nt = total_obs / std::max<int64_t>(1, n_obj);
    auto choose_split = [&](int64_t items, int64_t n_slots) {
        int64_t split = 1;
        if (items < 8 * n_slots && n_obj > 0) {
            const int64_t min_obs = (k == LSP_KERNEL_TENSOR) ? 256 : (k == LSP_KERNEL_FACTORED) ? 128 : 64;   // per split, to amortise prologue/epilogue
            const int64_t s_max = std::max<int64_t>(1, std::min<int64_t>(64, avg_nt / min_obs));
            double best_score = -1.0;
            for (int64_t cand = 1; cand <= s_max; ++cand) {
                const double waves = (double)(items * cand) / (double)n_slots;
                const double eff = waves / std::ceil(waves);               // occupancy of the average wave
                const double score = eff - 0.004 * (double)(cand - 1);     // each split adds a partial-sum pass
                if (score > best_score + 1e-9) { best_score = score; split = cand; }
                if (waves >= 8.0) break;
            }
        }
        if (k == LSP_KERNEL_TENSOR && n_obj > 0) {
            // The tensor cores add into their FP32 accumulators with truncation: the bias grows with the number of accumulations
            // (measured ~3e-8 of the sum per 16-observation stage).  Items are capped at 1024 stages so it stays below 1e-4 of max P.
            const int64_t nkb_avg = (avg_nt + kTcKB - 1) / kTcKB;
            split = std::max<int64_t>(split, (nkb_avg + 1023) / 1024);
        }
        return split;
    };
    int64_t split = choose_split(std::max<int64_t>(1, n_obj * s.n_tiles), slots);
    if (k == LSP_KERNEL_TENSOR) {
        // role shape by item length: stages (16 observations) per work item
        int64_t stages_per_item = (avg_nt / kTcKB) / std::max<int64_t>(1, split);
        s.tp.long_items = (p->tc_roles == 0) ? (stages_per_item >= 48 ? 1 : 0) : (p->tc_roles == 2 ? 1 : 0);
        // CTA pairs (cta_group::2; the long-item shape only): an item is a pair of tiles, one per CTA of a 2-CTA cluster, which
        // share every B stage (each CTA holds half of its columns).  Halves the shared-memory traffic per MMA, which bounds
        // the unpaired kernel; taken when the items stay long on half as many (twice as wide) scheduling slots.
        s.tp.pair = 0;
        if (allow_pair && p->tc_pair != 1 && s.n_tiles >= 2 && p->sm_count >= 2 && n_obj > 0 && (p->tc_pair == 2 || p->tc_roles != 1)) {
            const Schedule q = s;                                 // the unpaired schedule, restored if the paired one is rejected
            max_nl = kTcPairMaxNL;                                // narrower tiles: tensor-memory columns for a deeper A ring
            max_tile = (int64_t)kTcGroups * 2 * max_nl;
            const int64_t nt0 = (c.n_freq + max_tile - 1) / max_tile;
            tensor_tiles(nt0);
            if ((nt0 & 1) && nt0 > 1) {                           // an even tile count wastes no phantom tile: take it if NL shrinks
                const int nl0 = s.tp.nl;
                tensor_tiles(nt0 + 1);
                if (s.tp.nl >= nl0 || (s.n_tiles & 1)) tensor_tiles(nt0);
            }
            const int64_t n_tp = (s.n_tiles + 1) / 2;
            const int64_t split_p = choose_split(std::max<int64_t>(1, n_obj * n_tp), p->sm_count / 2);
            const int64_t stages_p = (avg_nt / kTcKB) / std::max<int64_t>(1, split_p);
            if (p->tc_pair == 2 || stages_p >= 48) {
                s.tp.pair = 1;
                s.tp.long_items = 1;
                split = split_p;
            } else {
                s = q;
            }
        }
        s.tp.b_plane_bytes = (s.tp.pair ? 1 : 2) * s.tp.nl * kTcKB * 2;
        s.tp.b_stage_bytes = s.tp.n_ops * 2 * s.tp.nl * kTcKB * 2 + kTcAuxBytes;
        s.tp.smem_stage_bytes = s.tp.n_ops * s.tp.b_plane_bytes + kTcAuxBytes;
        // B ring (TMA -> MMA; the generators read its aux blocks): as deep as shared memory allows, at most 8 stages
        const int ng = s.tp.pair ? kTcPairNG : (s.tp.long_items ? 4 : 3), ew = s.tp.long_items ? 4 : 8;
        const int reserve = tc_static_smem_of(ew, ng) + (int)tc_smem_bytes(0, 0) + 512;
        const int fit = (int)std::max<int64_t>(2, std::min<int64_t>(kTcMaxSB, (int64_t)(p->smem_optin - reserve) / s.tp.smem_stage_bytes));
        // the kernel's A-ring depth is a compile-time function of its largest tile; smaller tiles only leave more room
        const int need = ng + tc_a_depth(s.products == 1 ? 1 : (s.products == 3 ? 0 : 2), ew, ng, s.tp.pair != 0,
                                         s.tp.pair ? kTcPairMaxNL : kTcMaxNL);
        s.tp.stages_b = std::max(need, p->tc_stages_b > 0 ? std::min(p->tc_stages_b, fit) : fit);
        s.tp.fixup = split > 1 ? 1 : 0;
    }
    s.n_split = (int)split;
    return s;
}

template <typename T, bool FAST>
cudaError_t launch_main(lsp_plan* p, const Schedule& s, const GridParams& gp, int64_t n_obj_launch, const int64_t* d_off,
                        const void* d_t, const void* d_y, const ObjStats* stats, void* out, Best* partials,
                        void* sums, cudaStream_t st, const void* wgt = nullptr, const double* gls_yy = nullptr)
{
    using V4 = typename Vec4<T>::type;
    const int64_t grid = n_obj_launch * s.n_tiles * s.n_split;
    if (grid <= 0) return cudaSuccess;
    if (grid > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (s.kernel == LSP_KERNEL_TENSOR) {
        if constexpr (std::is_same<T, float>::value) {
            const size_t smem = tc_smem_bytes(s.tp.stages_b, s.tp.smem_stage_bytes);
            // pair mode: an item is (object, pair of tiles, split), one 2-CTA cluster per item slot
            const int64_t items = s.tp.pair ? n_obj_launch * ((s.n_tiles + 1) / 2) * s.n_split : grid;
            const unsigned ctas = s.tp.pair ? 2u * (unsigned)std::min<int64_t>(items, p->sm_count / 2)
                                            : (unsigned)std::min<int64_t>(items, p->sm_count);
            auto go = [&](auto kern, int threads) -> cudaError_t {
                const cudaError_t ea = optin_smem(p, kern, smem);
                if (ea != cudaSuccess) return ea;
                return launch_pdl(kern, ctas, (unsigned)threads, smem, st, s.tp.pair ? 2 : 1, gp, s.tp, d_off, (const TensorObj*)p->tc_objs.ptr,
                                  (const unsigned char*)p->tc_table.ptr, (float*)out, partials, (float4*)sums, n_obj_launch, (long long)items,
                                  gls_yy);
            };
            p->tensor_shape = s.tp.pair ? 3 : (s.tp.long_items ? 2 : 1);
            p->tensor_products = s.products;
            // precision mode of the kernel template: 1 = fast_math, 2 = two products (opt-in), 0 = three (the default)
            auto go_pm = [&](auto pm_tag) -> cudaError_t {
                constexpr int PM = decltype(pm_tag)::value;
                if (s.tp.weighted && s.tp.gls == 2)      // generalised mode, weighted W slot + ZK09's epilogue fused
                    return s.tp.long_items ? go(lsp_tensor_kernel<float, PM, 4, 4, 2>, TcRoles<4, 4>::kThreads)
                                           : go(lsp_tensor_kernel<float, PM, 8, 3, 2>, TcRoles<8, 3>::kThreads);
                if (s.tp.weighted)                       // generalised mode: the W slot carries the weights
                    return s.tp.long_items ? go(lsp_tensor_kernel<float, PM, 4, 4, 1>, TcRoles<4, 4>::kThreads)
                                           : go(lsp_tensor_kernel<float, PM, 8, 3, 1>, TcRoles<8, 3>::kThreads);
                if (s.tp.pair) return go(lsp_tensor_kernel<float, PM, 4, kTcPairNG, 0, true, kTcPairMaxNL>, TcRoles<4, kTcPairNG>::kThreads);
                return s.tp.long_items ? go(lsp_tensor_kernel<float, PM, 4, 4, 0>, TcRoles<4, 4>::kThreads)
                                       : go(lsp_tensor_kernel<float, PM, 8, 3, 0>, TcRoles<8, 3>::kThreads);
            };
            cudaError_t e;
            if (FAST) e = go_pm(std::integral_constant<int, 1>{});
            else if (s.products == 3) e = go_pm(std::integral_constant<int, 0>{});
            else e = go_pm(std::integral_constant<int, 2>{});
            if (e != cudaSuccess) return e;
        } else {
            return cudaErrorInvalidValue;      // rejected at plan creation
        }
    } else if (s.kernel == LSP_KERNEL_FACTORED) {
        cudaError_t e = cudaMemsetAsync(p->counter.ptr, 0, sizeof(unsigned long long), st);
        if (e != cudaSuccess) return e;
        const unsigned ctas = (unsigned)std::min<int64_t>(grid, p->sm_count);
        using V2 = typename FactoredCfg<T>::V2;
        const int64_t rows = p->ws_table_obs + WsCfg<T>::JC;
        const V2* tabV = (const V2*)p->ws_table.ptr;
        const V2* tabB1 = tabV + rows * 8;
        const V2* tabB2 = tabB1 + rows * FactoredCfg<T>::NL;
        auto go = [&](auto kern) -> cudaError_t {
            const cudaError_t ea = optin_smem(p, kern, ws_smem_bytes<T>());
            if (ea != cudaSuccess) return ea;
            kern<<<ctas, kWsThreads, ws_smem_bytes<T>(), st>>>(gp, d_off, (const T*)d_t, (const T*)d_y, stats, (T*)out, partials,
                                                              (V4*)sums, n_obj_launch, (long long)grid,
                                                              (unsigned long long*)p->counter.ptr, tabV, tabB1, tabB2, (const T*)wgt);
            return cudaSuccess;
        };
        e = wgt ? go(lsp_factored_ws_kernel<T, FAST, true>) : go(lsp_factored_ws_kernel<T, FAST, false>);
        if (e != cudaSuccess) return e;
    } else {
        auto go = [&](auto kern) {
            kern<<<(unsigned)grid, kDirectThreads, 0, st>>>(gp, d_off, (const T*)d_t, (const T*)d_y, stats, (T*)out, partials,
                                                            (V4*)sums, n_obj_launch, (const T*)wgt);
        };
        if (s.direct_r == 4) { if (wgt) go(lsp_direct_kernel<T, FAST, 4, true>); else go(lsp_direct_kernel<T, FAST, 4, false>); }
        else                 { if (wgt) go(lsp_direct_kernel<T, FAST, 1, true>); else go(lsp_direct_kernel<T, FAST, 1, false>); }
    }
    return cudaGetLastError();
}

// Launches steps 2-6' for objects [obj_base, obj_base + n_obj_launch) on `st`.
// `out` (device, may be NULL) receives rows relative to obj_base; partials (may be NULL) is indexed by the launch-local object.
struct RangeOpts {
    void* ext_sums = nullptr;     // write partial sums there and stop (generalised mode)
    const void* wgt = nullptr;    // generalised mode: per-observation weights (W slot = sum w e^{2 i theta}; the tensor pre-pass
                                  // stores them in the table's aux blocks)
    int w_pass = 0;               // generalised mode, the pass whose Z slot is sum w e^{i theta}: the tensor path takes w from the aux
                                  // blocks as the Z operand and skips the W contraction
    int skip_prepass = 0;         // tensor path: table and statistics of the previous launch (same objects, same grid) are reused
    int gls = 0;                  // tensor path, n_split = 1: 1 = the w pass writes (C, S) per element into ext_sums in the epilogue's
                                  // own order; 2 = the weighted pass reads them from ext_sums and evaluates ZK09's power in its epilogue
    const double* gls_yy = nullptr;   // chi0^2 per object (gls = 2)
};
lsp_status run_range(lsp_plan* p, const Schedule& s_in, const GridSpec& g, int64_t obj_base, int64_t n_obj_launch, int64_t obs_bound,
                     const int64_t* d_off, const void* d_t, const void* d_y, void* out, bool want_best, int* n_parts_out,
                     cudaStream_t st, const RangeOpts& opt = RangeOpts{})
{
    const lsp_config& c = p->cfg;
    Schedule s = s_in;
    void* ext_sums = opt.ext_sums;
    const bool tensor = s.kernel == LSP_KERNEL_TENSOR;
    const bool fixup = tensor && s.n_split > 1 && !ext_sums;      // the tensor kernel finishes split tiles itself
    if (tensor) {
        s.tp.fixup = fixup ? 1 : 0;
        s.tp.weighted = (opt.wgt && !opt.w_pass) ? 1 : 0;
        s.tp.z_only = s.tp.y_is_w = opt.w_pass;
        s.tp.gls = opt.gls;
        // pre-pass of the tensor path, ONE launch: the B-operand table (once per object, shared by all of its frequency tiles
        // and observation splits; each stage carries the aux block the generators read) and the per-object statistics
        const int64_t kb_bound = obs_bound / kTcKB + n_obj_launch;
        lsp_status e = ensure(p, p->tc_objs, (size_t)(n_obj_launch + 1) * sizeof(TensorObj));
        if (e != LSP_OK) return e;
        if ((e = ensure(p, p->tc_table, std::max<size_t>(256, (size_t)kb_bound * (size_t)s.tp.b_stage_bytes))) != LSP_OK) return e;
        GridParams gq{};
        gq.f_min = g.f_min;
        gq.df = (g.f_max - g.f_min) / (double)c.n_freq;
        gq.n_freq = (int)c.n_freq;
        gq.obj_base = (int)obj_base;
        const int64_t pre_grid = kb_bound + n_obj_launch;
        if (pre_grid > 0x7fffffffLL) return fail(p, LSP_ERR_INVALID_ARG, "batch too large for one launch");
        if (opt.skip_prepass) {
            // table and statistics of the previous launch (same objects, same grid) are still in place
        } else if (c.fast_math)
            lsp_tensor_prepass_kernel<true><<<(unsigned)pre_grid, kTcPreThreads, 0, st>>>(
                gq, s.tp, d_off, (const float*)d_t, (const float*)d_y, (const float*)opt.wgt, (TensorObj*)p->tc_objs.ptr,
                (int)n_obj_launch, (long long)kb_bound, g.center, g.normalize, (unsigned char*)p->tc_table.ptr);
        else
            lsp_tensor_prepass_kernel<false><<<(unsigned)pre_grid, kTcPreThreads, 0, st>>>(
                gq, s.tp, d_off, (const float*)d_t, (const float*)d_y, (const float*)opt.wgt, (TensorObj*)p->tc_objs.ptr,
                (int)n_obj_launch, (long long)kb_bound, g.center, g.normalize, (unsigned char*)p->tc_table.ptr);
        LSP_CUDA(p, cudaGetLastError());
        if (!opt.skip_prepass) ++p->n_launches;
    }
    GridParams gp;
    gp.f_min = g.f_min;
    gp.df = (g.f_max - g.f_min) / (double)c.n_freq;
    gp.n_freq = (int)c.n_freq;
    gp.n_tiles = s.n_tiles;
    gp.n_split = s.n_split;
    gp.obj_base = (int)obj_base;
    const ObjStats* stats = (g.center || g.normalize) ? (const ObjStats*)p->stats.ptr : nullptr;
    void* sums = nullptr;
    const int n_cparts = (int)((c.n_freq + kCombineThreads * kCombinePerThread - 1) / (kCombineThreads * kCombinePerThread));
    if (ext_sums) {
        sums = ext_sums;
    } else if (fixup) {
        // tensor path: one slot per (split, object, tile) in the epilogue's own element order (lsp_tensor.cuh)
        const size_t tile_elems = (size_t)((s.tp.nl + 15) / 16) * 16 * 128;
        const size_t need = (size_t)s.n_split * n_obj_launch * s.n_tiles * tile_elems * sizeof(float4);
        lsp_status e = ensure(p, p->sums, need);
        if (e != LSP_OK) return e;
        sums = p->sums.ptr;
    } else if (s.n_split > 1) {
        const size_t need = (size_t)s.n_split * n_obj_launch * c.n_freq * 4 * elem_size(c);
        lsp_status e = ensure(p, p->sums, need);
        if (e != LSP_OK) return e;
        sums = p->sums.ptr;
    }
    const bool combine = s.n_split > 1 && !ext_sums && !fixup;    // FMA-pipe / direct kernels: partial sums + lsp_combine_kernel
    const bool fused_gls = tensor && opt.gls == 2;                // powers and argmax partials come straight from the epilogue
    *n_parts_out = fused_gls ? s.n_tiles : (combine || ext_sums) ? n_cparts : (fixup ? s.n_tiles * kTcFixParts : s.n_tiles);
    if (want_best) {     // partials are indexed by the launch-local object: each launch's finalize follows it in-stream
        lsp_status e = ensure(p, p->partials, (size_t)n_obj_launch * (size_t)*n_parts_out * sizeof(Best));
        if (e != LSP_OK) return e;
    }

    Best* partials = want_best ? (Best*)p->partials.ptr : nullptr;

    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    if (p->timing) {
        if (p->t_used == p->t_start.size()) {
            cudaEvent_t a, b;
            LSP_CUDA(p, cudaEventCreate(&a));
            LSP_CUDA(p, cudaEventCreate(&b));
            p->t_start.push_back(a);
            p->t_stop.push_back(b);
        }
        ev0 = p->t_start[p->t_used];
        ev1 = p->t_stop[p->t_used];
        ++p->t_used;
        LSP_CUDA(p, cudaEventRecord(ev0, st));
    }
    cudaError_t e;
    void* main_out = (sums && !fused_gls) ? nullptr : out;       // kernels write partial sums instead of powers iff `sums` is set
    Best* main_partials = (sums && !fused_gls) ? nullptr : partials;
    if (c.dtype == LSP_F32) {
        const void* kw = opt.w_pass ? nullptr : opt.wgt;         // the w pass runs the unweighted instantiations
        e = c.fast_math ? launch_main<float, true>(p, s, gp, n_obj_launch, d_off, d_t, d_y, stats, main_out, main_partials, sums, st, kw, opt.gls_yy)
                        : launch_main<float, false>(p, s, gp, n_obj_launch, d_off, d_t, d_y, stats, main_out, main_partials, sums, st, kw, opt.gls_yy);
    } else {
        const void* kw = opt.w_pass ? nullptr : opt.wgt;
        e = launch_main<double, false>(p, s, gp, n_obj_launch, d_off, d_t, d_y, stats, main_out, main_partials, sums, st, kw);
    }
    if (e != cudaSuccess) return fail(p, LSP_ERR_CUDA, "periodogram kernel launch: %s", cudaGetErrorString(e));
    ++p->n_launches;
    if (ev1) LSP_CUDA(p, cudaEventRecord(ev1, st));

    if (fixup) {
        // tensor path: add the splits' partial slots in split order and finish the tiles (steps 5, 6, 6')
        const int64_t grid = n_obj_launch * (int64_t)s.n_tiles * kTcFixParts;
        if (grid > 0x7fffffffLL) return fail(p, LSP_ERR_INVALID_ARG, "batch too large for one launch");
        LSP_CUDA(p, launch_pdl(lsp_tensor_fix_kernel<float>, (unsigned)grid, (unsigned)kTcFixThreads, 0, st, 1, gp, s.tp, d_off,
                               (const TensorObj*)p->tc_objs.ptr, (const float4*)sums, (float*)out, partials, n_obj_launch));
        LSP_CUDA(p, cudaGetLastError());
        ++p->n_launches;
    }
    if (combine) {
        const int64_t grid = n_obj_launch * n_cparts;
        if (c.dtype == LSP_F32)
            lsp_combine_kernel<float><<<(unsigned)grid, kCombineThreads, 0, st>>>(gp, d_off, stats, (const float4*)sums, (float*)out,
                                                                                  partials, n_cparts, n_obj_launch);
        else
            lsp_combine_kernel<double><<<(unsigned)grid, kCombineThreads, 0, st>>>(gp, d_off, stats, (const double4*)sums, (double*)out,
                                                                                   partials, n_cparts, n_obj_launch);
        LSP_CUDA(p, cudaGetLastError());
        ++p->n_launches;
    }
    return LSP_OK;
}

lsp_status run_finalize(lsp_plan* p, int64_t obj_base, int64_t n_obj_launch, int n_parts, const int64_t* d_off,
                        void* d_best_period, void* d_best_power, int64_t* d_best_index, cudaStream_t st)
{
    const lsp_config& c = p->cfg;
    GridParams gp;
    gp.f_min = c.f_min;
    gp.df = (c.f_max - c.f_min) / (double)c.n_freq;
    gp.n_freq = (int)c.n_freq;
    gp.n_tiles = n_parts;
    gp.n_split = 1;
    gp.obj_base = (int)obj_base;
    const int wpb = 4;
    const unsigned grid = (unsigned)((n_obj_launch + wpb - 1) / wpb);
    if (c.dtype == LSP_F32)
        lsp_finalize_best_kernel<float><<<grid, wpb * 32, 0, st>>>(gp, d_off, (const Best*)p->partials.ptr, n_parts, n_obj_launch,
                                                                   (float*)d_best_period, (float*)d_best_power, d_best_index);
    else
        lsp_finalize_best_kernel<double><<<grid, wpb * 32, 0, st>>>(gp, d_off, (const Best*)p->partials.ptr, n_parts, n_obj_launch,
                                                                    (double*)d_best_period, (double*)d_best_power, d_best_index);
    LSP_CUDA(p, cudaGetLastError());
    ++p->n_launches;
    return LSP_OK;
}

// Pre-pass of the factored WS path: tile-independent phasors of every observation on grid `g`, once per call
// (per pass in the generalised mode).
lsp_status build_ws_table(lsp_plan* p, const Schedule& s, const GridSpec& g, const void* d_t, int64_t total_obs, cudaStream_t st)
{
    const lsp_config& c = p->cfg;
    if (s.kernel != LSP_KERNEL_FACTORED) return LSP_OK;
    GridParams gq{};
    gq.f_min = g.f_min;
    gq.df = (g.f_max - g.f_min) / (double)c.n_freq;
    gq.n_freq = (int)c.n_freq;
    p->ws_table_obs = total_obs;
    const size_t bytes = c.dtype == LSP_F32 ? ws_table_bytes<float>(total_obs) : ws_table_bytes<double>(total_obs);
    lsp_status e = ensure(p, p->ws_table, bytes);
    if (e != LSP_OK) return e;
    const int64_t jc = c.dtype == LSP_F32 ? WsCfg<float>::JC : WsCfg<double>::JC;
    const int64_t nl = c.dtype == LSP_F32 ? FactoredCfg<float>::NL : FactoredCfg<double>::NL;
    const int64_t rows = total_obs + jc;
    const unsigned blocks = (unsigned)std::min<int64_t>((rows * (8 + nl) + 255) / 256, (int64_t)p->sm_count * 32);
    if (c.dtype == LSP_F32) {
        float2* v = (float2*)p->ws_table.ptr;
        if (c.fast_math) lsp_ws_table_kernel<float, true><<<blocks, 256, 0, st>>>(gq, (const float*)d_t, total_obs, v, v + rows * 8, v + rows * (8 + nl));
        else lsp_ws_table_kernel<float, false><<<blocks, 256, 0, st>>>(gq, (const float*)d_t, total_obs, v, v + rows * 8, v + rows * (8 + nl));
    } else {
        double2* v = (double2*)p->ws_table.ptr;
        lsp_ws_table_kernel<double, false><<<blocks, 256, 0, st>>>(gq, (const double*)d_t, total_obs, v, v + rows * 8, v + rows * (8 + nl));
    }
    LSP_CUDA(p, cudaGetLastError());
    ++p->n_launches;
    return LSP_OK;
}

lsp_status run_call(lsp_plan* p, int64_t n_obj, const int64_t* d_off, const int64_t* h_off, const void* d_t,
                    const void* d_y, void* out_power, int out_is_host, void* d_best_period, void* d_best_power,
                    int64_t* d_best_index, void* cuda_stream)
{
    if (!p) return LSP_ERR_INVALID_ARG;
    const lsp_config& c = p->cfg;
    p->n_launches = p->n_pairs = p->n_chunks = 0;
    p->t_used = 0;
    p->tensor_shape = p->tensor_products = 0;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (n_obj < 0) return fail(p, LSP_ERR_INVALID_ARG, "n_obj < 0");
    const int n_best = (d_best_period != nullptr) + (d_best_power != nullptr) + (d_best_index != nullptr);
    if (n_best != 0 && n_best != 3) return fail(p, LSP_ERR_INVALID_ARG, "best_period/best_power/best_index: give all three or none");
    const bool want_best = n_best == 3;
    if (n_obj == 0) return LSP_OK;
    if (!out_power && !want_best) return fail(p, LSP_ERR_INVALID_ARG, "no output requested");
    if (!d_off) return fail(p, LSP_ERR_INVALID_ARG, "d_offsets is NULL");
    if (n_obj > 0x7fffffffLL) return fail(p, LSP_ERR_INVALID_ARG, "n_obj too large");
    LSP_CUDA(p, cudaSetDevice(c.device));

    int64_t total_obs;
    std::vector<int64_t> off_cache;      // host copy of the offsets when the caller gave none
    if (h_off) {
        if (h_off[0] != 0) return fail(p, LSP_ERR_INVALID_ARG, "offsets[0] != 0");
        for (int64_t o = 0; o < n_obj; ++o)
            if (h_off[o + 1] < h_off[o]) return fail(p, LSP_ERR_INVALID_ARG, "offsets decrease at object %lld", (long long)o);
        total_obs = h_off[n_obj];
    } else if (n_obj < (1 << 17)) {
        // one synchronous read-back of the whole (small) array instead of its last element now and the rest later (the
        // two-product tensor mode and the table-budget cuts look at the objects' lengths)
        off_cache.resize((size_t)n_obj + 1);
        LSP_CUDA(p, cudaMemcpyAsync(off_cache.data(), d_off, off_cache.size() * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        LSP_CUDA(p, cudaStreamSynchronize(st));
        total_obs = off_cache[(size_t)n_obj];
        if (total_obs < 0) return fail(p, LSP_ERR_INVALID_ARG, "offsets[n_obj] < 0");
    } else {
        if (!p->h_offsets_pinned) LSP_CUDA(p, cudaMallocHost((void**)&p->h_offsets_pinned, sizeof(int64_t)));
        LSP_CUDA(p, cudaMemcpyAsync(p->h_offsets_pinned, d_off + n_obj, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        LSP_CUDA(p, cudaStreamSynchronize(st));
        total_obs = p->h_offsets_pinned[0];
        if (total_obs < 0) return fail(p, LSP_ERR_INVALID_ARG, "offsets[n_obj] < 0");
    }
    if (total_obs > 0 && (!d_t || !d_y)) return fail(p, LSP_ERR_INVALID_ARG, "d_t / d_y is NULL");

    const Schedule s = make_schedule(p, n_obj, total_obs);
    p->kernel_used = s.kernel;
    p->n_split = s.n_split;
    p->n_pairs = total_obs * c.n_freq;

    if (c.center || c.normalize) {
        lsp_status e = ensure(p, p->stats, (size_t)n_obj * sizeof(ObjStats));
        if (e != LSP_OK) return e;
        if (c.dtype == LSP_F32)
            lsp_object_stats_kernel<float><<<(unsigned)n_obj, 128, 0, st>>>(d_off, (const float*)d_y, (ObjStats*)p->stats.ptr, c.center, c.normalize);
        else
            lsp_object_stats_kernel<double><<<(unsigned)n_obj, 128, 0, st>>>(d_off, (const double*)d_y, (ObjStats*)p->stats.ptr, c.center, c.normalize);
        LSP_CUDA(p, cudaGetLastError());
        ++p->n_launches;
    }

    const GridSpec g = plan_grid(c);
    {
        lsp_status e = build_ws_table(p, s, g, d_t, total_obs, st);
        if (e != LSP_OK) return e;
    }

    const size_t es = elem_size(c);
    const size_t row_bytes = (size_t)c.n_freq * es;
    // Host copy of the offsets (large batches without one: fetched only when needed).
    auto host_offsets = [&]() -> const int64_t* {
        if (h_off) return h_off;
        if (off_cache.empty()) {
            off_cache.resize((size_t)n_obj + 1);
            if (cudaMemcpyAsync(off_cache.data(), d_off, off_cache.size() * sizeof(int64_t), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                cudaStreamSynchronize(st) != cudaSuccess) {
                off_cache.clear();
                return nullptr;
            }
        }
        return off_cache.data();
    };
    // Steps 2-6' for objects [o0, o0 + no) holding `obs` observations, asynchronous on the caller's stream: `out` (device, may be
    // NULL) receives rows relative to o0.  One launch sequence, except on the tensor path when the B-operand table of the range
    // would exceed its memory budget: then the objects go in sub-ranges (same results: an object's sums never span launches).
    // two-product tensor mode (opt-in): the CALL's shortest object decides for every launch of the call (kTcMinNtTwoProducts), so
    // chunks, table-budget sub-ranges and the uncut device call give the same bits; needs the offsets on the host
    const bool need_min_nt = s.kernel == LSP_KERNEL_TENSOR && s.products == 2;
    if (need_min_nt && !host_offsets()) return fail(p, LSP_ERR_CUDA, "reading offsets back failed");
    const int64_t call_min_nt = need_min_nt ? range_min_nt(host_offsets(), 0, n_obj) : INT64_MAX;
    auto min_nt_of = [&](int64_t, int64_t) { return call_min_nt; };
    auto run_objs = [&](int64_t o0, int64_t no, int64_t obs, void* out) -> lsp_status {
        int n_parts = 0;
        const Schedule sc = make_schedule(p, no, obs, s.kernel, min_nt_of(o0, no));
        const bool cut = s.kernel == LSP_KERNEL_TENSOR &&
                         (size_t)(obs / kTcKB + no) * (size_t)sc.tp.b_stage_bytes > p->tc_table_budget;
        if (!cut) {
            lsp_status e = run_range(p, sc, g, o0, no, obs, d_off, d_t, d_y, out, want_best, &n_parts, st);
            if (e != LSP_OK) return e;
            return want_best ? run_finalize(p, o0, no, n_parts, d_off, d_best_period, d_best_power, d_best_index, st) : LSP_OK;
        }
        const int64_t* ho = host_offsets();
        if (!ho) return fail(p, LSP_ERR_CUDA, "reading offsets back failed");
        const int64_t kb_cap = (int64_t)(p->tc_table_budget / (size_t)sc.tp.b_stage_bytes);
        for (int64_t a0 = o0; a0 < o0 + no;) {
            int64_t na = 0, kbs = 0;
            while (a0 + na < o0 + no) {
                const int64_t k = tc_n_kb(ho[a0 + na + 1] - ho[a0 + na]) + 1;      // + 1: the table's per-object slack block
                if (na > 0 && kbs + k > kb_cap) break;
                kbs += k;
                ++na;
            }
            const int64_t obs_a = ho[a0 + na] - ho[a0];
            const Schedule sa = make_schedule(p, na, obs_a, s.kernel, min_nt_of(a0, na));
            lsp_status e = run_range(p, sa, g, a0, na, obs_a, d_off, d_t, d_y,
                                     out ? (char*)out + (size_t)(a0 - o0) * row_bytes : nullptr, want_best, &n_parts, st);
            if (e != LSP_OK) return e;
            if (want_best && (e = run_finalize(p, a0, na, n_parts, d_off, d_best_period, d_best_power, d_best_index, st)) != LSP_OK) return e;
            a0 += na;
        }
        return LSP_OK;
    };
    if (!out_power || !out_is_host) return run_objs(0, n_obj, total_obs, out_power);

    // ---- step 7: chunked compute -> event -> copy streams -> (pinned) host -------------------
    const size_t chunk_bytes = c.chunk_bytes > 0 ? (size_t)c.chunk_bytes : ((size_t)64 << 20);
    const int64_t objs_per_chunk = std::max<int64_t>(1, (int64_t)(chunk_bytes / row_bytes));
    const size_t slot_bytes = (size_t)objs_per_chunk * row_bytes;
    const int n_slots = (int)p->slot_ready.size();
    {
        lsp_status e = ensure(p, p->ring, slot_bytes * n_slots);
        if (e != LSP_OK) return e;
    }
    // A pinned (or registered) destination is written directly by the async copies.  A pageable one is either handed to
    // cudaMemcpyAsync as it is (the driver stages it; default) or goes the paper's way (L117; LSP_FLAG_PAGEABLE_STAGED): D2H into a
    // pinned staging slot, then a host-side memcpy into the caller's buffer run by the copy stream's callback thread, the
    // slot's "free" event covering both the device slot and its staging twin.  Measured on config 4 (4 GB): pinned 76 ms,
    // pageable plain 229 ms, pageable staged 283 ms -- the callback threads' memcpy (~14 GB/s) is slower than the driver's
    // own staging on this host, the opposite of the paper's Pascal-era result (Fig. 8: up to 1.91x for staging).
    bool staged = false;
    {
        cudaPointerAttributes attr{};
        const cudaError_t pe = cudaPointerGetAttributes(&attr, out_power);
        if (pe != cudaSuccess) cudaGetLastError();
        staged = (pe != cudaSuccess || attr.type == cudaMemoryTypeUnregistered) && p->pageable_mode == 0;
    }
    if (staged) {
        if (p->stage_host_bytes < slot_bytes * n_slots) {
            if (p->stage_host) LSP_CUDA(p, cudaFreeHost(p->stage_host));
            p->stage_host = nullptr;
            p->stage_host_bytes = 0;
            LSP_CUDA(p, cudaMallocHost(&p->stage_host, slot_bytes * n_slots));
            p->stage_host_bytes = slot_bytes * n_slots;
        }
        p->host_copies.assign((size_t)((n_obj + objs_per_chunk - 1) / objs_per_chunk), lsp_plan::HostCopy{});
    }
    std::fill(p->slot_used.begin(), p->slot_used.end(), 0);
    // a chunk's schedule is made for the chunk's own object and observation counts (so small chunks still split observations
    // and the tensor path's operand table is sized for the chunk, not the batch): the offsets are needed on the host
    const int64_t* ho = (n_obj > objs_per_chunk) ? host_offsets() : nullptr;
    if (n_obj > objs_per_chunk && !ho) return fail(p, LSP_ERR_CUDA, "reading offsets back failed");
    int64_t chunk = 0;
    for (int64_t o0 = 0; o0 < n_obj; o0 += objs_per_chunk, ++chunk) {
        const int64_t no = std::min(objs_per_chunk, n_obj - o0);
        const int slot = (int)(chunk % n_slots);
        char* dslot = (char*)p->ring.ptr + (size_t)slot * slot_bytes;
        if (p->slot_used[slot]) LSP_CUDA(p, cudaStreamWaitEvent(st, p->slot_free[slot], 0));
        lsp_status e = run_objs(o0, no, ho ? ho[o0 + no] - ho[o0] : total_obs, dslot);
        if (e != LSP_OK) return e;
        LSP_CUDA(p, cudaEventRecord(p->slot_ready[slot], st));
        cudaStream_t cs = p->copy_streams[chunk % p->copy_streams.size()];
        LSP_CUDA(p, cudaStreamWaitEvent(cs, p->slot_ready[slot], 0));
        if (staged) {
            char* hslot = (char*)p->stage_host + (size_t)slot * slot_bytes;
            LSP_CUDA(p, cudaMemcpyAsync(hslot, dslot, (size_t)no * row_bytes, cudaMemcpyDeviceToHost, cs));
            lsp_plan::HostCopy& hc = p->host_copies[(size_t)chunk];
            hc.dst = (char*)out_power + (size_t)o0 * row_bytes;
            hc.src = hslot;
            hc.bytes = (size_t)no * row_bytes;
            LSP_CUDA(p, cudaLaunchHostFunc(cs, [](void* u) {
                const lsp_plan::HostCopy* h = (const lsp_plan::HostCopy*)u;
                memcpy(h->dst, h->src, h->bytes);
            }, &hc));
        } else {
            LSP_CUDA(p, cudaMemcpyAsync((char*)out_power + (size_t)o0 * row_bytes, dslot, (size_t)no * row_bytes,
                                        cudaMemcpyDeviceToHost, cs));
        }
        LSP_CUDA(p, cudaEventRecord(p->slot_free[slot], cs));
        p->slot_used[slot] = 1;
    }
    p->n_chunks = chunk;
    for (cudaStream_t cs : p->copy_streams) LSP_CUDA(p, cudaStreamSynchronize(cs));
    return LSP_OK;
}

}  // namespace

// =============================================================================================================
extern "C" {

lsp_status lsp_plan_create(const lsp_config* cfg, lsp_plan** out_plan)
{
    if (out_plan) *out_plan = nullptr;
    if (!cfg || !out_plan) return fail(nullptr, LSP_ERR_INVALID_ARG, "cfg / out_plan is NULL");
    if (!(cfg->f_min > 0.0) || !(cfg->f_max > cfg->f_min) || !std::isfinite(cfg->f_max))
        return fail(nullptr, LSP_ERR_INVALID_ARG, "need 0 < f_min < f_max (got %g, %g)", cfg->f_min, cfg->f_max);
    if (cfg->n_freq < 1 || cfg->n_freq > 0x7fffffffLL) return fail(nullptr, LSP_ERR_INVALID_ARG, "n_freq out of range");
    if (cfg->dtype != LSP_F32 && cfg->dtype != LSP_F64) return fail(nullptr, LSP_ERR_INVALID_ARG, "unknown dtype");
    if (cfg->fast_math != 0 && cfg->fast_math != 1) return fail(nullptr, LSP_ERR_INVALID_ARG, "fast_math must be 0 or 1");
    if (cfg->fast_math && cfg->dtype == LSP_F64)
        return fail(nullptr, LSP_ERR_INVALID_ARG, "fast_math (MUFU sincos) is FP32-only");
    if (cfg->kernel < LSP_KERNEL_AUTO || cfg->kernel > LSP_KERNEL_TENSOR) return fail(nullptr, LSP_ERR_INVALID_ARG, "unknown kernel");
    if (cfg->kernel == LSP_KERNEL_TENSOR && cfg->dtype != LSP_F32)
        return fail(nullptr, LSP_ERR_INVALID_ARG, "the tensor-core kernel is FP32-mode only (FP16-split operands, FP32 accumulation)");
    if (cfg->flags & ~LSP_FLAG_PAGEABLE_STAGED) return fail(nullptr, LSP_ERR_INVALID_ARG, "unknown bit in flags");
    if (cfg->table_budget_bytes < 0) return fail(nullptr, LSP_ERR_INVALID_ARG, "table_budget_bytes < 0");
    if (cfg->tensor_roles < 0 || cfg->tensor_roles > 2) return fail(nullptr, LSP_ERR_INVALID_ARG, "tensor_roles must be 0, 1 or 2");
    if (cfg->tensor_b_stages != 0 && (cfg->tensor_b_stages < 2 || cfg->tensor_b_stages > 8))
        return fail(nullptr, LSP_ERR_INVALID_ARG, "tensor_b_stages must be 0 or 2..8");
    if (cfg->tensor_products != 0 && cfg->tensor_products != 2 && cfg->tensor_products != 3)
        return fail(nullptr, LSP_ERR_INVALID_ARG, "tensor_products must be 0, 2 or 3");
    if (cfg->tensor_pair < 0 || cfg->tensor_pair > 2) return fail(nullptr, LSP_ERR_INVALID_ARG, "tensor_pair must be 0, 1 or 2");
    if (cfg->n_copy_streams < 0 || cfg->n_copy_streams > 16 || cfg->chunk_bytes < 0 || cfg->max_objects < 0 || cfg->max_total_obs < 0)
        return fail(nullptr, LSP_ERR_INVALID_ARG, "negative / oversized sizing field");
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev <= 0) {
        cudaGetLastError();
        return fail(nullptr, LSP_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    }
    if (cfg->device < 0 || cfg->device >= n_dev) return fail(nullptr, LSP_ERR_INVALID_ARG, "device ordinal out of range");
    lsp_plan* p = new (std::nothrow) lsp_plan;
    if (!p) return fail(nullptr, LSP_ERR_OOM, "host allocation failed");
    p->cfg = *cfg;
    if (p->cfg.n_copy_streams == 0) p->cfg.n_copy_streams = 3;
    auto bail = [&](lsp_status st) {
        g_create_error = p->error;
        lsp_destroy(p);
        return st;
    };
#define LSP_CREATE_CUDA(call)                                                                   \
    do {                                                                                        \
        cudaError_t e_ = (call);                                                                \
        if (e_ != cudaSuccess) {                                                                \
            p->error = std::string(#call) + ": " + cudaGetErrorString(e_);                      \
            return bail(e_ == cudaErrorMemoryAllocation ? LSP_ERR_OOM : LSP_ERR_CUDA);          \
        }                                                                                       \
    } while (0)
    LSP_CREATE_CUDA(cudaSetDevice(cfg->device));
    cudaDeviceProp prop;
    LSP_CREATE_CUDA(cudaGetDeviceProperties(&prop, cfg->device));
    if (prop.major < 10) {
        p->error = "device is not sm_100 class (this library is built for sm_100a only)";
        return bail(LSP_ERR_UNSUPPORTED);
    }
    p->sm_count = prop.multiProcessorCount;
    p->smem_optin = (int)prop.sharedMemPerBlockOptin;
    if (cfg->table_budget_bytes > 0) p->tc_table_budget = (size_t)cfg->table_budget_bytes;
    p->pageable_mode = (cfg->flags & LSP_FLAG_PAGEABLE_STAGED) ? 0 : 1;
    p->tc_roles = cfg->tensor_roles;
    p->tc_products = cfg->tensor_products == 2 ? 2 : 3;            // three products unless the caller opts in to two
    p->tc_pair = cfg->tensor_pair;
    if (cfg->tensor_b_stages > 0) p->tc_stages_b = cfg->tensor_b_stages;
    const int n_slots = p->cfg.n_copy_streams + 1;
    for (int i = 0; i < p->cfg.n_copy_streams; ++i) {
        cudaStream_t s;
        LSP_CREATE_CUDA(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
        p->copy_streams.push_back(s);
    }
    for (int i = 0; i < n_slots; ++i) {
        cudaEvent_t a, b;
        LSP_CREATE_CUDA(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
        p->slot_ready.push_back(a);
        LSP_CREATE_CUDA(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
        p->slot_free.push_back(b);
    }
    p->slot_used.assign(n_slots, 0);
    if (ensure(p, p->counter, 64) != LSP_OK) return bail(LSP_ERR_OOM);
    if (cfg->max_objects > 0) {
        const int tile = cfg->dtype == LSP_F32 ? fac_tile<float>() : fac_tile<double>();
        const size_t parts = (size_t)std::max<int64_t>((cfg->n_freq + tile - 1) / tile,
                                                       (cfg->n_freq + kDirectThreads - 1) / kDirectThreads);
        if (ensure(p, p->partials, (size_t)cfg->max_objects * parts * sizeof(Best)) != LSP_OK) return bail(LSP_ERR_OOM);
        if (ensure(p, p->stats, (size_t)cfg->max_objects * sizeof(ObjStats)) != LSP_OK) return bail(LSP_ERR_OOM);
    }
#undef LSP_CREATE_CUDA
    *out_plan = p;
    return LSP_OK;
}

lsp_status lsp_periodogram_batched(lsp_plan* plan, int64_t n_obj, const int64_t* d_offsets, const int64_t* h_offsets,
                                   const void* d_t, const void* d_y, void* out_power, int32_t out_is_host,
                                   void* d_best_period, void* d_best_power, int64_t* d_best_index, void* cuda_stream)
{
    if (!plan) return LSP_ERR_INVALID_ARG;
    if (!out_power && n_obj != 0)
        return fail(plan, LSP_ERR_INVALID_ARG, "out_power is NULL (use lsp_best_period for best-only output)");
    return run_call(plan, n_obj, d_offsets, h_offsets, d_t, d_y, out_power, out_is_host, d_best_period, d_best_power,
                    d_best_index, cuda_stream);
}

lsp_status lsp_best_period(lsp_plan* plan, int64_t n_obj, const int64_t* d_offsets, const int64_t* h_offsets,
                           const void* d_t, const void* d_y, void* d_best_period, void* d_best_power,
                           int64_t* d_best_index, void* cuda_stream)
{
    if (!plan) return LSP_ERR_INVALID_ARG;
    if (!d_best_period || !d_best_power || !d_best_index)
        return fail(plan, LSP_ERR_INVALID_ARG, "best_period, best_power and best_index are all required");
    return run_call(plan, n_obj, d_offsets, h_offsets, d_t, d_y, nullptr, 0, d_best_period, d_best_power, d_best_index,
                    cuda_stream);
}

}  // extern "C"

namespace {
// The generalised call; `out_power` is a device pointer, or (out_is_host) a host pointer filled round by round through the plan's
// chunk ring and copy streams, like step 7 of the standard call.
lsp_status gls_call(lsp_plan* plan, int64_t n_obj, const int64_t* d_offsets, const int64_t* h_offsets,
                    const void* d_t, const void* d_y, const void* d_sigma, void* d_out_power, int out_is_host,
                    void* d_best_period, void* d_best_power, int64_t* d_best_index, void* cuda_stream)
{
    lsp_plan* p = plan;
    if (!p) return LSP_ERR_INVALID_ARG;
    p->n_launches = p->n_pairs = p->n_chunks = 0;
    p->t_used = 0;
    p->tensor_shape = p->tensor_products = 0;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (n_obj < 0) return fail(p, LSP_ERR_INVALID_ARG, "n_obj < 0");
    const int n_best = (d_best_period != nullptr) + (d_best_power != nullptr) + (d_best_index != nullptr);
    if (n_best != 0 && n_best != 3) return fail(p, LSP_ERR_INVALID_ARG, "best_period/best_power/best_index: give all three or none");
    const bool want_best = n_best == 3;
    if (n_obj == 0) return LSP_OK;
    if (!d_out_power && !want_best) return fail(p, LSP_ERR_INVALID_ARG, "no output requested");
    if (!d_offsets) return fail(p, LSP_ERR_INVALID_ARG, "d_offsets is NULL");
    if (n_obj > 0x7fffffffLL) return fail(p, LSP_ERR_INVALID_ARG, "n_obj too large");
    LSP_CUDA(p, cudaSetDevice(p->cfg.device));
    int64_t total_obs;
    if (h_offsets) {
        if (h_offsets[0] != 0) return fail(p, LSP_ERR_INVALID_ARG, "offsets[0] != 0");
        for (int64_t o = 0; o < n_obj; ++o)
            if (h_offsets[o + 1] < h_offsets[o]) return fail(p, LSP_ERR_INVALID_ARG, "offsets decrease at object %lld", (long long)o);
        total_obs = h_offsets[n_obj];
    } else {
        if (!p->h_offsets_pinned) LSP_CUDA(p, cudaMallocHost((void**)&p->h_offsets_pinned, sizeof(int64_t)));
        LSP_CUDA(p, cudaMemcpyAsync(p->h_offsets_pinned, d_offsets + n_obj, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        LSP_CUDA(p, cudaStreamSynchronize(st));
        total_obs = p->h_offsets_pinned[0];
        if (total_obs < 0) return fail(p, LSP_ERR_INVALID_ARG, "offsets[n_obj] < 0");
    }
    if (total_obs > 0 && (!d_t || !d_y || !d_sigma)) return fail(p, LSP_ERR_INVALID_ARG, "d_t / d_y / d_sigma is NULL");

    // Two passes of the standard kernels in their partial-sum form on derived inputs (lsp_gls.cuh): y is already weighted and
    // centred (center / normalize off).  The plan's configuration is never modified.
    const lsp_config& c = p->cfg;
    const size_t es = elem_size(c);
    lsp_status e;
    if ((e = ensure(p, p->gls_x, std::max<size_t>(16, (size_t)2 * total_obs * es))) != LSP_OK) return e;
    if ((e = ensure(p, p->gls_yy, (size_t)n_obj * sizeof(double))) != LSP_OK) return e;
    void* xa = p->gls_x.ptr;
    void* xb = (char*)p->gls_x.ptr + (size_t)total_obs * es;
    if (c.dtype == LSP_F32)
        lsp_gls_prep_kernel<float><<<(unsigned)n_obj, 256, 0, st>>>(d_offsets, (const float*)d_y, (const float*)d_sigma, (float*)xa, (float*)xb, (double*)p->gls_yy.ptr);
    else
        lsp_gls_prep_kernel<double><<<(unsigned)n_obj, 256, 0, st>>>(d_offsets, (const double*)d_y, (const double*)d_sigma, (double*)xa, (double*)xb, (double*)p->gls_yy.ptr);
    LSP_CUDA(p, cudaGetLastError());
    ++p->n_launches;

    Schedule s = make_schedule(p, n_obj, total_obs, -1, INT64_MAX, false);      // (the generalised passes run unpaired)
    if (s.kernel == LSP_KERNEL_TENSOR && s.products == 2) {      // two-product mode: the shortest object decides (kTcMinNtTwoProducts)
        std::vector<int64_t> off_cache;
        const int64_t* ho = h_offsets;
        if (!ho) {
            off_cache.resize((size_t)n_obj + 1);
            LSP_CUDA(p, cudaMemcpyAsync(off_cache.data(), d_offsets, off_cache.size() * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
            LSP_CUDA(p, cudaStreamSynchronize(st));
            ho = off_cache.data();
        }
        s = make_schedule(p, n_obj, total_obs, -1, range_min_nt(ho, 0, n_obj), false);
    }
    if (s.kernel == LSP_KERNEL_TENSOR &&
        (size_t)(total_obs / kTcKB + n_obj) * (size_t)s.tp.b_stage_bytes > p->tc_table_budget) {
        // the tensor path's operand table of the whole batch does not fit: AUTO falls back to the FMA-pipe kernel
        if (c.kernel != LSP_KERNEL_AUTO)
            return fail(p, LSP_ERR_UNSUPPORTED, "generalised mode on the tensor path: batch too large for the operand table (use kernel = factored)");
        s = make_schedule(p, n_obj, total_obs, LSP_KERNEL_FACTORED);
    }
    p->kernel_used = s.kernel;
    p->n_split = s.n_split;
    p->n_pairs = 2 * total_obs * c.n_freq;
    const GridSpec g{c.f_min, c.f_max, 0, 0};
    if ((e = build_ws_table(p, s, g, d_t, total_obs, st)) != LSP_OK) return e;      // FMA-pipe path: one table for both passes
    // objects per round so that the two sums buffers stay within ~12 GB
    // Tensor path, n_split = 1: ZK09's epilogue is fused into the kernel's -- the w pass leaves (C, S) per element (8 bytes, in the
    // epilogue's own order) and the weighted pass reads them back and writes powers / argmax partials itself; nothing else goes
    // through memory.  Otherwise both passes leave partial sums per grid frequency and lsp_gls_combine_kernel finishes.
    const bool fused = s.kernel == LSP_KERNEL_TENSOR && s.n_split == 1;
    const size_t tile_elems = fused ? (size_t)((s.tp.nl + 15) / 16) * 16 * 128 : 0;
    const size_t per_obj = fused ? (size_t)s.n_tiles * tile_elems * sizeof(float2) : (size_t)2 * s.n_split * c.n_freq * 4 * es;
    int64_t objs_per_round = std::max<int64_t>(1, (int64_t)(((size_t)12 << 30) / per_obj));
    const size_t row_bytes = (size_t)c.n_freq * es;
    const int n_cparts = (int)((c.n_freq + kCombineThreads * kCombinePerThread - 1) / (kCombineThreads * kCombinePerThread));
    // host output: a round is a chunk of the ring (step 7: compute into a ring slot, event, D2H on a copy stream, overlapped with
    // the next round's compute)
    const bool to_host = d_out_power && out_is_host;
    const int n_slots = (int)p->slot_ready.size();
    size_t slot_bytes = 0;
    if (to_host) {
        const size_t chunk_bytes = c.chunk_bytes > 0 ? (size_t)c.chunk_bytes : ((size_t)64 << 20);
        objs_per_round = std::min<int64_t>(objs_per_round, std::max<int64_t>(1, (int64_t)(chunk_bytes / row_bytes)));
        slot_bytes = (size_t)objs_per_round * row_bytes;
        if ((e = ensure(p, p->ring, slot_bytes * n_slots)) != LSP_OK) return e;
        std::fill(p->slot_used.begin(), p->slot_used.end(), 0);
    }
    int64_t round = 0;
    for (int64_t o0 = 0; o0 < n_obj; o0 += objs_per_round, ++round) {
        const int64_t no = std::min(objs_per_round, n_obj - o0);
        int n_parts = 0;
        const int slot = (int)(round % n_slots);
        void* const out = !d_out_power ? nullptr
                          : to_host    ? (void*)((char*)p->ring.ptr + (size_t)slot * slot_bytes)
                                       : (void*)((char*)d_out_power + (size_t)o0 * row_bytes);
        if (to_host && p->slot_used[slot]) LSP_CUDA(p, cudaStreamWaitEvent(st, p->slot_free[slot], 0));
        // after this round's kernels: hand the slot to a copy stream
        auto ship = [&]() -> lsp_status {
            if (!to_host) return LSP_OK;
            LSP_CUDA(p, cudaEventRecord(p->slot_ready[slot], st));
            cudaStream_t cs = p->copy_streams[round % p->copy_streams.size()];
            LSP_CUDA(p, cudaStreamWaitEvent(cs, p->slot_ready[slot], 0));
            LSP_CUDA(p, cudaMemcpyAsync((char*)d_out_power + (size_t)o0 * row_bytes, out, (size_t)no * row_bytes, cudaMemcpyDeviceToHost, cs));
            LSP_CUDA(p, cudaEventRecord(p->slot_free[slot], cs));
            p->slot_used[slot] = 1;
            ++p->n_chunks;
            return LSP_OK;
        };
        if (fused) {
            if ((e = ensure(p, p->gls_sums, (size_t)no * per_obj)) != LSP_OK) return e;
            RangeOpts ro;
            ro.ext_sums = p->gls_sums.ptr;
            ro.wgt = xb;
            ro.w_pass = 1;            // first the w pass (its launch also runs the pre-pass: y = w (y - ybar), aux w)
            ro.gls = 1;
            if ((e = run_range(p, s, g, o0, no, total_obs, d_offsets, d_t, xa, nullptr, false, &n_parts, st, ro)) != LSP_OK) return e;
            ro.w_pass = 0;
            ro.skip_prepass = 1;
            ro.gls = 2;
            ro.gls_yy = (const double*)p->gls_yy.ptr;
            if ((e = run_range(p, s, g, o0, no, total_obs, d_offsets, d_t, xa, out, want_best, &n_parts, st, ro)) != LSP_OK) return e;
            if (want_best && (e = run_finalize(p, o0, no, n_parts, d_offsets, d_best_period, d_best_power, d_best_index, st)) != LSP_OK) return e;
            if ((e = ship()) != LSP_OK) return e;
            continue;
        }
        const size_t pass_bytes = (size_t)s.n_split * no * c.n_freq * 4 * es;
        if ((e = ensure(p, p->gls_sums, 2 * pass_bytes)) != LSP_OK) return e;
        for (int pass = 0; pass < 2; ++pass) {
            RangeOpts ro;
            ro.ext_sums = (char*)p->gls_sums.ptr + (size_t)pass * pass_bytes;
            ro.wgt = xb;
            ro.w_pass = pass;
            ro.skip_prepass = pass;   // tensor path: pass 2 reuses pass 1's table and statistics
            e = run_range(p, s, g, o0, no, total_obs, d_offsets, d_t, pass == 0 ? xa : xb, nullptr, false, &n_parts, st, ro);
            if (e != LSP_OK) return e;
        }
        GridParams gp;
        gp.f_min = c.f_min;
        gp.df = (c.f_max - c.f_min) / (double)c.n_freq;
        gp.n_freq = (int)c.n_freq;
        gp.n_tiles = s.n_tiles;
        gp.n_split = s.n_split;
        gp.obj_base = (int)o0;
        if (want_best && (e = ensure(p, p->partials, (size_t)no * n_cparts * sizeof(Best))) != LSP_OK) return e;
        Best* partials = want_best ? (Best*)p->partials.ptr : nullptr;
        const int64_t grid = no * n_cparts;
        if (c.dtype == LSP_F32) {
            const float4* sa = (const float4*)p->gls_sums.ptr;
            lsp_gls_combine_kernel<float><<<(unsigned)grid, kCombineThreads, 0, st>>>(gp, (const double*)p->gls_yy.ptr, sa,
                sa + pass_bytes / sizeof(float4), (float*)out, partials, n_cparts, no);
        } else {
            const double4* sa = (const double4*)p->gls_sums.ptr;
            lsp_gls_combine_kernel<double><<<(unsigned)grid, kCombineThreads, 0, st>>>(gp, (const double*)p->gls_yy.ptr, sa,
                sa + pass_bytes / sizeof(double4), (double*)out, partials, n_cparts, no);
        }
        LSP_CUDA(p, cudaGetLastError());
        ++p->n_launches;
        if (want_best && (e = run_finalize(p, o0, no, n_cparts, d_offsets, d_best_period, d_best_power, d_best_index, st)) != LSP_OK) return e;
        if ((e = ship()) != LSP_OK) return e;
    }
    if (to_host)
        for (cudaStream_t cs : p->copy_streams) LSP_CUDA(p, cudaStreamSynchronize(cs));
    return LSP_OK;
}
}  // namespace

extern "C" {

lsp_status lsp_periodogram_generalized(lsp_plan* plan, int64_t n_obj, const int64_t* d_offsets, const int64_t* h_offsets,
                                       const void* d_t, const void* d_y, const void* d_sigma, void* d_out_power,
                                       void* d_best_period, void* d_best_power, int64_t* d_best_index, void* cuda_stream)
{
    return gls_call(plan, n_obj, d_offsets, h_offsets, d_t, d_y, d_sigma, d_out_power, 0, d_best_period, d_best_power, d_best_index,
                    cuda_stream);
}

lsp_status lsp_periodogram_generalized_host(lsp_plan* plan, int64_t n_obj, const int64_t* h_offsets, const void* h_t,
                                            const void* h_y, const void* h_sigma, void* h_out_power, void* h_best_period,
                                            void* h_best_power, int64_t* h_best_index, void* cuda_stream)
{
    lsp_plan* p = plan;
    if (!p) return LSP_ERR_INVALID_ARG;
    const lsp_config& c = p->cfg;
    if (n_obj < 0) return fail(p, LSP_ERR_INVALID_ARG, "n_obj < 0");
    const int n_best = (h_best_period != nullptr) + (h_best_power != nullptr) + (h_best_index != nullptr);
    if (n_best != 0 && n_best != 3) return fail(p, LSP_ERR_INVALID_ARG, "best_period/best_power/best_index: give all three or none");
    if (!h_out_power && n_best == 0) return fail(p, LSP_ERR_INVALID_ARG, "no output requested");
    p->n_launches = p->n_pairs = p->n_chunks = 0;
    if (n_obj == 0) return LSP_OK;
    if (!h_offsets) return fail(p, LSP_ERR_INVALID_ARG, "h_offsets is NULL");
    if (h_offsets[0] != 0) return fail(p, LSP_ERR_INVALID_ARG, "offsets[0] != 0");
    for (int64_t o = 0; o < n_obj; ++o)
        if (h_offsets[o + 1] < h_offsets[o]) return fail(p, LSP_ERR_INVALID_ARG, "offsets decrease at object %lld", (long long)o);
    const int64_t total_obs = h_offsets[n_obj];
    if (total_obs > 0 && (!h_t || !h_y || !h_sigma)) return fail(p, LSP_ERR_INVALID_ARG, "h_t / h_y / h_sigma is NULL");
    LSP_CUDA(p, cudaSetDevice(c.device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t es = elem_size(c);
    lsp_status e;
    if ((e = ensure(p, p->in_off, (size_t)(n_obj + 1) * sizeof(int64_t))) != LSP_OK) return e;
    if ((e = ensure(p, p->in_t, std::max<size_t>(16, (size_t)total_obs * es))) != LSP_OK) return e;
    if ((e = ensure(p, p->in_y, std::max<size_t>(16, (size_t)total_obs * es))) != LSP_OK) return e;
    if ((e = ensure(p, p->in_sigma, std::max<size_t>(16, (size_t)total_obs * es))) != LSP_OK) return e;
    LSP_CUDA(p, cudaMemcpyAsync(p->in_off.ptr, h_offsets, (size_t)(n_obj + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    if (total_obs > 0) {
        LSP_CUDA(p, cudaMemcpyAsync(p->in_t.ptr, h_t, (size_t)total_obs * es, cudaMemcpyHostToDevice, st));
        LSP_CUDA(p, cudaMemcpyAsync(p->in_y.ptr, h_y, (size_t)total_obs * es, cudaMemcpyHostToDevice, st));
        LSP_CUDA(p, cudaMemcpyAsync(p->in_sigma.ptr, h_sigma, (size_t)total_obs * es, cudaMemcpyHostToDevice, st));
    }
    char* d_bper = nullptr;
    char* d_bpow = nullptr;
    int64_t* d_bidx = nullptr;
    if (n_best) {
        if ((e = ensure(p, p->out_best, (size_t)n_obj * (2 * es + sizeof(int64_t)))) != LSP_OK) return e;
        d_bidx = (int64_t*)p->out_best.ptr;
        d_bper = (char*)p->out_best.ptr + (size_t)n_obj * sizeof(int64_t);
        d_bpow = d_bper + (size_t)n_obj * es;
    }
    e = gls_call(p, n_obj, (const int64_t*)p->in_off.ptr, h_offsets, p->in_t.ptr, p->in_y.ptr, p->in_sigma.ptr, h_out_power,
                 h_out_power ? 1 : 0, d_bper, d_bpow, d_bidx, cuda_stream);
    if (e != LSP_OK) return e;
    if (n_best) {
        LSP_CUDA(p, cudaMemcpyAsync(h_best_index, d_bidx, (size_t)n_obj * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        LSP_CUDA(p, cudaMemcpyAsync(h_best_period, d_bper, (size_t)n_obj * es, cudaMemcpyDeviceToHost, st));
        LSP_CUDA(p, cudaMemcpyAsync(h_best_power, d_bpow, (size_t)n_obj * es, cudaMemcpyDeviceToHost, st));
    }
    LSP_CUDA(p, cudaStreamSynchronize(st));
    return LSP_OK;
}

lsp_status lsp_periodogram_batched_host(lsp_plan* plan, int64_t n_obj, const int64_t* h_offsets, const void* h_t,
                                        const void* h_y, void* h_out_power, void* h_best_period, void* h_best_power,
                                        int64_t* h_best_index, void* cuda_stream)
{
    lsp_plan* p = plan;
    if (!p) return LSP_ERR_INVALID_ARG;
    const lsp_config& c = p->cfg;
    if (n_obj < 0) return fail(p, LSP_ERR_INVALID_ARG, "n_obj < 0");
    const int n_best = (h_best_period != nullptr) + (h_best_power != nullptr) + (h_best_index != nullptr);
    if (n_best != 0 && n_best != 3) return fail(p, LSP_ERR_INVALID_ARG, "best_period/best_power/best_index: give all three or none");
    if (!h_out_power && n_best == 0) return fail(p, LSP_ERR_INVALID_ARG, "no output requested");
    p->n_launches = p->n_pairs = p->n_chunks = 0;
    if (n_obj == 0) return LSP_OK;
    if (!h_offsets) return fail(p, LSP_ERR_INVALID_ARG, "h_offsets is NULL");
    if (h_offsets[0] != 0) return fail(p, LSP_ERR_INVALID_ARG, "offsets[0] != 0");
    for (int64_t o = 0; o < n_obj; ++o)
        if (h_offsets[o + 1] < h_offsets[o]) return fail(p, LSP_ERR_INVALID_ARG, "offsets decrease at object %lld", (long long)o);
    const int64_t total_obs = h_offsets[n_obj];
    if (total_obs > 0 && (!h_t || !h_y)) return fail(p, LSP_ERR_INVALID_ARG, "h_t / h_y is NULL");
    LSP_CUDA(p, cudaSetDevice(c.device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t es = elem_size(c);
    lsp_status e;
    if ((e = ensure(p, p->in_off, (size_t)(n_obj + 1) * sizeof(int64_t))) != LSP_OK) return e;
    if ((e = ensure(p, p->in_t, std::max<size_t>(16, (size_t)total_obs * es))) != LSP_OK) return e;
    if ((e = ensure(p, p->in_y, std::max<size_t>(16, (size_t)total_obs * es))) != LSP_OK) return e;
    LSP_CUDA(p, cudaMemcpyAsync(p->in_off.ptr, h_offsets, (size_t)(n_obj + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    if (total_obs > 0) {
        LSP_CUDA(p, cudaMemcpyAsync(p->in_t.ptr, h_t, (size_t)total_obs * es, cudaMemcpyHostToDevice, st));
        LSP_CUDA(p, cudaMemcpyAsync(p->in_y.ptr, h_y, (size_t)total_obs * es, cudaMemcpyHostToDevice, st));
    }
    char* d_bper = nullptr;
    char* d_bpow = nullptr;
    int64_t* d_bidx = nullptr;
    if (n_best) {
        if ((e = ensure(p, p->out_best, (size_t)n_obj * (2 * es + sizeof(int64_t)))) != LSP_OK) return e;
        d_bidx = (int64_t*)p->out_best.ptr;                       // int64 first: keeps every array aligned
        d_bper = (char*)p->out_best.ptr + (size_t)n_obj * sizeof(int64_t);
        d_bpow = d_bper + (size_t)n_obj * es;
    }
    e = run_call(p, n_obj, (const int64_t*)p->in_off.ptr, h_offsets, p->in_t.ptr, p->in_y.ptr, h_out_power,
                 h_out_power ? 1 : 0, d_bper, d_bpow, d_bidx, cuda_stream);
    if (e != LSP_OK) return e;
    if (n_best) {
        LSP_CUDA(p, cudaMemcpyAsync(h_best_index, d_bidx, (size_t)n_obj * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        LSP_CUDA(p, cudaMemcpyAsync(h_best_period, d_bper, (size_t)n_obj * es, cudaMemcpyDeviceToHost, st));
        LSP_CUDA(p, cudaMemcpyAsync(h_best_power, d_bpow, (size_t)n_obj * es, cudaMemcpyDeviceToHost, st));
    }
    LSP_CUDA(p, cudaStreamSynchronize(st));
    return LSP_OK;
}

lsp_status lsp_best_merge(lsp_plan* plan, int64_t n_obj, int32_t n_parts, const void* d_part_power,
                          const int64_t* d_part_index, void* d_best_period, void* d_best_power, int64_t* d_best_index,
                          void* cuda_stream)
{
    lsp_plan* p = plan;
    if (!p) return LSP_ERR_INVALID_ARG;
    if (n_obj < 0 || n_parts < 1) return fail(p, LSP_ERR_INVALID_ARG, "n_obj < 0 or n_parts < 1");
    if (n_obj == 0) return LSP_OK;
    if (!d_part_power || !d_part_index || !d_best_period || !d_best_power || !d_best_index)
        return fail(p, LSP_ERR_INVALID_ARG, "lsp_best_merge: NULL argument");
    const lsp_config& c = p->cfg;
    LSP_CUDA(p, cudaSetDevice(c.device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    GridParams gp{};
    gp.f_min = c.f_min;
    gp.df = (c.f_max - c.f_min) / (double)c.n_freq;
    gp.n_freq = (int)c.n_freq;
    const unsigned grid = (unsigned)((n_obj + 127) / 128);
    if (c.dtype == LSP_F32)
        lsp_merge_best_kernel<float><<<grid, 128, 0, st>>>(gp, (const float*)d_part_power, d_part_index, n_parts, n_obj,
                                                          (float*)d_best_period, (float*)d_best_power, d_best_index);
    else
        lsp_merge_best_kernel<double><<<grid, 128, 0, st>>>(gp, (const double*)d_part_power, d_part_index, n_parts, n_obj,
                                                           (double*)d_best_period, (double*)d_best_power, d_best_index);
    LSP_CUDA(p, cudaGetLastError());
    p->n_launches = 1;
    return LSP_OK;
}

void lsp_destroy(lsp_plan* p)
{
    if (!p) return;
    cudaSetDevice(p->cfg.device);
    for (cudaStream_t s : p->copy_streams) {
        cudaStreamSynchronize(s);
        cudaStreamDestroy(s);
    }
    for (cudaEvent_t e : p->slot_ready) cudaEventDestroy(e);
    for (cudaEvent_t e : p->slot_free) cudaEventDestroy(e);
    for (cudaEvent_t e : p->t_start) cudaEventDestroy(e);
    for (cudaEvent_t e : p->t_stop) cudaEventDestroy(e);
    for (DeviceBuffer* b : {&p->ring, &p->partials, &p->sums, &p->stats, &p->counter, &p->ws_table, &p->gls_x, &p->gls_yy, &p->gls_sums, &p->tc_objs, &p->tc_table, &p->in_off, &p->in_t, &p->in_y, &p->in_sigma, &p->out_best})
        if (b->ptr) cudaFree(b->ptr);
    if (p->h_offsets_pinned) cudaFreeHost(p->h_offsets_pinned);
    if (p->stage_host) cudaFreeHost(p->stage_host);
    cudaGetLastError();
    delete p;
}

const char* lsp_last_error(const lsp_plan* plan)
{
    return plan ? plan->error.c_str() : g_create_error.c_str();
}

void lsp_last_call_info(const lsp_plan* p, int64_t* n_launches, int64_t* n_pairs, int32_t* kernel_used, int32_t* n_split,
                        int64_t* n_chunks, int32_t* tensor_shape, int32_t* tensor_products)
{
    if (!p) return;
    if (tensor_shape) *tensor_shape = p->tensor_shape;
    if (tensor_products) *tensor_products = p->tensor_products;
    if (n_launches) *n_launches = p->n_launches;
    if (n_pairs) *n_pairs = p->n_pairs;
    if (kernel_used) *kernel_used = p->kernel_used;
    if (n_split) *n_split = p->n_split;
    if (n_chunks) *n_chunks = p->n_chunks;
}

void lsp_set_timing(lsp_plan* p, int32_t on)
{
    if (p) p->timing = on != 0;
}

float lsp_last_kernel_ms(lsp_plan* p)
{
    if (!p || !p->timing || p->t_used == 0) return -1.f;
    float total = 0.f;
    for (size_t i = 0; i < p->t_used; ++i) {
        float ms = 0.f;
        if (cudaEventSynchronize(p->t_stop[i]) != cudaSuccess) return -1.f;
        if (cudaEventElapsedTime(&ms, p->t_start[i], p->t_stop[i]) != cudaSuccess) return -1.f;
        total += ms;
    }
    return total;
}

const char* lsp_version(void)
{
    return "lsp-b200 0.6 (sm_100a; kernels: direct, factored-ffma2, factored-dfma, tensor-tcgen05 (A operands in TMEM, CTA pairs; three FP16 products by default); modes: standard, generalised; allocation-free best period: lsp_best_period_static)";
}

}  // extern "C"

// =============================================================================================================
// lsp_best_period_static: the one entry point that allocates nothing (include/lsp.h says who needs that and why).
//
// It is the best-period route of the direct kernel family -- lsp_object_stats_kernel (only with center / normalize),
// lsp_direct_kernel with the fused argmax, lsp_finalize_best_kernel: the very kernels the plan-based calls launch -- with
// the scratch those kernels need (per-CTA argmax candidates, per-object statistics) taken from the file-scope array below
// instead of plan-owned cudaMalloc memory.  No plan exists on this path, so there are no streams, events or host vectors
// to create either.
namespace {

// The scratch itself.  It lives in the library's device image: each GPU context that loads the library gets its own
// zero-filled copy at load time and keeps it until the process exits.  256-byte alignment keeps both sub-arrays below
// (16-byte elements) naturally aligned and the base on a memory-sector boundary.
static __device__ __align__(256) unsigned char g_static_scratch[LSP_STATIC_SCRATCH_BYTES];

// Host code must never pass `g_static_scratch` itself to a kernel.  On the host that name is only nvcc's handle for the
// symbol -- an ordinary host variable whose address means nothing to the GPU (a kernel given it faults, or on a system where
// the GPU can reach host memory it quietly scribbles over that handle).  The real address is per device and comes from
// cudaGetSymbolAddress, asked once per device while that device is current, and kept here.
constexpr int kStaticMaxDevices = 64;
struct StaticDevice {
    unsigned char* scratch;   // DEVICE address of g_static_scratch on this device; NULL = set-up not done yet
    int sm_count;
};
StaticDevice g_static_devices[kStaticMaxDevices];   // zero-initialised
std::mutex g_static_mutex;                          // guards the table above (first calls from several host threads)

// One-time set-up for `device`; the caller has already made it current.  Two queries, no allocation.
lsp_status static_device_setup(int device, StaticDevice* out)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& d = g_static_devices[device];
    if (!d.scratch) {
        int major = 0, sms = 0;
        LSP_CUDA(nullptr, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
        if (major < 10)
            return fail(nullptr, LSP_ERR_UNSUPPORTED, "device is not sm_100 class (this library is built for sm_100a only)");
        LSP_CUDA(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
        unsigned char* ptr = nullptr;
        LSP_CUDA(nullptr, cudaGetSymbolAddress((void**)&ptr, g_static_scratch));
        if (!ptr) return fail(nullptr, LSP_ERR_CUDA, "cudaGetSymbolAddress returned a NULL address for the static scratch");
        d.sm_count = sms;
        d.scratch = ptr;
    }
    *out = d;
    return LSP_OK;
}

template <typename T, bool FAST>
lsp_status static_launch(const lsp_config& c, const StaticDevice& dev, int64_t n_obj, const int64_t* d_off, const T* d_t,
                         const T* d_y, T* d_best_period, T* d_best_power, int64_t* d_best_index, cudaStream_t st)
{
    using V4 = typename Vec4<T>::type;
    // schedule: as make_schedule does for the direct kernel, with n_split fixed at 1 (partial sums would need N_f-sized scratch)
    const int64_t tiles4 = (c.n_freq + 4 * kDirectThreads - 1) / (4 * kDirectThreads);
    const int r = (n_obj * tiles4 >= (int64_t)dev.sm_count * 8) ? 4 : 1;
    const int64_t n_tiles = (c.n_freq + (int64_t)r * kDirectThreads - 1) / ((int64_t)r * kDirectThreads);
    // scratch layout: ObjStats[n_obj] | Best[n_obj * n_tiles], both 16-byte elements
    static_assert(sizeof(ObjStats) == 16 && sizeof(Best) == 16, "scratch layout assumes 16-byte elements");
    const int64_t need = 16 * n_obj * (n_tiles + 1);
    if (need > (int64_t)LSP_STATIC_SCRATCH_BYTES)      // not reachable past the documented check in the caller; kept as the guard
        return fail(nullptr, LSP_ERR_UNSUPPORTED, "static scratch too small: need %lld bytes, have %lld", (long long)need,
                    (long long)LSP_STATIC_SCRATCH_BYTES);
    ObjStats* stats = (ObjStats*)dev.scratch;
    Best* partials = (Best*)(dev.scratch + (size_t)n_obj * sizeof(ObjStats));
    const bool use_stats = c.center || c.normalize;
    if (use_stats) {
        lsp_object_stats_kernel<T><<<(unsigned)n_obj, 128, 0, st>>>(d_off, d_y, stats, c.center, c.normalize);
        LSP_CUDA(nullptr, cudaGetLastError());
    }
    GridParams gp;
    gp.f_min = c.f_min;
    gp.df = (c.f_max - c.f_min) / (double)c.n_freq;
    gp.n_freq = (int)c.n_freq;
    gp.n_tiles = (int)n_tiles;
    gp.n_split = 1;
    gp.obj_base = 0;
    // Every CTA (object, tile) stores its candidate, and the finalize kernel reads exactly those n_obj * n_tiles slots (and the
    // statistics kernel above wrote the n_obj entries the main kernel reads): whatever an earlier call left in the array is
    // overwritten before it is looked at, so nothing is cleared here.
    const unsigned grid = (unsigned)(n_obj * n_tiles);
    const ObjStats* ks = use_stats ? stats : nullptr;
    if (r == 4)
        lsp_direct_kernel<T, FAST, 4, false><<<grid, kDirectThreads, 0, st>>>(gp, d_off, d_t, d_y, ks, (T*)nullptr, partials,
                                                                             (V4*)nullptr, n_obj, (const T*)nullptr);
    else
        lsp_direct_kernel<T, FAST, 1, false><<<grid, kDirectThreads, 0, st>>>(gp, d_off, d_t, d_y, ks, (T*)nullptr, partials,
                                                                             (V4*)nullptr, n_obj, (const T*)nullptr);
    LSP_CUDA(nullptr, cudaGetLastError());
    const int wpb = 4;
    lsp_finalize_best_kernel<T><<<(unsigned)((n_obj + wpb - 1) / wpb), wpb * 32, 0, st>>>(gp, d_off, partials, (int)n_tiles, n_obj,
                                                                                         d_best_period, d_best_power, d_best_index);
    LSP_CUDA(nullptr, cudaGetLastError());
    return LSP_OK;
}

}  // namespace

extern "C" lsp_status lsp_best_period_static(const lsp_config* cfg, int64_t n_obj, const int64_t* d_offsets, const void* d_t,
                                             const void* d_y, void* d_best_period, void* d_best_power, int64_t* d_best_index,
                                             void* cuda_stream)
{
    if (!cfg) return fail(nullptr, LSP_ERR_INVALID_ARG, "cfg is NULL");
    const lsp_config& c = *cfg;
    if (!(c.f_min > 0.0) || !(c.f_max > c.f_min) || !std::isfinite(c.f_max))
        return fail(nullptr, LSP_ERR_INVALID_ARG, "need 0 < f_min < f_max (got %g, %g)", c.f_min, c.f_max);
    if (c.n_freq < 1 || c.n_freq > 0x7fffffffLL) return fail(nullptr, LSP_ERR_INVALID_ARG, "n_freq out of range");
    if (c.dtype != LSP_F32 && c.dtype != LSP_F64) return fail(nullptr, LSP_ERR_INVALID_ARG, "unknown dtype");
    if (c.fast_math != 0 && c.fast_math != 1) return fail(nullptr, LSP_ERR_INVALID_ARG, "fast_math must be 0 or 1");
    if (c.fast_math && c.dtype == LSP_F64) return fail(nullptr, LSP_ERR_INVALID_ARG, "fast_math (MUFU sincos) is FP32-only");
    if (n_obj < 0) return fail(nullptr, LSP_ERR_INVALID_ARG, "n_obj < 0");
    if (n_obj > 0 && (!d_offsets || !d_t || !d_y || !d_best_period || !d_best_power || !d_best_index))
        return fail(nullptr, LSP_ERR_INVALID_ARG, "lsp_best_period_static: NULL argument (offsets, t, y and all three outputs are required)");
    // the documented limit, checked on the host before any CUDA call: 16 B x n_obj x (ceil(n_freq / 1024) + 1)
    const int64_t tiles_doc = (c.n_freq + 1023) / 1024 + 1;
    const int64_t max_slots = (int64_t)LSP_STATIC_SCRATCH_BYTES / 16;
    if (n_obj > max_slots / tiles_doc)
        return fail(nullptr, LSP_ERR_UNSUPPORTED,
                    "request exceeds the static scratch: n_obj (%lld) x (ceil(n_freq / 1024) + 1 = %lld) x 16 bytes > %lld bytes; "
                    "run the batch as object ranges of at most %lld objects",
                    (long long)n_obj, (long long)tiles_doc, (long long)LSP_STATIC_SCRATCH_BYTES, (long long)(max_slots / tiles_doc));
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev <= 0) {
        cudaGetLastError();
        return fail(nullptr, LSP_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    }
    if (c.device < 0 || c.device >= n_dev || c.device >= kStaticMaxDevices)
        return fail(nullptr, LSP_ERR_INVALID_ARG, "device ordinal out of range");
    LSP_CUDA(nullptr, cudaSetDevice(c.device));
    StaticDevice dev{};
    const lsp_status es = static_device_setup(c.device, &dev);
    if (es != LSP_OK) return es;
    if (n_obj == 0) return LSP_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (c.dtype == LSP_F64)
        return static_launch<double, false>(c, dev, n_obj, d_offsets, (const double*)d_t, (const double*)d_y, (double*)d_best_period,
                                            (double*)d_best_power, d_best_index, st);
    return c.fast_math ? static_launch<float, true>(c, dev, n_obj, d_offsets, (const float*)d_t, (const float*)d_y,
                                                    (float*)d_best_period, (float*)d_best_power, d_best_index, st)
                       : static_launch<float, false>(c, dev, n_obj, d_offsets, (const float*)d_t, (const float*)d_y,
                                                     (float*)d_best_period, (float*)d_best_power, d_best_index, st);
}
