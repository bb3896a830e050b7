/*
 * lsp.h -- C ABI of the B200-native batched Lomb-Scargle periodogram library (liblsp_b200.so).
 *
 * What the library computes (arXiv 2105.04006, section 2):
 *   - time series (t_j, X_j), j = 1..N_t, unevenly sampled, assumed zero-mean
 *   - omega = 2*pi*f; Scargle offset  tan 2 omega tau = sum sin 2 omega t_j / sum cos 2 omega t_j   Eq. 1
 *   - P_LS(f) = 1/2 ( [sum X_j cos omega(t_j-tau)]^2 / sum cos^2 omega(t_j-tau)
 *                   + [sum X_j sin omega(t_j-tau)]^2 / sum sin^2 omega(t_j-tau) )      Eq. 2
 *   - evenly spaced grid on [f_min, f_max): df = (f_max - f_min)/N_f, f_k = f_min + k df, k = 0..N_f-1
 *   - one grid shared by every object of a batch
 *   - FP32 or FP64 selectable
 *   - returning the periodogram is optional; best period = argmax_k P(f_k)
 *   - periodograms returned to the host go through several CUDA streams and pinned memory, overlapped
 *     with the computation of later objects
 *
 * Conventions:
 *   - f is CYCLIC (cycles per unit of t), omega = 2 pi f is formed inside; period = 1/f          (a1)
 *   - f_max itself is not sampled                                                                (a2)
 *   - output is Eq. 2 exactly as printed ("non-normalised"); normalize=1 divides by 1/2 sum y^2   (a3)
 *   - y is used as given; center=1 subtracts the per-object mean first                           (a4)
 *   - argmax: lowest index wins exact ties, NaN never wins                                       (a7)
 *   - the LS period 1/f_k* is returned, never doubled                                            (a8)
 *
 * All entry points are plain C: pointers are labelled HOST or DEVICE, sizes are int64_t, no C++ or
 * torch types cross this boundary.  No entry point throws or aborts; every failure is a status code,
 * with a message available from lsp_last_error().  There is no CPU fallback anywhere: without a CUDA
 * device lsp_plan_create fails with LSP_ERR_CUDA.
 */
#ifndef LSP_B200_H
#define LSP_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lsp_plan lsp_plan; /* opaque; created by lsp_plan_create, freed by lsp_destroy */

typedef enum { LSP_F32 = 0, LSP_F64 = 1 } lsp_dtype;

typedef enum {
    LSP_OK = 0,
    LSP_ERR_INVALID_ARG = 1,
    LSP_ERR_CUDA = 2,
    LSP_ERR_OOM = 3,
    LSP_ERR_UNSUPPORTED = 4
} lsp_status;

/* Which periodogram kernel family runs steps 2-5 of the hot path. */
typedef enum {
    LSP_KERNEL_AUTO = 0,     /* library picks: tensor (FP32) / factored (FP64), direct for grids under 1024 points */
    LSP_KERNEL_DIRECT = 1,   /* one sincos per (t,f) pair, thread = frequency (the paper's Listing 1 shape,
                                PAPER.md:L137-216, with smem staging L121-125 and range-reduced phase)     */
    LSP_KERNEL_FACTORED = 2, /* angle-addition outer product: no sincos in the O(N_t N_f) loop, 4 FMA/pair */
    LSP_KERNEL_TENSOR = 3    /* FP32 mode only: the same contraction on the tensor cores (tcgen05.mma kind::f16, FP32
                                accumulators in TMEM).  Operands are FP16 hi(+lo) pairs, two or three MMAs per product
                                (lsp_config.tensor_products; fast_math = 1: hi only, one MMA, MUFU sincos); phases
                                stay FP64-reduced.                                                                  */
} lsp_kernel;

typedef struct lsp_config {
    double  f_min;          /* cycles per unit of t; 0 < f_min < f_max                                     */
    double  f_max;          /* NOT sampled: last frequency is f_max - df */
    int64_t n_freq;         /* N_f >= 1 (<= 2^31 - 1)                                                      */
    int32_t dtype;          /* lsp_dtype: element type of t, y, power, best_period, best_power             */
    int32_t fast_math;      /* FP32 only: 1 = MUFU.SIN/COS (__sincosf class), 0 = accurate   */
    int32_t normalize;      /* 0 = Eq. 2 as printed; 1 = divide by (1/2) sum_j y_j^2 per object            */
    int32_t center;         /* 0 = y as given (paper: caller centres); 1 = subtract mean */
    int32_t device;         /* CUDA device ordinal                                                         */
    int32_t n_copy_streams; /* D2H streams for host output (paper: 3); 0 = default (3)      */
    int64_t chunk_bytes;    /* device staging chunk for host output (paper: 8 MiB); 0 = library default    */
    int64_t max_objects;    /* scratch sizing hints; 0 = size on first use (scratch grows when needed)     */
    int64_t max_total_obs;
    int32_t kernel;         /* lsp_kernel                                                                  */
    int32_t flags;          /* bit set of LSP_FLAG_*; unknown bits are rejected                            */
    int64_t table_budget_bytes; /* tensor path: cap on the per-launch B-operand table; larger batches run in
                                   object ranges (same results); 0 = library default (12 GiB)              */
    int32_t tensor_roles;   /* tensor path warp-role shape: 0 = chosen by item length, 1 = short-item shape
                                   (8 epilogue warps), 2 = long-item shape (4 epilogue warps)               */
    int32_t tensor_b_stages;/* tensor path: depth of the B-operand (TMA) ring, 2..8; 0 = library default    */
    int32_t tensor_products;/* tensor path, fast_math = 0: FP16 tcgen05 products per multiply-accumulate.
                                   3 (= 0, default): a_hi b_hi + a_hi b_lo + a_lo b_hi -- both operands FP16 pairs
                                   (22 significand bits): within the FP32 tolerance on every cadence tested, ~1e-6 of max P;
                                   2 (opt-in, ~1.35x faster on long objects, no gain on short ones): a_hi (b_hi + b_lo) --
                                   the generated operand a = y e^{i alpha} is ONE FP16 (11 bits).  Its error follows the
                                   conditioning of the 2 x 2 system: <= 4.5e-4 of max P on year-long cadences, but several
                                   1e-3 (over the 1e-3 tolerance) on noise-only objects observed on <= 12 nights inside a
                                   0.05 d window -- choose it only for well-sampled data.  A call that holds
                                   an object of fewer than 32 observations runs with 3 all the same                 */
    int32_t tensor_pair;    /* tensor path: CTA pairs (2-CTA clusters, tcgen05 cta_group::2: two frequency tiles of one
                                   object share every tabulated-operand stage).  0 = when work items are long (>= 48
                                   stages of 16 observations), 1 = never, 2 = whenever the grid has >= 2 tiles         */
} lsp_config;

/* lsp_config.flags */
#define LSP_FLAG_PAGEABLE_STAGED 1 /* host output into PAGEABLE memory goes through a plan-owned pinned staging ring and
                                      host-side copies on the copy streams' callback threads (the paper's scheme,
                                      PAPER.md:L117) instead of plain cudaMemcpyAsync into the pageable buffer      */

/*
 * Create a plan: validates cfg, selects the device, creates the D2H copy streams and events and
 * allocates scratch (argmax partials, split-N_t partial sums, the device chunk ring for host output).
 * The plan owns all of that; the caller owns every buffer passed to the calls below.
 * Errors: LSP_ERR_INVALID_ARG (f_min <= 0, f_max <= f_min, n_freq < 1, fast_math with FP64, unknown
 * enum or flag bit, tensor_roles / tensor_b_stages / tensor_products / tensor_pair out of range), LSP_ERR_CUDA (no device / runtime failure), LSP_ERR_OOM.  *out_plan is NULL on
 * failure.  A plan is not thread-safe; distinct plans are independent.
 */
lsp_status lsp_plan_create(const lsp_config* cfg /* HOST */, lsp_plan** out_plan /* HOST */);

/*
 * Full periodogram of a CSR batch (hot-path steps 1-6, and 7 when the output is on the host;
 * PAPER.md:L85, L103, L109, L113, L117).
 *   n_obj        objects in the batch (>= 0; 1 = the paper's single-object mode)
 *   d_offsets    DEVICE, int64[n_obj+1], offsets[0] = 0, non-decreasing; object o owns [offsets[o], offsets[o+1])
 *   h_offsets    HOST copy of the same array, or NULL (the library then reads offsets back itself:
 *                one small synchronous D2H on the call's stream)
 *   d_t, d_y     DEVICE, offsets[n_obj] elements of cfg.dtype: times and magnitudes, concatenated
 *   out_power    n_obj * n_freq elements of cfg.dtype, row-major by object:
 *                a DEVICE pointer when out_is_host == 0, else a HOST pointer filled through the plan's chunk ring and copy
 *                streams: a pinned (or registered) buffer is written directly by the async copies and overlaps with compute;
 *                a pageable one is handed to cudaMemcpyAsync as it is (works, does not overlap), or, with
 *                LSP_FLAG_PAGEABLE_STAGED in cfg.flags, goes through a plan-owned pinned staging ring and
 *                per-chunk host-side copies run by the copy streams' callback threads (PAPER.md:L117's scheme)
 *   d_best_*     DEVICE, optional (all three NULL or all three non-NULL): per object best period
 *                (cfg.dtype), its power (cfg.dtype) and grid index (int64; -1 and NaN period when N_t = 0)
 *   cuda_stream  cudaStream_t as void* (NULL = default stream).  Device-output calls are asynchronous
 *                on it; host-output calls return after the last chunk has landed in out_power.
 * Errors: LSP_ERR_INVALID_ARG (NULL where required, n_obj < 0, bad offsets when h_offsets is given),
 * LSP_ERR_CUDA, LSP_ERR_OOM.  Outputs are unspecified after an error.
 */
lsp_status lsp_periodogram_batched(lsp_plan* plan, int64_t n_obj,
                                   const int64_t* d_offsets, const int64_t* h_offsets,
                                   const void* d_t, const void* d_y,
                                   void* out_power, int32_t out_is_host,
                                   void* d_best_period, void* d_best_power, int64_t* d_best_index,
                                   void* cuda_stream);

/*
 * Best period per object with the argmax fused into the periodogram kernels: the N_obj x N_f array
 * is never written to memory (space O(N_t + N_o)).  Arguments as above; all three
 * outputs are required.  Asynchronous on cuda_stream.
 */
lsp_status lsp_best_period(lsp_plan* plan, int64_t n_obj,
                           const int64_t* d_offsets, const int64_t* h_offsets,
                           const void* d_t, const void* d_y,
                           void* d_best_period, void* d_best_power, int64_t* d_best_index,
                           void* cuda_stream);

/*
 * Generalised Lomb-Scargle periodogram: floating mean + per-point errors (section 4.11; Zechmeister &
 * Kuerster 2009).  With weights w_j = sigma_j^-2 / sum sigma^-2 the output is the relative chi^2 reduction
 *     P(f_k) = (chi0^2 - chi^2(f_k)) / chi0^2  in [0, 1],
 * chi0^2 of the weighted-mean model, chi^2(f) of the weighted least-squares fit a cos 2 pi f t + b sin 2 pi f t + c
 * (reading a15).  Same grid, layout and best-period conventions as lsp_periodogram_batched; `center` and
 * `normalize` of the plan do not apply (the mean floats; the power is normalised by construction).
 *   d_sigma      DEVICE, offsets[n_obj] elements of the plan's dtype, all > 0 (1-sigma errors of y).
 *   d_out_power  DEVICE, n_obj * n_freq elements, or NULL when only the best period is wanted.
 *   d_best_*     DEVICE, n_obj elements each: all three or none.
 * Asynchronous on cuda_stream.  Runs the standard contraction kernels twice in their partial-sum form -- pass 1: sums of
 * w (y - ybar) e^{i theta} and, in the doubled-angle slot, w e^{2 i theta}; pass 2: sums of w e^{i theta} (the tensor-core
 * path skips the doubled-angle contraction there) -- and one combine kernel: about 2x the cost of lsp_periodogram_batched
 * on the FMA-pipe kernels, ~1.5x on the tensor-core path (the paper's own implementation: 2.06-2.14x).
 * kernel = AUTO selects as lsp_periodogram_batched does, except that it falls back from the tensor-core kernel to the FMA-pipe
 * one when the batch's operand table would exceed the plan's budget (LSP_ERR_UNSUPPORTED if kernel = TENSOR was forced).
 * Other errors as lsp_periodogram_batched.
 */
lsp_status lsp_periodogram_generalized(lsp_plan* plan, int64_t n_obj,
                                       const int64_t* d_offsets, const int64_t* h_offsets,
                                       const void* d_t, const void* d_y, const void* d_sigma,
                                       void* d_out_power,
                                       void* d_best_period, void* d_best_power, int64_t* d_best_index,
                                       void* cuda_stream);

/*
 * The generalised periodogram for callers whose data lives on the HOST: every pointer is a HOST pointer (h_sigma like h_t, h_y;
 * h_out_power may be NULL for best-period-only output).  Inputs are copied to plan-owned device buffers on cuda_stream; full
 * periodograms come back round by round through the plan's chunk ring and copy streams (chunk_bytes per round: the D2H of one
 * round overlaps the kernels of the next), best-period arrays by one small D2H each.  Returns after everything
 * has landed on the host.  LSP_FLAG_PAGEABLE_STAGED does not apply to this call: a pageable h_out_power is handed to
 * cudaMemcpyAsync as it is (the staged scheme belongs to lsp_periodogram_batched / _batched_host).
 * Errors as lsp_periodogram_generalized.
 */
lsp_status lsp_periodogram_generalized_host(lsp_plan* plan, int64_t n_obj,
                                            const int64_t* h_offsets, const void* h_t, const void* h_y, const void* h_sigma,
                                            void* h_out_power,
                                            void* h_best_period, void* h_best_power, int64_t* h_best_index,
                                            void* cuda_stream);

/*
 * End-to-end form of lsp_periodogram_batched / lsp_best_period for callers whose data lives on the HOST (the paper's own call
 * shape: H2D of the concatenated (t, y) arrays, kernel, D2H of periodograms and/or periods,
 * PAPER.md:L85-91, L103-117).  Every pointer is a HOST pointer (pinned memory lets the copies overlap;
 * pageable memory works but serialises):
 *   h_offsets    int64[n_obj+1]   (validated: offsets[0] = 0, non-decreasing)
 *   h_t, h_y     offsets[n_obj] elements of cfg.dtype
 *   h_out_power  n_obj * n_freq elements of cfg.dtype, or NULL for best-period-only output (the
 *                N_obj x N_f array is then never written anywhere)
 *   h_best_*     optional (all three NULL or all three non-NULL; required when h_out_power is NULL)
 * The inputs are copied to plan-owned device buffers on cuda_stream, the same kernels run, full
 * periodograms come back through the chunk ring and copy streams (step 7) and the best-period arrays by
 * one small D2H each.  The call returns after everything has landed on the host.
 * Errors as for lsp_periodogram_batched.
 */
lsp_status lsp_periodogram_batched_host(lsp_plan* plan, int64_t n_obj,
                                        const int64_t* h_offsets, const void* h_t, const void* h_y,
                                        void* h_out_power,
                                        void* h_best_period, void* h_best_power, int64_t* h_best_index,
                                        void* cuda_stream);

/*
 * Best period over FREQUENCY SHARDS (a single huge object, or any batch, whose grid was cut into contiguous index ranges that
 * ran as separate plans, possibly on different GPUs).  `plan` is a plan for the GLOBAL grid (its f_min,
 * f_max, n_freq and dtype are used; no periodogram is computed).  For every object the candidates of the n_parts shards are
 * merged with the library's own rule (reading a7: largest power, lowest grid index on exact ties, NaN or
 * index -1 never wins) and period = 1/f_k on the global grid.
 *   d_part_power   DEVICE, [n_parts][n_obj] of cfg.dtype: each shard's best power per object
 *   d_part_index   DEVICE, int64 [n_parts][n_obj]: each shard's best GLOBAL grid index per object, or -1
 *   d_best_*       DEVICE, n_obj elements each (index -1, power 0, period NaN when no shard had a candidate)
 * Asynchronous on cuda_stream.  Errors: LSP_ERR_INVALID_ARG, LSP_ERR_CUDA.
 */
lsp_status lsp_best_merge(lsp_plan* plan, int64_t n_obj, int32_t n_parts,
                          const void* d_part_power, const int64_t* d_part_index,
                          void* d_best_period, void* d_best_power, int64_t* d_best_index,
                          void* cuda_stream);

/*
 * Best period per object WITHOUT ANY ALLOCATION: no plan, no cudaMalloc / cudaFree / cudaMallocHost, no stream or event
 * creation, nothing that grows on the device or on the host.
 *
 * Who this is for.  Every other call works on a plan, and a plan allocates (lsp_plan_create up front, the calls whenever their
 * scratch has to grow).  Some programs cannot afford that at the point where they need a period search: a service whose whole
 * HBM has been handed to its own pool or caching allocator, so that a raw cudaMalloc from a library fails or eats into a budget
 * it does not own; a real-time or latency-bound loop, where cudaMalloc / cudaFree stall every stream of the device; a plug-in
 * that runs under a host application's rule "no driver allocations after start-up".  Such a caller passes its inputs and its
 * three output arrays, all allocated by itself, and the library brings its own scratch: one fixed array of
 * LSP_STATIC_SCRATCH_BYTES that is part of the library image.  Every GPU whose context loads the library holds that array
 * from then until the process exits, whether or not this function is ever called.
 *
 * What runs: the fused-argmax route of lsp_best_period on the direct kernel family (LSP_KERNEL_DIRECT, one sincos per (t, f)
 * pair; best period PAPER.md:L87, L105), always with one observation split, followed by the same finalize
 * kernel; the per-CTA (power, index) candidates and, with center / normalize, the per-object statistics live in the static
 * array instead of plan-owned memory.  Same grid, tie rule and empty-object convention as lsp_best_period (readings a1, a2,
 * a7, a8).  Results agree with lsp_best_period on a LSP_KERNEL_DIRECT plan to rounding (bit for bit when that plan also runs
 * one split), and with the other kernel families within the library's tolerances.
 *
 *   cfg          HOST.  Read: f_min, f_max, n_freq, dtype, fast_math, normalize, center, device.  Every other field is ignored
 *                (a plan's lsp_config can be passed as it is; `kernel` does not select anything here).
 *   n_obj        objects (>= 0).  n_obj = 0 does the one-time set-up described below and nothing else.
 *   d_offsets    DEVICE, int64[n_obj+1], non-decreasing, indices into d_t / d_y.  offsets[0] need not be 0, so an object range
 *                [o0, o0+n) of a larger batch is (d_offsets + o0, same d_t and d_y, d_best_* + o0).
 *   d_t, d_y     DEVICE, elements of cfg.dtype, as for lsp_best_period.
 *   d_best_*     DEVICE, n_obj elements each, all three required: period and power (cfg.dtype), grid index (int64; -1, power 0
 *                and NaN period for an object without observations).
 *   cuda_stream  cudaStream_t as void* (NULL = default stream); the call is asynchronous on it.
 *
 * Limit.  The scratch need is 16 bytes x n_obj x (ceil(n_freq / 1024) + 1) and must not exceed LSP_STATIC_SCRATCH_BYTES
 * (16 MiB: n_obj x (ceil(n_freq / 1024) + 1) <= 1,048,576 -- e.g. 10,000 objects on a 100,000-point grid, or one object on
 * a grid of a billion points).  A larger request is rejected with LSP_ERR_UNSUPPORTED before anything is launched; run it as
 * object ranges.
 *
 * Set-up.  The first call for a given device looks up where that device keeps the array and how many SMs it has (two queries,
 * no allocation) and remembers both for the life of the process; it makes cfg.device current to do so, as every call of this
 * library does.  Make that first call (n_obj = 0 is enough) before the device is inside a stream capture.
 *
 * Sharing.  There is ONE array per device for the whole process.  Nothing in it has to start at zero -- each call writes every
 * slot it later reads -- so no clearing is done and a call leaves its candidates behind for the next one to overwrite.  Two
 * calls that can overlap on the same GPU (different streams, different host threads, different "plans" of the caller) would
 * write the same slots: they RACE and both results are garbage.  Order them on one stream or with events.  Plan-based calls
 * never touch the array and may overlap with it freely.
 *
 * Errors: LSP_ERR_INVALID_ARG (bad grid / dtype / fast_math with FP64 / device ordinal, NULL pointer with n_obj > 0, n_obj < 0),
 * LSP_ERR_UNSUPPORTED (over the limit above; device not sm_100), LSP_ERR_CUDA.  The message is read with lsp_last_error(NULL).
 */
#define LSP_STATIC_SCRATCH_BYTES (16 << 20)
lsp_status lsp_best_period_static(const lsp_config* cfg /* HOST */, int64_t n_obj,
                                  const int64_t* d_offsets, const void* d_t, const void* d_y,
                                  void* d_best_period, void* d_best_power, int64_t* d_best_index,
                                  void* cuda_stream);

/* Frees the plan and everything it owns (synchronises its streams first).  NULL is a no-op. */
void lsp_destroy(lsp_plan* plan);

/* Message of the last failure on this plan (plan-owned, valid until the next call on the plan); with
 * plan == NULL, the message of the last failed lsp_plan_create or lsp_best_period_static on this thread.  Never NULL. */
const char* lsp_last_error(const lsp_plan* plan);

/* Bookkeeping of the LAST call on the plan, for benchmarks and tests: how many of the library's kernels it launched,
 * (t,f) pairs evaluated, the kernel family used (lsp_kernel), observation splits per (object, tile), -- host-output
 * calls only -- chunks copied, the tensor kernel's warp-role shape (0 = tensor kernel not used, 1 = short-item
 * shape, 2 = long-item shape, 3 = long-item shape on CTA pairs; see lsp_config.tensor_roles, tensor_pair) and its FP16 products per multiply-accumulate in the last
 * launch (0 = tensor kernel not used; 1 = fast_math; 2 or 3: lsp_config.tensor_products -- a call that holds an object
 * of fewer than 32 observations runs with 3 whatever the plan says).  Any pointer may be NULL. */
void lsp_last_call_info(const lsp_plan* plan, int64_t* n_launches, int64_t* n_pairs, int32_t* kernel_used,
                        int32_t* n_split, int64_t* n_chunks, int32_t* tensor_shape, int32_t* tensor_products);

/*
 * Device time of the periodogram kernel(s) of the LAST call, in milliseconds, measured with CUDA events
 * recorded on the launching stream around the dominant kernel (bench.py's roofline.achieved).  Enabled by
 * lsp_set_timing(plan, 1); the query synchronises on the stop event.  Returns < 0 if timing was off.
 */
void  lsp_set_timing(lsp_plan* plan, int32_t on);
float lsp_last_kernel_ms(lsp_plan* plan);

/* Library version / build string (static). */
const char* lsp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LSP_B200_H */
