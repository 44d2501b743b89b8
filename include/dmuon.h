/*
 * dmuon.h -- C ABI of libdmuon: the single-GPU Muon optimizer step of DMuon (arxiv/paper_2606_27153)
 * for NVIDIA B200 (sm_100a).
 *
 * The path (Eq. 1; Eq. 2; Gram form PAPER.md:170; Algorithm 1 l.12-16, PAPER.md:232-239;
 * conventions the paper does not print are the readings N1..N17 of DESIGN.md):
 *
 *     M' = mu M + G ;  U = bf16( G + mu M' )                         Nesterov momentum + the bf16 cast
 *     X0 = U / (||U||_F + 1e-7)        (the Gram matrix is taken on the smaller side)
 *     k times:  A = X X^T ;  B = b A + c A A ;  X <- a X + B X       Newton-Schulz quintic, Gram form
 *     W' = W - lr ( sqrt(max(1, rows/cols)) X_k + wd W )             Eq. 1 with shape scale + decoupled decay
 *                                                                    (applied in the last X update's epilogue)
 *
 * Every step runs in hand-written CUDA kernels (tcgen05/TMEM/TMA grouped GEMMs, vectorised elementwise
 * kernels).  There is no CPU fallback: on a machine without an sm_100 device every compute entry point
 * returns DMUON_ERR_UNSUPPORTED_DEVICE.
 *
 * Conventions for all entry points
 *   - matrices: bfloat16, row-major, contiguous (leading dimension == cols), base pointer 16-byte aligned,
 *     rows >= 1, cols >= 1.  DEVICE pointers unless the function name ends in _host.
 *   - `shapes`: HOST array of count*2 int32 = {rows, cols} per matrix.  Pointer arrays are HOST arrays.
 *     All host arrays are copied before the call returns.
 *   - ownership: the caller owns every tensor.  `grads` are never written.  `params`, `momenta` (and `ptrs` of
 *     dmuon_ns_batched) are updated in place.  Two entries of one call must not alias or overlap (undefined).
 *   - asynchrony: work is enqueued on `stream` (a cudaStream_t) and the call returns without synchronising,
 *     EXCEPT the first call for a shape set not seen before, which builds a plan, allocates workspace and
 *     autotunes tile configurations on scratch buffers (never on caller data) and synchronises the device.
 *   - errors: return value 0 = DMUON_OK, negative = error; dmuon_last_error() gives a message for the calling
 *     thread's last failure.  Nothing throws or aborts across this boundary.  Non-finite inputs propagate.
 *   - count == 0 is a valid no-op.
 *   - threads: every entry point takes one process-wide mutex for its whole host-side duration, so calls from several
 *     host threads are safe and run one after another (the enqueued GPU work still overlaps only as its streams
 *     allow, and the per-device workspace is shared: see "devices").  dmuon_last_error() is per thread.
 *   - CUDA graphs: once a shape set's plan exists (first call, or dmuon_warmup) a step only enqueues kernels and one
 *     pointer-table upload, and may be captured.  The captured graph keeps RAW POINTERS into that plan's device tables
 *     and into the workspace, and its replay re-uploads the tensors it was captured with.  The library therefore
 *     (a) records the upload in every capture and, after a plan has been captured once, uploads on every later eager
 *     call too, so replays and eager calls with other tensors can be mixed in any order on one stream;
 *     (b) never evicts a captured plan from its cache of 8 plans, and REFUSES (DMUON_ERR_INVALID_ARG) what would free
 *     memory a graph may still use: dmuon_set_workspace, a new shape set that needs a larger shared workspace, a
 *     ninth plan when all eight are captured.  Warm up the largest shape set before capturing.  After destroying
 *     the graphs, dmuon_set_option("graphs_destroyed", "1") lifts (a) and (b); dmuon_shutdown frees everything
 *     regardless, so destroy the graphs first.
 *   - devices: every call works on the CURRENT CUDA device (cudaSetDevice before the call); plans, workspaces and
 *     kernel attributes are kept per device.  Calls that share a device share that device's workspace: issue them
 *     on one stream, or order the streams yourself.
 */
#ifndef DMUON_H_
#define DMUON_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define DMUON_API __attribute__((visibility("default")))
#else
#define DMUON_API
#endif

#define DMUON_OK 0
#define DMUON_ERR_INVALID_ARG (-1)        /* null pointer, count < 0, dimension <= 0, steps < 0, misaligned pointer, bad option */
#define DMUON_ERR_UNSUPPORTED_DEVICE (-2) /* current device is not compute capability 10.x, or no device */
#define DMUON_ERR_OOM (-3)                /* workspace allocation failed, or a caller workspace is too small */
#define DMUON_ERR_CUDA (-4)               /* a CUDA runtime / driver call failed */
#define DMUON_ERR_INTERNAL (-5)

/* A cudaStream_t, spelled without including CUDA headers. */
typedef struct CUstream_st* dmuon_stream_t;

/*
 * Batched Newton-Schulz orthogonalisation (Eq. 2 in the Gram form of :170, batched by shape as in :180).
 *   ptrs    HOST array[count] of DEVICE pointers; matrix i is shapes[2i] x shapes[2i+1] bf16 and is OVERWRITTEN in
 *           place by NS_steps( X / (||X||_F + 1e-7) ), rounded to bf16, in the input's own orientation.
 *   steps   number of NS steps k >= 0 (0 = normalisation only).
 *   coeffs  HOST, exactly 3 floats {a, b, c} used at every step; NULL = {3.4445, -4.7750, 2.0315}.
 */
DMUON_API int dmuon_ns_batched(void* const* ptrs, const int32_t* shapes, int32_t count, int32_t steps,
                               const float* coeffs, dmuon_stream_t stream);

/* Same with a per-step schedule: coeffs is HOST [steps][3] (e.g. Polar Express; values are the caller's). */
DMUON_API int dmuon_ns_batched_sched(void* const* ptrs, const int32_t* shapes, int32_t count, int32_t steps,
                                     const float* coeffs, dmuon_stream_t stream);

/*
 * One Muon optimizer step over `count` 2-D parameters (Eq. 1; Alg. 1 l.12-15).
 *   params   HOST array[count] of DEVICE pointers to W (bf16), updated in place.
 *   grads    HOST array[count] of DEVICE pointers to G (bf16), read only.
 *   momenta  HOST array[count] of DEVICE pointers to M (bf16), updated in place to mu M + G.
 *   lr, mu, wd  learning rate, momentum, decoupled weight decay.
 * Uses the NS step count and coefficients set through dmuon_set_option ("steps", "coeffs" or "coeffs_sched";
 * defaults 5 and the standard quintic).
 */
DMUON_API int dmuon_muon_step(void* const* params, const void* const* grads, void* const* momenta,
                              const int32_t* shapes, int32_t count, float lr, float mu, float wd,
                              dmuon_stream_t stream);

/*
 * The Muon step with fp32 master weights ("the orthogonalized update is cast to fp32 and applied to the
 * fp32 master weights, and then cast back to the parameter's working dtype").  As dmuon_muon_step, but the update
 *     master' = master - lr * (sqrt(max(1, rows/cols)) * O + wd * master)       (fp32, one expression)
 * is applied to masters[i] (DEVICE fp32, row-major, contiguous, 32-byte aligned, updated in place) and params[i] (bf16)
 * is OVERWRITTEN with the round-to-nearest-even bf16 of the new master; its previous contents are not read.
 */
DMUON_API int dmuon_muon_step_master(void* const* params, void* const* masters, const void* const* grads,
                                     void* const* momenta, const int32_t* shapes, int32_t count, float lr, float mu,
                                     float wd, dmuon_stream_t stream);

/*
 * The same step for tensors that live in HOST memory (pinned memory gives asynchronous copies): copies W, G, M of
 * every matrix to device staging buffers owned by the library, runs dmuon_muon_step there, and copies W and M
 * back.  The matrix list is processed in up to 32 groups of whole repetitions of its shape pattern (layers) through
 * a ring of four staging slots (four groups resident, not the whole set; option "host_pipeline"), so that the
 * host->device copies of one group, the step of the previous one and the device->host copies of the one before
 * overlap (two library-owned copy streams, both PCIe directions busy).  On an error return nothing is left in flight.  All work is ordered after what `stream`
 * held at the call and `stream` waits for all of it: the caller synchronises `stream` before reading the results.
 * Host buffers should be pinned (pageable memory makes the copies synchronous).
 */
DMUON_API int dmuon_muon_step_host(void* const* params_host, const void* const* grads_host,
                                   void* const* momenta_host, const int32_t* shapes, int32_t count, float lr,
                                   float mu, float wd, dmuon_stream_t stream);

/*
 * Non-matrix parameters (embeddings, norms, biases; Alg. 1 l.16 "non-matrix params: AdamW"): one
 * decoupled-weight-decay AdamW step (the paper's citation [16]; the convention of torch.optim.AdamW) over `count`
 * tensors in ONE launch:
 *     m <- beta1 m + (1 - beta1) g ;  v <- beta2 v + (1 - beta2) g^2
 *     p <- p (1 - lr wd) - lr / (1 - beta1^step) * m / ( sqrt(v) / sqrt(1 - beta2^step) + eps )
 *   params      HOST array[count] of DEVICE pointers, bf16, updated in place (fp32 arithmetic, one RNE rounding)
 *   grads       HOST array[count] of DEVICE pointers, bf16, read only
 *   exp_avg, exp_avg_sq   HOST arrays[count] of DEVICE pointers, fp32, updated in place
 *   numel       HOST array[count], elements per tensor (> 0); all pointers 16-byte aligned
 *   step        1-based step count (bias correction)
 */
DMUON_API int dmuon_adamw_step(void* const* params, const void* const* grads, void* const* exp_avg,
                               void* const* exp_avg_sq, const int64_t* numel, int32_t count, float lr, float beta1,
                               float beta2, float eps, float wd, int32_t step, dmuon_stream_t stream);

/*
 * dmuon_adamw_step for callers that cannot allocate device memory.
 *
 * Who that is: an optimizer step that runs inside a training process whose framework allocator has already taken
 * (nearly) all of the GPU's memory for its own pool, so a raw cudaMalloc from a library fails although the framework
 * could still hand out tensors; a step issued while collectives of another stream are in flight, where cudaMalloc and
 * cudaFree are unwelcome because they synchronise the whole device; and tight loops that cannot afford that
 * synchronisation at all.  dmuon_adamw_step allocates its per-call work table (one record per tensor) with cudaMalloc
 * whenever the tensor list changes.  This entry point never does: the table lives in a fixed array that is part of the
 * library's device image, 192 KiB on every GPU that has loaded libdmuon, held until the process exits.
 *
 * Arguments, arithmetic and results are those of dmuon_adamw_step (same kernel; results are bitwise equal).  Differences:
 *   - count must be <= DMUON_ADAMW_NOALLOC_MAX_TENSORS, else DMUON_ERR_INVALID_ARG and nothing is enqueued.  Longer
 *     lists: several calls on one stream.
 *   - no cudaMalloc, cudaFree, cudaMallocHost or other allocating routine is called, on any call.
 *   - the FIRST call on each device looks up the array's address on that device (cudaGetSymbolAddress, with the
 *     caller's current device) and remembers it.  Make that first call during start-up, on the device you will use and
 *     before any stream capture begins.
 *   - the table is uploaded from host memory at every call (two small asynchronous copies on `stream` ahead of the kernel), so the
 *     call may wait for earlier work of `stream` to drain before it returns; everything it enqueues is ordered on `stream`.
 *   - ALL calls on a device share the one array.  Each call rewrites every table entry its kernel reads, so nothing
 *     from an earlier call is reused and nothing needs clearing; but two calls whose GPU work can overlap (different
 *     streams without an event between them) race on the table and may update the wrong tensors.  Keep the calls of a
 *     device on one stream, or order the streams yourself.
 *   - launches are not recorded by the "profile" option.
 */
#define DMUON_ADAMW_NOALLOC_MAX_TENSORS 4096
DMUON_API int dmuon_adamw_step_noalloc(void* const* params, const void* const* grads, void* const* exp_avg,
                                       void* const* exp_avg_sq, const int64_t* numel, int32_t count, float lr,
                                       float beta1, float beta2, float eps, float wd, int32_t step,
                                       dmuon_stream_t stream);

/*
 * c_{s,b} of PAPER.md:194: the measured time (ms) of the owner-local Muon update of ONE batch of `batch` matrices of
 * shape rows x cols "including the complete execution path selected by the runtime" (bucketing, tuned tile
 * configurations, block schedule, fused epilogue), averaged over `reps` steps after two warm-up steps.  Runs on
 * library-owned scratch tensors; synchronises the device.
 */
DMUON_API int dmuon_measure_cost(int32_t rows, int32_t cols, int32_t batch, int32_t reps, float* ms_out,
                                 dmuon_stream_t stream);

/*
 * Owner assignment from a measured cost model (Eq. 5).  HOST ONLY, no device needed.
 *     minimise  max_r sum_{s,b} c[s,b] x[s,b,r]    subject to   sum_{r,b} b x[s,b,r] = n_s  for every shape s
 *   counts       [num_shapes] n_s, matrices of shape s
 *   num_batches  [num_shapes] |B_s|, candidate batch sizes of shape s (must contain 1 when n_s > 0)
 *   batch_sizes, costs   concatenated over shapes: b and c[s,b] (e.g. from dmuon_measure_cost)
 *   mode         0 greedy (longest processing time first, over several batch-size caps); 1 exact (branch and bound);
 *                -1 exact when (sum_s |B_s|) * num_ranks <= threshold (S_thr of PAPER.md:206), greedy otherwise
 *   x_out        [(sum_s |B_s|) * num_ranks] batches of configuration k = (s, b) given to rank r at x_out[k * R + r]
 *   makespan_out the largest per-rank cost of the returned assignment
 * Returns 1 when the result is a proven optimum, 0 for a greedy result, negative on error (an exact search that
 * exceeds its node budget falls back to greedy and returns 0).
 */
DMUON_API int dmuon_assign_owners(const int32_t* counts, const int32_t* num_batches, const int32_t* batch_sizes,
                                  const double* costs, int32_t num_shapes, int32_t num_ranks, int32_t mode,
                                  int32_t threshold, int32_t* x_out, double* makespan_out);

/* Plan + allocate + autotune for a shape set ahead of time (what the first dmuon_muon_step would do). */
DMUON_API int dmuon_warmup(const int32_t* shapes, int32_t count, dmuon_stream_t stream);

/* Bytes of device workspace a step over this shape set needs with the current options (0 on bad arguments): the
 * largest bucket's buffers, since buckets run one after another in one region ("chunk_mb" bounds a bucket). */
DMUON_API size_t dmuon_workspace_bytes(const int32_t* shapes, int32_t count);

/* Hand the library a caller-owned DEVICE workspace (256-byte aligned) to use instead of its own allocation;
 * (NULL, 0) returns to library-owned workspace.  Drops all cached plans. */
DMUON_API int dmuon_set_workspace(void* dev_ptr, size_t bytes);

/*
 * Options (string key/value).  Keys:
 *   "steps"       NS steps of dmuon_muon_step (default "5")
 *   "coeffs"      "a,b,c" used by dmuon_muon_step (default "3.4445,-4.7750,2.0315")
 *   "coeffs_sched" "a0,b0,c0;a1,b1,c1;..." one triple per NS step for the Muon-step entry points (per-step sets such
 *                 as Polar Express; the values are the caller's); must hold exactly "steps" triples when
 *                 a step runs; "" = off (default)
 *   "mode"        "tc"  = fp16 operands on tcgen05 tensor cores, fp32 accumulation in TMEM (default; PAPER.md:262 runs NS in fp16);
 *                 "fp32_check" = fp32 operands, plain SIMT kernels: the <= 1e-4 check mode, small shapes only
 *   "schedule"    "auto" = on wide buckets (n >= 1.5 m, m >= 256) run the k steps as Gram blocks: G = X X^T once per block,
 *                 G_{i+1} = P_i G_i P_i in the m x m Gram space (Eq. 4), Q = prod P_i, one X <- Q X per
 *                 block; blocks of 3 then 2 steps for k = 5 (restarts keep fp16 storage stable).  An exact
 *                 reformulation of Eq. 2: same result up to rounding (default).
 *                 "x" = the plain iteration X <- (a I + B) X at every step, on every bucket
 *   "autotune"    "1"/"0": pick each bucket's tile configuration by on-device measurement (default "1")
 *   "fuse_epilogue" "1"/"0": for matrices whose rows and cols are multiples of 128, apply W' = W - lr (scale O + wd W)
 *                 (or write the bf16 NS output) in the epilogue of the last X update instead of a separate pass
 *                 (default "1").  Results agree to the rounding of the unfused path's fp16 O
 *   "small_fused" "1"/"0": matrices whose padded oriented shape is 256 x 256 run ALL their NS steps in one on-chip
 *                 kernel (X, G, B resident in the shared memory of a CTA pair; nothing stored between products), up to
 *                 16 steps (default "1"; "0" = the grouped per-product launches, as for every other shape)
 *   "graphs_destroyed" "1": a statement, not a setting: every CUDA graph captured from calls of this library has been
 *                 destroyed (see "CUDA graphs" at the top).
 *   "keep_ns_output" "1"/"0": keep every matrix's unrounded NS result readable after the call (dmuon_read_ns_output):
 *                 fused epilogues also store it and buckets get disjoint workspace regions (default "0")
 *   "chunk_mb"    workspace a bucket may use, MiB (default "12288"): a bucket whose matrices need more runs as
 *                 chunks of fewer matrices, one after the other, through the same region
 *   "host_pipeline" "groups,slots" of dmuon_muon_step_host (default "32,4")
 *   "program"     "auto" (default) / "1" / "0": run ALL products of a bucket's NS program in ONE launch, chained by
 *                 per-matrix completion counters instead of kernel boundaries, the matrices taken in groups whose
 *                 buffers fit the L2 ("l2_group_mb").  "auto" = buckets whose small side is >= 2048 (there it is 5-10 %
 *                 faster: fewer DRAM bytes, more clock under the power cap); "1" = every bucket with a small side
 *                 >= 256 and <= 32 products; "0" = one launch per product everywhere.  Same arithmetic either way
 *                 (work units are handed out dynamically to the CTAs that are running, so the launch also makes progress
 *                 while kernels of other streams occupy part of the GPU)
 *   "l2_group_mb" budget for the buffers of one group of matrices in the program kernel, MiB (default "64"; a group is
 *                 never smaller than three waves of work units)
 *   "tune_ms"     autotune: milliseconds each candidate runs back to back (default "40": long enough for the
 *                 board's power cap to act, as it does in the step)
 *   "variants"    "s,q,b": force the tile configuration (see dmuon_ns_gemm) of the SYRK, m x m and X-update products of
 *                 plans built from now on; -1 = measured / cached choice (default "-1,-1,-1")
 *   "cache_path"  file for the persistent tuning cache ("" disables; default $DMUON_CACHE or ~/.cache/dmuon/tune.txt)
 *   "profile"     "1"/"0": record CUDA events around every kernel launch (read with dmuon_profile_read)
 * Returns DMUON_ERR_INVALID_ARG for an unknown key or unparsable value.
 */
DMUON_API int dmuon_set_option(const char* key, const char* value);

/*
 * Describe how a shape set is executed: writes a JSON object
 *   {"buckets": [{"m": m_pad, "n": n_pad, "kind": "wide" | "tall" | "generic", "count": matrices, "blocks": [3, 2],
 *                 "variants": [gram, sq, xupdate], "fused": bool, "onchip": bool, "program": bool, "xscale": c, "gscale": g}, ...],   (execution order;
 *    "workspace_bytes": B, "tune_seconds": t, "tune_cache_entries": n}                     chunks of a shape repeat)
 * for `steps` NS steps with the current options into buf (NUL terminated, truncated to
 * len); builds the plan if needed (like dmuon_warmup).  Returns the bytes needed (excluding the NUL) or a negative error.
 */
DMUON_API int dmuon_describe_plan(const int32_t* shapes, int32_t count, int32_t steps, char* buf, size_t len,
                                  dmuon_stream_t stream);

/*
 * Host-only (no device needed): the block schedule the library would use for ONE rows x cols matrix and `steps` NS
 * steps under the current "schedule" option.  coeffs: HOST, 3 floats (per_step = 0), [steps][3] (per_step = 1) or
 * NULL (defaults).  Writes up to `cap` block lengths into out (sum = steps) and returns the number of blocks, or a
 * negative error.  A block of length 1 is the plain step; longer blocks run in the Gram space (see "schedule").
 */
DMUON_API int dmuon_block_schedule(int32_t rows, int32_t cols, int32_t steps, const float* coeffs, int32_t per_step,
                                   int32_t* out, int32_t cap);

/* Thread's last error message ("" if none).  The pointer stays valid until the thread's next failing call. */
DMUON_API const char* dmuon_last_error(void);

/*
 * With option profile=1: synchronises the recorded events and writes a JSON object
 *   {"kernels": {"<name>": {"launches": L, "ms": total}, ...}, "launches": total}
 * accumulated since the last dmuon_profile_reset into buf (NUL terminated, truncated to len).  Returns the number
 * of bytes needed (excluding the NUL), or a negative error.
 */
DMUON_API int dmuon_profile_read(char* buf, size_t len);
DMUON_API int dmuon_profile_reset(void);

/*
 * Building block of the NS iteration, exposed for tests and benchmarks: ONE grouped launch over `count`
 * same-shape problems on fp16 row-major DEVICE matrices whose dimensions are multiples of 128.
 *   op 0 (SYRK, step a3):  C[m x m] = alpha * X X^T                X = in0[i] is m x k;  in1 ignored
 *   op 1 (SQ,   step a4):  C[m x m] = alpha * A A + beta * A       A = in0[i] is m x m, symmetric;  in1 ignored
 *   op 2 (BX,   step a5):  C[m x n] = alpha * B X + beta * X       B = in0[i] is m x m;  X = in1[i] is m x n
 *   op 4 (SYRK_T):         C[m x m] = alpha * Y^T Y                Y = in0[i] is n x m (a tall matrix as stored)
 *   op 5 (XB):             C[n x m] = alpha * Y B + beta * Y       B = in0[i] is m x m SYMMETRIC;  Y = in1[i] is n x m
 * For ops 0 and 4 `n` is the contraction length; for op 1 it is ignored.  Symmetric ops compute upper-triangular
 * tiles only and mirror them.  in0/in1/out are HOST arrays[count] of DEVICE pointers; out must not alias an input.
 * variant: -1 = the default tile configuration, >= 0 selects configuration `variant`: 0..3 = one CTA per unit,
 * UMMA 128 x 256 (0, 2) or 128 x 128 (1, 3), column-panel-major (0, 1) or row-major (2, 3) unit order; 4, 5 = CTA
 * pair (cta_group::2), UMMA 256 x 256, panel-major / row-major; 6, 7 = the CTA pair with 8 epilogue warps (two per
 * TMEM lane quarter: for short contractions, where the epilogue sets the pace).  The symmetric ops accept 0, 1, 4, 6 only.
 */
DMUON_API int dmuon_ns_gemm(int32_t op, const void* const* in0, const void* const* in1, void* const* out,
                            int32_t m, int32_t n, int32_t count, float alpha, float beta, int32_t variant,
                            dmuon_stream_t stream);

/*
 * The symmetric m x m product of the Gram blocks (Eq. 4), for tests: ONE grouped launch of
 *   C = alpha * A B^T + beta * D + beta2 * D2
 * over `count` problems; every matrix is fp16 m x m row-major on the DEVICE, m a multiple of 128.  The RESULT is
 * assumed symmetric (A, B commuting symmetric matrices): only upper-triangular tiles are computed and mirrored.
 * d and/or d2 may be NULL (term absent; d2 requires d).  a/b/d/d2/out: HOST arrays[count] of DEVICE pointers; out
 * must not alias an input.  variant as for dmuon_ns_gemm op 1.  Synchronises `stream` before returning (test entry).
 */
DMUON_API int dmuon_ns_sym_mm(const void* const* a, const void* const* b, const void* const* d, const void* const* d2,
                              void* const* out, int32_t m, int32_t count, float alpha, float beta, float beta2,
                              int32_t variant, dmuon_stream_t stream);

/* Number of tile-configuration variants dmuon_ns_gemm accepts for `op`. */
DMUON_API int dmuon_ns_gemm_variants(int32_t op);

/*
 * Test hook: copies the Newton-Schulz result O = NS_k(X0) of matrix `index` of the MOST RECENT dmuon_muon_step /
 * dmuon_ns_batched call out of the library's workspace, before any rounding to bf16, as fp32 into out_dev
 * (DEVICE, rows*cols floats, the matrix's stored orientation).  Valid until the next call that uses the workspace.
 * Needs option keep_ns_output=1 set BEFORE that call unless the call had a single bucket and no fused epilogue
 * (otherwise buckets reuse one workspace region and the fused epilogue never stores O): DMUON_ERR_INVALID_ARG.
 */
DMUON_API int dmuon_read_ns_output(int32_t index, float* out_dev, dmuon_stream_t stream);

/* Free every plan, workspace, staging buffer and event; the library can be used again afterwards. */
DMUON_API void dmuon_shutdown(void);

/* Library version string. */
DMUON_API const char* dmuon_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DMUON_H_ */
