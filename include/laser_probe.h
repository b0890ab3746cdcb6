/*
 * laser_probe.h — C ABI of the B200-native LASER confidence probe.
 *
 * One call, laser_probe_confidence(), runs the whole data-parallel hot path of LASER's serving loop
 * (arxiv/paper_2606_31580; citations are /root/reference/PAPER.md line numbers) for every in-flight
 * request at a probe point (an "action transition point"):
 *
 *   a1  logits[n,v] = sum_k hidden[n,k] * W[v,k]          LM-head projection of the trial-answer
 *                                                         tokens' final hidden states
 *   a2  pmax[n] = max_v softmax(logits[n,:]),  argmax[n]  online softmax over the vocabulary; the
 *                                                         [N,V] logits never leave the SM
 *   a3  conf[r] = mean_{n in request r} pmax[n]           confidence C_i^(k)
 *   a4  tau[r]  = clamp(lambda_base - beta*tanh(gamma*(load[r]-L_target)/L_target),
 *                       lambda_min, lambda_max)           Eq. 5 + clamp
 *   a5  exit[r] = conf[r] > tau[r]   (strict)             PAPER.md:61, 70, 122 (Algorithm 1 step 6)
 *
 * Device code is sm_100a only (TMA + tcgen05/TMEM).  There is no fallback of any kind: on another
 * device the call returns LASER_E_ARCH.  The library never allocates device memory per call, never
 * synchronises the host with the device (outside the *_host entry points) and never reads device
 * data on the host; all work is enqueued on the caller's stream.  Internal state: one 64 KB control
 * block per device, allocated at first use (the counters with which the CTAs of the fused kernel
 * hand over to its last phase; never the caller's workspace), and probe handles - explicit
 * (laser_probe_handle_create) or implicit, cached per thread - holding the launch plan and the
 * encoded TMA descriptors.
 *
 * All functions return an int status (LASER_OK == 0, errors negative); none throws or aborts.
 */
#ifndef LASER_PROBE_H_
#define LASER_PROBE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    LASER_OK = 0,
    LASER_E_NULL = -1,      /* a required pointer is NULL                                             */
    LASER_E_DIMS = -2,      /* d <= 0, V <= 0, N < 0, R < 0, d % 8 != 0 (TMA row pitch must be 16 B)  */
    LASER_E_ALIGN = -3,     /* hidden / W not 16-byte aligned                                         */
    LASER_E_PARAMS = -4,    /* lambda_min > lambda_max, l_target <= 0, or a non-finite parameter      */
    LASER_E_WORKSPACE = -5, /* workspace NULL or smaller than laser_probe_workspace_bytes()           */
    LASER_E_ARCH = -6,      /* current device is not compute capability 10.0 (B200)                   */
    LASER_E_CUDA = -7,      /* a CUDA runtime / driver call failed; see laser_last_error()            */
    LASER_E_MODE = -8,      /* unknown aggregate / probability / kernel mode                          */
    LASER_E_STATIC_LIMIT = -9 /* laser_probe_confidence_static: the batch needs more scratch than the
                                 built-in LASER_STATIC_SCRATCH_BYTES array holds                       */
};

/* Hyper-parameters of Eq. 5; defaults are the paper's.  `l_target` and load[] share
 * one unit: the paper counts active requests (L_target = 10); only the ratio enters Eq. 5. */
typedef struct {
    float lambda_base; /* 0.95 */
    float beta;        /* 0.04 */
    float gamma;       /* 1.0  */
    float l_target;    /* 10   */
    float lambda_min;  /* 0.88 */
    float lambda_max;  /* 0.97 */
} laser_tau_params;

/* N = rows allocated in `hidden` (valid rows are [0, req_offsets[R])), d = hidden size,
 * V = vocabulary size, R = number of requests. */
typedef struct {
    int32_t N, d, V, R;
} laser_probe_dims;

/* How a call is laid out on the GPU (informational; filled by laser_probe_plan_query).  splits /
 * tiles_per_split / work_items describe a batch whose N rows are all valid; when req_offsets[R] < N
 * leaves whole token tiles of padding, the kernels skip them and re-deal the vocabulary tiles over the
 * remaining token tiles on the device (same tile_n), so padding rows cost no tensor work. */
typedef struct {
    int32_t num_sms;         /* SMs the plan was made for                                             */
    int32_t m_tiles;         /* ceil(N / tile_m) token tiles                                          */
    int32_t splits;          /* vocabulary splits S                                                   */
    int32_t tiles_per_split; /* vocab tiles per split T                                               */
    int32_t tile_n;          /* vocab rows per tile BN (multiple of 16; 32 in pair mode; <= 256)      */
    int32_t k_blocks;        /* ceil(d / 64)                                                          */
    int32_t stages;          /* shared-memory pipeline depth                                          */
    int32_t grid;            /* CTAs of the fused kernel (persistent, <= num_sms)                     */
    int32_t work_items;      /* m_tiles * splits                                                      */
    int32_t smem_bytes;      /* dynamic shared memory per CTA                                         */
    int32_t kernel_launches; /* kernels one laser_probe_confidence call enqueues: 1 (a3-a5 run in the
                                fused kernel's tail; mixed schedule: 2) or one more (LASER_TAIL_SEPARATE) */
    int32_t tile_m;          /* token rows per work item: 128 (one CTA) or 256 (CTA pair)             */
    int32_t cta_pair;        /* 1: clusters of two CTAs, tcgen05 cta_group::2; 0: one CTA per item    */
    int32_t ws_records;      /* 16-byte workspace records (the most any re-plan of the batch writes)  */
    int32_t tail_cache;      /* requests whose {offset, threshold} the fused kernel's tail keeps in the
                                shared memory the pipeline leaves over (0: read from global memory)    */
    /* Mixed schedule (AUTO for N > 1024 rows, LASER_MODE_MIXED for N > 256): the fields above describe the CTA-pair kernel (256-row
     * items); when the number of 128-row tiles that hold rows is odd, the last tile runs on single CTAs
     * in a second kernel beside it.  The split of the SMs is decided on the device from
     * req_offsets[R].  kernel_launches = 2: tail-tile kernel, pair kernel (a3-a5 in the tail of
     * whichever of the two has the work; of the pair kernel when both have). */
    int32_t mixed;           /* 1: mixed schedule                                                     */
    int32_t tail_tile_n;     /* vocab rows per tile of the single-CTA tail-tile kernel                */
    int32_t tail_stages;     /* its pipeline depth                                                    */
    int32_t tail_smem_bytes; /* its dynamic shared memory per CTA                                     */
    int32_t tail_grid;       /* its CTAs (those it does not need exit at once)                        */
    /* Flex kernel (LASER_MODE_FLEX up to 4096 rows; AUTO for 129 <= N <= 1024 rows except exactly
     * 256): vocabulary on the MMA M axis (tile_n = 256 rows of W per CTA pair), tokens on N in chunks of flex_n_tok rows (a multiple of 16, <= 256), so that a batch pays for at most 15 padding
     * rows per chunk.  m_tiles = chunks, splits / tiles_per_split per chunk, all for a batch whose N
     * rows are valid; the kernel looks the decomposition for req_offsets[R] up in a table the host
     * planned (laser_probe_flex_query).  One launch per call. */
    int32_t flex;            /* 1: flex kernel                                                        */
    int32_t flex_n_tok;      /* token rows per chunk for a dense batch                                */
    int32_t flex_max_tok;    /* the largest chunk any valid-row count takes (sizes the pipeline stage) */
} laser_probe_plan;

/* Kernel variant (laser_probe_options.kernel_mode).  AUTO (default): one single-CTA kernel for
 * N <= 128 rows; the flex kernel (vocabulary on the MMA M axis, token chunks of a multiple of 16 rows on
 * N, decided on the device from req_offsets[R]) for 129..1024 rows except exactly 256 (and not where it
 * measures slower: hidden sizes below 1280 above 384 rows / below 768 at all; vocabularies whose 256-row
 * tiles would leave the busiest CTA pair more than 15 % above an even share); one CTA-pair
 * kernel for N = 256 (a single 256-row item); above 1024 rows the mixed schedule (CTA pairs for the
 * even part of the 128-row tiles that hold rows, single CTAs for an odd last tile, decided on the
 * device).  SINGLE / PAIR force one variant for every shape (tuning and tests; both are exact; PAIR
 * pads an odd tile count); FLEX forces the flex kernel up to 4096 rows, MIXED the schedule AUTO uses
 * above 1024 rows for every N > 128. */
enum { LASER_MODE_AUTO = 0, LASER_MODE_SINGLE = 1, LASER_MODE_PAIR = 2, LASER_MODE_FLEX = 3, LASER_MODE_MIXED = 4 };

/* Where merge + a3-a5 run (laser_probe_options.tail).
 *   FUSED     in the tail of the fused kernel: every CTA counts itself in when its records are in the
 *             workspace, the last min(grid, R, 32) CTAs to arrive wait for the count and share the
 *             requests.  One launch per call (mixed schedule: its two fused kernels; the tail runs in
 *             the one that has the work, in the pair kernel when both have).  Needs a control slot of
 *             the library's per-device control block.  The waiting CTAs hold their SMs; with at most
 *             32 of them per call, up to FOUR fused-tail calls may be in flight on one device at the
 *             same time (different streams) and the CTAs they wait for always find a free SM.  Callers
 *             that run more probe calls than that concurrently, or beside other kernels that pin most
 *             of the SMs, use SEPARATE (a call that does starve traps after ~4 s rather than hang).
 *   SEPARATE  one more kernel (laser_probe_finalize_kernel) behind the fused one(s).  Nothing waits.
 *   AUTO      FUSED for strict calls of at most 64 requests when a control slot is available (the only
 *             case where none is: the very first call on a device is made under CUDA stream capture,
 *             where nothing can be allocated); SEPARATE for more requests (32 finalizers would take
 *             them several apiece; a block per request is faster) and for overlap = 1 calls (measured
 *             faster there: the tiny second kernel runs beside the next call's CTAs instead of holding
 *             their SMs). */
enum { LASER_TAIL_AUTO = 0, LASER_TAIL_FUSED = 1, LASER_TAIL_SEPARATE = 2 };

/* Ordering against the kernel ahead of the call on the stream (laser_probe_options.overlap).  The
 * fused kernel is launched with programmatic dependent launch, i.e. it may become resident while
 * that kernel is still running.
 * 0 (default, strict): `hidden`, `req_offsets`, `load` and `token_ids` are read only after the kernel
 *    ahead has completed (griddepcontrol.wait), whatever that kernel is - e.g. the forward pass that
 *    writes `hidden` (Algorithm 1).  W IS READ EARLIER: it is the model's LM-head
 *    weight, and the call requires that the kernel ahead of it on the stream does not write W.  The
 *    kernel requests the first W tiles of every CTA ahead of the wait, so the head of the W stream
 *    overlaps the tail of the preceding kernel.  laser_probe_options.w_ordered = 1 turns this off for
 *    callers whose W is written on the stream (then W too is read after the wait).
 * 1 (overlap): every input may be read while the kernel ahead is still running; only the kernel's
 *    stores (workspace, outputs) wait for it.  Exact whenever hidden, W, req_offsets, load are
 *    complete when the preceding kernel STARTS - true for a loop of probe calls over resident
 *    inputs, false behind a producer of `hidden`. */

/* Layout of the W buffer a call is given (laser_probe_options.w_layout).
 *   ROWMAJOR (default)  bf16 [V, d], the LM-head matrix as the model stores it.
 *   KBLOCKED            bf16 [ceil(d/64)][V][64]: K-block-major, written once per model by
 *                       laser_probe_pack_w (W is weight: pack it at load time).  The kernels read W one
 *                       (vocabulary tile x 64-column k-block) box at a time; in this layout such a box
 *                       is ONE contiguous run of tile_rows x 128 bytes in HBM instead of tile_rows
 *                       separate 128-byte pieces 2*d bytes apart, which HBM serves ~3 % faster (C2:
 *                       76.8 -> 74.3 us per strict step on one box).  Same arithmetic, same results bit
 *                       for bit; only the HBM-bound regime (N <= ~256 rows) gains.  Columns d..64*ceil(d/64)
 *                       of the packed buffer are zero. */
enum { LASER_W_ROWMAJOR = 0, LASER_W_KBLOCKED = 1 };

/* Bytes of the K-block-major copy of a [V, d] bf16 matrix: ceil(d/64) * V * 128.  0 for invalid sizes.  Host. */
size_t laser_probe_packed_w_bytes(int32_t V, int32_t d);

/* W (device, bf16 [V, d] row-major, 16-byte aligned, d % 8 == 0) -> W_packed (device,
 * laser_probe_packed_w_bytes(V, d) bytes, 16-byte aligned, must not overlap W), K-block-major.
 * Asynchronous on `stream`; one elementwise kernel, run once per model.  A vocabulary shard
 * (laser_probe_partial) is packed on its own: V = rows of the shard. */
int laser_probe_pack_w(const void* W, int32_t V, int32_t d, void* W_packed, void* stream);

/* Aggregate that turns the per-token max probabilities of a request into its confidence.
 * The paper does not fix it; MEAN is the default reading (A1). */
enum { LASER_AGG_MEAN = 0, LASER_AGG_GEOMEAN = 1, LASER_AGG_MIN = 2 };

/* Writes the paper's defaults.  Host. */
int laser_tau_params_default(laser_tau_params* out);

/* Device scratch laser_probe_confidence needs for `dims`, in bytes: 16 * ws_records of the larger of
 * the two kernel variants' plans (so one buffer serves every kernel_mode), at least 16.  Returns 0
 * for invalid dims.  Host; needs no GPU. */
size_t laser_probe_workspace_bytes(const laser_probe_dims* dims);

/* Fills *plan for `dims` (LASER_MODE_AUTO / the given kernel_mode).  Host; needs no GPU (assumes 148
 * SMs when no device is present). */
int laser_probe_plan_query(const laser_probe_dims* dims, laser_probe_plan* plan);
int laser_probe_plan_query_mode(const laser_probe_dims* dims, int kernel_mode, laser_probe_plan* plan);

/* What the mixed schedule does for a batch of dims->N allocated rows of which n_valid (= what
 * req_offsets[R] will say) hold requests: the entry of the table the kernels look up on the device.
 * Informational (tests, tuning); host; needs no GPU.  mixed = 0: dims take a single kernel. */
typedef struct {
    int32_t mixed;          /* 1: the fields below apply                                              */
    int32_t schedule;       /* 0 pair items only, 1 pair items + one single-CTA tile, 2 single-CTA tiles only */
    int32_t k_pair;         /* 256-row items on CTA pairs                                             */
    int32_t j_single;       /* 128-row tiles on single CTAs (behind the pair items)                   */
    int32_t u_pair;         /* CTA pairs that take part                                               */
    int32_t u_single;       /* single CTAs that take part                                             */
    int32_t splits_pair;    /* vocabulary splits per pair item                                        */
    int32_t splits_single;  /* vocabulary splits per single-CTA tile                                  */
    float model_us;         /* the planner's cost-model estimate of the fused kernels, microseconds   */
} laser_probe_mixed;
int laser_probe_mixed_query(const laser_probe_dims* dims, int32_t n_valid, laser_probe_mixed* out);

/* What the flex kernel does for n_valid (<= 4096) valid rows at vocabulary size dims->V: the entry of
 * its device-side table.  Informational; host; needs no GPU. */
typedef struct {
    int32_t chunks;         /* token chunks C                                                         */
    int32_t n_tok;          /* token rows per chunk (multiple of 16)                                  */
    int32_t splits;         /* vocabulary splits per chunk S (a row gets 2 S workspace records)       */
    int32_t tiles_per_split;/* 256-row vocabulary tiles per split                                     */
    int32_t rounds;         /* work items the busiest CTA pair takes                                  */
    float model_cost;       /* the planner's relative cost (rounds x tiles x per-tile cost)           */
} laser_probe_flex;
int laser_probe_flex_query(const laser_probe_dims* dims, int32_t n_valid, laser_probe_flex* out);

/*
 * The hot path a1-a5.  Asynchronous on `stream`; returns after enqueueing.
 *
 *   hidden       device, bf16 [N, d] row-major, 16-byte aligned, d % 8 == 0.  Post-final-norm states.
 *   W            device, bf16 [V, d] row-major, 16-byte aligned (LM-head / unembedding matrix).
 *   req_offsets  device, int32 [R+1], non-decreasing, [0] == 0, [R] <= N (CSR over rows; a
 *                precondition: the library never reads device data on the host.  With the
 *                environment variable LASER_DEBUG=1 a one-warp kernel checks it on the device ahead
 *                of every call and traps on a violation - the call then surfaces as a CUDA error).
 *                Two more debugging switches are read from the environment, once per process:
 *                LASER_NO_PDL=1 launches every kernel without programmatic dependent launch (full
 *                stream order, slower), LASER_NO_STAGE_KERNEL=1 makes the *_host entry points copy
 *                `hidden` with cudaMemcpyAsync instead of their staging kernel.  Same results.
 *                Rows >= req_offsets[R] are padding.
 *   load         device, float [R]: smoothed load Lbar of each request's probe point, unit of l_target.
 *   tau_params   HOST pointer; copied by value into the launch.
 *   out_conf     device, float [R].   Empty request -> 0.  NaN in a request's rows -> NaN.
 *   out_argmax   device, int32 [N].   Lowest vocabulary index attaining the row maximum; -1 for
 *                padding rows.
 *   out_exit     device, uint8 [R].   1 iff conf > tau (strict); NaN conf -> 0.
 *   dims         HOST pointer.
 *   workspace    device scratch >= laser_probe_workspace_bytes(dims), 16-byte aligned; contents are
 *                overwritten; may be reused by the next call on the same stream.
 *   stream       cudaStream_t (NULL = legacy default stream).
 *   out_tau_opt  device float [R] or NULL: the thresholds.
 *   out_pmax_opt device float [N] or NULL: per-row max probability (NaN for padding rows).
 *
 * All buffers are caller-owned.  N == 0 or R == 0 is a successful no-op on conf/exit (argmax of all
 * N rows is still set to -1 when R == 0).
 */
int laser_probe_confidence(const void* hidden, const void* W, const int32_t* req_offsets,
                           const float* load, const laser_tau_params* tau_params, float* out_conf,
                           int32_t* out_argmax, uint8_t* out_exit, const laser_probe_dims* dims,
                           void* workspace, size_t workspace_bytes, void* stream,
                           float* out_tau_opt, float* out_pmax_opt);

/* Same, with an explicit aggregate (LASER_AGG_*). */
int laser_probe_confidence_agg(const void* hidden, const void* W, const int32_t* req_offsets,
                               const float* load, const laser_tau_params* tau_params,
                               float* out_conf, int32_t* out_argmax, uint8_t* out_exit,
                               const laser_probe_dims* dims, void* workspace,
                               size_t workspace_bytes, void* stream, float* out_tau_opt,
                               float* out_pmax_opt, int aggregate_mode);

/* Which probability of a trial-answer token enters the aggregate.  PAPER.md:61 says the confidence
 * is "computed from the token probabilities" and does not say which (A2):
 *   LASER_PROB_MAX    the row maximum max_v softmax(logits[n,:]) (default; equals the emitted token's
 *                     probability under greedy decoding)
 *   LASER_PROB_TOKEN  the probability of a given token, softmax(logits[n,:])[token_ids[n]] - the token
 *                     the engine actually emitted at that position.  A token id outside [0, V) has
 *                     probability 0.  out_argmax is still the row argmax. */
enum { LASER_PROB_MAX = 0, LASER_PROB_TOKEN = 1 };

/* Options of laser_probe_confidence_opt / laser_probe_handle_create / laser_probe_partial /
 * laser_probe_combine (HOST struct, copied by value; per call, so two threads or streams may use
 * different settings).  laser_probe_options_default() fills the defaults (all zero). */
typedef struct {
    int32_t aggregate_mode;    /* LASER_AGG_*                                                        */
    int32_t prob_mode;         /* LASER_PROB_*                                                       */
    const int32_t* token_ids;  /* device, int32 [N]; required for LASER_PROB_TOKEN, else may be NULL */
    int32_t kernel_mode;       /* LASER_MODE_*                                                       */
    int32_t overlap;           /* 0 strict (default) / 1 overlap, see above                          */
    int32_t tail;              /* LASER_TAIL_*                                                       */
    int32_t w_layout;          /* LASER_W_*: how the buffer passed as W is laid out (default row-major) */
    int32_t w_ordered;         /* 0 (default): strict calls read W AHEAD of the kernel ahead's completion (see
                                  `overlap` above) - right for resident weights.  1: W is read in stream order
                                  like every other input.  Set it when W is PRODUCED on the stream just ahead of
                                  the call by a kernel that lets its dependents start early (a dequantise / cast /
                                  LoRA-merge kernel launched with programmatic dependent launch, a weight swap):
                                  such a W would otherwise be read stale, silently.  Costs the overlap of the head
                                  of the W stream with the preceding kernel's tail (a few us per call).  Applies to
                                  laser_probe_partial's W_shard as well.  laser_probe_pack_w is an ordinary launch:
                                  it reads W in stream order and its output is complete before the next kernel. */
} laser_probe_options;
int laser_probe_options_default(laser_probe_options* out);

/* laser_probe_confidence with options (NULL options = defaults: mean of the row maxima).  With
 * LASER_PROB_TOKEN, out_pmax_opt receives the token probabilities.  Costs no extra HBM traffic: the
 * token's logit rides in the spare word of the 16-byte statistics record. */
int laser_probe_confidence_opt(const void* hidden, const void* W, const int32_t* req_offsets,
                               const float* load, const laser_tau_params* tau_params,
                               float* out_conf, int32_t* out_argmax, uint8_t* out_exit,
                               const laser_probe_dims* dims, void* workspace,
                               size_t workspace_bytes, void* stream, float* out_tau_opt,
                               float* out_pmax_opt, const laser_probe_options* options);

/*
 * The probe for callers that cannot allocate device memory.
 *
 * Who this is for.  Every other entry point needs a device `workspace` from the caller, and the
 * default tail additionally makes the library cudaMalloc its per-device control block on first use.
 * Some callers can do neither: a plug-in that runs inside an inference engine whose memory pool
 * owns the whole GPU (a cudaMalloc there fails or fragments the pool, and the pool's allocator is not
 * reachable from C), a process started with nearly all of the GPU's memory already reserved by its
 * host application, or a latency-critical serving loop that must not take the driver's allocation
 * lock (cudaMalloc / cudaFree serialise against every other thread's CUDA calls and may synchronise
 * the device).  Such a caller has its inputs and outputs - the engine gave it those - and nothing
 * else.
 *
 * What it does.  Same a1-a5 as laser_probe_confidence, same kernels, same results.  The only scratch
 * the path needs - the 16-byte per-row statistics records the vocabulary splits hand to the merge -
 * goes to a fixed array of LASER_STATIC_SCRATCH_BYTES that is part of the library's device image
 * instead of a caller workspace, and merge + a3-a5 run as the second small kernel
 * (LASER_TAIL_SEPARATE), which needs no control block.  The call makes no cudaMalloc / cudaFree /
 * cudaMemset / cudaMemcpy and calls no library routine that allocates device memory; it enqueues its
 * kernels on `stream` and returns.
 *
 * Limit.  The array is LASER_STATIC_SCRATCH_BYTES (4 MiB) per GPU, resident on every GPU the library's
 * device code is loaded on from that load until the process exits, used or not.  A batch is accepted
 * iff laser_probe_workspace_bytes(dims) <= LASER_STATIC_SCRATCH_BYTES (checkable ahead of time, on the
 * host, without a GPU): at the paper's model shapes that is every batch up to about 1024 rows
 * (C4: 2.5 MB); 4096 rows at V = 151936 need 13.6 MB and are refused with LASER_E_STATIC_LIMIT
 * (laser_last_error() names both numbers).  Nothing is launched in that case.  Larger batches need
 * laser_probe_confidence with a workspace.
 *
 * First call on a device.  It looks the array's device address up (cudaGetSymbolAddress, once per
 * device, with that device current; this may make the CUDA runtime load the library's device code,
 * which is the runtime's allocation, not a call of ours), raises the kernels' shared-memory limit
 * and encodes the TMA descriptors.  Make that first call ahead of any stream capture, on every
 * device you will use; later calls with the same dims only launch.
 *
 * Sharing.  There is ONE array per GPU and every call on that GPU uses it.  Nothing in it has to start
 * at zero and nothing is cleared: a call writes every record it later reads, and what the previous
 * call left behind is never looked at.  But two calls whose kernels can be on the GPU at the same time
 * - different streams, or different threads, on one device - overwrite each other's records and return
 * wrong results without any error.  Keep all calls of this entry point on one device in ONE stream
 * order (one stream, or streams joined by events); calls with a caller workspace are not affected.
 *
 * Arguments: as laser_probe_confidence without workspace / workspace_bytes; options NULL = defaults.
 * options->tail is ignored (always SEPARATE); kernel_mode, overlap, aggregate, token_ids, w_layout
 * apply as usual.
 */
#define LASER_STATIC_SCRATCH_BYTES (4u << 20)
int laser_probe_confidence_static(const void* hidden, const void* W, const int32_t* req_offsets,
                                  const float* load, const laser_tau_params* tau_params,
                                  float* out_conf, int32_t* out_argmax, uint8_t* out_exit,
                                  const laser_probe_dims* dims, void* stream, float* out_tau_opt,
                                  float* out_pmax_opt, const laser_probe_options* options);

/*
 * Probe handles.  A handle fixes dims and options once and caches what does not change between
 * calls: the launch plan, the encoded TMA descriptors of the hidden / W buffers it has been called
 * with (2 / 4 most recent), the device-mapped addresses of pinned host buffers, and its control slot.
 * A call through a handle takes no lock, hashes nothing and queries no pointer attributes; it is what
 * a serving engine that probes the same shape every step should hold.  The handle-less entry points
 * above use implicit handles from a small per-thread cache keyed by (device, dims, options,
 * workspace).
 *
 * Thread safety: any number of handles may be used concurrently from any number of threads and
 * streams with LASER_TAIL_SEPARATE, and up to four calls in flight at once per device with the fused
 * tail (see LASER_TAIL_FUSED above: its finalizer CTAs wait on the GPU); ONE handle must be used by one
 * thread at a time, and the calls made through it must be stream-ordered with respect to each other
 * (they share the handle's control slot, like calls that share a workspace).
 *
 * Lifetime: a handle - explicit, or the implicit one behind a handle-less call - owns a control slot
 * whose address is baked into the launches made through it.  Destroy a handle (and call laser_shutdown,
 * which drops the implicit ones) only after the work enqueued through it has completed, and keep it
 * alive as long as a CUDA graph captured through it may be replayed: the slot goes back to a free list
 * and a later handle may be given it.  Implicit handles are keyed by (device, dims, options, workspace),
 * 16 per thread, least recently used evicted: a serving loop whose N or R change from step to step
 * should hold explicit handles of the capacity (N_alloc, R_max) instead - padding rows and empty
 * requests cost nothing - rather than churn implicit ones.
 *
 * laser_probe_handle_create   host; the current device must be a B200 (else LASER_E_ARCH).  options
 *                             NULL = defaults; options->token_ids (LASER_PROB_TOKEN) is remembered.
 * laser_probe_handle_run      laser_probe_confidence_opt with the handle's dims and options.
 * laser_probe_handle_run_host laser_probe_confidence_host[_async] (synchronize != 0 / == 0).
 * laser_probe_handle_plan     the handle's plan; kernel_launches says whether the tail is fused.
 */
typedef struct laser_probe_handle_s laser_probe_handle;
int laser_probe_handle_create(laser_probe_handle** out, const laser_probe_dims* dims,
                              const laser_probe_options* options);
int laser_probe_handle_destroy(laser_probe_handle* h);
int laser_probe_handle_plan(const laser_probe_handle* h, laser_probe_plan* plan);
size_t laser_probe_handle_workspace_bytes(const laser_probe_handle* h);
int laser_probe_handle_run(laser_probe_handle* h, const void* hidden, const void* W,
                           const int32_t* req_offsets, const float* load,
                           const laser_tau_params* tau_params, float* out_conf, int32_t* out_argmax,
                           uint8_t* out_exit, void* workspace, size_t workspace_bytes, void* stream,
                           float* out_tau_opt, float* out_pmax_opt);
int laser_probe_handle_run_host(laser_probe_handle* h, const void* h_hidden, const void* W,
                                const int32_t* h_req_offsets, const float* h_load,
                                const laser_tau_params* tau_params, float* h_out_conf,
                                int32_t* h_out_argmax, uint8_t* h_out_exit, void* workspace,
                                size_t workspace_bytes, void* d_staging, size_t staging_bytes,
                                void* stream, int synchronize);

/*
 * Vocabulary-parallel probe (SURVEY.md §8 e: the LM head's tensor-parallel layout).  GPU g holds the
 * rows [v_offset_g, v_offset_g + V_g) of W and the whole batch; the path becomes
 *
 *   every GPU:  laser_probe_partial  a1 + a2 over its shard -> one 16-byte record per row
 *   exchange :  the records of all G shards meet on every GPU, laid out [G, N]
 *   every GPU:  laser_probe_combine  merge of the G records per row, then a3, a4, a5 as above
 *
 * The merge is the associative operator the split-V path already uses, so the result equals the
 * single-GPU call up to the rounding order of the sum of exponentials.  The exchange is either a
 * collective of the caller (NCCL all-gather of N*16 bytes per GPU), or done by the producer itself:
 * with `peers`, laser_probe_partial stores each record straight into every GPU's gathered buffer
 * through peer-mapped pointers (NVLink) and then raises a flag there; laser_probe_combine waits for
 * the G flags.  No collective call, no host synchronisation.
 */
typedef struct {
    float m;       /* max logit over the shard (-inf: empty / padding row)                            */
    float s;       /* sum_v exp(logit - m) over the shard                                            */
    int32_t a;     /* GLOBAL vocabulary index of the lowest-index maximum (INT32_MAX: none)          */
    float l_tok;   /* logit of the row's token if the shard holds it, else -inf (LASER_PROB_TOKEN)   */
} laser_row_stats;

enum { LASER_MAX_PEERS = 16 };
/* Peer-push exchange (HOST struct).  peer_stats[g] / peer_flags[g] are device pointers valid on THIS
 * GPU that address GPU g's gathered buffer [world, N] and flag array [world] (peer-mapped, e.g.
 * CUDA IPC or symmetric memory; entry [rank] is this GPU's own).  `epoch` must increase by one per
 * exchange on every GPU and never be 0 (flags start at 0).  A gathered buffer may be rewritten two
 * exchanges later: alternate two (stats, flags) sets by epoch parity. */
typedef struct {
    int32_t rank, world;                       /* 0 <= rank < world <= LASER_MAX_PEERS */
    uint32_t epoch;
    laser_row_stats* peer_stats[LASER_MAX_PEERS];
    uint32_t* peer_flags[LASER_MAX_PEERS];
} laser_probe_peers;

/* a1 + a2 over one vocabulary shard.  dims->V = rows of W_shard; v_offset = global index of its row
 * 0; token_ids_opt (device int32 [N], GLOBAL ids) or NULL.  out_stats: device [N] or NULL (rows >=
 * req_offsets[R] get the neutral record {-inf, 0, INT32_MAX, -inf}).  peers_opt: see above; at least
 * one of out_stats / peers_opt must be given.  workspace as for laser_probe_confidence with the same
 * dims.  options: NULL or kernel_mode / overlap / tail (the aggregate fields are ignored here).
 * Asynchronous on `stream`.  One kernel: the tail of the fused kernel merges each row's records,
 * stores / pushes them, and the last CTA to finish raises the flags.  With LASER_TAIL_SEPARATE:
 * three kernels with peers (fused, reduce, signal), else two. */
int laser_probe_partial(const void* hidden, const void* W_shard, const int32_t* req_offsets,
                        const int32_t* token_ids_opt, const laser_probe_dims* dims, int32_t v_offset,
                        laser_row_stats* out_stats, const laser_probe_peers* peers_opt,
                        void* workspace, size_t workspace_bytes, void* stream,
                        const laser_probe_options* options);

/* Merge + a3-a5 over gathered statistics.  stats: device [G, N] (shard-major).  dims->N and dims->R
 * are used (d, V ignored but must be valid).  wait_flags_opt: device uint32 [G] or NULL; when given
 * every block first waits until all G flags have reached `epoch` (peer-push exchange); a flag that
 * does not arrive within ~5 s makes the kernel trap (LASER_E_CUDA on the next call / sync) instead of
 * hanging the GPU.  One kernel. */
int laser_probe_combine(const laser_row_stats* stats, int32_t G, const int32_t* req_offsets,
                        const float* load, const laser_tau_params* tau_params, float* out_conf,
                        int32_t* out_argmax, uint8_t* out_exit, const laser_probe_dims* dims,
                        void* stream, float* out_tau_opt, float* out_pmax_opt,
                        const laser_probe_options* options, const uint32_t* wait_flags_opt,
                        uint32_t epoch);

/*
 * End-to-end form with HOST buffers for the per-step tensors (W stays resident on the device: it is
 * the model's weight, not a per-step input).  Copies hidden / req_offsets / load to the device
 * staging buffers, runs laser_probe_confidence, copies conf / argmax / exit back, and synchronises
 * `stream` before returning.  Host buffers should be pinned for the copies to be asynchronous; when
 * req_offsets, load and the three outputs are pinned AND device-mapped (cudaHostAlloc,
 * cudaHostRegister, torch pin_memory) the kernels access them in place over PCIe and only `hidden`
 * is copied (one transfer per call instead of six).  Pageable buffers take the staged path.
 *
 *   h_*          host pointers (same shapes and dtypes as above)
 *   d_staging    device scratch >= laser_probe_staging_bytes(dims), 256-byte aligned
 *   W, workspace as above (device)
 */
size_t laser_probe_staging_bytes(const laser_probe_dims* dims);
int laser_probe_confidence_host(const void* h_hidden, const void* W, const int32_t* h_req_offsets,
                                const float* h_load, const laser_tau_params* tau_params,
                                float* h_out_conf, int32_t* h_out_argmax, uint8_t* h_out_exit,
                                const laser_probe_dims* dims, void* workspace,
                                size_t workspace_bytes, void* d_staging, size_t staging_bytes,
                                void* stream);
/* Same without the final synchronisation: returns after enqueueing the copies and the kernels on
 * `stream`; results are in the host buffers once `stream` has been synchronised by the caller.  With
 * two (staging, workspace, output) sets on two streams a serving loop overlaps the host->device copy
 * of batch i+1 with the kernels of batch i.  Host buffers must stay valid until then. */
int laser_probe_confidence_host_async(const void* h_hidden, const void* W,
                                      const int32_t* h_req_offsets, const float* h_load,
                                      const laser_tau_params* tau_params, float* h_out_conf,
                                      int32_t* h_out_argmax, uint8_t* h_out_exit,
                                      const laser_probe_dims* dims, void* workspace,
                                      size_t workspace_bytes, void* d_staging, size_t staging_bytes,
                                      void* stream);

/* Host, scalar-array version of a4 (Eq. 5 + clamp) in the same float arithmetic as the kernel. */
int laser_tau_from_load(const float* load, int32_t R, const laser_tau_params* tau_params,
                        float* out_tau);

/* Control-plane helpers either side of the probe in Algorithm 1 (host scalars, "O(1)").
 * EMA: lbar <- alpha*L + (1-alpha)*lbar, in place over R independent trackers. */
int laser_ema_update(float* lbar, const float* L, int32_t R, float alpha);

/* Budget pre-allocation, Eq. 6-8; defaults PAPER.md:166, 195.  IEEE double
 * throughout.  Eq. 6 takes the floor of a real-number product; its binary evaluation can land a hair
 * below an integer the exact product reaches (paper defaults, |p| = 100: f_diff = 0.6 + 50/225 * 0.9
 * = 0.8 exactly, B = floor(10 * 0.8) = 8, yet 0.6 + 50.0/225.0*0.9 = 0.7999999999999999 in binary).
 * The floor is therefore taken of product + LASER_BUDGET_FLOOR_EPS (reading A19). */
#define LASER_BUDGET_FLOOR_EPS 1e-9
typedef struct {
    double b_base;   /* 10  */
    double b_min;    /* 2   */
    double f_min;    /* 0.6 */
    double f_max;    /* 1.5 */
    double p_min;    /* 50  */
    double p_max;    /* 275 */
    double l_target; /* 10  */
} laser_budget_params;
int laser_budget_params_default(laser_budget_params* out);
int laser_allocate_budget(const int32_t* prompt_tokens, const float* L, int32_t R,
                          const laser_budget_params* params, int32_t* out_budget);

/*
 * Per-kernel timing for bench / profiling (thread-local; off by default).  While enabled, each
 * laser_probe_confidence* call on this thread records CUDA events on its stream before the fused
 * kernel, after it and after the finalize kernel if the call has one (up to 512 calls; programmatic
 * dependent launch is not used for those calls).  With the fused tail ms_finalize_sum is 0: merge and
 * a3-a5 are inside the fused kernel's duration.  laser_profile_read() waits for the last recorded
 * call, returns the summed durations in milliseconds and the number of calls, and resets the count.
 */
int laser_profile_enable(int on);
int laser_profile_read(float* ms_fused_sum, float* ms_finalize_sum, int32_t* calls);

/* Text for a status code; never NULL. */
const char* laser_status_string(int status);
/* Detail of the last LASER_E_CUDA on this thread ("" if none). */
const char* laser_last_error(void);
/* Number of kernels this library has enqueued since load (all threads). */
uint64_t laser_kernel_launch_count(void);
/* Drops the implicit handles (the calling thread's at once, every other thread's at that thread's next
 * call) with their cached TMA descriptors, and frees a device's control block once no handle holds a slot
 * of it any more (explicit handles are the caller's to destroy first).  Call it when the work enqueued
 * through the library has completed.  The library stays usable: the next call builds what it needs again.
 * The 4 MiB array of laser_probe_confidence_static is part of the device image and stays. */
int laser_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* LASER_PROBE_H_ */
