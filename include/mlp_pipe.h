/*
 * mlp_pipe.h -- C ABI of the CTA-pipelined chained GEMM for one B200 (sm_100a).
 *
 * What the library computes (the hot path of arxiv/paper_2607_07862, "CTA-Pipelining"):
 *
 *     A^0 = X;   A^l = bf16( act_l( A^{l-1} . W_l ) ),  l = 1..L;   Y = A^L
 *
 *   - "two-layer GEMM workload ... where the output of the first GEMM is directly
 *     consumed by the subsequent GEMM"                 PAPER.md:107 (section III-B)
 *   - "Y = XAB"; bf16 in / bf16 out, fp32 tensor-core accumulator
 *                                                      PAPER.md:161
 *   - every intermediate A^l is a kernel OUTPUT materialised in global memory
 *     (arrow (1)), hence rounded to bf16 before the next layer reads it
 *   - act_l is applied on the fp32 accumulator for l < L and is the identity for l = L
 *     (the activation comes from BASELINE.json's configs; the paper omits it)
 *
 * and how: producer tiles (layer l) and consumer tiles (layer l+1) run at the same time
 * inside ONE persistent launch.  A producer's epilogue stores its output tile and then
 * publishes a ready counter (the paper's fence + scoreboard update, PAPER.md:95 steps
 * (1)-(4)); a consumer's prologue polls the counters it depends on before it loads the
 * intermediate (PAPER.md:95 step (5)); work is handed out by a global atomic ticket that
 * orders all tiles of layer l before those of layer l+1 (the ordering knob of
 * PAPER.md:99-101).  The same kernel also runs as the two baselines the paper compares
 * against: stream-ordered SEQUENTIAL launches and static MICROBATCH
 * chunk pipelining.
 *
 * Conventions for every entry point
 *   - plain C, no exceptions cross the boundary; every function returns an MLP_* status
 *     (0 = ok) unless stated otherwise.
 *   - "device pointer" = address in the current CUDA device's global memory (e.g.
 *     torch.Tensor.data_ptr()); "host pointer" = ordinary (ideally pinned) host memory.
 *   - bf16 = the upper 16 bits of an IEEE binary32, stored as uint16_t.
 *   - layouts: X [M x K] row-major (K contiguous); W_l [N_l x K_l] row-major (K_l
 *     contiguous, i.e. nn.Linear.weight; logical W_l[k][n] = stored[n][k]); Y [M x N_L]
 *     row-major.  The paper is silent on layout (its CUTLASS profiler chose).
 *   - every K_l, N_l must be a multiple of 8 and every pointer 16-byte aligned (TMA
 *     requirement); M >= 1 is arbitrary.
 *   - the caller owns X, W_l, Y and the stream; the library owns the hidden activations
 *     H_l, tickets, counters, the split-K workspace, tensor maps and internal streams.
 *   - a handle is NOT re-entrant: runs on one handle must be stream-ordered after one
 *     another (all counters are per handle).
 *   - co-residency: a persistent launch needs all its CTAs (<= one per SM) on the device at the
 *     same time, because waiting CTAs wait on work owned by other CTAs of the launch.  Launches
 *     that can wait are therefore cooperative (they queue behind other work instead of starting
 *     partially); see MLP_FLAG_NO_COOPERATIVE.
 *   - limits: ceil(N_l / 128) * ceil(M / tile_m) <= 65535 output tiles and K_l <= 64 * 65535 per
 *     layer (MLP_ERR_UNSUPPORTED beyond).
 *   - there is no CPU fallback: without an sm_100 device mlp_pipe_create fails with
 *     MLP_ERR_UNSUPPORTED.
 */
#ifndef MLP_PIPE_H_
#define MLP_PIPE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mlp_pipe mlp_pipe; /* opaque, library-owned */

enum { MLP_OK = 0, MLP_ERR_INVALID = 1, MLP_ERR_UNSUPPORTED = 2, MLP_ERR_CUDA = 3, MLP_ERR_OOM = 4, MLP_ERR_TIMEOUT = 5 };

/* dtype: bf16 in / bf16 out, fp32 accumulate -- the only one. */
enum { MLP_BF16 = 0 };

/* activation between layers (BASELINE.json configs; readings c1, c2).
 * GELU_TANH: g(x) = 0.5 x (1 + tanh(sqrt(2/pi) (x + 0.044715 x^3))). */
enum { MLP_ACT_NONE = 0, MLP_ACT_RELU = 1, MLP_ACT_GELU_TANH = 2 };

/* execution mode */
enum {
    MLP_SEQUENTIAL = 0,   /* one launch per layer, stream-ordered, no flags      */
    MLP_MICROBATCH = 1,   /* X split by rows into `chunks`; layer l of chunk i on stream l, after an
                             event on layer l-1 of chunk i */
    MLP_CTA_PIPELINED = 2 /* ONE persistent launch; tickets + ready counters */
};

#define MLP_MAX_LAYERS 8

/* mlp_mode.flags */
#define MLP_FLAG_TILE_MAJOR   0x1u  /* consumer layers hand out units tile-major (all K-slices of an
                                       output tile adjacent) instead of K-slice-major (default)      */
#define MLP_FLAG_DEBUG_DELAY  0x2u  /* test hook: producers of layer 1 sleep a pseudo-random time
                                       before publishing (adversarial schedule for the protocol)     */
#define MLP_FLAG_DEBUG_REVERSE 0x4u /* test hook: layer-1 units are handed out in reverse order       */
#define MLP_FLAG_NO_W_EVICT_FIRST 0x8u /* do not tag weight loads L2 evict-first                      */
#define MLP_FLAG_ACQUIRE_LOADS 0x40u /* consumer prologue polls every ready counter with ld.acquire.gpu (the literal
                                       form) instead of ld.relaxed.gpu + one fence.acq_rel.gpu per group of counters;
                                       also switches the scheduler's look-ahead fast path off                       */
/* Measurement knobs, each REMOVES one ingredient of the protocol to price it (results may be wrong; tests use them
 * only to show that the ingredient matters or what it costs): */
#define MLP_FLAG_EXP_NO_ACQUIRE_FENCE 0x10u /* no fence.acq_rel.gpu after the relaxed polls of the activation loader */
#define MLP_FLAG_EXP_NO_PROXY_FENCE   0x20u /* no fence.proxy.async between the acquire and the TMA loads of H       */
#define MLP_FLAG_EXP_NO_FAST_PATH     0x80u /* the scheduler never pre-checks a unit's ready counters                */
#define MLP_FLAG_EXP_NO_PREISSUE      0x100u /* the first weight / activation ring is not requested during setup     */
#define MLP_FLAG_PDL 0x800u         /* SEQUENTIAL only: layers 2.. are launched as PROGRAMMATIC DEPENDENTS of the layer
                                       before (cudaLaunchAttributeProgrammaticStreamSerialization; not in the paper, whose baseline
                                       only removes launch bubbles with CUDA Graphs): their
                                       CTAs start as SMs become free, set up and prefetch weights, and execute
                                       griddepcontrol.wait before the first load of the previous layer's output.  A
                                       stronger stream-ordered baseline than plain back-to-back launches.               */
#define MLP_FLAG_WORKQUEUE 0x1000u  /* CTA_PIPELINED only: the paper's literal protocol instead of polled ready
                                       counters.  Producer epilogue: dependency array -> scoreboard update -> push of the
                                       now-ready consumer units into a work queue; consumer prologue: a ticket is a queue
                                       POSITION, the CTA spins until an entry appears there and remaps its unit to it (units
                                       run in the order in which they became ready; the weights of a unit cannot be
                                       prefetched before the pop).  Split tiles are summed by the last-arriving slice.       */
#define MLP_FLAG_PAIR 0x2000u       /* CTA pairs (thread-block clusters of 2, tcgen05 cta_group::2):
                                       a pair executes one unit of 256 weight rows -- each CTA stages its own 128 rows and HALF
                                       of the activation tile, the leader schedules (one ticket per pair) and issues one MMA of
                                       M = 256 for both tensor cores; counters, partials and outputs stay per 128-row block.
                                       Halves the activation bytes an SM pulls per weight byte.  tile_m must be a multiple of
                                       32 (UNSUPPORTED otherwise), grid even, not with MLP_FLAG_WORKQUEUE.                      */
#define MLP_FLAG_DEBUG_DROP_PUBLISH 0x4000u /* test hook: the producer of output tile 0 of the first layer never publishes its
                                       ready counter, so its consumers starve until the flag-poll watchdog (timeout_ms) expires:
                                       the deterministic way to exercise MLP_ERR_TIMEOUT.  One-shot: only the FIRST run of the
                                       handle drops the publish, so the runs after the reset are clean                            */
#define MLP_FLAG_NO_COOPERATIVE 0x8000u /* launch WITHOUT cudaLaunchAttributeCooperative.  By default every launch in which a CTA
                                       may wait on another CTA (CTA_PIPELINED, also as the two kernels of MLP_FLAG_TWO_KERNEL;
                                       split-K reduce units in any mode, also in the sibling launches of MLP_FLAG_MB_CORESIDENT)
                                       is cooperative: the grid starts only when all its CTAs fit on the device at once.  The one
                                       exception is MLP_FLAG_PDL, whose dependent launches are meant to start while the launch
                                       before still holds SMs (measured: cooperative costs the sibling modes nothing).  With this flag the
                                       caller guarantees that (an otherwise idle GPU, no second handle running concurrently);
                                       otherwise waiting CTAs can starve CTAs that are not yet resident until the watchdog.   */
#define MLP_FLAG_MB_CORESIDENT 0x10000u /* MICROBATCH only: every launch gets num_SMs / min(L, chunks) CTAs instead of one per SM, so
                                       that the launches of different layers on their different streams fit on the device
                                       TOGETHER and layer l of chunk i+1 really overlaps layer l+1 of chunk i (PAPER.md:173,
                                       Fig. 3a).  Without it every launch is a full persistent grid that holds all SMs (shared
                                       memory allows one CTA per SM), and the second stream only gets SMs as the first's CTAs exit. */
#define MLP_FLAG_TWO_KERNEL 0x20000u /* CTA_PIPELINED, 2 layers: the paper's host organisation on one GPU (
                                       SURVEY.md NEXT-4).  The producer layer is a kernel of its own on an internal stream over
                                       sm_split x num_SMs CTAs (0 or 1 = one half), the consumer layer a second kernel on a
                                       second stream over the remaining SMs, gated by cuStreamWaitValue32 on the first ready
                                       counter reaching this run's value; inside the consumer kernel every unit polls its ready
                                       counters as usual.  Not capturable into a CUDA graph (the wait value is per run), not
                                       with MLP_FLAG_WORKQUEUE / PAIR / AUTOTUNE, not on a grid of 1 CTA -- each kernel needs
                                       one of its own -- and not for chains other than 2 layers (UNSUPPORTED, from create and
                                       from mlp_pipe_plan alike).                                                              */
#define MLP_FLAG_AUTOTUNE 0x400u    /* measured plan search: the FIRST mlp_pipe_run on the handle (outside stream
                                       capture) tries the planner's candidate K-splits / ticket orders (and, unless tile_n is given,
                                       both unit heights 128 / 256; for M >= 1024, where they can pay, also CTA pairs as under
                                       MLP_FLAG_PAIR, if the handle could have been created with that flag) on the
                                       caller's buffers, timing each with the in-kernel clock, and keeps the
                                       fastest.  That one call synchronises the device, may allocate, and takes
                                       tens of milliseconds (up to a second or two for M in the thousands); Y is valid after it.  Results are remembered per
                                       process for equal (shape, mode).  MICROBATCH candidates are timed from fork to join
                                       with CUDA events (its launches overlap).  If the
                                       first run is being captured into a CUDA graph the search is skipped for good. */

typedef struct {
    int kind;        /* MLP_SEQUENTIAL | MLP_MICROBATCH | MLP_CTA_PIPELINED                           */
    int chunks;      /* MICROBATCH: number of row chunks, must divide M; ignored otherwise            */
    float sm_split;  /* CTA_PIPELINED: fraction in (0,1] of the CTAs that draw layer-1 units first;
                        the others start on layer 2 at once (prefetch W_2, poll for H).  1 = the pure
                        single-ticket scheme.  0 is read as 1.                                         */
    int tile_m;      /* tokens per tile (the tcgen05 N extent): 0 = auto, else a multiple of 16 <= 256 */
    int tile_n;      /* weight rows per unit: 0 = auto, 128, or 256 (two 128-row MMAs per K step that share
                        the activation tile; needs 2 * tile_m <= 512 TMEM columns)                      */
    int tile_k;      /* contraction elements per pipeline stage: 0 or 64                               */
    int stages;      /* shared-memory ring depth: 0 = as many as fit                                   */
    int kslice_tiles;/* producer tiles per ready counter: 0 or 1 (one counter per (M-block, K-slice))  */
    int split_k;     /* split of the contraction per output tile: 0 = auto, else applied to all layers */
    unsigned flags;  /* MLP_FLAG_*                                                                     */
    int split_k_layer[MLP_MAX_LAYERS]; /* per-layer override of split_k (0 = use split_k / auto)       */
    int grid;        /* CTAs of the persistent launch: 0 = one per SM                                  */
    int w_group;     /* weight K-blocks (128-byte row pieces) requested back to back: 0 = auto, <= stages   */
    int timeout_ms;  /* flag-poll watchdog: 0 = 2000 ms.  On expiry the kernel stops waiting, finishes
                        with undefined output and the handle reports MLP_ERR_TIMEOUT                   */
    int a_stages;    /* activation ring depth: 0 = as deep as the weight ring (the two rings then share their
                        barriers: one wait + one commit per K-block); another value gives the ring its own  */
} mlp_mode;

/*
 * Create a handle for Y = act(X.W1).W2, X [M x K], W1 [N1 x K], W2 [N2 x N1].
 * mode == NULL selects CTA_PIPELINED with every field auto.  Allocates all library-owned
 * device memory here; *out is set only on MLP_OK.
 * Errors: INVALID (null out, non-positive dims, dims not multiples of 8, bad mode fields,
 * chunks not dividing M), UNSUPPORTED (no sm_100 device, dtype != MLP_BF16, tile shape outside
 * the compiled set), OOM, CUDA.
 */
int mlp_pipe_create(mlp_pipe** out, int M, int K, int N1, int N2, int dtype, int act, const mlp_mode* mode);

/*
 * Same for an L-layer chain ("intermediate kernels act as both producers and
 * consumers"; BASELINE.json configs[4]).  widths[0..n_layers] = K, N_1, ..., N_L (host
 * pointer, copied).  1 <= n_layers <= MLP_MAX_LAYERS.  act after layers 1..L-1, none after L.
 */
int mlp_pipe_create_chain(mlp_pipe** out, int M, int n_layers, const int* widths, int dtype, int act,
                          const mlp_mode* mode);

/*
 * One pass of the whole path.  X, W1, W2, Y: device pointers (layouts above).  cuda_stream:
 * a cudaStream_t (NULL = the legacy default stream).  Asynchronous: enqueues on the stream
 * and returns; no host synchronisation, no allocation.  Y is fully overwritten.
 * Errors: INVALID (null / misaligned pointer), CUDA (launch failure, see last_error),
 * TIMEOUT (a previous run on this handle hit the watchdog: the kernel mirrors its status word into
 * pinned host memory, so the first mlp_pipe_run AFTER the expired kernel has finished sees it without
 * a device round trip, synchronises, resets the handle's protocol state and returns TIMEOUT once; the
 * output of the expired run, and of runs that were already queued behind it, is undefined).
 */
int mlp_pipe_run(mlp_pipe* h, const void* X, const void* W1, const void* W2, void* Y, void* cuda_stream);

/* Chain form: W = host array of n_layers device pointers. */
int mlp_pipe_run_chain(mlp_pipe* h, const void* X, const void* const* W, void* Y, void* cuda_stream);

/*
 * End-to-end form with HOST buffers (bench.py's e2e leg): copies X and every W_l host->device
 * into library-owned staging buffers, runs, copies Y device->host and synchronises the stream
 * before returning.  X, W[l], Y are host pointers (pinned memory makes the copies asynchronous
 * and fast; pageable memory works).  h2d_bytes / d2h_bytes (optional) receive the bytes moved.
 */
int mlp_pipe_run_host(mlp_pipe* h, const void* X, const void* const* W, void* Y, void* cuda_stream,
                      size_t* h2d_bytes, size_t* d2h_bytes);

/*
 * Test hook: device pointer and size of hidden activation H_layer = A^layer, 1 <= layer < L
 * ([M x N_layer] bf16 row-major).  Valid until destroy.
 */
int mlp_pipe_hidden(mlp_pipe* h, int layer, void** dev_ptr, size_t* bytes);

/* Test hook: fill every H_l with the 16-bit pattern `pattern` (e.g. a bf16 NaN) on the stream,
 * so that a consumer that reads H before it is published poisons Y. */
int mlp_pipe_poison_hidden(mlp_pipe* h, uint16_t pattern, void* cuda_stream);

/*
 * Statistics of the most recent run.  Synchronises the device.  Fills as much of `out` as
 * `bytes` allows.  Also the place where a watchdog expiry is reported (returns MLP_ERR_TIMEOUT).
 */
typedef struct {
    int n_layers, grid, stages, tile_m;           /* resolved launch configuration                    */
    int split_k[MLP_MAX_LAYERS];                  /* resolved per-layer split                         */
    int units[MLP_MAX_LAYERS];                    /* tickets per layer (tiles x split MMA units + the
                                                     reduce units of split tiles, if any)             */
    int producer_ctas;                            /* CTAs that start on layer 1 (sm_split)            */
    uint32_t status;                              /* 0 ok, else device-side abort code                */
    uint64_t runs;                                /* completed launches counted by the device epoch   */
    uint64_t flag_stall_cycles_sum;               /* sum over CTAs of SM cycles spent polling flags    */
    uint64_t flag_stall_cycles_max;               /* max over CTAs                                    */
    uint64_t flag_polls;                          /* polls (relaxed, or ld.acquire with MLP_FLAG_ACQUIRE_LOADS) that found the slice not ready */
    uint64_t kernel_cycles_max;                   /* max over CTAs of the CTA's lifetime in SM cycles */
    uint32_t units_done[MLP_MAX_LAYERS];          /* units executed per layer, summed over CTAs       */
    uint32_t units_by_consumer_ctas[MLP_MAX_LAYERS]; /* of which by CTAs in the consumer-first group  */
    uint32_t ready_ok;                            /* 1 if every ready counter / ticket / arrival
                                                     counter holds its expected post-run value       */
    int tile_n;                                   /* resolved weight rows per unit (128 or 256)       */
    int reduce_mode[MLP_MAX_LAYERS];              /* how split tiles are summed: 0 not split, 1 by the
                                                     last-arriving slice, 2 by reduce units           */
} mlp_stats;
int mlp_pipe_stats(mlp_pipe* h, mlp_stats* out, size_t bytes);

/*
 * Profiling hook (the paper's in-kernel timestamp instrumentation): per-CTA records
 * of the most recent launch of launch class `cls` (0 for CTA_PIPELINED; the layer index for
 * SEQUENTIAL / MICROBATCH / the two kernels of MLP_FLAG_TWO_KERNEL).  Copies min(max_records, CTAs of that class's
 * launch) records to the host array `out` -- the grid, except under MLP_FLAG_TWO_KERNEL, where each kernel has its own
 * share of it -- and returns the number copied through *n_out.  Synchronises the device.
 */
#define MLP_UNIT_TRACE 12
typedef struct {
    uint64_t flag_stall_cycles;   /* SM cycles the consumer prologue spent polling                        */
    uint64_t flag_polls;          /* unsuccessful polls                                                   */
    uint64_t cycles;              /* CTA lifetime in SM cycles                                            */
    uint64_t ts[8];               /* globaltimer ns: 0 CTA start, 1 setup done, 2 first ticket decoded,
                                     3 first weight TMA issued, 4 first stage landed, 5 first accumulator
                                     complete, 6 first unit stored (+published), 7 CTA exit               */
    uint64_t wait[8];             /* SM cycles: 0 weight loader inside its waits for a free stage (every wait is timed: one
                                     that succeeds at once still costs ~100 cycles per K-block), 1 reducer summing
                                     partials (gather loads + adds), 2 MMA blocked on operands, 3 MMA blocked
                                     on a free accumulator, 4 epilogue blocked on an accumulator, 5 reduce unit
                                     blocked on the arrival counter of its tile, 6 storing split-K partials,
                                     7 direct epilogue (TMEM -> act -> bf16 -> global)                      */
    uint32_t units[MLP_MAX_LAYERS]; /* units this CTA executed, per layer                                 */
    uint64_t unit_ts[MLP_UNIT_TRACE][4]; /* first MLP_UNIT_TRACE units of the CTA, globaltimer ns: weight
                                     loader starts the unit, weight loader has issued its last load,
                                     accumulator complete (T_mma), epilogue done incl. publish (T1)       */
    uint32_t unit_id[MLP_UNIT_TRACE]; /* layer << 28 | tile << 8 | K-slice (reduce unit: 0x80 | first column / 16) */
} mlp_cta_record;
int mlp_pipe_cta_records(mlp_pipe* h, int cls, mlp_cta_record* out, int max_records, int* n_out);

/*
 * The launch plan the library would use for this problem on a device with `num_sms` SMs, WITHOUT touching
 * a device (host logic only; works on a CPU-only box): tile shape, ring depths, per-layer split of the
 * contraction, how split tiles are summed, and the planner's latency estimate.  The ticket order itself
 * (step a1: the order in which work is handed out is the scheduling knob) is returned by
 * mlp_pipe_plan_units: unit i of `layer` is what ticket i of that layer executes.
 */
typedef struct {
    int tile_m, tile_n, m_blks, stages, a_stages, acc_stages, grid, producer_ctas, smem_bytes;
    int tiles[MLP_MAX_LAYERS];       /* output tiles per layer (m_blks x ceil(N / tile_n))               */
    int split_k[MLP_MAX_LAYERS];     /* K-slices per output tile                                          */
    int reduce_mode[MLP_MAX_LAYERS]; /* 0 not split, 1 last-arriving slice sums, 2 reduce units           */
    int ready_inc[MLP_MAX_LAYERS];   /* ready-counter increments per tile and run                         */
    int units[MLP_MAX_LAYERS];       /* tickets per layer                                                 */
    double model_us;                 /* planner's estimate of one run (device time, microseconds)         */
} mlp_plan;
typedef struct {
    uint16_t tile;     /* m_blk * n_blks + n_blk                                                          */
    uint8_t kind;      /* 0 = MMA unit over K-blocks [begin, end) (64 elements each); 1 = reduce unit over
                          token columns [begin, end) of the tile                                          */
    uint8_t k_slice;   /* MMA unit: index of its K-slice                                                  */
    uint16_t begin, end;
} mlp_unit;
int mlp_pipe_plan(int M, int n_layers, const int* widths, const mlp_mode* mode, int num_sms, mlp_plan* out);
/* Copies min(max_units, n) units of `layer` to out; *n_out = n, the number of tickets of that layer. */
int mlp_pipe_plan_units(int M, int n_layers, const int* widths, const mlp_mode* mode, int num_sms, int layer,
                        mlp_unit* out, int max_units, int* n_out);

/*
 * The same CTA-pipelined pass (one persistent launch, plan of a default CTA_PIPELINED handle) for
 * callers that cannot let this library allocate -- no handle, no cudaMalloc, no cudaFree, no pinned-memory or
 * stream / event creation, on the first call or on any later one.
 *
 * Who needs this.  mlp_pipe_create reserves the hidden activations, the split-K partials, the tickets and counters and
 * the unit tables with cudaMalloc.  Two kinds of caller cannot afford that: a serving process whose own memory manager
 * has already claimed the free HBM at start-up (KV-cache pools and the like), where a later cudaMalloc fails or eats into
 * a budget the library knows nothing about; and a decode loop that shares the GPU with other streams, where a
 * cudaMalloc / cudaFree in the middle of the loop can stall the whole device, not just the calling stream.  For them all of
 * that scratch lives in one fixed array of MLP_STATIC_SCRATCH_BYTES that is part of the library image: every GPU on which
 * the library runs a kernel holds these 32 MiB from the moment the library's code is loaded there until the process
 * exits, whether or not this function is ever called.
 *
 * Arguments: M tokens; widths[0..n_layers] = K, N_1, .., N_L (host pointer, 1 <= n_layers <= MLP_MAX_LAYERS); act as for
 * mlp_pipe_create; X [M x K], W[l] [N_{l+1} x N_l] (W = host array of n_layers DEVICE pointers), Y [M x N_L]: device
 * pointers owned by the caller, layouts and alignment as above; cuda_stream as for mlp_pipe_run.  Asynchronous: clears
 * the part of the array that must start at zero, sends the unit tables (a few KB, only when the shape differs from the
 * previous call's) and launches, all on the caller's stream, and returns.  The clear costs 2-3 us per call over
 * mlp_pipe_run on a handle, which keeps its counters from run to run instead (B200: 54 vs 51 us on the decode config).  Y is fully overwritten; plan and kernel are those of a handle created with mode == NULL, and so is the result.
 *
 * Limit: the plan's scratch (sum over layers of M x N_l x 2 bytes of hidden activations + tiles x split x tile bytes of
 * fp32 partials + a few hundred KB of counters, tables and records) must fit MLP_STATIC_SCRATCH_BYTES; all five
 * BASELINE.json configs do (the 4-layer chain needs about 24 MiB).  A larger problem is rejected with
 * MLP_ERR_UNSUPPORTED before anything is enqueued, and mlp_pipe_last_error(NULL) names the bytes it would have needed.
 *
 * Set-up: the FIRST call on each device looks up where that device keeps the array (a symbol look-up, which may load
 * the library's device code) with that device current; make that first call during start-up, before any stream capture
 * begins.  The first call for a new shape also plans it on the host (tens of milliseconds for the large configs); calls
 * that repeat the previous shape reuse that plan.
 *
 * Sharing: there is ONE array per device and every call uses it, whatever its shape, and finds in it what the call
 * before left behind.  Calls must therefore not overlap on the GPU: order them on one stream, or with events.  Two calls
 * in flight at once (two streams, two threads) clear and overwrite each other's counters and activations -- wrong output,
 * or CTAs that wait until the watchdog (2 s) lets them go.  Handles made by mlp_pipe_create have their own memory and may
 * run alongside.  This entry point keeps no pinned status mirror, so it cannot report a watchdog expiry; it returns only
 * what can be known at enqueue time.
 * Errors: INVALID (null / misaligned pointer, bad dims or act), UNSUPPORTED (no sm_100 device, scratch limit, unit-table
 * limits), CUDA (symbol look-up, memset, copy or launch failure).  Messages: mlp_pipe_last_error(NULL).
 */
#define MLP_STATIC_SCRATCH_BYTES (32u << 20)
int mlp_pipe_run_static(int M, int n_layers, const int* widths, int act, const void* X, const void* const* W, void* Y,
                        void* cuda_stream);

/* Free everything the handle owns (synchronises the device).  NULL is ignored. */
void mlp_pipe_destroy(mlp_pipe* h);

/* Static strings; never NULL. */
const char* mlp_status_string(int status);
/* Message of the last failing call on this handle (or on create, with h == NULL). */
const char* mlp_pipe_last_error(const mlp_pipe* h);

/* Library self-description: "mlp_pipe <version> sm_100a ..." */
const char* mlp_pipe_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MLP_PIPE_H_ */
