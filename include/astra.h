/*
 * astra.h -- C-ABI of the B200-native cycle-synchronous cache-line collective simulator.
 *
 * The hot path of ASTRA-sim 3.0 (arxiv/paper_2606_10440): compute units (CUs) of each simulated
 * GPU run wavefronts that issue one 128 B load from local HBM per cycle and store the line to a
 * peer GPU; the stores cross the links and switches of an InfraGraph-style topology; store-acks
 * return; a per-GPU step DAG releases the next step.  Many independent design points run as one
 * batch on one B200.  Every state variable and every output is an integer.
 *
 * Paper passages behind each call (PAPER.md line numbers; cycle-level rules are the readings
 * R1-R14 listed in DESIGN.md section 3, because the paper prints no equations):
 *   astra_load_infragraph  L225, L259 (InfraGraph = directed attributed graph, fully qualified
 *                          node/edge list), L49 + L221 (alpha-beta links, modular routing)
 *   astra_load_collective  L73, L173 (per-GPU, per-workgroup operation lists; control
 *                          dependencies), L150 (MemcpyOp = Load, Waitcnt, Store per cache line)
 *   astra_set_gpu          L189 (CUs), L165 (wavefronts), L209-L215 + L297 (in-flight cap),
 *                          L221 (memory channels -> HBM lines/cycle)
 *   astra_run_batch        L191, L203-L209 (per-cycle Wavefront Request injection), L35 (4-stage
 *                          put path), L289 (acknowledgment after remote Store)
 *   astra_read_results     L277 (collective time), plus per-step and per-link counters
 *
 * Conventions
 *   - All pointers are HOST pointers unless a parameter says "device".  The library copies every
 *     input array during the call; callers keep ownership and may free theirs at once.
 *   - Results are copied into caller-allocated host buffers.
 *   - astra_ctx owns all host and device memory it allocates; astra_destroy frees it.  One ctx is
 *     not thread-safe; separate ctxs are independent.  Loaded objects live until astra_destroy.
 *   - A batch runs as ONE cooperative kernel launch whose CTAs wait on each other (one CTA group per
 *     large design point): the CUDA runtime either makes the whole grid resident or refuses the
 *     launch.  While another kernel (another ctx, another stream, another process under MPS)
 *     occupies SMs, astra_run_batch may therefore fail with ASTRA_ELIMIT / ASTRA_ECUDA instead of
 *     running; it never hangs: group barriers give up after a few seconds without progress and the
 *     call returns ASTRA_ECUDA.
 *   - Every call returns 0 or a negative ASTRA_E* code and never throws or aborts;
 *     astra_last_error gives a message valid until the next call on the same ctx.
 *   - There is no CPU fallback: without a usable CUDA device astra_create fails with ASTRA_ECUDA.
 */
#ifndef ASTRA_H
#define ASTRA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ASTRA_OK            0
#define ASTRA_EINVAL       (-1)  /* malformed input (see validation rules below)            */
#define ASTRA_ENOMEM       (-2)  /* host or device allocation failed                        */
#define ASTRA_ECUDA        (-3)  /* CUDA runtime error / no device                          */
#define ASTRA_EUNREACHABLE (-4)  /* some step's owner has no route to its dst               */
#define ASTRA_ELIMIT       (-5)  /* exceeds an engine limit (see ASTRA_MAX_*)               */
#define ASTRA_ESTATE       (-6)  /* bad id, read before run, run while another is pending   */

/* Engine limits (flit bit widths: step 20 bits, wavefront 12 bits, slot 6 bits). */
#define ASTRA_MAX_STEPS            (1u << 20)
#define ASTRA_MAX_WAVEFRONTS       4096u      /* cus * wavefronts_per_cu per GPU */
#define ASTRA_MAX_OUTSTANDING      64u        /* per wavefront                    */
#define ASTRA_MAX_GPUS             65535u
#define ASTRA_MAX_LINK_LATENCY     (1u << 24) /* latency + node_latency           */
#define ASTRA_MAX_BW_Q8            (31u * 256u) /* at most 31 lines/cycle per link */
#define ASTRA_MAX_HBM_LINES        1023u      /* hbm_lines_per_cycle (10-bit slot index inside a cycle's cell) */
#define ASTRA_MAX_CYCLES           (0xffffffffull - (1ull << 25)) /* cycle counters are 32 bits on the device:
                                                 astra_run_batch CLAMPS max_cycles to this value, so a run that
                                                 needs more cycles reports ASTRA_STATUS_MAX_CYCLES at this cycle */

/* Dependency kinds: which timestamp of the producer step the consumer waits for (R3). */
#define ASTRA_DEP_DELIVERED 0    /* producer's last line reached its dst;  needs dst(p)   == owner(s) */
#define ASTRA_DEP_ACKED     1    /* producer's last ack processed at owner; needs owner(p) == owner(s) */
#define ASTRA_DEP_ISSUED    2    /* producer's last line issued;            needs owner(p) == owner(s) */

/* astra_create flags */
#define ASTRA_FLAG_NONE           0ull
#define ASTRA_FLAG_NO_WINDOW_SKIP 1ull   /* step through every lookahead window (testing I8)   */
#define ASTRA_FLAG_WINDOW_1       2ull   /* force a 1-cycle lookahead window (testing I8)      */
#define ASTRA_FLAG_SERIAL_ISSUE   4ull   /* always take the cycle-serial issue path (testing)  */
#define ASTRA_FLAG_NO_HEAVY        16ull  /* no warp-per-wavefront issue path (testing)         */
#define ASTRA_FLAG_NO_PRIORITY_SWEEP 32ull /* budget-bound windows take the cycle-serial path (testing) */
#define ASTRA_FLAG_RUN_AHEAD     64ull  /* one-CTA points of up to 32 nodes: no block barrier per window, a node starts its next
                                         * window as soon as the nodes it depends on have completed the current one.  Same
                                         * results; measured slower on B200 (config 4 +11 %: the barrier keeps the warps of a
                                         * CTA in the same stage and so in the same instruction-cache lines), hence opt-in */
#define ASTRA_FLAG_SERIAL_ARRIVALS 8ull  /* one task per in-link, no chunking (testing)        */
#define ASTRA_FLAG_WARPS(w) (((uint64_t)(w) & 0x3full) << 20) /* CTA shape: w in {1,2,4,8,16} warps per CTA, 16/w CTAs per SM
                                            (0 = engine's choice) */
#define ASTRA_FLAG_GROUP(g) (((uint64_t)(g) & 0xffull) << 8) /* run every design point on a group of g
                                            CTAs (1..255, at most the co-resident CTAs of the device), one node range each; 0 = engine's choice */

/* Per-point simulation outcome */
#define ASTRA_STATUS_DONE       0
#define ASTRA_STATUS_MAX_CYCLES 1    /* watchdog: cycle max_cycles reached before completion */
#define ASTRA_STATUS_DEADLOCK   2    /* no pending event and not finished                    */
#define ASTRA_STATUS_INTERNAL   3    /* engine self-check failed (ring overflow guard etc.)  */

#define ASTRA_TS_NONE UINT64_MAX     /* a timestamp that never happened */

typedef struct astra_ctx astra_ctx;  /* opaque */

typedef struct {
    uint32_t topo_id, coll_id, gpu_id, reserved;
} astra_point;

typedef struct {
    int32_t  status;            /* ASTRA_STATUS_*                                              */
    uint32_t n_steps, n_links;
    uint32_t window;            /* lookahead window (cycles) the engine used, diagnostic       */
    uint64_t completion_cycle;  /* max over steps of t_ack (R14)                               */
    uint64_t total_lines;       /* sum of lines over steps == transactions simulated           */
    uint64_t busy_cycles;       /* diagnostic: node-cycles actually stepped, summed over nodes */
    uint64_t skipped_cycles;    /* diagnostic: node-cycles skipped as idle, summed over nodes  */
} astra_summary;

/* Create a context bound to CUDA device `cuda_device`.  Fails with ASTRA_ECUDA when no such
 * device is usable.  `flags`: ASTRA_FLAG_*. */
int32_t astra_create(astra_ctx** out, int32_t cuda_device, uint64_t flags);
int32_t astra_destroy(astra_ctx* ctx);
const char* astra_last_error(const astra_ctx* ctx);

/* Optional: run on a caller-provided CUDA stream (a cudaStream_t passed as void*; e.g. the
 * torch current stream).  NULL = the ctx's own stream.  The stream stays owned by the caller. */
int32_t astra_set_stream(astra_ctx* ctx, void* cuda_stream);

/* Topology (R4, R5).  Nodes 0..n_gpus-1 are GPUs (node id == rank); n_gpus..n_gpus+n_switches-1
 * are switches.  CSR by TAIL node: links of node v are [row_ptr[v], row_ptr[v+1]); link id == CSR
 * position.  Within a row heads must be strictly ascending (no parallel links), no self loops.
 *   node_latency [V]   cycles added when a line TRANSITS (or enters) the node; GPUs normally 0
 *   row_ptr      [V+1]
 *   head         [E]
 *   bw_q8        [E]   lines/cycle * 256, 0 < bw_q8 <= ASTRA_MAX_BW_Q8
 *   latency      [E]   cycles, >= 1
 * EINVAL on malformed CSR / zero bandwidth / zero latency; ELIMIT beyond the limits above. */
int32_t astra_load_infragraph(astra_ctx* ctx, uint32_t n_gpus, uint32_t n_switches,
                              const uint32_t* node_latency, const uint32_t* row_ptr,
                              const uint32_t* head, const uint32_t* bw_q8, const uint32_t* latency,
                              uint32_t* out_topo_id);

/* Collective (R3, R11).  Step s: GPU owner[s] sends lines[s] 128 B lines to dst[s], executed by
 * CUs [cu_lo[s], cu_lo[s]+cu_n[s]) of the owner.  Dependencies of s are
 * dep_step[dep_ptr[s] .. dep_ptr[s+1]) with kinds dep_kind[] (ASTRA_DEP_*); every dependency id
 * must be < s and locally observable (see ASTRA_DEP_*).  EINVAL otherwise, or when lines == 0,
 * cu_n == 0, owner == dst, owner/dst >= n_gpus. */
int32_t astra_load_collective(astra_ctx* ctx, uint32_t n_gpus, uint32_t n_steps,
                              const uint32_t* owner, const uint32_t* dst, const uint32_t* lines,
                              const uint32_t* cu_lo, const uint32_t* cu_n,
                              const uint32_t* dep_ptr, const uint32_t* dep_step,
                              const uint8_t* dep_kind, uint32_t* out_coll_id);

/* GPU model (R11-R13): cus CUs, wavefronts_per_cu wavefronts each issuing at most one line per
 * cycle, at most max_outstanding un-acked lines per wavefront, at most hbm_lines_per_cycle load
 * grants per GPU per cycle.  All must be >= 1. */
int32_t astra_set_gpu(astra_ctx* ctx, uint32_t cus, uint32_t wavefronts_per_cu,
                      uint32_t max_outstanding, uint32_t hbm_lines_per_cycle, uint32_t* out_gpu_id);

/* The same GPU model with the paper's per-CU readings of two rules switched on by `mode` bits (DESIGN.md
 * section 3, R12' and R2'; astra_set_gpu is mode 0, the per-wavefront reading the BASELINE configs use):
 *   ASTRA_GPU_ISSUE_PER_CU  a CU dispatches at most one line per cycle, from its lowest-id ready wavefront
 *                           ("it can dispatch one cache-line-sized Wavefront Request in each
 *                           cycle", L191 "chooses a wavefront that is ready")
 *   ASTRA_GPU_CAP_PER_CU    max_outstanding bounds the un-acked lines of all wavefronts of a CU together
 *                           ("maximum number of outstanding requests per CU")
 * Such GPUs are stepped on the engine's cycle-serial issue path.  ELIMIT when wavefronts_per_cu > 32. */
#define ASTRA_GPU_ISSUE_PER_CU 1u
#define ASTRA_GPU_CAP_PER_CU   2u
int32_t astra_set_gpu_ex(astra_ctx* ctx, uint32_t cus, uint32_t wavefronts_per_cu,
                         uint32_t max_outstanding, uint32_t hbm_lines_per_cycle, uint32_t mode,
                         uint32_t* out_gpu_id);

/* Simulate n_points independent design points, each from t = 0 with empty queues (R1), until
 * every step is acked (R14) or cycle max_cycles (clamped to ASTRA_MAX_CYCLES) is reached.  Synchronous: returns when the
 * results are ready on the device.  EINVAL when a point's collective and topology disagree on
 * n_gpus or a CU range exceeds the GPU's CUs; EUNREACHABLE when a step has no route. */
int32_t astra_run_batch(astra_ctx* ctx, uint32_t n_points, const astra_point* points,
                        uint64_t max_cycles);

/* As astra_run_batch but only enqueues the device work on the ctx's stream; astra_sync waits.
 * A prepared batch (tables resident in device memory) is reused when the same points are run
 * again, so repeated calls measure device work only. */
int32_t astra_run_batch_async(astra_ctx* ctx, uint32_t n_points, const astra_point* points,
                              uint64_t max_cycles);
int32_t astra_sync(astra_ctx* ctx);

/* Results of design point `point` of the last batch (ESTATE before any run / bad index).
 *   step_ts    [4*n_steps] or NULL: release, issued, delivered, acked per step (ASTRA_TS_NONE
 *              if it never happened)
 *   link_lines [n_links]   or NULL: lines accepted per link */
int32_t astra_read_results(astra_ctx* ctx, uint32_t point, astra_summary* out,
                           uint64_t* step_ts, uint64_t* link_lines);

/* Diagnostics (libraries built with -DASTRA_DIAG only, ESTATE otherwise; the default build carries no
 * instrumentation): SM clocks of CTA `cta_rank` of the group that ran design point `point` of the last
 * batch.  out144[144]: [0] lookahead windows stepped, [5] state initialisation, [6] budget-bound
 * GPU-windows; then for each of the CTA's 16 warp sets s (a set steps one simulated node at a time)
 * eight counters at [16 + 8 s ..]: arrivals + ack discovery, release events, wavefront runs, budget check /
 * commit / cycle-serial path, placement, multi-feeder merge, link service, wait at the end-of-window barrier
 * -- clocks of the set's first warp, summed over the set's nodes and all windows. */
int32_t astra_read_diag(astra_ctx* ctx, uint32_t point, uint32_t cta_rank, uint64_t* out144);

/* Number of CTAs the engine assigned to design point `point` of the prepared batch (1 = one CTA). */
int32_t astra_point_group(astra_ctx* ctx, uint32_t point, uint32_t* group);

/* Diagnostics: device milliseconds (CUDA events on the ctx's stream) of the last batch and the
 * number of kernels it launched; bytes of device memory held by the prepared batch. */
int32_t astra_last_run_info(astra_ctx* ctx, float* device_ms, uint32_t* kernel_launches,
                            uint64_t* device_bytes);

/* Diagnostics: host->device bytes copied when the last batch was prepared (tables, descriptors,
 * queue order) and device->host bytes a full read-back of its results copies. */
int32_t astra_last_transfer_bytes(astra_ctx* ctx, uint64_t* h2d_bytes, uint64_t* d2h_bytes);

/* ---------------------------------------------------------------------------------------------
 * No-allocation entry point.  Some callers cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  For them one design point can be run with the
 * engine's whole scratch state (link rings, ack records, wavefront state, queue counters) in a
 * file-scope `static __device__` array of the library, ASTRA_NOALLOC_SCRATCH_BYTES large; every
 * GPU that loads the library holds that array until the process exits.
 *
 * Set-up (may allocate host memory; resolves the array's device address once per device):
 *   astra_pack_point  plans ONE design point (A0: routing, tables, array placement) for a single
 *                     CTA and writes its inputs -- constant tables, descriptor -- as one relocatable
 *                     blob of info->in_bytes bytes into host_buf (NULL / too small: only *info is
 *                     filled, ELIMIT when host_buf is non-NULL but too small).  The caller copies
 *                     that blob to device memory of its own (256-byte aligned).
 * Run (allocates nothing: no cudaMalloc / cudaFree / allocating library call, host or device):
 *   astra_run_packed_noalloc  enqueues on `cuda_stream` (NULL = the ctx's stream) a clear of the
 *                     scratch header and the step kernel on one CTA; inputs = the caller's device
 *                     copy of the blob (d_in), outputs = caller's device buffer d_out of
 *                     info->out_bytes bytes (256-byte aligned): step timestamps u64[4*n_steps] at
 *                     byte offset info->off_step_ts, lines per link u64[n_links] at
 *                     info->off_link_lines, an astra_summary at info->off_summary.  Asynchronous:
 *                     the caller synchronises the stream before reading d_out.
 * ELIMIT ("scratch ... exceeds") when info->scratch_bytes > ASTRA_NOALLOC_SCRATCH_BYTES; EINVAL on
 * a bad info / NULL buffers.  Same results as astra_run_batch on the same point.
 * All calls on a device share the one array, which keeps the previous call's contents: the entry
 * point clears what must start at zero (the queue / abort header) and the kernel initialises the
 * state arrays itself, but two calls that overlap on the GPU (different streams, two contexts,
 * two processes' worth of threads on one device) RACE -- serialise them.                       */
#define ASTRA_NOALLOC_SCRATCH_BYTES (16ull << 20)
#define ASTRA_PACKED_MAGIC 0x41535452504b3031ull   /* "ASTRPK01" */
typedef struct {
    uint64_t magic;             /* ASTRA_PACKED_MAGIC                                          */
    uint64_t in_bytes;          /* size of the packed input blob                               */
    uint64_t out_bytes;         /* size of the output buffer                                   */
    uint64_t scratch_bytes;     /* scratch the point needs (header + one CTA's workspace)      */
    uint64_t off_const, off_desc, off_order;            /* inside the input blob               */
    uint64_t off_step_ts, off_link_lines, off_summary;  /* inside the output buffer            */
    uint32_t n_steps, n_links, hot_bytes, warps;
} astra_packed_info;
int32_t astra_pack_point(astra_ctx* ctx, const astra_point* point, uint64_t max_cycles,
                         void* host_buf, uint64_t host_buf_bytes, astra_packed_info* info);
int32_t astra_run_packed_noalloc(astra_ctx* ctx, const astra_packed_info* info,
                                 const void* d_in, void* d_out, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* ASTRA_H */
