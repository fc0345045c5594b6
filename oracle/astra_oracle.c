/*
 * astra_oracle.c -- CPU ORACLE for the cycle-synchronous cache-line collective simulation.
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code with
 * the CUDA engine (paper_2606_10440_b200/csrc): no headers, no helpers, no tables.
 *
 * What it is: the method itself, executed one cycle at a time, single-threaded, with plain
 * growable queues -- the paper's fine-grained Load-Store simulation (section 4.1,
 * 4.4, 4.5) under the cycle rules R1-R14 of SURVEY.md 8(c) (restated in DESIGN.md section 3,
 * "Readings", because the paper itself prints no equations).  Per cycle t:
 *
 *   phase A1  arrivals    PAPER.md:L35 (iii)(iv), L221   -- pipes -> deliver | forward (R7)
 *   phase A2  inject      PAPER.md:L35 (ii)              -- lines issued at t-1 enter first hop
 *   phase A3  acks        PAPER.md:L289, L140            -- slot return, ack count, t_ack (R6)
 *   phase B   link accept PAPER.md:L49 (alpha-beta), L221 -- credit refill, FIFO -> pipe (R9)
 *   phase C   release     PAPER.md:L73                   -- step DAG (R3, R10)
 *   phase D   issue       PAPER.md:L165, L191, L203, L209 -- per-GPU fixed-priority scan (R11-R13)
 *
 * Routing (R5, "modular routing function"): static, destination based, minimum
 * total effective latency, candidates sorted by link id, candidate index (dst mod k).
 *
 * Nothing here is blocked, fused or reordered beyond that order.  Two bookkeeping shortcuts
 * that cannot change any decision are used and are individually switchable for testing:
 *   - phase C is re-evaluated only on cycles after some timestamp was stamped (its inputs
 *     are exactly the timestamps);
 *   - with ORACLE_FLAG_PRUNED_SCAN, phase D visits only wavefronts whose state changed since
 *     they were last found unable to issue (ack received, step of their CU range released,
 *     or they issued).  Every visited wavefront runs the same full check.  The default (flag
 *     clear) is the plain scan over all wavefronts; tests assert both give identical output.
 *
 * Round 2 adds the paper's own per-CU readings of two rules as OPTIONS (both off by default, so nothing above
 * changes, R12' and R2'):
 *   ORACLE_FLAG_ISSUE_PER_CU  a CU dispatches at most one line per cycle ("it can dispatch one
 *                             cache-line-sized Wavefront Request in each cycle", L203), choosing its lowest-id ready
 *                             wavefront (L191 "chooses a wavefront that is ready");
 *   ORACLE_FLAG_CAP_PER_CU    max_outstanding bounds the un-acked lines of all wavefronts of a CU together
 *                             ("maximum number of outstanding requests per CU").
 * Pinned by hand traces H1-H3 (tests/golden/pins_survey_8c.json).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): hand traces P1-P3, closed forms CF1/CF2,
 * config 1 in full (P4: completion 38,623), alpha-beta convergence P5, config 2 ring/direct
 * formulas P6/P7, invariants I1-I9, and agreement with an independently structured tiny
 * Python simulator on random cases.  Configs 3-5 have no closed form: "parity unpinned by
 * closed form" -- they are covered by the invariants and the brute-force cross-check only.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK            0
#define ORACLE_EINVAL       -1
#define ORACLE_ENOMEM       -2
#define ORACLE_EUNREACHABLE -4
#define ORACLE_EINTERNAL    -100

#define ORACLE_FLAG_PRUNED_SCAN 1u
#define ORACLE_FLAG_ISSUE_PER_CU 2u
#define ORACLE_FLAG_CAP_PER_CU   4u

#define DEP_DELIVERED 0
#define DEP_ACKED     1
#define DEP_ISSUED    2

#define TS_NONE UINT64_MAX
#define INF_DIST UINT64_MAX

typedef struct { uint32_t step, wf; } token_t;
typedef struct { uint64_t arrival; token_t tok; } pipe_entry_t;

/* ---- growable ring deques (logical FIFOs are unbounded, SURVEY "Capacity") ---- */
typedef struct { token_t *buf; uint64_t cap, head, len; } tokq_t;
typedef struct { pipe_entry_t *buf; uint64_t cap, head, len; } pipeq_t;

static int tokq_push(tokq_t *q, token_t v) {
    if (q->len == q->cap) {
        uint64_t ncap = q->cap ? q->cap * 2 : 16;
        token_t *nb = (token_t *)malloc(ncap * sizeof(token_t));
        if (!nb) return -1;
        for (uint64_t i = 0; i < q->len; i++) nb[i] = q->buf[(q->head + i) % q->cap];
        free(q->buf); q->buf = nb; q->cap = ncap; q->head = 0;
    }
    q->buf[(q->head + q->len) % q->cap] = v; q->len++;
    return 0;
}
static token_t tokq_pop(tokq_t *q) {
    token_t v = q->buf[q->head]; q->head = (q->head + 1) % q->cap; q->len--; return v;
}
static int pipeq_push(pipeq_t *q, pipe_entry_t v) {
    if (q->len == q->cap) {
        uint64_t ncap = q->cap ? q->cap * 2 : 16;
        pipe_entry_t *nb = (pipe_entry_t *)malloc(ncap * sizeof(pipe_entry_t));
        if (!nb) return -1;
        for (uint64_t i = 0; i < q->len; i++) nb[i] = q->buf[(q->head + i) % q->cap];
        free(q->buf); q->buf = nb; q->cap = ncap; q->head = 0;
    }
    q->buf[(q->head + q->len) % q->cap] = v; q->len++;
    return 0;
}
static pipe_entry_t pipeq_pop(pipeq_t *q) {
    pipe_entry_t v = q->buf[q->head]; q->head = (q->head + 1) % q->cap; q->len--; return v;
}
typedef struct { token_t *buf; uint64_t cap, len; } tokv_t;
static int tokv_push(tokv_t *q, token_t v) {
    if (q->len == q->cap) {
        uint64_t ncap = q->cap ? q->cap * 2 : 8;
        token_t *nb = (token_t *)realloc(q->buf, ncap * sizeof(token_t));
        if (!nb) return -1;
        q->buf = nb; q->cap = ncap;
    }
    q->buf[q->len++] = v; return 0;
}

/* ------------------------------------------------------------------------------------ */
/* Routing, R4 + R5.  dist[v*G+d] = minimum sum of Leff from node v to GPU d.            */
/* ------------------------------------------------------------------------------------ */
static int build_routes(uint32_t G, uint32_t V, uint32_t E,
                        const uint32_t *row_ptr, const uint32_t *head, const uint32_t *tail,
                        const uint64_t *leff, uint64_t *dist, uint32_t *next_link) {
    for (uint64_t i = 0; i < (uint64_t)V * G; i++) { dist[i] = INF_DIST; next_link[i] = UINT32_MAX; }
    for (uint32_t d = 0; d < G; d++) {
        dist[(uint64_t)d * G + d] = 0;
        /* Bellman-Ford relaxation towards d until nothing changes */
        int changed = 1;
        while (changed) {
            changed = 0;
            for (uint32_t e = 0; e < E; e++) {
                uint64_t dh = dist[(uint64_t)head[e] * G + d];
                if (dh == INF_DIST) continue;
                uint64_t cand = dh + leff[e];
                if (cand < dist[(uint64_t)tail[e] * G + d]) { dist[(uint64_t)tail[e] * G + d] = cand; changed = 1; }
            }
        }
        for (uint32_t v = 0; v < V; v++) {
            if (v == d) continue;
            uint64_t dv = dist[(uint64_t)v * G + d];
            if (dv == INF_DIST) continue;
            uint32_t k = 0;
            for (uint32_t e = row_ptr[v]; e < row_ptr[v + 1]; e++) {   /* ascending link id */
                uint64_t dh = dist[(uint64_t)head[e] * G + d];
                if (dh != INF_DIST && dh + leff[e] == dv) k++;
            }
            uint32_t want = d % k, idx = 0;
            for (uint32_t e = row_ptr[v]; e < row_ptr[v + 1]; e++) {
                uint64_t dh = dist[(uint64_t)head[e] * G + d];
                if (dh != INF_DIST && dh + leff[e] == dv) {
                    if (idx == want) { next_link[(uint64_t)v * G + d] = e; break; }
                    idx++;
                }
            }
        }
    }
    return 0;
}

static int validate_topology(uint32_t G, uint32_t NS, const uint32_t *row_ptr, const uint32_t *head,
                             const uint32_t *bw_q8, const uint32_t *latency) {
    uint32_t V = G + NS;
    if (G < 1) return ORACLE_EINVAL;
    if (row_ptr[0] != 0) return ORACLE_EINVAL;
    for (uint32_t v = 0; v < V; v++) {
        if (row_ptr[v + 1] < row_ptr[v]) return ORACLE_EINVAL;
        for (uint32_t e = row_ptr[v]; e < row_ptr[v + 1]; e++) {
            if (head[e] >= V || head[e] == v) return ORACLE_EINVAL;
            if (e > row_ptr[v] && head[e] <= head[e - 1]) return ORACLE_EINVAL;
            if (bw_q8[e] == 0 || latency[e] == 0) return ORACLE_EINVAL;
        }
    }
    return ORACLE_OK;
}

/* Exported for tests: routing tables only. dist as u64 [V*G], next_link u32 [V*G]. */
int oracle_route(uint32_t n_gpus, uint32_t n_switches, const uint32_t *node_latency,
                 const uint32_t *row_ptr, const uint32_t *head, const uint32_t *bw_q8,
                 const uint32_t *latency, uint64_t *dist_out, uint32_t *next_link_out) {
    uint32_t G = n_gpus, V = n_gpus + n_switches;
    int rc = validate_topology(G, n_switches, row_ptr, head, bw_q8, latency);
    if (rc) return rc;
    uint32_t E = row_ptr[V];
    uint32_t *tail = (uint32_t *)malloc(sizeof(uint32_t) * (E ? E : 1));
    uint64_t *leff = (uint64_t *)malloc(sizeof(uint64_t) * (E ? E : 1));
    if (!tail || !leff) { free(tail); free(leff); return ORACLE_ENOMEM; }
    for (uint32_t v = 0; v < V; v++)
        for (uint32_t e = row_ptr[v]; e < row_ptr[v + 1]; e++) {
            tail[e] = v; leff[e] = (uint64_t)latency[e] + node_latency[head[e]];
        }
    build_routes(G, V, E, row_ptr, head, tail, leff, dist_out, next_link_out);
    free(tail); free(leff);
    return ORACLE_OK;
}

/* trace record kinds */
#define TR_ISSUE   0
#define TR_ACCEPT  1
#define TR_DELIVER 2
#define TR_ACK     3
#define TR_RELEASE 4

#define TRACE(kind_, x_, y_, z_) do { \
    if (trace && tr_len < trace_cap) { uint64_t *r_ = trace + 5 * tr_len; \
        r_[0] = t; r_[1] = (kind_); r_[2] = (x_); r_[3] = (y_); r_[4] = (z_); } \
    tr_len++; } while (0)

/*
 * Run one design point.  All arrays are caller-owned.  step_ts is [4*S]:
 * release, issued, delivered, acked (TS_NONE if never).  stats (optional, [8]):
 * 0 cycles simulated, 1 max FIFO occupancy, 2 max pipe occupancy, 3 max acks in one cycle,
 * 4 max per-GPU issues in one cycle, 5 max `out` seen, 6 wavefront visits in phase D.
 * trace (optional): 5 u64 per event: cycle, kind, step, gpu*65536+wf... see TR_* (accept: z=link).
 */
int oracle_run(uint32_t n_gpus, uint32_t n_switches, const uint32_t *node_latency,
               const uint32_t *row_ptr, const uint32_t *head, const uint32_t *bw_q8,
               const uint32_t *latency,
               uint32_t n_steps, const uint32_t *owner, const uint32_t *dst, const uint32_t *lines,
               const uint32_t *cu_lo, const uint32_t *cu_n,
               const uint32_t *dep_ptr, const uint32_t *dep_step, const uint8_t *dep_kind,
               uint32_t cus, uint32_t wpc, uint32_t K, uint32_t H,
               uint64_t max_cycles, uint32_t flags,
               int32_t *status_out, uint64_t *completion_out, uint64_t *total_lines_out,
               uint64_t *step_ts, uint64_t *link_lines, uint64_t *stats,
               uint64_t *trace, uint64_t trace_cap, uint64_t *trace_len_out) {
    const uint32_t G = n_gpus, V = n_gpus + n_switches, S = n_steps;
    int rc = validate_topology(G, n_switches, row_ptr, head, bw_q8, latency);
    if (rc) return rc;
    const uint32_t E = row_ptr[V];
    if (cus == 0 || wpc == 0 || K == 0 || H == 0) return ORACLE_EINVAL;
    if (dep_ptr[0] != 0) return ORACLE_EINVAL;
    for (uint32_t s = 0; s < S; s++) {
        if (owner[s] >= G || dst[s] >= G || owner[s] == dst[s]) return ORACLE_EINVAL;
        if (lines[s] == 0 || cu_n[s] == 0) return ORACLE_EINVAL;
        if ((uint64_t)cu_lo[s] + cu_n[s] > cus) return ORACLE_EINVAL;
        if (dep_ptr[s + 1] < dep_ptr[s]) return ORACLE_EINVAL;
        for (uint32_t i = dep_ptr[s]; i < dep_ptr[s + 1]; i++) {
            uint32_t p = dep_step[i];
            if (p >= s) return ORACLE_EINVAL;
            if (dep_kind[i] == DEP_DELIVERED) { if (dst[p] != owner[s]) return ORACLE_EINVAL; }
            else if (dep_kind[i] == DEP_ACKED || dep_kind[i] == DEP_ISSUED) { if (owner[p] != owner[s]) return ORACLE_EINVAL; }
            else return ORACLE_EINVAL;
        }
    }

    const uint32_t WF = cus * wpc;              /* wavefronts per GPU, id = cu*wpc + w */
    int ret = ORACLE_OK;
    uint64_t tr_len = 0;

    /* ---- derived topology ---- */
    uint32_t *tail = (uint32_t *)calloc(E ? E : 1, sizeof(uint32_t));
    uint64_t *leff = (uint64_t *)calloc(E ? E : 1, sizeof(uint64_t));
    uint64_t *dist = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)V * G);
    uint32_t *next_link = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)V * G);
    uint32_t *in_ptr = (uint32_t *)calloc(V + 1, sizeof(uint32_t));
    uint32_t *in_link = (uint32_t *)calloc(E ? E : 1, sizeof(uint32_t));
    /* ---- per-link state ---- */
    tokq_t *fifo = (tokq_t *)calloc(E ? E : 1, sizeof(tokq_t));
    pipeq_t *pipe = (pipeq_t *)calloc(E ? E : 1, sizeof(pipeq_t));
    uint64_t *credit = (uint64_t *)calloc(E ? E : 1, sizeof(uint64_t));
    uint64_t *cap = (uint64_t *)calloc(E ? E : 1, sizeof(uint64_t));
    /* ---- per-step state ---- */
    uint64_t *issued_cnt = (uint64_t *)calloc(S ? S : 1, sizeof(uint64_t));
    uint64_t *deliv_cnt = (uint64_t *)calloc(S ? S : 1, sizeof(uint64_t));
    uint64_t *ack_cnt = (uint64_t *)calloc(S ? S : 1, sizeof(uint64_t));
    /* ---- per-CU step lists (R11) ---- */
    uint32_t *cul_ptr = (uint32_t *)calloc((size_t)G * cus + 1, sizeof(uint32_t));
    uint32_t *cul = NULL;
    /* ---- per-wavefront state ---- */
    uint32_t *wf_cur = (uint32_t *)calloc((size_t)G * WF, sizeof(uint32_t));   /* index into its CU list */
    uint32_t *wf_rem = (uint32_t *)calloc((size_t)G * WF, sizeof(uint32_t));   /* quota left; UINT32_MAX = not loaded */
    uint32_t *wf_out = (uint32_t *)calloc((size_t)G * WF, sizeof(uint32_t));
    uint32_t *cu_out = (uint32_t *)calloc((size_t)G * cus, sizeof(uint32_t));      /* un-acked lines per CU (R2') */
    uint64_t *cu_issued = (uint64_t *)calloc((size_t)G * cus, sizeof(uint64_t));   /* t + 1 of the CU's last issue (R12') */
    uint8_t *wf_maybe = (uint8_t *)malloc((size_t)G * WF);                     /* pruned scan only */
    uint32_t *gpu_unfinished = (uint32_t *)calloc(G, sizeof(uint32_t));        /* wavefronts with list not exhausted */
    uint32_t *gpu_maybe_cnt = (uint32_t *)calloc(G, sizeof(uint32_t));         /* pruned scan only: #wf_maybe set */
    tokv_t *pending = (tokv_t *)calloc(G, sizeof(tokv_t));                     /* issued at t-1, inject at t */
    tokv_t *acks = NULL;  uint64_t Tcal = 0;

    if (!tail || !leff || !dist || !next_link || !in_ptr || !in_link || !fifo || !pipe || !credit || !cap ||
        !issued_cnt || !deliv_cnt || !ack_cnt || !cul_ptr || !wf_cur || !wf_rem || !wf_out || !cu_out || !cu_issued || !wf_maybe ||
        !gpu_unfinished || !gpu_maybe_cnt || !pending) { ret = ORACLE_ENOMEM; goto done; }

    for (uint32_t v = 0; v < V; v++)
        for (uint32_t e = row_ptr[v]; e < row_ptr[v + 1]; e++) {
            tail[e] = v;
            leff[e] = (uint64_t)latency[e] + node_latency[head[e]];      /* R4 */
            in_ptr[head[e] + 1]++;
        }
    for (uint32_t v = 0; v < V; v++) in_ptr[v + 1] += in_ptr[v];
    {   /* in-links per head node, ascending link id */
        uint32_t *fill = (uint32_t *)calloc(V, sizeof(uint32_t));
        if (!fill) { ret = ORACLE_ENOMEM; goto done; }
        for (uint32_t e = 0; e < E; e++) { uint32_t h = head[e]; in_link[in_ptr[h] + fill[h]++] = e; }
        free(fill);
    }
    build_routes(G, V, E, row_ptr, head, tail, leff, dist, next_link);
    uint64_t max_alpha = 1, total_lines = 0;
    for (uint32_t s = 0; s < S; s++) {
        uint64_t a = dist[(uint64_t)owner[s] * G + dst[s]];
        if (a == INF_DIST) { ret = ORACLE_EUNREACHABLE; goto done; }
        if (a > max_alpha) max_alpha = a;
        total_lines += lines[s];
    }
    Tcal = max_alpha + 1;
    acks = (tokv_t *)calloc(Tcal, sizeof(tokv_t));
    if (!acks) { ret = ORACLE_ENOMEM; goto done; }

    for (uint32_t e = 0; e < E; e++) {
        cap[e] = 256ull * (((uint64_t)bw_q8[e] + 255) / 256);              /* R9 */
        credit[e] = cap[e];
        link_lines[e] = 0;
    }
    /* per-CU in-order step lists: steps whose CU range contains the CU, ascending id */
    for (uint32_t s = 0; s < S; s++)
        for (uint32_t c = cu_lo[s]; c < cu_lo[s] + cu_n[s]; c++) cul_ptr[(size_t)owner[s] * cus + c + 1]++;
    for (size_t i = 0; i < (size_t)G * cus; i++) cul_ptr[i + 1] += cul_ptr[i];
    cul = (uint32_t *)malloc(sizeof(uint32_t) * (cul_ptr[(size_t)G * cus] ? cul_ptr[(size_t)G * cus] : 1));
    if (!cul) { ret = ORACLE_ENOMEM; goto done; }
    {
        uint32_t *fill = (uint32_t *)calloc((size_t)G * cus, sizeof(uint32_t));
        if (!fill) { ret = ORACLE_ENOMEM; goto done; }
        for (uint32_t s = 0; s < S; s++)
            for (uint32_t c = cu_lo[s]; c < cu_lo[s] + cu_n[s]; c++) {
                size_t k = (size_t)owner[s] * cus + c;
                cul[cul_ptr[k] + fill[k]++] = s;
            }
        free(fill);
    }
    for (uint32_t g = 0; g < G; g++)
        for (uint32_t wf = 0; wf < WF; wf++) {
            size_t k = (size_t)g * cus + wf / wpc;
            wf_rem[(size_t)g * WF + wf] = UINT32_MAX;
            if (cul_ptr[k + 1] > cul_ptr[k]) gpu_unfinished[g]++;
        }
    memset(wf_maybe, 1, (size_t)G * WF);
    for (uint32_t g = 0; g < G; g++) gpu_maybe_cnt[g] = WF;
    for (uint32_t s = 0; s < 4 * S; s++) step_ts[s] = TS_NONE;

    uint64_t n_acked_steps = 0, in_flight = 0, completion = 0;
    uint64_t st_max_fifo = 0, st_max_pipe = 0, st_max_acks = 0, st_max_issue = 0, st_max_out = 0, st_visits = 0;
    int status = 1;
    int dirty_release = 1;          /* phase C must run at t = 0 */
    uint64_t t;

    for (t = 0; t < max_cycles; t++) {
        uint64_t issued_this_cycle = 0, released_this_cycle = 0;

        /* ---------------- phase A1: arrivals (R7) ---------------- */
        for (uint32_t v = 0; v < V; v++) {
            for (uint32_t ii = in_ptr[v]; ii < in_ptr[v + 1]; ii++) {
                uint32_t e = in_link[ii];
                pipeq_t *p = &pipe[e];
                while (p->len && p->buf[p->head].arrival == t) {
                    pipe_entry_t pe = pipeq_pop(p);
                    uint32_t s = pe.tok.step;
                    if (v == dst[s]) {
                        deliv_cnt[s]++;
                        TRACE(TR_DELIVER, s, (uint64_t)owner[s] * 65536 + pe.tok.wf, e);
                        if (deliv_cnt[s] == lines[s]) { step_ts[4 * s + 2] = t; dirty_release = 1; }
                        uint64_t a = dist[(uint64_t)owner[s] * G + dst[s]];          /* R6 */
                        if (tokv_push(&acks[(t + a) % Tcal], pe.tok)) { ret = ORACLE_ENOMEM; goto done; }
                    } else {
                        uint32_t f = next_link[(uint64_t)v * G + dst[s]];
                        if (tokq_push(&fifo[f], pe.tok)) { ret = ORACLE_ENOMEM; goto done; }
                        if (fifo[f].len > st_max_fifo) st_max_fifo = fifo[f].len;
                    }
                }
                if (p->len && p->buf[p->head].arrival < t) { ret = ORACLE_EINTERNAL; goto done; }
            }
        }
        /* ---------------- phase A2: inject lines issued at t-1 (R7) ---------------- */
        for (uint32_t g = 0; g < G; g++) {
            tokv_t *pd = &pending[g];
            for (uint64_t i = 0; i < pd->len; i++) {             /* already in ascending wavefront id */
                token_t tk = pd->buf[i];
                uint32_t f = next_link[(uint64_t)g * G + dst[tk.step]];
                if (tokq_push(&fifo[f], tk)) { ret = ORACLE_ENOMEM; goto done; }
                if (fifo[f].len > st_max_fifo) st_max_fifo = fifo[f].len;
            }
            pd->len = 0;
        }
        /* ---------------- phase A3: acks due at t (R6, R7) ---------------- */
        {
            tokv_t *b = &acks[t % Tcal];
            if (b->len > st_max_acks) st_max_acks = b->len;
            for (uint64_t i = 0; i < b->len; i++) {
                token_t tk = b->buf[i];
                uint32_t s = tk.step, g = owner[s];
                size_t w = (size_t)g * WF + tk.wf;
                if (wf_out[w] == 0) { ret = ORACLE_EINTERNAL; goto done; }
                wf_out[w]--;
                cu_out[(size_t)g * cus + tk.wf / wpc]--;
                if (!wf_maybe[w]) { wf_maybe[w] = 1; gpu_maybe_cnt[g]++; }
                if (flags & ORACLE_FLAG_CAP_PER_CU)            /* the slot returns to the CU's pool: any of its wavefronts may use it */
                    for (uint32_t x = (tk.wf / wpc) * wpc; x < (tk.wf / wpc + 1) * wpc; x++)
                        if (!wf_maybe[(size_t)g * WF + x]) { wf_maybe[(size_t)g * WF + x] = 1; gpu_maybe_cnt[g]++; }
                in_flight--;
                ack_cnt[s]++;
                TRACE(TR_ACK, s, (uint64_t)g * 65536 + tk.wf, 0);
                if (ack_cnt[s] == lines[s]) {
                    step_ts[4 * s + 3] = t; dirty_release = 1;
                    n_acked_steps++;
                    if (t > completion) completion = t;
                }
            }
            b->len = 0;
        }
        /* ---------------- phase B: link acceptance (R9) ---------------- */
        for (uint32_t e = 0; e < E; e++) {
            uint64_t c = credit[e] + bw_q8[e];
            if (c > cap[e]) c = cap[e];
            while (c >= 256 && fifo[e].len) {
                token_t tk = tokq_pop(&fifo[e]);
                pipe_entry_t pe; pe.arrival = t + leff[e]; pe.tok = tk;
                if (pipeq_push(&pipe[e], pe)) { ret = ORACLE_ENOMEM; goto done; }
                if (pipe[e].len > st_max_pipe) st_max_pipe = pipe[e].len;
                c -= 256;
                link_lines[e]++;
                TRACE(TR_ACCEPT, tk.step, (uint64_t)owner[tk.step] * 65536 + tk.wf, e);
            }
            credit[e] = c;
        }
        /* ---------------- phase C: DAG release (R10) ---------------- */
        if (dirty_release) {
            dirty_release = 0;
            for (uint32_t s = 0; s < S; s++) {
                if (step_ts[4 * s + 0] != TS_NONE) continue;
                int ok = 1;
                for (uint32_t i = dep_ptr[s]; i < dep_ptr[s + 1] && ok; i++) {
                    uint32_t p = dep_step[i];
                    uint64_t ts = dep_kind[i] == DEP_DELIVERED ? step_ts[4 * p + 2]
                                : dep_kind[i] == DEP_ACKED ? step_ts[4 * p + 3] : step_ts[4 * p + 1];
                    if (ts == TS_NONE || ts > t) ok = 0;
                }
                if (ok) {
                    step_ts[4 * s + 0] = t; released_this_cycle++;
                    TRACE(TR_RELEASE, s, 0, 0);
                    if (flags & ORACLE_FLAG_PRUNED_SCAN) {
                        uint32_t g = owner[s];
                        for (uint32_t wf = cu_lo[s] * wpc; wf < (cu_lo[s] + cu_n[s]) * wpc; wf++)
                            if (!wf_maybe[(size_t)g * WF + wf]) { wf_maybe[(size_t)g * WF + wf] = 1; gpu_maybe_cnt[g]++; }
                    }
                }
            }
        }
        /* ---------------- phase D: issue (R11, R12, R13) ---------------- */
        for (uint32_t g = 0; g < G; g++) {
            if (gpu_unfinished[g] == 0) continue;
            if ((flags & ORACLE_FLAG_PRUNED_SCAN) && gpu_maybe_cnt[g] == 0) continue;
            uint32_t budget = H;
            uint64_t issued_g = 0;
            for (uint32_t wf = 0; wf < WF && budget; wf++) {
                size_t w = (size_t)g * WF + wf;
                if ((flags & ORACLE_FLAG_PRUNED_SCAN) && !wf_maybe[w]) continue;
                uint32_t cu = wf / wpc, lane = wf % wpc;
                size_t ck = (size_t)g * cus + cu;
                if ((flags & ORACLE_FLAG_ISSUE_PER_CU) && cu_issued[ck] == t + 1) continue;   /* R12': the CU has dispatched this cycle */
                st_visits++;
                uint32_t len = cul_ptr[ck + 1] - cul_ptr[ck];
                int can = 0; uint32_t s = 0;
                while (wf_cur[w] < len) {                      /* in-order list, lazy advance (R11) */
                    s = cul[cul_ptr[ck] + wf_cur[w]];
                    if (step_ts[4 * s + 0] == TS_NONE) break;      /* not released: wait */
                    if (wf_rem[w] == UINT32_MAX) {
                        uint32_t m = cu_n[s] * wpc;
                        uint32_t j = (cu - cu_lo[s]) * wpc + lane;
                        wf_rem[w] = lines[s] / m + (j < lines[s] % m ? 1u : 0u);
                    }
                    if (wf_rem[w] == 0) {                         /* quota fully issued: move on */
                        wf_cur[w]++; wf_rem[w] = UINT32_MAX;
                        if (wf_cur[w] == len) gpu_unfinished[g]--;
                        continue;
                    }
                    can = 1; break;
                }
                if (can && ((flags & ORACLE_FLAG_CAP_PER_CU) ? cu_out[ck] < K : wf_out[w] < K)) {      /* R2 / R2' */
                    wf_out[w]++; cu_out[ck]++; cu_issued[ck] = t + 1; wf_rem[w]--; in_flight++;
                    if (wf_out[w] > st_max_out) st_max_out = wf_out[w];
                    issued_cnt[s]++;
                    TRACE(TR_ISSUE, s, (uint64_t)g * 65536 + wf, 0);
                    if (issued_cnt[s] == lines[s]) { step_ts[4 * s + 1] = t; dirty_release = 1; }
                    token_t tk; tk.step = s; tk.wf = wf;
                    if (tokv_push(&pending[g], tk)) { ret = ORACLE_ENOMEM; goto done; }
                    budget--; issued_g++;
                    /* it may issue again next cycle: stays a candidate */
                } else {
                    if (wf_maybe[w]) { wf_maybe[w] = 0; gpu_maybe_cnt[g]--; } /* cannot issue until ack / release */
                }
            }
            issued_this_cycle += issued_g;
            if (issued_g > st_max_issue) st_max_issue = issued_g;
        }
        /* ---------------- R14 termination ---------------- */
        if (n_acked_steps == S) { status = 0; t++; break; }
        if (in_flight == 0 && issued_this_cycle == 0 && released_this_cycle == 0 && !dirty_release) {
            status = 2; t++; break;                                /* nothing can ever change */
        }
    }

    if (status == 0) {
        /* I1: everything drained */
        for (uint32_t e = 0; e < E; e++) if (fifo[e].len || pipe[e].len) { ret = ORACLE_EINTERNAL; goto done; }
        for (uint64_t i = 0; i < Tcal; i++) if (acks[i].len) { ret = ORACLE_EINTERNAL; goto done; }
        if (in_flight) { ret = ORACLE_EINTERNAL; goto done; }
    }
    *status_out = status;
    *completion_out = completion;
    *total_lines_out = total_lines;
    if (stats) {
        stats[0] = t; stats[1] = st_max_fifo; stats[2] = st_max_pipe; stats[3] = st_max_acks;
        stats[4] = st_max_issue; stats[5] = st_max_out; stats[6] = st_visits; stats[7] = max_alpha;
    }
    if (trace_len_out) *trace_len_out = tr_len;

done:
    if (fifo) for (uint32_t e = 0; e < E; e++) free(fifo[e].buf);
    if (pipe) for (uint32_t e = 0; e < E; e++) free(pipe[e].buf);
    if (pending) for (uint32_t g = 0; g < G; g++) free(pending[g].buf);
    if (acks) for (uint64_t i = 0; i < Tcal; i++) free(acks[i].buf);
    free(tail); free(leff); free(dist); free(next_link); free(in_ptr); free(in_link);
    free(fifo); free(pipe); free(credit); free(cap);
    free(issued_cnt); free(deliv_cnt); free(ack_cnt);
    free(cul_ptr); free(cul); free(wf_cur); free(wf_rem); free(wf_out); free(cu_out); free(cu_issued); free(wf_maybe);
    free(gpu_unfinished); free(gpu_maybe_cnt); free(pending); free(acks);
    return ret;
}
