// astra_internal.h -- structures shared by the host loader and the CUDA engine.
// Not part of the public ABI (include/astra.h is).  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

typedef uint32_t u32;
typedef uint64_t u64;

// ---------------------------------------------------------------------------------------------
// Flit: one 128 B line in flight, 64 bits.
//   [0,20)  step id      [20,32) wavefront id within the owner GPU (cu*W + w)
//   [32,38) outstanding-slot index inside the wavefront (ack addressing)
//   [38,64) time field, 26 bits:
//             queued in a link FIFO : cycle of the FIFO append relative to the window start
//             accepted by the link  : arrival cycle at the link's head, mod 2^26
//             inject record         : append cycle (10 bits) | slot index in the cell << 10
// ---------------------------------------------------------------------------------------------
#define ASTRA_FLIT_TIME_SHIFT 38
#define ASTRA_FLIT_PAYLOAD_MASK ((1ull << ASTRA_FLIT_TIME_SHIFT) - 1)
#define ASTRA_TMASK26 0x3ffffffu
#define ASTRA_T_INF 0xffffffffu
#define ASTRA_NOTLOADED 0xffffffffu
#define ASTRA_TS_NONE32 0xffffffffu
#define ASTRA_NONE32 0xffffffffu
#ifndef ASTRA_WMAX
#define ASTRA_WMAX 512u                   // cap of the lookahead window in cycles (< 1024: 10-bit cycle fields in the flit)
#endif
#ifndef ASTRA_HOT_BUDGET_SINGLE
#define ASTRA_HOT_BUDGET_SINGLE (48u << 10)  // bytes of shared memory for hot arrays, batches of one-CTA points (the rest of the SM's 256 KB is L1)
#endif
#define ASTRA_HOT_BUDGET_GROUPS (64u << 10)  // ... batches with CTA groups
#define ASTRA_NW_MAX 4096                 // window bins per GPU and per link (route latency / lookahead window + 2, rounded up to a power of two)
#define ASTRA_ACK_LIST_CAP 4096u           // ack discovery list entries per (GPU, window bin); beyond: bitmap scan
#ifndef ASTRA_HEAVY_MIN
#define ASTRA_HEAVY_MIN 8u                // possible issues in a window from which a wavefront gets a warp of its own
#endif
#define ASTRA_HEAVY_MAX_PER_WORD 16        // more such wavefronts among 32 consecutive ones: they stay on their threads
#ifndef ASTRA_SPARSE_CELLS_BELOW
#define ASTRA_SPARSE_CELLS_BELOW 0.125    // expected share of non-empty cells under which a multi-feeder link keeps a bitmap of them
#endif
#define ASTRA_LF_DELIVER_ONLY 1u           // lflag: every line over the link terminates at its head
#define ASTRA_LF_FORWARD_ONLY 2u           // lflag: every line over the link goes on to the single-feeder link lfwd[e]
#define ASTRA_LF_CELLS 3u                  // lflag: lines terminate at the head or go on to multi-feeder links only (cells)
#define ASTRA_GF_ISSUED_DEPS 1u            // gflag: some step of the GPU has an ISSUED-kind successor
#define ASTRA_GF_SERIAL 2u                 // gflag: the GPU model couples the wavefronts of a CU: cycle-serial issue path

// Link service kinds (R9): how the acceptance times of a FIFO are computed for a whole window.
#define ASTRA_LK_INT     0u               // bw = B*256: B lines every cycle, no carried credit
#define ASTRA_LK_PERIOD  1u               // 256 % bw == 0: one line every P = 256/bw cycles
#define ASTRA_LK_GENERAL 2u               // any other bw: saturating credit walked entry by entry

// Constant tables of a design point (u32 arrays in the batch's constant blob).
#define ASTRA_CONST_TABLES(X) \
    X(in_ptr) X(in_link) X(head) X(tail) X(leff) X(next_link) X(row_ptr) \
    X(step_od) X(lines) X(cu_lo) X(cu_n) X(succ_ptr) X(succ) X(ndeps) \
    X(step_q) X(step_r) X(first_link) X(step_alpha) X(step_aq) X(step_ar) X(cul_ptr) X(cul) X(rel_off) X(init_rel) X(init_rel_cnt) \
    X(ev_off) X(ring_off) X(ring_mask) X(lkind) X(ceilb) X(lstate0_init) X(mask_off) X(pre_off) X(nz_off) X(classoff) \
    X(nd_mw) X(nd_injoff) X(inj_off) X(part) X(predmask) X(gflag) X(gdirect) X(lflag) X(lfwd) X(lscr_off)

// Mutable arrays of a design point.  X(name, element type, init) with init: 0 zero, 1 0xff bytes,
// 2 written by the kernel's own initialisation, 3 scratch (no initialisation).
// Ordered by how often the per-window stages touch them: the loader places them in shared memory
// in this order until the budget is spent, the rest in the CTA group's global workspace.
#define ASTRA_WS_ARRAYS(X) \
    X(pipe_head, u32, 0) X(fifo_head, u32, 0) X(ltail, u32, 0) X(run, u32, 0) X(lstate0, u32, 2) X(lstate1, u32, 0) \
    X(link_lines, u32, 0) X(dirty, u32, 0) X(ndue, u32, 0) X(due_cnt, u32, 0) X(tl_lo, u32, 3) X(tl_n, u32, 3) X(tl_base, u32, 3) X(tbase, u32, 3) X(pcnt, u32, 2) X(ev_cnt, u32, 0) X(ack_n, u32, 0) \
    X(inj_n, u32, 0) X(want, u32, 0) X(freeb, u32, 2) X(amask, u32, 0) X(gmode, u32, 0) X(nheavy, u32, 0) X(turn, u32, 0) X(cnt, u32, 3) X(hist, u32, 3) X(sel, u32, 3) X(nz, u32, 0) X(masks, u32, 0) X(pre, u32, 3) \
    X(t_release, u32, 2) X(issued_cnt, u32, 0) X(t_issued, u32, 0) X(deliv_cnt, u32, 0) X(t_deliv, u32, 0) \
    X(ack_cnt, u32, 0) X(t_ack, u32, 0) X(ndep_left, u32, 2) X(rel_time, u32, 0) X(plist, u32, 2) X(ev_list, u32, 3) \
    X(bin_cnt, u32, 0) X(cu_out, u32, 0) X(wf_busy, u64, 0) X(wf_rem, u32, 1) X(wf_cur, u32, 2) \
    X(hlist, u32, 3) X(undo_busy, u64, 3) X(undo_rem, u32, 3) X(undo_cur, u32, 3) X(undo_want, u32, 3) X(undo_freeb, u32, 3) \
    X(lscr, u32, 3) X(bitmap, u32, 0) X(ack_list, u32, 3) X(inj_list, u64, 3) X(ack_rec, u64, 3) X(ack_tmp, u64, 3) X(ack_sorted, u64, 3) X(evb, u64, 3) X(ring, u64, 3)

enum AstraConstId {
#define X(n) ASTRA_C_##n,
    ASTRA_CONST_TABLES(X)
#undef X
    ASTRA_C_COUNT
};
enum AstraArrId {
#define X(n, t, i) ASTRA_A_##n,
    ASTRA_WS_ARRAYS(X)
#undef X
    ASTRA_A_COUNT
};

#define ASTRA_DIAG_WORDS 144                // u64 per CTA: 16 common + 16 warp sets x 8 stage clocks (ASTRA_DIAG builds)
#define ASTRA_PLACE_SMEM (1ull << 63)     // a_off flag: offset is into the CTA's shared-memory hot region
#define ASTRA_PLACE_LOCAL (1ull << 62)    // a_off flag (CTA groups): the array holds only the CTA's own GPUs; indexed by absolute GPU id
                                          // through a pointer moved back by g_lo strides (hist: by the first out-link of g_lo)
// Arrays indexed by GPU (X(name, elements per GPU as an expression of P, bytes per element)): in a CTA group each CTA keeps only its GPUs' part.
#define ASTRA_GPU_ARRAYS(X) \
    X(want, P.nwords, 4) X(freeb, P.nwords, 4) X(amask, P.nwords, 4) X(undo_want, P.nwords, 4) X(undo_freeb, P.nwords, 4) \
    X(cnt, P.Wcyc, 4) X(sel, P.H, 4) X(wf_busy, P.CW, 8) X(undo_busy, P.CW, 8) X(wf_rem, P.CW, 4) X(wf_cur, P.CW, 4) \
    X(undo_rem, P.CW, 4) X(undo_cur, P.CW, 4) X(hlist, P.CW, 4)

// Per design point descriptor.  c_off are byte offsets into the batch's constant blob, a_off byte
// offsets into the hot region (flag set) or the workspace of the CTA group running the point,
// r_* byte offsets into the results blob.
struct PointDesc {
    u32 G, V, E, S;
    u32 C, Wv, K, H;
    u32 CW, nwords, slots, bmwords;
    u32 Wcyc, NW, kdiv_magic, NC;              // Wcyc lookahead window in cycles; NW power of two; kdiv_magic = ceil(2^32 / K); NC = W + 1
    u32 flags, group;                          // group: CTAs cooperating on this point
    u32 pcu, run_ahead;                        // pcu: ASTRA_GPU_ISSUE_PER_CU | ASTRA_GPU_CAP_PER_CU of the point's GPU model;
                                               // run_ahead: buffers are sized for nodes two windows apart (one CTA, <= 32 nodes)
    u32 hot_bytes, alcap;                      // alcap: entries per (GPU, window bin) ack discovery list
    u64 max_cycles;
    u64 total_lines;
    u64 ws_bytes;
    u64 c_off[ASTRA_C_COUNT];
    u64 a_off[ASTRA_A_COUNT];
    u64 a_bytes[ASTRA_A_COUNT];
    u64 r_step_ts, r_link_lines, r_summary, r_diag;
};

struct DeviceSummary {          // mirrors astra_summary, written by the kernel
    int32_t status; u32 n_steps, n_links, window;
    u64 completion_cycle, total_lines, busy_cycles, skipped_cycles;
};

// Control block of one CTA group in global memory (multi-CTA design points).
struct GroupCtl {
    u32 bar;            // monotone barrier counter; alone in its 128-byte line: every CTA of the group polls it
    u32 pad0[31];
    u32 point;          // queue index the group is running
    u32 acked;          // steps fully acked, all CTAs
    u32 err;
    u32 completion;     // max t_ack
    u32 hint[3];        // next-event time, rotated per window
    u32 pad[25];
};

// ---------------------------------------------------------------------------------------------
// Host-side objects
// ---------------------------------------------------------------------------------------------
struct HostTopo {
    u32 G = 0, NS = 0, V = 0, E = 0;
    std::vector<u32> node_lat, row_ptr, head, tail, bw, lat, leff;
    std::vector<u32> in_ptr, in_link;
    std::vector<u32> next_link;       // [V*G], 0xffffffff = none
    std::vector<u32> dist;            // [V*G], 0xffffffff = unreachable
    u32 min_leff = 0, max_leff = 0;
};

struct HostColl {
    u32 G = 0, S = 0;
    std::vector<u32> owner, dst, lines, cu_lo, cu_n;
    std::vector<u32> dep_ptr, dep_step; std::vector<uint8_t> dep_kind;
    std::vector<u32> succ_ptr, succ, ndeps;    // successor CSR (kind in bits 30..31), deduplicated deps
    u32 max_cu_end = 0;
    u64 total_lines = 0;
};

struct HostGpu { u32 C = 0, Wv = 0, K = 0, H = 0, mode = 0; };

struct Blob {                       // append-only byte buffer with 16-byte aligned sections
    std::vector<uint8_t> bytes;
    u64 add(const void* p, size_t n);
    template <class T> u64 add(const std::vector<T>& v) { return add(v.data(), v.size() * sizeof(T)); }
};

struct PlanOptions {
    u64 flags = 0;
    u64 max_cycles = 0;
    u32 group = 1;                  // CTAs per design point
    u32 hot_budget = 0;             // bytes of shared memory available for hot arrays
};

// loader entry points (astra_loader.cpp)
int32_t astra_build_topo(HostTopo& t, std::string& err);
int32_t astra_build_coll(HostColl& c, std::string& err);
int32_t astra_plan_point(const HostTopo& t, const HostColl& c, const HostGpu& g, const PlanOptions& opt,
                         const u64* topo_off, const u64* coll_off, Blob& blob, PointDesc& out, double& cost,
                         std::string& err);
double astra_point_cost(const HostTopo& t, const HostColl& c, u64 flags);
#define ASTRA_N_TOPO_TABLES 7
#define ASTRA_N_COLL_TABLES 7

// engine entry points (astra_engine.cu)
struct EngineLaunch {
    const uint8_t* d_const; uint8_t* d_ws; uint8_t* d_results;
    const PointDesc* d_points; const u32* d_order; u32* d_queue; GroupCtl* d_groups;
    u32 n_points;
    // scheduling classes: order[0, n_big) are the points that run on a group of `group` CTAs (n_slots
    // groups, workspace d_ws + slot * ws_big_stride), the rest run on one CTA each (workspace
    // d_ws + ws_single_off + cta * ws_single_stride); a group whose queue is empty turns into single CTAs
    u32 n_big, n_slots, group, grid;
    u64 ws_big_stride, ws_single_off, ws_single_stride;
    u32 warps_per_cta, hot_bytes;
    bool stage;                     // the CTAs carry the staging area for per-step constant tables (some point of the batch fits it)
    u32 variant;                    // 1: one CTA per SM (128 registers per thread), 2: two CTAs per SM (64)
};
int32_t astra_engine_launch(const EngineLaunch& L, void* stream, std::string& err);
int32_t astra_engine_occupancy(u32 warps_per_cta, u32 hot_bytes, u32 variant, bool stage, u32* ctas_per_sm, u32* n_sms, std::string& err);
u32 astra_engine_fixed_smem(u32 warps_per_cta, bool stage);
bool astra_engine_stageable(u32 warps_per_cta, u32 n_steps);   // the point's per-step constant tables fit the staging area
bool astra_engine_has_diag();
// No-allocation path (include/astra.h, astra_run_packed_noalloc): the library's static device scratch.
#define ASTRA_NOALLOC_HEADER_BYTES 512u    // queue counters + abort flag, one GroupCtl; cleared by every call
int32_t astra_engine_static_scratch(int device, uint8_t** ptr, std::string& err);       // set-up: once per device, that device current
int32_t astra_engine_launch_noalloc(int device, const uint8_t* d_const, const PointDesc* d_point, const u32* d_order,
                                    uint8_t* d_results, u64 ws_bytes, u32 warps_per_cta, u32 hot_bytes, u32 n_steps, void* stream, std::string& err);
