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
//   [38,64) arrival cycle mod 2^26 (meaningful in link latency pipes only)
// ---------------------------------------------------------------------------------------------
#define ASTRA_FLIT_TIME_SHIFT 38
#define ASTRA_TMASK26 0x3ffffffu
#define ASTRA_T_INF 0xffffffffu
#define ASTRA_NOTLOADED 0xffffffffu
#define ASTRA_TS_NONE32 0xffffffffu
#define ASTRA_WMAX_LOG2 9                 // lookahead window capped at 512 cycles (per-warp smem histogram)
#define ASTRA_CAND_PAD 0xffffffffu        // padding entry in candidate tables

// Candidate table entry (per node, for in-links and out-links): link id, ceil(B), k.
//   [10,32) link id   [5,10) ceil(bw)   [0,5) k
// A link's block of candidates never straddles a 32-entry chunk.
static inline u32 astra_cand_pack(u32 link, u32 ceilb, u32 k) { return (link << 10) | (ceilb << 5) | k; }

// Per design point descriptor.  c_* are byte offsets into the batch's constant blob, w_* byte
// offsets into the workspace of the CTA slot running the point, r_* byte offsets into the results
// blob.
struct PointDesc {
    u32 G, V, E, S;
    u32 C, Wv, K, H;
    u32 CW, nwords, slots, bmwords;
    u32 logW, NW, kdiv_magic, n_rel_total;     // NW power of two; kdiv_magic = ceil(2^32 / K)
    u32 flags, pad0;
    u64 max_cycles;
    u64 total_lines;
    u64 ws_bytes, ws_zero_bytes, ws_ff_off, ws_ff_bytes;
    // topology tables
    u64 c_row_ptr, c_in_ptr, c_in_link, c_leff, c_bw, c_icand_ptr, c_icand, c_ocand_ptr, c_ocand, c_next_link;
    // collective tables
    u64 c_step_od, c_lines, c_cu_lo, c_cu_n, c_succ_ptr, c_succ, c_ndeps;
    // plan tables (topology x collective x gpu)
    u64 c_step_q, c_step_r, c_first_link, c_step_alpha, c_cul_ptr, c_cul, c_rel_off, c_init_rel, c_init_rel_cnt;
    u64 c_fifo_off, c_fifo_mask, c_pipe_off, c_pipe_mask, c_credit_cap;
    // workspace: zero-initialised region
    u64 w_fifo_head, w_fifo_tail, w_pipe_tail, w_pipe_tail_pub, w_pipe_head, w_pipe_tsnap, w_credit_time, w_link_lines;
    u64 w_issued_cnt, w_deliv_cnt, w_ack_cnt, w_wf_busy, w_want, w_freeb, w_pend_cnt, w_rel_cnt;
    u64 w_bitmap, w_bin_cnt, w_node_next, w_node_busy, w_node_acked;
    // workspace: 0xff-initialised region
    u64 w_t_release, w_t_issued, w_t_deliv, w_t_ack, w_wf_rem;
    // workspace: specially initialised
    u64 w_credit, w_ndep_left, w_wf_cur, w_rel_list;
    // workspace: uninitialised
    u64 w_fifo_buf, w_pipe_buf, w_pend, w_pend_link, w_sel, w_ack_rec, w_ack_tmp, w_ack_sorted;   // ack_tmp / ack_sorted hold u64 entries
    // results
    u64 r_step_ts, r_link_lines, r_summary;
};

struct DeviceSummary {          // mirrors astra_summary, written by the kernel
    int32_t status; u32 n_steps, n_links, window;
    u64 completion_cycle, total_lines, busy_cycles, skipped_cycles;
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
    std::vector<u32> icand_ptr, icand, ocand_ptr, ocand;
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

struct HostGpu { u32 C = 0, Wv = 0, K = 0, H = 0; };

struct Blob {                       // append-only byte buffer with 16-byte aligned sections
    std::vector<uint8_t> bytes;
    u64 add(const void* p, size_t n);
    template <class T> u64 add(const std::vector<T>& v) { return add(v.data(), v.size() * sizeof(T)); }
};

struct PlanResult { int32_t rc = 0; std::string err; };

// loader entry points (astra_loader.cpp)
int32_t astra_build_topo(HostTopo& t, std::string& err);
int32_t astra_build_coll(HostColl& c, std::string& err);
int32_t astra_plan_point(const HostTopo& t, const HostColl& c, const HostGpu& g, u64 flags, u64 max_cycles,
                         u64 topo_off[10], u64 coll_off[7], Blob& blob, PointDesc& out, double& cost,
                         std::string& err);

// engine entry points (astra_engine.cu)
struct EngineLaunch {
    const uint8_t* d_const; uint8_t* d_ws; uint8_t* d_results;
    const PointDesc* d_points; const u32* d_order; u32* d_queue;
    u32 n_points; u64 ws_stride; u32 grid, warps_per_cta;
};
int32_t astra_engine_launch(const EngineLaunch& L, void* stream, std::string& err);
int32_t astra_engine_occupancy(u32 warps_per_cta, u32* ctas_per_sm, u32* n_sms, std::string& err);
