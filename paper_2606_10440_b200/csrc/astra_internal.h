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
//   [38,64) arrival cycle mod 2^26 (meaningful once the link has accepted the line)
// ---------------------------------------------------------------------------------------------
#define ASTRA_FLIT_TIME_SHIFT 38
#define ASTRA_FLIT_PAYLOAD_MASK ((1ull << ASTRA_FLIT_TIME_SHIFT) - 1)
#define ASTRA_TMASK26 0x3ffffffu
#define ASTRA_T_INF 0xffffffffu
#define ASTRA_NOTLOADED 0xffffffffu
#define ASTRA_TS_NONE32 0xffffffffu
#define ASTRA_WMAX_LOG2 9                 // lookahead window capped at 512 cycles (per-warp smem scratch)
#define ASTRA_NW_MAX 256                  // ack window bins per point (smem counters)

// Link service kinds (R9): how the acceptance times of a FIFO are computed for a whole window.
#define ASTRA_LK_INT     0u               // bw = B*256: B lines every cycle, no carried credit
#define ASTRA_LK_PERIOD  1u               // 256 % bw == 0: one line every P = 256/bw cycles
#define ASTRA_LK_GENERAL 2u               // any other bw: saturating credit walked entry by entry

// Per design point descriptor.  c_* are byte offsets into the batch's constant blob, w_* byte
// offsets into the workspace of the CTA slot running the point, r_* byte offsets into the results
// blob.
struct PointDesc {
    u32 G, V, E, S;
    u32 C, Wv, K, H;
    u32 CW, nwords, slots, bmwords;
    u32 logW, NW, kdiv_magic, NC;              // NW power of two; kdiv_magic = ceil(2^32 / K); NC = W + 1
    u32 flags, pad0;
    u64 max_cycles;
    u64 total_lines;
    u64 ws_bytes, ws_zero_bytes, ws_ff_off, ws_ff_bytes;
    // topology tables
    u64 c_in_ptr, c_in_link, c_head, c_tail, c_leff, c_bw, c_next_link;
    // collective tables
    u64 c_step_od, c_lines, c_cu_lo, c_cu_n, c_succ_ptr, c_succ, c_ndeps;
    // plan tables (topology x collective x gpu)
    u64 c_step_q, c_step_r, c_first_link, c_step_alpha, c_cul_ptr, c_cul, c_rel_off, c_init_rel, c_init_rel_cnt;
    u64 c_ev_off;
    u64 c_ring_off, c_ring_mask, c_lkind, c_ceilb, c_lstate0_init, c_stage_off, c_mask_off, c_classoff;
    u64 c_nd_cellcap, c_nd_mw, c_nd_injoff;
    // workspace: zero-initialised region
    u64 w_pipe_head, w_fifo_head, w_tail, w_lstate1, w_link_lines, w_masks;
    u64 w_issued_cnt, w_t_issued, w_deliv_cnt, w_t_deliv, w_ack_cnt, w_t_ack, w_rel_time;
    u64 w_wf_busy, w_want, w_bitmap, w_bin_cnt, w_ack_n, w_ev_cnt;
    // workspace: 0xff-initialised region
    u64 w_wf_rem;
    // workspace: specially initialised
    u64 w_lstate0, w_t_release, w_ndep_left, w_wf_cur, w_freeb, w_plist, w_pcnt;
    // workspace: uninitialised
    u64 w_ring, w_stage, w_sel, w_ack_rec, w_ack_tmp, w_ack_sorted, w_ev_list;
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

#define ASTRA_N_TOPO_TABLES 7
#define ASTRA_N_COLL_TABLES 7

// loader entry points (astra_loader.cpp)
int32_t astra_build_topo(HostTopo& t, std::string& err);
int32_t astra_build_coll(HostColl& c, std::string& err);
int32_t astra_plan_point(const HostTopo& t, const HostColl& c, const HostGpu& g, u64 flags, u64 max_cycles,
                         const u64* topo_off, const u64* coll_off, Blob& blob, PointDesc& out, double& cost,
                         std::string& err);

// engine entry points (astra_engine.cu)
struct EngineLaunch {
    const uint8_t* d_const; uint8_t* d_ws; uint8_t* d_results;
    const PointDesc* d_points; const u32* d_order; u32* d_queue;
    u32 n_points; u64 ws_stride; u32 grid, warps_per_cta;
};
int32_t astra_engine_launch(const EngineLaunch& L, void* stream, std::string& err);
int32_t astra_engine_occupancy(u32 warps_per_cta, u32* ctas_per_sm, u32* n_sms, std::string& err);
