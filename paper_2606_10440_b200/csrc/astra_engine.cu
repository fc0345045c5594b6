// astra_engine.cu -- the sm_100a window-batched step kernel of the cycle-synchronous cache-line
// simulator.
//
// The paper's simulator is an event-driven CPU program.  This engine is organised
// around one structural fact instead: a line accepted by a link at cycle a cannot reach the next
// node before a + Leff, and an ack cannot reach its owner before t_deliv + alpha >= t_deliv +
// min Leff.  With W <= min Leff, nothing a node does inside the window [kW, (k+1)W) can
// influence another node inside the same window.  So simulated time advances a whole window at a
// time, every stage of a window is node-local, and inside a window every phase of rules R7-R12
// is a data-parallel pass over ALL events of the window instead of a serial walk over cycles:
//
//   stage 1  arrivals (R7 A1) and ack discovery (R6, A3) as a flat list of chunk tasks: the lines
//            due on every in-link are known (link service counted them per arrival window), so
//            links are cut into independent 32-entry chunks -- deliveries (slot-addressed ack
//            record + bitmap bit), forwards to a single-feeder link (position = base + index),
//            forwards to multi-feeder links (one bit in the (out-link, cycle) cell at a slot fixed
//            by (in-link, rank inside the cycle)); the ack bitmap into 32-word chunks.
//   stage 2  release + issue (R10-R13): events -> release times; every wavefront runs through the
//            window as if the HBM budget never bound, on a thread (wf_sim) or a warp (wf_heavy,
//            prefix maximum over the issue index); per-cycle counts prove it (gpu_binds), or the
//            exact fixed-priority grants are computed word by word (wf_priority_word); issues are
//            ranked inside their cycle by wavefront id (ev_place) = FIFO position / cell slot.
//   stage 3  merge (R7/R8 append order) per out-link with several feeders: prefix sum of the
//            cell popcounts = FIFO position of every slot; the feeders then write their lines
//            straight to those positions.  No atomically allocated slot, no sort.
//   stage 4  link service (R9)  one warp per link: acceptance times of the whole FIFO follow from
//            a prefix-max scan (integer and 1/P bandwidths) or a credit walk (any other), and the
//            accepted lines are stamped with their arrival cycle in the link's ring.
//   stage 5  next non-idle window (A7): min over pending arrivals, acks, backlog and ready work.
//
// Hot per-node state (link cursors, cells, ready masks, wavefront records, step counters) lives
// in shared memory whenever the loader could fit it (PointDesc::a_off placement flags); rings and
// ack records stream through L2/HBM.  One CTA, or a group of CTAs with one node range each and one
// group barrier per window, simulates one design point; a persistent grid pulls points from two
// cost-sorted queues (grouped / single), see classify() in astra_api.cpp.
#include "astra_internal.h"
#include "../../include/astra.h"

#include <cuda_runtime.h>

#define FULL 0xffffffffu
#define ASTRA_COLD            // measured: real calls (__noinline__) for the rarely taken paths cost 3 % on every config
#define STAGE_BYTES (24u << 10)   // shared-memory copy of a point's per-step constant tables (TMA bulk copies at the point's start)
#define STAGE_TABLES 10u          // step_od, lines, cu_lo, cu_n, step_q, step_r, first_link, step_alpha, step_aq, step_ar
#define SCR_WORDS 1088u   // per-warp scratch words: 32 lanes x 64 16-bit ack keys (wf_sim, wf_priority_word), 513 counters (ack_sort), 512 (ack_chunk)

struct Ctx {   // resolved pointers of the point a CTA is running; lives in shared memory
    u32 G, V, E, S, C, Wv, K, H, CW, nwords, slots, bmwords, W, NC, NWmask, NW, kmagic, tmax, flags, alcap, pcu;
    u32 group, rank, v_lo, v_hi, g_lo, g_hi, e_lo, e_hi, i_lo, i_hi;
    u64 fullmask;
#define X(n) const u32* n;
    ASTRA_CONST_TABLES(X)
#undef X
#define X(n, t, i) t* n;
    ASTRA_WS_ARRAYS(X)
#undef X
    u64 *r_step_ts, *r_link_lines, *r_diag; DeviceSummary* r_summary;
};

struct Ctl {   // per-CTA control block in shared memory
    u32 point;          // index into the order array
    u32 acked;          // steps fully acked by this CTA's GPUs (single CTA: running total; group: since the last reduction)
    u32 completion;     // max t_ack
    u32 err;            // engine self-check flags
    u32 hint[3];        // min over everything pending of its next event time; slot seq % 3 is the window's (A7)
    u32 g_hint, g_acked, g_err, g_completion;   // group mode: the group-wide values after the window's group barrier
    u32 abort;          // a group barrier timed out somewhere: leave the kernel
    // run-ahead windows (one-CTA points of up to 32 nodes, one node per warp set): no block barrier per window
    u32 prog[32];       // windows completed by node (set) i
    u32 shint[32][2];   // next-event hint of node i's current window (slot: window ordinal & 1)
    u32 hint8[8];       // the point's hint per window ordinal & 7
    u32 stop;           // 1 + final status once a node has decided that the run ends
    u32 stage_phase, stage_wait;   // mbarrier phase of the next / the current point's staged tables
    // link service by all warps of a set (link_service_set)
    int ls_max[32];     // per warp: maximum of its block
    u32 ls_acc[32], ls_last[32];   // per set: lines accepted, last acceptance cycle
#ifdef ASTRA_DIAG
    u64 clk[16];        // [0] windows, [5] init clocks, [6] budget-bound GPU-windows, [7] clocks on that path, [8] windows with such a GPU
    u64 sclk[16][8];    // per warp set (clocks of its first warp, summed over its nodes and windows): 0 arrivals+acks,
                        // 1 release events, 2 wavefront runs, 3 budget check / commit, 4 placement, 5 merge, 6 link service,
                        // 7 waiting at the end-of-window barrier (block + group)
#endif
};

#ifdef ASTRA_DIAG
#define DIAG_CLK(slot) do { if (diag_lane) { const long long ck_ = clock64(); ctl.sclk[set][slot] += (u64)(ck_ - dck); dck = ck_; } } while (0)
#define DIAG_ADD(slot, v) do { atomicAdd((unsigned long long*)&ctl.clk[slot], (unsigned long long)(v)); } while (0)
#else
#define DIAG_CLK(slot) do { } while (0)
#define DIAG_ADD(slot, v) do { } while (0)
#endif

__device__ const unsigned char k_arr_init[ASTRA_A_COUNT] = {
#define X(n, t, i) i,
    ASTRA_WS_ARRAYS(X)
#undef X
};

// Arrays that the loader may place in shared OR global memory and that another CTA of a group may
// have written: a volatile generic load (never served from a stale L1 line, legal on both spaces).
__device__ __forceinline__ u32 ld_vol(const u32* p) { return *(const volatile u32*)p; }

__device__ __forceinline__ u32 lanemask_lt() { u32 m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m; }

__device__ __forceinline__ u32 warp_incl_scan(u32 v, u32 lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { u32 n = __shfl_up_sync(FULL, v, d); if (lane >= (u32)d) v += n; }
    return v;
}
__device__ __forceinline__ int warp_incl_max(int v, u32 lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { int n = __shfl_up_sync(FULL, v, d); if (lane >= (u32)d) v = max(v, n); }
    return v;
}

// Mark slot `slot` of the cell (out-link o at node v, cycle t0 + d) occupied (R7/R8).  A multi-feeder link that the
// loader expects to see lines in few cycles of a window (nz_off set) also keeps one bit per cycle, "this cell is not
// empty": its prefix pass and its clean-up look only at the marked cells instead of sweeping all of them.
__device__ __forceinline__ void cell_set(const Ctx& __restrict__ c, u32 o, u32 v, u32 cb, u32 d, u32 slot) {
    u32 ci = cb + d; if (ci >= c.NC) ci -= c.NC;
    atomicOr(&c.masks[c.mask_off[o] + ci * c.nd_mw[v] + (slot >> 5)], 1u << (slot & 31));
    const u32 nzo = c.nz_off[o];
    if (nzo != ASTRA_NONE32) atomicOr(&c.nz[nzo + (d >> 5)], 1u << (d & 31));
    c.dirty[o] = 1u;
}
// FIFO position, relative to the tail at the window start, of the line in slot `slot` of that cell.
__device__ __forceinline__ u32 cell_pos(const Ctx& __restrict__ c, u32 o, u32 v, u32 cb, u32 d, u32 slot) {
    u32 ci = cb + d; if (ci >= c.NC) ci -= c.NC;
    const u32 mw = c.nd_mw[v];
    const u32* words = c.masks + c.mask_off[o] + ci * mw;
    u32 r = c.pre[c.pre_off[o] + d];
    const u32 sw = slot >> 5;
    #pragma unroll 1
    for (u32 w = 0; w < sw; w++) r += __popc(words[w]);
    return r + __popc(words[sw] & ((1u << (slot & 31)) - 1u));
}

// ---------------------------------------------------------------------------------------------
// stage 1a / 3b: arrivals on in-link stream i during [t0, t0 + wlen)   (R7 A1)
// PASS 1 delivers, appends to single-feeder out-links and marks cells; PASS 3 (after the prefix
// sums) writes the lines that go to multi-feeder out-links at their FIFO positions.
// ---------------------------------------------------------------------------------------------
template <int PASS>
__device__ void arrivals_link(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 i, u32 n_due, u32 k, u32 t0, u32 wlen, u32 cb, u32 lane) {
    const u32 e = c.in_link[i];
    const u32 lo = c.pipe_head[e];
    // pass 1: the lines due this window were counted by the link's service when it accepted them
    const u32 hi = lo + (PASS == 1 ? n_due : c.ndue[e]);
    if (lo == hi) return;
    const u32 v = c.head[e];
    const u64* ring = c.ring + c.ring_off[e];
    const u32 rmask = c.ring_mask[e], coff = c.classoff[e];
    if (PASS == 1 && lane == 0 && hi - lo > rmask + 1) atomicOr(&ctl.err, 1u);
    u32 carry_d = 0xffffffffu, carry_cnt = 0, idx = lo, ndue = 0, hint = ASTRA_T_INF;
    bool any_p3 = false;
    #pragma unroll 1
    for (;;) {
        const u32 ii = idx + lane;
        const bool valid = (int32_t)(hi - ii) > 0;
        const u64 flit = valid ? __ldcg(&ring[ii & rmask]) : 0ull;
        const u32 d = ((u32)(flit >> ASTRA_FLIT_TIME_SHIFT) - t0) & ASTRA_TMASK26;
        const bool due = valid && d < wlen;
        const u32 duemask = __ballot_sync(FULL, due);
        if (PASS == 1 && valid && !due) hint = min(hint, t0 + d);
        if (duemask) {
            // position of the line among the lines this link delivers in the same cycle
            u32 r = 0;
            if (due) {
                const u32 grp = __match_any_sync(duemask, d);
                r = __popc(grp & lanemask_lt()) + (d == carry_d ? carry_cnt : 0u);
            }
            const u32 last = 31 - __clz(duemask);
            const u32 nd_last = __shfl_sync(FULL, d, last);
            const u32 nc_last = __shfl_sync(FULL, r, last) + 1;
            carry_d = nd_last; carry_cnt = nc_last;

            const u32 step = (u32)flit & 0xfffffu;
            const u32 od = due ? c.step_od[step] : 0;
            const u32 dstg = od & 0xffffu;
            const bool deliver = due && dstg == v;
            const bool transit = due && !deliver;
            u32 o = 0, moff = 0;
            if (transit) { o = c.next_link[(size_t)v * c.G + dstg]; moff = c.mask_off[o]; }
            const bool direct = transit && moff == ASTRA_NONE32;
            const bool merged = transit && !direct;
            if (PASS == 1) {
                if (merged) { cell_set(c, o, v, cb, d, coff + r); any_p3 = true; }
                const u32 dm = __ballot_sync(FULL, direct);
                if (dm) {       // this stream is the only feeder of o: append in stream order
                    u32 grp = 0, base = 0;
                    if (direct) {
                        grp = __match_any_sync(dm, o);
                        base = c.run[o];
                        const u32 pos = base + __popc(grp & lanemask_lt());
                        c.ring[c.ring_off[o] + (pos & c.ring_mask[o])] =
                            (flit & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)d << ASTRA_FLIT_TIME_SHIFT);
                    }
                    __syncwarp();
                    if (direct && (grp & lanemask_lt()) == 0) c.run[o] = base + __popc(grp);
                    __syncwarp();
                }
                const u32 dmask = __ballot_sync(FULL, deliver);
                if (dmask) {
                    bool completed = false;
                    if (deliver) {
                        const u32 owner = od >> 16;
                        const u32 wf = ((u32)flit >> 20) & 0xfffu, slot = (u32)(flit >> 32) & 63u;
                        const u32 ta = t0 + d + c.step_alpha[step];                       // R6
                        const u32 bit = wf * c.K + slot;
                        c.ack_rec[(size_t)owner * c.slots + bit] = ((u64)step << 32) | ta;
                        const u32 bin = owner * c.NW + ((k + c.step_aq[step] + (d + c.step_ar[step] >= c.W ? 1u : 0u)) & c.NWmask);
                        atomicOr(&c.bitmap[(size_t)bin * c.bmwords + (bit >> 5)], 1u << (bit & 31));
                        const u32 mb = __match_any_sync(dmask, bin);
                        u32 lpos = 0;                                        // discovery list of the bin: position from the count
                        if ((mb & lanemask_lt()) == 0) { if (c.alcap) lpos = atomicAdd(&c.bin_cnt[bin], (u32)__popc(mb)); else atomicAdd(&c.bin_cnt[bin], (u32)__popc(mb)); }
                        hint = min(hint, ta);
                        const u32 m = __match_any_sync(dmask, step);
                        const u32 dmax = __reduce_max_sync(m, d);
                        if ((m & lanemask_lt()) == 0) {
                            const u32 dc = c.deliv_cnt[step] + __popc(m);
                            c.deliv_cnt[step] = dc;
                            if (dc == c.lines[step]) { c.t_deliv[step] = t0 + dmax; completed = true; }
                        }
                        if (c.alcap) { lpos = __shfl_sync(mb, lpos, __ffs(mb) - 1) + __popc(mb & lanemask_lt()); if (lpos < c.alcap) c.ack_list[(size_t)bin * c.alcap + lpos] = bit; }
                    }
                    if (completed) {      // DELIVERED event at GPU v (dst of the step)
                        const u32 pos = atomicAdd(&c.ev_cnt[v], 1u);
                        c.ev_list[c.ev_off[v] + pos] = step | ((u32)ASTRA_DEP_DELIVERED << 30);
                    }
                }
            } else if (merged) {
                const u32 pos = c.ltail[o] + cell_pos(c, o, v, cb, d, coff + r);
                c.ring[c.ring_off[o] + (pos & c.ring_mask[o])] =
                    (flit & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)d << ASTRA_FLIT_TIME_SHIFT);
            }
            ndue += __popc(duemask);
        }
        if (duemask != FULL) break;
        idx += 32;
    }
    if (PASS == 1) {
        hint = __reduce_min_sync(FULL, hint);
        any_p3 = __any_sync(FULL, any_p3);
        if (lane == 0) {
            if (any_p3) c.ndue[e] = ndue;           // pass 3 walks the same entries again
            else c.pipe_head[e] = lo + ndue;
            if (hint != ASTRA_T_INF) atomicMin(hp, hint);
        }
    } else if (lane == 0) {
        c.pipe_head[e] = lo + ndue;
        c.ndue[e] = 0;
    }
}

// ---------------------------------------------------------------------------------------------
// Cycle-serial path only: consume the window's ack bits of GPU g into ack_sorted, counting-sorted
// by cycle (low word: cycle << 18 | wavefront << 6 | slot).
__device__ ASTRA_COLD void ack_sort(const Ctx& __restrict__ c, Ctl& ctl, u32 g, u32 k, u32 t0, u32 wlen, u32* scnt, u32 lane) {
    const u32 bin = k & c.NWmask;
    const u32 n = c.ack_n[g];
    if (n == 0) return;
    #pragma unroll 1
    for (u32 i = lane; i <= wlen; i += 32) scnt[i] = 0;
    __syncwarp();
    u32* bm = c.bitmap + (size_t)(g * c.NW + bin) * c.bmwords;
    const u64* rec = c.ack_rec + (size_t)g * c.slots;
    u64* tmp = c.ack_tmp + (size_t)g * c.slots;
    u64* srt = c.ack_sorted + (size_t)g * c.slots;
    u32 total = 0;
    #pragma unroll 1
    for (u32 wb = 0; wb < c.bmwords; wb += 32) {
        const u32 wi = wb + lane;
        u32 w = (wi < c.bmwords) ? __ldcg(&bm[wi]) : 0;
        if (w) bm[wi] = 0;
        const u32 cnt = __popc(w);
        const u32 incl = warp_incl_scan(cnt, lane);
        u32 pos = total + incl - cnt;
        total += __shfl_sync(FULL, incl, 31);
        #pragma unroll 1
        while (w) {
            const u32 b = __ffs(w) - 1; w &= w - 1;
            const u32 idx = wi * 32 + b;
            const u64 rc = __ldcg(&rec[idx]);
            const u32 cyc = (u32)rc - t0;
            const u32 wf = c.K == 1 ? idx : (u32)(((u64)idx * c.kmagic) >> 32);
            const u32 slot = idx - wf * c.K;
            atomicAdd(&scnt[cyc], 1u);
            tmp[pos++] = (rc & 0xffffffff00000000ull) | (cyc << 18) | (wf << 6) | slot;
        }
    }
    __syncwarp();
    u32 carry = 0;
    #pragma unroll 1
    for (u32 b = 0; b < wlen; b += 32) {
        const u32 i = b + lane;
        const u32 vv = (i < wlen) ? scnt[i] : 0;
        const u32 incl = warp_incl_scan(vv, lane);
        if (i < wlen) scnt[i] = carry + incl - vv;
        carry += __shfl_sync(FULL, incl, 31);
    }
    __syncwarp();
    #pragma unroll 1
    for (u32 b = 0; b < total; b += 32) {
        const u32 i = b + lane;
        if (i < total) {
            const u64 ent = tmp[i];
            const u32 pos = atomicAdd(&scnt[(u32)ent >> 18], 1u);
            srt[pos] = ent;
        }
    }
    if (lane == 0) {
        c.bin_cnt[g * c.NW + bin] = 0;
        if (total != n) atomicOr(&ctl.err, 2u);
    }
    __syncwarp();
}

// ---------------------------------------------------------------------------------------------
// stage 1 as a flat task list.  The number of lines due on every in-link this window is known
// (link_service counted them per arrival window), so a link whose lines all terminate at its head,
// or all go on to one single-feeder link, is cut into independent chunks of 32 pipe entries; any
// other link stays one task (arrivals_link).  Ack discovery is cut into chunks of 32 bitmap words.
// ---------------------------------------------------------------------------------------------
__device__ void stage1_setup_gpu(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 g, u32 k, u32 lane) {
    u32 best = ASTRA_T_INF;                                     // earliest later window with acks pending (A7)
    #pragma unroll 1
    for (u32 j = 1 + lane; j < c.NW; j += 32)
        if (ld_vol(&c.bin_cnt[g * c.NW + ((k + j) & c.NWmask)])) { best = j; break; }
    best = __reduce_min_sync(FULL, best);
    if (lane == 0) {
        if (best != ASTRA_T_INF) {
            const u64 tw = (u64)(k + best) * c.W;
            atomicMin(hp, tw >= ASTRA_T_INF ? ASTRA_T_INF - 1 : (u32)tw);
        }
        c.ack_n[g] = ld_vol(&c.bin_cnt[g * c.NW + (k & c.NWmask)]);
    }
}

// In-link e has lines in flight that arrive after this window: the earliest later window with lines
// due is a candidate for the next non-idle window (A7).  Arrival windows of a link lie at most
// Leff / W + 1 windows ahead.  One link per lane.  Also the ring overflow guard of the reading side.
__device__ __forceinline__ void link_inflight_hint(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 e, u32 lo, u32 k) {
    const u32* dcb = &c.due_cnt[(size_t)e * c.NW];
    const u32 span = min(c.NW - 1, c.leff[e] / c.W + 2);
    u32 best = ASTRA_T_INF;
    {   // the first eight bins in flight together (the counts are other CTAs' writes in a group: volatile loads)
        u32 dv[8];
#pragma unroll
        for (u32 q = 0; q < 8; q++) dv[q] = q < span ? ld_vol(&dcb[(k + q + 1) & c.NWmask]) : 0u;
#pragma unroll
        for (int q = 7; q >= 0; q--) if (dv[q]) best = (u32)q + 1u;
    }
    if (best == ASTRA_T_INF)
#pragma unroll 1
        for (u32 j = 9; j <= span; j++)
            if (ld_vol(&dcb[(k + j) & c.NWmask])) { best = j; break; }
    if (best != ASTRA_T_INF) {
        const u64 tw = (u64)(k + best) * c.W;
        atomicMin(hp, tw >= ASTRA_T_INF ? ASTRA_T_INF - 1 : (u32)tw);
    }
    if (ld_vol(&c.fifo_head[e]) - lo > c.ring_mask[e] + 1) atomicOr(&ctl.err, 1u);
}

// 128 entries of the discovery list of GPU g's ack bin (deliveries appended the slot ids of their acks, in
// any order): per-step ack counts, t_ack, ACKED events, amask (R6, A3).  Everything here commutes.
__device__ void ack_list_chunk(const Ctx& __restrict__ c, Ctl& ctl, u32 g, u32 chunk, u32 n, u32 k, u32 t1, u32 lane) {
    const u32 bin = k & c.NWmask;
    const u32* list = c.ack_list + (size_t)(g * c.NW + bin) * c.alcap;
    const u64* rec = c.ack_rec + (size_t)g * c.slots;
    u32* am = c.amask + (size_t)g * c.nwords;
    const u32 K = c.K, kmagic = c.kmagic;
    const u32* lines = c.lines;
    const u32 j0 = chunk * 128;
    u32 idx[4]; u64 rc[4];
#pragma unroll
    for (int q = 0; q < 4; q++) { const u32 j = j0 + q * 32 + lane; idx[q] = j < n ? __ldcg(&list[j]) : 0xffffffffu; }
#pragma unroll
    for (int q = 0; q < 4; q++) rc[q] = idx[q] != 0xffffffffu ? __ldcg(&rec[idx[q]]) : 0ull;
    u32 tmax = 0, cs = 0xffffffffu, cc = 0, cm = 0;
#pragma unroll
    for (int q = 0; q < 4; q++) {
        if (idx[q] == 0xffffffffu) continue;
        const u32 ta = (u32)rc[q];
        const u32 wf = K == 1 ? idx[q] : (u32)(((u64)idx[q] * kmagic) >> 32);   // idx / K
        atomicOr(&am[wf >> 5], 1u << (wf & 31));
        if (ta >= t1) continue;                              // beyond the watchdog cut: not processed
        const u32 step = (u32)(rc[q] >> 32);
        tmax = max(tmax, ta);
        if (step != cs) {
            if (cc) {
                atomicMax(&c.t_ack[cs], cm);
                if (atomicAdd(&c.ack_cnt[cs], cc) + cc == lines[cs]) {
                    c.ev_list[c.ev_off[g] + atomicAdd(&c.ev_cnt[g], 1u)] = cs | ((u32)ASTRA_DEP_ACKED << 30);
                    atomicAdd(&ctl.acked, 1u);
                }
            }
            cs = step; cc = 0; cm = 0;
        }
        cc++; cm = max(cm, ta);
    }
    {   // final flush, aggregated over the lanes that hold the same step
        const u32 key = cc ? cs : 0xffffffffu;
        const u32 m = __match_any_sync(FULL, key);
        const u32 csum = __reduce_add_sync(m, cc), cmax = __reduce_max_sync(m, cm);
        if (cc && (m & lanemask_lt()) == 0) {
            atomicMax(&c.t_ack[cs], cmax);
            if (atomicAdd(&c.ack_cnt[cs], csum) + csum == lines[cs]) {
                c.ev_list[c.ev_off[g] + atomicAdd(&c.ev_cnt[g], 1u)] = cs | ((u32)ASTRA_DEP_ACKED << 30);
                atomicAdd(&ctl.acked, 1u);
            }
        }
    }
    tmax = __reduce_max_sync(FULL, tmax);
    if (lane == 0 && tmax) atomicMax(&ctl.completion, tmax);
}

// Fallback when a bin received more acks than its list holds: the bitmap itself is scanned.
// 32 bitmap words of GPU g's ack bin: per-step ack counts, t_ack, ACKED events, amask (R6, A3).
// The set bits are first compacted into the warp's scratch so that every lane handles the same
// number of acks whatever their spread over the words, four record loads in flight per lane.
__device__ ASTRA_COLD void ack_chunk(const Ctx& __restrict__ c, Ctl& ctl, u32 g, u32 chunk, u32 k, u32 t1, u32* scr, u32 lane) {
    const u32 CAP = 512;
    const u32 bin = k & c.NWmask;
    const u32* bm = c.bitmap + (size_t)(g * c.NW + bin) * c.bmwords;
    const u64* rec = c.ack_rec + (size_t)g * c.slots;
    u32* am = c.amask + (size_t)g * c.nwords;
    const u32 wi = chunk * 32 + lane;
    const u32 w = (wi < c.bmwords) ? __ldcg(&bm[wi]) : 0;
    const u32 cntw = __popc(w);
    const u32 incl = warp_incl_scan(cntw, lane);
    const u32 excl = incl - cntw, total = __shfl_sync(FULL, incl, 31);
    if (total == 0) return;
    const u32 K = c.K, kmagic = c.kmagic;
    const u32* lines = c.lines;
    u32 tmax = 0;
    // per-lane caches: consecutive acks of a lane mostly belong to one step and one amask word
    u32 cs = 0xffffffffu, cc = 0, cm = 0, aw = 0xffffffffu, ab = 0;
    #pragma unroll 1
    for (u32 base = 0; base < total; base += CAP) {
        {
            u32 pos = excl, ww = w;
            #pragma unroll 1
            while (ww) {
                const u32 b = __ffs(ww) - 1; ww &= ww - 1;
                if (pos >= base && pos < base + CAP) scr[pos - base] = (lane << 5) | b;
                pos++;
            }
        }
        __syncwarp();
        const u32 nn = min(CAP, total - base);
        #pragma unroll 1
        for (u32 j0 = 0; j0 < nn; j0 += 128) {
            u32 idx[4]; u64 rc[4];
#pragma unroll
            for (int q = 0; q < 4; q++) { const u32 j = j0 + q * 32 + lane; idx[q] = j < nn ? chunk * 1024 + scr[j] : 0xffffffffu; }
#pragma unroll
            for (int q = 0; q < 4; q++) rc[q] = idx[q] != 0xffffffffu ? __ldcg(&rec[idx[q]]) : 0ull;
#pragma unroll
            for (int q = 0; q < 4; q++) {
                if (idx[q] == 0xffffffffu) continue;
                const u32 ta = (u32)rc[q];
                const u32 wf = K == 1 ? idx[q] : (u32)(((u64)idx[q] * kmagic) >> 32);   // idx / K
                if ((wf >> 5) != aw) { if (ab) atomicOr(&am[aw], ab); aw = wf >> 5; ab = 0; }
                ab |= 1u << (wf & 31);
                if (ta >= t1) continue;                          // beyond the watchdog cut: not processed
                const u32 step = (u32)(rc[q] >> 32);
                tmax = max(tmax, ta);
                if (step != cs) {
                    if (cc) {                                    // flush the cached step
                        atomicMax(&c.t_ack[cs], cm);
                        if (atomicAdd(&c.ack_cnt[cs], cc) + cc == lines[cs]) {
                            c.ev_list[c.ev_off[g] + atomicAdd(&c.ev_cnt[g], 1u)] = cs | ((u32)ASTRA_DEP_ACKED << 30);
                            atomicAdd(&ctl.acked, 1u);
                        }
                    }
                    cs = step; cc = 0; cm = 0;
                }
                cc++; cm = max(cm, ta);
            }
        }
        __syncwarp();
    }
    if (ab) atomicOr(&am[aw], ab);
    // final flush, aggregated over the lanes that hold the same step
    {
        const u32 key = cc ? cs : 0xffffffffu;
        const u32 m = __match_any_sync(FULL, key);
        const u32 csum = __reduce_add_sync(m, cc), cmax = __reduce_max_sync(m, cm);
        if (cc && (m & lanemask_lt()) == 0) {
            atomicMax(&c.t_ack[cs], cmax);
            if (atomicAdd(&c.ack_cnt[cs], csum) + csum == lines[cs]) {
                c.ev_list[c.ev_off[g] + atomicAdd(&c.ev_cnt[g], 1u)] = cs | ((u32)ASTRA_DEP_ACKED << 30);
                atomicAdd(&ctl.acked, 1u);
            }
        }
    }
    tmax = __reduce_max_sync(FULL, tmax);
    if (lane == 0 && tmax) atomicMax(&ctl.completion, tmax);
}

// 32 pipe entries of a link whose lines all terminate at its head GPU (R7 A1, deliveries)
__device__ void deliver_chunk(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 e, u32 lo, u32 n, u32 chunk, u32 k, u32 t0, u32 wlen, u32 lane) {
    const u32 ii = lo + chunk * 32 + lane;
    bool valid = (int32_t)(lo + n - ii) > 0;
    u64 flit0 = 0;
    if (valid) {
        flit0 = __ldcg(&c.ring[c.ring_off[e] + (ii & c.ring_mask[e])]);
        valid = (((u32)(flit0 >> ASTRA_FLIT_TIME_SHIFT) - t0) & ASTRA_TMASK26) < wlen;   // watchdog cut inside the window
    }
    const u32 amk = __ballot_sync(FULL, valid);
    u32 hint = ASTRA_T_INF;
    if (valid) {
        const u32 v = c.head[e];
        const u64 flit = flit0;
        const u32 d = ((u32)(flit >> ASTRA_FLIT_TIME_SHIFT) - t0) & ASTRA_TMASK26;
        const u32 step = (u32)flit & 0xfffffu;
        const u32 owner = c.step_od[step] >> 16;
        const u32 wf = ((u32)flit >> 20) & 0xfffu, slot = (u32)(flit >> 32) & 63u;
        const u32 ta = t0 + d + c.step_alpha[step];                       // R6
        const u32 bit = wf * c.K + slot;
        c.ack_rec[(size_t)owner * c.slots + bit] = ((u64)step << 32) | ta;
        const u32 bin = owner * c.NW + ((k + c.step_aq[step] + (d + c.step_ar[step] >= c.W ? 1u : 0u)) & c.NWmask);
        atomicOr(&c.bitmap[(size_t)bin * c.bmwords + (bit >> 5)], 1u << (bit & 31));
        const u32 mb = __match_any_sync(amk, bin);
        u32 lpos = 0;                                        // discovery list of the bin: position from the count
        if ((mb & lanemask_lt()) == 0) { if (c.alcap) lpos = atomicAdd(&c.bin_cnt[bin], (u32)__popc(mb)); else atomicAdd(&c.bin_cnt[bin], (u32)__popc(mb)); }
        hint = ta;
        const u32 m = __match_any_sync(amk, step);
        const u32 dmax = __reduce_max_sync(m, d);
        if ((m & lanemask_lt()) == 0) {
            atomicMax(&c.t_deliv[step], t0 + dmax);
            const u32 cntm = __popc(m);
            const u32 old = atomicAdd(&c.deliv_cnt[step], cntm);
            if (old + cntm == c.lines[step]) {                  // DELIVERED event at GPU v (dst of the step)
                const u32 pos = atomicAdd(&c.ev_cnt[v], 1u);
                c.ev_list[c.ev_off[v] + pos] = step | ((u32)ASTRA_DEP_DELIVERED << 30);
            }
        }
        hint = __reduce_min_sync(amk, hint);
        if ((amk & lanemask_lt()) == 0) atomicMin(hp, hint);
        if (c.alcap) { lpos = __shfl_sync(mb, lpos, __ffs(mb) - 1) + __popc(mb & lanemask_lt()); if (lpos < c.alcap) c.ack_list[(size_t)bin * c.alcap + lpos] = bit; }
    }
}

// Pipe entries of a link whose lines terminate at its head or go on to multi-feeder links (R7 A1).
// A line's cell slot is (in-link's slot base + its rank among the lines this link delivers in the
// same cycle); lines of one cycle are consecutive in the stream, so the rank is a look at the
// neighbours -- inside the chunk, and at most ceil(B)-1 entries back across its start.
// Pass 1 (here) delivers, marks cells and records (out-link, slot) per line; the placement pass
// (cells_place_chunk, after the cell prefix sums) writes the FIFO entries.

// the lines of one half-chunk that end at the link's head GPU v: ack record, ack bin, delivery count (R6, R7 A1)
__device__ __forceinline__ void cells_deliver(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 v, u32 k, u32 t0, u64 flit, u32 d, u32 od,
                                              bool deliver, u32 vmask) {
    const u32 dmask = __ballot_sync(vmask, deliver);
    if (!deliver) return;
    const u32 step = (u32)flit & 0xfffffu;
    const u32 owner = od >> 16;
    const u32 wf = ((u32)flit >> 20) & 0xfffu, slot = (u32)(flit >> 32) & 63u;
    const u32 ta = t0 + d + c.step_alpha[step];                       // R6
    const u32 bit = wf * c.K + slot;
    c.ack_rec[(size_t)owner * c.slots + bit] = ((u64)step << 32) | ta;
    const u32 bin = owner * c.NW + ((k + c.step_aq[step] + (d + c.step_ar[step] >= c.W ? 1u : 0u)) & c.NWmask);
    atomicOr(&c.bitmap[(size_t)bin * c.bmwords + (bit >> 5)], 1u << (bit & 31));
    const u32 mb = __match_any_sync(dmask, bin);
    u32 lpos = 0;                                        // discovery list of the bin: position from the count
    if ((mb & lanemask_lt()) == 0) { if (c.alcap) lpos = atomicAdd(&c.bin_cnt[bin], (u32)__popc(mb)); else atomicAdd(&c.bin_cnt[bin], (u32)__popc(mb)); }
    const u32 m = __match_any_sync(dmask, step);
    const u32 dmax = __reduce_max_sync(m, d);
    if ((m & lanemask_lt()) == 0) {
        atomicMax(&c.t_deliv[step], t0 + dmax);
        const u32 cntm = __popc(m);
        const u32 old = atomicAdd(&c.deliv_cnt[step], cntm);
        if (old + cntm == c.lines[step]) {
            const u32 pos = atomicAdd(&c.ev_cnt[v], 1u);
            c.ev_list[c.ev_off[v] + pos] = step | ((u32)ASTRA_DEP_DELIVERED << 30);
        }
    }
    const u32 hint = __reduce_min_sync(dmask, ta);
    if ((dmask & lanemask_lt()) == 0) atomicMin(hp, hint);
    if (c.alcap) { lpos = __shfl_sync(mb, lpos, __ffs(mb) - 1) + __popc(mb & lanemask_lt()); if (lpos < c.alcap) c.ack_list[(size_t)bin * c.alcap + lpos] = bit; }
}

// A task is 64 entries, handled as two halves in lock step: the ring loads (and the look-back), then the step
// lookups, then the route lookups of both halves are in flight together.
__device__ void cells_chunk(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 e, u32 lo, u32 n, u32 chunk, u32 k, u32 t0, u32 wlen, u32 cb, u32 lane) {
    const u32 i0 = lo + chunk * 64;
    const u64* ring = c.ring + c.ring_off[e];
    const u32 rmask = c.ring_mask[e];
    const u32 nb = c.ceilb[e] - 1;                            // at most ceil(B) lines per cycle
    const bool in0 = (int32_t)(lo + n - (i0 + lane)) > 0, in1 = (int32_t)(lo + n - (i0 + 32 + lane)) > 0;
    const bool inb = lane < nb && (int32_t)(i0 - 1 - lane - lo) >= 0;
    const u64 fa = in0 ? __ldcg(&ring[(i0 + lane) & rmask]) : 0ull;
    const u64 fb = in1 ? __ldcg(&ring[(i0 + 32 + lane) & rmask]) : 0ull;
    const u64 fz = inb ? __ldcg(&ring[(i0 - 1 - lane) & rmask]) : 0ull;
    const u32 v = c.head[e], coff = c.classoff[e], G = c.G;
    const u32 da = in0 ? (((u32)(fa >> ASTRA_FLIT_TIME_SHIFT) - t0) & ASTRA_TMASK26) : 0xffffffffu;
    const u32 db = in1 ? (((u32)(fb >> ASTRA_FLIT_TIME_SHIFT) - t0) & ASTRA_TMASK26) : 0xfffffffeu;
    const u32 dz = inb ? (((u32)(fz >> ASTRA_FLIT_TIME_SHIFT) - t0) & ASTRA_TMASK26) : 0xfffffffdu;
    const u32 da0 = __shfl_sync(FULL, da, 0), db0 = __shfl_sync(FULL, db, 0);
    const u32 back_a = __popc(__ballot_sync(FULL, dz == da0));          // same-cycle lines before the task
    const u32 back_b = __popc(__ballot_sync(FULL, da == db0));          // ... before its second half
    const bool va = in0 && da < wlen, vb = in1 && db < wlen;            // d >= wlen: watchdog cut inside the window
    const u32 vma = __ballot_sync(FULL, va), vmb = __ballot_sync(FULL, vb);
    const u32 oda = va ? c.step_od[(u32)fa & 0xfffffu] : 0u;
    const u32 odb = vb ? c.step_od[(u32)fb & 0xfffffu] : 0u;
    u32 ra = 0, rb = 0;
    if (va) ra = __popc(__match_any_sync(vma, da) & lanemask_lt()) + (da == da0 ? back_a : 0u);
    if (vb) rb = __popc(__match_any_sync(vmb, db) & lanemask_lt()) + (db == db0 ? back_b : 0u);
    const bool dla = va && (oda & 0xffffu) == v, dlb = vb && (odb & 0xffffu) == v;
    const bool tra = va && !dla, trb = vb && !dlb;
    const u32 oa = tra ? c.next_link[(size_t)v * G + (oda & 0xffffu)] : 0u;
    const u32 ob = trb ? c.next_link[(size_t)v * G + (odb & 0xffffu)] : 0u;
    u32* scr = c.lscr + c.lscr_off[e] + chunk * 64 + lane;
    if (va) { if (tra) { cell_set(c, oa, v, cb, da, coff + ra); scr[0] = (oa << 12) | (coff + ra); } else scr[0] = ASTRA_NONE32; }
    if (vb) { if (trb) { cell_set(c, ob, v, cb, db, coff + rb); scr[32] = (ob << 12) | (coff + rb); } else scr[32] = ASTRA_NONE32; }
    if (__any_sync(FULL, tra || trb) && lane == 0) c.tl_base[e] = 1u;   // the placement pass has work on this link
    if (__any_sync(FULL, dla)) { if (va) cells_deliver(c, ctl, hp, v, k, t0, fa, da, oda, dla, vma); }
    if (__any_sync(FULL, dlb)) { if (vb) cells_deliver(c, ctl, hp, v, k, t0, fb, db, odb, dlb, vmb); }
}

// Placement pass of such a link (after the cell prefix sums): the lines that go on are written to their
// FIFO positions; out-link and cell slot of every line were recorded by pass 1.
__device__ void cells_place_chunk(const Ctx& __restrict__ c, u32 e, u32 lo, u32 n, u32 chunk, u32 t0, u32 wlen, u32 cb, u32 lane) {
    const u64* ring = c.ring + c.ring_off[e];
    const u32 rmask = c.ring_mask[e];
    const u32* scr = c.lscr + c.lscr_off[e];
    const u32 v = c.head[e], mw = c.nd_mw[v], NC = c.NC;
    u64 fl[2]; u32 sc[2], d[2], o[2], pb[2], tl[2], moff[2]; bool ok[2];
    // both halves in lock step: flit + record, then cursors and prefix, then the cell words
#pragma unroll
    for (int h = 0; h < 2; h++) {
        const u32 r = chunk * 64 + h * 32 + lane;
        fl[h] = r < n ? __ldcg(&ring[(lo + r) & rmask]) : 0ull;
        sc[h] = r < n ? scr[r] : ASTRA_NONE32;
    }
#pragma unroll
    for (int h = 0; h < 2; h++) {
        d[h] = ((u32)(fl[h] >> ASTRA_FLIT_TIME_SHIFT) - t0) & ASTRA_TMASK26;
        ok[h] = chunk * 64 + h * 32 + lane < n && d[h] < wlen && sc[h] != ASTRA_NONE32;      // d >= wlen: watchdog cut inside the window
        o[h] = ok[h] ? sc[h] >> 12 : 0u;
        pb[h] = ok[h] ? c.pre[c.pre_off[o[h]] + d[h]] : 0u;
        tl[h] = ok[h] ? c.ltail[o[h]] : 0u;
        moff[h] = ok[h] ? c.mask_off[o[h]] : 0u;
    }
#pragma unroll
    for (int h = 0; h < 2; h++) {
        if (!ok[h]) continue;
        const u32 slot = sc[h] & 0xfffu;
        u32 ci = cb + d[h]; if (ci >= NC) ci -= NC;
        const u32* words = c.masks + moff[h] + ci * mw;
        u32 r = pb[h];
        const u32 swd = slot >> 5;
        #pragma unroll 1
        for (u32 w = 0; w < swd; w++) r += __popc(words[w]);
        r += __popc(words[swd] & ((1u << (slot & 31)) - 1u));
        const u32 pos = tl[h] + r;
        c.ring[c.ring_off[o[h]] + (pos & c.ring_mask[o[h]])] = (fl[h] & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)d[h] << ASTRA_FLIT_TIME_SHIFT);
    }
}

// 32 pipe entries of a link whose lines all go on to the single-feeder link lfwd[e] (R7 A1, transit):
// stream order is FIFO order, so the position is the base plus the index in the stream
__device__ void forward_chunk(const Ctx& __restrict__ c, u32 e, u32 lo, u32 n, u32 base, u32 chunk, u32 t0, u32 wlen, u32 lane) {
    const u32 ii = lo + chunk * 32 + lane;
    if ((int32_t)(lo + n - ii) <= 0) return;
    const u64 flit = __ldcg(&c.ring[c.ring_off[e] + (ii & c.ring_mask[e])]);
    const u32 d = ((u32)(flit >> ASTRA_FLIT_TIME_SHIFT) - t0) & ASTRA_TMASK26;
    if (d >= wlen) return;                                      // watchdog cut inside the window
    const u32 o = c.lfwd[e];
    const u32 pos = base + (ii - lo);
    c.ring[c.ring_off[o] + (pos & c.ring_mask[o])] = (flit & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)d << ASTRA_FLIT_TIME_SHIFT);
}

// ---------------------------------------------------------------------------------------------
// stage 2 helpers
// ---------------------------------------------------------------------------------------------
// A step's timestamp of kind `kind` was stamped at cycle `time` on GPU g: count down its
// successors (R3, R10).  A successor whose last dependency this was is released at the max over
// its dependencies' times and joins g's pending-release list.  Whole warp, warp-uniform p.
__device__ __forceinline__ void on_event(const Ctx& __restrict__ c, u32 g, u32 p, u32 kind, u32 time, u32 lane) {
    const u32 lo = c.succ_ptr[p], hi = c.succ_ptr[p + 1];
    #pragma unroll 1
    for (u32 b = lo; b < hi; b += 32) {
        const u32 i = b + lane; bool ready = false; u32 s2 = 0;
        if (i < hi) {
            const u32 sk = c.succ[i];
            if ((sk >> 30) == kind) {
                s2 = sk & 0xfffffu;
                const u32 rt = max(c.rel_time[s2], time);
                c.rel_time[s2] = rt;
                const u32 nd = c.ndep_left[s2] - 1; c.ndep_left[s2] = nd;
                if (nd == 0) { ready = true; c.t_release[s2] = rt; }
            }
        }
        const u32 rm = __ballot_sync(FULL, ready);
        if (rm) {
            const u32 cnt = c.pcnt[g];
            if (ready) c.plist[c.rel_off[g] + cnt + __popc(rm & lanemask_lt())] = s2;
            __syncwarp();
            if (lane == 0) c.pcnt[g] = cnt + __popc(rm);
        }
        __syncwarp();
    }
}

// Walk wavefront (g, wf)'s in-order list from `cur` to the first entry that is not released by
// cycle t or has quota for it (R11).  Returns true when quota was loaded (the wavefront wants to
// issue).
__device__ __forceinline__ bool wf_advance(const Ctx& __restrict__ c, u32 g, u32 wf, u32& cur, u32& rem, u32 t) {
    const u32 end = c.cul_ptr[g * c.C + wf / c.Wv + 1];
    rem = ASTRA_NOTLOADED;
    #pragma unroll 1
    while (cur < end) {
        const u32 s = c.cul[cur];
        if (c.t_release[s] > t) return false;           // NONE (0xffffffff) or a later cycle
        const u32 q = c.step_q[s] + (((wf - c.cu_lo[s] * c.Wv) < c.step_r[s]) ? 1u : 0u);
        if (q) { rem = q; return true; }
        cur++;
    }
    return false;
}

// Per-CU cap (R2'): the "has a free slot" bits of the W wavefronts of CU `cu` follow the CU's pool together.
__device__ __forceinline__ void cu_set_free(u32* freeb, u32 cu, u32 Wv, bool free_now) {
    const u32 lo = cu * Wv, hi = lo + Wv;                       // Wv <= 32: at most two words
    const u32 w0 = lo >> 5, w1 = (hi - 1) >> 5;
    const u32 m0 = (w0 == w1 ? ((Wv == 32 ? ~0u : ((1u << Wv) - 1u)) << (lo & 31)) : (~0u << (lo & 31)));
    if (free_now) atomicOr(&freeb[w0], m0); else atomicAnd(&freeb[w0], ~m0);
    if (w1 != w0) { const u32 m1 = (1u << (hi & 31)) - 1u; if (free_now) atomicOr(&freeb[w1], m1); else atomicAnd(&freeb[w1], ~m1); }
}

// ---------------------------------------------------------------------------------------------
// stage 2: release + issue of GPU g over [t0, t1)   (R10 - R13, slot return of R7 A3)
// ---------------------------------------------------------------------------------------------
__device__ ASTRA_COLD void issue_window(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 g, u32 t0, u32 t1, u32 cb, u32 lane) {
    const u32 ack_n = c.ack_n[g];
    const u32 pcu = c.pcu;                                      // bit 0: one line per CU per cycle (R12'), bit 1: cap per CU (R2')
    const u64* srt = c.ack_sorted + (size_t)g * c.slots;
    u32* plist = c.plist + c.rel_off[g];
    u32* want = c.want + (size_t)g * c.nwords;
    u32* freeb = c.freeb + (size_t)g * c.nwords;
    u32* sel = c.sel + (size_t)g * c.H;
    u64* inj = c.inj_list + c.inj_off[g];
    const u32 inj_cap = c.inj_off[g + 1] - c.inj_off[g];
    u32 n_inj = c.inj_n[g];
    const u32 injoff = c.nd_injoff[g];
    // sorted acks are consumed from a register window of 32 entries
    u32 ack_pos = 0, abase = 0;
    u32 abuf = (lane < ack_n) ? (u32)srt[lane] : 0xffffffffu;       // low word: cyc << 18 | wf << 6 | slot
    u32 t_ack_next = ack_n ? t0 + (__shfl_sync(FULL, abuf, 0) >> 18) : ASTRA_T_INF;
    u32 t_rel_next = ASTRA_T_INF;
    {
        const u32 np = c.pcnt[g];
        #pragma unroll 1
        for (u32 i = lane; i < np; i += 32) t_rel_next = min(t_rel_next, c.t_release[plist[i]]);
        t_rel_next = __reduce_min_sync(FULL, t_rel_next);
    }
    bool more;
    {
        u32 any = 0;
        #pragma unroll 1
        for (u32 wi = lane; wi < c.nwords; wi += 32) any |= want[wi] & freeb[wi];
        more = __ballot_sync(FULL, any != 0) != 0;
    }
    u32 t = min(min(t_ack_next, t_rel_next), more ? t0 : ASTRA_T_INF);
    if (t < t0) t = t0;

    #pragma unroll 1
    while (t < t1) {
        more = false;
        // ---- slot return: acks due at t (R7 A3) ----
        if (t_ack_next == t) {
            const u32 cyc = t - t0;
            #pragma unroll 1
            for (;;) {
                const u32 j0 = ack_pos - abase;
                const bool now = lane >= j0 && abase + lane < ack_n && (abuf >> 18) == cyc;
                const u32 nm = __ballot_sync(FULL, now);
                if (now) {
                    const u32 wf = (abuf >> 6) & 0xfffu, slot = abuf & 63u;
                    // several acks of one wavefront may land in the same cycle
                    const u32 mw = __match_any_sync(nm, wf);
                    const u32 blo = __reduce_or_sync(mw, slot < 32 ? (1u << slot) : 0u);
                    const u32 bhi = __reduce_or_sync(mw, slot >= 32 ? (1u << (slot - 32)) : 0u);
                    if ((mw & lanemask_lt()) == 0) {
                        u64 busy = c.wf_busy[(size_t)g * c.CW + wf];
                        busy &= ~(((u64)bhi << 32) | blo);
                        c.wf_busy[(size_t)g * c.CW + wf] = busy;
                    }
                    if (pcu & 2u) {                                  // R2': the slots return to the CU's pool
                        const u32 cu = wf / c.Wv;
                        const u32 mc = __match_any_sync(nm, cu);
                        if ((mc & lanemask_lt()) == 0) { c.cu_out[(size_t)g * c.C + cu] -= (u32)__popc(mc); cu_set_free(freeb, cu, c.Wv, true); }
                    } else {
                        const u32 wi = wf >> 5;
                        const u32 mi = __match_any_sync(nm, wi);
                        const u32 bits = __reduce_or_sync(mi, 1u << (wf & 31));
                        if ((mi & lanemask_lt()) == 0) freeb[wi] |= bits;
                    }
                }
                ack_pos += __popc(nm);
                __syncwarp();                                        // the pool counts of one round are seen by the next
                if (ack_pos - abase < 32 || ack_pos >= ack_n) break;
                abase = ack_pos;                                     // register window exhausted: refill
                abuf = (abase + lane < ack_n) ? (u32)srt[abase + lane] : 0xffffffffu;
            }
            __syncwarp();
            if (ack_pos >= ack_n) t_ack_next = ASTRA_T_INF;
            else {
                if (ack_pos - abase >= 32) { abase = ack_pos; abuf = (abase + lane < ack_n) ? (u32)srt[abase + lane] : 0xffffffffu; }
                t_ack_next = t0 + (__shfl_sync(FULL, abuf, ack_pos - abase) >> 18);
            }
        }

        // ---- phase C: releases that take effect at t (R10) ----
        if (t_rel_next == t) {
            const u32 np = c.pcnt[g];
            u32 keep = 0, tn = ASTRA_T_INF;
            #pragma unroll 1
            for (u32 b = 0; b < np; b += 32) {
                const u32 i = b + lane;
                const u32 s = (i < np) ? plist[i] : 0;
                const u32 tr = (i < np) ? c.t_release[s] : ASTRA_T_INF;
                const bool now = (i < np) && tr == t;
                const bool later = (i < np) && !now;
                u32 nowm = __ballot_sync(FULL, now);
                const u32 laterm = __ballot_sync(FULL, later);
                __syncwarp();
                if (later) { plist[keep + __popc(laterm & lanemask_lt())] = s; tn = min(tn, tr); }
                keep += __popc(laterm);
                #pragma unroll 1
                while (nowm) {
                    const u32 src = __ffs(nowm) - 1; nowm &= nowm - 1;
                    const u32 sr = __shfl_sync(FULL, s, src);
                    const u32 lo = c.cu_lo[sr] * c.Wv, hi = lo + c.cu_n[sr] * c.Wv;
                    #pragma unroll 1
                    for (u32 wb = lo & ~31u; wb < hi; wb += 32) {
                        const u32 wf = wb + lane;
                        bool setw = false;
                        if (wf >= lo && wf < hi) {
                            const size_t gw = (size_t)g * c.CW + wf;
                            u32 cur = c.wf_cur[gw];
                            if (c.wf_rem[gw] == ASTRA_NOTLOADED && cur < c.cul_ptr[g * c.C + wf / c.Wv + 1] && c.cul[cur] == sr) {
                                u32 rem;
                                setw = wf_advance(c, g, wf, cur, rem, t);
                                c.wf_cur[gw] = cur; c.wf_rem[gw] = rem;
                            }
                        }
                        const u32 bits = __ballot_sync(FULL, setw);
                        if (bits && lane == 0) want[wb >> 5] |= bits;
                    }
                }
            }
            __syncwarp();
            if (lane == 0) c.pcnt[g] = keep;
            t_rel_next = __reduce_min_sync(FULL, tn);
            __syncwarp();
        }

        // ---- phase D: issue (R11 - R13) ----
        u32 budget = c.H, nsel = 0;
        bool left_over = false;
        if (pcu) {
            // per-CU readings: one CU per lane.  Of its ready wavefronts a CU may dispatch the lowest one (R12') or as
            // many as its pool has room for (R2'); then the first H of all of them in ascending wavefront id (R12).
            const u32 Wv = c.Wv;
            #pragma unroll 1
            for (u32 cb0 = 0; cb0 < c.C; cb0 += 32) {
                const u32 cu = cb0 + lane;
                u32 keep = 0, lo = 0;
                bool more_ready = false;
                if (cu < c.C) {
                    lo = cu * Wv;
                    const u32 w0 = lo >> 5, sh = lo & 31;
                    u64 r2 = (u64)(want[w0] & freeb[w0]);
                    if (w0 + 1 < c.nwords) r2 |= (u64)(want[w0 + 1] & freeb[w0 + 1]) << 32;
                    u32 bits = (u32)(r2 >> sh) & (Wv == 32 ? ~0u : ((1u << Wv) - 1u));
                    u32 room = Wv;
                    if (pcu & 1u) room = 1u;
                    if (pcu & 2u) room = min(room, c.K - c.cu_out[(size_t)g * c.C + cu]);
                    #pragma unroll 1
                    for (u32 q = 0; q < room && bits; q++) { const u32 low = bits & (0u - bits); keep |= low; bits ^= low; }
                    more_ready = bits != 0u;
                }
                const u32 cntc = __popc(keep);
                const u32 incl = warp_incl_scan(cntc, lane);
                const u32 tot = __shfl_sync(FULL, incl, 31);
                if (__any_sync(FULL, more_ready)) left_over = true;
                if (tot == 0) continue;
                if (budget == 0) { left_over = true; break; }
                const u32 excl = incl - cntc;
                const u32 take = excl >= budget ? 0 : min(cntc, budget - excl);
                #pragma unroll 1
                for (u32 i = 0; i < take; i++) {
                    const u32 b = __ffs(keep) - 1; keep &= keep - 1;
                    sel[nsel + excl + i] = lo + b;
                }
                const u32 got = min(tot, budget);
                if (tot > got) left_over = true;
                nsel += got; budget -= got;
            }
        } else
        #pragma unroll 1
        for (u32 wb = 0; wb < c.nwords; wb += 32) {
            const u32 wi = wb + lane;
            u32 r = (wi < c.nwords) ? (want[wi] & freeb[wi]) : 0;
            const u32 cnt = __popc(r);
            const u32 incl = warp_incl_scan(cnt, lane);
            const u32 tot = __shfl_sync(FULL, incl, 31);
            if (tot == 0) continue;
            if (budget == 0) { left_over = true; break; }
            const u32 excl = incl - cnt;
            const u32 take = excl >= budget ? 0 : min(cnt, budget - excl);
            #pragma unroll 1
            for (u32 i = 0; i < take; i++) {
                const u32 b = __ffs(r) - 1; r &= r - 1;
                sel[nsel + excl + i] = wi * 32 + b;
            }
            const u32 got = min(tot, budget);
            if (tot > got) left_over = true;
            nsel += got; budget -= got;
        }
        __syncwarp();
        const u32 d = t + 1 - t0;     // injected at t + 1 into the first-hop FIFO, after that cycle's transit lines (R7 A2)
        #pragma unroll 1
        for (u32 b = 0; b < nsel; b += 32) {
            const u32 j = b + lane; const bool act = j < nsel;
            u32 wf = 0, s = 0, o = 0, moff = 0; bool full = false, keepw = true;
            u64 payload = 0;
            if (act) {
                wf = sel[j];
                const size_t gw = (size_t)g * c.CW + wf;
                u32 cur = c.wf_cur[gw];
                s = c.cul[cur];
                u32 rem = c.wf_rem[gw] - 1;
                u64 busy = c.wf_busy[gw];
                const u32 slot = __ffsll((long long)~busy) - 1;
                busy |= 1ull << slot;
                c.wf_busy[gw] = busy;
                full = (busy == c.fullmask);
                payload = (u64)s | ((u64)wf << 20) | ((u64)slot << 32);
                o = c.first_link[s]; moff = c.mask_off[o];
                if (rem == 0) { cur++; keepw = wf_advance(c, g, wf, cur, rem, t); c.wf_cur[gw] = cur; }
                c.wf_rem[gw] = rem;
            }
            const u32 amask = __ballot_sync(FULL, act);
            const bool direct = act && moff == ASTRA_NONE32;
            const bool merged = act && !direct;
            const u32 dm = __ballot_sync(FULL, direct);
            if (dm) {            // this GPU is the only feeder of o: append in wavefront order
                u32 grp = 0, base = 0;
                if (direct) {
                    grp = __match_any_sync(dm, o);
                    base = c.run[o];
                    const u32 pos = base + __popc(grp & lanemask_lt());
                    c.ring[c.ring_off[o] + (pos & c.ring_mask[o])] = payload | ((u64)d << ASTRA_FLIT_TIME_SHIFT);
                }
                __syncwarp();
                if (direct && (grp & lanemask_lt()) == 0) c.run[o] = base + __popc(grp);
                __syncwarp();
            }
            const u32 mm = __ballot_sync(FULL, merged);
            if (mm) {
                if (merged) {
                    cell_set(c, o, g, cb, d, injoff + j);
                    const u32 p = n_inj + __popc(mm & lanemask_lt());
                    if (p < inj_cap) inj[p] = payload | ((u64)(d | (j << 10)) << ASTRA_FLIT_TIME_SHIFT);
                    else atomicOr(&ctl.err, 4u);
                }
                n_inj += __popc(mm);
            }
            bool completed = false;
            if (act) {
                const u32 ms = __match_any_sync(amask, s);
                if ((ms & lanemask_lt()) == 0) {
                    const u32 ic = c.issued_cnt[s] + __popc(ms);
                    c.issued_cnt[s] = ic;
                    if (ic == c.lines[s]) { c.t_issued[s] = t; completed = true; }
                }
                const u32 wi = wf >> 5;
                const u32 mi = __match_any_sync(amask, wi);
                const u32 clrf = __reduce_or_sync(mi, (full && !(pcu & 2u)) ? (1u << (wf & 31)) : 0u);
                const u32 clrw = __reduce_or_sync(mi, keepw ? 0u : (1u << (wf & 31)));
                if ((mi & lanemask_lt()) == 0) {
                    if (clrf) atomicAnd(&freeb[wi], ~clrf);
                    if (clrw) want[wi] &= ~clrw;
                }
                if (pcu & 2u) {                                  // R2': the CU's pool fills
                    const u32 cu = wf / c.Wv;
                    const u32 mc = __match_any_sync(amask, cu);
                    if ((mc & lanemask_lt()) == 0) {
                        const u32 nout = c.cu_out[(size_t)g * c.C + cu] + (u32)__popc(mc);
                        c.cu_out[(size_t)g * c.C + cu] = nout;
                        if (nout >= c.K) cu_set_free(freeb, cu, c.Wv, false);
                    }
                }
            }
            u32 cm = __ballot_sync(FULL, completed);
            #pragma unroll 1
            while (cm) {
                const u32 src = __ffs(cm) - 1; cm &= cm - 1;
                const u32 p = __shfl_sync(FULL, s, src);
                on_event(c, g, p, ASTRA_DEP_ISSUED, t + 1, lane);      // visible to phase C of t + 1 (R10)
                t_rel_next = ASTRA_T_INF;                               // recomputed below
            }
            __syncwarp();                                               // counters of one batch of 32 are seen by the next
        }
        __syncwarp();
        if (nsel) more = true;            // an issuing wavefront may issue again at t + 1
        if (left_over) more = true;
        if (t_rel_next == ASTRA_T_INF) {
            const u32 np = c.pcnt[g];
            u32 tn = ASTRA_T_INF;
            #pragma unroll 1
            for (u32 i = lane; i < np; i += 32) tn = min(tn, c.t_release[plist[i]]);
            t_rel_next = __reduce_min_sync(FULL, tn);
        }
        // ---- next cycle of this GPU where something can change (A7) ----
        u32 tn = min(t_ack_next, t_rel_next);
        if (more) tn = min(tn, t + 1);
        t = tn;
    }
    if (lane == 0) {
        c.inj_n[g] = n_inj;
        if (t != ASTRA_T_INF) atomicMin(hp, t);
    }
}

// ---------------------------------------------------------------------------------------------
// stage 2, wavefront-parallel path.  Inside a window every input of a wavefront's issue decisions
// is known up front -- its acks (stage 1b), the release times of its steps (events of stage 1) --
// EXCEPT the HBM budget H shared by the GPU's wavefronts (R12).  So every wavefront that can change
// state this window is simulated on its own thread as if the budget never bound, the issues are
// counted per (first-hop link, cycle), and the GPU's warp checks that no cycle exceeded H.  If none
// did, the unconstrained run IS the fixed-priority run (no wavefront was ever denied), and its
// issues are ranked (cycle, wavefront id) by counting into per-cycle buckets: that rank is the
// FIFO position (direct out-link) or the cell slot (multi-feeder out-link) R7 A2 prescribes.
// A GPU-window where the budget binds, or whose steps have ISSUED-kind successors (their release
// times depend on this window's issues), takes the cycle-serial path (issue_window) instead.
// ---------------------------------------------------------------------------------------------

// stage 2a: dependency events -> release times (R10); the set of wavefronts to look at; the mode.
__device__ void gpu_prepare(const Ctx& __restrict__ c, Ctl& ctl, u32 g, u32 t0, u32 t1, u32 lane) {
    {
        const u32 nev = c.ev_cnt[g];
        #pragma unroll 1
        for (u32 j = 0; j < nev; j++) {
            const u32 ek = c.ev_list[c.ev_off[g] + j];
            const u32 p = ek & 0xfffffu, kind = ek >> 30;
            const u32 time = kind == ASTRA_DEP_DELIVERED ? c.t_deliv[p] : c.t_ack[p];
            on_event(c, g, p, kind, time, lane);
        }
        __syncwarp();
        if (lane == 0 && nev) c.ev_cnt[g] = 0;
    }
    u32* am = c.amask + (size_t)g * c.nwords;
    const u32* want = c.want + (size_t)g * c.nwords;
    const u32* freeb = c.freeb + (size_t)g * c.nwords;
    // wavefronts of the CU range of every step released inside this window
    const u32 np = c.pcnt[g];
    const u32* plist = c.plist + c.rel_off[g];
    #pragma unroll 1
    for (u32 i = 0; i < np; i++) {
        const u32 s = plist[i];
        if (c.t_release[s] >= t1) continue;
        const u32 lo = c.cu_lo[s] * c.Wv, hi = lo + c.cu_n[s] * c.Wv;
        #pragma unroll 1
        for (u32 wi = (lo >> 5) + lane; wi <= ((hi - 1) >> 5); wi += 32) {
            const u32 b0 = wi * 32;
            u32 m = ~0u;
            if (lo > b0) m &= ~0u << (lo - b0);
            if (hi < b0 + 32) m &= (1u << (hi - b0)) - 1u;
            am[wi] |= m;
        }
        __syncwarp();
    }
    u32 any = 0;
    #pragma unroll 1
    for (u32 wi = lane; wi < c.nwords; wi += 32) {
        const u32 a = am[wi] | (want[wi] & freeb[wi]);
        am[wi] = a; any |= a;
    }
    const bool active = __ballot_sync(FULL, any != 0) != 0;
    u32 mode = 0;
    if (active) mode = ((c.gflag[g] & (ASTRA_GF_ISSUED_DEPS | ASTRA_GF_SERIAL)) || (c.flags & (u32)ASTRA_FLAG_SERIAL_ISSUE)) ? 2u : 1u;
    if (mode == 1) {
        const u32 e0 = c.row_ptr[g], deg = c.row_ptr[g + 1] - e0;
        u32* cnt = c.cnt + (size_t)g * c.W;
        #pragma unroll 1
        for (u32 i = lane; i < c.W; i += 32) cnt[i] = 0;
        if (lane == 0) c.nheavy[g] = 0;
        if (deg > 1) {                                          // per-cycle issue counts of the direct out-links
            u32 dm = deg > 32 ? 0u : c.gdirect[g];
            if (deg > 32) { u32* h = c.hist + (size_t)e0 * c.W; for (u32 i = lane; i < deg * c.W; i += 32) h[i] = 0; }
            #pragma unroll 1
            while (dm) {
                const u32 x = __ffs(dm) - 1; dm &= dm - 1;
                u32* h = c.hist + (size_t)(e0 + x) * c.W;
                #pragma unroll 1
                for (u32 i = lane; i < c.W; i += 32) h[i] = 0;
            }
        }
    }
    if (lane == 0) c.gmode[g] = mode;
}

// stage 2b: the 32 wavefronts of word wi of GPU g, each on its own thread, run through the window as
// if the HBM budget never bound.  Issues go to the bucket of their cycle (first H of a cycle are
// kept: more than H means the budget binds and the GPU-window is redone cycle-serially).  The new
// wavefront state is written in place, the old one kept in the undo arrays for that case.
__device__ void wf_sim(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 g, u32 wi, u32 k, u32 t0, u32 t1, u32* scr, u32 lane) {
    const u32 nwords = c.nwords;
    const u32 am0 = c.amask[(size_t)g * nwords + wi];
    if (am0 == 0) return;
    const bool active = (am0 >> lane) & 1u;
    const u32 wf = wi * 32 + lane;
    const u32 W = c.W, H = c.H, K = c.K;
    const u64 fullmask = c.fullmask;
    bool wantb = false, freebit = false, hint = false, heavy = false;
    const size_t gw = (size_t)g * c.CW + wf;
    const u32 b0 = wf * K, w0 = b0 >> 5, sh = b0 & 31;
    u32 cur = 0, rem = 0;
    u64 busy = 0, rb = 0;
    if (active) {
        cur = c.wf_cur[gw]; rem = c.wf_rem[gw]; busy = c.wf_busy[gw];
        // this wavefront's ack bits of the window's bin: bits [wf*K, wf*K + K) of the GPU's bitmap
        if (c.ack_n[g]) {
            const u32 bmwords = c.bmwords;
            const u32* bm = c.bitmap + (size_t)(g * c.NW + (k & c.NWmask)) * bmwords;
            const u32 x0 = __ldcg(&bm[w0]);
            const u32 x1 = (w0 + 1 < bmwords) ? __ldcg(&bm[w0 + 1]) : 0u;
            const u32 x2 = (sh && w0 + 2 < bmwords) ? __ldcg(&bm[w0 + 2]) : 0u;
            rb = ((((u64)x1 << 32) | x0) >> sh);
            if (sh) rb |= (u64)x2 << (64 - sh);
            rb &= fullmask;
        }
        // a wavefront that may issue many lines this window, in a word where few do, gets a warp of
        // its own (wf_heavy); when most of the word does, the lanes run the same long loop together
        heavy = min(K - (u32)__popcll(busy) + (u32)__popcll(rb), t1 - t0) >= ASTRA_HEAVY_MIN && !(c.flags & (u32)ASTRA_FLAG_NO_HEAVY);
    }
    __syncwarp();
    if (__popc(__ballot_sync(FULL, heavy)) > ASTRA_HEAVY_MAX_PER_WORD) heavy = false;
    if (heavy) {
        const u32 hp = atomicAdd(&c.nheavy[g], 1u);
        c.hlist[(size_t)g * c.CW + hp] = wf;
    }
    if (active) {
        const u32 e0 = c.row_ptr[g], deg = c.row_ptr[g + 1] - e0;
        u32* const cnt = c.cnt + (size_t)g * W;
        u32* const h = c.hist + (size_t)e0 * W;
        u64* const evb = c.evb + (size_t)g * H * W;
        const u32* const t_release = c.t_release;
        const u32* const cul = c.cul;
      if (!heavy) {
        c.undo_cur[gw] = cur; c.undo_rem[gw] = rem; c.undo_busy[gw] = busy;
        // the wavefront's acks of the window, sorted by cycle: (cycle - t0) << 6 | slot, 15 bits each, in the
        // warp's shared-memory scratch (entry j of this lane at aq[32 j]: no bank conflicts, no local memory)
        unsigned short* const aq = reinterpret_cast<unsigned short*>(scr) + lane;
        u32 na = 0, ai = 0;
        if (rb) {
            const u64* rec = c.ack_rec + (size_t)g * c.slots + b0;
            u64 x = rb;
            #pragma unroll 1
            while (x) {                                         // four loads in flight at a time
                u32 b[4]; u32 v[4]; int m = 0;
#pragma unroll
                for (int q = 0; q < 4; q++) { b[q] = 0; if (x) { b[q] = __ffsll((long long)x) - 1; x &= x - 1; m = q + 1; } }
#pragma unroll
                for (int q = 0; q < 4; q++) v[q] = (q < m) ? (u32)__ldcg(&rec[b[q]]) : 0u;
#pragma unroll
                for (int q = 0; q < 4; q++) if (q < m) aq[32 * na++] = (unsigned short)(((v[q] - t0) << 6) | b[q]);
            }
            #pragma unroll 1
            for (u32 i = 1; i < na; i++) {
                const u32 xv = aq[32 * i]; u32 j = i;
                #pragma unroll 1
                while (j > 0 && aq[32 * (j - 1)] > xv) { aq[32 * j] = aq[32 * (j - 1)]; j--; }
                aq[32 * j] = (unsigned short)xv;
            }
        }
        u32 nq = na ? aq[0] : 0xffffffffu;                       // earliest ack not applied yet (packed)
        const u32 end = c.cul_ptr[g * c.C + wf / c.Wv + 1];
        const u32 wlen = t1 - t0;
        const u32 gdir = c.gdirect[g];                          // out-links that need their per-cycle issue counts
        bool hx = false;
        u32 tt = 0, s = 0, ox = 0, last_issue = 0xffffffffu;    // tt: candidate cycle relative to t0
        u32 eq0 = 0, eq1 = 0, eq2 = 0, eq3 = 0, nb = 0;             // buffered issues: cycle << 6 | slot
        bool have_s = false;
        #pragma unroll 1
        for (;;) {
            if (rem == ASTRA_NOTLOADED) {
                bool got = false;
                #pragma unroll 1
                while (cur < end) {
                    const u32 s2 = cul[cur];
                    const u32 tr = t_release[s2];
                    if (tr >= t1) break;                        // not released by the end of the window
                    if (tr > t0 + tt) tt = tr - t0;
                    const u32 q = c.step_q[s2] + (((wf - c.cu_lo[s2] * c.Wv) < c.step_r[s2]) ? 1u : 0u);   // R11
                    if (q) { rem = q; got = true; break; }
                    cur++;
                }
                if (!got) break;
                have_s = false;
            }
            if (!have_s) { s = cul[cur]; ox = c.first_link[s] - e0; hx = deg > 1 && ((gdir >> (ox & 31u)) & 1u); have_s = true; }
            if (busy == fullmask) {                             // all K slots in flight: wait for the next ack
                if (ai >= na) break;
                tt = max(tt, nq >> 6);
            }
            #pragma unroll 1
            while ((nq >> 6) <= tt) {                           // slots returned by this cycle (A3 before D)
                busy &= ~(1ull << (nq & 63u)); ai++;
                nq = ai < na ? aq[32 * ai] : 0xffffffffu;
            }
            if (tt >= wlen) break;
            const u32 slot = __ffsll((long long)~busy) - 1;
            busy |= 1ull << slot;
            // issues are buffered four at a time so that their bucket-slot atomics overlap
            eq3 = eq2; eq2 = eq1; eq1 = eq0; eq0 = (tt << 6) | slot; nb++;
            last_issue = tt;
            rem--; tt++;
            if (nb == 4 || rem == 0) {
                u32 pp[4]; const u32 bb[4] = {eq0, eq1, eq2, eq3};
#pragma unroll
                for (int q = 0; q < 4; q++) pp[q] = (u32)q < nb ? atomicAdd(&cnt[bb[q] >> 6], 1u) : 0u;
#pragma unroll
                for (int q = 0; q < 4; q++) if ((u32)q < nb) {
                    const u32 t2 = bb[q] >> 6;
                    if (pp[q] < H) evb[(size_t)t2 * H + pp[q]] = (u64)s | ((u64)wf << 20) | ((u64)(bb[q] & 63u) << 32) | ((u64)(t2 + 1) << ASTRA_FLIT_TIME_SHIFT) | ((u64)ox << 48);
                    if (hx) atomicAdd(&h[ox * W + t2], 1u);
                }
                nb = 0;
            }
            if (rem == 0) { cur++; rem = ASTRA_NOTLOADED; }
        }
        if (nb) {
            u32 pp[4]; const u32 bb[4] = {eq0, eq1, eq2, eq3};
#pragma unroll
            for (int q = 0; q < 4; q++) pp[q] = (u32)q < nb ? atomicAdd(&cnt[bb[q] >> 6], 1u) : 0u;
#pragma unroll
            for (int q = 0; q < 4; q++) if ((u32)q < nb) {
                const u32 t2 = bb[q] >> 6;
                if (pp[q] < H) evb[(size_t)t2 * H + pp[q]] = (u64)s | ((u64)wf << 20) | ((u64)(bb[q] & 63u) << 32) | ((u64)(t2 + 1) << ASTRA_FLIT_TIME_SHIFT) | ((u64)ox << 48);
                if (hx) atomicAdd(&h[ox * W + t2], 1u);
            }
        }
        #pragma unroll 1
        for (; ai < na; ai++) busy &= ~(1ull << (aq[32 * ai] & 63u));   // acks later in the window than the last look
        c.wf_cur[gw] = cur; c.wf_rem[gw] = rem; c.wf_busy[gw] = busy;
        wantb = rem != ASTRA_NOTLOADED;
        freebit = busy != fullmask;
        hint = (wantb && freebit) || last_issue == wlen - 1;
      }
    }
    __syncwarp();
    const u32 wm = __ballot_sync(FULL, wantb), fm = __ballot_sync(FULL, freebit);
    const bool anyh = __any_sync(FULL, hint);
    const u32 am = am0 & ~__ballot_sync(FULL, heavy);         // heavy wavefronts update their own bits later
    if (lane == 0) {
        u32* want = c.want + (size_t)g * nwords + wi;
        u32* freeb = c.freeb + (size_t)g * nwords + wi;
        const u32 ow = *want, of = *freeb;
        c.undo_want[(size_t)g * nwords + wi] = ow; c.undo_freeb[(size_t)g * nwords + wi] = of;
        *want = (ow & ~am) | wm;
        *freeb = (of & ~am) | fm;
        if (anyh) atomicMin(hp, t1);
    }
}

// One wavefront with many issues in the window, on a whole warp: lane = issue index.  The i-th
// issue of the window needs a slot -- one of the F0 slots free at the window start, else the
// (i - F0)-th ack in cycle order -- and its step released, and comes at least one cycle after the
// (i-1)-th: x_i = max(x_{i-1} + 1, c_i), a prefix maximum of c_j - j.  Same result as wf_sim.
__device__ void wf_heavy(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 g, u32 wf, u32 k, u32 t0, u32 t1, u32* scr, u32 lane) {
    const u32 W = c.W, H = c.H, K = c.K, nwords = c.nwords;
    const u64 fullmask = c.fullmask;
    const u32 e0 = c.row_ptr[g], deg = c.row_ptr[g + 1] - e0;
    u32* const cnt = c.cnt + (size_t)g * W;
    u32* const h = c.hist + (size_t)e0 * W;
    u64* const evb = c.evb + (size_t)g * H * W;
    const u32* const t_release = c.t_release;
    const u32* const cul = c.cul;
    const size_t gw = (size_t)g * c.CW + wf;
    u32 cur = c.wf_cur[gw], rem = c.wf_rem[gw];
    const u64 busy = c.wf_busy[gw];
    if (lane == 0) { c.undo_cur[gw] = cur; c.undo_rem[gw] = rem; c.undo_busy[gw] = busy; }
    const u32 b0 = wf * K, w0 = b0 >> 5, sh = b0 & 31;
    u64 rb = 0;
    if (c.ack_n[g]) {
        const u32 bmwords = c.bmwords;
        const u32* bm = c.bitmap + (size_t)(g * c.NW + (k & c.NWmask)) * bmwords;
        const u32 x0 = __ldcg(&bm[w0]);
        const u32 x1 = (w0 + 1 < bmwords) ? __ldcg(&bm[w0 + 1]) : 0u;
        const u32 x2 = (sh && w0 + 2 < bmwords) ? __ldcg(&bm[w0 + 2]) : 0u;
        rb = ((((u64)x1 << 32) | x0) >> sh);
        if (sh) rb |= (u64)x2 << (64 - sh);
        rb &= fullmask;
    }
    const u32 na = __popcll(rb);
    const u64 fb = ~busy & fullmask;
    const u32 F0 = __popcll(fb);
    // scr[64 ..): positions of the set bits of rb (acked slots); scr[128 ..): of fb (free slots)
    {
        const u32 rlo = (u32)rb, rhi = (u32)(rb >> 32), flo = (u32)fb, fhi = (u32)(fb >> 32), lt = lanemask_lt();
        if ((rlo >> lane) & 1u) scr[64 + __popc(rlo & lt)] = lane;
        if ((rhi >> lane) & 1u) scr[64 + __popc(rlo) + __popc(rhi & lt)] = 32 + lane;
        if ((flo >> lane) & 1u) scr[128 + __popc(flo & lt)] = lane;
        if ((fhi >> lane) & 1u) scr[128 + __popc(flo) + __popc(fhi & lt)] = 32 + lane;
        __syncwarp();
    }
    // acks sorted by (cycle, slot) into scr[0 .. na): rank = number of smaller keys
    {
        const u64* rec = c.ack_rec + (size_t)g * c.slots + b0;
        u32 key0 = 0xffffffffu, key1 = 0xffffffffu;
        if (lane < na) { const u32 b = scr[64 + lane]; key0 = (((u32)__ldcg(&rec[b]) - t0) << 6) | b; }
        if (lane + 32 < na) { const u32 b = scr[96 + lane]; key1 = (((u32)__ldcg(&rec[b]) - t0) << 6) | b; }
        u32 r0 = 0, r1 = 0;
        if (na > 32) {
#pragma unroll 2
            for (u32 j = 0; j < 32; j++) {
                const u32 k0 = __shfl_sync(FULL, key0, j), k1 = __shfl_sync(FULL, key1, j);
                r0 += (k0 < key0) + (k1 < key0); r1 += (k0 < key1) + (k1 < key1);
            }
        } else if (na > 1) {
#pragma unroll 4
            for (u32 j = 0; j < 32; j++) r0 += __shfl_sync(FULL, key0, j) < key0;
        }
        if (lane < na) scr[r0] = key0;
        if (lane + 32 < na) scr[r1] = key1;
        __syncwarp();
    }
    const u32 end = c.cul_ptr[g * c.C + wf / c.Wv + 1];
    const u32 wlen = t1 - t0;
    u32 idx = 0, xp = 0, last_issue = 0xffffffffu;              // xp: earliest cycle (relative to t0) of the next issue
    u32 im_lo = 0, im_hi = 0;                                   // slots taken by this lane's issues
    bool stop = false;
    #pragma unroll 1
    while (!stop) {
        if (rem == ASTRA_NOTLOADED) {
            bool got = false;
            #pragma unroll 1
            while (cur < end) {
                const u32 s2 = cul[cur];
                const u32 tr = t_release[s2];
                if (tr >= t1) break;
                if (tr > t0 + xp) xp = tr - t0;
                const u32 q = c.step_q[s2] + (((wf - c.cu_lo[s2] * c.Wv) < c.step_r[s2]) ? 1u : 0u);   // R11
                if (q) { rem = q; got = true; break; }
                cur++;
            }
            if (!got) break;
        }
        const u32 s = cul[cur];
        const u32 ox = c.first_link[s] - e0;
        const bool hx = deg > 1 && ((c.gdirect[g] >> (ox & 31u)) & 1u);
        #pragma unroll 1
        while (rem > 0) {
            const u32 i = idx + lane;
            const u32 want_n = min(32u, rem);
            const bool cand = lane < want_n && i < F0 + na;
            const u32 key = (cand && i >= F0) ? scr[i - F0] : 0u;
            const int val = cand ? (int)(key >> 6) - (int)lane : INT_MIN;
            const int y = max(warp_incl_max(val, lane), (int)xp);
            const u32 x = lane + (u32)y;
            const bool valid = cand && x < wlen;
            const u32 nv = __popc(__ballot_sync(FULL, valid));
            if (valid) {
                const u32 slot = i < F0 ? scr[128 + i] : (key & 63u);
                if (slot < 32) im_lo |= 1u << slot; else im_hi |= 1u << (slot - 32);
                const u32 p = atomicAdd(&cnt[x], 1u);
                if (p < H) evb[(size_t)x * H + p] = (u64)s | ((u64)wf << 20) | ((u64)slot << 32) | ((u64)(x + 1) << ASTRA_FLIT_TIME_SHIFT) | ((u64)ox << 48);
                if (hx) atomicAdd(&h[ox * W + x], 1u);
            }
            if (nv) {
                last_issue = __shfl_sync(FULL, x, nv - 1);
                xp = last_issue + 1; idx += nv; rem -= nv;
            }
            if (nv < want_n) { stop = true; break; }            // out of slots or out of window
        }
        if (!stop && rem == 0) { cur++; rem = ASTRA_NOTLOADED; }
    }
    im_lo = __reduce_or_sync(FULL, im_lo); im_hi = __reduce_or_sync(FULL, im_hi);
    if (lane == 0) {
        const u64 nbusy = (busy & ~rb) | (((u64)im_hi << 32) | im_lo);
        c.wf_cur[gw] = cur; c.wf_rem[gw] = rem; c.wf_busy[gw] = nbusy;
        const bool wantb = rem != ASTRA_NOTLOADED, freebit = nbusy != fullmask;
        u32* want = c.want + (size_t)g * nwords + (wf >> 5);
        u32* freeb = c.freeb + (size_t)g * nwords + (wf >> 5);
        const u32 bit = 1u << (wf & 31);
        if (wantb) atomicOr(want, bit); else atomicAnd(want, ~bit);
        if (freebit) atomicOr(freeb, bit); else atomicAnd(freeb, ~bit);
        if ((wantb && freebit) || last_issue == wlen - 1) atomicMin(hp, t1);
    }
    __syncwarp();
}

// The budget bound: put the wavefronts of word wi of GPU g back to their state at the window start.
__device__ ASTRA_COLD void wf_restore_word(const Ctx& __restrict__ c, u32 g, u32 wi, u32 lane) {
    const u32 am = c.amask[(size_t)g * c.nwords + wi];
    if (am == 0) return;
    if ((am >> lane) & 1u) {
        const size_t gw = (size_t)g * c.CW + wi * 32 + lane;
        c.wf_cur[gw] = c.undo_cur[gw]; c.wf_rem[gw] = c.undo_rem[gw]; c.wf_busy[gw] = c.undo_busy[gw];
    }
    if (lane == 0) {
        c.want[(size_t)g * c.nwords + wi] = c.undo_want[(size_t)g * c.nwords + wi];
        c.freeb[(size_t)g * c.nwords + wi] = c.undo_freeb[(size_t)g * c.nwords + wi];
    }
    __syncwarp();
}

// The words of a budget-bound GPU-window are swept in ascending order (word w needs the grants of all lower
// words), but by several warps: each loads and sorts its word's inputs on its own, then waits for its turn.
__device__ __forceinline__ void turn_wait(u32* turn, u32 wi, u32 lane) {
    if (lane == 0) while (*(volatile u32*)turn != wi) __nanosleep(40);
    __syncwarp();
    __threadfence_block();
}
__device__ __forceinline__ void turn_pass(u32* turn, u32 wi, u32 lane) {
    __syncwarp();
    __threadfence_block();
    if (lane == 0) *(volatile u32*)turn = wi + 1u;
}

// The budget binds in this GPU-window: exact fixed-priority grants (R12), word by word in ascending
// wavefront id.  A wavefront is granted at cycle t iff it is ready and fewer than H wavefronts with a
// lower id are granted at t; occ[t] (the cnt array) holds the grants of all lower words, so the 32
// wavefronts of a word step together through the cycles where one of them is ready and occ[t] < H,
// a ballot giving the rank inside the word.  That rank is the bucket position of the issue.
__device__ ASTRA_COLD void wf_priority_word(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 g, u32 wi, u32 k, u32 t0, u32 t1, u32* scr, u32* turn, u32 lane) {
    const u32 nwords = c.nwords;
    const u32 am = c.amask[(size_t)g * nwords + wi];
    if (am == 0) { if (turn) { turn_wait(turn, wi, lane); turn_pass(turn, wi, lane); } return; }
    const bool active = (am >> lane) & 1u;
    const u32 wf = wi * 32 + lane;
    const u32 W = c.W, H = c.H, K = c.K, wlen = t1 - t0;
    const u64 fullmask = c.fullmask;
    const u32 e0 = c.row_ptr[g], deg = c.row_ptr[g + 1] - e0;
    u32* const occ = c.cnt + (size_t)g * W;
    u32* const h = c.hist + (size_t)e0 * W;
    u64* const evb = c.evb + (size_t)g * H * W;
    const u32* const t_release = c.t_release;
    const u32* const cul = c.cul;
    const size_t gw = (size_t)g * c.CW + wf;
    u32 cur = 0, rem = ASTRA_NOTLOADED, end = 0;
    u64 busy = fullmask;
    unsigned short* const aq = reinterpret_cast<unsigned short*>(scr) + lane;      // as in wf_sim: entry j at aq[32 j]
    u32 na = 0, ai = 0;
    if (active) {
        cur = c.wf_cur[gw]; rem = c.wf_rem[gw]; busy = c.wf_busy[gw];
        end = c.cul_ptr[g * c.C + wf / c.Wv + 1];
        const u32 b0 = wf * K, w0 = b0 >> 5, sh = b0 & 31;
        u64 rb = 0;
        if (c.ack_n[g]) {
            const u32 bmwords = c.bmwords;
            const u32* bm = c.bitmap + (size_t)(g * c.NW + (k & c.NWmask)) * bmwords;
            const u32 x0 = __ldcg(&bm[w0]);
            const u32 x1 = (w0 + 1 < bmwords) ? __ldcg(&bm[w0 + 1]) : 0u;
            const u32 x2 = (sh && w0 + 2 < bmwords) ? __ldcg(&bm[w0 + 2]) : 0u;
            rb = ((((u64)x1 << 32) | x0) >> sh);
            if (sh) rb |= (u64)x2 << (64 - sh);
            rb &= fullmask;
        }
        const u64* rec = c.ack_rec + (size_t)g * c.slots + b0;
        #pragma unroll 1
        while (rb) { const u32 b = __ffsll((long long)rb) - 1; rb &= rb - 1; aq[32 * na++] = (unsigned short)((((u32)__ldcg(&rec[b]) - t0) << 6) | b); }
        #pragma unroll 1
        for (u32 i = 1; i < na; i++) {
            const u32 xv = aq[32 * i]; u32 j = i;
            #pragma unroll 1
            while (j > 0 && aq[32 * (j - 1)] > xv) { aq[32 * j] = aq[32 * (j - 1)]; j--; }
            aq[32 * j] = (unsigned short)xv;
        }
    }
    u32 nq = na ? aq[0] : 0xffffffffu;
    u32 s = 0, ox = 0, last_issue = 0xffffffffu;
    bool have_s = false, hx = false;
    const u32 gdir = c.gdirect[g];
    u32 T = 0;
    if (turn) turn_wait(turn, wi, lane);                       // the grants of all lower words are in occ[] now
    #pragma unroll 1
    for (;;) {
        // bring the lane to cycle T: slots returned by T, step loaded if released by T
        u32 np = 0xffffffffu;                                   // earliest cycle this lane can be ready
        if (active) {
            #pragma unroll 1
            while ((nq >> 6) <= T) { busy &= ~(1ull << (nq & 63u)); ai++; nq = ai < na ? aq[32 * ai] : 0xffffffffu; }
            if (rem == ASTRA_NOTLOADED) {
                #pragma unroll 1
                while (cur < end) {
                    const u32 s2 = cul[cur];
                    const u32 tr = t_release[s2];
                    if (tr >= t1) break;
                    if (tr > t0 + T) { np = tr - t0; break; }
                    const u32 q = c.step_q[s2] + (((wf - c.cu_lo[s2] * c.Wv) < c.step_r[s2]) ? 1u : 0u);   // R11
                    if (q) { rem = q; have_s = false; break; }
                    cur++;
                }
            }
            if (rem != ASTRA_NOTLOADED) np = busy != fullmask ? T : (ai < na ? (nq >> 6) : 0xffffffffu);
        }
        const u32 tmin = __reduce_min_sync(FULL, np);
        if (tmin >= wlen) break;
        if (tmin > T) { T = tmin; continue; }
        const u32 o = occ[T];
        if (o >= H) {                                           // cycle taken by lower ids: next cycle with room
            u32 t2 = T + 1;
            #pragma unroll 1
            for (;;) {
                const bool room = t2 + lane < wlen && occ[t2 + lane] < H;
                const u32 rm2 = __ballot_sync(FULL, room);
                if (rm2) { t2 += __ffs(rm2) - 1; break; }
                t2 += 32;
                if (t2 >= wlen) break;
            }
            if (t2 >= wlen) break;
            T = t2; continue;
        }
        const bool ready = active && rem != ASTRA_NOTLOADED && busy != fullmask;
        const u32 rm = __ballot_sync(FULL, ready);
        const u32 rank = o + __popc(rm & lanemask_lt());
        const bool granted = ready && rank < H;
        if (granted) {
            if (!have_s) { s = cul[cur]; ox = c.first_link[s] - e0; hx = deg > 1 && ((gdir >> (ox & 31u)) & 1u); have_s = true; }
            const u32 slot = __ffsll((long long)~busy) - 1;
            busy |= 1ull << slot;
            evb[(size_t)T * H + rank] = (u64)s | ((u64)wf << 20) | ((u64)slot << 32) | ((u64)(T + 1) << ASTRA_FLIT_TIME_SHIFT) | ((u64)ox << 48);
            if (hx) atomicAdd(&h[ox * W + T], 1u);
            last_issue = T;
            if (--rem == 0) { cur++; rem = ASTRA_NOTLOADED; }
        }
        __syncwarp();
        if (lane == 0) occ[T] = min(H, o + (u32)__popc(rm));
        __syncwarp();
        T++;
        if (T >= wlen) break;
    }
    if (turn) turn_pass(turn, wi, lane);
    bool wantb = false, freebit = false, hint = false;
    if (active) {
        #pragma unroll 1
        for (; ai < na; ai++) busy &= ~(1ull << (aq[32 * ai] & 63u));
        if (rem == ASTRA_NOTLOADED) {                           // a step released by the end of the window is loaded (as in wf_sim)
            #pragma unroll 1
            while (cur < end) {
                const u32 s2 = cul[cur];
                if (t_release[s2] >= t1) break;
                const u32 q = c.step_q[s2] + (((wf - c.cu_lo[s2] * c.Wv) < c.step_r[s2]) ? 1u : 0u);
                if (q) { rem = q; break; }
                cur++;
            }
        }
        c.wf_cur[gw] = cur; c.wf_rem[gw] = rem; c.wf_busy[gw] = busy;
        wantb = rem != ASTRA_NOTLOADED; freebit = busy != fullmask;
        hint = (wantb && freebit) || last_issue == wlen - 1;
    }
    __syncwarp();
    const u32 wm = __ballot_sync(FULL, wantb), fm = __ballot_sync(FULL, freebit);
    const bool anyh = __any_sync(FULL, hint);
    if (lane == 0) {
        u32* want = c.want + (size_t)g * nwords + wi;
        u32* freeb = c.freeb + (size_t)g * nwords + wi;
        *want = (*want & ~am) | wm;
        *freeb = (*freeb & ~am) | fm;
        if (anyh) atomicMin(hp, t1);
    }
    __syncwarp();
}

// stage 2c: did the HBM budget bind in any cycle (R12)?  If not, the run stands: exclusive prefix of
// the per-cycle counts (item enumeration), FIFO positions of every (direct out-link, cycle), new
// tails, and the window's ack bits / released steps are consumed.
__device__ bool gpu_binds(const Ctx& __restrict__ c, u32 g, u32 wlen, u32 lane) {
    const u32* cnt = c.cnt + (size_t)g * c.W;
    bool bind = false;
    #pragma unroll 1
    for (u32 tt = lane; tt < wlen; tt += 32) if (cnt[tt] > c.H) bind = true;
    return __any_sync(FULL, bind);
}

// The run stands (no cycle exceeded H, or the exact grants were computed): three independent parts that
// different warps of the set take -- (a) exclusive prefix of the per-cycle issue counts = item enumeration
// of the window (in place: every warp has finished its budget check by then, see node_window), (b) per
// out-link the absolute FIFO position of each cycle's first line, (c) the window's ack bits are consumed.
__device__ void gpu_finalize_counts(const Ctx& __restrict__ c, u32 g, u32 k, u32 wlen, u32 lane) {
    const u32 W = c.W;
    u32* cnt = c.cnt + (size_t)g * W;
    u32 carry = 0;
    #pragma unroll 1
    for (u32 b = 0; b < W; b += 32) {
        const u32 i = b + lane;
        const u32 v = (i < wlen) ? cnt[i] : 0;
        const u32 incl = warp_incl_scan(v, lane);
        if (i < W) cnt[i] = carry + incl - v;
        carry += __shfl_sync(FULL, incl, 31);
    }
    const u32 e0 = c.row_ptr[g], deg = c.row_ptr[g + 1] - e0;
    if (lane == 0) {
        if (deg == 1 && carry && c.mask_off[e0] == ASTRA_NONE32) c.run[e0] += carry;
        c.sel[(size_t)g * c.H] = carry;                         // issues of the GPU this window (sel is free on this path)
        c.pcnt[g] = 0;
        c.bin_cnt[g * c.NW + (k & c.NWmask)] = 0;
    }
}
__device__ void gpu_finalize_link(const Ctx& __restrict__ c, u32 e, u32 wlen, u32 lane) {
    const u32 W = c.W;
    u32* h = c.hist + (size_t)e * W;
    const bool direct = c.mask_off[e] == ASTRA_NONE32;
    u32 acc = direct ? c.run[e] : 0u;
    const u32 acc0 = acc;
    #pragma unroll 1
    for (u32 b = 0; b < W; b += 32) {
        const u32 i = b + lane;
        const u32 v = (i < wlen) ? h[i] : 0;
        const u32 incl = warp_incl_scan(v, lane);
        if (i < W) h[i] = acc + incl - v;
        acc += __shfl_sync(FULL, incl, 31);
    }
    __syncwarp();
    if (lane == 0 && direct && acc != acc0) c.run[e] = acc;
}
__device__ void gpu_finalize_acks(const Ctx& __restrict__ c, u32 g, u32 k, u32 lane) {
    const u32 n_ack = c.ack_n[g];
    if (n_ack) {
        u32* bm = c.bitmap + (size_t)(g * c.NW + (k & c.NWmask)) * c.bmwords;
        if (n_ack <= c.alcap) {     // every bit of the bin's words is consumed this window: whole words can go
            const u32* list = c.ack_list + (size_t)(g * c.NW + (k & c.NWmask)) * c.alcap;
            #pragma unroll 1
            for (u32 i = lane; i < n_ack; i += 32) bm[__ldcg(&list[i]) >> 5] = 0;
        } else for (u32 i = lane; i < c.bmwords; i += 32) bm[i] = 0;
    }
    #pragma unroll 1
    for (u32 wi = lane; wi < c.nwords; wi += 32) c.amask[(size_t)g * c.nwords + wi] = 0;
}
__device__ void gpu_finalize(const Ctx& __restrict__ c, u32 g, u32 k, u32 wlen, u32 lane) {   // all parts on one warp
    gpu_finalize_counts(c, g, k, wlen, lane);
    const u32 e0 = c.row_ptr[g], deg = c.row_ptr[g + 1] - e0;
    if (deg > 1) for (u32 x = 0; x < deg; x++) if (deg > 32 || ((c.gdirect[g] >> x) & 1u)) gpu_finalize_link(c, e0 + x, wlen, lane);
    gpu_finalize_acks(c, g, k, lane);
    __syncwarp();
}

// stage 2e: rank the issues of GPU g inside their cycle (ascending wavefront id, R7 A2 / R12) and
// put each line where that rank says: FIFO position on a direct out-link, cell slot + injection
// record on a multi-feeder one.  Item i of the window is entry i - cnt[tt] of the bucket of the
// last cycle tt with cnt[tt] <= i (cnt = exclusive prefix of the per-cycle issue counts).
__device__ void ev_place(const Ctx& __restrict__ c, Ctl& ctl, u32 g, u32 chunk, u32 t0, u32 cb, u32 lane) {
    const u32 nev = c.sel[(size_t)g * c.H];
    const u32 cs = chunk * 32, i = cs + lane;
    const bool act = i < nev;
    const u32 amk = __ballot_sync(FULL, act);
    const u32 W = c.W, H = c.H;
    const u32* cnt = c.cnt + (size_t)g * W;                    // by now the exclusive prefix of the per-cycle issue counts
    const u32 e0 = c.row_ptr[g], deg = c.row_ptr[g + 1] - e0;
    u32 tt = 0xffffffffu, st = 0, n = 0, s = 0, wf = 0, o = 0;
    u64 rec = 0;
    const u64* bucket = nullptr;
    if (act) {
        u32 lo = 0, hi = W;                                     // first index with cnt > i
        #pragma unroll 1
        while (lo < hi) { const u32 mid = (lo + hi) >> 1; if (cnt[mid] > i) hi = mid; else lo = mid + 1; }
        tt = lo - 1;
        st = cnt[tt]; n = (tt + 1 < W ? cnt[tt + 1] : nev) - st;
        bucket = c.evb + ((size_t)g * W + tt) * H;
        rec = bucket[i - st];
        s = (u32)rec & 0xfffffu; wf = ((u32)rec >> 20) & 0xfffu;
        o = c.first_link[s];
    }
    if (!act) return;
    // rank among the issues of the same cycle (j) and, for a single-feeder out-link of a GPU with several, among those
    // that take the same out-link (jo); a bucket holds at most H records, each with its wavefront id and out-link
    // (bits 48.. of the record).  The budget-bound sweep writes its buckets in wavefront order already (nheavy marks it).
    u32 j = 0, jo = 0;
    const u32 oxm = o - e0;
    const bool need_jo = deg > 1 && c.mask_off[o] == ASTRA_NONE32;
    if (c.nheavy[g] == ASTRA_NONE32) {
        j = i - st;
        if (need_jo)
#pragma unroll 1
            for (u32 x = 0; x < j; x++) jo += (u32)(bucket[x] >> 48) == oxm;
    } else if (need_jo) {
#pragma unroll 1
        for (u32 x = 0; x < n; x++) {
            const u64 r2 = bucket[x];
            const bool lower = (((u32)r2 >> 20) & 0xfffu) < wf;
            j += lower;
            jo += lower && (u32)(r2 >> 48) == oxm;
        }
    } else {
#pragma unroll 1
        for (u32 x = 0; x < n; x++) j += (((u32)bucket[x] >> 20) & 0xfffu) < wf;
    }
    if (deg == 1) jo = j;
    const u32 d = tt + 1;
    if (c.mask_off[o] == ASTRA_NONE32) {
        const u32 pos = (deg == 1 ? c.run[o] - nev + st : c.hist[(size_t)o * W + tt]) + jo;
        c.ring[c.ring_off[o] + (pos & c.ring_mask[o])] = (rec & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)d << ASTRA_FLIT_TIME_SHIFT);
    } else {
        cell_set(c, o, g, cb, d, c.nd_injoff[g] + j);
        const u32 mm = __activemask();                          // one counter bump for the lanes that record an injection
        u32 p = 0;
        if ((mm & lanemask_lt()) == 0) p = atomicAdd(&c.inj_n[g], (u32)__popc(mm));
        p = __shfl_sync(mm, p, __ffs(mm) - 1) + __popc(mm & lanemask_lt());
        if (p < c.inj_off[g + 1] - c.inj_off[g]) c.inj_list[c.inj_off[g] + p] = (rec & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)(d | (j << 10)) << ASTRA_FLIT_TIME_SHIFT);
        else atomicOr(&ctl.err, 4u);
    }
    // issued counts and the cycle of each step's last issue (R3)
    const u32 ms = __match_any_sync(amk, s);
    const u32 tmax = __reduce_max_sync(ms, t0 + tt);
    if ((ms & lanemask_lt()) == 0) { atomicAdd(&c.issued_cnt[s], (u32)__popc(ms)); atomicMax(&c.t_issued[s], tmax); }
}

// ---------------------------------------------------------------------------------------------
// stage 3a: FIFO positions of the cells of multi-feeder out-link o: exclusive prefix over the
// cell popcounts of the window (R7/R8: cycle by cycle, slot order inside a cycle).
// ---------------------------------------------------------------------------------------------
// every cycle of the window is looked at: links that carry a line per cycle or more
__device__ void link_prefix_dense(const Ctx& __restrict__ c, u32 o, u32 wlen, u32 cb, u32 lane) {
    const u32 v = c.tail[o];
    const u32 mw = c.nd_mw[v], NC = c.NC;
    const u32* masks = c.masks + c.mask_off[o];
    u32* pre = c.pre + c.pre_off[o];
    u32 n_new = 0;
    // four consecutive cycles per lane: their cell words are loaded together, one warp scan per 128 cycles
#pragma unroll 1
    for (u32 b = 0; b < wlen; b += 128) {
        u32 cq[4];
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const u32 tau = b + 4 * lane + q;
            cq[q] = 0;
            if (tau < wlen) {
                u32 ci = cb + tau; if (ci >= NC) ci -= NC;
                for (u32 w = 0; w < mw; w++) cq[q] += __popc(masks[ci * mw + w]);
            }
        }
        const u32 tot = cq[0] + cq[1] + cq[2] + cq[3];
        const u32 incl = warp_incl_scan(tot, lane);
        u32 run = n_new + incl - tot;
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const u32 tau = b + 4 * lane + q;
            if (tau < wlen) pre[tau] = run;
            run += cq[q];
        }
        n_new += __shfl_sync(FULL, incl, 31);
    }
    if (lane == 0) c.run[o] = c.ltail[o] + n_new;
}

// only the cycles marked in the link's bitmap of non-empty cells are looked at: links below one line per cycle
__device__ void link_prefix(const Ctx& __restrict__ c, u32 o, u32 wlen, u32 cb, u32* scr, u32 lane) {
    const u32 v = c.tail[o];
    const u32 mw = c.nd_mw[v], NC = c.NC;
    const u32* masks = c.masks + c.mask_off[o];
    u32* pre = c.pre + c.pre_off[o];
    if (c.nz_off[o] == ASTRA_NONE32) { link_prefix_dense(c, o, wlen, cb, lane); return; }
    const u32* nz = c.nz + c.nz_off[o];
    const u32 nzw = (wlen + 31) / 32;
    // the non-empty cycles of the window (cycle wlen belongs to the next one), in ascending order, into the warp's scratch
    u32 total = 0;
    #pragma unroll 1
    for (u32 wb = 0; wb < nzw; wb += 32) {
        const u32 wi = wb + lane;
        u32 w = wi < nzw ? nz[wi] : 0u;
        if (wi == (wlen >> 5)) w &= (1u << (wlen & 31)) - 1u;
        const u32 cw = __popc(w);
        const u32 incl = warp_incl_scan(cw, lane);
        u32 pos = total + incl - cw;
        #pragma unroll 1
        while (w) { const u32 b = __ffs(w) - 1; w &= w - 1; scr[pos++] = wi * 32 + b; }
        total += __shfl_sync(FULL, incl, 31);
    }
    __syncwarp();
    // cell popcounts and their exclusive prefix, 32 non-empty cycles per step
    u32 n_new = 0;
    #pragma unroll 1
    for (u32 b = 0; b < total; b += 32) {
        const u32 j = b + lane;
        u32 cq = 0, tau = 0;
        if (j < total) {
            tau = scr[j];
            u32 ci = cb + tau; if (ci >= NC) ci -= NC;
            #pragma unroll 1
            for (u32 w = 0; w < mw; w++) cq += __popc(masks[ci * mw + w]);
        }
        const u32 incl = warp_incl_scan(cq, lane);
        if (j < total) pre[tau] = n_new + incl - cq;
        n_new += __shfl_sync(FULL, incl, 31);
    }
    __syncwarp();
    if (lane == 0) c.run[o] = c.ltail[o] + n_new;
}

// stage 3b: GPU g's recorded injections go to their FIFO positions; the ones that enter at the
// first cycle of the next window stay recorded.
__device__ void inject_place(const Ctx& __restrict__ c, u32 g, u32 wlen, u32 cb, u32 lane) {
    const u32 n = c.inj_n[g];
    if (n == 0) return;
    u64* inj = c.inj_list + c.inj_off[g];
    const u32 injoff = c.nd_injoff[g];
    u32 keep = 0;
    #pragma unroll 1
    for (u32 b = 0; b < n; b += 32) {
        const u32 i = b + lane;
        const bool act = i < n;
        const u64 rec = act ? inj[i] : 0ull;
        const u32 tf = (u32)(rec >> ASTRA_FLIT_TIME_SHIFT);
        const u32 d = tf & 0x3ffu, j = (tf >> 10) & 0x3ffu;
        const bool place = act && d < wlen;
        const bool carry = act && !place;
        if (place) {
            const u32 o = c.first_link[(u32)rec & 0xfffffu];
            const u32 pos = c.ltail[o] + cell_pos(c, o, g, cb, d, injoff + j);
            c.ring[c.ring_off[o] + (pos & c.ring_mask[o])] = (rec & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)d << ASTRA_FLIT_TIME_SHIFT);
        }
        const u32 cm = __ballot_sync(FULL, carry);
        __syncwarp();
        // records are in cycle order: the carried ones are the last; dst index <= src index
        if (carry) inj[keep + __popc(cm & lanemask_lt())] = (rec & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)(j << 10) << ASTRA_FLIT_TIME_SHIFT);
        keep += __popc(cm);
        __syncwarp();
    }
    if (lane == 0) c.inj_n[g] = keep;
}

// ---------------------------------------------------------------------------------------------
// stage 4: link e over [t0, t1): acceptance times of the whole FIFO (R9), arrival stamps.
// ---------------------------------------------------------------------------------------------
__device__ void link_service(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 e, u32 k, u32 t0, u32 t1, u32 cb, u32 lane) {
    const u32 wlen = t1 - t0;
    const u32 fh = c.fifo_head[e], tl = c.ltail[e], tn = c.run[e];
    if (c.dirty[e]) {                                        // consume the cells of the window
        const u32 v = c.tail[e];
        const u32 mw = c.nd_mw[v], NC = c.NC;
        u32* masks = c.masks + c.mask_off[e];
        bool carry = false;                                  // injections that enter at t1 (cycle wlen) keep the link marked
        if (c.nz_off[e] == ASTRA_NONE32) {
            // cells [cb, cb + wlen) of the circular array: one or two contiguous word ranges
            const u32 end1 = min(cb + wlen, NC);
            #pragma unroll 1
            for (u32 x = cb * mw + lane; x < end1 * mw; x += 32) masks[x] = 0;
            if (cb + wlen > NC) for (u32 x = lane; x < (cb + wlen - NC) * mw; x += 32) masks[x] = 0;
            __syncwarp();
            u32 ci = cb + wlen; if (ci >= NC) ci -= NC;
            #pragma unroll 1
            for (u32 w = lane; w < mw; w += 32) carry |= masks[ci * mw + w] != 0u;
            carry = __any_sync(FULL, carry);
        } else {                                             // only the marked cells
            u32* nz = c.nz + c.nz_off[e];
            const u32 NZW = (NC + 31) / 32;
            #pragma unroll 1
            for (u32 wi = lane; wi < NZW; wi += 32) {
                u32 w = nz[wi];
                if (w == 0u) continue;
                nz[wi] = 0u;
                if (wi == (wlen >> 5) && ((w >> (wlen & 31)) & 1u)) { carry = true; w &= ~(1u << (wlen & 31)); }
                #pragma unroll 1
                while (w) {
                    const u32 b = __ffs(w) - 1; w &= w - 1;
                    u32 ci = cb + wi * 32 + b; if (ci >= NC) ci -= NC;
                    #pragma unroll 1
                    for (u32 x = 0; x < mw; x++) masks[ci * mw + x] = 0u;
                }
            }
            carry = __any_sync(FULL, carry);
            if (lane == 0 && carry) nz[0] = 1u;                // cycle wlen is cycle 0 of the next window
        }
        if (lane == 0) c.dirty[e] = carry ? 1u : 0u;
        __syncwarp();
    }
    const u32 n_back = tl - fh, n_new = tn - tl;
    const u32 n_tot = n_back + n_new;
    if (n_tot == 0) return;
    u64* ring = c.ring + c.ring_off[e];
    const u32 rmask = c.ring_mask[e];
    if (lane == 0 && tn - ld_vol(&c.pipe_head[e]) > rmask + 1) atomicOr(&ctl.err, 1u);     // ring overflow guard
    const u32 lk = c.lkind[e];
    const u32 kind = lk & 3u, param = lk >> 2;
    const u32 leff = c.leff[e];
    const u32 lq = leff / c.W, lr = leff % c.W;             // arrival window = k + lq + (x + lr >= W)
    const u32 scan_limit = min(n_tot, c.ceilb[e] * wlen);
    // carried service state
    int run_max = INT_MIN;                                  // INT: prefix max of B*a - i ; PERIOD: of a - P*i
    int xn_rel = 0;                                         // PERIOD: earliest next accept, relative to t0
    u32 cr = 0, tc = 0;                                     // GENERAL: credit after the pops of cycle tc
    if (kind == ASTRA_LK_PERIOD) {
        const u32 xn = c.lstate0[e];
        xn_rel = xn > t0 ? (int)(xn - t0) : 0;
    } else if (kind == ASTRA_LK_GENERAL) { cr = c.lstate0[e]; tc = c.lstate1[e]; }
    const u32 capq = c.ceilb[e] * 256u;
    u32 n_acc = 0, first_x = 0, last_x = 0;
    if (kind != ASTRA_LK_GENERAL) {
        // 128 entries per step, four consecutive ones per lane: local running max, then one warp scan
        const int P = (int)param;
        const u32 bmagic = 0xffffffffu / param + 1u;           // n / param == umulhi(n, bmagic) for n < 2^32 / 32 (param <= 31)
        u64 nx[4];                                           // next step's entries, loaded one step ahead
#pragma unroll
        for (int q = 0; q < 4; q++) nx[q] = 4 * lane + q < scan_limit ? ring[(fh + 4 * lane + q) & rmask] : 0ull;
        #pragma unroll 1
        for (u32 base = 0; base < scan_limit; base += 128) {
            const u32 j0 = base + 4 * lane;
            u64 fl[4]; int val[4]; u32 xx[4]; bool act[4];
#pragma unroll
            for (int q = 0; q < 4; q++) { act[q] = j0 + q < scan_limit; fl[q] = nx[q]; }
#pragma unroll
            for (int q = 0; q < 4; q++) nx[q] = j0 + 128 + q < scan_limit ? ring[(fh + j0 + 128 + q) & rmask] : 0ull;
            int m = INT_MIN;
#pragma unroll
            for (int q = 0; q < 4; q++) {
                const u32 j = j0 + q;
                const int a = (act[q] && j >= n_back) ? (int)((u32)(fl[q] >> ASTRA_FLIT_TIME_SHIFT) & 0x3ffu) : 0;
                const int v = kind == ASTRA_LK_INT ? P * a - (int)j : a - P * (int)j;
                m = act[q] ? max(m, v) : m;
                val[q] = m;                                  // running max inside the lane
            }
            // exclusive prefix max of the lane totals, seeded with the carried maximum
            int incl = warp_incl_max(m, lane);
            int excl = __shfl_up_sync(FULL, incl, 1);
            if (lane == 0) excl = INT_MIN;
            excl = max(excl, run_max);
            run_max = max(run_max, __shfl_sync(FULL, incl, 31));
            u32 cnt_acc = 0, cnt_act = 0, xmax = 0;
#pragma unroll
            for (int q = 0; q < 4; q++) {
                const u32 j = j0 + q;
                const int pm = max(excl, val[q]);
                xx[q] = kind == ASTRA_LK_INT ? (param == 1 ? (u32)((int)j + pm) : __umulhi((u32)((int)j + pm), bmagic)) : (u32)(P * (int)j + max(pm, xn_rel));
                const bool acc = act[q] && xx[q] < wlen;
                cnt_act += act[q]; cnt_acc += acc;
                if (acc) {
                    xmax = xx[q];
                    ring[(fh + j) & rmask] = (fl[q] & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)((t0 + xx[q] + leff) & ASTRA_TMASK26) << ASTRA_FLIT_TIME_SHIFT);
                } else xx[q] = 0xffffffffu;
            }
            const u32 tot_acc = __reduce_add_sync(FULL, cnt_acc), tot_act = __reduce_add_sync(FULL, cnt_act);
            if (tot_acc) {
                const u32 x_first = __shfl_sync(FULL, xx[0], 0);   // acceptance is a prefix: entry `base` is the first
                if (n_acc == 0) first_x = x_first;
                last_x = __reduce_max_sync(FULL, xmax);
                n_acc += tot_acc;
                // arrivals of one step fall in at most two lookahead windows
                const u32 w_first = k + lq + (x_first + lr >= c.W ? 1u : 0u);
                u32 c0 = 0;
#pragma unroll
                for (int q = 0; q < 4; q++) c0 += (xx[q] != 0xffffffffu) && (k + lq + (xx[q] + lr >= c.W ? 1u : 0u)) == w_first;
                c0 = __reduce_add_sync(FULL, c0);
                if (lane == 0) {
                    atomicAdd(&c.due_cnt[(size_t)e * c.NW + (w_first & c.NWmask)], c0);
                    if (tot_acc != c0) atomicAdd(&c.due_cnt[(size_t)e * c.NW + ((w_first + 1) & c.NWmask)], tot_acc - c0);
                }
            }
            if (tot_acc != tot_act) break;                   // FIFO: nothing behind a waiting line is accepted
        }
    } else {
    // ring loads run two chunks ahead of the scan
    u64 fq0 = lane < scan_limit ? ring[(fh + lane) & rmask] : 0ull;
    u64 fq1 = 32 + lane < scan_limit ? ring[(fh + 32 + lane) & rmask] : 0ull;
    #pragma unroll 1
    for (u32 base = 0; base < scan_limit; base += 32) {
        const u32 i = base + lane;
        const bool act = i < scan_limit;
        const u32 pos = (fh + i) & rmask;
        const u64 flit = fq0;
        fq0 = fq1;
        fq1 = i + 64 < scan_limit ? ring[(fh + i + 64) & rmask] : 0ull;
        // append cycle relative to t0: backlog was appended before the window
        const u32 a = (act && i >= n_back) ? ((u32)(flit >> ASTRA_FLIT_TIME_SHIFT) & 0x3ffu) : 0u;
        u32 x = 0xffffffffu;                                 // acceptance cycle relative to t0
        if (kind == ASTRA_LK_INT) {
            int val = act ? (int)(param * a) - (int)i : INT_MIN;
            int pm = warp_incl_max(val, lane);
            pm = max(pm, run_max);
            run_max = __shfl_sync(FULL, pm, 31);
            if (act) x = (u32)((int)i + pm) / param;
        } else if (kind == ASTRA_LK_PERIOD) {
            int val = act ? (int)a - (int)(param * i) : INT_MIN;
            int pm = warp_incl_max(val, lane);
            pm = max(pm, run_max);
            run_max = __shfl_sync(FULL, pm, 31);
            // x_i = max(a_i, x_{i-1} + P) with x_{-1} + P = xn_rel
            if (act) x = (u32)((int)(param * i) + max(pm, xn_rel));
        } else {
            // saturating credit walked in FIFO order; every lane tracks the same state
            const u32 bw = param;
            #pragma unroll 1
            for (u32 j = 0; j < 32; j++) {
                if (base + j >= scan_limit) break;
                const u32 aj = t0 + __shfl_sync(FULL, a, j);
                u32 tt = max(aj, tc);
                u64 avail = min((u64)cr + (u64)(tt - tc) * bw, (u64)capq);
                if (avail < 256) {
                    const u32 wait = (u32)((256 - avail + bw - 1) / bw);
                    tt += wait;
                    avail = min(avail + (u64)wait * bw, (u64)capq);
                }
                if (tt >= t1) break;                     // not in this window: state stays at the last accept
                cr = (u32)avail - 256u; tc = tt;
                if (j == lane) x = tt - t0;
            }
        }
        const bool acc = act && x < wlen;
        const u32 accm = __ballot_sync(FULL, acc);
        const u32 actm = __ballot_sync(FULL, act);
        if (accm) {
            if (n_acc == 0) first_x = __shfl_sync(FULL, x, __ffs(accm) - 1);
            last_x = __shfl_sync(FULL, x, 31 - __clz(accm));
            n_acc += __popc(accm);
        }
        if (acc) {
            ring[pos] = (flit & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)((t0 + x + leff) & ASTRA_TMASK26) << ASTRA_FLIT_TIME_SHIFT);
            // lines due at the head per lookahead window: stage 1 of that window reads the count
        }
        if (accm) {                                          // arrivals of a chunk fall in at most two windows
            const u32 wa = k + lq + (x + lr >= c.W ? 1u : 0u);
            const u32 w_first = __shfl_sync(FULL, wa, __ffs(accm) - 1);
            const u32 m0 = __ballot_sync(FULL, acc && wa == w_first);
            if (lane == 0) {
                atomicAdd(&c.due_cnt[(size_t)e * c.NW + (w_first & c.NWmask)], (u32)__popc(m0));
                if (accm != m0) atomicAdd(&c.due_cnt[(size_t)e * c.NW + ((w_first + 1) & c.NWmask)], (u32)__popc(accm & ~m0));
            }
        }
        if (accm != actm) break;                             // FIFO: nothing behind a waiting line is accepted
    }
    }
    if (lane == 0) {
        c.fifo_head[e] = fh + n_acc;
        c.ltail[e] = tn;
        if (n_acc) {
            c.link_lines[e] += n_acc;
            atomicMin(hp, t0 + first_x + leff);
            if (kind == ASTRA_LK_PERIOD) c.lstate0[e] = t0 + last_x + param;
        }
        if (kind == ASTRA_LK_GENERAL) { c.lstate0[e] = cr; c.lstate1[e] = tc; }
        if (n_tot > n_acc) atomicMin(hp, t1);
    }
}

__device__ void resolve_ctx(Ctx& c, const PointDesc& P, const uint8_t* cb, uint8_t* ws, uint8_t* hot, uint8_t* rs, u32 rank) {
    c.G = P.G; c.V = P.V; c.E = P.E; c.S = P.S; c.C = P.C; c.Wv = P.Wv; c.K = P.K; c.H = P.H;
    c.CW = P.CW; c.nwords = P.nwords; c.slots = P.slots; c.bmwords = P.bmwords;
    c.W = P.Wcyc; c.NC = P.NC; c.NW = P.NW; c.NWmask = P.NW - 1; c.kmagic = P.kdiv_magic;
    c.tmax = (u32)P.max_cycles; c.flags = P.flags; c.alcap = P.alcap; c.pcu = P.pcu;
    c.fullmask = P.K >= 64 ? ~0ull : ((1ull << P.K) - 1);
    c.group = P.group; c.rank = rank;
#define X(n) c.n = (const u32*)(cb + P.c_off[ASTRA_C_##n]);
    ASTRA_CONST_TABLES(X)
#undef X
#define X(n, t, i) c.n = (t*)(((P.a_off[ASTRA_A_##n] & ASTRA_PLACE_SMEM) ? hot : ws) + (P.a_off[ASTRA_A_##n] & ~(ASTRA_PLACE_SMEM | ASTRA_PLACE_LOCAL)));
    ASTRA_WS_ARRAYS(X)
#undef X
    // node range of this CTA (the whole graph when the point runs on one CTA)
    c.v_lo = c.part[rank]; c.v_hi = c.part[rank + 1];
    c.g_lo = min(c.v_lo, c.G); c.g_hi = min(c.v_hi, c.G);
    // arrays that hold only this CTA's GPUs are indexed by absolute GPU id through a pointer moved back by g_lo strides
#define X(n, per_gpu, eb) if (P.a_off[ASTRA_A_##n] & ASTRA_PLACE_LOCAL) c.n -= (size_t)c.g_lo * (per_gpu);
    ASTRA_GPU_ARRAYS(X)
#undef X
    if (P.a_off[ASTRA_A_hist] & ASTRA_PLACE_LOCAL) c.hist -= (size_t)c.row_ptr[c.g_lo] * P.Wcyc;
    c.e_lo = c.row_ptr[c.v_lo]; c.e_hi = c.row_ptr[c.v_hi];
    c.i_lo = c.in_ptr[c.v_lo]; c.i_hi = c.in_ptr[c.v_hi];
    c.r_step_ts = (u64*)(rs + P.r_step_ts);
    c.r_link_lines = (u64*)(rs + P.r_link_lines);
    c.r_summary = (DeviceSummary*)(rs + P.r_summary);
    c.r_diag = (u64*)(rs + P.r_diag);
}

// Barrier over the CTAs of a group.  The grid is launched cooperatively (astra_engine_launch), so all
// CTAs are co-resident or the launch fails; the spin is bounded all the same: after ASTRA_SPIN_CLOCKS
// without progress the CTA raises the kernel-wide abort flag and every CTA leaves.
// `target` = number of arrivals that completes this barrier.  Returns false on abort.
#define ASTRA_SPIN_CLOCKS (1ll << 34)     // about 8 s at 2 GHz
__device__ __forceinline__ bool group_barrier(GroupCtl* gc, u32 target, u32* abort_flag, Ctl& ctl) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const u32 mine = atomicAdd(&gc->bar, 1u) + 1u;           // the last to arrive knows it from its own count: no poll
        const long long start = clock64();
        u32 spins = 0;
        #pragma unroll 1
        while ((int32_t)(mine - target) < 0 && (int32_t)(*(volatile u32*)&gc->bar - target) < 0) {
            if ((++spins & 0x3ffu) == 0) {
                if (*(volatile u32*)abort_flag) { ctl.abort = 1u; break; }
                if (clock64() - start > ASTRA_SPIN_CLOCKS) { atomicExch(abort_flag, 1u); ctl.abort = 1u; break; }
            }
        }
        __threadfence();
    }
    __syncthreads();
    return ctl.abort == 0u;
}

// Barrier over the `ws` warps that work on one simulated node (named barrier 1 + set; a single warp
// needs only its own lanes).  Orders the set's shared- and global-memory accesses like __syncthreads.
__device__ __forceinline__ void set_sync(u32 ws, u32 set) {
    if (ws == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" :: "r"(set + 1u), "r"(ws * 32u) : "memory");
}

// Link service of one link by all ws warps of a node's set (a GPU's one or two FIFOs of several hundred entries and
// sixteen warps): warp r takes entries [128 r, 128 r + 128), the blocks' maxima are combined through shared memory.
// Integer and 1/P bandwidths, single-feeder links, 129 .. 128 ws entries; anything else falls to one warp.
__device__ void link_service_set(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 e, u32 k, u32 t0, u32 t1, u32 cb,
                                 u32 lane, u32 sw, u32 ws, u32 set) {
    const u32 wlen = t1 - t0;
    const u32 fh = c.fifo_head[e], tl = c.ltail[e], tn = c.run[e];
    const u32 n_back = tl - fh, n_tot = tn - fh;
    const u32 lk = c.lkind[e];
    const u32 kind = lk & 3u, param = lk >> 2;
    const u32 scan_limit = min(n_tot, c.ceilb[e] * wlen);
    if (kind == ASTRA_LK_GENERAL || scan_limit > 128u * ws || scan_limit <= 128u || c.dirty[e]) {
        set_sync(ws, set);                  // every warp has taken this decision before warp 0 moves the link's cursors
        if (sw == 0) link_service(c, ctl, hp, e, k, t0, t1, cb, lane);
        return;
    }
    u64* ring = c.ring + c.ring_off[e];
    const u32 rmask = c.ring_mask[e];
    const u32 leff = c.leff[e];
    const u32 lq = leff / c.W, lr = leff % c.W;
    const int P = (int)param;
    const u32 bmagic = 0xffffffffu / param + 1u;
    int xn_rel = 0;
    if (kind == ASTRA_LK_PERIOD) { const u32 xn = c.lstate0[e]; xn_rel = xn > t0 ? (int)(xn - t0) : 0; }
    const u32 warp = threadIdx.x >> 5;
    // phase 1: the block's entries, running maxima inside the lane, the block's maximum
    const u32 j0 = 128u * sw + 4u * lane;
    u64 fl[4]; int val[4]; bool act[4];
    int m = INT_MIN;
#pragma unroll
    for (int q = 0; q < 4; q++) { act[q] = j0 + q < scan_limit; fl[q] = act[q] ? ring[(fh + j0 + q) & rmask] : 0ull; }
#pragma unroll
    for (int q = 0; q < 4; q++) {
        const u32 j = j0 + q;
        const int a = (act[q] && j >= n_back) ? (int)((u32)(fl[q] >> ASTRA_FLIT_TIME_SHIFT) & 0x3ffu) : 0;
        const int v = kind == ASTRA_LK_INT ? P * a - (int)j : a - P * (int)j;
        m = act[q] ? max(m, v) : m;
        val[q] = m;
    }
    const int incl = warp_incl_max(m, lane);
    int excl = __shfl_up_sync(FULL, incl, 1);
    if (lane == 0) excl = INT_MIN;
    if (lane == 31) ctl.ls_max[warp] = incl;
    set_sync(ws, set);
    // phase 2: maxima of the blocks before this one, acceptance cycles, arrival stamps
    {
        const int bm = lane < sw ? ctl.ls_max[warp - sw + lane] : INT_MIN;
        excl = max(excl, (int)__reduce_max_sync(FULL, bm));
    }
    u32 xx[4], cnt_acc = 0, xmax = 0;
#pragma unroll
    for (int q = 0; q < 4; q++) {
        const u32 j = j0 + q;
        const int pm = max(excl, val[q]);
        xx[q] = kind == ASTRA_LK_INT ? (param == 1 ? (u32)((int)j + pm) : __umulhi((u32)((int)j + pm), bmagic)) : (u32)(P * (int)j + max(pm, xn_rel));
        const bool acc = act[q] && xx[q] < wlen;
        cnt_acc += acc;
        if (acc) {
            xmax = xx[q];
            ring[(fh + j) & rmask] = (fl[q] & ASTRA_FLIT_PAYLOAD_MASK) | ((u64)((t0 + xx[q] + leff) & ASTRA_TMASK26) << ASTRA_FLIT_TIME_SHIFT);
        } else xx[q] = 0xffffffffu;
    }
    const u32 tot_acc = __reduce_add_sync(FULL, cnt_acc);
    if (tot_acc) {
        const u32 x_first = __shfl_sync(FULL, xx[0], 0);       // acceptance is a prefix: the block's first entry is its first accepted one
        const u32 x_last = __reduce_max_sync(FULL, xmax);
        const u32 w_first = k + lq + (x_first + lr >= c.W ? 1u : 0u);
        u32 c0 = 0;
#pragma unroll
        for (int q = 0; q < 4; q++) c0 += (xx[q] != 0xffffffffu) && (k + lq + (xx[q] + lr >= c.W ? 1u : 0u)) == w_first;
        c0 = __reduce_add_sync(FULL, c0);
        if (lane == 0) {
            atomicAdd(&c.due_cnt[(size_t)e * c.NW + (w_first & c.NWmask)], c0);
            if (tot_acc != c0) atomicAdd(&c.due_cnt[(size_t)e * c.NW + ((w_first + 1) & c.NWmask)], tot_acc - c0);
            atomicAdd(&ctl.ls_acc[set], tot_acc);
            atomicMax(&ctl.ls_last[set], x_last);
            if (sw == 0) atomicMin(hp, t0 + x_first + leff);
        }
    }
    set_sync(ws, set);
    if (sw == 0 && lane == 0) {
        const u32 n_acc = ctl.ls_acc[set], last_x = ctl.ls_last[set];
        ctl.ls_acc[set] = 0u; ctl.ls_last[set] = 0u;
        c.fifo_head[e] = fh + n_acc;
        c.ltail[e] = tn;
        if (n_acc) {
            c.link_lines[e] += n_acc;
            if (kind == ASTRA_LK_PERIOD) c.lstate0[e] = t0 + last_x + param;
        }
        if (n_tot > n_acc) atomicMin(hp, t1);
        if (tn - ld_vol(&c.pipe_head[e]) > rmask + 1) atomicOr(&ctl.err, 1u);     // ring overflow guard
    }
}

// The rest of a node's window after the issue decisions: placement of the window's issues (or the cycle-serial
// issue path), merge into multi-feeder out-links, link service.  e_l .. fl_l: the node's first 32 in-links, one per
// lane (id, lines due, read cursor, arrival path), as loaded by stage 1.
__device__ void node_tail(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 v, u32 k, u32 t0, u32 t1, u32 cb,
                          u32* scr, u32 lane, u32 sw, u32 ws, u32 set, bool diag_lane, u32 mode,
                          u32 e_l, u32 n_l, u32 lo_l, u32 fl_l) {
#ifdef ASTRA_DIAG
    long long dck = clock64();
#endif
    const u32 wlen = t1 - t0;
    const bool is_gpu = v < c.G;
    const u32 g = v;
    const u32 i_lo = c.in_ptr[v], i_hi = c.in_ptr[v + 1];
    const u32 e_lo = c.row_ptr[v], e_hi = c.row_ptr[v + 1];
    const bool serial_arr = (c.flags & (u32)ASTRA_FLAG_SERIAL_ARRIVALS) != 0;
    const u32 kb = k & c.NWmask;
    if (mode == 2u) {                        // cycle-serial path
        if (sw == 0) {
            ack_sort(c, ctl, g, k, t0, wlen, scr, lane);
            issue_window(c, ctl, hp, g, t0, t1, cb, lane);
            #pragma unroll 1
            for (u32 wi = lane; wi < c.nwords; wi += 32) c.amask[(size_t)g * c.nwords + wi] = 0;
        }
        set_sync(ws, set);
    } else if (mode == 1u) {
        const u32 nch = (c.sel[(size_t)g * c.H] + 31) / 32;
        #pragma unroll 1
        for (u32 ch = sw; ch < nch; ch += ws) ev_place(c, ctl, g, ch, t0, cb, lane);
        set_sync(ws, set);
    }
    DIAG_CLK(4);

    // ---- stage 3: merge into multi-feeder out-links of v (skipped when none received a line) ----
    bool any_dirty = false;
    #pragma unroll 1
    for (u32 e = e_lo + lane; e < e_hi; e += 32) any_dirty |= c.dirty[e] != 0u;
    any_dirty = __any_sync(FULL, any_dirty);
    if (any_dirty) {
        #pragma unroll 1
        for (u32 e = e_lo + sw; e < e_hi; e += ws)
            if (c.dirty[e]) link_prefix(c, e, wlen, cb, scr, lane);
        set_sync(ws, set);
        if (is_gpu && sw == ws - 1) inject_place(c, v, wlen, cb, lane);
        u32 tmod3 = 0;
        #pragma unroll 1
        for (u32 ib = i_lo; ib < i_hi; ib += 32) {
            const u32 i = ib + lane;
            u32 e_b = e_l, n_b = n_l, lo_b = lo_l, fl_b = fl_l;
            if (ib != i_lo) {
                e_b = n_b = lo_b = fl_b = 0;
                if (i < i_hi) {
                    e_b = c.in_link[i]; n_b = ld_vol(&c.due_cnt[(size_t)e_b * c.NW + kb]);
                    lo_b = c.pipe_head[e_b]; fl_b = serial_arr ? 0u : c.lflag[e_b];
                }
            }
            // links that marked cells in pass 1 go over the same lines again, now with the FIFO positions known
            const bool again = i < i_hi && (fl_b == 0u ? c.ndue[e_b] != 0u : (fl_b == ASTRA_LF_CELLS && c.tl_base[e_b] != 0u));
            u32 nm = __ballot_sync(FULL, again);
            #pragma unroll 1
            while (nm) {
                const u32 src = __ffs(nm) - 1; nm &= nm - 1;
                const u32 e = __shfl_sync(FULL, e_b, src), n = __shfl_sync(FULL, n_b, src);
                const u32 lo = __shfl_sync(FULL, lo_b, src), fl = __shfl_sync(FULL, fl_b, src);
                const u32 first = (sw + ws - tmod3) % ws;
                if (fl == 0u) { if (first == 0u) arrivals_link<3>(c, ctl, hp, ib + src, 0u, k, t0, wlen, cb, lane); tmod3 = (tmod3 + 1) % ws; continue; }
                #pragma unroll 1
                for (u32 ch = first; ch * 64 < n; ch += ws) cells_place_chunk(c, e, lo, n, ch, t0, wlen, cb, lane);
                tmod3 = (tmod3 + (n + 63) / 64) % ws;
            }
        }
        set_sync(ws, set);
    }
    DIAG_CLK(5);

    // ---- stage 4: link service of v's out-links (R9); the in-links' cursors move past the window ----
    if (sw == ws - 1) {
        #pragma unroll 1
        for (u32 ib = i_lo; ib < i_hi; ib += 32) {
            const u32 i = ib + lane;
            if (i >= i_hi) continue;
            u32 e = e_l, n = n_l, fl = fl_l;
            if (ib != i_lo) { e = c.in_link[i]; n = ld_vol(&c.due_cnt[(size_t)e * c.NW + kb]); fl = serial_arr ? 0u : c.lflag[e]; }
            if (n == 0) continue;
            c.due_cnt[(size_t)e * c.NW + kb] = 0;
            if (fl != 0u) { c.pipe_head[e] += n; c.tl_base[e] = 0; }
        }
    }
    if (ws >= 8u * (e_hi - e_lo)) {                              // one or two links and many warps: every link by the whole set
#pragma unroll 1
        for (u32 e = e_lo; e < e_hi; e++) link_service_set(c, ctl, hp, e, k, t0, t1, cb, lane, sw, ws, set);
    } else
#pragma unroll 1
    for (u32 e = e_lo + sw; e < e_hi; e += ws) link_service(c, ctl, hp, e, k, t0, t1, cb, lane);
    DIAG_CLK(6);
}

// ---------------------------------------------------------------------------------------------
// One lookahead window of one simulated node v, by the warp set that owns it (sw = warp index in the
// set of ws warps).  Inside a window nothing a node does can reach another node (W <= min Leff), so
// the stages of a node order only against each other: set barriers, no block barrier.
// ---------------------------------------------------------------------------------------------
__device__ void node_window(const Ctx& __restrict__ c, Ctl& ctl, u32* hp, u32 v, u32 k, u32 t0, u32 t1, u32 cb,
                            u32* scr, u32 lane, u32 sw, u32 ws, u32 set, bool diag_lane) {
#ifdef ASTRA_DIAG
    long long dck = clock64();
#endif
    const u32 wlen = t1 - t0;
    const bool is_gpu = v < c.G;
    const u32 i_lo = c.in_ptr[v], i_hi = c.in_ptr[v + 1];
    const u32 e_lo = c.row_ptr[v], e_hi = c.row_ptr[v + 1];
    const bool serial_arr = (c.flags & (u32)ASTRA_FLAG_SERIAL_ARRIVALS) != 0;
    const u32 kb = k & c.NWmask;

    // ---- stage 1: ack discovery (A3) and arrivals (A1) as chunk tasks over the set's warps ----
    // Task t of the stage (all its chunks numbered through) is taken by warp t mod ws: tmod is the running
    // task count mod ws, the same in every warp, and `(sw + ws - tmod) % ws` the first chunk of the next group
    // that falls to this warp.
    bool any_fwd = false;
    u32 tmod = 0;
    if (is_gpu) {
        if (sw == ws - 1) stage1_setup_gpu(c, ctl, hp, v, k, lane);
        const u32 n_ack = ld_vol(&c.bin_cnt[v * c.NW + kb]);
        if (n_ack && n_ack <= c.alcap) {                         // alcap == 0: no list, the bitmap is scanned
            #pragma unroll 1
            for (u32 ch = sw; ch * 128 < n_ack; ch += ws) ack_list_chunk(c, ctl, v, ch, n_ack, k, t1, lane);
            tmod = ((n_ack + 127) / 128) % ws;
        } else if (n_ack) {
            const u32 nch = (c.bmwords + 31) / 32;
            #pragma unroll 1
            for (u32 ch = sw; ch < nch; ch += ws) ack_chunk(c, ctl, v, ch, k, t1, scr, lane);
            tmod = nch % ws;
        }
    }
    // the node's in-links, one per lane: id, lines due this window (counted by the link's service when it
    // accepted them), read cursor, arrival path -- all loads of a batch of 32 links in flight at once
    u32 e_l = 0, n_l = 0, lo_l = 0, fl_l = 0;
    #pragma unroll 1
    for (u32 ib = i_lo; ib < i_hi; ib += 32) {
        const u32 i = ib + lane;
        u32 e_b = 0, n_b = 0, lo_b = 0, fl_b = 0;
        if (i < i_hi) {
            e_b = c.in_link[i];
            n_b = ld_vol(&c.due_cnt[(size_t)e_b * c.NW + kb]);
            lo_b = c.pipe_head[e_b];
            fl_b = serial_arr ? 0u : c.lflag[e_b];
            if (sw == (i - i_lo) % ws) link_inflight_hint(c, ctl, hp, e_b, lo_b, k);
        }
        if (ib == i_lo) { e_l = e_b; n_l = n_b; lo_l = lo_b; fl_l = fl_b; }     // first batch stays in registers for stages 3 and 4
        u32 nm = __ballot_sync(FULL, n_b != 0u);
        #pragma unroll 1
        while (nm) {
            const u32 src = __ffs(nm) - 1; nm &= nm - 1;
            const u32 e = __shfl_sync(FULL, e_b, src), n = __shfl_sync(FULL, n_b, src);
            const u32 lo = __shfl_sync(FULL, lo_b, src), fl = __shfl_sync(FULL, fl_b, src);
            const u32 first = (sw + ws - tmod) % ws;
            if (fl == 0u) { if (first == 0u) arrivals_link<1>(c, ctl, hp, ib + src, n, k, t0, wlen, cb, lane); tmod = (tmod + 1) % ws; continue; }
            if (fl == ASTRA_LF_DELIVER_ONLY) {
                #pragma unroll 1
                for (u32 ch = first; ch * 32 < n; ch += ws) deliver_chunk(c, ctl, hp, e, lo, n, ch, k, t0, wlen, lane);
            } else if (fl == ASTRA_LF_FORWARD_ONLY) {
                const u32 base = c.run[c.lfwd[e]];
                #pragma unroll 1
                for (u32 ch = first; ch * 32 < n; ch += ws) forward_chunk(c, e, lo, n, base, ch, t0, wlen, lane);
                any_fwd = true;
            } else {
                #pragma unroll 1
                for (u32 ch = first; ch * 64 < n; ch += ws) cells_chunk(c, ctl, hp, e, lo, n, ch, k, t0, wlen, cb, lane);
            }
            tmod = (tmod + (fl == ASTRA_LF_CELLS ? (n + 63) / 64 : (n + 31) / 32)) % ws;
        }
    }
    set_sync(ws, set);
    if (any_fwd && sw == 0) {                    // forwarded lines are now in the next link's FIFO
        #pragma unroll 1
        for (u32 ib = i_lo; ib < i_hi; ib += 32) {
            const u32 i = ib + lane;
            if (i >= i_hi) continue;
            const u32 e = ib == i_lo ? e_l : c.in_link[i];
            if (!serial_arr && c.lflag[e] == ASTRA_LF_FORWARD_ONLY) c.run[c.lfwd[e]] += ld_vol(&c.due_cnt[(size_t)e * c.NW + kb]);
        }
    }
    DIAG_CLK(0);

    // ---- stage 2: release + issue of GPU v (R10 - R13) ----
    u32 mode = 0;
    const u32 g = v;
    if (is_gpu) {
        if (sw == 0) gpu_prepare(c, ctl, g, t0, t1, lane);
        set_sync(ws, set);
        DIAG_CLK(1);
        mode = c.gmode[g];
    }
    if (mode == 1u) {
        #pragma unroll 1
        for (u32 wi = sw; wi < c.nwords; wi += ws) wf_sim(c, ctl, hp, g, wi, k, t0, t1, scr, lane);
        set_sync(ws, set);
        const u32 nh = c.nheavy[g];
        if (nh) {
            #pragma unroll 1
            for (u32 j = sw; j < nh; j += ws) wf_heavy(c, ctl, hp, g, c.hlist[(size_t)g * c.CW + j], k, t0, t1, scr, lane);
            set_sync(ws, set);
        }
        DIAG_CLK(2);
        const bool bind = gpu_binds(c, g, wlen, lane);     // every warp checks: the same answer everywhere ...
        set_sync(ws, set);                                  // ... before anybody writes over the counts
        const u32 deg = e_hi - e_lo;
        if (!bind) {                                        // the parts of the commit are dealt out
            if (sw == 0) gpu_finalize_counts(c, g, k, wlen, lane);
            if (deg > 1) for (u32 x = (sw + ws - 1) % ws; x < deg; x += ws) if (deg > 32 || ((c.gdirect[g] >> x) & 1u)) gpu_finalize_link(c, e_lo + x, wlen, lane);
            if (sw == ws - 1) gpu_finalize_acks(c, g, k, lane);
        } else if (c.flags & (u32)ASTRA_FLAG_NO_PRIORITY_SWEEP) {      // testing: back to the window start, cycle-serial path
            #pragma unroll 1
            for (u32 wi = sw; wi < c.nwords; wi += ws) wf_restore_word(c, g, wi, lane);
            if (sw == 0 && lane == 0) c.gmode[g] = 2u;
        } else {
            // The budget binds: back to the window start, then the exact grants word by word (wf_priority_word).
            // The sweep is ordered, but every warp of the set loads and sorts its words' inputs on its own and then
            // waits for its turn (a CTA-wide version for one-warp sets was measured: no gain on config 4).
            if (sw == 0 && lane == 0) DIAG_ADD(6, 1);
            #pragma unroll 1
            for (u32 i = sw * 32 + lane; i < c.W; i += ws * 32) c.cnt[(size_t)g * c.W + i] = 0;
            if (deg > 1) for (u32 x = 0; x < deg; x++)
                if (deg > 32 || ((c.gdirect[g] >> x) & 1u)) for (u32 i = sw * 32 + lane; i < c.W; i += ws * 32) c.hist[(size_t)(e_lo + x) * c.W + i] = 0;
            if (sw == 0 && lane == 0) c.turn[g] = 0u;
            set_sync(ws, set);
            #pragma unroll 1
            for (u32 wi = sw; wi < c.nwords; wi += ws) {
                wf_restore_word(c, g, wi, lane);
                wf_priority_word(c, ctl, hp, g, wi, k, t0, t1, scr, ws > 1 ? &c.turn[g] : nullptr, lane);
            }
            set_sync(ws, set);
            if (sw == 0) { gpu_finalize(c, g, k, wlen, lane); if (lane == 0) c.nheavy[g] = ASTRA_NONE32; }     // buckets are in wavefront order (ev_place)
        }
        set_sync(ws, set);
        mode = c.gmode[g];
    } else if (!is_gpu && any_fwd) set_sync(ws, set);
    DIAG_CLK(3);
    node_tail(c, ctl, hp, v, k, t0, t1, cb, scr, lane, sw, ws, set, diag_lane, mode, e_l, n_l, lo_l, fl_l);
}

// Run-ahead windows: wait until the nodes of `pm` have completed `need_pred` windows and all nodes `need_all`.
// Returns 0, or 1 + final status when the run has ended meanwhile (or an internal error / a time-out ends it).
__device__ u32 wait_prog(Ctl& ctl, u32 lane, u32 n_nodes, u32 pm, u32 need_pred, u32 allm, u32 need_all) {
    const long long start = clock64();
#pragma unroll 1
    for (u32 spins = 0;; spins++) {
        const u32 p = lane < n_nodes ? *(volatile u32*)&ctl.prog[lane] : 0xffffffffu;
        const u32 okp = __ballot_sync(FULL, p >= need_pred), oka = __ballot_sync(FULL, p >= need_all);
        const u32 stop = *(volatile u32*)&ctl.stop;
        if (stop) return stop;
        if (*(volatile u32*)&ctl.err || ((spins & 0xfffu) == 0xfffu && clock64() - start > ASTRA_SPIN_CLOCKS)) {
            if (lane == 0) { atomicOr(&ctl.err, 16u); atomicCAS(&ctl.stop, 0u, 1u + (u32)ASTRA_STATUS_INTERNAL); }
            __syncwarp();
            return 1u + (u32)ASTRA_STATUS_INTERNAL;
        }
        if ((okp & pm) == pm && (oka & allm) == allm) { __threadfence_block(); return 0u; }
        __nanosleep(64);
    }
}

// TMA bulk copy global -> shared memory, completion counted in bytes on an mbarrier (all addresses and the size
// multiples of 16 bytes).  One thread issues; everybody waits on the barrier's phase.
__device__ __forceinline__ void bulk_g2s(u32 dst_smem, const void* src, u32 bytes, u32 mbar_smem) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst_smem), "l"(src), "r"(bytes), "r"(mbar_smem) : "memory");
}
__device__ __forceinline__ void mbar_wait(u32 mbar_smem, u32 phase) {
    u32 ok;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(mbar_smem), "r"(phase) : "memory");
    } while (!ok);
}

// One thread: the ten per-step constant tables of the point -> the staging area (TMA bulk copies counted on the
// mbarrier 128 bytes below it); the Ctx then points at the copies.  A call of its own: keeps its registers out of the kernel body.
__device__ __noinline__ void stage_tables(Ctx& c, Ctl& ctl, uint8_t* stage, u32 stage_pad) {
    const u32 stage_s = (u32)__cvta_generic_to_shared(stage), mbar_s = stage_s - 128u;
    ctl.stage_wait = ctl.stage_phase; ctl.stage_phase ^= 1u;        // the phase everybody waits for
    const u32* src[STAGE_TABLES] = {c.step_od, c.lines, c.cu_lo, c.cu_n, c.step_q, c.step_r, c.first_link, c.step_alpha, c.step_aq, c.step_ar};
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // the last point's generic reads of the area are done
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(mbar_s), "r"(STAGE_TABLES * stage_pad) : "memory");
#pragma unroll
    for (u32 q = 0; q < STAGE_TABLES; q++) bulk_g2s(stage_s + q * stage_pad, src[q], stage_pad, mbar_s);
    const u32* const st = (const u32*)stage;
    const u32 w = stage_pad / 4u;
    c.step_od = st; c.lines = st + w; c.cu_lo = st + 2 * w; c.cu_n = st + 3 * w; c.step_q = st + 4 * w; c.step_r = st + 5 * w;
    c.first_link = st + 6 * w; c.step_alpha = st + 7 * w; c.step_aq = st + 8 * w; c.step_ar = st + 9 * w;
}

__device__ __forceinline__ void
step_kernel_body(const uint8_t* __restrict__ cblob, uint8_t* __restrict__ ws_base, uint8_t* __restrict__ results,
                  const PointDesc* __restrict__ points, const u32* __restrict__ order, u32* queue,
                  GroupCtl* groups, u32 n_points, u32 n_big, u32 n_slots, u32 group0,
                  u64 ws_big_stride, u64 ws_single_off, u64 ws_single_stride, u32 hot_off) {
    extern __shared__ __align__(16) uint8_t smem[];
    Ctx& c = *reinterpret_cast<Ctx*>(smem);
    Ctl& ctl = *reinterpret_cast<Ctl*>(smem + ((sizeof(Ctx) + 15) & ~size_t(15)));
    u32* scr_all = reinterpret_cast<u32*>(smem + ((sizeof(Ctx) + 15) & ~size_t(15)) + ((sizeof(Ctl) + 15) & ~size_t(15)));
    uint8_t* hot = smem + hot_off;
    const u32 tid = threadIdx.x, nthr = blockDim.x;
    const u32 lane = tid & 31, warp = tid >> 5, nwarps = nthr >> 5;
    u32* scr = scr_all + warp * SCR_WORDS;
    u32* const abort_flag = queue + 2;
    // CTAs [0, n_slots * group0) form the groups that run the big points; every CTA can run small ones
    const bool in_slot = blockIdx.x < n_slots * group0;
    u32 group = in_slot ? group0 : 1u;
    u32 rank = in_slot ? blockIdx.x % group0 : 0u;
    const u32 gid = in_slot ? blockIdx.x / group0 : 0u;
    uint8_t* ws = in_slot ? ws_base + (size_t)gid * ws_big_stride : ws_base + ws_single_off + (size_t)blockIdx.x * ws_single_stride;
    GroupCtl* gc = groups + gid;
    u32 bar_target = 0;                 // arrivals that complete the next group barrier
    // staging area of the per-step constant tables and its mbarrier, right below the hot region -- present when the launch
    // reserved it (astra_engine_fixed_smem): the hot region then starts 128 + STAGE_BYTES above the per-warp scratch
#define HAS_STAGE (nwarps == 16u && hot_off >= (u32)((((sizeof(Ctx) + 15) & ~size_t(15)) + ((sizeof(Ctl) + 15) & ~size_t(15)) + (size_t)nwarps * SCR_WORDS * sizeof(u32) + 127) & ~size_t(127)) + 128u + STAGE_BYTES)
#define STAGE_S ((u32)__cvta_generic_to_shared(hot) - STAGE_BYTES)
#define MBAR_S (STAGE_S - 128u)
    if (HAS_STAGE && tid == 0) {
        ctl.stage_phase = 0u;
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(MBAR_S) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid == 0) ctl.abort = 0u;

    #pragma unroll 1
    for (;;) {
        __syncthreads();
        if (group == 1) {
            if (tid == 0) {
                const u32 q = *(volatile u32*)abort_flag ? ASTRA_NONE32 : atomicAdd(&queue[1], 1u);
                ctl.point = q < n_points - n_big ? n_big + q : ASTRA_NONE32;
            }
            __syncthreads();
        } else {
            bar_target += group;
            if (!group_barrier(gc, bar_target, abort_flag, ctl)) break;     // everyone is done with the previous point's control block
            if (rank == 0 && tid == 0) {
                const u32 q = atomicAdd(&queue[0], 1u);
                gc->point = q < n_big ? q : ASTRA_NONE32;
                gc->acked = 0; gc->err = 0; gc->completion = 0;
                gc->hint[0] = gc->hint[1] = gc->hint[2] = ASTRA_T_INF;
            }
            bar_target += group;
            if (!group_barrier(gc, bar_target, abort_flag, ctl)) break;
            if (tid == 0) ctl.point = *(volatile u32*)&gc->point;
            __syncthreads();
        }
        const u32 qi = ctl.point;
        if (qi == ASTRA_NONE32) {
            if (group == 1) break;
            // no big point left: the CTAs of the group go on alone with the small ones
            group = 1; rank = 0;
            ws = ws_base + ws_single_off + (size_t)blockIdx.x * ws_single_stride;
            continue;
        }
        const u32 pi = order[qi];
        const PointDesc& P = points[pi];
        // The ten per-step constant tables are looked up on every delivery, issue and ack: where they fit (config 2: 4.5 KB,
        // config 4: <= 19 KB) one thread copies them to shared memory with TMA bulk copies and the point runs on the copies.
        const u32 stage_pad = (4u * P.S + 15u) & ~15u;
        const bool staged = HAS_STAGE && P.S > 0u && STAGE_TABLES * stage_pad <= STAGE_BYTES;
        if (tid == 0) {
            resolve_ctx(c, P, cblob, ws, hot, results, rank);
            if (staged) stage_tables(c, ctl, hot - STAGE_BYTES, stage_pad);
            ctl.acked = 0; ctl.completion = 0; ctl.err = 0;
            ctl.hint[0] = ctl.hint[1] = ctl.hint[2] = ASTRA_T_INF;
            for (int i = 0; i < 32; i++) { ctl.ls_acc[i] = 0u; ctl.ls_last[i] = 0u; }
            ctl.g_hint = ASTRA_T_INF; ctl.g_acked = 0; ctl.g_err = 0; ctl.g_completion = 0;
#ifdef ASTRA_DIAG
            #pragma unroll 1
            for (int i = 0; i < 16; i++) ctl.clk[i] = 0;
            #pragma unroll 1
            for (int i = 0; i < 128; i++) (&ctl.sclk[0][0])[i] = 0;
#endif
        }
#ifdef ASTRA_DIAG
        long long dck = clock64();
#endif
        __syncthreads();
        if (staged) mbar_wait(MBAR_S, ctl.stage_wait);                          // the tables have landed in shared memory
        // ---- state init: shared-memory arrays by their CTA, global arrays split over the group ----
        #pragma unroll 1
        for (u32 a = 0; a < ASTRA_A_COUNT; a++) {
            const u32 kind = k_arr_init[a];
            if (kind > 1) continue;
            const u64 off = P.a_off[a];
            const bool in_smem = (off & ASTRA_PLACE_SMEM) != 0;
            uint8_t* base = (in_smem ? hot : ws) + (off & ~(ASTRA_PLACE_SMEM | ASTRA_PLACE_LOCAL));
            const u32 pat = kind ? ~0u : 0u;
            const u64 n16 = P.a_bytes[a] / 16;              // arrays are padded to 16 bytes
            uint4* p = reinterpret_cast<uint4*>(base);
            const uint4 v4 = make_uint4(pat, pat, pat, pat);
            if (in_smem || group == 1) { for (u64 i = tid; i < n16; i += nthr) p[i] = v4; }
            else { for (u64 i = (u64)rank * nthr + tid; i < n16; i += (u64)group * nthr) p[i] = v4; }
        }
        if (group > 1) { bar_target += group; if (!group_barrier(gc, bar_target, abort_flag, ctl)) break; } else __syncthreads();
        #pragma unroll 1
        for (u32 e = c.e_lo + tid; e < c.e_hi; e += nthr) c.lstate0[e] = c.lstate0_init[e];
        #pragma unroll 1
        for (u32 s = tid; s < c.S; s += nthr) {
            const u32 ow = c.step_od[s] >> 16;
            if (ow < c.g_lo || ow >= c.g_hi) continue;
            c.ndep_left[s] = c.ndeps[s];
            // steps without deps are released at t = 0 (R10) -- unless the watchdog allows no cycle at all
            c.t_release[s] = (c.ndeps[s] || c.tmax == 0u) ? ASTRA_TS_NONE32 : 0u;
        }
        #pragma unroll 1
        for (u32 gq = c.g_lo; gq < c.g_hi; gq++) {
            #pragma unroll 1
            for (u32 j = c.rel_off[gq] + tid; j < c.rel_off[gq + 1]; j += nthr) c.plist[j] = c.init_rel[j];
            #pragma unroll 1
            for (u32 wf = tid; wf < c.CW; wf += nthr) c.wf_cur[(size_t)gq * c.CW + wf] = c.cul_ptr[gq * c.C + wf / c.Wv];
            #pragma unroll 1
            for (u32 wi = tid; wi < c.nwords; wi += nthr) {
                const u32 nb = c.CW - wi * 32;
                c.freeb[(size_t)gq * c.nwords + wi] = nb >= 32 ? ~0u : ((1u << nb) - 1u);
            }
            if (tid == 0) c.pcnt[gq] = c.init_rel_cnt[gq];
        }
        if (group > 1) { bar_target += group; if (!group_barrier(gc, bar_target, abort_flag, ctl)) break; } else __syncthreads();
#ifdef ASTRA_DIAG
        if (tid == 0) ctl.clk[5] = (u64)(clock64() - dck);
#endif

        // ---- warp sets: the CTA's nodes are dealt round robin to nsets sets of ws warps each ----
        const u32 n_nodes = c.v_hi - c.v_lo;
        const u32 nsets = max(1u, min(n_nodes, nwarps));
        const u32 wset = nwarps / nsets;                   // warps per set (left-over warps idle through the window)
        const u32 set = warp / wset, sw = warp % wset;
        const bool in_set = set < nsets;

        // ---- window loop ----
        u32 k = 0, seq = 0;
        int32_t status = ASTRA_STATUS_DONE;
        const u32 W = c.W;
        u64 busy = 0, skipped = 0;
        bool aborted = false;
        // Run-ahead windows (ASTRA_FLAG_RUN_AHEAD; off by default, see include/astra.h).  Inside a window a node depends on nothing; between windows only on the nodes that feed
        // its in-links and that receive its lines (predmask).  So there is no barrier per window: a node whose own
        // pending events fall into the next window knows that window is the next one for everybody and starts it as
        // soon as its predecessors have completed the current one (and every node the one before: buffers are sized
        // for a distance of two windows).  A node without such an event waits for all nodes and takes the point's
        // hint, as the barrier version does.  All nodes step through the same sequence of windows.
        const bool run_ahead = P.run_ahead != 0u && group == 1u && nsets == n_nodes && n_nodes > 1u && n_nodes <= 32u;
        if (run_ahead) {
            if (tid < 32) ctl.prog[tid] = 0u;
            if (tid < 8) ctl.hint8[tid] = ASTRA_T_INF;
            if (tid == 0) ctl.stop = 0u;
            __syncthreads();
            if (in_set) {
                const u32 pm = c.predmask[c.v_lo + set];
                const u32 allm = n_nodes == 32u ? ~0u : (1u << n_nodes) - 1u;
                const bool leader = sw == 0 && lane == 0;
                u32 n = 0;                                  // ordinal of the window in the sequence all nodes step through
#pragma unroll 1
                for (;;) {
                    const u64 t0l = (u64)k * W;
                    if (t0l >= c.tmax) { if (leader) atomicCAS(&ctl.stop, 0u, 1u + (u32)ASTRA_STATUS_MAX_CYCLES); break; }
                    const u32 t0 = (u32)t0l;
                    const u32 t1 = (u32)min((u64)c.tmax, t0l + W);
                    const u32 cb = t0 % c.NC;
                    u32* const hp = &ctl.shint[set][n & 1u];
#ifdef ASTRA_DIAG
                    dck = clock64();
#endif
                    if (n > 0 && wait_prog(ctl, lane, n_nodes, pm, n, allm, n - 1u)) break;
#ifdef ASTRA_DIAG
                    if (leader) ctl.sclk[set][7] += (u64)(clock64() - dck);
#endif
                    if (leader) *hp = ASTRA_T_INF;
                    set_sync(wset, set);
                    busy += t1 - t0;
                    node_window(c, ctl, hp, c.v_lo + set, k, t0, t1, cb, scr, lane, sw, wset, set, leader);
                    set_sync(wset, set);
                    const u32 own = *(volatile u32*)hp;
                    if (leader) {
                        atomicMin(&ctl.hint8[n & 7u], own);
                        ctl.hint8[(n + 4u) & 7u] = ASTRA_T_INF;  // last read before anybody started window n - 2, next written after n + 3
                        __threadfence_block();
                        *(volatile u32*)&ctl.prog[set] = n + 1u;
#ifdef ASTRA_DIAG
                        if (set == 0) ctl.clk[0]++;
#endif
                    }
                    const bool last = (u64)(k + 1) * W >= c.tmax;
                    if (!last && own / W <= k + 1u) { k++; n++; continue; }      // the next window is k + 1 for everybody
                    // the point's decision after this window, from what all nodes have posted
#ifdef ASTRA_DIAG
                    dck = clock64();
#endif
                    if (wait_prog(ctl, lane, n_nodes, 0u, 0u, allm, n + 1u)) break;
#ifdef ASTRA_DIAG
                    if (leader) ctl.sclk[set][7] += (u64)(clock64() - dck);
#endif
                    const u32 hint = *(volatile u32*)&ctl.hint8[n & 7u];
                    int32_t st = -1;
                    if (*(volatile u32*)&ctl.acked == c.S) st = ASTRA_STATUS_DONE;
                    else if (*(volatile u32*)&ctl.err) st = ASTRA_STATUS_INTERNAL;
                    else if (last) st = ASTRA_STATUS_MAX_CYCLES;       // events past the watchdog cut are not looked at
                    else if (hint == ASTRA_T_INF) st = ASTRA_STATUS_DEADLOCK;
                    if (st >= 0) { if (leader) atomicCAS(&ctl.stop, 0u, 1u + (u32)st); break; }
                    u32 nk = k + 1;
                    if (!(c.flags & (u32)ASTRA_FLAG_NO_WINDOW_SKIP)) nk = max(nk, hint / W);
                    skipped += (u64)(nk - k - 1) * W;
                    k = nk; n++;
                }
            }
            __syncthreads();
            status = (int32_t)ctl.stop - 1;
        } else
        #pragma unroll 1
        for (;;) {
            const u64 t0l = (u64)k * W;
            if (t0l >= c.tmax) { status = ASTRA_STATUS_MAX_CYCLES; break; }
            const u32 t0 = (u32)t0l;
            const u32 t1 = (u32)min((u64)c.tmax, t0l + W);
            const u32 cb = t0 % c.NC;
            u32* const hp = &ctl.hint[seq % 3];
            busy += t1 - t0;
            if (in_set)
#pragma unroll 1
                for (u32 j = set; j < n_nodes; j += nsets)
                    node_window(c, ctl, hp, c.v_lo + j, k, t0, t1, cb, scr, lane, sw, wset, set, sw == 0 && lane == 0);
            // ---- stage 5: next non-idle window (A7), one block barrier per window ----
#ifdef ASTRA_DIAG
            dck = clock64();
#endif
            u32 hint, acked_total, err;
            if (group > 1) {
                __syncthreads();
                if (tid == 0) {
                    atomicMin(&gc->hint[seq % 3], *hp);
                    if (ctl.acked) { atomicAdd(&gc->acked, ctl.acked); atomicMax(&gc->completion, ctl.completion); ctl.acked = 0; }
                    if (ctl.err) atomicOr(&gc->err, ctl.err);
                    if (rank == 0) gc->hint[(seq + 1) % 3] = ASTRA_T_INF;
                    ctl.hint[(seq + 2) % 3] = ASTRA_T_INF;
                }
                bar_target += group;
                if (!group_barrier(gc, bar_target, abort_flag, ctl)) { aborted = true; break; }
                if (tid == 0) {
                    ctl.g_hint = *(volatile u32*)&gc->hint[seq % 3];
                    ctl.g_acked = *(volatile u32*)&gc->acked;
                    ctl.g_err = *(volatile u32*)&gc->err;
                    ctl.g_completion = *(volatile u32*)&gc->completion;
                }
                __syncthreads();
                hint = ctl.g_hint; acked_total = ctl.g_acked; err = ctl.g_err;
            } else {
                __syncthreads();
                hint = *hp; acked_total = ctl.acked; err = ctl.err;
                // slot (seq + 2) % 3 was last read before this barrier and is next written after the next one
                if (tid == 0) ctl.hint[(seq + 2) % 3] = ASTRA_T_INF;
            }
#ifdef ASTRA_DIAG
            if (in_set && sw == 0 && lane == 0) ctl.sclk[set][7] += (u64)(clock64() - dck);
            if (tid == 0) ctl.clk[0]++;
#endif
            seq++;
            // every thread takes the same decision from the same values
            if (acked_total == c.S) { status = ASTRA_STATUS_DONE; break; }
            if (err) { status = ASTRA_STATUS_INTERNAL; break; }
            if ((u64)(k + 1) * W >= c.tmax) { status = ASTRA_STATUS_MAX_CYCLES; break; }   // events past the watchdog cut are not looked at
            if (hint == ASTRA_T_INF) { status = ASTRA_STATUS_DEADLOCK; break; }
            u32 nk = k + 1;
            if (!(c.flags & (u32)ASTRA_FLAG_NO_WINDOW_SKIP)) nk = max(nk, hint / W);
            skipped += (u64)(nk - k - 1) * W;
            k = nk;
        }
        if (aborted) break;
        __syncthreads();
        // ---- A8: write-out (each CTA the steps / links of its own nodes) ----
        u32 cmax = 0;                                       // completion = max t_ack over fully acked steps (R14)
        #pragma unroll 1
        for (u32 s = tid; s < c.S; s += nthr) {
            const u32 n = c.lines[s];
            const u32 od = c.step_od[s];
            const u32 ow = od >> 16, ds = od & 0xffffu;
            if (ow >= c.g_lo && ow < c.g_hi) {
                const u32 a = c.t_release[s];
                c.r_step_ts[4 * (size_t)s + 0] = a == ASTRA_TS_NONE32 ? ~0ull : a;
                c.r_step_ts[4 * (size_t)s + 1] = c.issued_cnt[s] == n ? (u64)c.t_issued[s] : ~0ull;
                const bool acked = c.ack_cnt[s] == n;
                c.r_step_ts[4 * (size_t)s + 3] = acked ? (u64)c.t_ack[s] : ~0ull;
                if (acked) cmax = max(cmax, c.t_ack[s]);
            }
            if (ds >= c.g_lo && ds < c.g_hi)
                c.r_step_ts[4 * (size_t)s + 2] = c.deliv_cnt[s] == n ? (u64)c.t_deliv[s] : ~0ull;
        }
        #pragma unroll 1
        for (u32 e = c.e_lo + tid; e < c.e_hi; e += nthr) c.r_link_lines[e] = c.link_lines[e];
        cmax = __reduce_max_sync(FULL, cmax);
        if (tid == 0) ctl.completion = 0;
        __syncthreads();
        if (lane == 0 && cmax) atomicMax(&ctl.completion, cmax);
        __syncthreads();
        if (group > 1) {
            if (tid == 0) { gc->completion = 0; }
            bar_target += group; if (!group_barrier(gc, bar_target, abort_flag, ctl)) break;
            if (tid == 0) atomicMax(&gc->completion, ctl.completion);
            bar_target += group; if (!group_barrier(gc, bar_target, abort_flag, ctl)) break;
            if (tid == 0) ctl.completion = *(volatile u32*)&gc->completion;
            __syncthreads();
        }
        if (tid == 0 && rank == 0) {
            DeviceSummary sm;
            sm.status = status; sm.n_steps = c.S; sm.n_links = c.E; sm.window = W;
            sm.completion_cycle = ctl.completion; sm.total_lines = P.total_lines;
            sm.busy_cycles = busy; sm.skipped_cycles = skipped;
            *c.r_summary = sm;
        }
#ifdef ASTRA_DIAG
        __syncthreads();
        if (tid < 16) c.r_diag[(size_t)rank * ASTRA_DIAG_WORDS + tid] = ctl.clk[tid];
        if (tid < 128) c.r_diag[(size_t)rank * ASTRA_DIAG_WORDS + 16 + tid] = (&ctl.sclk[0][0])[tid];
#endif
    }
}

// The step kernel: 128 registers per thread; 16 warps per CTA and one CTA per SM unless ASTRA_FLAG_WARPS says otherwise.
extern "C" __global__ void __launch_bounds__(512, 1)
astra_step_kernel(const uint8_t* __restrict__ cblob, uint8_t* __restrict__ ws_base, uint8_t* __restrict__ results,
                  const PointDesc* __restrict__ points, const u32* __restrict__ order, u32* queue,
                  GroupCtl* groups, u32 n_points, u32 n_big, u32 n_slots, u32 group0,
                  u64 ws_big_stride, u64 ws_single_off, u64 ws_single_stride, u32 hot_off) {
    step_kernel_body(cblob, ws_base, results, points, order, queue, groups, n_points, n_big, n_slots, group0,
                     ws_big_stride, ws_single_off, ws_single_stride, hot_off);
}
// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
bool astra_engine_has_diag() {
#ifdef ASTRA_DIAG
    return true;
#else
    return false;
#endif
}

bool astra_engine_stageable(u32 warps, u32 n_steps) {
    return warps == 16 && n_steps > 0 && (u64)STAGE_TABLES * ((4ull * n_steps + 15) & ~15ull) <= STAGE_BYTES;
}

u32 astra_engine_fixed_smem(u32 warps, bool stage) {
    size_t s = ((sizeof(Ctx) + 15) & ~size_t(15)) + ((sizeof(Ctl) + 15) & ~size_t(15)) + (size_t)warps * SCR_WORDS * sizeof(u32);
    s = (s + 127) & ~size_t(127);
    if (stage && warps == 16) s += 128 + STAGE_BYTES;        // mbarrier + staging area of the per-step constant tables, right below the hot region
    return (u32)s;
}

static const void* kernel_variant(u32) { return (const void*)astra_step_kernel; }

int32_t astra_engine_occupancy(u32 warps_per_cta, u32 hot_bytes, u32 variant, bool stage, u32* ctas_per_sm, u32* n_sms, std::string& err) {
    int dev = 0, sms = 0, occ = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    size_t sm = (size_t)astra_engine_fixed_smem(warps_per_cta, stage) + hot_bytes;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kernel_variant(variant), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel_variant(variant), (int)warps_per_cta * 32, sm);
    if (e != cudaSuccess) { err = std::string("occupancy query: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    *ctas_per_sm = (u32)occ; *n_sms = (u32)sms;
    return ASTRA_OK;
}

int32_t astra_engine_launch(const EngineLaunch& L, void* stream, std::string& err) {
    const u32 fixed = astra_engine_fixed_smem(L.warps_per_cta, L.stage);
    size_t sm = (size_t)fixed + L.hot_bytes;
    cudaError_t e = cudaFuncSetAttribute(kernel_variant(L.variant), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) { err = std::string("smem attribute: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    e = cudaMemsetAsync(L.d_queue, 0, 4 * sizeof(u32), (cudaStream_t)stream);
    if (e == cudaSuccess && L.n_slots) e = cudaMemsetAsync(L.d_groups, 0, sizeof(GroupCtl) * L.n_slots, (cudaStream_t)stream);
    if (e != cudaSuccess) { err = std::string("queue reset: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    // Cooperative launch: the CTAs of a group spin on each other, so the whole grid must be co-resident.
    // The runtime guarantees that or refuses the launch (cudaErrorCooperativeLaunchTooLarge) -- never a hang.
    const uint8_t* a0 = L.d_const; uint8_t* a1 = L.d_ws; uint8_t* a2 = L.d_results; const PointDesc* a3 = L.d_points;
    const u32* a4 = L.d_order; u32* a5 = L.d_queue; GroupCtl* a6 = L.d_groups;
    u32 a7 = L.n_points, a8 = L.n_big, a9 = L.n_slots, a10 = L.group;
    u64 a11 = L.ws_big_stride, a12 = L.ws_single_off, a13 = L.ws_single_stride; u32 a14 = fixed;
    void* args[] = {&a0, &a1, &a2, &a3, &a4, &a5, &a6, &a7, &a8, &a9, &a10, &a11, &a12, &a13, &a14};
    e = cudaLaunchCooperativeKernel(kernel_variant(L.variant), dim3(L.grid), dim3(L.warps_per_cta * 32), args, sm,
                                    (cudaStream_t)stream);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        err = std::string("cooperative kernel launch: ") + cudaGetErrorString(e);
        return e == cudaErrorCooperativeLaunchTooLarge ? ASTRA_ELIMIT : ASTRA_ECUDA;
    }
    return ASTRA_OK;
}


// ---------------------------------------------------------------------------------------------
// No-allocation path (include/astra.h: astra_run_packed_noalloc).  The scratch of one single-CTA
// design point -- queue header + the CTA's workspace -- lives in this file-scope array instead of
// a cudaMalloc'ed buffer.  In host code the array's name is only a stand-in: its device address
// is resolved once per device with cudaGetSymbolAddress (that device current) and handed to the
// kernel as its workspace pointer.  Every call on a device shares the array.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char astra_noalloc_scratch[ASTRA_NOALLOC_SCRATCH_BYTES];

#define ASTRA_NOALLOC_MAX_DEVICES 64
static uint8_t* g_noalloc_ptr[ASTRA_NOALLOC_MAX_DEVICES];     // device address of the array, per device (nullptr: not resolved yet)

int32_t astra_engine_static_scratch(int device, uint8_t** ptr, std::string& err) {
    if (device < 0 || device >= ASTRA_NOALLOC_MAX_DEVICES) { err = "device index beyond the static-scratch table"; return ASTRA_ELIMIT; }
    if (!g_noalloc_ptr[device]) {
        int cur = -1;
        cudaError_t e = cudaGetDevice(&cur);
        if (e == cudaSuccess && cur != device) { err = "static scratch: the device is not current"; return ASTRA_ESTATE; }
        void* p = nullptr;
        if (e == cudaSuccess) e = cudaGetSymbolAddress(&p, astra_noalloc_scratch);
        if (e != cudaSuccess || !p) { (void)cudaGetLastError(); err = std::string("cudaGetSymbolAddress(static scratch): ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
        // the kernel's shared-memory opt-in is set here too, so that the run itself only clears and launches
        e = cudaFuncSetAttribute((const void*)astra_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)(astra_engine_fixed_smem(16, true) + ASTRA_HOT_BUDGET_SINGLE));
        if (e != cudaSuccess) { (void)cudaGetLastError(); err = std::string("smem attribute: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
        g_noalloc_ptr[device] = (uint8_t*)p;
    }
    *ptr = g_noalloc_ptr[device];
    return ASTRA_OK;
}

// One design point on one CTA: [0, 16) of the array = queue counters + abort flag, [256, 256 + sizeof(GroupCtl)) an
// (unused) group block, [ASTRA_NOALLOC_HEADER_BYTES, ...) the CTA's workspace.  The header must start at zero.
int32_t astra_engine_launch_noalloc(int device, const uint8_t* d_const, const PointDesc* d_point, const u32* d_order,
                                    uint8_t* d_results, u64 ws_bytes, u32 warps_per_cta, u32 hot_bytes, u32 n_steps, void* stream, std::string& err) {
    if ((u64)ASTRA_NOALLOC_HEADER_BYTES + ws_bytes > ASTRA_NOALLOC_SCRATCH_BYTES) { err = "scratch exceeds the static scratch array"; return ASTRA_ELIMIT; }
    if (hot_bytes > ASTRA_HOT_BUDGET_SINGLE || warps_per_cta != 16) { err = "packed point was planned for another CTA shape"; return ASTRA_EINVAL; }
    uint8_t* scratch = nullptr;
    int32_t rc = astra_engine_static_scratch(device, &scratch, err);
    if (rc) return rc;
    cudaError_t e = cudaMemsetAsync(scratch, 0, ASTRA_NOALLOC_HEADER_BYTES, (cudaStream_t)stream);
    if (e != cudaSuccess) { (void)cudaGetLastError(); err = std::string("scratch header clear: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    const u32 fixed = astra_engine_fixed_smem(warps_per_cta, astra_engine_stageable(warps_per_cta, n_steps));
    const size_t sm = (size_t)fixed + hot_bytes;
    // the other path sets this attribute to its own batch's size before each of its launches: set ours (no allocation)
    e = cudaFuncSetAttribute((const void*)astra_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) { (void)cudaGetLastError(); err = std::string("smem attribute: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    const uint8_t* a0 = d_const; uint8_t* a1 = scratch + ASTRA_NOALLOC_HEADER_BYTES; uint8_t* a2 = d_results; const PointDesc* a3 = d_point;
    const u32* a4 = d_order; u32* a5 = (u32*)scratch; GroupCtl* a6 = (GroupCtl*)(scratch + 256);
    u32 a7 = 1, a8 = 0, a9 = 0, a10 = 1;
    u64 a11 = 0, a12 = 0, a13 = (ws_bytes + 255) & ~255ull; u32 a14 = fixed;
    void* args[] = {&a0, &a1, &a2, &a3, &a4, &a5, &a6, &a7, &a8, &a9, &a10, &a11, &a12, &a13, &a14};
    e = cudaLaunchCooperativeKernel((const void*)astra_step_kernel, dim3(1), dim3(warps_per_cta * 32), args, sm, (cudaStream_t)stream);
    if (e != cudaSuccess) { (void)cudaGetLastError(); err = std::string("kernel launch: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    return ASTRA_OK;
}
