// astra_engine.cu -- the sm_100a step kernel of the cycle-synchronous cache-line simulator.
//
// Design.  The paper's simulator is an event-driven CPU program
// (PAPER.md:L19); this engine is organised around one structural fact instead: a line accepted
// by a link at cycle a cannot reach the next node before a + Leff, and an ack cannot reach its
// owner before t_deliv + alpha >= t_deliv + min Leff.  With W = 2^k <= min Leff, nothing a node
// does inside the window [kW, (k+1)W) can influence another node inside the same window.  So:
//
//   * one WARP advances one simulated node (GPU or switch) through a whole window, cycle by
//     cycle, touching only node-private state -- no barrier per cycle;
//   * nodes exchange data only through single-producer/single-consumer link pipes (ring buffers
//     of 64-bit flits tagged with their arrival cycle) and slot-addressed ack records with a
//     per-window discovery bitmap; both are read one window after they are written;
//   * one CTA barrier per window (not per cycle) separates producers from consumers;
//   * inside a node every per-cycle phase (R7 A1-A3, R9 B, R10 C, R12 D) is warp-parallel:
//     lanes are (link, k) candidates or wavefronts, same-cycle FIFO append order (R8) comes
//     from ballot/match ranks, never from atomics;
//   * idle cycles are skipped per node with a warp min-reduction over the next arrival, next
//     ack, next credit-sufficient cycle and "work pending".
//
// One CTA simulates one design point at a time and pulls the next from a cost-sorted queue.
#include "astra_internal.h"
#include "../../include/astra.h"

#include <cuda_runtime.h>

#define FULL 0xffffffffu

struct Ctx {   // resolved pointers of the point a CTA is running; lives in shared memory
    u32 G, V, E, S, C, Wv, K, H, CW, nwords, slots, bmwords, logW, W, NWmask, NW, kmagic, tmax;
    u64 fullmask;
    const u32 *row_ptr, *in_ptr, *in_link, *leff, *bw, *icand_ptr, *icand, *ocand_ptr, *ocand, *next_link;
    const u32 *step_od, *lines, *cu_lo, *cu_n, *succ_ptr, *succ, *ndeps;
    const u32 *step_q, *step_r, *first_link, *step_alpha, *cul_ptr, *cul, *rel_off, *init_rel, *init_rel_cnt;
    const u32 *fifo_off, *fifo_mask, *pipe_off, *pipe_mask, *credit_cap;
    u32 *fifo_head, *fifo_tail, *pipe_tail, *pipe_tail_pub, *pipe_head, *pipe_tsnap, *credit, *credit_time, *link_lines;
    u64 *fifo_buf, *pipe_buf;
    u32 *t_release, *issued_cnt, *t_issued, *deliv_cnt, *t_deliv, *ack_cnt, *t_ack, *ndep_left;
    u32 *wf_rem, *wf_cur; u64 *wf_busy;
    u32 *want, *freeb; u64 *pend; u32 *pend_link, *pend_cnt, *rel_list, *rel_cnt, *sel;
    u64 *ack_rec, *ack_tmp, *ack_sorted; u32 *bitmap, *bin_cnt; u32 flags;
    u32 *node_next; u64 *node_busy; u32 *node_acked;
    u64 *r_step_ts, *r_link_lines; DeviceSummary *r_summary;
};

struct Ctl {   // per-CTA control block in shared memory
    u32 point;          // index into the order array
    u32 acked;          // steps fully acked so far
    u32 completion;     // max t_ack
    u32 err;            // engine self-check flags
    u32 done;
    u32 next_hint;      // min over nodes of their next event time
    u32 decision;       // 0 = run window `next_k`, else 1 + status
    u32 next_k;
    u64 busy, skipped;
};

__device__ __forceinline__ u32 lane_id() { return threadIdx.x & 31; }
__device__ __forceinline__ u32 lanemask_lt() { u32 m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m; }
__device__ __forceinline__ u64 ldcg64(const u64* p) { return __ldcg((const unsigned long long*)p); }
__device__ __forceinline__ u32 ldcg32(const u32* p) { return __ldcg(p); }

__device__ __forceinline__ u32 warp_incl_scan(u32 v, u32 lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { u32 n = __shfl_up_sync(FULL, v, d); if (lane >= (u32)d) v += n; }
    return v;
}

// Append one flit per lane of `mask` to the FIFO of its out-link `eo`, in lane order (R8).
__device__ __forceinline__ void fifo_append(Ctx& c, u32 mask, bool act, u32 eo, u64 flit, u32& err) {
    u32 m = 0, rank = 0, base = 0;
    if (act) {
        m = __match_any_sync(mask, eo);
        rank = __popc(m & lanemask_lt());
        base = c.fifo_tail[eo];
        c.fifo_buf[c.fifo_off[eo] + ((base + rank) & c.fifo_mask[eo])] = flit;
    }
    __syncwarp();
    if (act && rank == 0) {
        u32 nt = base + __popc(m);
        if (nt - c.fifo_head[eo] > c.fifo_mask[eo] + 1) err |= 1u;     // ring overflow guard
        c.fifo_tail[eo] = nt;
    }
    __syncwarp();
}

// A step's timestamp of kind `kind` was stamped on node g: count down its successors (R3, R10).
// Called by the whole warp with a warp-uniform step p.  Newly ready steps join g's release list.
__device__ __forceinline__ void on_event(Ctx& c, u32 g, u32 p, u32 kind, u32 lane) {
    u32 lo = c.succ_ptr[p], hi = c.succ_ptr[p + 1];
    for (u32 b = lo; b < hi; b += 32) {
        u32 i = b + lane; bool ready = false; u32 s2 = 0;
        if (i < hi) {
            u32 sk = c.succ[i];
            if ((sk >> 30) == kind) {
                s2 = sk & 0xfffffu;
                u32 nd = c.ndep_left[s2] - 1; c.ndep_left[s2] = nd;
                ready = (nd == 0);
            }
        }
        u32 rm = __ballot_sync(FULL, ready);
        if (rm) {
            u32 cnt = c.rel_cnt[g];
            if (ready) c.rel_list[c.rel_off[g] + cnt + __popc(rm & lanemask_lt())] = s2;
            __syncwarp();
            if (lane == 0) c.rel_cnt[g] = cnt + __popc(rm);
        }
        __syncwarp();
    }
}

// Walk wavefront (g, wf)'s in-order list from `cur` to the first entry that is unreleased or has
// quota for it (R11).  Returns true when quota was loaded (the wavefront wants to issue).
__device__ __forceinline__ bool wf_advance(Ctx& c, u32 g, u32 wf, u32& cur, u32& rem) {
    u32 end = c.cul_ptr[g * c.C + wf / c.Wv + 1];
    rem = ASTRA_NOTLOADED;
    while (cur < end) {
        u32 s = c.cul[cur];
        if (c.t_release[s] == ASTRA_TS_NONE32) return false;
        u32 q = c.step_q[s] + (((wf - c.cu_lo[s] * c.Wv) < c.step_r[s]) ? 1u : 0u);
        if (q) { rem = q; return true; }
        cur++;
    }
    return false;
}

// Counting sort of this window's acks of GPU g by cycle (R6, R7 A3).  Returns their number.
__device__ u32 ack_prologue(Ctx& c, u32 g, u32 k, u32 t0, u32* scnt, u32 lane) {
    u32 bin = k & c.NWmask;
    u32 n = ldcg32(&c.bin_cnt[g * c.NW + bin]);
    if (n == 0) return 0;
    const u32 W = c.W;
    for (u32 i = lane; i <= W; i += 32) scnt[i] = 0;
    __syncwarp();
    u32* bm = c.bitmap + (size_t)(g * c.NW + bin) * c.bmwords;
    const u64* rec = c.ack_rec + (size_t)g * c.slots;
    u64* tmp = c.ack_tmp + (size_t)g * c.slots;
    u64* srt = c.ack_sorted + (size_t)g * c.slots;
    // pass 1: discover, histogram by cycle, compact into tmp
    u32 total = 0;
    for (u32 wb = 0; wb < c.bmwords; wb += 32) {
        u32 wi = wb + lane;
        u32 w = (wi < c.bmwords) ? ldcg32(&bm[wi]) : 0;
        if (w) bm[wi] = 0;
        u32 cnt = __popc(w);
        u32 incl = warp_incl_scan(cnt, lane);
        u32 pos = total + incl - cnt;
        total += __shfl_sync(FULL, incl, 31);
        while (w) {
            u32 b = __ffs(w) - 1; w &= w - 1;
            u32 idx = wi * 32 + b;
            u64 rc = ldcg64(&rec[idx]);
            u32 cyc = (u32)rc - t0;
            u32 wf = c.K == 1 ? idx : (u32)(((u64)idx * c.kmagic) >> 32);   // idx / K (magic overflows for K == 1)
            u32 slot = idx - wf * c.K;
            atomicAdd(&scnt[cyc], 1u);
            tmp[pos++] = (rc & 0xffffffff00000000ull) | (cyc << 18) | (wf << 6) | slot;
        }
    }
    __syncwarp();
    // exclusive scan of the histogram
    u32 carry = 0;
    for (u32 b = 0; b < W; b += 32) {
        u32 i = b + lane;
        u32 v = (i < W) ? scnt[i] : 0;
        u32 incl = warp_incl_scan(v, lane);
        if (i < W) scnt[i] = carry + incl - v;
        carry += __shfl_sync(FULL, incl, 31);
    }
    __syncwarp();
    // pass 2: scatter into cycle order
    for (u32 i = lane; i < total; i += 32) {
        u64 ent = tmp[i];
        u32 pos = atomicAdd(&scnt[(u32)ent >> 18], 1u);
        srt[pos] = ent;
    }
    if (lane == 0) c.bin_cnt[g * c.NW + bin] = 0;
    __syncwarp();
    return total;
}

// Minimum arrival time over the heads of v's in-link pipes (entries visible in this window).
__device__ u32 peek_arrivals(Ctx& c, u32 v, u32 tref, u32 lane) {
    u32 tn = ASTRA_T_INF;
    for (u32 i = c.in_ptr[v] + lane; i < c.in_ptr[v + 1]; i += 32) {
        u32 e = c.in_link[i];
        u32 head = c.pipe_head[e];
        if ((int32_t)(c.pipe_tsnap[e] - head) > 0) {
            u64 f = ldcg64(&c.pipe_buf[c.pipe_off[e] + (head & c.pipe_mask[e])]);
            u32 d = ((u32)(f >> ASTRA_FLIT_TIME_SHIFT) - tref) & ASTRA_TMASK26;
            tn = min(tn, tref + d);
        }
    }
    return __reduce_min_sync(FULL, tn);
}

// Advance node v through the window [t0, t1).  One warp.
__device__ void node_window(Ctx& c, Ctl& ctl, u32 v, u32 k, u32 t0, u32 t1, u32* scnt, u32 lane) {
    const bool isgpu = v < c.G;
    const u32 g = v;
    const u32 ic_lo = c.icand_ptr[v], ic_hi = c.icand_ptr[v + 1];
    const u32 oc_lo = c.ocand_ptr[v], oc_hi = c.ocand_ptr[v + 1];
    u32 err = 0;

    // ---- prologue: snapshot producer tails, sort this window's acks ----
    for (u32 i = c.in_ptr[v] + lane; i < c.in_ptr[v + 1]; i += 32) {
        u32 e = c.in_link[i];
        c.pipe_tsnap[e] = ldcg32(&c.pipe_tail_pub[e]);
    }
    __syncwarp();
    u32 ack_n = 0, ack_pos = 0;
    const u64* srt = c.ack_sorted + (size_t)g * c.slots;
    if (isgpu) ack_n = ack_prologue(c, g, k, t0, scnt, lane);
    u32 t_ack_next = ack_n ? t0 + ((u32)srt[0] >> 18) : ASTRA_T_INF;
    u32 t_arr_next = peek_arrivals(c, v, t0, lane);
    u32 t_local = c.node_next[v];                 // work pending from the previous window
    u32 t = min(min(t_arr_next, t_ack_next), max(t_local, t0));
    u32 stepped = 0, acked_steps = 0, completion = 0;
    u32 t_last = t0;
    u32 local_next = ASTRA_T_INF;
    u32 push_hint = ASTRA_T_INF;      // earliest arrival / ack this node created for others

    while (t < t1) {
        stepped++;
        t_last = t;
        u32 t_link_next = ASTRA_T_INF;
        bool more = false;          // something forces a visit at t + 1

        // ================= phase A1: arrivals (R7) =================
        if (t_arr_next == t) {
            u32 tn = ASTRA_T_INF;
            for (u32 cb = ic_lo; cb < ic_hi; cb += 32) {
                u32 j = cb + lane;
                u32 pk = (j < ic_hi) ? c.icand[j] : ASTRA_CAND_PAD;
                bool act = pk != ASTRA_CAND_PAD;
                u32 e = pk >> 10, ceilb = (pk >> 5) & 31, kk = pk & 31;
                bool valid = false, due = false; u64 flit = 0; u32 head = 0;
                if (act) {
                    head = c.pipe_head[e];
                    u32 idx = head + kk;
                    valid = (int32_t)(c.pipe_tsnap[e] - idx) > 0;
                    if (valid) {
                        flit = ldcg64(&c.pipe_buf[c.pipe_off[e] + (idx & c.pipe_mask[e])]);
                        u32 d = ((u32)(flit >> ASTRA_FLIT_TIME_SHIFT) - t) & ASTRA_TMASK26;
                        due = (d == 0);
                        if (!due) tn = min(tn, t + d);
                    }
                }
                u32 duemask = __ballot_sync(FULL, due);
                if (duemask == 0) continue;
                // pops per link: the k == 0 lane of each block advances the head
                if (act && kk == 0) {
                    u32 blk = ((2u << ceilb) - 1u) << lane;       // lanes [lane, lane + ceilb]
                    u32 npop = __popc(duemask & blk);
                    if (npop) c.pipe_head[e] = head + npop;
                }
                u32 step = (u32)flit & 0xfffffu;
                u32 od = due ? c.step_od[step] : 0;
                u32 dstg = od & 0xffffu;
                bool deliver = due && dstg == v;
                bool transit = due && !deliver;
                u32 tmask = __ballot_sync(FULL, transit);
                u32 dmask = __ballot_sync(FULL, deliver);
                if (tmask) {
                    u32 eo = transit ? c.next_link[v * c.G + dstg] : 0;
                    fifo_append(c, tmask, transit, eo, flit, err);
                }
                if (dmask) {
                    bool completed = false;
                    if (deliver) {
                        u32 owner = od >> 16;
                        u32 wf = ((u32)flit >> 20) & 0xfffu, slot = (u32)(flit >> 32) & 63u;
                        u32 ta = t + c.step_alpha[step];
                        push_hint = min(push_hint, ta);
                        u32 bit = wf * c.K + slot;
                        c.ack_rec[(size_t)owner * c.slots + bit] = ((u64)step << 32) | ta;
                        u32 bin = (ta >> c.logW) & c.NWmask;
                        atomicOr(&c.bitmap[(size_t)(owner * c.NW + bin) * c.bmwords + (bit >> 5)], 1u << (bit & 31));
                        atomicAdd(&c.bin_cnt[owner * c.NW + bin], 1u);
                        u32 m = __match_any_sync(dmask, step);
                        if ((m & lanemask_lt()) == 0) {
                            u32 dc = c.deliv_cnt[step] + __popc(m);
                            c.deliv_cnt[step] = dc;
                            if (dc == c.lines[step]) { c.t_deliv[step] = t; completed = true; }
                        }
                    }
                    u32 cm = __ballot_sync(FULL, completed);
                    while (cm) {
                        u32 src = __ffs(cm) - 1; cm &= cm - 1;
                        u32 p = __shfl_sync(FULL, step, src);
                        on_event(c, g, p, ASTRA_DEP_DELIVERED, lane);
                    }
                }
            }
            __syncwarp();
            t_arr_next = __reduce_min_sync(FULL, tn);
        }

        // ================= phase A2: inject lines issued at t-1 (R7) =================
        if (isgpu) {
            u32 np = c.pend_cnt[g];
            if (np) {
                for (u32 b = 0; b < np; b += 32) {
                    u32 j = b + lane; bool act = j < np;
                    u64 flit = act ? c.pend[(size_t)g * c.H + j] : 0;
                    u32 eo = act ? c.pend_link[(size_t)g * c.H + j] : 0;
                    u32 amask = __ballot_sync(FULL, act);
                    fifo_append(c, amask, act, eo, flit, err);
                }
                if (lane == 0) c.pend_cnt[g] = 0;
                __syncwarp();
            }
        }

        // ================= phase A3: acks due at t (R6, R7) =================
        if (t_ack_next == t) {
            const u32 cyc = t - t0;
            while (ack_pos < ack_n) {
                u32 j = ack_pos + lane;
                u64 ent64 = (j < ack_n) ? srt[j] : ~0ull;
                u32 ent = (u32)ent64;
                bool now = (j < ack_n) && (ent >> 18) == cyc;
                u32 nm = __ballot_sync(FULL, now);
                if (nm == 0) break;
                bool completed = false; u32 step = 0;
                if (now) {
                    u32 wf = (ent >> 6) & 0xfffu, slot = ent & 63u;
                    step = (u32)(ent64 >> 32);
                    // return the slot (several acks of one wavefront may land in the same cycle)
                    u32 mw = __match_any_sync(nm, wf);
                    u32 lo = __reduce_or_sync(mw, slot < 32 ? (1u << slot) : 0u);
                    u32 hi = __reduce_or_sync(mw, slot >= 32 ? (1u << (slot - 32)) : 0u);
                    if ((mw & lanemask_lt()) == 0) {
                        u64 busy = c.wf_busy[(size_t)g * c.CW + wf];
                        busy &= ~(((u64)hi << 32) | lo);
                        c.wf_busy[(size_t)g * c.CW + wf] = busy;
                    }
                    // its free bit
                    u32 wi = wf >> 5;
                    u32 mi = __match_any_sync(nm, wi);
                    u32 bits = __reduce_or_sync(mi, 1u << (wf & 31));
                    if ((mi & lanemask_lt()) == 0) c.freeb[g * c.nwords + wi] |= bits;
                    // ack count of the step
                    u32 ms = __match_any_sync(nm, step);
                    if ((ms & lanemask_lt()) == 0) {
                        u32 ac = c.ack_cnt[step] + __popc(ms);
                        c.ack_cnt[step] = ac;
                        if (ac == c.lines[step]) { c.t_ack[step] = t; completed = true; }
                    }
                }
                u32 cm = __ballot_sync(FULL, completed);
                if (cm) {
                    acked_steps += __popc(cm);
                    completion = t;
                    while (cm) {
                        u32 src = __ffs(cm) - 1; cm &= cm - 1;
                        u32 p = __shfl_sync(FULL, step, src);
                        on_event(c, g, p, ASTRA_DEP_ACKED, lane);
                    }
                }
                ack_pos += __popc(nm);
                if (__popc(nm) < 32) break;
            }
            __syncwarp();
            t_ack_next = (ack_pos < ack_n) ? t0 + ((u32)srt[ack_pos] >> 18) : ASTRA_T_INF;
        }

        // ================= phase B: link acceptance (R9) =================
        for (u32 cb = oc_lo; cb < oc_hi; cb += 32) {
            u32 j = cb + lane;
            u32 pk = (j < oc_hi) ? c.ocand[j] : ASTRA_CAND_PAD;
            bool act = pk != ASTRA_CAND_PAD;
            u32 e = pk >> 10, ceilb = (pk >> 5) & 31, kk = pk & 31;
            u32 nacc = 0, head = 0, ptail = 0, tl = ASTRA_T_INF;
            if (act && kk == 0) {
                head = c.fifo_head[e];
                u32 len = c.fifo_tail[e] - head;
                if (len) {
                    u32 bw = c.bw[e], cap = ceilb << 8;
                    u64 cr = (u64)c.credit[e] + (u64)(t - c.credit_time[e]) * bw;
                    if (cr > cap) cr = cap;
                    nacc = min((u32)cr >> 8, len);
                    u32 crn = (u32)cr - (nacc << 8);
                    c.credit[e] = crn; c.credit_time[e] = t;
                    ptail = c.pipe_tail[e];
                    if (nacc) {
                        c.fifo_head[e] = head + nacc;
                        c.pipe_tail[e] = ptail + nacc;
                        c.link_lines[e] += nacc;
                        push_hint = min(push_hint, t + c.leff[e]);
                    }
                    if (len > nacc) tl = (crn + bw >= 256u) ? t + 1 : t + (256u - crn + bw - 1) / bw;
                }
            }
            u32 src = lane - kk;
            nacc = __shfl_sync(FULL, nacc, src & 31);
            head = __shfl_sync(FULL, head, src & 31);
            ptail = __shfl_sync(FULL, ptail, src & 31);
            if (act && kk < nacc) {
                u64 flit = c.fifo_buf[c.fifo_off[e] + ((head + kk) & c.fifo_mask[e])];
                flit = (flit & ((1ull << ASTRA_FLIT_TIME_SHIFT) - 1)) |
                       ((u64)((t + c.leff[e]) & ASTRA_TMASK26) << ASTRA_FLIT_TIME_SHIFT);
                c.pipe_buf[c.pipe_off[e] + ((ptail + kk) & c.pipe_mask[e])] = flit;
            }
            t_link_next = min(t_link_next, tl);
        }
        __syncwarp();
        t_link_next = __reduce_min_sync(FULL, t_link_next);

        if (isgpu) {
            // ================= phase C: DAG release (R10) =================
            u32 nr = c.rel_cnt[g];
            if (nr) {
                const u32* rl = c.rel_list + c.rel_off[g];
                for (u32 i = lane; i < nr; i += 32) c.t_release[rl[i]] = t;
                __syncwarp();
                for (u32 i = 0; i < nr; i++) {
                    u32 s = rl[i];
                    u32 lo = c.cu_lo[s] * c.Wv, hi = lo + c.cu_n[s] * c.Wv;
                    for (u32 wb = lo & ~31u; wb < hi; wb += 32) {
                        u32 wf = wb + lane;
                        bool setw = false;
                        if (wf >= lo && wf < hi) {
                            size_t gw = (size_t)g * c.CW + wf;
                            u32 cur = c.wf_cur[gw];
                            if (c.wf_rem[gw] == ASTRA_NOTLOADED && cur < c.cul_ptr[g * c.C + wf / c.Wv + 1] && c.cul[cur] == s) {
                                u32 rem;
                                setw = wf_advance(c, g, wf, cur, rem);
                                c.wf_cur[gw] = cur; c.wf_rem[gw] = rem;
                            }
                        }
                        u32 bits = __ballot_sync(FULL, setw);
                        if (bits && lane == 0) c.want[g * c.nwords + (wb >> 5)] |= bits;
                    }
                }
                if (lane == 0) c.rel_cnt[g] = 0;
                __syncwarp();
            }

            // ================= phase D: issue (R11-R13) =================
            u32 budget = c.H, nsel = 0;
            u32* sel = c.sel + (size_t)g * c.H;
            for (u32 wb = 0; wb < c.nwords && budget; wb += 32) {
                u32 wi = wb + lane;
                u32 r = (wi < c.nwords) ? (c.want[g * c.nwords + wi] & c.freeb[g * c.nwords + wi]) : 0;
                u32 cnt = __popc(r);
                u32 incl = warp_incl_scan(cnt, lane);
                u32 tot = __shfl_sync(FULL, incl, 31);
                if (tot == 0) continue;
                u32 excl = incl - cnt;
                u32 take = excl >= budget ? 0 : min(cnt, budget - excl);
                for (u32 i = 0; i < take; i++) {
                    u32 b = __ffs(r) - 1; r &= r - 1;
                    sel[nsel + excl + i] = wi * 32 + b;
                }
                u32 got = min(tot, budget);
                nsel += got; budget -= got;
            }
            __syncwarp();
            for (u32 b = 0; b < nsel; b += 32) {
                u32 j = b + lane; bool act = j < nsel;
                u32 wf = 0, s = 0; bool full = false, keepw = true;
                if (act) {
                    wf = sel[j];
                    size_t gw = (size_t)g * c.CW + wf;
                    u32 cur = c.wf_cur[gw];
                    s = c.cul[cur];
                    u32 rem = c.wf_rem[gw] - 1;
                    u64 busy = c.wf_busy[gw];
                    u32 slot = __ffsll((long long)~busy) - 1;
                    busy |= 1ull << slot;
                    c.wf_busy[gw] = busy;
                    full = (busy == c.fullmask);
                    c.pend[(size_t)g * c.H + j] = (u64)s | ((u64)wf << 20) | ((u64)slot << 32);
                    c.pend_link[(size_t)g * c.H + j] = c.first_link[s];
                    if (rem == 0) { cur++; keepw = wf_advance(c, g, wf, cur, rem); c.wf_cur[gw] = cur; }
                    c.wf_rem[gw] = rem;
                }
                u32 amask = __ballot_sync(FULL, act);
                bool completed = false;
                if (act) {
                    u32 ms = __match_any_sync(amask, s);
                    if ((ms & lanemask_lt()) == 0) {
                        u32 ic = c.issued_cnt[s] + __popc(ms);
                        c.issued_cnt[s] = ic;
                        if (ic == c.lines[s]) { c.t_issued[s] = t; completed = true; }
                    }
                    u32 wi = wf >> 5;
                    u32 mi = __match_any_sync(amask, wi);
                    u32 clrf = __reduce_or_sync(mi, full ? (1u << (wf & 31)) : 0u);
                    u32 clrw = __reduce_or_sync(mi, keepw ? 0u : (1u << (wf & 31)));
                    if ((mi & lanemask_lt()) == 0) {
                        if (clrf) c.freeb[g * c.nwords + wi] &= ~clrf;
                        if (clrw) c.want[g * c.nwords + wi] &= ~clrw;
                    }
                }
                u32 cm = __ballot_sync(FULL, completed);
                while (cm) {
                    u32 src = __ffs(cm) - 1; cm &= cm - 1;
                    u32 p = __shfl_sync(FULL, s, src);
                    on_event(c, g, p, ASTRA_DEP_ISSUED, lane);      // released at t + 1 (R10)
                }
            }
            if (nsel) { if (lane == 0) c.pend_cnt[g] = nsel; more = true; }
            __syncwarp();
            if (c.rel_cnt[g]) more = true;
            if (!more) {
                u32 any = 0;
                for (u32 wi = lane; wi < c.nwords; wi += 32) any |= c.want[g * c.nwords + wi] & c.freeb[g * c.nwords + wi];
                if (__ballot_sync(FULL, any != 0)) more = true;
            }
        }

        // ================= next non-idle cycle of this node (A7) =================
        u32 tn = min(min(t_arr_next, t_ack_next), t_link_next);
        if (more) tn = min(tn, t + 1);
        local_next = more ? t + 1 : t_link_next;
        t = tn;
    }

    // ---- epilogue: publish producer tails, carry local work over, account ----
    for (u32 i = c.row_ptr[v] + lane; i < c.row_ptr[v + 1]; i += 32) c.pipe_tail_pub[i] = c.pipe_tail[i];
    // hint for window skipping: the earliest thing this node knows about -- its own pending work,
    // visible arrivals, what it pushed to others, and acks waiting in its future bins
    u32 hint = min(min(t_arr_next, t_ack_next), push_hint);
    if (isgpu) {
        for (u32 j = lane; j < c.NW; j += 32) {
            u32 w = k + ((j - k) & c.NWmask);
            if (w != k && ldcg32(&c.bin_cnt[g * c.NW + j]) != 0) {
                u64 tw = (u64)w << c.logW;
                hint = min(hint, tw >= ASTRA_T_INF ? ASTRA_T_INF - 1 : (u32)tw);
            }
        }
    }
    hint = __reduce_min_sync(FULL, hint);
    err = __reduce_or_sync(FULL, err);
    if (lane == 0) {
        if (stepped) c.node_next[v] = local_next;          // else unchanged
        hint = min(hint, c.node_next[v]);
        u32 span = t1 - t0;
        atomicAdd((unsigned long long*)&ctl.busy, (unsigned long long)stepped);
        atomicAdd((unsigned long long*)&ctl.skipped, (unsigned long long)(span - stepped));
        if (acked_steps) { atomicAdd(&ctl.acked, acked_steps); atomicMax(&ctl.completion, completion); }
        if (err) atomicOr(&ctl.err, err);
        atomicMin(&ctl.next_hint, hint);
    }
    (void)t_last;
}

__device__ void resolve_ctx(Ctx& c, const PointDesc& P, const uint8_t* cb, uint8_t* ws, uint8_t* rs) {
    c.G = P.G; c.V = P.V; c.E = P.E; c.S = P.S; c.C = P.C; c.Wv = P.Wv; c.K = P.K; c.H = P.H;
    c.CW = P.CW; c.nwords = P.nwords; c.slots = P.slots; c.bmwords = P.bmwords;
    c.logW = P.logW; c.W = 1u << P.logW; c.NW = P.NW; c.NWmask = P.NW - 1; c.kmagic = P.kdiv_magic;
    c.tmax = (u32)P.max_cycles; c.flags = P.flags;
    c.fullmask = P.K >= 64 ? ~0ull : ((1ull << P.K) - 1);
#define CP(name) c.name = (const u32*)(cb + P.c_##name)
    CP(row_ptr); CP(in_ptr); CP(in_link); CP(leff); CP(bw); CP(icand_ptr); CP(icand); CP(ocand_ptr); CP(ocand); CP(next_link);
    CP(step_od); CP(lines); CP(cu_lo); CP(cu_n); CP(succ_ptr); CP(succ); CP(ndeps);
    CP(step_q); CP(step_r); CP(first_link); CP(step_alpha); CP(cul_ptr); CP(cul); CP(rel_off); CP(init_rel); CP(init_rel_cnt);
    CP(fifo_off); CP(fifo_mask); CP(pipe_off); CP(pipe_mask); CP(credit_cap);
#undef CP
#define WP(name, type) c.name = (type*)(ws + P.w_##name)
    WP(fifo_head, u32); WP(fifo_tail, u32); WP(pipe_tail, u32); WP(pipe_tail_pub, u32); WP(pipe_head, u32); WP(pipe_tsnap, u32);
    WP(credit, u32); WP(credit_time, u32); WP(link_lines, u32);
    WP(fifo_buf, u64); WP(pipe_buf, u64);
    WP(t_release, u32); WP(issued_cnt, u32); WP(t_issued, u32); WP(deliv_cnt, u32); WP(t_deliv, u32);
    WP(ack_cnt, u32); WP(t_ack, u32); WP(ndep_left, u32);
    WP(wf_rem, u32); WP(wf_cur, u32); WP(wf_busy, u64);
    WP(want, u32); WP(freeb, u32); WP(pend, u64); WP(pend_link, u32); WP(pend_cnt, u32); WP(rel_list, u32); WP(rel_cnt, u32); WP(sel, u32);
    WP(ack_rec, u64); WP(bitmap, u32); WP(bin_cnt, u32); WP(ack_tmp, u64); WP(ack_sorted, u64);
    WP(node_next, u32); WP(node_busy, u64); WP(node_acked, u32);
#undef WP
    c.r_step_ts = (u64*)(rs + P.r_step_ts);
    c.r_link_lines = (u64*)(rs + P.r_link_lines);
    c.r_summary = (DeviceSummary*)(rs + P.r_summary);
}

extern "C" __global__ void __launch_bounds__(512, 1)
astra_step_kernel(const uint8_t* __restrict__ cblob, uint8_t* __restrict__ ws_base, uint8_t* __restrict__ results,
                  const PointDesc* __restrict__ points, const u32* __restrict__ order, u32* queue,
                  u32 n_points, u64 ws_stride) {
    extern __shared__ __align__(16) uint8_t smem[];
    Ctx& c = *reinterpret_cast<Ctx*>(smem);
    Ctl& ctl = *reinterpret_cast<Ctl*>(smem + ((sizeof(Ctx) + 15) & ~size_t(15)));
    u32* scnt_all = reinterpret_cast<u32*>(smem + ((sizeof(Ctx) + 15) & ~size_t(15)) + ((sizeof(Ctl) + 15) & ~size_t(15)));
    const u32 tid = threadIdx.x, nthr = blockDim.x;
    const u32 lane = tid & 31, warp = tid >> 5, nwarps = nthr >> 5;
    u32* scnt = scnt_all + warp * ((1u << ASTRA_WMAX_LOG2) + 32);
    uint8_t* ws = ws_base + (size_t)blockIdx.x * ws_stride;

    for (;;) {
        __syncthreads();
        if (tid == 0) ctl.point = atomicAdd(queue, 1u);
        __syncthreads();
        const u32 qi = ctl.point;
        if (qi >= n_points) break;
        const u32 pi = order[qi];
        const PointDesc& P = points[pi];
        if (tid == 0) {
            resolve_ctx(c, P, cblob, ws, results);
            ctl.acked = 0; ctl.completion = 0; ctl.err = 0; ctl.done = 0; ctl.next_hint = ASTRA_T_INF;
            ctl.busy = 0; ctl.skipped = 0;
        }
        // ---- workspace init ----
        {
            uint4 z = make_uint4(0, 0, 0, 0), f = make_uint4(~0u, ~0u, ~0u, ~0u);
            uint4* pz = reinterpret_cast<uint4*>(ws);
            for (u64 i = tid; i < P.ws_zero_bytes / 16; i += nthr) pz[i] = z;
            uint4* pf = reinterpret_cast<uint4*>(ws + P.ws_ff_off);
            for (u64 i = tid; i < P.ws_ff_bytes / 16; i += nthr) pf[i] = f;
        }
        __syncthreads();
        for (u32 e = tid; e < c.E; e += nthr) c.credit[e] = c.credit_cap[e];
        for (u32 s = tid; s < c.S; s += nthr) c.ndep_left[s] = c.ndeps[s];
        for (u32 i = tid; i < c.G * c.CW; i += nthr) {
            u32 gq = i / c.CW, wf = i - gq * c.CW;
            c.wf_cur[i] = c.cul_ptr[gq * c.C + wf / c.Wv];
        }
        for (u32 gq = tid; gq < c.G; gq += nthr) c.rel_cnt[gq] = c.init_rel_cnt[gq];
        for (u32 s = tid; s < c.S; s += nthr) c.rel_list[s] = c.init_rel[s];
        for (u32 i = tid; i < c.G * c.nwords; i += nthr) {
            u32 wi = i % c.nwords;
            u32 nb = c.CW - wi * 32;
            c.freeb[i] = nb >= 32 ? ~0u : ((1u << nb) - 1u);
        }
        __syncthreads();

        // ---- window loop ----
        u32 k = 0;
        int32_t status = ASTRA_STATUS_DONE;
        const u32 W = c.W;
        for (;;) {
            u64 t0l = (u64)k << c.logW;
            if (t0l >= c.tmax) { status = ASTRA_STATUS_MAX_CYCLES; break; }
            u32 t0 = (u32)t0l;
            u32 t1 = (u32)min((u64)c.tmax, t0l + W);
            for (u32 v = warp; v < c.V; v += nwarps) node_window(c, ctl, v, k, t0, t1, scnt, lane);
            __syncthreads();
            if (tid == 0) {                     // the only thread touching ctl between the two barriers
                u32 hint = ctl.next_hint;
                ctl.next_hint = ASTRA_T_INF;
                u32 dec = 0, nk = k + 1;
                if (ctl.acked == c.S) dec = 1 + ASTRA_STATUS_DONE;
                else if (ctl.err) dec = 1 + ASTRA_STATUS_INTERNAL;
                else if (hint == ASTRA_T_INF) dec = 1 + ASTRA_STATUS_DEADLOCK;
                else if (!(c.flags & (u32)ASTRA_FLAG_NO_WINDOW_SKIP)) nk = max(nk, hint >> c.logW);
                ctl.decision = dec; ctl.next_k = nk;
            }
            __syncthreads();
            u32 dec = ctl.decision;
            if (dec) { status = (int32_t)dec - 1; break; }
            k = ctl.next_k;
        }
        __syncthreads();
        // ---- A8: write-out ----
        for (u32 s = tid; s < c.S; s += nthr) {
            u32 a = c.t_release[s], b = c.t_issued[s], d = c.t_deliv[s], e = c.t_ack[s];
            c.r_step_ts[4 * (size_t)s + 0] = a == ASTRA_TS_NONE32 ? ~0ull : a;
            c.r_step_ts[4 * (size_t)s + 1] = b == ASTRA_TS_NONE32 ? ~0ull : b;
            c.r_step_ts[4 * (size_t)s + 2] = d == ASTRA_TS_NONE32 ? ~0ull : d;
            c.r_step_ts[4 * (size_t)s + 3] = e == ASTRA_TS_NONE32 ? ~0ull : e;
        }
        for (u32 e = tid; e < c.E; e += nthr) c.r_link_lines[e] = c.link_lines[e];
        if (tid == 0) {
            DeviceSummary sm;
            sm.status = status; sm.n_steps = c.S; sm.n_links = c.E; sm.window = W;
            sm.completion_cycle = ctl.completion; sm.total_lines = P.total_lines;
            sm.busy_cycles = ctl.busy; sm.skipped_cycles = ctl.skipped;
            *c.r_summary = sm;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
static size_t smem_bytes(u32 warps) {
    return ((sizeof(Ctx) + 15) & ~size_t(15)) + ((sizeof(Ctl) + 15) & ~size_t(15)) +
           (size_t)warps * ((1u << ASTRA_WMAX_LOG2) + 32) * sizeof(u32);
}

int32_t astra_engine_occupancy(u32 warps_per_cta, u32* ctas_per_sm, u32* n_sms, std::string& err) {
    int dev = 0, sms = 0, occ = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    size_t sm = smem_bytes(warps_per_cta);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(astra_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, astra_step_kernel, (int)warps_per_cta * 32, sm);
    if (e != cudaSuccess) { err = std::string("occupancy query: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    *ctas_per_sm = (u32)occ; *n_sms = (u32)sms;
    return ASTRA_OK;
}

int32_t astra_engine_launch(const EngineLaunch& L, void* stream, std::string& err) {
    size_t sm = smem_bytes(L.warps_per_cta);
    cudaError_t e = cudaFuncSetAttribute(astra_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) { err = std::string("smem attribute: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    e = cudaMemsetAsync(L.d_queue, 0, sizeof(u32), (cudaStream_t)stream);
    if (e != cudaSuccess) { err = std::string("queue reset: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    astra_step_kernel<<<L.grid, L.warps_per_cta * 32, sm, (cudaStream_t)stream>>>(
        L.d_const, L.d_ws, L.d_results, L.d_points, L.d_order, L.d_queue, L.n_points, L.ws_stride);
    e = cudaGetLastError();
    if (e != cudaSuccess) { err = std::string("kernel launch: ") + cudaGetErrorString(e); return ASTRA_ECUDA; }
    return ASTRA_OK;
}
