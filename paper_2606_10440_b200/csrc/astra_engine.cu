// astra_engine.cu -- the sm_100a window-batched step kernel of the cycle-synchronous cache-line
// simulator.
//
// The paper's simulator is an event-driven CPU program.  This engine is organised
// around one structural fact instead: a line accepted by a link at cycle a cannot reach the next
// node before a + Leff, and an ack cannot reach its owner before t_deliv + alpha >= t_deliv +
// min Leff.  With W = 2^k <= min Leff, nothing a node does inside the window [kW, (k+1)W) can
// influence another node inside the same window.  So simulated time advances a whole window at a
// time, and inside a window every phase of rules R7-R12 is a data-parallel pass over ALL events
// of the window instead of a serial walk over cycles:
//
//   stage 1  arrivals (R7 A1)   one warp per link, 32 pipe entries per step: deliveries bump
//            the step counters and post slot-addressed ack records; transit lines drop into the
//            staging cell (out-link, cycle) at a slot fixed by (in-link, position) -- the FIFO
//            append order of R8 without atomics or sorting.
//            ack gather (R6, A3) one warp per GPU: this window's acks, counting-sorted by cycle,
//            per-step ack counts and t_ack.
//   stage 2  release + issue (R10-R13) one warp per GPU: dependency events of the window become
//            timed releases; the fixed-priority HBM grant scan walks only the cycles of the
//            window where something can change; issued lines drop into their staging cell.
//   stage 3  link service (R9)  one warp per link: the occupied staging slots of the window, read
//            in slot order, are the FIFO appends; acceptance times of the whole FIFO follow from
//            a prefix-max scan (integer and 1/P bandwidths) or a credit walk (any other), and the
//            accepted lines are stamped with their arrival cycle in the link's ring.
//   stage 4  next non-idle window (A7): min over pending arrivals, acks, backlog and ready work.
//
// One CTA simulates one design point at a time and pulls the next from a cost-sorted queue.
#include "astra_internal.h"
#include "../../include/astra.h"

#include <cuda_runtime.h>

#define FULL 0xffffffffu
#define SCR_WORDS ((1u << ASTRA_WMAX_LOG2) + 64)   // per-warp scratch words

struct Ctx {   // resolved pointers of the point a CTA is running; lives in shared memory
    u32 G, V, E, S, C, Wv, K, H, CW, nwords, slots, bmwords, logW, W, NC, NWmask, NW, kmagic, tmax, flags;
    u64 fullmask;
    const u32 *in_ptr, *in_link, *head, *tail, *leff, *bw, *next_link;
    const u32 *step_od, *lines, *cu_lo, *cu_n, *succ_ptr, *succ, *ndeps;
    const u32 *step_q, *step_r, *first_link, *step_alpha, *cul_ptr, *cul, *rel_off, *init_rel, *init_rel_cnt, *ev_off;
    const u32 *ring_off, *ring_mask, *lkind, *ceilb, *lstate0_init, *stage_off, *mask_off, *classoff;
    const u32 *nd_cellcap, *nd_mw, *nd_injoff;
    u32 *pipe_head, *fifo_head, *ltail, *lstate0, *lstate1, *link_lines, *masks;
    u64 *ring, *stage;
    u32 *t_release, *issued_cnt, *t_issued, *deliv_cnt, *t_deliv, *ack_cnt, *t_ack, *ndep_left, *rel_time;
    u32 *wf_rem, *wf_cur; u64 *wf_busy;
    u32 *want, *freeb, *sel, *plist, *pcnt, *ev_list, *ev_cnt, *ack_n;
    u64 *ack_rec, *ack_tmp, *ack_sorted; u32 *bitmap, *bin_cnt;
    u64 *r_step_ts, *r_link_lines; DeviceSummary *r_summary;
};

struct Ctl {   // per-CTA control block in shared memory
    u32 point;          // index into the order array
    u32 acked;          // steps fully acked so far
    u32 completion;     // max t_ack
    u32 err;            // engine self-check flags
    u32 next_hint;      // min over everything pending of its next event time
    u32 decision;       // 0 = run window `next_k`, else 1 + status
    u32 next_k;
    u32 pad;
    u64 busy, skipped;
    u32 ackwin[ASTRA_NW_MAX];   // acks posted per future window bin
};

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

// Put one flit payload into the staging cell (out-link o, cycle t0 + d) at `slot` (R7/R8).
__device__ __forceinline__ void stage_put(Ctx& c, u32 o, u32 v, u32 cb, u32 d, u32 slot, u64 payload) {
    u32 ci = cb + d; if (ci >= c.NC) ci -= c.NC;
    c.stage[(size_t)c.stage_off[o] + (size_t)ci * c.nd_cellcap[v] + slot] = payload;
    atomicOr(&c.masks[(size_t)c.mask_off[o] + (size_t)ci * c.nd_mw[v] + (slot >> 5)], 1u << (slot & 31));
}

// ---------------------------------------------------------------------------------------------
// stage 1a: arrivals on link e during [t0, t0 + wlen)   (R7 A1)
// ---------------------------------------------------------------------------------------------
__device__ void arrivals_link(Ctx& c, Ctl& ctl, u32 e, u32 t0, u32 wlen, u32 cb, u32 lane) {
    const u32 lo = c.pipe_head[e], hi = c.fifo_head[e];
    if (lo == hi) return;
    const u32 v = c.head[e];
    const u64* ring = c.ring + c.ring_off[e];
    const u32 rmask = c.ring_mask[e], coff = c.classoff[e];
    u32 carry_d = 0xffffffffu, carry_cnt = 0, idx = lo, ndue = 0, hint = ASTRA_T_INF;
    for (;;) {
        const u32 i = idx + lane;
        const bool valid = (int32_t)(hi - i) > 0;
        const u64 flit = valid ? ring[i & rmask] : 0ull;
        const u32 d = ((u32)(flit >> ASTRA_FLIT_TIME_SHIFT) - t0) & ASTRA_TMASK26;
        const bool due = valid && d < wlen;
        const u32 duemask = __ballot_sync(FULL, due);
        if (valid && !due) hint = min(hint, t0 + d);
        if (duemask) {
            // position of the line among the lines this link delivers in the same cycle
            u32 r = 0, grp = 0;
            if (due) {
                grp = __match_any_sync(duemask, d);
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
            if (transit) {
                const u32 o = c.next_link[(size_t)v * c.G + dstg];
                stage_put(c, o, v, cb, d, coff + r, flit & ASTRA_FLIT_PAYLOAD_MASK);
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
                    const u32 bin = (ta >> c.logW) & c.NWmask;
                    atomicOr(&c.bitmap[(size_t)(owner * c.NW + bin) * c.bmwords + (bit >> 5)], 1u << (bit & 31));
                    atomicAdd(&c.bin_cnt[owner * c.NW + bin], 1u);
                    atomicAdd(&ctl.ackwin[bin], 1u);
                    const u32 m = __match_any_sync(dmask, step);
                    const u32 dmax = __reduce_max_sync(m, d);
                    if ((m & lanemask_lt()) == 0) {
                        const u32 dc = c.deliv_cnt[step] + __popc(m);
                        c.deliv_cnt[step] = dc;
                        if (dc == c.lines[step]) { c.t_deliv[step] = t0 + dmax; completed = true; }
                    }
                }
                if (completed) {      // DELIVERED event at GPU v (dst of the step)
                    const u32 pos = atomicAdd(&c.ev_cnt[v], 1u);
                    c.ev_list[c.ev_off[v] + pos] = step | ((u32)ASTRA_DEP_DELIVERED << 30);
                }
            }
            ndue += __popc(duemask);
        }
        if (duemask != FULL) break;
        idx += 32;
    }
    hint = __reduce_min_sync(FULL, hint);
    if (lane == 0) {
        c.pipe_head[e] = lo + ndue;
        if (hint != ASTRA_T_INF) atomicMin(&ctl.next_hint, hint);
    }
}

// ---------------------------------------------------------------------------------------------
// stage 1b: this window's acks of GPU g, counting-sorted by cycle; per-step ack counts (R6, A3)
// ---------------------------------------------------------------------------------------------
__device__ void ack_gather(Ctx& c, Ctl& ctl, u32 g, u32 k, u32 t0, u32 wlen, u32* scnt, u32 lane) {
    const u32 bin = k & c.NWmask;
    const u32 n = c.bin_cnt[g * c.NW + bin];
    if (lane == 0) c.ack_n[g] = n;
    if (n == 0) return;
    for (u32 i = lane; i <= wlen; i += 32) scnt[i] = 0;
    __syncwarp();
    u32* bm = c.bitmap + (size_t)(g * c.NW + bin) * c.bmwords;
    const u64* rec = c.ack_rec + (size_t)g * c.slots;
    u64* tmp = c.ack_tmp + (size_t)g * c.slots;
    u64* srt = c.ack_sorted + (size_t)g * c.slots;
    // pass 1: discover, histogram by cycle, compact into tmp
    u32 total = 0;
    for (u32 wb = 0; wb < c.bmwords; wb += 32) {
        const u32 wi = wb + lane;
        u32 w = (wi < c.bmwords) ? bm[wi] : 0;
        if (w) bm[wi] = 0;
        const u32 cnt = __popc(w);
        const u32 incl = warp_incl_scan(cnt, lane);
        u32 pos = total + incl - cnt;
        total += __shfl_sync(FULL, incl, 31);
        while (w) {
            const u32 b = __ffs(w) - 1; w &= w - 1;
            const u32 idx = wi * 32 + b;
            const u64 rc = rec[idx];
            const u32 cyc = (u32)rc - t0;
            const u32 wf = c.K == 1 ? idx : (u32)(((u64)idx * c.kmagic) >> 32);   // idx / K (magic overflows for K == 1)
            const u32 slot = idx - wf * c.K;
            atomicAdd(&scnt[cyc], 1u);
            tmp[pos++] = (rc & 0xffffffff00000000ull) | (cyc << 18) | (wf << 6) | slot;
        }
    }
    __syncwarp();
    // exclusive scan of the histogram
    u32 carry = 0;
    for (u32 b = 0; b < wlen; b += 32) {
        const u32 i = b + lane;
        const u32 vv = (i < wlen) ? scnt[i] : 0;
        const u32 incl = warp_incl_scan(vv, lane);
        if (i < wlen) scnt[i] = carry + incl - vv;
        carry += __shfl_sync(FULL, incl, 31);
    }
    __syncwarp();
    // pass 2: scatter into cycle order; count acks per step, stamp t_ack (R3, R14)
    u32 acked_steps = 0, completion = 0;
    for (u32 b = 0; b < total; b += 32) {
        const u32 i = b + lane;
        const bool act = i < total;
        const u64 ent = act ? tmp[i] : 0ull;
        const u32 amask = __ballot_sync(FULL, act);
        bool completed = false;
        if (act) {
            const u32 cyc = (u32)ent >> 18;
            const u32 pos = atomicAdd(&scnt[cyc], 1u);
            srt[pos] = ent;
            const u32 step = (u32)(ent >> 32);
            const u32 m = __match_any_sync(amask, step);
            const u32 cmax = __reduce_max_sync(m, cyc);
            if ((m & lanemask_lt()) == 0) {
                const u32 ac = c.ack_cnt[step] + __popc(m);
                const u32 tm = max(c.t_ack[step], t0 + cmax);
                c.ack_cnt[step] = ac; c.t_ack[step] = tm;
                if (ac == c.lines[step]) {
                    completed = true;
                    const u32 pos2 = atomicAdd(&c.ev_cnt[g], 1u);
                    c.ev_list[c.ev_off[g] + pos2] = step | ((u32)ASTRA_DEP_ACKED << 30);
                }
            }
            if (completed) completion = max(completion, max(c.t_ack[step], t0 + cmax));
        }
        acked_steps += __popc(__ballot_sync(FULL, completed));
    }
    completion = __reduce_max_sync(FULL, completion);
    if (lane == 0) {
        c.bin_cnt[g * c.NW + bin] = 0;
        atomicSub(&ctl.ackwin[bin], total);
        if (total != n) atomicOr(&ctl.err, 2u);
        if (acked_steps) { atomicAdd(&ctl.acked, acked_steps); atomicMax(&ctl.completion, completion); }
    }
    __syncwarp();
}

// ---------------------------------------------------------------------------------------------
// stage 2 helpers
// ---------------------------------------------------------------------------------------------
// A step's timestamp of kind `kind` was stamped at cycle `time` on GPU g: count down its
// successors (R3, R10).  A successor whose last dependency this was is released at the max over
// its dependencies' times and joins g's pending-release list.  Whole warp, warp-uniform p.
__device__ __forceinline__ void on_event(Ctx& c, u32 g, u32 p, u32 kind, u32 time, u32 lane) {
    const u32 lo = c.succ_ptr[p], hi = c.succ_ptr[p + 1];
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
__device__ __forceinline__ bool wf_advance(Ctx& c, u32 g, u32 wf, u32& cur, u32& rem, u32 t) {
    const u32 end = c.cul_ptr[g * c.C + wf / c.Wv + 1];
    rem = ASTRA_NOTLOADED;
    while (cur < end) {
        const u32 s = c.cul[cur];
        if (c.t_release[s] > t) return false;           // NONE (0xffffffff) or a later cycle
        const u32 q = c.step_q[s] + (((wf - c.cu_lo[s] * c.Wv) < c.step_r[s]) ? 1u : 0u);
        if (q) { rem = q; return true; }
        cur++;
    }
    return false;
}

// ---------------------------------------------------------------------------------------------
// stage 2: release + issue of GPU g over [t0, t1)   (R10 - R13, slot return of R7 A3)
// ---------------------------------------------------------------------------------------------
__device__ void issue_window(Ctx& c, Ctl& ctl, u32 g, u32 t0, u32 t1, u32 cb, u32 lane) {
    // dependency events of this window (DELIVERED from stage 1a, ACKED from stage 1b)
    {
        const u32 nev = c.ev_cnt[g];
        for (u32 j = 0; j < nev; j++) {
            const u32 ek = c.ev_list[c.ev_off[g] + j];
            const u32 p = ek & 0xfffffu, kind = ek >> 30;
            const u32 time = kind == ASTRA_DEP_DELIVERED ? c.t_deliv[p] : c.t_ack[p];
            on_event(c, g, p, kind, time, lane);
        }
        __syncwarp();
        if (lane == 0 && nev) c.ev_cnt[g] = 0;
    }
    const u32 ack_n = c.ack_n[g];
    u32 ack_pos = 0;
    const u64* srt = c.ack_sorted + (size_t)g * c.slots;
    u32* plist = c.plist + c.rel_off[g];
    u32* want = c.want + (size_t)g * c.nwords;
    u32* freeb = c.freeb + (size_t)g * c.nwords;
    u32* sel = c.sel + (size_t)g * c.H;
    const u32 injoff = c.nd_injoff[g];
    u32 t_ack_next = ack_n ? t0 + ((u32)srt[0] >> 18) : ASTRA_T_INF;
    u32 t_rel_next = ASTRA_T_INF;
    {
        const u32 np = c.pcnt[g];
        for (u32 i = lane; i < np; i += 32) t_rel_next = min(t_rel_next, c.t_release[plist[i]]);
        t_rel_next = __reduce_min_sync(FULL, t_rel_next);
    }
    bool more;
    {
        u32 any = 0;
        for (u32 wi = lane; wi < c.nwords; wi += 32) any |= want[wi] & freeb[wi];
        more = __ballot_sync(FULL, any != 0) != 0;
    }
    u32 t = min(min(t_ack_next, t_rel_next), more ? t0 : ASTRA_T_INF);
    if (t < t0) t = t0;

    while (t < t1) {
        more = false;
        // ---- slot return: acks due at t (R7 A3) ----
        if (t_ack_next == t) {
            const u32 cyc = t - t0;
            while (ack_pos < ack_n) {
                const u32 j = ack_pos + lane;
                const u64 ent64 = (j < ack_n) ? srt[j] : ~0ull;
                const u32 ent = (u32)ent64;
                const bool now = (j < ack_n) && (ent >> 18) == cyc;
                const u32 nm = __ballot_sync(FULL, now);
                if (nm == 0) break;
                if (now) {
                    const u32 wf = (ent >> 6) & 0xfffu, slot = ent & 63u;
                    // several acks of one wavefront may land in the same cycle
                    const u32 mw = __match_any_sync(nm, wf);
                    const u32 blo = __reduce_or_sync(mw, slot < 32 ? (1u << slot) : 0u);
                    const u32 bhi = __reduce_or_sync(mw, slot >= 32 ? (1u << (slot - 32)) : 0u);
                    if ((mw & lanemask_lt()) == 0) {
                        u64 busy = c.wf_busy[(size_t)g * c.CW + wf];
                        busy &= ~(((u64)bhi << 32) | blo);
                        c.wf_busy[(size_t)g * c.CW + wf] = busy;
                    }
                    const u32 wi = wf >> 5;
                    const u32 mi = __match_any_sync(nm, wi);
                    const u32 bits = __reduce_or_sync(mi, 1u << (wf & 31));
                    if ((mi & lanemask_lt()) == 0) freeb[wi] |= bits;
                }
                ack_pos += __popc(nm);
                if (__popc(nm) < 32) break;
            }
            __syncwarp();
            t_ack_next = (ack_pos < ack_n) ? t0 + ((u32)srt[ack_pos] >> 18) : ASTRA_T_INF;
        }

        // ---- phase C: releases that take effect at t (R10) ----
        if (t_rel_next == t) {
            const u32 np = c.pcnt[g];
            u32 keep = 0, tn = ASTRA_T_INF;
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
                while (nowm) {
                    const u32 src = __ffs(nowm) - 1; nowm &= nowm - 1;
                    const u32 sr = __shfl_sync(FULL, s, src);
                    const u32 lo = c.cu_lo[sr] * c.Wv, hi = lo + c.cu_n[sr] * c.Wv;
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
            for (u32 i = 0; i < take; i++) {
                const u32 b = __ffs(r) - 1; r &= r - 1;
                sel[nsel + excl + i] = wi * 32 + b;
            }
            const u32 got = min(tot, budget);
            if (tot > got) left_over = true;
            nsel += got; budget -= got;
        }
        __syncwarp();
        for (u32 b = 0; b < nsel; b += 32) {
            const u32 j = b + lane; const bool act = j < nsel;
            u32 wf = 0, s = 0; bool full = false, keepw = true;
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
                // injected at t + 1 into the first-hop FIFO, after that cycle's transit lines (R7 A2)
                stage_put(c, c.first_link[s], g, cb, t + 1 - t0, injoff + j, (u64)s | ((u64)wf << 20) | ((u64)slot << 32));
                if (rem == 0) { cur++; keepw = wf_advance(c, g, wf, cur, rem, t); c.wf_cur[gw] = cur; }
                c.wf_rem[gw] = rem;
            }
            const u32 amask = __ballot_sync(FULL, act);
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
                const u32 clrf = __reduce_or_sync(mi, full ? (1u << (wf & 31)) : 0u);
                const u32 clrw = __reduce_or_sync(mi, keepw ? 0u : (1u << (wf & 31)));
                if ((mi & lanemask_lt()) == 0) {
                    if (clrf) freeb[wi] &= ~clrf;
                    if (clrw) want[wi] &= ~clrw;
                }
            }
            u32 cm = __ballot_sync(FULL, completed);
            while (cm) {
                const u32 src = __ffs(cm) - 1; cm &= cm - 1;
                const u32 p = __shfl_sync(FULL, s, src);
                on_event(c, g, p, ASTRA_DEP_ISSUED, t + 1, lane);      // visible to phase C of t + 1 (R10)
                t_rel_next = ASTRA_T_INF;                               // recomputed below
            }
        }
        __syncwarp();
        if (nsel) more = true;            // an issuing wavefront may issue again at t + 1
        if (left_over) more = true;
        if (t_rel_next == ASTRA_T_INF) {
            const u32 np = c.pcnt[g];
            u32 tn = ASTRA_T_INF;
            for (u32 i = lane; i < np; i += 32) tn = min(tn, c.t_release[plist[i]]);
            t_rel_next = __reduce_min_sync(FULL, tn);
        }
        // ---- next cycle of this GPU where something can change (A7) ----
        u32 tn = min(t_ack_next, t_rel_next);
        if (more) tn = min(tn, t + 1);
        t = tn;
    }
    if (lane == 0 && t != ASTRA_T_INF) atomicMin(&ctl.next_hint, t);
}

// ---------------------------------------------------------------------------------------------
// stage 3: link e over [t0, t1): FIFO appends of the window in slot order, acceptance times of
// the whole FIFO (R9), arrival stamps.  `pre` is per-warp scratch of >= wlen + 1 words.
// ---------------------------------------------------------------------------------------------
__device__ void link_window(Ctx& c, Ctl& ctl, u32 e, u32 t0, u32 t1, u32 cb, u32* pre, u32 lane) {
    const u32 wlen = t1 - t0;
    const u32 v = c.tail[e];
    const u32 cap = c.nd_cellcap[v], mw = c.nd_mw[v];
    u32* masks = c.masks + c.mask_off[e];
    const u64* stage = c.stage + c.stage_off[e];
    // ---- appends per cycle of the window: exclusive prefix over the cells ----
    u32 n_new = 0;
    for (u32 b = 0; b < wlen; b += 32) {
        const u32 tau = b + lane; u32 cnt = 0;
        if (tau < wlen) {
            u32 ci = cb + tau; if (ci >= c.NC) ci -= c.NC;
            for (u32 w = 0; w < mw; w++) cnt += __popc(masks[ci * mw + w]);
        }
        const u32 incl = warp_incl_scan(cnt, lane);
        if (tau < wlen) pre[tau] = n_new + incl - cnt;
        n_new += __shfl_sync(FULL, incl, 31);
    }
    const u32 fh = c.fifo_head[e], tl = c.ltail[e];
    const u32 n_back = tl - fh;
    if (n_new == 0 && n_back == 0) return;
    if (lane == 0) pre[wlen] = n_new;
    __syncwarp();
    u64* ring = c.ring + c.ring_off[e];
    const u32 rmask = c.ring_mask[e];
    if (lane == 0 && (tl + n_new) - c.pipe_head[e] > rmask + 1) atomicOr(&ctl.err, 1u);   // ring overflow guard
    const u32 n_tot = n_back + n_new;
    const u32 lk = c.lkind[e];
    const u32 kind = lk & 3u, param = lk >> 2;
    const u32 leff = c.leff[e];
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
    bool saturated = (scan_limit == 0);

    for (u32 base = 0; base < n_tot; base += 32) {
        if (saturated && base + 32 <= n_back) {              // backlog that stays queued: nothing to do
            base = (n_back & ~31u);
            if (base >= n_tot) break;
        }
        const u32 i = base + lane;
        const bool act = i < n_tot;
        const bool isnew = act && i >= n_back;
        u32 a = 0, tau = 0, q = 0;
        if (isnew) {                                         // append cycle of the line: search the cell prefix
            const u32 p = i - n_back;
            u32 lo = 0, hi = wlen;                           // largest tau with pre[tau] <= p
            while (hi - lo > 1) { const u32 mid = (lo + hi) >> 1; if (pre[mid] <= p) lo = mid; else hi = mid; }
            tau = lo; q = p - pre[lo]; a = tau;
        }
        u32 x = 0xffffffffu;                                 // acceptance cycle relative to t0
        if (!saturated) {
            const bool in_scan = i < scan_limit;
            if (kind == ASTRA_LK_INT) {
                int val = in_scan ? (int)(param * a) - (int)i : INT_MIN;
                int pm = warp_incl_max(val, lane);
                pm = max(pm, run_max);
                run_max = __shfl_sync(FULL, pm, 31);
                if (in_scan) x = (u32)((int)i + pm) / param;
            } else if (kind == ASTRA_LK_PERIOD) {
                int val = in_scan ? (int)a - (int)(param * i) : INT_MIN;
                int pm = warp_incl_max(val, lane);
                pm = max(pm, run_max);
                run_max = __shfl_sync(FULL, pm, 31);
                if (in_scan) {
                    // x_i = max(a_i, x_{i-1} + P) with x_{-1} + P = xn_rel
                    const int xi = (int)(param * i) + max(pm, xn_rel);
                    x = (u32)xi;
                }
            } else {
                // saturating credit walked in FIFO order; every lane tracks the same state
                const u32 bw = param;
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
        }
        const bool acc = act && x < wlen;
        const u32 accm = __ballot_sync(FULL, acc);
        const u32 actm = __ballot_sync(FULL, act);
        if (accm) {
            if (n_acc == 0) first_x = __shfl_sync(FULL, x, __ffs(accm) - 1);
            last_x = __shfl_sync(FULL, x, 31 - __clz(accm));
            n_acc += __popc(accm);
        }
        if (accm != actm) saturated = true;
        const u64 stamp = acc ? ((u64)((t0 + x + leff) & ASTRA_TMASK26) << ASTRA_FLIT_TIME_SHIFT) : 0ull;
        if (isnew) {
            u32 ci = cb + tau; if (ci >= c.NC) ci -= c.NC;
            u32 slot = 0, qq = q;
            for (u32 w = 0; w < mw; w++) {
                const u32 word = masks[ci * mw + w];
                const u32 pc = __popc(word);
                if (qq < pc) { slot = w * 32 + __fns(word, 0, qq + 1); break; }
                qq -= pc;
            }
            const u64 payload = stage[(size_t)ci * cap + slot];
            ring[(tl + (i - n_back)) & rmask] = payload | stamp;
        } else if (acc) {
            const u32 pos = (fh + i) & rmask;
            ring[pos] = (ring[pos] & ASTRA_FLIT_PAYLOAD_MASK) | stamp;
        }
    }
    __syncwarp();
    // consume the cells
    if (n_new) {
        for (u32 tau = lane; tau < wlen; tau += 32) {
            u32 ci = cb + tau; if (ci >= c.NC) ci -= c.NC;
            for (u32 w = 0; w < mw; w++) masks[ci * mw + w] = 0;
        }
    }
    if (lane == 0) {
        c.fifo_head[e] = fh + n_acc;
        c.ltail[e] = tl + n_new;
        if (n_acc) {
            c.link_lines[e] += n_acc;
            atomicMin(&ctl.next_hint, t0 + first_x + leff);
            if (kind == ASTRA_LK_PERIOD) c.lstate0[e] = t0 + last_x + param;
        }
        if (kind == ASTRA_LK_GENERAL) { c.lstate0[e] = cr; c.lstate1[e] = tc; }
        if (n_tot > n_acc) atomicMin(&ctl.next_hint, t1);
    }
}

__device__ void resolve_ctx(Ctx& c, const PointDesc& P, const uint8_t* cb, uint8_t* ws, uint8_t* rs) {
    c.G = P.G; c.V = P.V; c.E = P.E; c.S = P.S; c.C = P.C; c.Wv = P.Wv; c.K = P.K; c.H = P.H;
    c.CW = P.CW; c.nwords = P.nwords; c.slots = P.slots; c.bmwords = P.bmwords;
    c.logW = P.logW; c.W = 1u << P.logW; c.NC = P.NC; c.NW = P.NW; c.NWmask = P.NW - 1; c.kmagic = P.kdiv_magic;
    c.tmax = (u32)P.max_cycles; c.flags = P.flags;
    c.fullmask = P.K >= 64 ? ~0ull : ((1ull << P.K) - 1);
#define CP(name) c.name = (const u32*)(cb + P.c_##name)
    CP(in_ptr); CP(in_link); CP(head); CP(tail); CP(leff); CP(bw); CP(next_link);
    CP(step_od); CP(lines); CP(cu_lo); CP(cu_n); CP(succ_ptr); CP(succ); CP(ndeps);
    CP(step_q); CP(step_r); CP(first_link); CP(step_alpha); CP(cul_ptr); CP(cul); CP(rel_off); CP(init_rel); CP(init_rel_cnt); CP(ev_off);
    CP(ring_off); CP(ring_mask); CP(lkind); CP(ceilb); CP(lstate0_init); CP(stage_off); CP(mask_off); CP(classoff);
    CP(nd_cellcap); CP(nd_mw); CP(nd_injoff);
#undef CP
#define WP(name, type) c.name = (type*)(ws + P.w_##name)
    WP(pipe_head, u32); WP(fifo_head, u32); c.ltail = (u32*)(ws + P.w_tail); WP(lstate0, u32); WP(lstate1, u32);
    WP(link_lines, u32); WP(masks, u32); WP(ring, u64); WP(stage, u64);
    WP(t_release, u32); WP(issued_cnt, u32); WP(t_issued, u32); WP(deliv_cnt, u32); WP(t_deliv, u32);
    WP(ack_cnt, u32); WP(t_ack, u32); WP(ndep_left, u32); WP(rel_time, u32);
    WP(wf_rem, u32); WP(wf_cur, u32); WP(wf_busy, u64);
    WP(want, u32); WP(freeb, u32); WP(sel, u32); WP(plist, u32); WP(pcnt, u32); WP(ev_list, u32); WP(ev_cnt, u32); WP(ack_n, u32);
    WP(ack_rec, u64); WP(bitmap, u32); WP(bin_cnt, u32); WP(ack_tmp, u64); WP(ack_sorted, u64);
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
    u32* scr_all = reinterpret_cast<u32*>(smem + ((sizeof(Ctx) + 15) & ~size_t(15)) + ((sizeof(Ctl) + 15) & ~size_t(15)));
    const u32 tid = threadIdx.x, nthr = blockDim.x;
    const u32 lane = tid & 31, warp = tid >> 5, nwarps = nthr >> 5;
    u32* scr = scr_all + warp * SCR_WORDS;
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
            ctl.acked = 0; ctl.completion = 0; ctl.err = 0; ctl.next_hint = ASTRA_T_INF;
            ctl.busy = 0; ctl.skipped = 0;
        }
        for (u32 i = tid; i < ASTRA_NW_MAX; i += nthr) ctl.ackwin[i] = 0;
        // ---- workspace init ----
        {
            uint4 z = make_uint4(0, 0, 0, 0), f = make_uint4(~0u, ~0u, ~0u, ~0u);
            uint4* pz = reinterpret_cast<uint4*>(ws);
            for (u64 i = tid; i < P.ws_zero_bytes / 16; i += nthr) pz[i] = z;
            uint4* pf = reinterpret_cast<uint4*>(ws + P.ws_ff_off);
            for (u64 i = tid; i < P.ws_ff_bytes / 16; i += nthr) pf[i] = f;
        }
        __syncthreads();
        for (u32 e = tid; e < c.E; e += nthr) c.lstate0[e] = c.lstate0_init[e];
        for (u32 s = tid; s < c.S; s += nthr) {
            c.ndep_left[s] = c.ndeps[s];
            c.t_release[s] = c.ndeps[s] ? ASTRA_TS_NONE32 : 0u;      // steps without deps are released at t = 0 (R10)
            c.plist[s] = c.init_rel[s];
        }
        for (u32 i = tid; i < c.G * c.CW; i += nthr) {
            u32 gq = i / c.CW, wf = i - gq * c.CW;
            c.wf_cur[i] = c.cul_ptr[gq * c.C + wf / c.Wv];
        }
        for (u32 gq = tid; gq < c.G; gq += nthr) c.pcnt[gq] = c.init_rel_cnt[gq];
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
        u64 busy = 0, skipped = 0;
        for (;;) {
            const u64 t0l = (u64)k << c.logW;
            if (t0l >= c.tmax) { status = ASTRA_STATUS_MAX_CYCLES; break; }
            const u32 t0 = (u32)t0l;
            const u32 t1 = (u32)min((u64)c.tmax, t0l + W);
            const u32 wlen = t1 - t0;
            const u32 cb = t0 % c.NC;
            busy += wlen;
            // stage 1: arrivals per link, ack gather per GPU
            for (u32 task = warp; task < c.E + c.G; task += nwarps) {
                if (task < c.G) ack_gather(c, ctl, task, k, t0, wlen, scr, lane);
                else arrivals_link(c, ctl, task - c.G, t0, wlen, cb, lane);
            }
            __syncthreads();
            // stage 2: release + issue per GPU
            for (u32 g = warp; g < c.G; g += nwarps) issue_window(c, ctl, g, t0, t1, cb, lane);
            __syncthreads();
            // stage 3: link service per link
            for (u32 e = warp; e < c.E; e += nwarps) link_window(c, ctl, e, t0, t1, cb, scr, lane);
            __syncthreads();
            // stage 4: next non-idle window
            if (tid == 0) {
                u32 hint = ctl.next_hint;
                ctl.next_hint = ASTRA_T_INF;
                for (u32 j = 1; j < c.NW; j++) {
                    if (ctl.ackwin[(k + j) & c.NWmask]) {
                        u64 tw = (u64)(k + j) << c.logW;
                        hint = min(hint, tw >= ASTRA_T_INF ? ASTRA_T_INF - 1 : (u32)tw);
                        break;
                    }
                }
                u32 dec = 0, nk = k + 1;
                if (ctl.acked == c.S) dec = 1 + ASTRA_STATUS_DONE;
                else if (ctl.err) dec = 1 + ASTRA_STATUS_INTERNAL;
                else if (hint == ASTRA_T_INF) dec = 1 + ASTRA_STATUS_DEADLOCK;
                else if (!(c.flags & (u32)ASTRA_FLAG_NO_WINDOW_SKIP)) nk = max(nk, hint >> c.logW);
                ctl.decision = dec; ctl.next_k = nk;
            }
            __syncthreads();
            const u32 dec = ctl.decision;
            if (dec) { status = (int32_t)dec - 1; break; }
            skipped += (u64)(ctl.next_k - k - 1) << c.logW;
            k = ctl.next_k;
        }
        __syncthreads();
        // ---- A8: write-out ----
        for (u32 s = tid; s < c.S; s += nthr) {
            const u32 n = c.lines[s];
            const u32 a = c.t_release[s];
            c.r_step_ts[4 * (size_t)s + 0] = a == ASTRA_TS_NONE32 ? ~0ull : a;
            c.r_step_ts[4 * (size_t)s + 1] = c.issued_cnt[s] == n ? (u64)c.t_issued[s] : ~0ull;
            c.r_step_ts[4 * (size_t)s + 2] = c.deliv_cnt[s] == n ? (u64)c.t_deliv[s] : ~0ull;
            c.r_step_ts[4 * (size_t)s + 3] = c.ack_cnt[s] == n ? (u64)c.t_ack[s] : ~0ull;
        }
        for (u32 e = tid; e < c.E; e += nthr) c.r_link_lines[e] = c.link_lines[e];
        if (tid == 0) {
            DeviceSummary sm;
            sm.status = status; sm.n_steps = c.S; sm.n_links = c.E; sm.window = W;
            sm.completion_cycle = ctl.completion; sm.total_lines = P.total_lines;
            sm.busy_cycles = busy; sm.skipped_cycles = skipped;
            *c.r_summary = sm;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
static size_t smem_bytes(u32 warps) {
    return ((sizeof(Ctx) + 15) & ~size_t(15)) + ((sizeof(Ctl) + 15) & ~size_t(15)) +
           (size_t)warps * SCR_WORDS * sizeof(u32);
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
