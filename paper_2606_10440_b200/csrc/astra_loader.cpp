// astra_loader.cpp -- host loader of the engine (untimed prep):
// validation (include/astra.h rules), min-latency routing with the (dst mod k) tie-break (R5,
// PAPER.md:L221 "modular routing function"), successor CSR of the step DAG (R3), per-CU in-order
// step lists and quota split (R11), link ring capacities, link service kinds (R9), the per-window
// staging cells that fix the same-cycle FIFO append order (R7/R8), the lookahead window, and the
// SoA workspace layout.
//
// Independent of oracle/: the oracle routes with Bellman-Ford sweeps, this file with a heap
// Dijkstra; they share no code.
#include "astra_internal.h"
#include "../../include/astra.h"

#include <algorithm>
#include <cstring>
#include <queue>

u64 Blob::add(const void* p, size_t n) {
    size_t off = (bytes.size() + 15) & ~size_t(15);
    bytes.resize(off + n);
    if (n) std::memcpy(bytes.data() + off, p, n);
    return off;
}

static u32 pow2ceil(u64 x) { u32 p = 1; while ((u64)p < x && p < (1u << 31)) p <<= 1; return p; }

// ---------------------------------------------------------------------------------------------
// Topology: validation, effective latencies (R4), routing (R5), candidate tables
// ---------------------------------------------------------------------------------------------
int32_t astra_build_topo(HostTopo& t, std::string& err) {
    const u32 V = t.G + t.NS;
    t.V = V;
    if (t.G < 1) { err = "n_gpus must be >= 1"; return ASTRA_EINVAL; }
    if (t.G > ASTRA_MAX_GPUS) { err = "too many GPUs"; return ASTRA_ELIMIT; }
    if (t.row_ptr.size() != (size_t)V + 1 || t.row_ptr[0] != 0) { err = "row_ptr malformed"; return ASTRA_EINVAL; }
    for (u32 v = 0; v < V; v++)
        if (t.row_ptr[v + 1] < t.row_ptr[v]) { err = "row_ptr not monotone"; return ASTRA_EINVAL; }
    t.E = t.row_ptr[V];
    if (t.E >= (1u << 22)) { err = "too many links"; return ASTRA_ELIMIT; }
    if (t.head.size() != t.E || t.bw.size() != t.E || t.lat.size() != t.E) { err = "link arrays wrong size"; return ASTRA_EINVAL; }
    t.tail.assign(t.E, 0); t.leff.assign(t.E, 0);
    t.min_leff = 0xffffffffu; t.max_leff = 0;
    for (u32 v = 0; v < V; v++) {
        for (u32 e = t.row_ptr[v]; e < t.row_ptr[v + 1]; e++) {
            if (t.head[e] >= V || t.head[e] == v) { err = "link head out of range or self loop"; return ASTRA_EINVAL; }
            if (e > t.row_ptr[v] && t.head[e] <= t.head[e - 1]) { err = "heads not strictly ascending in a row"; return ASTRA_EINVAL; }
            if (t.bw[e] == 0 || t.lat[e] == 0) { err = "zero bandwidth or latency"; return ASTRA_EINVAL; }
            if (t.bw[e] > ASTRA_MAX_BW_Q8) { err = "bandwidth above ASTRA_MAX_BW_Q8"; return ASTRA_ELIMIT; }
            u64 le = (u64)t.lat[e] + t.node_lat[t.head[e]];
            if (le >= ASTRA_MAX_LINK_LATENCY) { err = "latency above ASTRA_MAX_LINK_LATENCY"; return ASTRA_ELIMIT; }
            t.tail[e] = v; t.leff[e] = (u32)le;
            t.min_leff = std::min(t.min_leff, (u32)le); t.max_leff = std::max(t.max_leff, (u32)le);
        }
    }
    if (t.E == 0) { t.min_leff = 1; t.max_leff = 1; }
    // in-links per head node, ascending link id (counting sort keeps id order)
    t.in_ptr.assign(V + 1, 0);
    for (u32 e = 0; e < t.E; e++) t.in_ptr[t.head[e] + 1]++;
    for (u32 v = 0; v < V; v++) t.in_ptr[v + 1] += t.in_ptr[v];
    t.in_link.assign(t.E, 0);
    { std::vector<u32> fill(V, 0); for (u32 e = 0; e < t.E; e++) { u32 h = t.head[e]; t.in_link[t.in_ptr[h] + fill[h]++] = e; } }

    // Dijkstra towards every destination GPU over reversed links
    const u32 G = t.G;
    t.dist.assign((size_t)V * G, 0xffffffffu);
    t.next_link.assign((size_t)V * G, 0xffffffffu);
    std::vector<u64> d(V);
    typedef std::pair<u64, u32> QE;
    for (u32 dst = 0; dst < G; dst++) {
        std::fill(d.begin(), d.end(), ~0ull);
        std::priority_queue<QE, std::vector<QE>, std::greater<QE>> pq;
        d[dst] = 0; pq.push(QE(0, dst));
        while (!pq.empty()) {
            QE top = pq.top(); pq.pop();
            u32 v = top.second;
            if (top.first != d[v]) continue;
            for (u32 i = t.in_ptr[v]; i < t.in_ptr[v + 1]; i++) {
                u32 e = t.in_link[i], u = t.tail[e];
                u64 nd = top.first + t.leff[e];
                if (nd < d[u]) { d[u] = nd; pq.push(QE(nd, u)); }
            }
        }
        for (u32 v = 0; v < V; v++) {
            if (d[v] == ~0ull) continue;
            if (d[v] >= 0xfffffff0ull) { err = "route latency overflows 32 bits"; return ASTRA_ELIMIT; }
            t.dist[(size_t)v * G + dst] = (u32)d[v];
            if (v == dst) continue;
            u32 k = 0;
            for (u32 e = t.row_ptr[v]; e < t.row_ptr[v + 1]; e++)
                if (d[t.head[e]] != ~0ull && d[t.head[e]] + t.leff[e] == d[v]) k++;
            u32 want = dst % k, idx = 0;
            for (u32 e = t.row_ptr[v]; e < t.row_ptr[v + 1]; e++)
                if (d[t.head[e]] != ~0ull && d[t.head[e]] + t.leff[e] == d[v]) {
                    if (idx == want) { t.next_link[(size_t)v * G + dst] = e; break; }
                    idx++;
                }
        }
    }
    return ASTRA_OK;
}

// ---------------------------------------------------------------------------------------------
// Collective: validation (R3) and successor CSR
// ---------------------------------------------------------------------------------------------
int32_t astra_build_coll(HostColl& c, std::string& err) {
    const u32 S = c.S, G = c.G;
    if (G < 1 || G > ASTRA_MAX_GPUS) { err = "bad n_gpus"; return G < 1 ? ASTRA_EINVAL : ASTRA_ELIMIT; }
    if (S >= ASTRA_MAX_STEPS) { err = "too many steps"; return ASTRA_ELIMIT; }
    if (c.dep_ptr.size() != (size_t)S + 1 || c.dep_ptr[0] != 0) { err = "dep_ptr malformed"; return ASTRA_EINVAL; }
    c.total_lines = 0; c.max_cu_end = 0;
    for (u32 s = 0; s < S; s++) {
        if (c.owner[s] >= G || c.dst[s] >= G || c.owner[s] == c.dst[s]) { err = "bad owner/dst"; return ASTRA_EINVAL; }
        if (c.lines[s] == 0 || c.cu_n[s] == 0) { err = "zero lines or cu_n"; return ASTRA_EINVAL; }
        if ((u64)c.cu_lo[s] + c.cu_n[s] > ASTRA_MAX_WAVEFRONTS) { err = "CU range too large"; return ASTRA_ELIMIT; }
        if (c.dep_ptr[s + 1] < c.dep_ptr[s] || c.dep_ptr[s + 1] > c.dep_step.size()) { err = "dep_ptr not monotone"; return ASTRA_EINVAL; }
        c.max_cu_end = std::max(c.max_cu_end, c.cu_lo[s] + c.cu_n[s]);
        c.total_lines += c.lines[s];
        for (u32 i = c.dep_ptr[s]; i < c.dep_ptr[s + 1]; i++) {
            u32 p = c.dep_step[i]; u32 k = c.dep_kind[i];
            if (p >= s) { err = "dependency id must be < step id"; return ASTRA_EINVAL; }
            if (k == ASTRA_DEP_DELIVERED) { if (c.dst[p] != c.owner[s]) { err = "DELIVERED dep not local"; return ASTRA_EINVAL; } }
            else if (k == ASTRA_DEP_ACKED || k == ASTRA_DEP_ISSUED) { if (c.owner[p] != c.owner[s]) { err = "ACKED/ISSUED dep not local"; return ASTRA_EINVAL; } }
            else { err = "unknown dependency kind"; return ASTRA_EINVAL; }
        }
    }
    // successor lists, duplicates (same producer, same kind) collapsed
    std::vector<std::vector<u32>> succ(S);
    c.ndeps.assign(S, 0);
    for (u32 s = 0; s < S; s++) {
        std::vector<u32> seen;
        for (u32 i = c.dep_ptr[s]; i < c.dep_ptr[s + 1]; i++) {
            u32 key = c.dep_step[i] | ((u32)c.dep_kind[i] << 30);
            if (std::find(seen.begin(), seen.end(), key) != seen.end()) continue;
            seen.push_back(key);
            succ[c.dep_step[i]].push_back(s | ((u32)c.dep_kind[i] << 30));
            c.ndeps[s]++;
        }
    }
    c.succ_ptr.assign(S + 1, 0); c.succ.clear();
    for (u32 s = 0; s < S; s++) { c.succ_ptr[s] = (u32)c.succ.size(); c.succ.insert(c.succ.end(), succ[s].begin(), succ[s].end()); }
    c.succ_ptr[S] = (u32)c.succ.size();
    return ASTRA_OK;
}

// ---------------------------------------------------------------------------------------------
// Plan one design point: plan tables into the blob, workspace layout into the descriptor.
// topo_off / coll_off are the blob offsets of the shared topology / collective tables.
//
// Staging cells (R7/R8).  The same-cycle append order into a link FIFO is fixed: transit lines
// by ascending in-link id of the node, each in pipe order, then the node's own injections by
// ascending wavefront id.  The engine gives every out-link of node v one cell per cycle of the
// window with a FIXED slot layout: in-link i of v owns ceil(B_i) consecutive slots (a link
// delivers at most ceil(B) lines per cycle), then H slots for injections (at most H issues per
// GPU per cycle).  A line's slot is therefore known without any atomic allocation, and reading
// a cell's occupied slots in slot order IS the FIFO order.
// ---------------------------------------------------------------------------------------------
int32_t astra_plan_point(const HostTopo& t, const HostColl& c, const HostGpu& g, u64 flags, u64 max_cycles,
                         const u64* topo_off, const u64* coll_off, Blob& blob, PointDesc& P, double& cost,
                         std::string& err) {
    std::memset(&P, 0, sizeof(P));
    const u32 G = t.G, V = t.V, E = t.E, S = c.S;
    if (c.G != G) { err = "collective and topology disagree on n_gpus"; return ASTRA_EINVAL; }
    if (c.max_cu_end > g.C) { err = "a step's CU range exceeds the GPU's CUs"; return ASTRA_EINVAL; }
    const u32 CW = g.C * g.Wv;
    const u32 slots = CW * g.K;
    P.G = G; P.V = V; P.E = E; P.S = S; P.C = g.C; P.Wv = g.Wv; P.K = g.K; P.H = g.H;
    P.CW = CW; P.nwords = (CW + 31) / 32; P.slots = slots; P.bmwords = (slots + 31) / 32;
    P.kdiv_magic = (u32)(((1ull << 32) + g.K - 1) / g.K);
    P.total_lines = c.total_lines;
    P.flags = (u32)flags;
    u64 tmax = std::min<u64>(max_cycles, 0xffffffffull - (1u << 25));
    P.max_cycles = tmax;

    // lookahead window: largest power of two <= min Leff, capped
    u32 logW = 0;
    if (!(flags & ASTRA_FLAG_WINDOW_1)) {
        while ((2u << logW) <= t.min_leff && logW + 1 <= ASTRA_WMAX_LOG2) logW++;
    }
    P.logW = logW;
    const u32 W = 1u << logW;
    const u32 NC = W + 1;
    P.NC = NC;

    std::vector<u32> step_q(S), step_r(S), first_link(S), step_alpha(S);
    u32 alpha_max = 1;
    for (u32 s = 0; s < S; s++) {
        u32 a = t.dist[(size_t)c.owner[s] * G + c.dst[s]];
        if (a == 0xffffffffu) { err = "a step's owner has no route to its dst"; return ASTRA_EUNREACHABLE; }
        step_alpha[s] = a; alpha_max = std::max(alpha_max, a);
        first_link[s] = t.next_link[(size_t)c.owner[s] * G + c.dst[s]];
        u32 m = c.cu_n[s] * g.Wv;
        step_q[s] = c.lines[s] / m; step_r[s] = c.lines[s] % m;
    }
    u64 nw64 = pow2ceil((u64)(alpha_max + W - 1) / W + 2);
    if (nw64 > ASTRA_NW_MAX) { err = "route latency / lookahead window ratio above the engine limit"; return ASTRA_ELIMIT; }
    P.NW = (u32)nw64;

    // per-CU in-order step lists (R11), per-owner release-list regions, per-GPU event-list regions
    std::vector<u32> cul_ptr((size_t)G * g.C + 1, 0), rel_off(G + 1, 0), ev_off(G + 1, 0);
    for (u32 s = 0; s < S; s++) {
        for (u32 cu = c.cu_lo[s]; cu < c.cu_lo[s] + c.cu_n[s]; cu++) cul_ptr[(size_t)c.owner[s] * g.C + cu + 1]++;
        rel_off[c.owner[s] + 1]++;
        ev_off[c.owner[s] + 1]++; ev_off[c.dst[s] + 1]++;     // one ACKED event at the owner, one DELIVERED at dst
    }
    for (size_t i = 0; i < (size_t)G * g.C; i++) cul_ptr[i + 1] += cul_ptr[i];
    for (u32 i = 0; i < G; i++) { rel_off[i + 1] += rel_off[i]; ev_off[i + 1] += ev_off[i]; }
    std::vector<u32> cul(cul_ptr.back());
    {
        std::vector<u32> fill((size_t)G * g.C, 0);
        for (u32 s = 0; s < S; s++)
            for (u32 cu = c.cu_lo[s]; cu < c.cu_lo[s] + c.cu_n[s]; cu++) {
                size_t k = (size_t)c.owner[s] * g.C + cu;
                cul[cul_ptr[k] + fill[k]++] = s;
            }
    }
    std::vector<u32> init_rel(S ? S : 1, 0), init_rel_cnt(G, 0);
    for (u32 s = 0; s < S; s++)
        if (c.ndeps[s] == 0) { u32 o = c.owner[s]; init_rel[rel_off[o] + init_rel_cnt[o]++] = s; }

    // ring capacities: lines that can sit in / fly over link e are bounded by the outstanding
    // lines of the owners routed through it.
    std::vector<u64> bound(E, 0);
    {
        std::vector<std::vector<u32>> by_owner(G);
        for (u32 s = 0; s < S; s++) by_owner[c.owner[s]].push_back(s);
        std::vector<u64> via(E, 0); std::vector<u32> touched;
        for (u32 o = 0; o < G; o++) {
            touched.clear();
            for (u32 s : by_owner[o]) {
                u32 v = o, d = c.dst[s], hops = 0;
                while (v != d) {
                    u32 e = t.next_link[(size_t)v * G + d];
                    if (via[e] == 0) touched.push_back(e);
                    via[e] += c.lines[s];
                    v = t.head[e];
                    if (++hops > V) { err = "routing loop"; return ASTRA_EINVAL; }
                }
                cost += (double)c.lines[s] * hops;
            }
            for (u32 e : touched) { bound[e] += std::min<u64>(slots, via[e]); via[e] = 0; }
        }
    }
    // staging cells: slot layout per node, regions per link
    std::vector<u32> nd_cellcap(V), nd_mw(V), nd_injoff(V), classoff(E, 0);
    for (u32 v = 0; v < V; v++) {
        u32 off = 0;
        for (u32 i = t.in_ptr[v]; i < t.in_ptr[v + 1]; i++) {
            u32 e = t.in_link[i];
            classoff[e] = off;
            off += (t.bw[e] + 255) / 256;
        }
        nd_injoff[v] = off;
        nd_cellcap[v] = off + (v < G ? g.H : 0);
        if (nd_cellcap[v] == 0) nd_cellcap[v] = 1;
        nd_mw[v] = (nd_cellcap[v] + 31) / 32;
    }
    std::vector<u32> ring_off(E), ring_mask(E), lkind(E), ceilb_v(E), credit_cap(E), lstate0(E), stage_off(E), mask_off(E);
    u64 ring_total = 0, stage_total = 0, mask_total = 0;
    for (u32 e = 0; e < E; e++) {
        u32 ceilb = (t.bw[e] + 255) / 256;
        ceilb_v[e] = ceilb;
        credit_cap[e] = ceilb * 256;
        if (t.bw[e] % 256 == 0) { lkind[e] = ASTRA_LK_INT | ((t.bw[e] / 256) << 2); lstate0[e] = 0; }
        else if (256 % t.bw[e] == 0) { lkind[e] = ASTRA_LK_PERIOD | ((256 / t.bw[e]) << 2); lstate0[e] = 0; }   // next accept not before cycle 0
        else { lkind[e] = ASTRA_LK_GENERAL | (t.bw[e] << 2); lstate0[e] = credit_cap[e]; }
        u32 rc = std::max<u32>(32, pow2ceil(bound[e]));
        if (ring_total + rc >= (1ull << 32)) { err = "ring space exceeds 2^32 entries"; return ASTRA_ELIMIT; }
        ring_off[e] = (u32)ring_total; ring_mask[e] = rc - 1; ring_total += rc;
        u32 v = t.tail[e];
        u64 st = (u64)NC * nd_cellcap[v], mk = (u64)NC * nd_mw[v];
        if (stage_total + st >= (1ull << 32)) { err = "staging space exceeds 2^32 entries"; return ASTRA_ELIMIT; }
        stage_off[e] = (u32)stage_total; stage_total += st;
        mask_off[e] = (u32)mask_total; mask_total += mk;
    }

    // constant tables
    P.c_in_ptr = topo_off[0]; P.c_in_link = topo_off[1]; P.c_head = topo_off[2]; P.c_tail = topo_off[3];
    P.c_leff = topo_off[4]; P.c_bw = topo_off[5]; P.c_next_link = topo_off[6];
    P.c_step_od = coll_off[0]; P.c_lines = coll_off[1]; P.c_cu_lo = coll_off[2]; P.c_cu_n = coll_off[3];
    P.c_succ_ptr = coll_off[4]; P.c_succ = coll_off[5]; P.c_ndeps = coll_off[6];
    P.c_step_q = blob.add(step_q); P.c_step_r = blob.add(step_r); P.c_first_link = blob.add(first_link);
    P.c_step_alpha = blob.add(step_alpha); P.c_cul_ptr = blob.add(cul_ptr); P.c_cul = blob.add(cul);
    P.c_rel_off = blob.add(rel_off); P.c_init_rel = blob.add(init_rel); P.c_init_rel_cnt = blob.add(init_rel_cnt);
    P.c_ev_off = blob.add(ev_off);
    P.c_ring_off = blob.add(ring_off); P.c_ring_mask = blob.add(ring_mask); P.c_lkind = blob.add(lkind);
    P.c_ceilb = blob.add(ceilb_v); P.c_lstate0_init = blob.add(lstate0);
    P.c_stage_off = blob.add(stage_off); P.c_mask_off = blob.add(mask_off); P.c_classoff = blob.add(classoff);
    P.c_nd_cellcap = blob.add(nd_cellcap); P.c_nd_mw = blob.add(nd_mw); P.c_nd_injoff = blob.add(nd_injoff);

    // workspace layout
    u64 off = 0;
    auto take = [&](u64 bytes) { u64 o = off; off = (off + bytes + 15) & ~15ull; return o; };
    const u64 GW = (u64)G * CW;
    const u32 nw = P.NW;
    // zero region
    P.w_pipe_head = take(4ull * E); P.w_fifo_head = take(4ull * E); P.w_tail = take(4ull * E);
    P.w_lstate1 = take(4ull * E); P.w_link_lines = take(4ull * E); P.w_masks = take(4ull * mask_total);
    P.w_issued_cnt = take(4ull * S); P.w_t_issued = take(4ull * S); P.w_deliv_cnt = take(4ull * S);
    P.w_t_deliv = take(4ull * S); P.w_ack_cnt = take(4ull * S); P.w_t_ack = take(4ull * S); P.w_rel_time = take(4ull * S);
    P.w_wf_busy = take(8ull * GW); P.w_want = take(4ull * G * P.nwords);
    P.w_bitmap = take(4ull * G * nw * P.bmwords); P.w_bin_cnt = take(4ull * G * nw);
    P.w_ack_n = take(4ull * G); P.w_ev_cnt = take(4ull * G);
    P.ws_zero_bytes = off;
    // 0xff region
    P.ws_ff_off = off;
    P.w_wf_rem = take(4ull * GW);
    P.ws_ff_bytes = off - P.ws_ff_off;
    // specially initialised
    P.w_lstate0 = take(4ull * E); P.w_t_release = take(4ull * S); P.w_ndep_left = take(4ull * S);
    P.w_wf_cur = take(4ull * GW); P.w_freeb = take(4ull * G * P.nwords);
    P.w_plist = take(4ull * (S ? S : 1)); P.w_pcnt = take(4ull * G);
    // uninitialised
    P.w_ring = take(8ull * ring_total); P.w_stage = take(8ull * stage_total);
    P.w_sel = take(4ull * G * g.H);
    P.w_ack_rec = take(8ull * G * slots); P.w_ack_tmp = take(8ull * G * slots); P.w_ack_sorted = take(8ull * G * slots);
    P.w_ev_list = take(4ull * (ev_off[G] ? ev_off[G] : 1));
    P.ws_bytes = off;
    return ASTRA_OK;
}
