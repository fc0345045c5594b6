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

// Cost proxy of a design point for the scheduler (A0): lookahead windows it will step through
// (bottleneck link occupancy / window) and line-hop events.  Only ratios between points matter.
double astra_point_cost(const HostTopo& t, const HostColl& c, u64 flags) {
    const u32 G = t.G, E = t.E;
    std::vector<u64> via(E, 0);
    double events = 0;
    u64 alpha_max = 1;
    for (u32 s = 0; s < c.S; s++) {
        u32 v = c.owner[s], d = c.dst[s], hops = 0;
        if (v >= G || d >= G || t.dist[(size_t)v * G + d] == 0xffffffffu) continue;
        alpha_max = std::max<u64>(alpha_max, t.dist[(size_t)v * G + d]);
        while (v != d && hops <= t.V) { u32 e = t.next_link[(size_t)v * G + d]; via[e] += c.lines[s]; v = t.head[e]; hops++; }
        events += (double)c.lines[s] * (hops + 2);
    }
    double cycles = 0;
    for (u32 e = 0; e < E; e++) cycles = std::max(cycles, (double)via[e] * 256.0 / t.bw[e]);
    cycles += 4.0 * alpha_max;
    u32 W = 1;
    if (!(flags & ASTRA_FLAG_WINDOW_1)) { W = std::max<u32>(1, std::min<u32>(t.min_leff, (u32)ASTRA_WMAX)); if (W >= 64) W &= ~63u; }
    // measured: a window costs a CTA about 20 k clocks plus 3.5 k per GPU and per link it steps; events are cheap
    return cycles / W * (20000.0 + 3500.0 * (t.G + E)) + events * 10.0;
}

// ---------------------------------------------------------------------------------------------
// Plan one design point: plan tables into the blob, array placement into the descriptor.
// topo_off / coll_off are the blob offsets of the shared topology / collective tables.
//
// Append order (R7/R8).  The same-cycle append order into a link FIFO is fixed: transit lines
// by ascending in-link id of the node, each in pipe order, then the node's own injections by
// ascending wavefront id.  An out-link that only ever receives lines from ONE feeder (one in-link
// or the node's own injections, decided here by walking every step's route) is appended to
// directly by that feeder.  Every other out-link of node v gets one cell per cycle of the window
// with a FIXED slot layout: in-link i of v owns ceil(B_i) consecutive slots (a link delivers at
// most ceil(B) lines per cycle), then H slots for injections (at most H issues per GPU per
// cycle).  A line's slot is known without any atomic allocation; one bit per slot is kept, and
// the prefix sum of the popcounts in (cycle, slot) order IS the FIFO position.
// ---------------------------------------------------------------------------------------------
int32_t astra_plan_point(const HostTopo& t, const HostColl& c, const HostGpu& g, const PlanOptions& opt,
                         const u64* topo_off, const u64* coll_off, Blob& blob, PointDesc& P, double& cost,
                         std::string& err) {
    std::memset(&P, 0, sizeof(P));
    const u32 G = t.G, V = t.V, E = t.E, S = c.S;
    if (c.G != G) { err = "collective and topology disagree on n_gpus"; return ASTRA_EINVAL; }
    if (c.max_cu_end > g.C) { err = "a step's CU range exceeds the GPU's CUs"; return ASTRA_EINVAL; }
    const u32 CW = g.C * g.Wv;
    const u32 slots = CW * g.K;
    const u32 group = std::max<u32>(1, opt.group);
    P.G = G; P.V = V; P.E = E; P.S = S; P.C = g.C; P.Wv = g.Wv; P.K = g.K; P.H = g.H;
    P.CW = CW; P.nwords = (CW + 31) / 32; P.slots = slots; P.bmwords = (slots + 31) / 32;
    P.kdiv_magic = (u32)(((1ull << 32) + g.K - 1) / g.K);
    P.total_lines = c.total_lines;
    P.flags = (u32)opt.flags;
    P.group = group;
    P.pcu = g.mode & 3u;
    u64 tmax = std::min<u64>(opt.max_cycles, ASTRA_MAX_CYCLES);       // documented clamp (include/astra.h)
    P.max_cycles = tmax;

    // lookahead window: min Leff (any value, not only powers of two), capped
    u32 W = 1;
    if (!(opt.flags & ASTRA_FLAG_WINDOW_1)) {
        W = std::max<u32>(1, std::min<u32>(t.min_leff, (u32)ASTRA_WMAX));
        if (W >= 64) W &= ~63u;                 // whole 32-entry chunks per link and window at the usual bandwidths
    }
    P.Wcyc = W;
    const u32 NC = W + 1;
    P.NC = NC;

    std::vector<u32> step_q(S), step_r(S), first_link(S), step_alpha(S), step_aq(S), step_ar(S);
    u32 alpha_max = 1;
    for (u32 s = 0; s < S; s++) {
        u32 a = t.dist[(size_t)c.owner[s] * G + c.dst[s]];
        if (a == 0xffffffffu) { err = "a step's owner has no route to its dst"; return ASTRA_EUNREACHABLE; }
        step_alpha[s] = a; alpha_max = std::max(alpha_max, a);
        step_aq[s] = a / W; step_ar[s] = a % W;             // ack window = delivery window + aq + (d + ar >= W)
        first_link[s] = t.next_link[(size_t)c.owner[s] * G + c.dst[s]];
        u32 m = c.cu_n[s] * g.Wv;
        step_q[s] = c.lines[s] / m; step_r[s] = c.lines[s] % m;
    }
    // ASTRA_FLAG_RUN_AHEAD: one-CTA points of up to 32 nodes let a node run ahead of the nodes it does not depend on, at
    // most two windows apart (step_kernel_body): one more window bin, 2 W ceil(B) more ring entries per link for the
    // lagging reader.
    bool run_ahead = group == 1 && V <= 32 && (opt.flags & ASTRA_FLAG_RUN_AHEAD);
    if (run_ahead && pow2ceil((u64)(alpha_max + W - 1) / W + 3) > ASTRA_NW_MAX) run_ahead = false;     // no room for the extra bin
    P.run_ahead = run_ahead ? 1u : 0u;
    u64 nw64 = pow2ceil((u64)(alpha_max + W - 1) / W + (run_ahead ? 3 : 2));
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

    // Walk every step's route: ring capacities (lines that can sit in / fly over link e are bounded
    // by the outstanding lines of the owners routed through it), feeders of every link, node loads.
    std::vector<u64> bound(E, 0);
    std::vector<u32> feeder(E, ASTRA_NONE32);       // first feeder seen: in-link id, or E for injections
    std::vector<uint8_t> multi(E, 0);
    std::vector<uint8_t> delivers(E, 0), transits(E, 0), multi_fwd(E, 0);
    std::vector<u32> fwd(E, ASTRA_NONE32);       // the one link that lines arriving over e are forwarded to
    std::vector<double> load(V, 0.0);
    std::vector<u64> via_tot(E, 0);                 // lines routed over every link, all owners
    double t_win = 1.0;                             // run length if only the outstanding caps bound it (cycles)
    {
        std::vector<std::vector<u32>> by_owner(G);
        for (u32 s = 0; s < S; s++) by_owner[c.owner[s]].push_back(s);
        std::vector<u64> via(E, 0); std::vector<u32> touched;
        for (u32 o = 0; o < G; o++) {
            touched.clear();
            double t_own = 0.0;
            for (u32 s : by_owner[o]) {
                u32 v = o, d = c.dst[s], hops = 0, prev = E;
                while (v != d) {
                    u32 e = t.next_link[(size_t)v * G + d];
                    if (via[e] == 0) touched.push_back(e);
                    via[e] += c.lines[s];
                    if (feeder[e] == ASTRA_NONE32) feeder[e] = prev;
                    else if (feeder[e] != prev) multi[e] = 1;
                    load[v] += c.lines[s]; load[t.head[e]] += c.lines[s];
                    if (t.head[e] == d) delivers[e] = 1;
                    else {
                        transits[e] = 1;
                        u32 e2 = t.next_link[(size_t)t.head[e] * G + d];
                        if (fwd[e] == ASTRA_NONE32) fwd[e] = e2; else if (fwd[e] != e2) multi_fwd[e] = 1;
                    }
                    prev = e;
                    v = t.head[e];
                    if (++hops > V) { err = "routing loop"; return ASTRA_EINVAL; }
                }
                load[o] += 2.0 * c.lines[s];
                t_own += (double)c.lines[s] * (2.0 * step_alpha[s] + 1.0) / (double)slots;
                cost += (double)c.lines[s] * hops;
            }
            for (u32 e : touched) { bound[e] += std::min<u64>(slots, via[e]); via_tot[e] += via[e]; via[e] = 0; }
            t_win = std::max(t_win, t_own);
        }
    }
    // cells: slot layout per node, cell and prefix regions per multi-feeder link
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
    // A multi-feeder link whose cells are expected to be mostly empty keeps a bitmap of the non-empty ones (see cell_set).
    // Estimate: run length = the longer of the bottleneck link's occupancy and the outstanding-cap bound; a link with
    // via lines over that time sees them in bursts of ceil(B) per cycle, so about via / (ceil(B) * cycles) of its cells
    // are marked.  Sparse below 1/8.  (Performance only: both paths give the same result.)
    std::vector<uint8_t> sparse_cells(E, 0);
    {
        double t_bw = 1.0;
        for (u32 e = 0; e < E; e++) t_bw = std::max(t_bw, (double)via_tot[e] * 256.0 / t.bw[e]);
        const double t_run = std::max(t_bw, t_win);
        for (u32 e = 0; e < E; e++) {
            const double cb_ = std::max(1.0, t.bw[e] / 256.0);
            sparse_cells[e] = (double)via_tot[e] / (cb_ * t_run) < ASTRA_SPARSE_CELLS_BELOW;
        }
    }
    std::vector<u32> ring_off(E), ring_mask(E), lkind(E), ceilb_v(E), lstate0(E), mask_off(E), pre_off(E), nz_off(E, ASTRA_NONE32), inj_off(G + 1, 0);
    u64 ring_total = 0, mask_total = 0, pre_total = 0, nz_total = 0;
    const u32 NZW = (NC + 31) / 32;            // words of a link's bitmap of non-empty cells (one bit per cycle of the window)
    for (u32 e = 0; e < E; e++) {
        u32 ceilb = (t.bw[e] + 255) / 256;
        ceilb_v[e] = ceilb;
        if (t.bw[e] % 256 == 0) { lkind[e] = ASTRA_LK_INT | ((t.bw[e] / 256) << 2); lstate0[e] = 0; }
        else if (256 % t.bw[e] == 0) { lkind[e] = ASTRA_LK_PERIOD | ((256 / t.bw[e]) << 2); lstate0[e] = 0; }   // next accept not before cycle 0
        else { lkind[e] = ASTRA_LK_GENERAL | (t.bw[e] << 2); lstate0[e] = ceilb * 256; }
        // a group's writer checks the ring against a reader cursor that may lag one window: 2x
        u32 rc = std::max<u32>(32, pow2ceil(run_ahead ? bound[e] + 2ull * W * ceilb : bound[e] * (group > 1 ? 2 : 1)));
        if (ring_total + rc >= (1ull << 32)) { err = "ring space exceeds 2^32 entries"; return ASTRA_ELIMIT; }
        ring_off[e] = (u32)ring_total; ring_mask[e] = rc - 1; ring_total += rc;
        u32 v = t.tail[e];
        if (multi[e]) {
            u64 mk = (u64)NC * nd_mw[v];
            if (mask_total + mk >= (1ull << 31) || pre_total + NC >= (1ull << 31)) { err = "cell space exceeds 2^31 words"; return ASTRA_ELIMIT; }
            mask_off[e] = (u32)mask_total; mask_total += mk;
            pre_off[e] = (u32)pre_total; pre_total += NC;
            if (sparse_cells[e]) { nz_off[e] = (u32)nz_total; nz_total += NZW; }
            if (v < G) inj_off[v + 1] = g.H * (W + 2);
        } else { mask_off[e] = ASTRA_NONE32; pre_off[e] = ASTRA_NONE32; }
    }
    for (u32 i = 0; i < G; i++) inj_off[i + 1] += inj_off[i];

    // node ranges of the CTAs of the group: contiguous, balanced by the lines each node handles
    std::vector<u32> part(group + 1, V);
    if (group >= V) {
        for (u32 j = 0; j <= group; j++) part[j] = std::min(j, V);     // one node per CTA
    } else {
        // contiguous ranges; the smallest bottleneck load is found by bisection over a greedy fill
        std::vector<double> w(V);
        double total = 0, wmax = 0;
        for (u32 v = 0; v < V; v++) { w[v] = load[v] + 1.0; total += w[v]; wmax = std::max(wmax, w[v]); }
        double lo = std::max(wmax, total / group), hi = total;
        auto fill = [&](double cap, std::vector<u32>* out) {
            u32 j = 1; double acc = 0;
            if (out) (*out)[0] = 0;
            for (u32 v = 0; v < V; v++) {
                if (acc + w[v] > cap && acc > 0) { if (j >= group) return false; if (out) (*out)[j] = v; j++; acc = 0; }
                acc += w[v];
            }
            if (out) for (; j <= group; j++) (*out)[j] = V;
            return true;
        };
        for (int it = 0; it < 50; it++) { double mid = 0.5 * (lo + hi); if (fill(mid, nullptr)) hi = mid; else lo = mid; }
        fill(hi, &part);
        part[group] = V;
        // The bottleneck is usually one heavy node (a switch), and the greedy fill then packs the light nodes
        // into few ranges and leaves CTAs without nodes.  A node costs its CTA time whatever its load (every
        // stage of a window is a chain of dependent accesses), so the spare CTAs take the largest ranges apart:
        // split the heaviest range with more than one node at its best balance point until every CTA has nodes.
        std::vector<u32> cuts;
        for (u32 j = 0; j <= group; j++) if (j == 0 || part[j] != part[j - 1]) cuts.push_back(part[j]);
        if (cuts.back() != V) cuts.push_back(V);
        std::vector<double> pre(V + 1, 0.0);
        for (u32 v = 0; v < V; v++) pre[v + 1] = pre[v] + w[v];
        while (cuts.size() - 1 < group) {
            size_t best = cuts.size(); double bw = -1.0;
            for (size_t j = 0; j + 1 < cuts.size(); j++)
                if (cuts[j + 1] - cuts[j] >= 2 && pre[cuts[j + 1]] - pre[cuts[j]] > bw) { bw = pre[cuts[j + 1]] - pre[cuts[j]]; best = j; }
            if (best == cuts.size()) break;
            u32 a = cuts[best], b = cuts[best + 1], cut = a + 1; double bal = 1e300;
            for (u32 m = a + 1; m < b; m++) {
                const double d = std::max(pre[m] - pre[a], pre[b] - pre[m]);
                if (d < bal) { bal = d; cut = m; }
            }
            cuts.insert(cuts.begin() + best + 1, cut);
        }
        for (u32 j = 0; j <= group; j++) part[j] = j < cuts.size() ? cuts[j] : V;
    }

    // all_merged[e]: every link that lines arriving over e are forwarded to has several feeders
    std::vector<uint8_t> all_merged(E, 1);
    for (u32 s = 0; s < S; s++) {
        u32 v = c.owner[s], d = c.dst[s];
        while (v != d) {
            u32 e = t.next_link[(size_t)v * G + d];
            u32 h = t.head[e];
            if (h != d && !multi[t.next_link[(size_t)h * G + d]]) all_merged[e] = 0;
            v = h;
        }
    }
    // per-link flags for the chunk-parallel arrival paths: every line over e terminates at head(e), or
    // every line over e is forwarded to the same single-feeder out-link
    std::vector<u32> lflag(E, 0), lfwd(E, 0);
    for (u32 e = 0; e < E; e++) {
        if (delivers[e] && !transits[e]) lflag[e] = ASTRA_LF_DELIVER_ONLY;
        else if (transits[e] && !delivers[e] && !multi_fwd[e] && !multi[fwd[e]]) { lflag[e] = ASTRA_LF_FORWARD_ONLY; lfwd[e] = fwd[e]; }
        else if (transits[e] && all_merged[e]) lflag[e] = ASTRA_LF_CELLS;
    }
    // links on the cell path record (out-link, cell slot) per line of a window for the placement pass: 20 + 12 bits
    std::vector<u32> lscr_off(E, 0);
    u64 lscr_total = 0;
    for (u32 e = 0; e < E; e++) {
        if (lflag[e] != ASTRA_LF_CELLS) continue;
        if (E >= (1u << 20) || nd_cellcap[t.head[e]] > 4096) { err = "too many links or cell slots for the merge path"; return ASTRA_ELIMIT; }
        lscr_off[e] = (u32)lscr_total;
        lscr_total += (u64)ceilb_v[e] * W;
        if (lscr_total >= (1ull << 31)) { err = "merge scratch exceeds 2^31 words"; return ASTRA_ELIMIT; }
    }
    // per-GPU flags: a GPU whose steps have ISSUED-kind successors always takes the cycle-serial issue path
    std::vector<u32> gflag(G, 0);
    for (u32 s = 0; s < S; s++)
        for (u32 i = c.succ_ptr[s]; i < c.succ_ptr[s + 1]; i++)
            if ((c.succ[i] >> 30) == ASTRA_DEP_ISSUED) gflag[c.owner[s]] |= ASTRA_GF_ISSUED_DEPS;
    if (g.mode & 3u) for (u32 q = 0; q < G; q++) gflag[q] |= ASTRA_GF_SERIAL;      // per-CU readings (R12', R2')

    // gdirect[g]: bit x set when out-link x of GPU g is single-feeder (the GPU appends its issues to it directly and
    // needs the per-cycle issue counts of that link); all ones for a GPU with more than 32 out-links
    std::vector<u32> gdirect(G, 0);
    for (u32 q = 0; q < G; q++) {
        const u32 e0 = t.row_ptr[q], deg = t.row_ptr[q + 1] - e0;
        if (deg > 32) { gdirect[q] = ~0u; continue; }
        for (u32 x = 0; x < deg; x++) if (!multi[e0 + x]) gdirect[q] |= 1u << x;
    }

    // predmask[v] (points of up to 32 nodes): the nodes whose window k - 1 must be complete before v starts window k --
    // the tails of v's in-links (lines, due counts) and the destinations of the steps v owns (their arrival stage
    // writes v's ack records and bins)
    std::vector<u32> predmask(V, 0);
    if (V <= 32) {
        for (u32 e = 0; e < E; e++) predmask[t.head[e]] |= 1u << t.tail[e];
        for (u32 s = 0; s < S; s++) predmask[c.owner[s]] |= 1u << c.dst[s];
        for (u32 v = 0; v < V; v++) predmask[v] &= ~(1u << v);
    }

    // constant tables
    u64* co = P.c_off;
    co[ASTRA_C_in_ptr] = topo_off[0]; co[ASTRA_C_in_link] = topo_off[1]; co[ASTRA_C_head] = topo_off[2];
    co[ASTRA_C_tail] = topo_off[3]; co[ASTRA_C_leff] = topo_off[4]; co[ASTRA_C_next_link] = topo_off[5];
    co[ASTRA_C_row_ptr] = topo_off[6];
    co[ASTRA_C_step_od] = coll_off[0]; co[ASTRA_C_lines] = coll_off[1]; co[ASTRA_C_cu_lo] = coll_off[2];
    co[ASTRA_C_cu_n] = coll_off[3]; co[ASTRA_C_succ_ptr] = coll_off[4]; co[ASTRA_C_succ] = coll_off[5];
    co[ASTRA_C_ndeps] = coll_off[6];
    co[ASTRA_C_step_q] = blob.add(step_q); co[ASTRA_C_step_r] = blob.add(step_r);
    co[ASTRA_C_first_link] = blob.add(first_link); co[ASTRA_C_step_alpha] = blob.add(step_alpha);
    co[ASTRA_C_step_aq] = blob.add(step_aq); co[ASTRA_C_step_ar] = blob.add(step_ar);
    co[ASTRA_C_cul_ptr] = blob.add(cul_ptr); co[ASTRA_C_cul] = blob.add(cul);
    co[ASTRA_C_rel_off] = blob.add(rel_off); co[ASTRA_C_init_rel] = blob.add(init_rel);
    co[ASTRA_C_init_rel_cnt] = blob.add(init_rel_cnt); co[ASTRA_C_ev_off] = blob.add(ev_off);
    co[ASTRA_C_ring_off] = blob.add(ring_off); co[ASTRA_C_ring_mask] = blob.add(ring_mask);
    co[ASTRA_C_lkind] = blob.add(lkind); co[ASTRA_C_ceilb] = blob.add(ceilb_v);
    co[ASTRA_C_lstate0_init] = blob.add(lstate0);
    co[ASTRA_C_mask_off] = blob.add(mask_off); co[ASTRA_C_pre_off] = blob.add(pre_off); co[ASTRA_C_nz_off] = blob.add(nz_off);
    co[ASTRA_C_classoff] = blob.add(classoff); co[ASTRA_C_nd_mw] = blob.add(nd_mw);
    co[ASTRA_C_nd_injoff] = blob.add(nd_injoff); co[ASTRA_C_inj_off] = blob.add(inj_off);
    co[ASTRA_C_part] = blob.add(part);
    co[ASTRA_C_predmask] = blob.add(predmask);
    co[ASTRA_C_gflag] = blob.add(gflag);
    co[ASTRA_C_gdirect] = blob.add(gdirect);
    co[ASTRA_C_lflag] = blob.add(lflag); co[ASTRA_C_lfwd] = blob.add(lfwd);
    co[ASTRA_C_lscr_off] = blob.add(lscr_off);

    // mutable arrays: sizes, then placement (shared memory in declaration order while it fits)
    const u64 GW = (u64)G * CW;
    u64* ab = P.a_bytes;
    for (u32 a : {ASTRA_A_pipe_head, ASTRA_A_fifo_head, ASTRA_A_ltail, ASTRA_A_run, ASTRA_A_lstate0, ASTRA_A_lstate1,
                  ASTRA_A_link_lines, ASTRA_A_dirty, ASTRA_A_ndue, ASTRA_A_tl_lo, ASTRA_A_tl_n, ASTRA_A_tl_base}) ab[a] = 4ull * E;
    ab[ASTRA_A_due_cnt] = 4ull * E * P.NW;
    ab[ASTRA_A_tbase] = 4ull * (E + 1);
    for (u32 a : {ASTRA_A_pcnt, ASTRA_A_ev_cnt, ASTRA_A_ack_n, ASTRA_A_inj_n}) ab[a] = 4ull * G;
    ab[ASTRA_A_want] = ab[ASTRA_A_freeb] = ab[ASTRA_A_amask] = 4ull * G * P.nwords;
    ab[ASTRA_A_gmode] = ab[ASTRA_A_nheavy] = ab[ASTRA_A_turn] = 4ull * G;
    ab[ASTRA_A_cnt] = 4ull * G * W;
    ab[ASTRA_A_undo_want] = ab[ASTRA_A_undo_freeb] = 4ull * G * P.nwords;
    ab[ASTRA_A_hist] = 4ull * ((u64)t.row_ptr[G] * W + 1);
    ab[ASTRA_A_evb] = 8ull * G * g.H * W;
    ab[ASTRA_A_sel] = 4ull * G * g.H;
    ab[ASTRA_A_masks] = 4ull * mask_total; ab[ASTRA_A_pre] = 4ull * pre_total; ab[ASTRA_A_nz] = 4ull * nz_total;
    for (u32 a : {ASTRA_A_t_release, ASTRA_A_issued_cnt, ASTRA_A_t_issued, ASTRA_A_deliv_cnt, ASTRA_A_t_deliv,
                  ASTRA_A_ack_cnt, ASTRA_A_t_ack, ASTRA_A_ndep_left, ASTRA_A_rel_time, ASTRA_A_plist}) ab[a] = 4ull * S;
    ab[ASTRA_A_ev_list] = 4ull * ev_off[G];
    ab[ASTRA_A_bin_cnt] = 4ull * G * P.NW;
    ab[ASTRA_A_cu_out] = (g.mode & 3u) ? 4ull * G * g.C : 0;
    ab[ASTRA_A_wf_busy] = ab[ASTRA_A_undo_busy] = 8ull * GW;
    ab[ASTRA_A_wf_rem] = ab[ASTRA_A_wf_cur] = ab[ASTRA_A_undo_rem] = ab[ASTRA_A_undo_cur] = ab[ASTRA_A_hlist] = 4ull * GW;
    ab[ASTRA_A_lscr] = 4ull * lscr_total;
    ab[ASTRA_A_bitmap] = 4ull * G * P.NW * P.bmwords;
    // Ack discovery: a list per (GPU, window bin) that deliveries append to -- or, when the bitmap of a bin is a
    // few 32-word chunks per warp of the node's set anyway, the scan of the bitmap itself (the append costs every
    // delivery the round trip of a counting atomic).
    {
        const u32 nodes_per_cta = (V + group - 1) / group;
        const u32 ws = std::max<u32>(1, 16 / std::min<u32>(16, nodes_per_cta));
        const u32 chunks = (P.bmwords + 31) / 32;
        P.alcap = chunks > 4 * ws ? std::min<u32>(slots, ASTRA_ACK_LIST_CAP) : 0u;
    }
    ab[ASTRA_A_ack_list] = 4ull * G * P.NW * P.alcap;      // 0 entries: no list
    ab[ASTRA_A_inj_list] = 8ull * inj_off[G];
    ab[ASTRA_A_ack_rec] = ab[ASTRA_A_ack_tmp] = ab[ASTRA_A_ack_sorted] = 8ull * G * slots;
    ab[ASTRA_A_ring] = 8ull * ring_total;
    // CTA groups: the arrays indexed by GPU (and hist, indexed by the GPUs' out-links) are kept per CTA for its own
    // GPUs only when that part fits in shared memory -- the whole point's arrays would crowd everything else out
    u32 maxG = 0, maxOut = 0;
    for (u32 r = 0; r < group; r++) {
        const u32 a0 = std::min(part[r], G), a1 = std::min(part[r + 1], G);
        maxG = std::max(maxG, a1 - a0); maxOut = std::max(maxOut, t.row_ptr[a1] - t.row_ptr[a0]);
    }
    u64 local_bytes[ASTRA_A_COUNT] = {0};
    if (group > 1) {
#define X(n, per_gpu, eb) local_bytes[ASTRA_A_##n] = (u64)(eb) * (per_gpu) * std::max<u32>(1, maxG);
        ASTRA_GPU_ARRAYS(X)
#undef X
        local_bytes[ASTRA_A_hist] = 4ull * ((u64)maxOut * W + 1);
    }
    u64 hot = 0, ws = 0;
    for (u32 a = 0; a < ASTRA_A_COUNT; a++) {
        if (local_bytes[a]) {
            const u64 lb = (std::max<u64>(local_bytes[a], 16) + 15) & ~15ull;
            if (hot + lb <= opt.hot_budget) { ab[a] = lb; P.a_off[a] = hot | ASTRA_PLACE_SMEM | ASTRA_PLACE_LOCAL; hot += lb; continue; }
        }
        ab[a] = (std::max<u64>(ab[a], 16) + 15) & ~15ull;
        // streamed arrays stay in global memory; so does, for a CTA group, what another CTA of the group
        // reads or writes: link cursors seen from both ends, ack records / bitmap / bin counts (written
        // at the destination, read at the owner).  Every other array is only ever touched by the CTA
        // that owns the node, so each CTA keeps its own shared-memory copy and uses its nodes' part.
        bool global_only = a == ASTRA_A_bitmap || a == ASTRA_A_ack_list || a == ASTRA_A_ack_rec || a == ASTRA_A_ack_tmp ||
                           a == ASTRA_A_ack_sorted || a == ASTRA_A_ring || a == ASTRA_A_evb ||
                           (group > 1 && (a == ASTRA_A_pipe_head || a == ASTRA_A_fifo_head || a == ASTRA_A_bin_cnt || a == ASTRA_A_due_cnt));
        if (!global_only && hot + ab[a] <= opt.hot_budget) { P.a_off[a] = hot | ASTRA_PLACE_SMEM; hot += ab[a]; }
        else { P.a_off[a] = ws; ws += ab[a]; }
    }
    P.hot_bytes = (u32)hot;
    P.ws_bytes = ws;
    return ASTRA_OK;
}
