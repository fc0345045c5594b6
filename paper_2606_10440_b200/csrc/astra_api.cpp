// astra_api.cpp -- the C-ABI of include/astra.h: object tables, batch preparation (constant blob,
// descriptors, cost-sorted queue, workspace sizing), launch, result read-back.
// No exception crosses the ABI; every entry point returns an ASTRA_E* code.
#include "astra_internal.h"
#include "../../include/astra.h"

#include <cuda_runtime_api.h>

#include <algorithm>
#include <cstring>
#include <map>
#include <new>
#include <numeric>
#include <thread>

struct astra_ctx {
    int device = 0;
    u64 flags = 0;
    std::string err;
    cudaStream_t own_stream = nullptr, stream = nullptr;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    std::vector<HostTopo> topos;
    std::vector<HostColl> colls;
    std::vector<HostGpu> gpus;
    // prepared batch
    bool prepared = false, ran = false, pending = false, results_cached = false;
    std::vector<astra_point> batch_points;
    u64 batch_max_cycles = 0;
    std::vector<PointDesc> descs;
    uint8_t *d_const = nullptr, *d_ws = nullptr, *d_results = nullptr;
    PointDesc* d_points = nullptr;
    u32 *d_order = nullptr, *d_queue = nullptr;
    GroupCtl* d_groups = nullptr;
    u64 const_bytes = 0, ws_big_stride = 0, ws_single_stride = 0, ws_single_off = 0, ws_total = 0, results_bytes = 0;
    u32 n_big = 0, n_slots = 0, grid = 1, group = 1, warps = 0, hot_bytes = 0, variant = 1;
    bool stage = false;
    std::vector<uint8_t> h_results;
    float last_ms = 0.f;
    u32 last_launches = 0;
};

static int32_t fail(astra_ctx* c, int32_t rc, const std::string& msg) { if (c) c->err = msg; return rc; }
static int32_t cuda_fail(astra_ctx* c, cudaError_t e, const char* what) {
    return fail(c, e == cudaErrorMemoryAllocation ? ASTRA_ENOMEM : ASTRA_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CUDA_TRY(ctx, call, what) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(ctx, e_, what); } while (0)

static void free_batch(astra_ctx* c) {
    cudaFree(c->d_const); cudaFree(c->d_ws); cudaFree(c->d_results); cudaFree(c->d_points);
    cudaFree(c->d_order); cudaFree(c->d_queue); cudaFree(c->d_groups);
    c->d_const = c->d_ws = c->d_results = nullptr; c->d_points = nullptr; c->d_order = c->d_queue = nullptr;
    c->d_groups = nullptr;
    c->prepared = false; c->ran = false; c->results_cached = false;
}

extern "C" int32_t astra_create(astra_ctx** out, int32_t cuda_device, uint64_t flags) {
    if (!out) return ASTRA_EINVAL;
    *out = nullptr;
    astra_ctx* c = new (std::nothrow) astra_ctx();
    if (!c) return ASTRA_ENOMEM;
    c->device = cuda_device; c->flags = flags;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || cuda_device < 0 || cuda_device >= n) { delete c; return ASTRA_ECUDA; }
    if (cudaSetDevice(cuda_device) != cudaSuccess || cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreate(&c->ev0) != cudaSuccess || cudaEventCreate(&c->ev1) != cudaSuccess) { delete c; return ASTRA_ECUDA; }
    c->stream = c->own_stream;
    *out = c;
    return ASTRA_OK;
}

extern "C" int32_t astra_destroy(astra_ctx* c) {
    if (!c) return ASTRA_EINVAL;
    cudaSetDevice(c->device);
    if (c->pending) cudaStreamSynchronize(c->stream);
    free_batch(c);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->own_stream) cudaStreamDestroy(c->own_stream);
    delete c;
    return ASTRA_OK;
}

extern "C" const char* astra_last_error(const astra_ctx* c) { return c ? c->err.c_str() : "null context"; }

extern "C" int32_t astra_set_stream(astra_ctx* c, void* s) {
    if (!c) return ASTRA_EINVAL;
    if (c->pending) return fail(c, ASTRA_ESTATE, "a batch is still running");
    c->stream = s ? (cudaStream_t)s : c->own_stream;
    return ASTRA_OK;
}

extern "C" int32_t astra_load_infragraph(astra_ctx* c, uint32_t n_gpus, uint32_t n_switches,
                                         const uint32_t* node_latency, const uint32_t* row_ptr,
                                         const uint32_t* head, const uint32_t* bw_q8, const uint32_t* latency,
                                         uint32_t* out_id) {
    if (!c) return ASTRA_EINVAL;
    if (!node_latency || !row_ptr || !out_id) return fail(c, ASTRA_EINVAL, "null argument");
    try {
        HostTopo t;
        t.G = n_gpus; t.NS = n_switches;
        u64 V = (u64)n_gpus + n_switches;
        if (V >= (1u << 24)) return fail(c, ASTRA_ELIMIT, "too many nodes");
        t.node_lat.assign(node_latency, node_latency + V);
        t.row_ptr.assign(row_ptr, row_ptr + V + 1);
        u32 E = t.row_ptr[V];
        if (E && (!head || !bw_q8 || !latency)) return fail(c, ASTRA_EINVAL, "null link arrays");
        if (E >= (1u << 22)) return fail(c, ASTRA_ELIMIT, "too many links");
        t.head.assign(head, head + E); t.bw.assign(bw_q8, bw_q8 + E); t.lat.assign(latency, latency + E);
        std::string err;
        int32_t rc = astra_build_topo(t, err);
        if (rc) return fail(c, rc, err);
        c->topos.push_back(std::move(t));
        *out_id = (u32)c->topos.size() - 1;
        return ASTRA_OK;
    } catch (const std::bad_alloc&) { return fail(c, ASTRA_ENOMEM, "host allocation failed"); }
      catch (...) { return fail(c, ASTRA_EINVAL, "unexpected error"); }
}

extern "C" int32_t astra_load_collective(astra_ctx* c, uint32_t n_gpus, uint32_t n_steps,
                                         const uint32_t* owner, const uint32_t* dst, const uint32_t* lines,
                                         const uint32_t* cu_lo, const uint32_t* cu_n,
                                         const uint32_t* dep_ptr, const uint32_t* dep_step,
                                         const uint8_t* dep_kind, uint32_t* out_id) {
    if (!c) return ASTRA_EINVAL;
    if (!dep_ptr || !out_id || (n_steps && (!owner || !dst || !lines || !cu_lo || !cu_n))) return fail(c, ASTRA_EINVAL, "null argument");
    try {
        HostColl h;
        h.G = n_gpus; h.S = n_steps;
        if (n_steps >= ASTRA_MAX_STEPS) return fail(c, ASTRA_ELIMIT, "too many steps");
        h.owner.assign(owner, owner + n_steps); h.dst.assign(dst, dst + n_steps); h.lines.assign(lines, lines + n_steps);
        h.cu_lo.assign(cu_lo, cu_lo + n_steps); h.cu_n.assign(cu_n, cu_n + n_steps);
        h.dep_ptr.assign(dep_ptr, dep_ptr + n_steps + 1);
        u32 nd = h.dep_ptr[n_steps];
        if (nd && (!dep_step || !dep_kind)) return fail(c, ASTRA_EINVAL, "null dependency arrays");
        h.dep_step.assign(dep_step, dep_step + nd); h.dep_kind.assign(dep_kind, dep_kind + nd);
        std::string err;
        int32_t rc = astra_build_coll(h, err);
        if (rc) return fail(c, rc, err);
        c->colls.push_back(std::move(h));
        *out_id = (u32)c->colls.size() - 1;
        return ASTRA_OK;
    } catch (const std::bad_alloc&) { return fail(c, ASTRA_ENOMEM, "host allocation failed"); }
      catch (...) { return fail(c, ASTRA_EINVAL, "unexpected error"); }
}

extern "C" int32_t astra_set_gpu_ex(astra_ctx* c, uint32_t cus, uint32_t wpc, uint32_t k, uint32_t h, uint32_t mode, uint32_t* out_id);

extern "C" int32_t astra_set_gpu(astra_ctx* c, uint32_t cus, uint32_t wpc, uint32_t k, uint32_t h, uint32_t* out_id) {
    return astra_set_gpu_ex(c, cus, wpc, k, h, 0u, out_id);
}

extern "C" int32_t astra_set_gpu_ex(astra_ctx* c, uint32_t cus, uint32_t wpc, uint32_t k, uint32_t h, uint32_t mode, uint32_t* out_id) {
    if (!c) return ASTRA_EINVAL;
    if (mode & ~(uint32_t)(ASTRA_GPU_ISSUE_PER_CU | ASTRA_GPU_CAP_PER_CU)) return fail(c, ASTRA_EINVAL, "unknown GPU mode bits");
    if (mode && wpc > 32) return fail(c, ASTRA_ELIMIT, "the per-CU modes need wavefronts_per_cu <= 32");
    if (!out_id) return fail(c, ASTRA_EINVAL, "null argument");
    if (!cus || !wpc || !k || !h) return fail(c, ASTRA_EINVAL, "GPU parameters must be >= 1");
    if ((u64)cus * wpc > ASTRA_MAX_WAVEFRONTS) return fail(c, ASTRA_ELIMIT, "cus * wavefronts_per_cu above ASTRA_MAX_WAVEFRONTS");
    if (k > ASTRA_MAX_OUTSTANDING) return fail(c, ASTRA_ELIMIT, "max_outstanding above ASTRA_MAX_OUTSTANDING");
    if (h > ASTRA_MAX_HBM_LINES) return fail(c, ASTRA_ELIMIT, "hbm_lines_per_cycle above ASTRA_MAX_HBM_LINES");
    HostGpu g; g.C = cus; g.Wv = wpc; g.K = k; g.H = h; g.mode = mode;
    c->gpus.push_back(g);
    *out_id = (u32)c->gpus.size() - 1;
    return ASTRA_OK;
}

// A0 scheduling policy.  Points are split in two classes by a cost proxy (lookahead windows x
// per-window overhead + line-hop events): "big" points, whose cost exceeds what one CTA's fair share
// of the batch is, run on a group of CTAs (one node range each, one group barrier per window); the
// rest run on one CTA each.  Groups whose queue is empty go on as single CTAs.
// ASTRA_FLAG_GROUP(g) overrides: every point on g CTAs (g = 1: every point on one).
static void classify(const astra_ctx* c, u32 n, const astra_point* pts, u32 n_ctas, std::vector<double>& cost,
                     std::vector<uint8_t>& big, u32* group) {
    cost.assign(n, 0.0); big.assign(n, 0);
    double total = 0, cmax = 0;
    for (u32 i = 0; i < n; i++) {
        cost[i] = astra_point_cost(c->topos[pts[i].topo_id], c->colls[pts[i].coll_id], c->flags & 0xff);
        total += cost[i]; cmax = std::max(cmax, cost[i]);
    }
    u32 g = (u32)((c->flags >> 8) & 0xff);
    if (g == 1 || n == 0) { *group = 1; return; }
    if (g > 1) { *group = std::min<u32>(g, std::max<u32>(2, n_ctas)); std::fill(big.begin(), big.end(), 1); return; }
    // Model: a group of g CTAs runs a point min(g, nodes) / 2 times faster than one CTA and costs
    // g CTAs for that time.  Try group sizes and how many of the most expensive points get one;
    // keep the pair with the smallest estimated makespan (critical point vs. total work / CTAs).
    std::vector<u32> idx(n);
    std::iota(idx.begin(), idx.end(), 0u);
    std::sort(idx.begin(), idx.end(), [&](u32 a, u32 b) { return cost[a] > cost[b]; });
    std::vector<double> pre(n + 1, 0.0);
    for (u32 i = 0; i < n; i++) pre[i + 1] = pre[i] + cost[idx[i]];
    double best = std::max(cmax, total / n_ctas);
    u32 best_g = 1, best_r = 0;
    const u32 gs[] = {2, 3, 4, 6, 8, 9, 12, 16, 24, 32, 48, 64, 96, 128, 148, 192, 255};
    for (u32 g2 : gs) {
        if (g2 > n_ctas) break;
        for (u32 r = 1; r <= n; r = r < 4 ? r + 1 : r + (r + 1) / 2) {
            u32 vmin = 0xffffffffu;
            for (u32 i = 0; i < std::min<u32>(r, 8); i++) vmin = std::min(vmin, c->topos[pts[idx[i]].topo_id].V);
            const double speed = 0.5 * std::min<u32>(g2, vmin);
            if (speed <= 1.0) continue;
            const u32 slots = std::max<u32>(1, std::min<u32>(r, n_ctas / g2));
            const double t_big = std::max(cost[idx[0]] / speed, pre[r] / speed / slots);      // critical point, big queue over its slots
            const double t_small = r < n ? cost[idx[r]] : 0.0;
            const double t_work = (pre[n] - pre[r] + pre[r] / speed * g2) / n_ctas;
            const double est = std::max(std::max(t_big, t_small), t_work);
            if (est < best * 0.97) { best = est; best_g = g2; best_r = r; }
        }
    }
    for (u32 i = 0; i < best_r; i++) big[idx[i]] = 1;
    *group = best_g;
}

static int32_t prepare(astra_ctx* c, uint32_t n, const astra_point* pts, uint64_t max_cycles) {
    free_batch(c);
    Blob blob;
    std::map<u32, std::vector<u64>> topo_off, coll_off;
    c->descs.assign(n, PointDesc());
    u64 roff = 0, ws_big_max = 0, ws_single_max = 0;
    for (u32 i = 0; i < n; i++) {
        const astra_point& p = pts[i];
        if (p.topo_id >= c->topos.size() || p.coll_id >= c->colls.size() || p.gpu_id >= c->gpus.size())
            return fail(c, ASTRA_ESTATE, "design point references an unknown id");
    }
    int dev = 0, sms = 0, smem_max = 0;
    CUDA_TRY(c, cudaGetDevice(&dev), "cudaGetDevice");
    CUDA_TRY(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "device attribute");
    CUDA_TRY(c, cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev), "device attribute");
    // CTA shape: 16 warps, one CTA per SM -- or, with ASTRA_FLAG_WARPS(w), 16 / w CTAs of w warps per SM
    // (128 registers per thread; the shared memory of the SM is split evenly between them)
    c->warps = 16;
    { const u32 wf = (u32)((c->flags >> 20) & 0x3f); if (wf == 1 || wf == 2 || wf == 4 || wf == 8 || wf == 16) c->warps = wf; }
    c->variant = 1u;
    const u32 ctas_per_sm = 16 / c->warps;
    std::vector<double> cost; std::vector<uint8_t> big;
    classify(c, n, pts, (u32)sms * ctas_per_sm, cost, big, &c->group);
    PlanOptions opt;
    opt.flags = c->flags & 0xffull; opt.max_cycles = max_cycles;
    c->stage = false;          // reserve the staging area only when some point's per-step tables fit it (it is taken from L1)
    for (u32 i = 0; i < n; i++) c->stage = c->stage || astra_engine_stageable(c->warps, c->colls[pts[i].coll_id].S);
    const u32 fixed = astra_engine_fixed_smem(c->warps, c->stage);
    int smem_sm = 0;
    CUDA_TRY(c, cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev), "device attribute");
    const u32 smem_cta = std::min<u32>((u32)smem_max, (u32)smem_sm / ctas_per_sm - 1024);    // 1 KB per CTA is reserved by the system
    opt.hot_budget = smem_cta > fixed + 1024 ? smem_cta - fixed - 1024 : 0;
    // Shared memory and L1 are one 256 KB array per SM, and the state that does not fit in shared memory (rings, ack
    // records, the constant tables) is read through L1: measured on the five configs, a hot region beyond 48 KB
    // (64 KB for batches with CTA groups) costs more in L1 misses than it saves (config 4: 157 KB -> 48 KB, -6 %).
    {
        bool any_big = false;
        for (u32 i = 0; i < n; i++) any_big |= big[i] != 0;
        opt.hot_budget = std::min<u32>(opt.hot_budget, any_big ? ASTRA_HOT_BUDGET_GROUPS : ASTRA_HOT_BUDGET_SINGLE);
    }
    u32 hot_max = 0, n_big = 0;
    // the tables shared by the points of a topology / a collective go into the blob once
    for (u32 i = 0; i < n; i++) {
        const astra_point& p = pts[i];
        const HostTopo& t = c->topos[p.topo_id];
        const HostColl& h = c->colls[p.coll_id];
        if (!topo_off.count(p.topo_id)) {
            std::vector<u64> o(ASTRA_N_TOPO_TABLES);
            o[0] = blob.add(t.in_ptr); o[1] = blob.add(t.in_link); o[2] = blob.add(t.head); o[3] = blob.add(t.tail);
            o[4] = blob.add(t.leff); o[5] = blob.add(t.next_link); o[6] = blob.add(t.row_ptr);
            topo_off[p.topo_id] = o;
        }
        if (!coll_off.count(p.coll_id)) {
            std::vector<u32> od(h.S);
            for (u32 s = 0; s < h.S; s++) od[s] = (h.owner[s] << 16) | h.dst[s];
            std::vector<u64> o(ASTRA_N_COLL_TABLES);
            o[0] = blob.add(od); o[1] = blob.add(h.lines); o[2] = blob.add(h.cu_lo); o[3] = blob.add(h.cu_n);
            o[4] = blob.add(h.succ_ptr); o[5] = blob.add(h.succ); o[6] = blob.add(h.ndeps);
            coll_off[p.coll_id] = o;
        }
    }
    // A0 per point (routing walk, cell layout, array placement): independent, spread over the host's cores; every
    // thread appends its points' own tables to a blob of its own, concatenated behind the shared tables afterwards
    const u32 n_thr = std::max<u32>(1, std::min<u32>({std::thread::hardware_concurrency(), 32u, (n + 15) / 16}));
    std::vector<Blob> tblob(n_thr);
    std::vector<int32_t> trc(n_thr, ASTRA_OK);
    std::vector<std::string> terr(n_thr);
    std::vector<u32> tfail(n_thr, 0);
    auto plan_range = [&](u32 th) {
        const u32 lo = (u32)((u64)n * th / n_thr), hi = (u32)((u64)n * (th + 1) / n_thr);
        try {
            for (u32 i = lo; i < hi && trc[th] == ASTRA_OK; i++) {
                const astra_point& p = pts[i];
                PlanOptions o2 = opt;
                o2.group = big[i] ? c->group : 1;
                double unused = 0;
                int32_t rc = astra_plan_point(c->topos[p.topo_id], c->colls[p.coll_id], c->gpus[p.gpu_id], o2,
                                              topo_off.find(p.topo_id)->second.data(), coll_off.find(p.coll_id)->second.data(),
                                              tblob[th], c->descs[i], unused, terr[th]);
                if (rc) { trc[th] = rc; tfail[th] = i; }
            }
        } catch (const std::bad_alloc&) { trc[th] = ASTRA_ENOMEM; terr[th] = "host allocation failed"; tfail[th] = lo; }
          catch (...) { trc[th] = ASTRA_EINVAL; terr[th] = "unexpected error"; tfail[th] = lo; }
    };
    if (n_thr == 1) plan_range(0);
    else {
        std::vector<std::thread> pool;
        for (u32 th = 0; th < n_thr; th++) pool.emplace_back(plan_range, th);
        for (auto& th : pool) th.join();
    }
    for (u32 th = 0; th < n_thr; th++)
        if (trc[th]) return fail(c, trc[th], "point " + std::to_string(tfail[th]) + ": " + terr[th]);
    {
        // c_off entries of the tables a point shares with others are offsets into the shared part already; the
        // point's own tables move behind it by the offset of its thread's blob
        bool shared_table[ASTRA_C_COUNT] = {false};
        for (u32 q : {ASTRA_C_in_ptr, ASTRA_C_in_link, ASTRA_C_head, ASTRA_C_tail, ASTRA_C_leff, ASTRA_C_next_link, ASTRA_C_row_ptr,
                      ASTRA_C_step_od, ASTRA_C_lines, ASTRA_C_cu_lo, ASTRA_C_cu_n, ASTRA_C_succ_ptr, ASTRA_C_succ, ASTRA_C_ndeps})
            shared_table[q] = true;
        u64 total = blob.bytes.size() + 16;
        for (u32 th = 0; th < n_thr; th++) total += tblob[th].bytes.size() + 16;
        blob.bytes.reserve(total);                                  // one allocation, no re-copy of what is there
        for (u32 th = 0; th < n_thr; th++) {
            const u64 base = blob.add(tblob[th].bytes.data(), tblob[th].bytes.size());
            const u32 lo = (u32)((u64)n * th / n_thr), hi = (u32)((u64)n * (th + 1) / n_thr);
            for (u32 i = lo; i < hi; i++)
                for (u32 q = 0; q < ASTRA_C_COUNT; q++)
                    if (!shared_table[q]) c->descs[i].c_off[q] += base;
            std::vector<uint8_t>().swap(tblob[th].bytes);
        }
    }
    for (u32 i = 0; i < n; i++) {
        PointDesc& P = c->descs[i];
        P.r_step_ts = roff; roff += 32ull * P.S;
        P.r_link_lines = roff; roff += 8ull * P.E;
        P.r_summary = roff; roff += (sizeof(DeviceSummary) + 15) & ~15ull;
        P.r_diag = roff; roff += 8ull * ASTRA_DIAG_WORDS * P.group;      // per CTA of the group (written by ASTRA_DIAG builds)
        if (big[i]) { ws_big_max = std::max(ws_big_max, P.ws_bytes); n_big++; }
        else ws_single_max = std::max(ws_single_max, P.ws_bytes);
        hot_max = std::max(hot_max, P.hot_bytes);
    }
    c->hot_bytes = hot_max;
    c->results_bytes = roff ? roff : 16;
    std::string err;
    u32 occ = 0, nsm = 0;
    int32_t rc = astra_engine_occupancy(c->warps, c->hot_bytes, c->variant, c->stage, &occ, &nsm, err);
    if (rc) return fail(c, rc, err);
    if (occ == 0) return fail(c, ASTRA_ECUDA, "kernel does not fit on an SM");
    // every CTA of the grid must be resident at once (persistent CTAs, group barriers)
    const u32 n_ctas = occ * nsm, n_small = n - n_big;
    c->n_big = n_big;
    c->n_slots = n_big ? std::max<u32>(1, std::min<u32>(n_big, n_ctas / c->group)) : 0;
    c->grid = std::max<u32>(1, std::min<u32>(n_ctas, c->n_slots * c->group + n_small));
    if (n_big && c->grid < c->n_slots * c->group) c->grid = c->n_slots * c->group;
    c->ws_big_stride = (ws_big_max + 255) & ~255ull;
    c->ws_single_stride = n_small ? (ws_single_max + 255) & ~255ull : 0;
    size_t free_b = 0, total_b = 0;
    CUDA_TRY(c, cudaMemGetInfo(&free_b, &total_b), "cudaMemGetInfo");
    u64 budget = (u64)(free_b * 0.85);
    u64 fixed_b = blob.bytes.size() + c->results_bytes + n * sizeof(PointDesc) + n * 4 + 4096;
    auto ws_need = [&]() { return (u64)c->n_slots * c->ws_big_stride + (u64)c->grid * c->ws_single_stride; };
    while (fixed_b + ws_need() > budget) {       // fewer resident CTAs until the workspaces fit
        if (c->grid > c->n_slots * c->group && c->grid > 1) c->grid--;
        else if (c->n_slots > 1) { c->n_slots--; c->grid = std::max<u32>(1, std::min(c->grid, std::max(c->n_slots * c->group, c->grid - c->group))); }
        else return fail(c, ASTRA_ENOMEM, "batch does not fit in device memory");
    }
    c->ws_single_off = (u64)c->n_slots * c->ws_big_stride;
    c->ws_total = ws_need();
    c->const_bytes = blob.bytes.size();

    // queue order: big points first (most expensive first), then the small ones (most expensive first)
    std::vector<u32> order(n);
    std::iota(order.begin(), order.end(), 0u);
    std::stable_sort(order.begin(), order.end(), [&](u32 a, u32 b) {
        if (big[a] != big[b]) return big[a] > big[b];
        return cost[a] > cost[b];
    });

    CUDA_TRY(c, cudaMalloc((void**)&c->d_const, blob.bytes.size() + 16), "cudaMalloc const");
    CUDA_TRY(c, cudaMalloc((void**)&c->d_ws, std::max<u64>(16, c->ws_total)), "cudaMalloc workspace");
    CUDA_TRY(c, cudaMalloc((void**)&c->d_results, c->results_bytes), "cudaMalloc results");
    CUDA_TRY(c, cudaMalloc((void**)&c->d_points, std::max<size_t>(16, n * sizeof(PointDesc))), "cudaMalloc points");
    CUDA_TRY(c, cudaMalloc((void**)&c->d_order, std::max<size_t>(16, n * 4)), "cudaMalloc order");
    CUDA_TRY(c, cudaMalloc((void**)&c->d_queue, 16), "cudaMalloc queue");
    CUDA_TRY(c, cudaMalloc((void**)&c->d_groups, sizeof(GroupCtl) * std::max<u32>(1, c->n_slots)), "cudaMalloc groups");
    CUDA_TRY(c, cudaMemcpyAsync(c->d_const, blob.bytes.data(), blob.bytes.size(), cudaMemcpyHostToDevice, c->stream), "H2D const");
    CUDA_TRY(c, cudaMemcpyAsync(c->d_points, c->descs.data(), n * sizeof(PointDesc), cudaMemcpyHostToDevice, c->stream), "H2D points");
    CUDA_TRY(c, cudaMemcpyAsync(c->d_order, order.data(), n * 4, cudaMemcpyHostToDevice, c->stream), "H2D order");
    CUDA_TRY(c, cudaStreamSynchronize(c->stream), "H2D sync");     // host staging buffers die here
    c->batch_points.assign(pts, pts + n);
    c->batch_max_cycles = max_cycles;
    c->prepared = true;
    return ASTRA_OK;
}

extern "C" int32_t astra_run_batch_async(astra_ctx* c, uint32_t n, const astra_point* pts, uint64_t max_cycles) {
    if (!c) return ASTRA_EINVAL;
    if (n && !pts) return fail(c, ASTRA_EINVAL, "null points");
    if (c->pending) return fail(c, ASTRA_ESTATE, "a batch is still running");
    try {
        CUDA_TRY(c, cudaSetDevice(c->device), "cudaSetDevice");
        bool same = c->prepared && c->batch_points.size() == n && c->batch_max_cycles == max_cycles &&
                    (n == 0 || std::memcmp(c->batch_points.data(), pts, n * sizeof(astra_point)) == 0);
        if (!same) { int32_t rc = prepare(c, n, pts, max_cycles); if (rc) return rc; }
        c->results_cached = false; c->ran = false;
        CUDA_TRY(c, cudaEventRecord(c->ev0, c->stream), "event record");
        c->last_launches = 0;
        if (n) {
            EngineLaunch L;
            L.d_const = c->d_const; L.d_ws = c->d_ws; L.d_results = c->d_results; L.d_points = c->d_points;
            L.d_order = c->d_order; L.d_queue = c->d_queue; L.d_groups = c->d_groups; L.n_points = n;
            L.n_big = c->n_big; L.n_slots = c->n_slots; L.group = c->group; L.grid = c->grid;
            L.ws_big_stride = c->ws_big_stride; L.ws_single_off = c->ws_single_off; L.ws_single_stride = c->ws_single_stride;
            L.warps_per_cta = c->warps; L.hot_bytes = c->hot_bytes; L.variant = c->variant; L.stage = c->stage;
            std::string err;
            int32_t rc = astra_engine_launch(L, (void*)c->stream, err);
            if (rc) return fail(c, rc, err);
            c->last_launches = 1;
        }
        CUDA_TRY(c, cudaEventRecord(c->ev1, c->stream), "event record");
        c->pending = true;
        return ASTRA_OK;
    } catch (const std::bad_alloc&) { return fail(c, ASTRA_ENOMEM, "host allocation failed"); }
      catch (...) { return fail(c, ASTRA_EINVAL, "unexpected error"); }
}

extern "C" int32_t astra_sync(astra_ctx* c) {
    if (!c) return ASTRA_EINVAL;
    if (!c->pending) return ASTRA_OK;
    c->pending = false;
    CUDA_TRY(c, cudaSetDevice(c->device), "cudaSetDevice");
    CUDA_TRY(c, cudaStreamSynchronize(c->stream), "kernel execution");
    CUDA_TRY(c, cudaEventElapsedTime(&c->last_ms, c->ev0, c->ev1), "event elapsed");
    if (c->d_queue && c->last_launches) {           // did a group barrier time out (kernel-wide abort flag)?
        u32 q[4] = {0, 0, 0, 0};
        CUDA_TRY(c, cudaMemcpy(q, c->d_queue, sizeof(q), cudaMemcpyDeviceToHost), "D2H queue");
        if (q[2]) return fail(c, ASTRA_ECUDA, "a CTA group barrier timed out: the batch was abandoned");
    }
    c->ran = true;
    return ASTRA_OK;
}

extern "C" int32_t astra_run_batch(astra_ctx* c, uint32_t n, const astra_point* pts, uint64_t max_cycles) {
    int32_t rc = astra_run_batch_async(c, n, pts, max_cycles);
    if (rc) return rc;
    return astra_sync(c);
}

extern "C" int32_t astra_read_results(astra_ctx* c, uint32_t point, astra_summary* out, uint64_t* step_ts, uint64_t* link_lines) {
    if (!c) return ASTRA_EINVAL;
    if (c->pending) { int32_t rc = astra_sync(c); if (rc) return rc; }
    if (!c->ran) return fail(c, ASTRA_ESTATE, "no batch has been run");
    if (point >= c->descs.size()) return fail(c, ASTRA_ESTATE, "point index out of range");
    try {
        if (!c->results_cached) {
            CUDA_TRY(c, cudaSetDevice(c->device), "cudaSetDevice");
            c->h_results.resize(c->results_bytes);
            CUDA_TRY(c, cudaMemcpy(c->h_results.data(), c->d_results, c->results_bytes, cudaMemcpyDeviceToHost), "D2H results");
            c->results_cached = true;
        }
    } catch (const std::bad_alloc&) { return fail(c, ASTRA_ENOMEM, "host allocation failed"); }
    const PointDesc& P = c->descs[point];
    const uint8_t* base = c->h_results.data();
    if (out) {
        DeviceSummary s; std::memcpy(&s, base + P.r_summary, sizeof(s));
        out->status = s.status; out->n_steps = s.n_steps; out->n_links = s.n_links; out->window = s.window;
        out->completion_cycle = s.completion_cycle; out->total_lines = s.total_lines;
        out->busy_cycles = s.busy_cycles; out->skipped_cycles = s.skipped_cycles;
    }
    if (step_ts) std::memcpy(step_ts, base + P.r_step_ts, 32ull * P.S);
    if (link_lines) std::memcpy(link_lines, base + P.r_link_lines, 8ull * P.E);
    return ASTRA_OK;
}

extern "C" int32_t astra_read_diag(astra_ctx* c, uint32_t point, uint32_t cta_rank, uint64_t* out144) {
    if (!c) return ASTRA_EINVAL;
    if (!out144) return fail(c, ASTRA_EINVAL, "null argument");
    if (!astra_engine_has_diag()) return fail(c, ASTRA_ESTATE, "this library was built without ASTRA_DIAG");
    int32_t rc = astra_read_results(c, point, nullptr, nullptr, nullptr);
    if (rc) return rc;
    if (cta_rank >= c->descs[point].group) return fail(c, ASTRA_ESTATE, "cta_rank beyond the point's CTA group");
    std::memcpy(out144, c->h_results.data() + c->descs[point].r_diag + 8ull * ASTRA_DIAG_WORDS * cta_rank, 8ull * ASTRA_DIAG_WORDS);
    return ASTRA_OK;
}

extern "C" int32_t astra_point_group(astra_ctx* c, uint32_t point, uint32_t* group) {
    if (!c) return ASTRA_EINVAL;
    if (!group) return fail(c, ASTRA_EINVAL, "null argument");
    if (!c->prepared || point >= c->descs.size()) return fail(c, ASTRA_ESTATE, "no such point in the prepared batch");
    *group = c->descs[point].group;
    return ASTRA_OK;
}

extern "C" int32_t astra_last_run_info(astra_ctx* c, float* ms, uint32_t* launches, uint64_t* bytes) {
    if (!c) return ASTRA_EINVAL;
    if (c->pending) { int32_t rc = astra_sync(c); if (rc) return rc; }
    if (ms) *ms = c->last_ms;
    if (launches) *launches = c->last_launches;
    if (bytes) *bytes = c->const_bytes + c->ws_total + c->results_bytes + c->descs.size() * sizeof(PointDesc);
    return ASTRA_OK;
}

extern "C" int32_t astra_last_transfer_bytes(astra_ctx* c, uint64_t* h2d, uint64_t* d2h) {
    if (!c) return ASTRA_EINVAL;
    if (!c->prepared) return fail(c, ASTRA_ESTATE, "no batch has been prepared");
    if (h2d) *h2d = c->const_bytes + c->descs.size() * (sizeof(PointDesc) + 4);
    if (d2h) *d2h = c->results_bytes;
    return ASTRA_OK;
}


// ---------------------------------------------------------------------------------------------
// No-allocation entry point (include/astra.h).  astra_pack_point is set-up: it plans one design
// point for a single CTA exactly as prepare() does for a one-CTA point and serialises what the
// kernel reads.  astra_run_packed_noalloc only clears the scratch header and launches.
// ---------------------------------------------------------------------------------------------
extern "C" int32_t astra_pack_point(astra_ctx* c, const astra_point* pt, uint64_t max_cycles,
                                    void* host_buf, uint64_t host_buf_bytes, astra_packed_info* info) {
    if (!c) return ASTRA_EINVAL;
    if (!pt || !info) return fail(c, ASTRA_EINVAL, "null argument");
    std::memset(info, 0, sizeof(*info));
    if (pt->topo_id >= c->topos.size() || pt->coll_id >= c->colls.size() || pt->gpu_id >= c->gpus.size())
        return fail(c, ASTRA_ESTATE, "design point references an unknown id");
    try {
        CUDA_TRY(c, cudaSetDevice(c->device), "cudaSetDevice");
        int smem_max = 0, smem_sm = 0;
        CUDA_TRY(c, cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device), "device attribute");
        CUDA_TRY(c, cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, c->device), "device attribute");
        std::string err;
        uint8_t* scratch = nullptr;
        int32_t rc = astra_engine_static_scratch(c->device, &scratch, err);     // once per device, this device current
        if (rc) return fail(c, rc, err);
        const u32 warps = 16;
        const u32 fixed = astra_engine_fixed_smem(warps, astra_engine_stageable(warps, c->colls[pt->coll_id].S));
        const u32 smem_cta = std::min<u32>((u32)smem_max, (u32)smem_sm - 1024);
        PlanOptions opt;
        opt.flags = c->flags & 0xffull; opt.max_cycles = max_cycles; opt.group = 1;
        opt.hot_budget = std::min<u32>(smem_cta > fixed + 1024 ? smem_cta - fixed - 1024 : 0, ASTRA_HOT_BUDGET_SINGLE);
        const HostTopo& t = c->topos[pt->topo_id];
        const HostColl& h = c->colls[pt->coll_id];
        Blob blob;
        u64 to[ASTRA_N_TOPO_TABLES], co[ASTRA_N_COLL_TABLES];
        to[0] = blob.add(t.in_ptr); to[1] = blob.add(t.in_link); to[2] = blob.add(t.head); to[3] = blob.add(t.tail);
        to[4] = blob.add(t.leff); to[5] = blob.add(t.next_link); to[6] = blob.add(t.row_ptr);
        std::vector<u32> od(h.S);
        for (u32 s = 0; s < h.S; s++) od[s] = (h.owner[s] << 16) | h.dst[s];
        co[0] = blob.add(od); co[1] = blob.add(h.lines); co[2] = blob.add(h.cu_lo); co[3] = blob.add(h.cu_n);
        co[4] = blob.add(h.succ_ptr); co[5] = blob.add(h.succ); co[6] = blob.add(h.ndeps);
        PointDesc P;
        double unused = 0;
        rc = astra_plan_point(t, h, c->gpus[pt->gpu_id], opt, to, co, blob, P, unused, err);
        if (rc) return fail(c, rc, err);
        u64 roff = 0;
        P.r_step_ts = roff; roff += 32ull * P.S;
        P.r_link_lines = roff; roff += 8ull * P.E;
        P.r_summary = roff; roff += (sizeof(DeviceSummary) + 15) & ~15ull;
        P.r_diag = roff; roff += 8ull * ASTRA_DIAG_WORDS;
        info->magic = ASTRA_PACKED_MAGIC;
        info->off_const = 0;
        info->off_desc = (blob.bytes.size() + 255) & ~255ull;
        info->off_order = info->off_desc + ((sizeof(PointDesc) + 255) & ~255ull);
        info->in_bytes = info->off_order + 256;
        info->out_bytes = (std::max<u64>(roff, 16) + 255) & ~255ull;
        info->scratch_bytes = (u64)ASTRA_NOALLOC_HEADER_BYTES + ((P.ws_bytes + 255) & ~255ull);
        info->off_step_ts = P.r_step_ts; info->off_link_lines = P.r_link_lines; info->off_summary = P.r_summary;
        info->n_steps = P.S; info->n_links = P.E; info->hot_bytes = P.hot_bytes; info->warps = warps;
        if (host_buf) {
            if (host_buf_bytes < info->in_bytes) return fail(c, ASTRA_ELIMIT, "host buffer smaller than info->in_bytes");
            uint8_t* hb = (uint8_t*)host_buf;
            std::memset(hb, 0, info->in_bytes);
            if (!blob.bytes.empty()) std::memcpy(hb + info->off_const, blob.bytes.data(), blob.bytes.size());
            std::memcpy(hb + info->off_desc, &P, sizeof(P));
            const u32 order0 = 0;
            std::memcpy(hb + info->off_order, &order0, sizeof(order0));
        }
        return ASTRA_OK;
    } catch (const std::bad_alloc&) { return fail(c, ASTRA_ENOMEM, "host allocation failed"); }
      catch (...) { return fail(c, ASTRA_EINVAL, "unexpected error"); }
}

// Allocates nothing: argument checks, one cudaMemsetAsync on the static scratch header, one kernel launch.
// (An error message is copied into the ctx on failure only.)
extern "C" int32_t astra_run_packed_noalloc(astra_ctx* c, const astra_packed_info* info, const void* d_in, void* d_out, void* stream) {
    if (!c) return ASTRA_EINVAL;
    if (!info || !d_in || !d_out) return fail(c, ASTRA_EINVAL, "null argument");
    if (info->magic != ASTRA_PACKED_MAGIC || info->off_order + 4 > info->in_bytes || info->off_desc + sizeof(PointDesc) > info->off_order)
        return fail(c, ASTRA_EINVAL, "not an astra_packed_info written by astra_pack_point");
    if (((uintptr_t)d_in | (uintptr_t)d_out) & 255u) return fail(c, ASTRA_EINVAL, "d_in and d_out must be 256-byte aligned");
    if (info->scratch_bytes > ASTRA_NOALLOC_SCRATCH_BYTES)
        return fail(c, ASTRA_ELIMIT, "scratch of " + std::to_string(info->scratch_bytes) + " bytes exceeds the library's static scratch of " +
                                     std::to_string((u64)ASTRA_NOALLOC_SCRATCH_BYTES) + " bytes (ASTRA_NOALLOC_SCRATCH_BYTES): use astra_run_batch");
    if (c->pending) return fail(c, ASTRA_ESTATE, "a batch is still running");
    CUDA_TRY(c, cudaSetDevice(c->device), "cudaSetDevice");
    const uint8_t* in = (const uint8_t*)d_in;
    std::string err;
    int32_t rc = astra_engine_launch_noalloc(c->device, in + info->off_const, (const PointDesc*)(in + info->off_desc),
                                             (const u32*)(in + info->off_order), (uint8_t*)d_out,
                                             info->scratch_bytes - ASTRA_NOALLOC_HEADER_BYTES, info->warps, info->hot_bytes, info->n_steps,
                                             stream ? stream : (void*)c->stream, err);
    if (rc) return fail(c, rc, err);
    return ASTRA_OK;
}
