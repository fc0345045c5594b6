"""A second, deliberately differently structured, pure-Python simulator of the same rules
(SURVEY.md 8(c) R1-R14 / DESIGN.md section 3) for brute-force agreement tests on tiny inputs.

It is NOT the oracle and is used only by tests/test_oracle_bruteforce.py to catch
implementation slips in oracle/astra_oracle.c (index, off-by-one, ordering).  It differs in
structure on purpose: Dijkstra with a heap instead of Bellman-Ford, per-line objects, dict
calendars for pipes and acks, quotas dealt round-robin, release recomputed every cycle, no
bookkeeping shortcuts.
"""
from __future__ import annotations

import heapq
from collections import defaultdict


class Line:
    __slots__ = ("step", "gpu", "wf")

    def __init__(self, step, gpu, wf):
        self.step, self.gpu, self.wf = step, gpu, wf


def simulate(topo, coll, gpu, max_cycles=1 << 22):
    G, V, E = topo.n_gpus, topo.n_nodes, topo.n_links
    tail = [0] * E
    out_links = [[] for _ in range(V)]
    in_links = [[] for _ in range(V)]
    for v in range(V):
        for e in range(int(topo.row_ptr[v]), int(topo.row_ptr[v + 1])):
            tail[e] = v
            out_links[v].append(e)
            in_links[int(topo.head[e])].append(e)
    head = [int(x) for x in topo.head]
    bw = [int(x) for x in topo.bw_q8]
    leff = [int(topo.latency[e]) + int(topo.node_latency[head[e]]) for e in range(E)]

    # Dijkstra from each destination over reversed links
    dist = [[None] * G for _ in range(V)]
    for d in range(G):
        dd = {d: 0}
        pq = [(0, d)]
        while pq:
            x, v = heapq.heappop(pq)
            if dd.get(v, 1 << 62) < x:
                continue
            for e in in_links[v]:
                u = tail[e]
                nx = x + leff[e]
                if nx < dd.get(u, 1 << 62):
                    dd[u] = nx
                    heapq.heappush(pq, (nx, u))
        for v, x in dd.items():
            dist[v][d] = x

    def next_link(v, d):
        cands = [e for e in sorted(out_links[v])
                 if dist[head[e]][d] is not None and leff[e] + dist[head[e]][d] == dist[v][d]]
        return cands[d % len(cands)]

    S = coll.n_steps
    owner = [int(x) for x in coll.owner]
    dst = [int(x) for x in coll.dst]
    lines = [int(x) for x in coll.lines]
    cu_lo = [int(x) for x in coll.cu_lo]
    cu_n = [int(x) for x in coll.cu_n]
    deps = [[(int(coll.dep_step[i]), int(coll.dep_kind[i]))
             for i in range(int(coll.dep_ptr[s]), int(coll.dep_ptr[s + 1]))] for s in range(S)]
    C, W, K, H = gpu.cus, gpu.wavefronts_per_cu, gpu.max_outstanding, gpu.hbm_lines_per_cycle
    per_cu_issue, per_cu_cap = bool(getattr(gpu, "mode", 0) & 1), bool(getattr(gpu, "mode", 0) & 2)     # R12', R2'

    # quota[(s, wf)]: deal the lines of step s round-robin over its wavefronts
    quota = {}
    for s in range(S):
        wfs = [c * W + w for c in range(cu_lo[s], cu_lo[s] + cu_n[s]) for w in range(W)]
        cnt = [0] * len(wfs)
        for i in range(lines[s]):
            cnt[i % len(wfs)] += 1
        for j, wf in enumerate(wfs):
            quota[(s, wf)] = cnt[j]
    # per wavefront work list: [(step, remaining)]
    work = {}
    for g in range(G):
        for wf in range(C * W):
            cu = wf // W
            work[(g, wf)] = [[s, quota[(s, wf)]] for s in range(S)
                             if owner[s] == g and cu_lo[s] <= cu < cu_lo[s] + cu_n[s]]
    outstanding = defaultdict(int)          # keyed (gpu, wavefront), or (gpu, 'cu', cu) for the per-CU pool

    ts = [[None] * 4 for _ in range(S)]   # release, issued, delivered, acked
    cnt_issued = [0] * S
    cnt_deliv = [0] * S
    cnt_ack = [0] * S
    fifo = [[] for _ in range(E)]
    pipe = [defaultdict(list) for _ in range(E)]       # arrival time -> lines in pipe order
    ack_cal = defaultdict(list)
    credit = [256 * -(-b // 256) for b in bw]
    capv = list(credit)
    link_lines = [0] * E
    injected_prev = [[] for _ in range(G)]

    t = 0
    done_steps = 0
    while t < max_cycles:
        # A1
        for v in range(V):
            for e in sorted(in_links[v]):
                for ln in pipe[e].pop(t, []):
                    s = ln.step
                    if dst[s] == v:
                        cnt_deliv[s] += 1
                        if cnt_deliv[s] == lines[s]:
                            ts[s][2] = t
                        ack_cal[t + dist[owner[s]][dst[s]]].append(ln)
                    else:
                        fifo[next_link(v, dst[s])].append(ln)
        # A2
        for g in range(G):
            for ln in sorted(injected_prev[g], key=lambda x: x.wf):
                fifo[next_link(g, dst[ln.step])].append(ln)
            injected_prev[g] = []
        # A3
        for ln in ack_cal.pop(t, []):
            outstanding[(ln.gpu, "cu", ln.wf // W) if per_cu_cap else (ln.gpu, ln.wf)] -= 1
            cnt_ack[ln.step] += 1
            if cnt_ack[ln.step] == lines[ln.step]:
                ts[ln.step][3] = t
                done_steps += 1
        # B
        for e in range(E):
            credit[e] = min(credit[e] + bw[e], capv[e])
            while credit[e] >= 256 and fifo[e]:
                ln = fifo[e].pop(0)
                pipe[e][t + leff[e]].append(ln)
                credit[e] -= 256
                link_lines[e] += 1
        # C
        for s in range(S):
            if ts[s][0] is None:
                ok = True
                for (p, k) in deps[s]:
                    stamp = ts[p][{0: 2, 1: 3, 2: 1}[k]]
                    if stamp is None or stamp > t:
                        ok = False
                if ok:
                    ts[s][0] = t
        # D
        for g in range(G):
            budget = H
            dispatched = set()                          # CUs that have issued this cycle
            for wf in range(C * W):
                if budget == 0:
                    break
                if per_cu_issue and wf // W in dispatched:
                    continue
                lst = work[(g, wf)]
                while lst and ts[lst[0][0]][0] is not None and lst[0][1] == 0:
                    lst.pop(0)
                if not lst or ts[lst[0][0]][0] is None:
                    continue
                slot_key = (g, "cu", wf // W) if per_cu_cap else (g, wf)
                if outstanding[slot_key] >= K:
                    continue
                s = lst[0][0]
                lst[0][1] -= 1
                outstanding[slot_key] += 1
                dispatched.add(wf // W)
                cnt_issued[s] += 1
                if cnt_issued[s] == lines[s]:
                    ts[s][1] = t
                injected_prev[g].append(Line(s, g, wf))
                budget -= 1
        if done_steps == S:
            break
        t += 1
    completion = max((x[3] for x in ts if x[3] is not None), default=0)
    return {"status": 0 if done_steps == S else 1, "completion": completion,
            "step_ts": ts, "link_lines": link_lines}
