"""Step-DAG generators for the textbook collectives the paper names (ring,
all-pairs/direct, double binary tree, recursive halving-doubling) plus the hierarchical
all-reduce and all-to-all of BASELINE configs 3 and 5.  Definitions follow SURVEY.md 8(d).

These are inputs, not the simulated method: they only lay out who sends how many lines to
whom, on which CUs, after which steps.
"""
from __future__ import annotations

from typing import List, Sequence

from .types import Collective, CollectiveBuilder, DEP_DELIVERED


def split_lines(total: int, parts: int) -> List[int]:
    """chunk i of `parts` gets floor(total/parts) + (i < total mod parts)."""
    q, r = divmod(total, parts)
    return [q + (1 if i < r else 0) for i in range(parts)]


def cu_slice(p: int, parts: int, cus: int):
    """CU slice p of `parts` over `cus` CUs: [floor(p*C/parts), floor((p+1)*C/parts))."""
    lo = (p * cus) // parts
    hi = ((p + 1) * cus) // parts
    return lo, hi - lo


def ring_allreduce(n: int, lines: int, cus: int, ranks: Sequence[int] | None = None,
                   b: CollectiveBuilder | None = None, first_deps=None,
                   n_gpus_total: int | None = None):
    """Ring all-reduce over `ranks` (default 0..n-1), `lines` split in n chunks.
    Step (s, i): ranks[i] -> ranks[(i+1)%n], chunk (i - s) mod n, s = 0..2n-3; step s>=1
    depends DELIVERED on step (s-1, i-1).  Returns (collective | None, ids[s][i])."""
    own = b is None
    if ranks is None:
        ranks = list(range(n))
    if b is None:
        b = CollectiveBuilder(n_gpus_total or n, f"ring_allreduce_n{n}_m{lines}")
    chunks = split_lines(lines, n)
    ids = [[-1] * n for _ in range(2 * (n - 1))]
    for s in range(2 * (n - 1)):
        for i in range(n):
            deps = []
            if s == 0:
                if first_deps is not None:
                    deps = list(first_deps[i])
            else:
                deps = [(ids[s - 1][(i - 1) % n], DEP_DELIVERED)]
            ids[s][i] = b.add(ranks[i], ranks[(i + 1) % n], chunks[(i - s) % n], 0, cus, deps)
    return (b.build() if own else None), ids


def direct_allreduce(n: int, lines: int, cus: int) -> Collective:
    """All-pairs all-reduce: reduce-scatter ids p*n+g (g sends chunk of dst to dst=(g+1+p)%n),
    all-gather ids (n-1)*n + p*n+g (g sends its own chunk), every all-gather step depending
    DELIVERED on all n-1 inbound reduce-scatter steps.  Peer p runs on CU slice p of n-1 when
    cus >= n-1, else on the single CU p mod cus."""
    b = CollectiveBuilder(n, f"direct_allreduce_n{n}_m{lines}")
    chunks = split_lines(lines, n)

    def cu_of(p):
        if cus >= n - 1:
            return cu_slice(p, n - 1, cus)
        return p % cus, 1

    rs = {}
    for p in range(n - 1):
        for g in range(n):
            d = (g + 1 + p) % n
            lo, cn = cu_of(p)
            rs[(p, g)] = b.add(g, d, chunks[d], lo, cn)
    for p in range(n - 1):
        for g in range(n):
            d = (g + 1 + p) % n
            lo, cn = cu_of(p)
            deps = [(rs[(pp, (g - 1 - pp) % n)], DEP_DELIVERED) for pp in range(n - 1)]
            b.add(g, d, chunks[g], lo, cn, deps)
    return b.build()


def halving_doubling_allreduce(n: int, lines: int, cus: int) -> Collective:
    """Recursive halving-doubling (n = 2^k): reduce-scatter rounds r=0..k-1 with partner
    g XOR (n>>(r+1)); the range is split at lo+ceil(len/2), the lower half is kept by the GPU
    whose bit is 0; then all-gather rounds in reverse.  ids round*n+g; each step depends
    DELIVERED on the previous-round step delivered into g."""
    k = n.bit_length() - 1
    if (1 << k) != n:
        raise ValueError("halving-doubling needs a power-of-two GPU count")
    if lines < n:
        raise ValueError("need at least n lines")
    b = CollectiveBuilder(n, f"hd_allreduce_n{n}_m{lines}")
    lo = [0] * n
    ln = [lines] * n
    ids = {}
    rnd = 0
    for r in range(k):
        mask = n >> (r + 1)
        new_lo, new_ln = list(lo), list(ln)
        for g in range(n):
            half_hi = (ln[g] + 1) // 2          # lower half length (ceil)
            bit = 1 if (g & mask) else 0
            if bit == 0:
                send = ln[g] - half_hi            # send upper half
                new_lo[g], new_ln[g] = lo[g], half_hi
            else:
                send = half_hi                    # send lower half
                new_lo[g], new_ln[g] = lo[g] + half_hi, ln[g] - half_hi
            deps = []
            if rnd > 0:
                prev_mask = n >> r
                deps = [(ids[(rnd - 1, g ^ prev_mask)], DEP_DELIVERED)]
            ids[(rnd, g)] = b.add(g, g ^ mask, send, 0, cus, deps)
        lo, ln = new_lo, new_ln
        rnd += 1
    prev_mask = 1       # the last halving round used mask n >> k == 1
    for j in range(k):
        mask = 1 << j
        new_lo, new_ln = list(lo), list(ln)
        for g in range(n):
            p = g ^ mask
            deps = [(ids[(rnd - 1, g ^ prev_mask)], DEP_DELIVERED)]
            ids[(rnd, g)] = b.add(g, p, ln[g], 0, cus, deps)
            new_lo[g] = min(lo[g], lo[p])
            new_ln[g] = ln[g] + ln[p]
        lo, ln = new_lo, new_ln
        prev_mask = mask
        rnd += 1
    return b.build()


def _t1_parent(r: int, n: int) -> int:
    """Tree T1: rank 0 is the root with the single child n/2; below it the
    in-order complete binary tree on 1..n-1."""
    bit = r & (-r)
    par = r - bit if ((r // (2 * bit)) & 1) else r + bit
    return par if 0 < par < n else 0


def dbt_parents(n: int):
    """Parents of both trees; parent[t][root] == -1.  T2 is T1 relabelled (r+1) mod n."""
    p1 = [-1] * n
    for r in range(1, n):
        p1[r] = _t1_parent(r, n)
    p2 = [-1] * n
    for r in range(n):
        x = (r + 1) % n
        p2[x] = -1 if p1[r] < 0 else (p1[r] + 1) % n
    return [p1, p2]


def double_binary_tree_allreduce(n: int, lines: int, cus: int, max_chunks: int = 4) -> Collective:
    """Double binary tree all-reduce: tree t carries ceil(M/2) / floor(M/2) lines in
    P = min(max_chunks, lines_t) pipeline chunks.  Reduce step child->parent depends DELIVERED
    on the child's children's same-chunk reduce steps; broadcast step parent->child depends on
    the parent's inbound same-chunk broadcast (root: on its child's reduce).  CU quarter
    2t+dir.  ids: all reduce steps ordered (chunk, tree, depth descending, rank), then all
    broadcast steps ordered (chunk, tree, depth ascending, parent rank, child)."""
    if cus < 4:
        raise ValueError("double binary tree layout needs >= 4 CUs")
    b = CollectiveBuilder(n, f"dbt_allreduce_n{n}_m{lines}")
    parents = dbt_parents(n)
    tree_lines = [(lines + 1) // 2, lines // 2]
    depth = []
    children = []
    for t in range(2):
        par = parents[t]
        d = [0] * n
        ch = [[] for _ in range(n)]
        for r in range(n):
            x, k = r, 0
            while par[x] >= 0:
                x = par[x]; k += 1
            d[r] = k
            if par[r] >= 0:
                ch[par[r]].append(r)
        for c in ch:
            c.sort()
        depth.append(d)
        children.append(ch)
    nchunks = [min(max_chunks, tl) for tl in tree_lines]
    chunk_lines = [split_lines(tree_lines[t], nchunks[t]) if nchunks[t] else [] for t in range(2)]
    red = {}
    for c in range(max(nchunks) if nchunks else 0):
        for t in range(2):
            if c >= nchunks[t]:
                continue
            lo, cn = cu_slice(2 * t + 0, 4, cus)
            order = sorted((r for r in range(n) if parents[t][r] >= 0),
                           key=lambda r: (-depth[t][r], r))
            for r in order:
                deps = [(red[(c, t, k)], DEP_DELIVERED) for k in children[t][r]]
                red[(c, t, r)] = b.add(r, parents[t][r], chunk_lines[t][c], lo, cn, deps)
    bc = {}
    for c in range(max(nchunks) if nchunks else 0):
        for t in range(2):
            if c >= nchunks[t]:
                continue
            lo, cn = cu_slice(2 * t + 1, 4, cus)
            order = sorted((r for r in range(n) if parents[t][r] >= 0),
                           key=lambda r: (depth[t][r], parents[t][r], r))
            for r in order:
                p = parents[t][r]
                if parents[t][p] < 0:      # p is the root: wait for its child's reduce
                    deps = [(red[(c, t, k)], DEP_DELIVERED) for k in children[t][p]]
                else:
                    deps = [(bc[(c, t, p)], DEP_DELIVERED)]
                bc[(c, t, r)] = b.add(p, r, chunk_lines[t][c], lo, cn, deps)
    return b.build()


def hierarchical_allreduce(n_nodes: int, gpus_per_node: int, lines: int, cus: int) -> Collective:
    """BASELINE config 3: intra-node direct reduce-scatter, inter-node ring all-reduce over the
    same-local GPUs on the node-local shard, intra-node direct all-gather."""
    G = n_nodes * gpus_per_node
    L = gpus_per_node
    if lines % L:
        raise ValueError("lines must divide by gpus_per_node")
    shard = lines // L
    b = CollectiveBuilder(G, f"hier_allreduce_{n_nodes}x{L}_m{lines}")
    p1 = {}
    for p in range(L - 1):
        for g in range(G):
            nd, loc = divmod(g, L)
            d = nd * L + (loc + 1 + p) % L
            lo, cn = cu_slice(p, L - 1, cus)
            p1[(p, g)] = b.add(g, d, shard, lo, cn)
    # phase 2: for every local index, a ring over the n_nodes same-local GPUs.  Step ids are
    # 448 + s*64 + g in the 8x8 case: emit in (s, g) order.
    chunks = split_lines(shard, n_nodes)
    p2 = {}
    for s in range(2 * (n_nodes - 1)):
        for g in range(G):
            nd, loc = divmod(g, L)
            d = ((nd + 1) % n_nodes) * L + loc
            if s == 0:
                deps = [(p1[(pp, nd * L + (loc - 1 - pp) % L)], DEP_DELIVERED) for pp in range(L - 1)]
            else:
                prev = ((nd - 1) % n_nodes) * L + loc
                deps = [(p2[(s - 1, prev)], DEP_DELIVERED)]
            p2[(s, g)] = b.add(g, d, chunks[(nd - s) % n_nodes], 0, cus, deps)
    last = 2 * (n_nodes - 1) - 1
    for p in range(L - 1):
        for g in range(G):
            nd, loc = divmod(g, L)
            d = nd * L + (loc + 1 + p) % L
            lo, cn = cu_slice(p, L - 1, cus)
            prev = ((nd - 1) % n_nodes) * L + loc
            b.add(g, d, shard, lo, cn, [(p2[(last, prev)], DEP_DELIVERED)])
    return b.build()


def all_to_all(n: int, pair_lines, cus: int) -> Collective:
    """BASELINE config 5: ids p*n+g, p=0..n-2, dst=(g+1+p)%n, no deps, CU = p mod cus
    (cu_n = 1).  pair_lines(g, d) -> lines for the ordered pair."""
    b = CollectiveBuilder(n, f"all_to_all_n{n}")
    for p in range(n - 1):
        for g in range(n):
            d = (g + 1 + p) % n
            b.add(g, d, pair_lines(g, d), p % cus, 1)
    return b.build()


def single_transfer(n_gpus: int, src: int, dst: int, lines: int, cu_lo: int, cu_n: int) -> Collective:
    b = CollectiveBuilder(n_gpus, f"p2p_{src}_{dst}_{lines}")
    b.add(src, dst, lines, cu_lo, cu_n)
    return b.build()


# ---------------------------------------------------------------------------------------------
# Control-path variants (PAPER.md:L137-138 SemaphoreAcquire / SemaphoreRelease,
# L165 "only wavefront zero" issues control messages, L279-289 put vs get).  Both are transforms of
# a step DAG into another step DAG: the control messages become one-line steps of their own, so
# they queue in the same FIFOs and use the same links as the data (no method arithmetic here).
# ---------------------------------------------------------------------------------------------
def put_with_signal(coll: Collective) -> Collective:
    """put + signal ("SemaphoreReleaseOp should follow after a remote Store", the
    receiver "must run SemaphoreAcquireOp before" it goes on): every step p that some step waits
    for with a DELIVERED dependency gets a SemaphoreRelease step right behind it -- one line from
    wavefront zero of p's first CU (cu_n = 1: the one line falls to wavefront 0 of that CU, R11)
    to the same destination, released when p's last line has been issued (ISSUED dependency on p)
    -- and the waiting steps wait for the DELIVERED stamp of that signal instead of p's.  The
    acquire is the local observation of the delivered semaphore line."""
    from .types import DEP_ISSUED
    S = coll.n_steps
    waited = set()
    for s in range(S):
        for i in range(int(coll.dep_ptr[s]), int(coll.dep_ptr[s + 1])):
            if int(coll.dep_kind[i]) == DEP_DELIVERED:
                waited.add(int(coll.dep_step[i]))
    b = CollectiveBuilder(coll.n_gpus, coll.name + "+signal")
    new_id, sig_id = {}, {}
    for s in range(S):
        deps = []
        for i in range(int(coll.dep_ptr[s]), int(coll.dep_ptr[s + 1])):
            p, kind = int(coll.dep_step[i]), int(coll.dep_kind[i])
            deps.append((sig_id[p], DEP_DELIVERED) if kind == DEP_DELIVERED else (new_id[p], kind))
        new_id[s] = b.add(coll.owner[s], coll.dst[s], coll.lines[s], coll.cu_lo[s], coll.cu_n[s], deps)
        if s in waited:
            sig_id[s] = b.add(coll.owner[s], coll.dst[s], 1, coll.cu_lo[s], 1, [(new_id[s], DEP_ISSUED)])
    return b.build()


def as_get(coll: Collective, chunk_lines: int = 0) -> Collective:
    """get ("requests to the remote GPU to send data"): every transfer p = (o -> d, n
    lines) is initiated by its destination.  d sends a one-line request to o from wavefront zero of
    p's first CU (posted as early as p's own dependencies on d allow: none here, the request is
    free), and o's response carries the data, released when the request has been DELIVERED at o and
    p's original dependencies hold.  With chunk_lines > 0 a transfer is cut into chunks of that many
    lines, one request each (the reading taken: one request per chunk, not per line)."""
    S = coll.n_steps
    b = CollectiveBuilder(coll.n_gpus, coll.name + "+get")
    last_id = {}                                  # original step -> all its response chunk steps
    for s in range(S):
        o, d, n = int(coll.owner[s]), int(coll.dst[s]), int(coll.lines[s])
        base = []
        for i in range(int(coll.dep_ptr[s]), int(coll.dep_ptr[s + 1])):
            p, kind = int(coll.dep_step[i]), int(coll.dep_kind[i])
            base += [(q, kind) for q in last_id[p]]
        sizes = [n] if chunk_lines <= 0 else [min(chunk_lines, n - x) for x in range(0, n, chunk_lines)]
        ids = []
        for m in sizes:
            req = b.add(d, o, 1, coll.cu_lo[s], 1)
            ids.append(b.add(o, d, m, coll.cu_lo[s], coll.cu_n[s], base + [(req, DEP_DELIVERED)]))
        last_id[s] = ids
    return b.build()


def with_barriers(coll: Collective, cus: int, scope: str = "workgroup", kind: int = 2) -> Collective:
    """NopOp / BarrierOp / memory fence between the operations of a GPU ("halts the
    execution of a workgroup until all its wavefronts reach this operation", BarrierOp "inter-workgroup
    synchronization"; L150 MemcpyOp "Waitcnt ... to enforce a memory fence") as dependencies between the
    steps a GPU owns: every step waits for the previous step on each of its CUs (scope "workgroup": NopOp
    between the operations of a workgroup) or for the previous step of every CU of the GPU (scope "gpu":
    BarrierOp).  kind 2 (ISSUED): the wavefronts have dispatched all requests of the previous operation;
    kind 1 (ACKED): its requests have also completed (Waitcnt 0, a fence).  `cus` = CUs per GPU."""
    S = coll.n_steps
    b = CollectiveBuilder(coll.n_gpus, coll.name + f"+{scope}_barriers{kind}")
    last = [[-1] * cus for _ in range(coll.n_gpus)]        # last step seen on (GPU, CU)
    for s in range(S):
        o, lo, cn = int(coll.owner[s]), int(coll.cu_lo[s]), int(coll.cu_n[s])
        deps = [(int(coll.dep_step[i]), int(coll.dep_kind[i])) for i in range(int(coll.dep_ptr[s]), int(coll.dep_ptr[s + 1]))]
        rng = range(lo, lo + cn) if scope == "workgroup" else range(cus)
        prev = sorted({last[o][cu] for cu in rng if last[o][cu] >= 0})
        deps += [(p, kind) for p in prev if (p, kind) not in deps]
        sid = b.add(o, coll.dst[s], coll.lines[s], lo, cn, deps)
        assert sid == s
        for cu in range(lo, lo + cn):
            last[o][cu] = s
    return b.build()
