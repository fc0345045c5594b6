/* Test-only driver: runs oracle_run() of oracle/astra_oracle.c on one design point read from a flat
 * binary file, so that the oracle can be executed under -fsanitize=address,undefined (SURVEY.md
 * section 5) without loading a sanitized shared object into the Python interpreter.
 * File layout (all little-endian u32 unless noted): G, NS, S, ND, cus, wpc, K, H, then u64
 * max_cycles, then node_latency[V], row_ptr[V+1], head[E], bw_q8[E], latency[E], owner[S], dst[S],
 * lines[S], cu_lo[S], cu_n[S], dep_ptr[S+1], dep_step[ND], dep_kind[ND] (u8).
 * Prints: status completion total_lines, then 4*S timestamps, then E link counts. */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

int oracle_run(uint32_t, uint32_t, const uint32_t *, const uint32_t *, const uint32_t *, const uint32_t *,
               const uint32_t *, uint32_t, const uint32_t *, const uint32_t *, const uint32_t *,
               const uint32_t *, const uint32_t *, const uint32_t *, const uint32_t *, const uint8_t *,
               uint32_t, uint32_t, uint32_t, uint32_t, uint64_t, uint32_t, int32_t *, uint64_t *, uint64_t *,
               uint64_t *, uint64_t *, uint64_t *, uint64_t *, uint64_t, uint64_t *);

static uint32_t *rd32(FILE *f, size_t n) {
    uint32_t *p = (uint32_t *)malloc(sizeof(uint32_t) * (n ? n : 1));
    if (!p || fread(p, sizeof(uint32_t), n, f) != n) { fprintf(stderr, "short read\n"); exit(3); }
    return p;
}

int main(int argc, char **argv) {
    if (argc < 3) return 2;
    FILE *f = fopen(argv[1], "rb");
    if (!f) return 2;
    uint32_t flags = (uint32_t)atoi(argv[2]);
    uint32_t *h = rd32(f, 8);
    uint32_t G = h[0], NS = h[1], S = h[2], ND = h[3], V = G + NS;
    uint64_t max_cycles;
    if (fread(&max_cycles, 8, 1, f) != 1) return 3;
    uint32_t *node_latency = rd32(f, V), *row_ptr = rd32(f, V + 1);
    uint32_t E = row_ptr[V];
    uint32_t *head = rd32(f, E), *bw = rd32(f, E), *lat = rd32(f, E);
    uint32_t *owner = rd32(f, S), *dst = rd32(f, S), *lines = rd32(f, S), *cu_lo = rd32(f, S), *cu_n = rd32(f, S);
    uint32_t *dep_ptr = rd32(f, S + 1), *dep_step = rd32(f, ND);
    uint8_t *dep_kind = (uint8_t *)malloc(ND ? ND : 1);
    if (fread(dep_kind, 1, ND, f) != ND) return 3;
    fclose(f);
    uint64_t *ts = (uint64_t *)malloc(sizeof(uint64_t) * (4 * (size_t)S + 1));
    uint64_t *ll = (uint64_t *)malloc(sizeof(uint64_t) * ((size_t)E + 1));
    uint64_t stats[8], completion = 0, total = 0, trlen = 0;
    int32_t status = -1;
    int rc = oracle_run(G, NS, node_latency, row_ptr, head, bw, lat, S, owner, dst, lines, cu_lo, cu_n,
                        dep_ptr, dep_step, dep_kind, h[4], h[5], h[6], h[7], max_cycles, flags,
                        &status, &completion, &total, ts, ll, stats, NULL, 0, &trlen);
    if (rc) { fprintf(stderr, "oracle_run rc %d\n", rc); return 4; }
    printf("%d %llu %llu\n", status, (unsigned long long)completion, (unsigned long long)total);
    for (uint32_t i = 0; i < 4 * S; i++) printf("%llu ", (unsigned long long)ts[i]);
    printf("\n");
    for (uint32_t e = 0; e < E; e++) printf("%llu ", (unsigned long long)ll[e]);
    printf("\n");
    free(h); free(node_latency); free(row_ptr); free(head); free(bw); free(lat); free(owner); free(dst);
    free(lines); free(cu_lo); free(cu_n); free(dep_ptr); free(dep_step); free(dep_kind); free(ts); free(ll);
    return 0;
}
