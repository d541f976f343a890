/* Config 5 -- single-source shortest paths by frontier Bellman-Ford.
 * TEST INFRASTRUCTURE (see oracle.h).  Source: PAPER.md:220 (section 5.1, workload 6: "Bellman-Ford graph traversal with
 * frontier-based relaxation"); SURVEY.md 8(f)4.  The paper gives no more than that sentence; readings S5-1..S5-4 in
 * DESIGN.md section 2:
 *   S5-1  graph in CSR (row_ptr[V+1], col[E], w[E]), directed, weights int32 >= 0, every path sum < 2^31
 *   S5-2  dist[src] = 0, unreachable vertices keep ORACLE_SSSP_INF = 2^31 - 1
 *   S5-3  frontier F_0 = {src}; round t relaxes every edge out of F_t against the distances as they were when the round
 *         began (synchronous rounds); F_{t+1} = vertices whose distance got smaller in round t; stop when F is empty
 *   S5-4  the result that is unique is dist[]; the round count depends on the relaxation order and is reported beside it
 * Written out step by step: no queue tricks, no early exit, O(rounds * (V + E)). */
#include "oracle.h"
#include <string.h>

int32_t oracle_sssp_frontier_bf(const int32_t *row_ptr, const int32_t *col, const int32_t *w, int64_t V, int32_t src,
                                int32_t *dist, int32_t *scratch) {
    int32_t *next = scratch;              /* distances at the end of the round                     */
    uint8_t *in_f = (uint8_t *)(scratch + V);      /* frontier of this round                        */
    uint8_t *out_f = in_f + V;                     /* frontier of the next round                    */
    for (int64_t v = 0; v < V; ++v) {
        dist[v] = ORACLE_SSSP_INF;
        in_f[v] = 0;
    }
    if (V <= 0 || src < 0 || src >= V) return 0;
    dist[src] = 0;
    in_f[src] = 1;
    int32_t rounds = 0;
    for (;;) {
        int any = 0;
        for (int64_t v = 0; v < V; ++v) any |= in_f[v];
        if (!any) break;
        rounds += 1;
        memcpy(next, dist, (size_t)V * sizeof(int32_t));
        memset(out_f, 0, (size_t)V);
        for (int64_t u = 0; u < V; ++u) {
            if (!in_f[u]) continue;
            for (int32_t e = row_ptr[u]; e < row_ptr[u + 1]; ++e) {
                int32_t v = col[e];
                int32_t nd = dist[u] + w[e];       /* dist[u] is finite: u entered the frontier by getting one */
                if (nd < next[v]) {
                    next[v] = nd;
                    out_f[v] = 1;
                }
            }
        }
        memcpy(dist, next, (size_t)V * sizeof(int32_t));
        memcpy(in_f, out_f, (size_t)V);
    }
    return rounds;
}

/* One job: image = [V, E, src, 0][row_ptr int32[V+1]][col int32[E]][w int32[E]] -> out = [dist int32[V]][rounds, 0, 0, 0].
 * scratch: int32[2V] + 2V bytes. */
void oracle_sssp_job(const int32_t *image, int32_t *out, int32_t *scratch) {
    int64_t V = image[0], E = image[1];
    int32_t src = image[2];
    const int32_t *row_ptr = image + 4, *col = row_ptr + V + 1, *w = col + E;
    int32_t rounds = oracle_sssp_frontier_bf(row_ptr, col, w, V, src, out, scratch);
    out[V] = rounds;
    out[V + 1] = out[V + 2] = out[V + 3] = 0;
}
