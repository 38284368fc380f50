/*
 * Native helper for the seeded workload generators (workloads.py).
 *
 * Holds NO annealing arithmetic: only sequential greedy graph colouring, which
 * is an INPUT of the method (BASELINE.json configs: "greedy colouring shipped
 * with the input") and is too slow as a Python loop at n = 1e6.
 * Served to both the oracle tests and the CUDA path through workloads.py.
 */
#include <stdint.h>
#include <stdlib.h>

/* Sequential greedy colouring: visit vertices in `order`, give each the
 * smallest colour not used by an already-coloured neighbour.
 * Returns the number of colours used, or -1 on allocation failure. */
int32_t wl_greedy_colour(int32_t n, const int64_t *row_ptr, const int32_t *col,
                         const int32_t *order, int32_t *colour_out)
{
    int32_t *mark = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n + 1));
    if (!mark) return -1;
    for (int32_t c = 0; c <= n; ++c) mark[c] = -1;
    for (int32_t i = 0; i < n; ++i) colour_out[i] = -1;
    int32_t n_colours = 0;
    for (int32_t k = 0; k < n; ++k) {
        int32_t v = order[k];
        for (int64_t e = row_ptr[v]; e < row_ptr[v + 1]; ++e) {
            int32_t c = colour_out[col[e]];
            if (c >= 0) mark[c] = v;
        }
        int32_t c = 0;
        while (mark[c] == v) ++c;
        colour_out[v] = c;
        if (c + 1 > n_colours) n_colours = c + 1;
    }
    free(mark);
    return n_colours;
}
