/* oracle/p3t_oracle_grid.c -- TEST INFRASTRUCTURE (see p3t_oracle.h).
 * Part I, continued: the neighbour lists of PAPER.md:66, :113 at sizes where the O(N^2) double loop
 * of p3t_o_neighbours takes hours ("brute force for N <= 131 072 and a uniform cell
 * grid, cell edge >= r_out, independent of the octree, above that").
 *
 * The result is DEFINED by the brute force: L(i) = { j != i : d2(i, j) < fl(r_out * r_out) } with the
 * fp32 predicate of reading R10.  The grid only restricts the candidates j that are tested:
 *   cells of edge h = 1.001 r_out (or larger, when the box would need more than 2^20 cells per axis);
 *   cell of a particle: c_a = floor((x_a - lo_a) / h) in fp64 (fp32 -> fp64 is exact);
 *   candidates of i: the particles of the 27 cells |c_a(j) - c_a(i)| <= 1.
 * Completeness: a particle outside those cells differs from i by at least 2 in one cell coordinate, so
 * |x_a(j) - x_a(i)| > h = 1.001 r_out on that axis; the fp32 d2 of R10 is >= fl(dx)^2 (fma and the sum of
 * squares are monotone), fl(dx) >= |dx| (1 - 2^-24) and fl(r_out * r_out) <= r_out^2 (1 + 2^-24): the
 * margin 1.001^2 is far outside those roundings, so no member is missed.  Every candidate then goes
 * through exactly the predicate of p3t_o_neighbours.  Pinned against p3t_o_neighbours at small N
 * (tests/test_oracle_direct.py): Plummer, King, duplicated points, a lattice, r_out > box.
 */
#include "p3t_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef struct { uint64_t key; int32_t id; } cell_ent;

static int cmp_ent(const void* a, const void* b)
{
    const cell_ent* x = (const cell_ent*)a; const cell_ent* y = (const cell_ent*)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return x->id < y->id ? -1 : (x->id > y->id ? 1 : 0);
}
static int cmp_i32(const void* a, const void* b)
{
    int32_t x = *(const int32_t*)a, y = *(const int32_t*)b;
    return x < y ? -1 : (x > y ? 1 : 0);
}

/* first entry with key >= k */
static int64_t lower_bound(const cell_ent* e, int64_t n, uint64_t k)
{
    int64_t lo = 0, hi = n;
    while (lo < hi) { int64_t mid = (lo + hi) >> 1; if (e[mid].key < k) lo = mid + 1; else hi = mid; }
    return lo;
}

/* Same contract as p3t_o_neighbours with fp32_predicate = 1: counts[nt] always; rows (ascending j) back to
 * back in indices when it is not NULL.  Returns the total, or -1 on allocation failure / bad input. */
int64_t p3t_o_neighbours_grid(int64_t n, const float* pm, float r_out,
                              int64_t nt, const int64_t* targets, int64_t* counts, int32_t* indices)
{
    if (n < 1 || !(r_out > 0.0f)) return -1;
    const float rout2f = r_out * r_out;
    double lo[3] = { pm[0], pm[1], pm[2] }, hi[3] = { pm[0], pm[1], pm[2] };
    for (int64_t i = 0; i < n; ++i)
        for (int a = 0; a < 3; ++a) {
            double v = pm[4 * i + a];
            if (v < lo[a]) lo[a] = v;
            if (v > hi[a]) hi[a] = v;
        }
    double ext = 0.0;
    for (int a = 0; a < 3; ++a) if (hi[a] - lo[a] > ext) ext = hi[a] - lo[a];
    double h = 1.001 * (double)r_out;
    if (ext / h > 1048575.0) h = ext / 1048575.0;            /* at most 2^20 cells per axis: 60-bit cell keys */
    int64_t dim[3];
    for (int a = 0; a < 3; ++a) dim[a] = (int64_t)floor((hi[a] - lo[a]) / h) + 1;

    cell_ent* ent = (cell_ent*)malloc(sizeof(cell_ent) * (size_t)n);
    int64_t* cc = (int64_t*)malloc(sizeof(int64_t) * 3 * (size_t)n);
    if (!ent || !cc) { free(ent); free(cc); return -1; }
    for (int64_t i = 0; i < n; ++i) {
        for (int a = 0; a < 3; ++a) {
            int64_t c = (int64_t)floor(((double)pm[4 * i + a] - lo[a]) / h);
            if (c < 0) c = 0;
            if (c >= dim[a]) c = dim[a] - 1;
            cc[3 * i + a] = c;
        }
        ent[i].key = ((uint64_t)cc[3 * i] * (uint64_t)dim[1] + (uint64_t)cc[3 * i + 1]) * (uint64_t)dim[2] + (uint64_t)cc[3 * i + 2];
        ent[i].id = (int32_t)i;
    }
    qsort(ent, (size_t)n, sizeof(cell_ent), cmp_ent);

    int64_t total = 0;
    for (int pass = 0; pass < 2; ++pass) {
        int64_t* off = NULL;
        if (pass == 1) {
            if (!indices) break;
            off = (int64_t*)malloc(sizeof(int64_t) * (size_t)(nt + 1));
            if (!off) { free(ent); free(cc); return -1; }
            off[0] = 0;
            for (int64_t t = 0; t < nt; ++t) off[t + 1] = off[t] + counts[t];
        }
        int64_t tot = 0;
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : tot)
        for (int64_t t = 0; t < nt; ++t) {
            const int64_t i = targets ? targets[t] : t;
            const float xi = pm[4 * i], yi = pm[4 * i + 1], zi = pm[4 * i + 2];
            int64_t c = 0, w = pass ? off[t] : 0;
            for (int64_t cx = cc[3 * i] - 1; cx <= cc[3 * i] + 1; ++cx) {
                if (cx < 0 || cx >= dim[0]) continue;
                for (int64_t cy = cc[3 * i + 1] - 1; cy <= cc[3 * i + 1] + 1; ++cy) {
                    if (cy < 0 || cy >= dim[1]) continue;
                    /* the three cells cz - 1 .. cz + 1 are consecutive keys */
                    int64_t z0 = cc[3 * i + 2] - 1, z1 = cc[3 * i + 2] + 1;
                    if (z0 < 0) z0 = 0;
                    if (z1 >= dim[2]) z1 = dim[2] - 1;
                    const uint64_t base = ((uint64_t)cx * (uint64_t)dim[1] + (uint64_t)cy) * (uint64_t)dim[2];
                    int64_t e = lower_bound(ent, n, base + (uint64_t)z0);
                    for (; e < n && ent[e].key <= base + (uint64_t)z1; ++e) {
                        const int64_t j = ent[e].id;
                        if (j == i) continue;                                   /* self excluded by index */
                        float dx = pm[4 * j] - xi, dy = pm[4 * j + 1] - yi, dz = pm[4 * j + 2] - zi;
                        float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));         /* reading R10, as in p3t_o_neighbours */
                        if (d2 < rout2f) {
                            if (pass) indices[w++] = (int32_t)j;
                            ++c;
                        }
                    }
                }
            }
            if (pass) qsort(indices + off[t], (size_t)c, sizeof(int32_t), cmp_i32);   /* rows ascending in j */
            else counts[t] = c;
            tot += c;
        }
        total = tot;
        free(off);
    }
    free(ent); free(cc);
    return total;
}
