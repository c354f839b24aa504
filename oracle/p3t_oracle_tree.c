/* oracle/p3t_oracle_tree.c -- TEST INFRASTRUCTURE (see p3t_oracle.h).
 * Part II: the reference octree, one step after the other, in the order of DESIGN.md R-S1..R-S8.
 * The paper says only "a GPU-enabled tree code provided by the BONSAI library ... opening angle
 * theta"; the rules below are this repo's readings and are shared with the GPU
 * path as RULES, never as code.  Integer stages and fp32 predicates are bit-specified; moments are
 * summed in fp64 over the particles of each cell (the definition) and rounded once to fp32;
 * forces are evaluated in fp64.  Compile with -ffp-contract=off.
 */
#include "p3t_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include "p3t_oracle_tree_priv.h"

/* R-S2: bit 3k+2 <- bit k of gx, 3k+1 <- gy, 3k <- gz */
uint64_t p3t_o_interleave(uint32_t gx, uint32_t gy, uint32_t gz, int bits)
{
    uint64_t key = 0;
    for (int k = 0; k < bits; ++k) {
        key |= (uint64_t)((gx >> k) & 1u) << (3 * k + 2);
        key |= (uint64_t)((gy >> k) & 1u) << (3 * k + 1);
        key |= (uint64_t)((gz >> k) & 1u) << (3 * k);
    }
    return key;
}

typedef struct { uint64_t key; uint32_t idx; } kv_t;
static int kv_cmp(const void* a, const void* b)
{
    const kv_t *p = (const kv_t*)a, *q = (const kv_t*)b;
    if (p->key != q->key) return p->key < q->key ? -1 : 1;
    return p->idx < q->idx ? -1 : (p->idx > q->idx);           /* R-S3: ties by original index */
}

static void grow_nodes(p3t_o_tree* t)
{
    int64_t c = t->cap ? 2 * t->cap : 1024;
    t->level = realloc(t->level, sizeof(int32_t) * c); t->begin = realloc(t->begin, sizeof(int32_t) * c);
    t->end = realloc(t->end, sizeof(int32_t) * c); t->first_child = realloc(t->first_child, sizeof(int32_t) * c);
    t->n_child = realloc(t->n_child, sizeof(int32_t) * c); t->prefix = realloc(t->prefix, sizeof(uint64_t) * c);
    t->cap = c;
}
static int64_t push_node(p3t_o_tree* t, int level, int32_t b, int32_t e, uint64_t prefix)
{
    if (t->nn == t->cap) grow_nodes(t);
    int64_t k = t->nn++;
    t->level[k] = level; t->begin[k] = b; t->end[k] = e; t->first_child[k] = -1; t->n_child[k] = 0; t->prefix[k] = prefix;
    return k;
}
static void push_group(p3t_o_tree* t, int32_t b, int32_t e)
{
    if (t->ng == t->gcap) {
        int64_t c = t->gcap ? 2 * t->gcap : 1024;
        t->gbegin = realloc(t->gbegin, sizeof(int32_t) * c); t->gend = realloc(t->gend, sizeof(int32_t) * c);
        t->gcap = c;
    }
    t->gbegin[t->ng] = b; t->gend[t->ng] = e; t->ng++;
}

/* R-S5 groups ("sibling runs"): below the first cell with more than NCRIT particles, consecutive
 * children with <= NCRIT particles are packed greedily, in octant order, into runs of <= NCRIT. */
static void make_groups(p3t_o_tree* t, int64_t node)
{
    int32_t b = t->begin[node], e = t->end[node];
    if (t->n_child[node] == 0) {                  /* over-full leaf at the deepest level */
        for (int32_t s = b; s < e; s += t->ncrit) push_group(t, s, s + t->ncrit < e ? s + t->ncrit : e);
        return;
    }
    int32_t rb = -1, re = -1;                     /* current run */
    for (int c = 0; c < t->n_child[node]; ++c) {
        int64_t ch = t->first_child[node] + c;
        int32_t cnt = t->end[ch] - t->begin[ch];
        if (cnt > t->ncrit) {
            if (rb >= 0) { push_group(t, rb, re); rb = -1; }
            make_groups(t, ch);
        } else if (rb >= 0 && (re - rb) + cnt <= t->ncrit) {
            re = t->end[ch];
        } else {
            if (rb >= 0) push_group(t, rb, re);
            rb = t->begin[ch]; re = t->end[ch];
        }
    }
    if (rb >= 0) push_group(t, rb, re);
}

p3t_o_tree* p3t_o_tree_build(int64_t n, const float* pm, int key_bits, int nleaf, int ncrit)
{
    if (n < 1 || (key_bits != 30 && key_bits != 63) || nleaf < 1 || ncrit < nleaf) return NULL;
    p3t_o_tree* t = (p3t_o_tree*)calloc(1, sizeof(*t));
    t->n = n; t->bits = key_bits / 3; t->nleaf = nleaf; t->ncrit = ncrit;
    const int B = t->bits;

    /* R-S1 cube: lo = per-axis minimum; ext = max_a fl32(hi_a - lo_a); side = 2^e with
     * ext = f 2^e, f in [1/2, 1) (frexpf), so side > ext; ext = 0 -> side = 1. */
    float lo[3], hi[3];
    for (int a = 0; a < 3; ++a) lo[a] = hi[a] = pm[a];
    for (int64_t i = 1; i < n; ++i)
        for (int a = 0; a < 3; ++a) {
            float v = pm[4 * i + a];
            if (v < lo[a]) lo[a] = v;
            if (v > hi[a]) hi[a] = v;
        }
    float ext = 0.0f;
    for (int a = 0; a < 3; ++a) { float d = hi[a] - lo[a]; if (d > ext) ext = d; }
    int ex = 0; float side = 1.0f;
    if (ext > 0.0f) { (void)frexpf(ext, &ex); side = ldexpf(1.0f, ex); }
    for (int a = 0; a < 3; ++a) t->lo[a] = lo[a];
    t->side = side;

    /* R-S2 keys: g_a = min(2^B - 1, (int) fl32( fl32(x_a - lo_a) * scale )), scale = 2^B / side */
    const float scale = ldexpf(1.0f, B) / side;            /* power of two: exact */
    const uint32_t gmax = (1u << B) - 1u;
    kv_t* kv = (kv_t*)malloc(sizeof(kv_t) * (size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        uint32_t g[3];
        for (int a = 0; a < 3; ++a) {
            float d = pm[4 * i + a] - lo[a];
            float s = d * scale;
            int64_t q = (int64_t)s;                          /* truncation */
            g[a] = q > (int64_t)gmax ? gmax : (uint32_t)q;
        }
        kv[i].key = p3t_o_interleave(g[0], g[1], g[2], B);
        kv[i].idx = (uint32_t)i;
    }
    /* R-S3 order */
    qsort(kv, (size_t)n, sizeof(kv_t), kv_cmp);
    t->keys = (uint64_t*)malloc(sizeof(uint64_t) * (size_t)n);
    t->order = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)n);
    t->spm = (float*)malloc(sizeof(float) * 4 * (size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        t->keys[i] = kv[i].key; t->order[i] = kv[i].idx;
        memcpy(t->spm + 4 * i, pm + 4 * (int64_t)kv[i].idx, 4 * sizeof(float));
    }
    free(kv);

    /* R-S4 topology: a cell is (level, 3*level-bit prefix); root is level 0.  A cell with more than
     * NLEAF particles and level < B is internal; its children are its non-empty octants in octant
     * order.  Anything else is a leaf.  Breadth-first numbering. */
    push_node(t, 0, 0, (int32_t)n, 0);
    for (int64_t k = 0; k < t->nn; ++k) {
        int lev = t->level[k]; int32_t b = t->begin[k], e = t->end[k];
        if (lev > t->max_level) t->max_level = lev;
        if (e - b <= nleaf || lev >= B) { t->n_leaves++; continue; }
        int shift = 3 * (B - lev - 1);
        int32_t s = b;
        while (s < e) {
            uint64_t oct = (t->keys[s] >> shift) & 7u;
            int32_t q = s;
            while (q < e && ((t->keys[q] >> shift) & 7u) == oct) ++q;
            int64_t ch = push_node(t, lev + 1, s, q, (t->prefix[k] << 3) | oct);
            if (t->n_child[k] == 0) t->first_child[k] = (int32_t)ch;
            t->n_child[k]++;
            s = q;
        }
    }

    /* R-S6 moments, from the definition, per cell, over its own particles, in fp64:
     * M = sum m; COM = sum m x / M; Q_ab = sum m (3 d_a d_b - |d|^2 delta_ab), d = x - COM
     * (traceless quadrupole; order xx yy zz xy xz yz); tight AABB = exact min/max;
     * delta = |COM - c_geo|, c_geo,a = lo_a + (p_a + 1/2) l, l = side / 2^level.
     * M, COM, Q, delta are rounded once to fp32.  M = 0 (all masses zero): reading R-S6a below.
     * SURVEY 8f NEXT-4 (octupole variant): T_abc = sum m d_a d_b d_c, the raw third moment about the COM,
     * order xxx yyy zzz xxy xxz xyy yyz xzz yzz xyz, likewise rounded once to fp32. */
    int64_t nn = t->nn;
    t->mass = malloc(sizeof(double) * nn); t->com = malloc(sizeof(double) * 3 * nn); t->quad = malloc(sizeof(double) * 6 * nn);
    t->fcom_m = malloc(sizeof(float) * 4 * nn); t->fquad = malloc(sizeof(float) * 6 * nn);
    t->oct = malloc(sizeof(double) * 10 * nn); t->foct = malloc(sizeof(float) * 10 * nn);
    t->clo = malloc(sizeof(float) * 3 * nn); t->chi = malloc(sizeof(float) * 3 * nn); t->delta = malloc(sizeof(float) * nn);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t k = 0; k < nn; ++k) {
        int32_t b = t->begin[k], e = t->end[k];
        double M = 0, s[3] = { 0, 0, 0 };
        float clo[3], chi[3];
        for (int a = 0; a < 3; ++a) clo[a] = chi[a] = t->spm[4 * (int64_t)b + a];
        for (int32_t i = b; i < e; ++i) {
            const float* p = t->spm + 4 * (int64_t)i;
            double m = p[3];
            M += m;
            for (int a = 0; a < 3; ++a) {
                s[a] += m * (double)p[a];
                if (p[a] < clo[a]) clo[a] = p[a];
                if (p[a] > chi[a]) chi[a] = p[a];
            }
        }
        double c[3] = { s[0] / M, s[1] / M, s[2] / M };
        if (M == 0.0)                      /* reading R-S6a: a cell of massless particles (tracers) has no centre of mass; */
            for (int a = 0; a < 3; ++a)    /* it takes the position of its first particle in sorted order (Q = 0, delta from it) */
                c[a] = t->spm[4 * (int64_t)b + a];
        double Q[6] = { 0, 0, 0, 0, 0, 0 }, T[10] = { 0, 0, 0, 0, 0, 0, 0, 0, 0, 0 };
        for (int32_t i = b; i < e; ++i) {
            const float* p = t->spm + 4 * (int64_t)i;
            double m = p[3], dx = p[0] - c[0], dy = p[1] - c[1], dz = p[2] - c[2];
            double d2 = dx * dx + dy * dy + dz * dz;
            Q[0] += m * (3 * dx * dx - d2); Q[1] += m * (3 * dy * dy - d2); Q[2] += m * (3 * dz * dz - d2);
            Q[3] += m * 3 * dx * dy; Q[4] += m * 3 * dx * dz; Q[5] += m * 3 * dy * dz;
            T[0] += m * dx * dx * dx; T[1] += m * dy * dy * dy; T[2] += m * dz * dz * dz;
            T[3] += m * dx * dx * dy; T[4] += m * dx * dx * dz; T[5] += m * dx * dy * dy;
            T[6] += m * dy * dy * dz; T[7] += m * dx * dz * dz; T[8] += m * dy * dz * dz; T[9] += m * dx * dy * dz;
        }
        /* integer cell coordinates from the prefix (x highest in every 3-bit digit) */
        int lev = t->level[k];
        uint32_t p3[3] = { 0, 0, 0 };
        for (int q = 0; q < lev; ++q) {
            uint64_t dgt = (t->prefix[k] >> (3 * q)) & 7u;
            p3[0] |= (uint32_t)((dgt >> 2) & 1u) << q; p3[1] |= (uint32_t)((dgt >> 1) & 1u) << q; p3[2] |= (uint32_t)(dgt & 1u) << q;
        }
        double l = (double)t->side / (double)(1ull << lev), dd = 0;
        for (int a = 0; a < 3; ++a) {
            double cg = (double)t->lo[a] + ((double)p3[a] + 0.5) * l;
            dd += (c[a] - cg) * (c[a] - cg);
        }
        t->mass[k] = M;
        for (int a = 0; a < 3; ++a) { t->com[3 * k + a] = c[a]; t->fcom_m[4 * k + a] = (float)c[a]; t->clo[3 * k + a] = clo[a]; t->chi[3 * k + a] = chi[a]; }
        t->fcom_m[4 * k + 3] = (float)M;
        for (int q = 0; q < 6; ++q) { t->quad[6 * k + q] = Q[q]; t->fquad[6 * k + q] = (float)Q[q]; }
        for (int q = 0; q < 10; ++q) { t->oct[10 * k + q] = T[q]; t->foct[10 * k + q] = (float)T[q]; }
        t->delta[k] = (float)sqrt(dd);
    }

    /* R-S5 groups and their tight boxes */
    if (n <= ncrit) push_group(t, 0, (int32_t)n); else make_groups(t, 0);
    t->glo = malloc(sizeof(float) * 3 * t->ng); t->ghi = malloc(sizeof(float) * 3 * t->ng);
    for (int64_t g = 0; g < t->ng; ++g)
        for (int a = 0; a < 3; ++a) {
            float mn = t->spm[4 * (int64_t)t->gbegin[g] + a], mx = mn;
            for (int32_t i = t->gbegin[g]; i < t->gend[g]; ++i) {
                float v = t->spm[4 * (int64_t)i + a];
                if (v < mn) mn = v;
                if (v > mx) mx = v;
            }
            t->glo[3 * g + a] = mn; t->ghi[3 * g + a] = mx;
        }
    return t;
}

void p3t_o_tree_free(p3t_o_tree* t)
{
    if (!t) return;
    free(t->keys); free(t->order); free(t->spm); free(t->level); free(t->begin); free(t->end);
    free(t->first_child); free(t->n_child); free(t->prefix); free(t->mass); free(t->com); free(t->quad);
    free(t->fcom_m); free(t->fquad); free(t->clo); free(t->chi); free(t->delta); free(t->oct); free(t->foct);
    free(t->gbegin); free(t->gend); free(t->glo); free(t->ghi); free(t);
}

void p3t_o_tree_sizes(const p3t_o_tree* t, int64_t out[6])
{
    out[0] = t->n; out[1] = t->nn; out[2] = t->n_leaves; out[3] = t->max_level; out[4] = t->ng; out[5] = t->bits;
}
void p3t_o_tree_cube(const p3t_o_tree* t, float lo[3], float* side)
{
    for (int a = 0; a < 3; ++a) lo[a] = t->lo[a];
    *side = t->side;
}
void p3t_o_tree_keys(const p3t_o_tree* t, uint64_t* k, uint32_t* o)
{
    memcpy(k, t->keys, sizeof(uint64_t) * t->n); memcpy(o, t->order, sizeof(uint32_t) * t->n);
}
void p3t_o_tree_nodes(const p3t_o_tree* t, int32_t* level, int32_t* begin, int32_t* end, int32_t* fc, int32_t* nc)
{
    size_t s = sizeof(int32_t) * t->nn;
    memcpy(level, t->level, s); memcpy(begin, t->begin, s); memcpy(end, t->end, s);
    memcpy(fc, t->first_child, s); memcpy(nc, t->n_child, s);
}
void p3t_o_tree_moments(const p3t_o_tree* t, float* com_m, float* quad, float* clo, float* chi, float* delta)
{
    memcpy(com_m, t->fcom_m, sizeof(float) * 4 * t->nn); memcpy(quad, t->fquad, sizeof(float) * 6 * t->nn);
    memcpy(clo, t->clo, sizeof(float) * 3 * t->nn); memcpy(chi, t->chi, sizeof(float) * 3 * t->nn);
    memcpy(delta, t->delta, sizeof(float) * t->nn);
}
void p3t_o_tree_octupoles(const p3t_o_tree* t, float* foct, double* oct)
{
    if (foct) memcpy(foct, t->foct, sizeof(float) * 10 * t->nn);
    if (oct) memcpy(oct, t->oct, sizeof(double) * 10 * t->nn);
}

void p3t_o_tree_moments64(const p3t_o_tree* t, double* mass, double* com, double* quad)
{
    memcpy(mass, t->mass, sizeof(double) * t->nn); memcpy(com, t->com, sizeof(double) * 3 * t->nn);
    memcpy(quad, t->quad, sizeof(double) * 6 * t->nn);
}
void p3t_o_tree_groups(const p3t_o_tree* t, int32_t* b, int32_t* e, float* glo, float* ghi)
{
    memcpy(b, t->gbegin, sizeof(int32_t) * t->ng); memcpy(e, t->gend, sizeof(int32_t) * t->ng);
    memcpy(glo, t->glo, sizeof(float) * 3 * t->ng); memcpy(ghi, t->ghi, sizeof(float) * 3 * t->ng);
}
