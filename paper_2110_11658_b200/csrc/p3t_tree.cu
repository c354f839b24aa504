// p3t_tree.cu -- steps a4-a6: canonical octree topology, bottom-up monopole +
// traceless quadrupole moments, target groups.  ONE cooperative kernel (grid = co-resident CTAs,
// grid-wide barriers between levels) so that the whole stage is a single launch.
// Rules: DESIGN.md R-S4 (topology), R-S5 (sibling-run groups), R-S6 (moments).
// The paper gives no detail of this stage ("the BONSAI library").
#include "p3t_internal.cuh"
#include <cooperative_groups.h>
namespace cg = cooperative_groups;

#define TREE_THREADS 256

struct tree_args {
    const uint64_t* keys;      // sorted
    const float4* spm;         // sorted bodies
    int n, B, nleaf, ncrit, node_cap;
    int32_t *nlevel, *nbegin, *nend, *nfirst, *nnchild;
    double* m64;               // [node][10] = M, sum m x (3), Q about COM (6: xx yy zz xy xz yz)
    float4 *ncom, *nlo, *nhi, *nq0;
    float2* nq1;
    int2* nlink;
    int32_t* scan_tmp;         // [gridDim]
    uint8_t* gflag;            // [n + 16] zeroed by the host side
    int32_t* gbegin;           // [n + 1]
    p3t_devinfo* info;
};

// exclusive scan of one int per thread over the block; returns the exclusive prefix, *total = block sum
__device__ __forceinline__ int block_exscan(int v, int* total, int* s_warp /* [TREE_THREADS/32 + 1] */)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    __syncthreads();                       // protect s_warp from the previous use
    if (lane == 31) s_warp[w] = x;
    __syncthreads();
    int add = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < TREE_THREADS / 32; ++k) { int t = s_warp[k]; if (k < w) add += t; tot += t; }
    *total = tot;
    return add + x - v;
}

// child boundaries of an internal cell: pos[o] = first position in [b, e) whose octant digit at
// `shift` is >= o.  The seven binary searches run in lockstep over the same interval, so that every
// step issues seven independent key loads (the searches are latency-bound: one dependent L2 round
// trip per step) instead of seven times as many dependent ones.
__device__ __forceinline__ void child_bounds(const uint64_t* __restrict__ keys, int b, int e, int shift, int pos[9])
{
    int lo[7], hi[7];
#pragma unroll
    for (int o = 0; o < 7; ++o) { lo[o] = b; hi[o] = e; }
    for (int span = e - b; span > 0; span >>= 1) {       // floor(log2(e - b)) + 1 halvings empty every interval
#pragma unroll
        for (int o = 0; o < 7; ++o) {
            if (lo[o] < hi[o]) {
                const int m = (lo[o] + hi[o]) >> 1;
                if (((uint32_t)(keys[m] >> shift) & 7u) < (uint32_t)(o + 1)) lo[o] = m + 1; else hi[o] = m;
            }
        }
    }
    pos[0] = b; pos[8] = e;
#pragma unroll
    for (int o = 0; o < 7; ++o) pos[o + 1] = lo[o];
}

__device__ __forceinline__ uint32_t compact3(uint64_t x)   // inverse of the 3-way bit spread
{
    x &= 0x1249249249249249ull;
    x = (x | (x >> 2))  & 0x10c30c30c30c30c3ull;
    x = (x | (x >> 4))  & 0x100f00f00f00f00full;
    x = (x | (x >> 8))  & 0x001f0000ff0000ffull;
    x = (x | (x >> 16)) & 0x001f00000000ffffull;
    x = (x | (x >> 32)) & 0x1fffffull;
    return (uint32_t)x;
}

// R-S6 output of one cell: fp32 rounding of the fp64 moments, delta, and the walk's link word
__device__ void store_node(const tree_args& A, int k, int level, int b, int e, int first, int nchild,
                           double M, const double s[3], const double Q[6], const float clo[3], const float chi[3])
{
    double* m = A.m64 + (size_t)k * 10;
    m[0] = M; m[1] = s[0]; m[2] = s[1]; m[3] = s[2];
#pragma unroll
    for (int q = 0; q < 6; ++q) m[4 + q] = Q[q];
    const double c[3] = { s[0] / M, s[1] / M, s[2] / M };
    // geometric centre from the integer cell coordinates (prefix of the first key)
    const uint64_t prefix = level == 0 ? 0ull : (A.keys[b] >> (3 * (A.B - level)));
    const uint32_t p3[3] = { compact3(prefix >> 2), compact3(prefix >> 1), compact3(prefix) };
    const double l = (double)A.info->side / (double)(1ull << level);
    double dd = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double cgeo = (double)A.info->lo[a] + ((double)p3[a] + 0.5) * l;
        dd += (c[a] - cgeo) * (c[a] - cgeo);
    }
    A.ncom[k] = make_float4((float)c[0], (float)c[1], (float)c[2], (float)M);
    A.nlo[k]  = make_float4(clo[0], clo[1], clo[2], (float)sqrt(dd));
    A.nhi[k]  = make_float4(chi[0], chi[1], chi[2], __int_as_float(level));
    A.nq0[k]  = make_float4((float)Q[0], (float)Q[1], (float)Q[2], (float)Q[3]);
    A.nq1[k]  = make_float2((float)Q[4], (float)Q[5]);
    // link: internal -> (first child, n_child); leaf -> (begin, -count)
    A.nlink[k] = nchild > 0 ? make_int2(first, nchild) : make_int2(b, -(e - b));
}

__global__ void __launch_bounds__(TREE_THREADS) k_tree(tree_args A)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ int s_warp[TREE_THREADS / 32 + 1];
    __shared__ int s_run;
    const int nb = gridDim.x, bid = blockIdx.x, tid = threadIdx.x;
    const uint64_t* __restrict__ keys = A.keys;

    // ---------------- a4 topology, level by level (R-S4) ----------------
    if (bid == 0 && tid == 0) {
        A.nlevel[0] = 0; A.nbegin[0] = 0; A.nend[0] = A.n;
        A.info->level_begin[0] = 0; A.info->level_begin[1] = 1;
    }
    grid.sync();
    int lb = 0, le = 1, n_leaves = 0, max_level = 0, overflow = 0;
    for (int lev = 0; lev <= A.B; ++lev) {
        const int cnt = le - lb;
        const int per = (cnt + nb - 1) / nb;
        const int cb = min(le, lb + bid * per), ce = min(le, cb + per);
        const int shift = 3 * (A.B - lev - 1);
        // phase 1: child counts
        int bsum = 0;
        for (int k0 = cb; k0 < ce; k0 += TREE_THREADS) {
            int k = k0 + tid, c = 0;
            if (k < ce) {
                int b = A.nbegin[k], e = A.nend[k];
                if (e - b > A.nleaf && lev < A.B) {
                    int pos[9];
                    child_bounds(keys, b, e, shift, pos);
#pragma unroll
                    for (int o = 0; o < 8; ++o) c += pos[o + 1] > pos[o];
                }
                A.nnchild[k] = c;
            }
            bsum += c;
        }
        {
            int tot; (void)block_exscan(bsum, &tot, s_warp);
            if (tid == 0) A.scan_tmp[bid] = tot;
        }
        grid.sync();
        // phase 2: numbering and child records
        int before = 0, total = 0;
        for (int k = tid; k < nb; k += TREE_THREADS) { int t = A.scan_tmp[k]; total += t; if (k < bid) before += t; }
        { int t2; (void)block_exscan(before, &t2, s_warp); before = t2; }
        { int t2; (void)block_exscan(total, &t2, s_warp); total = t2; }
        if (le + total > A.node_cap) { overflow = 1; total = 0; }
        int run = le + before;
        for (int k0 = cb; k0 < ce && total > 0; k0 += TREE_THREADS) {
            int k = k0 + tid;
            int c = k < ce ? A.nnchild[k] : 0, tot;
            int first = run + block_exscan(c, &tot, s_warp);
            run += tot;
            if (k < ce) {
                if (c > 0) {
                    int b = A.nbegin[k], e = A.nend[k], pos[9];
                    child_bounds(keys, b, e, shift, pos);
                    int w = first;
#pragma unroll
                    for (int o = 0; o < 8; ++o)
                        if (pos[o + 1] > pos[o]) { A.nlevel[w] = lev + 1; A.nbegin[w] = pos[o]; A.nend[w] = pos[o + 1]; ++w; }
                    A.nfirst[k] = first;
                } else A.nfirst[k] = -1;
            }
        }
        if (total == 0) {     // every cell of this level is a leaf (or capacity hit)
            for (int k = cb + tid; k < ce; k += TREE_THREADS) A.nfirst[k] = -1;
        }
        if (bid == 0 && tid == 0) A.info->level_begin[lev + 2 < 24 ? lev + 2 : 23] = le + total;
        max_level = lev;
        grid.sync();
        lb = le; le = le + total;
        if (total == 0) break;
    }
    const int nn = le;
    if (bid == 0 && tid == 0) {
        A.info->n_nodes = nn; A.info->max_level = max_level; A.info->node_overflow = overflow;
    }

    // ---------------- a5 moments (R-S6): leaves from their particles, fp64 ----------------
    for (int k = bid * TREE_THREADS + tid; k < nn; k += nb * TREE_THREADS) {
        if (A.nnchild[k] != 0) continue;
        ++n_leaves;
        const int b = A.nbegin[k], e = A.nend[k];
        double M = 0.0, s[3] = { 0.0, 0.0, 0.0 };
        float4 p0 = A.spm[b];
        float clo[3] = { p0.x, p0.y, p0.z }, chi[3] = { p0.x, p0.y, p0.z };
        for (int i = b; i < e; ++i) {
            float4 p = A.spm[i];
            double m = p.w;
            M += m; s[0] += m * (double)p.x; s[1] += m * (double)p.y; s[2] += m * (double)p.z;
            clo[0] = fminf(clo[0], p.x); clo[1] = fminf(clo[1], p.y); clo[2] = fminf(clo[2], p.z);
            chi[0] = fmaxf(chi[0], p.x); chi[1] = fmaxf(chi[1], p.y); chi[2] = fmaxf(chi[2], p.z);
        }
        const double c[3] = { s[0] / M, s[1] / M, s[2] / M };
        double Q[6] = { 0, 0, 0, 0, 0, 0 };
        for (int i = b; i < e; ++i) {
            float4 p = A.spm[i];
            double m = p.w, dx = p.x - c[0], dy = p.y - c[1], dz = p.z - c[2];
            double d2 = dx * dx + dy * dy + dz * dz;
            Q[0] += m * (3 * dx * dx - d2); Q[1] += m * (3 * dy * dy - d2); Q[2] += m * (3 * dz * dz - d2);
            Q[3] += m * 3 * dx * dy; Q[4] += m * 3 * dx * dz; Q[5] += m * 3 * dy * dz;
        }
        store_node(A, k, A.nlevel[k], b, e, -1, 0, M, s, Q, clo, chi);
    }
    {   // leaf count
        int tot; (void)block_exscan(n_leaves, &tot, s_warp);
        if (tid == 0 && tot) atomicAdd(&A.info->n_leaves, tot);
    }
    grid.sync();
    // internal cells bottom-up: parallel-axis combination of the children, fp64
    for (int lev = max_level - 1; lev >= 0; --lev) {
        const int l0 = A.info->level_begin[lev], l1 = A.info->level_begin[lev + 1];
        for (int k = l0 + bid * TREE_THREADS + tid; k < l1; k += nb * TREE_THREADS) {
            const int nc = A.nnchild[k];
            if (nc == 0) continue;
            const int fc = A.nfirst[k];
            double M = 0.0, s[3] = { 0.0, 0.0, 0.0 };
            float clo[3] = { INFINITY, INFINITY, INFINITY }, chi[3] = { -INFINITY, -INFINITY, -INFINITY };
            for (int c = fc; c < fc + nc; ++c) {
                const double* m = A.m64 + (size_t)c * 10;
                M += m[0]; s[0] += m[1]; s[1] += m[2]; s[2] += m[3];
                float4 lo = A.nlo[c], hi = A.nhi[c];
                clo[0] = fminf(clo[0], lo.x); clo[1] = fminf(clo[1], lo.y); clo[2] = fminf(clo[2], lo.z);
                chi[0] = fmaxf(chi[0], hi.x); chi[1] = fmaxf(chi[1], hi.y); chi[2] = fmaxf(chi[2], hi.z);
            }
            const double cm[3] = { s[0] / M, s[1] / M, s[2] / M };
            double Q[6] = { 0, 0, 0, 0, 0, 0 };
            for (int c = fc; c < fc + nc; ++c) {
                const double* m = A.m64 + (size_t)c * 10;
                const double Mc = m[0];
                const double dx = m[1] / Mc - cm[0], dy = m[2] / Mc - cm[1], dz = m[3] / Mc - cm[2];
                const double d2 = dx * dx + dy * dy + dz * dz;
                Q[0] += m[4] + Mc * (3 * dx * dx - d2); Q[1] += m[5] + Mc * (3 * dy * dy - d2); Q[2] += m[6] + Mc * (3 * dz * dz - d2);
                Q[3] += m[7] + Mc * 3 * dx * dy; Q[4] += m[8] + Mc * 3 * dx * dz; Q[5] += m[9] + Mc * 3 * dy * dz;
            }
            store_node(A, k, lev, A.nbegin[k], A.nend[k], fc, nc, M, s, Q, clo, chi);
        }
        grid.sync();
    }

    // ---------------- a6 groups (R-S5 sibling runs): flag every group start ----------------
    if (bid == 0 && tid == 0 && A.n <= A.ncrit) A.gflag[0] = 1;
    for (int k = bid * TREE_THREADS + tid; k < nn; k += nb * TREE_THREADS) {
        const int b = A.nbegin[k], e = A.nend[k];
        if (e - b <= A.ncrit) continue;
        const int nc = A.nnchild[k];
        if (nc == 0) {                                 // over-full leaf at the deepest level
            for (int s = b; s < e; s += A.ncrit) A.gflag[s] = 1;
            continue;
        }
        const int fc = A.nfirst[k];
        int run = -1;                                  // size of the open run, -1 = none
        for (int c = fc; c < fc + nc; ++c) {
            const int cb2 = A.nbegin[c], cnt = A.nend[c] - cb2;
            if (cnt > A.ncrit) run = -1;               // that child makes its own groups
            else if (run >= 0 && run + cnt <= A.ncrit) run += cnt;
            else { A.gflag[cb2] = 1; run = cnt; }
        }
    }
    grid.sync();
    // compaction of the flags into ascending group starts
    {
        const int n16 = (A.n + 15) / 16;               // 16 flags per thread step
        const int per = (n16 + nb - 1) / nb;
        const int cb = min(n16, bid * per), ce = min(n16, cb + per);
        const uint4* f4 = (const uint4*)A.gflag;
        int bsum = 0;
        for (int q = cb + tid; q < ce; q += TREE_THREADS) {
            uint4 v = f4[q];
            bsum += __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w);
        }
        int tot; (void)block_exscan(bsum, &tot, s_warp);
        if (tid == 0) A.scan_tmp[bid] = tot;
        grid.sync();
        int before = 0, total = 0;
        for (int k = tid; k < nb; k += TREE_THREADS) { int t = A.scan_tmp[k]; total += t; if (k < bid) before += t; }
        { int t2; (void)block_exscan(before, &t2, s_warp); before = t2; }
        { int t2; (void)block_exscan(total, &t2, s_warp); total = t2; }
        if (tid == 0) s_run = before;
        __syncthreads();
        for (int q0 = cb; q0 < ce; q0 += TREE_THREADS) {
            int q = q0 + tid, c = 0;
            uint4 v = make_uint4(0, 0, 0, 0);
            if (q < ce) { v = f4[q]; c = __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w); }
            int t3, ex = block_exscan(c, &t3, s_warp);
            int w = s_run + ex;
            if (c) {
                const uint32_t words[4] = { v.x, v.y, v.z, v.w };
#pragma unroll
                for (int j = 0; j < 16; ++j)
                    if ((words[j >> 2] >> (8 * (j & 3))) & 0xffu) A.gbegin[w++] = q * 16 + j;
            }
            __syncthreads();
            if (tid == 0) s_run += t3;
            __syncthreads();
        }
        if (bid == 0 && tid == 0) { A.gbegin[total] = A.n; A.info->n_groups = total; }
    }
}

// ---------------------------------------------------------------------------------------------
int p3t_tree_init(p3t_ctx* ctx)
{
    int per_sm = 0;
    P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_tree, TREE_THREADS, 0));
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 4) per_sm = 4;
    ctx->coop_blocks_tree = per_sm * ctx->num_sms;
    return P3T_OK;
}

int p3t_launch_tree(p3t_ctx* ctx)
{
    tree_args A;
    A.keys = P<uint64_t>(ctx->keys[0]); A.spm = P<float4>(ctx->spm);
    A.n = (int)ctx->n; A.B = ctx->bits; A.nleaf = ctx->nleaf; A.ncrit = ctx->ncrit; A.node_cap = (int)ctx->node_cap;
    A.nlevel = P<int32_t>(ctx->nlevel); A.nbegin = P<int32_t>(ctx->nbegin); A.nend = P<int32_t>(ctx->nend);
    A.nfirst = P<int32_t>(ctx->nfirst); A.nnchild = P<int32_t>(ctx->nnchild);
    A.m64 = P<double>(ctx->m64);
    A.ncom = P<float4>(ctx->ncom); A.nlo = P<float4>(ctx->nlo); A.nhi = P<float4>(ctx->nhi);
    A.nq0 = P<float4>(ctx->nq0); A.nq1 = P<float2>(ctx->nq1); A.nlink = P<int2>(ctx->nlink);
    A.scan_tmp = P<int32_t>(ctx->scan_tmp);
    A.gflag = P<uint8_t>(ctx->gflag); A.gbegin = P<int32_t>(ctx->gbegin);
    A.info = INFO(ctx);
    P3T_CUDA(ctx, cudaMemsetAsync(ctx->gflag.p, 0, (size_t)ctx->n + 32, ctx->stream));
    void* args[] = { &A };
    P3T_CUDA(ctx, cudaLaunchCooperativeKernel((void*)k_tree, dim3(ctx->coop_blocks_tree), dim3(TREE_THREADS), args, 0, ctx->stream));
    ctx->launches += 1;
    return P3T_OK;
}
