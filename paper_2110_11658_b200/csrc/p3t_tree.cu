// p3t_tree.cu -- steps a4-a6: canonical octree topology, bottom-up monopole +
// traceless quadrupole moments, target groups.
// Rules: DESIGN.md R-S4 (topology), R-S5 (sibling-run groups), R-S6 (moments).
// The paper gives no detail of this stage ("the BONSAI library").
//
// Topology without a level loop.  The canonical rule "a cell with more than NLEAF particles (and
// level < B) is split" makes the existence of a cell a LOCAL property of the sorted key array:
//   cl(i)  = number of leading octant digits that key[i-1] and key[i] share (cl(0) = -1):
//            particle i begins a new cell at every level l > cl(i);
//   a(i)   = number of leading digits that key[i] and key[i+NLEAF] share: the NLEAF+1 particles
//            i .. i+NLEAF lie in one cell down to level a(i);
//   P(i)   = max a(j), j in [i-NLEAF, i]  = the deepest level at which the cell of particle i
//            holds more than NLEAF particles (-1: not even the root);
//   lam(i) = min(P(i) + 1, B)             = the level of the leaf that holds particle i.
// The cell (l, i) -- level l, first particle i -- exists iff cl(i) < l <= lam(i) (and (0, 0), the
// root).  Numbering the cells by level, then by first particle, needs one multi-level prefix sum
// over the particles: three streaming kernels instead of two grid-wide barriers per level.
// Moments then climb the tree with one arrival counter per cell (the last child to arrive
// computes its parent, combining the children in their fixed order), again without barriers.
#include "p3t_internal.cuh"
#include <cooperative_groups.h>

#define TOPO_THREADS 256
#define TOPO_WARPS   (TOPO_THREADS / 32)
#define MAXLEV       22                  // levels 0 .. 21
#define NODE_THREADS 128

struct tree_args {
    const uint64_t* keys;      // sorted
    const float4* spm;         // sorted bodies
    int n, B, nleaf, ncrit, node_cap, nblk;
    int8_t *pcl, *plam;        // per particle: cl(i), lam(i)
    int32_t* blksum;           // [MAXLEV][nblk] starters per level and block -> exclusive prefix
    int32_t *nlevel, *nbegin, *nend, *nfirst, *nnchild, *nparent, *nfc, *ncount;
    double* m64;               // [node][13] = M, sum m x (3), Q about COM (6: xx yy zz xy xz yz), COM (3)
    float4 *ncom, *nlo, *nhi, *nq0;
    float2* nq1;
    int2* nlink;
    uint8_t* gflag;            // [n + 16] zeroed by the host side
    int32_t* gbegin;           // [n + 1]
    int32_t* gsum;             // block sums of the group-flag compaction
    p3t_devinfo* info;
};

// number of leading octant digits two keys of 3B bits share
__device__ __forceinline__ int common_digits(uint64_t a, uint64_t b, int B)
{
    const uint64_t x = a ^ b;
    if (x == 0) return B;
    return (__clzll((long long)x) - (64 - 3 * B)) / 3;
}

// ---------------- a4, pass 1: cl, lam, starters per level and block ----------------
__global__ void __launch_bounds__(TOPO_THREADS) k_topo_count(tree_args A)
{
    __shared__ uint64_t s_key[TOPO_THREADS + 2 * P3T_MAX_NCRIT + 1];
    __shared__ int8_t   s_a[TOPO_THREADS + P3T_MAX_NCRIT];
    __shared__ int      s_cnt[TOPO_WARPS][MAXLEV];
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int t0 = blockIdx.x * TOPO_THREADS, L = A.nleaf;
    // keys t0 - L - 1 .. t0 + 255 + L
    for (int q = tid; q < TOPO_THREADS + 2 * L + 1; q += TOPO_THREADS) {
        const int j = t0 - L - 1 + q;
        s_key[q] = (j >= 0 && j < A.n) ? A.keys[j] : 0ull;
    }
    __syncthreads();
    // a(j) for j = t0 - L .. t0 + 255
    for (int q = tid; q < TOPO_THREADS + L; q += TOPO_THREADS) {
        const int j = t0 - L + q;
        int a = -1;
        if (j >= 0 && j + L < A.n) a = common_digits(s_key[q + 1], s_key[q + 1 + L], A.B);
        s_a[q] = (int8_t)a;
    }
    __syncthreads();
    const int i = t0 + tid;
    int cl = MAXLEV, lam = -1;                  // idle threads start nothing
    if (i < A.n) {
        cl = i == 0 ? -1 : common_digits(s_key[tid + L], s_key[tid + L + 1], A.B);
        int P = -1;
        for (int q = tid; q <= tid + L; ++q) P = max(P, (int)s_a[q]);
        lam = min(P + 1, A.B);
        A.pcl[i] = (int8_t)cl; A.plam[i] = (int8_t)lam;
    }
    // only the levels at which some particle of the warp starts a cell (a handful around the leaf level of the
    // neighbourhood, not all 21): the others keep their zero
    if (lane < MAXLEV) s_cnt[w][lane] = 0;
    const int l_lo = max(1, __reduce_min_sync(0xffffffffu, cl + 1)), l_hi = min(A.B, __reduce_max_sync(0xffffffffu, lam));
    __syncwarp();
    for (int l = l_lo; l <= l_hi; ++l) {
        const uint32_t m = __ballot_sync(0xffffffffu, cl < l && l <= lam);
        if (lane == 0) s_cnt[w][l] = __popc(m);
    }
    __syncthreads();
    if (tid >= 1 && tid <= A.B) {
        int t = 0;
#pragma unroll
        for (int k = 0; k < TOPO_WARPS; ++k) t += s_cnt[k][tid];
        A.blksum[(size_t)tid * A.nblk + blockIdx.x] = t;
    }
}

// ---------------- a4, pass 2: exclusive prefix over the blocks, one block per level ----------------
#define TSCAN_THREADS 1024
__global__ void __launch_bounds__(TSCAN_THREADS) k_topo_scan(tree_args A)
{
    __shared__ int s_w[TSCAN_THREADS / 32];
    __shared__ int s_run;
    __shared__ int s_last;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, l = blockIdx.x + 1;       // levels 1 .. B
    int32_t* row = A.blksum + (size_t)l * A.nblk;
    if (threadIdx.x == 0) s_run = 0;
    __syncthreads();
    for (int b0 = 0; b0 < A.nblk; b0 += TSCAN_THREADS) {
        const int b = b0 + threadIdx.x;
        const int v = b < A.nblk ? row[b] : 0;
        int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) s_w[w] = x;
        __syncthreads();
        int add = s_run, tot = 0;
#pragma unroll
        for (int k = 0; k < TSCAN_THREADS / 32; ++k) { const int t = s_w[k]; if (k < w) add += t; tot += t; }
        if (b < A.nblk) row[b] = add + x - v;
        __syncthreads();
        if (threadIdx.x == 0) s_run += tot;
        __syncthreads();
    }
    // the last level to finish turns the totals into the level offsets
    if (threadIdx.x == 0) {
        A.info->level_tot[l] = s_run;
        __threadfence();
        s_last = atomicAdd(&A.info->topo_done, 1) == (int)gridDim.x - 1;
    }
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        __threadfence();
        int off = 1, maxl = 0;                    // the root is cell 0
        A.info->level_begin[0] = 0; A.info->level_begin[1] = 1;
        for (int k = 1; k <= A.B; ++k) {
            const int t = *(volatile int32_t*)&A.info->level_tot[k];
            if (t > 0) maxl = k;
            off += t;
            A.info->level_begin[k + 1 < 24 ? k + 1 : 23] = off;
        }
        for (int k = A.B + 2; k < 24; ++k) A.info->level_begin[k] = off;
        A.info->n_nodes = off; A.info->max_level = maxl;
        A.info->node_overflow = off > A.node_cap ? 1 : 0;
    }
}

// ---------------- a4, pass 3: the cells ----------------
__global__ void __launch_bounds__(TOPO_THREADS) k_topo_nodes(tree_args A)
{
    __shared__ int s_cnt[TOPO_WARPS][MAXLEV + 1];   // starters per warp and level, then exclusive over the warps
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int i = blockIdx.x * TOPO_THREADS + tid;
    int cl = MAXLEV, lam = -1;
    if (i < A.n) { cl = A.pcl[i]; lam = A.plam[i]; }
    const int* __restrict__ lb = A.info->level_begin;
    if (A.info->node_overflow) return;
    if (lane <= MAXLEV) s_cnt[w][lane] = 0;
    const int l_lo = max(1, __reduce_min_sync(0xffffffffu, cl + 1)), l_hi = min(A.B, __reduce_max_sync(0xffffffffu, lam));
    __syncwarp();
    for (int l = l_lo; l <= l_hi; ++l) {                 // the levels at which the warp starts cells (see k_topo_count)
        const uint32_t m = __ballot_sync(0xffffffffu, cl < l && l <= lam);
        if (lane == 0) s_cnt[w][l] = __popc(m);
    }
    __syncthreads();
    if (tid <= A.B) {
        int run = tid == 0 ? 0 : A.blksum[(size_t)tid * A.nblk + blockIdx.x];
#pragma unroll
        for (int k = 0; k < TOPO_WARPS; ++k) { const int t = s_cnt[k][tid]; s_cnt[k][tid] = run; run += t; }
    }
    __syncthreads();
    // rank of particle i among the starters of level l = s_cnt[w][l] + popc(ballot_l & lanes below);
    // level 0 has the single starter (0, 0)
    if (i == 0) {                                // the root
        A.nlevel[0] = 0; A.nbegin[0] = 0; A.nparent[0] = -1;
        A.nfc[0] = 1;                            // rank 0 among the level-1 starters
    }
    uint32_t m_prev = 0, m_cur = __ballot_sync(0xffffffffu, cl < l_lo && l_lo <= lam);
    // starters of level l_lo - 1 before i: none of them is in this warp (level 0: the root, before everybody but i = 0)
    int r_prev = l_lo == 1 ? (i > 0 ? 1 : 0) : s_cnt[w][l_lo - 1];
    for (int l = l_lo; l <= l_hi; ++l) {
        const uint32_t m_next = l < A.B ? __ballot_sync(0xffffffffu, cl < l + 1 && l + 1 <= lam) : 0u;
        const int r_cur = s_cnt[w][l] + __popc(m_cur & lt_mask);
        if (cl < l && l <= lam) {
            const int id = lb[l] + r_cur;
            const int r_next = l < A.B ? s_cnt[w][l + 1] + __popc(m_next & lt_mask) : 0;
            A.nlevel[id] = l; A.nbegin[id] = i;
            A.nfc[id] = lb[l + 1 < 24 ? l + 1 : 23] + r_next;
            A.nparent[id] = lb[l - 1] + r_prev - (cl < l - 1 ? 0 : 1);
        }
        r_prev = r_cur; m_prev = m_cur; m_cur = m_next;
    }
    (void)m_prev;
}

// ---------------- a4, pass 4: ranges and child links ----------------
// Children tile their parent: the range of a cell ends where its next sibling begins, and the last
// child ends where its parent ends (climb until a cell has a next sibling).  The children of a cell
// are numbered consecutively; their number is the distance to the first child of the next cell of
// the same level.
__global__ void __launch_bounds__(NODE_THREADS) k_topo_link(tree_args A)
{
    const int nn = A.info->n_nodes;
    const int* __restrict__ lb = A.info->level_begin;
    if (A.info->node_overflow) return;
    int leaves = 0;
    // the cell count is only known on the device: a fixed grid strides over the cells (a grid sized by the host's bound
    // on the count would be ten times too large, and empty blocks are not free)
    for (int k = blockIdx.x * NODE_THREADS + threadIdx.x; k < nn; k += gridDim.x * NODE_THREADS) {
        const int lev = A.nlevel[k];
        int end = A.n;
        for (int w = k, l = lev; l > 0; --l) {
            const int v = w + 1;
            const int p = A.nparent[w];
            if (v < lb[l + 1] && A.nparent[v] == p) { end = A.nbegin[v]; break; }
            w = p;
        }
        A.nend[k] = end;
        const int fc = A.nfc[k];
        const int fc_next = k + 1 < lb[lev + 1] ? A.nfc[k + 1] : lb[lev + 2 < 24 ? lev + 2 : 23];
        const int nc = lev < A.B ? fc_next - fc : 0;
        A.nnchild[k] = nc; A.nfirst[k] = nc > 0 ? fc : -1;
        A.ncount[k] = 0;
        leaves += nc == 0;
    }
    // block sum of the leaf counts
    const int tot = leaves;
    __shared__ int s_leaf[NODE_THREADS / 32];
    int x = tot;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if ((threadIdx.x & 31) == 0) s_leaf[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int k = 0; k < NODE_THREADS / 32; ++k) t += s_leaf[k];
        if (t) atomicAdd(&A.info->n_leaves, t);
    }
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
// key0 = Morton key of the cell's first particle (a leaf reads it, a parent takes its first child's: no dependent load)
__device__ void store_node(const tree_args& A, int k, int level, int b, int e, int first, int nchild, uint64_t key0,
                           double M, const double s[3], const double c[3], const double Q[6], const float clo[3], const float chi[3])
{
    P3T_CHECK(k >= 0 && k < A.node_cap && b >= 0 && e <= A.n && b < e);
    double* m = A.m64 + (size_t)k * M64_STRIDE;
    m[0] = M; m[1] = s[0]; m[2] = s[1]; m[3] = s[2];
#pragma unroll
    for (int q = 0; q < 6; ++q) m[4 + q] = Q[q];
    m[10] = c[0]; m[11] = c[1]; m[12] = c[2];       // the parent reads the quotient instead of dividing again (same bits)
    m[13] = __longlong_as_double((long long)key0);
    // geometric centre from the integer cell coordinates (prefix of the first key)
    const uint64_t prefix = level == 0 ? 0ull : (key0 >> (3 * (A.B - level)));
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

// ---------------- a5 moments (R-S6), fp64 ----------------
// One cooperative launch.  Phase 0: every leaf from its particles (one thread per leaf).  Then the internal cells level
// by level from the deepest up (cells are numbered breadth-first, so a level is a contiguous range), a grid barrier
// between two levels.  An internal cell is combined by eight lanes, one per child: each lane loads its child's fp64
// record (one round trip for the whole cell), the sums go through a fixed xor tree over the eight lanes (idle lanes add
// exact zeros), so the result does not depend on timing: bit-reproducible, and no atomics or fences are needed.
// (Rounds 1's version climbed from the leaves with one arrival counter per cell: a chain of L2 round trips per level
// in ever fewer, diverged threads -- 0.12 ms at N = 2^20.)
__device__ __forceinline__ double shfl_xor_f64(double v, int o)
{
    int lo = __double2loint(v), hi = __double2hiint(v);
    lo = __shfl_xor_sync(0xffffffffu, lo, o); hi = __shfl_xor_sync(0xffffffffu, hi, o);
    return __hiloint2double(hi, lo);
}
__device__ __forceinline__ double shfl_up_f64(double v, int o)
{
    int lo = __double2loint(v), hi = __double2hiint(v);
    lo = __shfl_up_sync(0xffffffffu, lo, o); hi = __shfl_up_sync(0xffffffffu, hi, o);
    return __hiloint2double(hi, lo);
}
__device__ __forceinline__ double shfl_idx_f64(double v, int src)
{
    int lo = __double2loint(v), hi = __double2hiint(v);
    lo = __shfl_sync(0xffffffffu, lo, src); hi = __shfl_sync(0xffffffffu, hi, src);
    return __hiloint2double(hi, lo);
}
__device__ __forceinline__ double seg8_sum(double v)
{
    v += shfl_xor_f64(v, 1); v += shfl_xor_f64(v, 2); v += shfl_xor_f64(v, 4);
    return v;
}
__device__ __forceinline__ float seg8_min(float v)
{
    v = fminf(v, __shfl_xor_sync(0xffffffffu, v, 1)); v = fminf(v, __shfl_xor_sync(0xffffffffu, v, 2)); v = fminf(v, __shfl_xor_sync(0xffffffffu, v, 4));
    return v;
}
__device__ __forceinline__ float seg8_max(float v)
{
    v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1)); v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2)); v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 4));
    return v;
}

__device__ void leaf_moments(const tree_args& A, int k)
{
    const int b = A.nbegin[k], e = A.nend[k];
    double M = 0.0, s[3] = { 0.0, 0.0, 0.0 };
    const uint64_t key0 = A.keys[b];
    const float4 p0 = A.spm[b];
    float clo[3] = { p0.x, p0.y, p0.z }, chi[3] = { p0.x, p0.y, p0.z };
    for (int i0 = b; i0 < e; i0 += 4) {                     // four loads in flight; summed in particle order
        float4 q[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) q[j] = A.spm[min(i0 + j, e - 1)];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (i0 + j >= e) break;
            const float4 p = q[j];
            const double m = p.w;
            M += m; s[0] += m * (double)p.x; s[1] += m * (double)p.y; s[2] += m * (double)p.z;
            clo[0] = fminf(clo[0], p.x); clo[1] = fminf(clo[1], p.y); clo[2] = fminf(clo[2], p.z);
            chi[0] = fmaxf(chi[0], p.x); chi[1] = fmaxf(chi[1], p.y); chi[2] = fmaxf(chi[2], p.z);
        }
    }
    // R-S6a: a cell of massless particles takes the position of its first particle (sorted order) as its centre
    const bool massless = M == 0.0;
    const double c[3] = { massless ? (double)p0.x : s[0] / M, massless ? (double)p0.y : s[1] / M, massless ? (double)p0.z : s[2] / M };
    double Q[6] = { 0, 0, 0, 0, 0, 0 };
    for (int i0 = b; i0 < e; i0 += 4) {
        float4 q[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) q[j] = A.spm[min(i0 + j, e - 1)];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (i0 + j >= e) break;
            const float4 p = q[j];
            const double m = p.w, dx = p.x - c[0], dy = p.y - c[1], dz = p.z - c[2];
            const double d2 = dx * dx + dy * dy + dz * dz;
            Q[0] += m * (3 * dx * dx - d2); Q[1] += m * (3 * dy * dy - d2); Q[2] += m * (3 * dz * dz - d2);
            Q[3] += m * 3 * dx * dy; Q[4] += m * 3 * dx * dz; Q[5] += m * 3 * dy * dz;
        }
    }
    store_node(A, k, A.nlevel[k], b, e, -1, 0, key0, M, s, c, Q, clo, chi);
}

// Grid barrier of k_moments (the launch is cooperative, so every block is resident): one monotone arrival counter;
// cooperative_groups' grid.sync() measured 8.8 us per barrier here (444 blocks), 75 % of the kernel.  Writes of the level
// below are fenced before the arrival and read past L1 (__ldcg) after it.
__device__ __forceinline__ void grid_barrier(uint32_t* bar, uint32_t nblocks)
{
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const uint32_t arrived = atomicAdd(bar, 1u) + 1u;
        const uint32_t target = (arrived + nblocks - 1u) / nblocks * nblocks;      // end of this round
        while (*(volatile uint32_t*)bar < target) { }
        __threadfence();
    }
    __syncthreads();
}

#define MOM_THREADS 256
__global__ void __launch_bounds__(MOM_THREADS) k_moments(tree_args A)
{
    const int nn = A.info->n_nodes;
    if (A.info->node_overflow) return;                       // uniform over the grid: nobody reaches a barrier
    const int gtid = blockIdx.x * MOM_THREADS + threadIdx.x, gsize = gridDim.x * MOM_THREADS;
    for (int k = gtid; k < nn; k += gsize)
        if (A.nnchild[k] == 0) leaf_moments(A, k);
    __shared__ int lb[24];                                       // level offsets: read once (a dependent load per level otherwise)
    if (threadIdx.x < 24) lb[threadIdx.x] = A.info->level_begin[threadIdx.x];
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int gwarp = gtid >> 5, nwarps = gsize >> 5;
    const int max_level = A.info->max_level;
    // Level l from level l + 1: the children of a cell are consecutive cells of the next level, so a warp takes a window
    // of 32 consecutive CHILDREN (coalesced loads of their fp64 records, no search for the internal cells among the leaves)
    // and sums every run of siblings by a segmented scan over the lanes (runs are at most 8 long: distances 1, 2, 4).
    // Windows advance by 25 = 32 - 7, so every run lies wholly inside the window in which its first child is among the
    // first 25 lanes: that window, and only that one, stores the parent.
    for (int l = max_level - 1; l >= 0; --l) {
        grid_barrier(&A.info->grid_bar, gridDim.x);
        const int c_begin = lb[l + 1], c_end = lb[l + 2 < 24 ? l + 2 : 23];
        for (int c0 = c_begin + 25 * gwarp; c0 < c_end; c0 += 25 * nwarps) {
            const int c = c0 + lane;
            const bool have = c < c_end;
            int p = -1 - lane, p_before = -1, cb = 0, ce = 0;    // inactive lanes: all different, never equal to a cell
            double cM = 0.0, cs[3] = { 0, 0, 0 }, cQ[6] = { 0, 0, 0, 0, 0, 0 }, cc[3] = { 0, 0, 0 }, ckey = 0.0;
            float lo[3] = { INFINITY, INFINITY, INFINITY }, hi[3] = { -INFINITY, -INFINITY, -INFINITY };
            if (have) {
                p = A.nparent[c];
                if (lane == 0 && c > c_begin) p_before = A.nparent[c - 1];     // does a run start at lane 0, or continue?
                cb = A.nbegin[c]; ce = A.nend[c];
                const double* m = A.m64 + (size_t)c * M64_STRIDE;  // read past L1: another SM wrote it in this launch
                ckey = __ldcg(m + 13);
                cM = __ldcg(m); cs[0] = __ldcg(m + 1); cs[1] = __ldcg(m + 2); cs[2] = __ldcg(m + 3);
#pragma unroll
                for (int q = 0; q < 6; ++q) cQ[q] = __ldcg(m + 4 + q);
                cc[0] = __ldcg(m + 10); cc[1] = __ldcg(m + 11); cc[2] = __ldcg(m + 12);
                const float4 l4 = __ldcg(&A.nlo[c]), h4 = __ldcg(&A.nhi[c]);
                lo[0] = l4.x; lo[1] = l4.y; lo[2] = l4.z; hi[0] = h4.x; hi[1] = h4.y; hi[2] = h4.z;
            }
            // run structure: same[o] = the lane o below belongs to the same parent
            bool same[3];
#pragma unroll
            for (int t = 0; t < 3; ++t) { const int q = __shfl_up_sync(0xffffffffu, p, 1 << t); same[t] = lane >= (1 << t) && q == p; }
            const bool head = !same[0];
            const int p_next = __shfl_down_sync(0xffffffffu, p, 1);             // every lane takes part (no short-circuit around it)
            const uint32_t lastmask = __ballot_sync(0xffffffffu, lane == 31 || p_next != p);
            const int run_end = lane + __ffs(lastmask >> lane) - 1;               // last lane of this lane's run
            const int run_head = 31 - __clz(__ballot_sync(0xffffffffu, head) & ((2u << lane) - 1u));
            auto seg_sum = [&](double x) {
#pragma unroll
                for (int t = 0; t < 3; ++t) { const double y = shfl_up_f64(x, 1 << t); if (same[t]) x += y; }
                return shfl_idx_f64(x, run_end);
            };
            auto seg_min = [&](float x) {
#pragma unroll
                for (int t = 0; t < 3; ++t) { const float y = __shfl_up_sync(0xffffffffu, x, 1 << t); if (same[t]) x = fminf(x, y); }
                return __shfl_sync(0xffffffffu, x, run_end);
            };
            auto seg_max = [&](float x) {
#pragma unroll
                for (int t = 0; t < 3; ++t) { const float y = __shfl_up_sync(0xffffffffu, x, 1 << t); if (same[t]) x = fmaxf(x, y); }
                return __shfl_sync(0xffffffffu, x, run_end);
            };
            const double M = seg_sum(cM);
            double s[3] = { seg_sum(cs[0]), seg_sum(cs[1]), seg_sum(cs[2]) };
            float clo[3], chi[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) { clo[a] = seg_min(lo[a]); chi[a] = seg_max(hi[a]); }
            // R-S6a: massless cell: the centre of its first child, i.e. its first particle in sorted order
            const bool massless = M == 0.0;
            double cm[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const double first = shfl_idx_f64(cc[a], run_head);
                cm[a] = massless ? first : s[a] / M;
            }
            double Q[6];
            {
                const double dx = cc[0] - cm[0], dy = cc[1] - cm[1], dz = cc[2] - cm[2];
                const double d2 = dx * dx + dy * dy + dz * dz;
                const double t[6] = { cQ[0] + cM * (3 * dx * dx - d2), cQ[1] + cM * (3 * dy * dy - d2), cQ[2] + cM * (3 * dz * dz - d2),
                                      cQ[3] + cM * 3 * dx * dy, cQ[4] + cM * 3 * dx * dz, cQ[5] + cM * 3 * dy * dz };
#pragma unroll
                for (int q = 0; q < 6; ++q) Q[q] = seg_sum(have ? t[q] : 0.0);
            }
            // the run's first lane stores the parent, if the run starts here (lane 0 may hold the tail of a run of the
            // previous window) and among the first 25 lanes
            const int e_run = __shfl_sync(0xffffffffu, ce, run_end);              // the parent's range: first child's begin .. last child's end
            if (have && head && lane < 25 && p_before != p)
                store_node(A, p, l, cb, e_run, c, run_end - lane + 1, (uint64_t)__double_as_longlong(ckey), M, s, cm, Q, clo, chi);
        }
    }
}

// ---------------- a6 groups (R-S5 sibling runs): flag every group start, then compact ----------------
__global__ void __launch_bounds__(NODE_THREADS) k_group_flags(tree_args A)
{
    const int nn = A.info->n_nodes;
    if (blockIdx.x == 0 && threadIdx.x == 0 && A.n <= A.ncrit) A.gflag[0] = 1;
    if (A.info->node_overflow) return;
    for (int k = blockIdx.x * NODE_THREADS + threadIdx.x; k < nn; k += gridDim.x * NODE_THREADS) {
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
}

#define GC_THREADS 256
__device__ __forceinline__ int flags16(const uint4 v) { return __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w); }

__global__ void __launch_bounds__(GC_THREADS) k_group_count(tree_args A)
{
    const int n16 = (A.n + 15) / 16;
    const int q = blockIdx.x * GC_THREADS + threadIdx.x;
    const int c = q < n16 ? flags16(((const uint4*)A.gflag)[q]) : 0;
    const int tot = c;
    // block sum by warp shuffles
    __shared__ int s_w[GC_THREADS / 32];
    int x = tot;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
#pragma unroll
        for (int k = 0; k < GC_THREADS / 32; ++k) t += s_w[k];
        A.gsum[blockIdx.x] = t;
    }
}

__global__ void __launch_bounds__(1024) k_group_scan(tree_args A, int nb)
{
    __shared__ int s_w[32];
    __shared__ int s_run;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_run = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nb; b0 += 1024) {
        const int b = b0 + threadIdx.x;
        const int v = b < nb ? A.gsum[b] : 0;
        int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) s_w[w] = x;
        __syncthreads();
        int add = s_run, tot = 0;
        for (int k = 0; k < 32; ++k) { const int t = s_w[k]; if (k < w) add += t; tot += t; }
        if (b < nb) A.gsum[b] = add + x - v;
        __syncthreads();
        if (threadIdx.x == 0) s_run += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) { A.gbegin[s_run] = A.n; A.info->n_groups = s_run; A.info->shard_g0 = 0; A.info->shard_g1 = s_run; }
}

__global__ void __launch_bounds__(GC_THREADS) k_group_compact(tree_args A)
{
    __shared__ int s_w[GC_THREADS / 32];
    const int n16 = (A.n + 15) / 16;
    const int q = blockIdx.x * GC_THREADS + threadIdx.x, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint4 v = make_uint4(0, 0, 0, 0);
    if (q < n16) v = ((const uint4*)A.gflag)[q];
    const int c = flags16(v);
    int x = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) s_w[w] = x;
    __syncthreads();
    int out = A.gsum[blockIdx.x] + x - c;
    for (int k = 0; k < w; ++k) out += s_w[k];
    if (c) {
        const uint32_t words[4] = { v.x, v.y, v.z, v.w };
#pragma unroll
        for (int j = 0; j < 16; ++j)
            if ((words[j >> 2] >> (8 * (j & 3))) & 0xffu) A.gbegin[out++] = q * 16 + j;
    }
}

// ---------------------------------------------------------------------------------------------

int p3t_launch_tree(p3t_ctx* ctx)
{
    tree_args A;
    const int n = (int)ctx->n;
    A.keys = P<uint64_t>(ctx->keys[0]); A.spm = P<float4>(ctx->spm);
    A.n = n; A.B = ctx->bits; A.nleaf = ctx->nleaf; A.ncrit = ctx->ncrit; A.node_cap = (int)ctx->node_cap;
    A.nblk = (n + TOPO_THREADS - 1) / TOPO_THREADS;
    A.pcl = P<int8_t>(ctx->pcl); A.plam = P<int8_t>(ctx->plam); A.blksum = P<int32_t>(ctx->scan_tmp);
    A.nlevel = P<int32_t>(ctx->nlevel); A.nbegin = P<int32_t>(ctx->nbegin); A.nend = P<int32_t>(ctx->nend);
    A.nfirst = P<int32_t>(ctx->nfirst); A.nnchild = P<int32_t>(ctx->nnchild);
    A.nparent = P<int32_t>(ctx->nparent); A.nfc = P<int32_t>(ctx->nfc); A.ncount = P<int32_t>(ctx->ncount);
    A.m64 = P<double>(ctx->m64);
    A.ncom = P<float4>(ctx->ncom); A.nlo = P<float4>(ctx->nlo); A.nhi = P<float4>(ctx->nhi);
    A.nq0 = P<float4>(ctx->nq0); A.nq1 = P<float2>(ctx->nq1); A.nlink = P<int2>(ctx->nlink);
    A.gflag = P<uint8_t>(ctx->gflag); A.gbegin = P<int32_t>(ctx->gbegin);
    A.gsum = P<int32_t>(ctx->gsum);
    A.info = INFO(ctx);
    cudaStream_t st = ctx->stream;
    P3T_CUDA(ctx, cudaMemsetAsync(ctx->gflag.p, 0, (size_t)n + 32, st));
    k_topo_count<<<A.nblk, TOPO_THREADS, 0, st>>>(A);
    k_topo_scan<<<A.B, TSCAN_THREADS, 0, st>>>(A);
    k_topo_nodes<<<A.nblk, TOPO_THREADS, 0, st>>>(A);
    // one thread per cell, striding: the cell count is only known on the device (about n / 4 for the paper's
    // workloads; the hard bound node_cap is ten times that), so the grid is sized for n / 2 cells, and for the device
    long long want = ((long long)n / 2 + NODE_THREADS - 1) / NODE_THREADS;
    const long long full = (long long)ctx->num_sms * 16;
    const int nodes_grid = (int)(want < 1 ? 1 : want < full ? want : full);
    k_topo_link<<<nodes_grid, NODE_THREADS, 0, st>>>(A);
    {   // cooperative: every block resident (grid barriers between the levels)
        if (!ctx->occ_moments) {
            P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->occ_moments, k_moments, MOM_THREADS, 0));
            if (ctx->occ_moments < 1) ctx->occ_moments = 1;
        }
        long long mb = ((long long)n / 2 + MOM_THREADS - 1) / MOM_THREADS;
        const long long mfull = (long long)ctx->occ_moments * ctx->num_sms;
        const int mom_grid = (int)(mb < 1 ? 1 : mb < mfull ? mb : mfull);
        void* args[] = { (void*)&A };
        P3T_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)k_moments, dim3(mom_grid), dim3(MOM_THREADS), args, 0, st));
    }
    k_group_flags<<<nodes_grid, NODE_THREADS, 0, st>>>(A);
    const int n16 = (n + 15) / 16, gcb = (n16 + GC_THREADS - 1) / GC_THREADS;
    k_group_count<<<gcb, GC_THREADS, 0, st>>>(A);
    k_group_scan<<<1, 1024, 0, st>>>(A, gcb);
    k_group_compact<<<gcb, GC_THREADS, 0, st>>>(A);
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 9;
    if (ctx->shard_nranks > 1) return p3t_launch_shard_range(ctx);
    return P3T_OK;
}
