// p3t_internal.cuh -- context record and launcher prototypes shared by the .cu files of libp3t.so.
// Nothing here is shared with oracle/ (the CPU checker); the two only agree on RULES.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "p3t.h"

// -DP3T_CHECKS (python -m paper_2110_11658_b200.build --checks): index assertions inside the kernels; a failed check
// prints the condition and traps (the call then returns P3T_ECUDA).  Stands in for compute-sanitizer's memcheck on
// boxes where that tool is not available (profiles/r02_sanitizer.md).  Compiled out of the product build.
#ifdef P3T_CHECKS
#include <stdio.h>
#define P3T_CHECK(c) do { if (!(c)) { printf("P3T_CHECK failed: %s (%s:%d)\n", #c, __FILE__, __LINE__); __trap(); } } while (0)
#else
#define P3T_CHECK(c) ((void)0)
#endif

#define M64_STRIDE 14                                         // doubles per cell in m64: M, sum m x (3), Q (6), COM (3), first key (bits)
#define P3T_RADIX_BITS 8
#define P3T_RADIX      256
#define P3T_SORT_THREADS 256
#define P3T_SORT_ITEMS_MIN 4                                 // keys per thread in one sort tile: 4 (n <= 2^18) or P3T_SORT_ITEMS_BIG
#define P3T_SORT_ITEMS_BIG 16
#define P3T_SORT_TILE_MIN  (P3T_SORT_THREADS * P3T_SORT_ITEMS_MIN) // the smallest tile sizes the histogram buffer

// device-side counters written by the build and force kernels (one small record)
struct p3t_devinfo {
    float    lo[3];          // bounding cube, R-S1
    float    side;
    float    scale;          // 2^B / side
    int32_t  bad_input;      // NaN/Inf seen
    int32_t  n_nodes;
    int32_t  n_leaves;
    int32_t  max_level;
    int32_t  n_groups;
    int32_t  node_overflow;
    int32_t  level_begin[24]; // first node of each level; level_begin[max_level+1] = n_nodes
    uint32_t group_cursor;   // dynamic group scheduler of the walk kernels
    uint32_t group_cursor2;
    uint32_t group_cursor3;
    unsigned long long n_pp, n_pc, n_pp_list, n_pc_list;
    unsigned long long nb_total;
    int32_t  nb_max;
    int32_t  stack_overflow;
    int32_t  pool_overflow;  // a walker warp ran out of list space (the call is repeated with larger pools)
    uint32_t need_pc, need_pp; // largest per-warp list space used, in entries
    uint32_t minmax[6];      // order-preserving uint encodings of min xyz / max xyz
    int32_t  shard_g0, shard_g1; // target groups of this context's shard (all groups unless p3t_set_shard)
    int32_t  nb_overflow;    // the neighbour total exceeds the capacity of the index buffers: nothing was emitted (repaired by the host)
    int32_t  spin_abort;     // a force warp waited too long for a group's lists (no co-resident walker): those groups are repaired
    int32_t  topo_done;      // k_topo_scan: blocks (levels) that have finished their row
    int32_t  level_tot[24];  // k_topo_scan: cells per level
    uint32_t grid_bar;       // k_moments: arrivals at its grid barrier (monotone; the record is cleared per build)
};

// State of a target group's interaction lists in p3t_ctx::gready, relative to the call's epoch `base` (values of older
// calls are smaller, so the array is never cleared): base + 1 = lists published by a walker warp, base + 2 = no lists
// (pool or stack overflow, or a force warp gave up waiting), base + 3 = lists rebuilt by the host's repair pass.
#define G_READY  1
#define G_FAILED 2
#define G_REDONE 3

// arguments of the force call in flight (p3t_force_begin .. p3t_force_finish)
struct p3t_pending {
    float r_out, r_in, theta, r_list, half_dt;
    int pot_mode, active, overlapped, repaired;
    int flags;                       // P3T_FF_* of the call (p3t_stats::force_flags)
    float4 *acc_pot, *vel;
};

struct p3t_buf { void* p; size_t bytes; };

struct p3t_ctx {
    int device;
    cudaStream_t stream;
    cudaStream_t copy_stream;        // p3t_step_host: device-to-host copies that overlap the force kernel (created on first use)
    int num_sms;
    int occ_moments;                 // resident CTAs per SM of k_moments (cooperative launch)
    int occ_walk[2], occ_force;      // resident CTAs per SM of k_walk<COUNT / LISTS> and k_force on this device (0 = not asked yet)
    int nleaf, ncrit;
    int order;               // multipole order of the p-c terms: 2 (default) or 1
    int state;               // 0 = created, 1 = built, 2 = force done
    int64_t n;
    int key_bits, bits;      // bits per axis
    int64_t node_cap;
    char err[256];
    int sticky;
    // device buffers (grow-only)
    p3t_buf keys[2], idx[2];         // uint64 / uint32 ping-pong; after the sort [0] holds the result
    p3t_buf spm;                     // float4 sorted bodies
    p3t_buf rank;                    // int32: original id -> sorted position
    p3t_buf hist;                    // sort: per-block digit counts
    p3t_buf nlevel, nbegin, nend, nfirst, nnchild;        // int32 per node
    p3t_buf m64;                     // double[M64_STRIDE] per node: M, sum m x [3], Q[6], COM[3], first key
    p3t_buf ncom, nlo, nhi, nq0, nq1, nlink;              // walk SoA (see p3t_tree.cu)
    p3t_buf scan_tmp;                // tree build: starters per level and block [22][blocks]
    p3t_buf pcl, plam;               // int8 per particle: cl(i), lam(i) (p3t_tree.cu)
    p3t_buf nparent, nfc, ncount;    // int32 per node: parent, first-child rank, arrival counter
    p3t_buf gsum;                    // block sums of the group compaction
    p3t_buf gflag, gbegin;           // group start flags [n+1] / compacted starts [n_groups+1]
    p3t_buf gnpp, gnpc;              // per-group list lengths
    p3t_buf nbcount, nboff, nbidx;   // neighbour CSR: counts (sorted order) -> offsets (original order), indices
    p3t_buf nbcur;                   // int64 per sorted particle: write cursor base
    p3t_buf nbcnt, part;             // k_force<SPLIT>: row cursors (int32 per particle), partial sums [nseg][n][4] fp64
    p3t_buf spill;                   // walk stack spill
    p3t_buf pcpool, pppool;          // interaction lists: node ids / sorted particle positions, per-warp regions
    p3t_buf glist;                   // uint4 per group: pc offset/32, n_pc, pp offset/32, n_pp
    int64_t pool_cap_pc, pool_cap_pp;// entries per walker warp (multiples of 32)
    int64_t walk_warps_max, walk_list_warps;
    p3t_buf info;                    // p3t_devinfo
    p3t_buf stage_in, stage_out;     // p3t_step_host staging
    int64_t nb_total_host;           // valid after p3t_neighbours
    int nb_valid;
    cudaEvent_t ev[6];               // build begin/end, sort begin/end ... force begin/end, walk begin/end
    cudaEvent_t evw[4];
    cudaEvent_t evi[2];              // irregular-force kernel begin/end
    cudaEvent_t evc[2];              // core-quantity kernels begin/end
    p3t_buf core;                    // double[6]: result of k_core_reduce
    p3t_buf irrpv;                   // k_irregular<PV>: float4[n][2] position + velocity records, original order
    p3t_buf psitab;                  // k_irregular: Hermite table of the pair-potential integral (p3t_irregular.cu)
    float psitab_host[256 * 8]; float psitab_rout, psitab_rin;
    p3t_buf o64, noct, octcnt;       // octupole variant (p3t_octupole.cu): fp64 third moments [node][11], fp32 [node][3] float4, arrival counters
    int oct_built;                   // the third moments belong to the current tree
    cudaEvent_t evo[2];              // octupole add kernel begin/end
    int core_done;
    int irr_done;
    p3t_stats last;
    float r_out, r_in, theta, r_list;
    int shard_rank, shard_nranks;    // p3t_set_shard: this context walks the groups of one Morton range
    p3t_buf shard_nominal;           // int64[nranks+1]: caller's cuts in sorted positions (unused when shard_has_nominal = 0)
    p3t_buf shard_cuts;              // int32[2][nranks+1]: group-aligned cuts as group index / sorted position
    int shard_has_nominal;
    int64_t launches;                // kernels launched so far
    // walk / force overlap (p3t_force.cu): per-group list state, the epoch of the current call, the walker stream
    p3t_buf gready;                  // int32 per group (see G_READY)
    int32_t epoch;
    cudaStream_t walk_stream;        // created on first use (non-blocking)
    cudaEvent_t ev_tree, ev_scan, ev_wdone;
    int overlap;                     // 1 (default): walkers and force kernel run concurrently; 0: one after the other (p3t_diag_set_overlap)
    int walk_ctas_per_sm;            // CTAs per SM given to the list walk while the force kernel runs (p3t_diag_set_overlap, default 2: measured 9.03 vs 9.06 ms at config 3)
    int64_t nb_cap;                  // capacity of nbidx / the raw row buffer in entries (grow-only, from the previous call's total)
    int nb_max_hint;                 // longest row of the previous call (chooses the row-sort variant; any value is correct)
    p3t_pending pend;
    int test_fault;                  // p3t_diag_set_fault (tests only), bits: 1 = the force kernel gives up waiting at once, 2 = no walk-stack spill,
                                     // 4 = p3t_step_host meets a CUDA failure while its force call is in flight
};

#define P3T_CUDA(ctx, call)                                                              \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) return p3t_fail_cuda((ctx), e_, #call, __LINE__);         \
    } while (0)

int  p3t_fail_cuda(p3t_ctx* ctx, cudaError_t e, const char* what, int line);
int  p3t_reserve(p3t_ctx* ctx, p3t_buf* b, size_t bytes);

template <typename T> static inline T* P(p3t_buf& b) { return (T*)b.p; }
static inline p3t_devinfo* INFO(p3t_ctx* c) { return (p3t_devinfo*)c->info.p; }

// p3t_sort.cu : a1-a3
size_t p3t_sort_scratch_bytes(int64_t n);                            // ctx->hist: digit totals, tickets, look-back words
int p3t_launch_cube_keys(p3t_ctx* ctx, const float4* pos_mass);
int p3t_launch_sort(p3t_ctx* ctx);
int p3t_launch_permute(p3t_ctx* ctx, const float4* pos_mass);
// p3t_tree.cu : a4-a6
int p3t_launch_tree(p3t_ctx* ctx);
// p3t_octupole.cu : SURVEY 8f NEXT-4, octupole variant
int p3t_launch_octupoles(p3t_ctx* ctx);
int p3t_launch_octupole_add(p3t_ctx* ctx, float4* acc_pot, float half_dt, float4* vel, int base, int mode, int evalall);
// p3t_shard.cu : SURVEY 8e, target groups split among the ranks of a node
int p3t_launch_shard_range(p3t_ctx* ctx);
// p3t_walk.cu : a7 (interaction lists), a10 (neighbour counts)
int p3t_walk_init(p3t_ctx* ctx);
int p3t_launch_walk_reset(p3t_ctx* ctx, cudaStream_t st);
int p3t_walk_reserve(p3t_ctx* ctx, int ctas_per_sm);                 // spill + list pools for a walk with this share of the device
int p3t_launch_walk_count(p3t_ctx* ctx, float r_list, float theta, cudaStream_t st);   // r_list: neighbour search radius (>= r_out)
// base: epoch of the call (gready); repair: host repair pass (every group again, failed ones become G_REDONE);
// ctas_per_sm: 0 = the whole device, else the share left to the walk while the force kernel runs
int p3t_launch_walk_lists(p3t_ctx* ctx, float r_list, float theta, cudaStream_t st, int base, int repair, int ctas_per_sm);
// p3t_core.cu : SURVEY 8f NEXT-3
int p3t_launch_core(p3t_ctx* ctx, int64_t ns, const int32_t* sample, int K, int32_t* nbr, float* d2k, double* rho, double* core_dev);
// p3t_irregular.cu : SURVEY 8f NEXT-1
int p3t_launch_irregular(p3t_ctx* ctx, const float4* vel, float4* acc, float4* jerk);
// p3t_force.cu : a8-a11
// p3t_force_begin enqueues the whole call (count walk, offsets, list walk and force kernel, row sort) without a host
// synchronisation; p3t_force_finish synchronises once, reports errors and repairs what an undersized buffer left out.
int p3t_force_begin(p3t_ctx* ctx, float r_out, float r_in, float theta, int pot_mode, float4* acc_pot,
                    float r_list, float half_dt, float4* vel);
int p3t_force_finish(p3t_ctx* ctx);
void p3t_force_abandon(p3t_ctx* ctx);        // p3t_destroy with a call in flight: the stream is drained, the device's overlap slot released

// group-state helpers shared by the walk, force and octupole kernels
__device__ __forceinline__ int ld_acquire_gpu(const int32_t* p)
{
    int v; asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ int cas_release_gpu(int32_t* p, int cmp, int val)
{
    int old; asm volatile("atom.release.gpu.global.cas.b32 %0, [%1], %2, %3;" : "=r"(old) : "l"(p), "r"(cmp), "r"(val) : "memory"); return old;
}
__device__ __forceinline__ bool g_decided(int v, int base) { return v >= base + G_READY && v <= base + G_REDONE; }
