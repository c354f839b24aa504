// p3t_walk.cu -- steps a7 and a10: the group tree walk.
//
// One warp walks one target group (R-S5) breadth-first: 32 cells per iteration, one per lane, the
// opening rule R-S7 evaluated in bit-specified fp32, ballot / popc compaction, a shared-memory
// stack with a global spill.  Two kernels share the traversal:
//
//   k_walk<WALK_COUNT>  walks only the cells within r_out of the group box and counts, per target,
//                       the neighbours d2 < r_out^2 (R10): the sizes of the CSR rows (a10).
//   k_walk<WALK_LISTS>  the full walk (a7).  It evaluates nothing: accepted cells (node ids) and the
//                       particles of opened leaves (sorted positions) are appended to the group's
//                       interaction lists in HBM.  The force kernel (p3t_force.cu) streams them.
//
// Why the lists go through HBM on B200: the walk is a serial, latency-bound pointer chase that
// needs few registers and many resident warps; the force evaluation is an FP32-pipe-bound stream
// that needs many registers.  Fused in one kernel (this library's first version) the two phases of
// a warp alternate and the FP32 pipe idles for 30-40 % of the time (profiles/r01b_force_walk_full_config3.md).  Writing
// 4 bytes per interaction-list entry costs 0.57 GB of HBM traffic at N = 2^20 (< 0.2 ms at the
// measured 6.5 TB/s) and lets either kernel run with its own register budget -- side by side on every SM: k_walk<WALK_LISTS>
// runs on its own stream while the force kernel evaluates the groups it has already published (p3t_force.cu).
// The paper gives no detail of this stage ("the BONSAI library").
#include "p3t_internal.cuh"
#include "p3t_f32x2.cuh"
#include <stdlib.h>

#define WALK_WARPS   8
#define WALK_THREADS (WALK_WARPS * 32)
#define STACK_CAP    384                  // per-warp node stack in shared memory; deeper entries spill
#define SPILL_CAP    8192                 // per-warp spill (global memory), entries
#define WALK_COUNT   0
#define WALK_LISTS   1

struct walk_args {
    const float4* spm; const uint32_t* order;
    const float4 *ncom, *nlo, *nhi; const int2* nlink;
    const int32_t* gbegin;
    int32_t *gnpp, *gnpc;
    int32_t* nbcount;           // WALK_COUNT out: per ORIGINAL id
    int32_t *pcpool, *pppool;   // WALK_LISTS out
    uint4* glist;               // WALK_LISTS out
    long long cap_pc, cap_pp;   // list space per warp, entries (multiples of 32)
    int32_t* spill;
    p3t_devinfo* info;
    float rout2, theta;
    int n;                      // particles (P3T_CHECKS)
    int32_t* gready;            // WALK_LISTS: per-group list state (p3t_internal.cuh: G_READY ...)
    int base, repair;           // epoch of the call; repair = host repair pass (no force kernel is waiting)
    int spill_cap;              // <= SPILL_CAP (smaller only under p3t_diag_set_fault bit 2, to exercise the overflow report)
};

struct __align__(16) warp_smem {
    int   stack[STACK_CAP];
    int   pcid[64];             // WALK_LISTS: accepted node ids waiting for a 32-wide store
    int   ppid[64];             // WALK_LISTS: sorted positions of leaf particles, likewise
};
struct __align__(16) count_smem {   // WALK_COUNT: positions of the leaf particles of one round
    float x[32], y[32], z[32];
};

__device__ __forceinline__ int stack_get(const warp_smem& S, const int32_t* spill, int i)
{
    return i < STACK_CAP ? S.stack[i] : spill[i - STACK_CAP];
}
__device__ __forceinline__ void stack_put(warp_smem& S, int32_t* spill, int i, int v)
{
    P3T_CHECK(i >= 0 && i < STACK_CAP + SPILL_CAP);
    if (i < STACK_CAP) S.stack[i] = v; else spill[i - STACK_CAP] = v;
}

// ids wait in a 64-entry staging row; once 32 are there they leave as one coalesced 128-byte store.
// ptr counts entries even when the region is full, so that the host learns the space needed.
__device__ __forceinline__ void list_flush(int* stage, int& fill, int32_t* pool, long long& ptr, long long end, int lane, int& ovf)
{
    if (fill >= 32) {
        if (ptr + 32 <= end) pool[ptr + lane] = stage[lane]; else ovf = 1;
        ptr += 32;
        const int v = stage[32 + lane];
        __syncwarp();
        stage[lane] = v;
        fill -= 32;
        __syncwarp();
    }
}

template <int MODE>
__device__ void walk_group(const walk_args& A, warp_smem& S, count_smem* C, int32_t* spill, int g, int gb, int ge,
                           const float* s_lt /* [24] fl(l/theta) per level */,
                           long long& pc_ptr, long long pc_end, long long& pp_ptr, long long pp_end)
{
    const int lane = threadIdx.x & 31;
    const uint32_t lt_mask = (1u << lane) - 1u;
    // targets: two slots per lane (P3T_MAX_NCRIT = 64); the group box is the exact fp32 min/max
    float tx[2], ty[2], tz[2]; int tid[2], cnt[2] = { 0, 0 };
    float glo[3] = { INFINITY, INFINITY, INFINITY }, ghi[3] = { -INFINITY, -INFINITY, -INFINITY };
    const float4 pfirst = A.spm[gb];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const int i = gb + s * 32 + lane;
        const bool v = i < ge;
        const float4 p = v ? A.spm[i] : pfirst;
        tx[s] = p.x; ty[s] = p.y; tz[s] = p.z; tid[s] = v ? i : -1;
        glo[0] = fminf(glo[0], p.x); glo[1] = fminf(glo[1], p.y); glo[2] = fminf(glo[2], p.z);
        ghi[0] = fmaxf(ghi[0], p.x); ghi[1] = fmaxf(ghi[1], p.y); ghi[2] = fmaxf(ghi[2], p.z);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            glo[a] = fminf(glo[a], __shfl_xor_sync(0xffffffffu, glo[a], o));
            ghi[a] = fmaxf(ghi[a], __shfl_xor_sync(0xffffffffu, ghi[a], o));
        }

    // every group's lists start on a 32-entry (128-byte) boundary
    const long long pc_begin = pc_ptr, pp_begin = pp_ptr;
    int top = 1, npc = 0, npp = 0, fill_pc = 0, fill_pp = 0, overflow = 0, ovf = 0;
    if (lane == 0) S.stack[0] = 0;
    __syncwarp();
    while (top > 0) {
        const int take = min(top, 32);
        top -= take;
        const bool valid = lane < take;
        int node = 0;
        if (valid) node = stack_get(S, spill, top + lane);
        P3T_CHECK(node >= 0 && node < A.info->n_nodes);
        bool open = false;
        int2 link = make_int2(0, 0);
        if (valid) {
            const float4 com = A.ncom[node];
            const float4 lo = A.nlo[node], hi = A.nhi[node];
            link = A.nlink[node];
            // R-S7, every operation one fp32 rounding
            const float fx = fmaxf(fmaxf(0.0f, __fsub_rn(glo[0], hi.x)), __fsub_rn(lo.x, ghi[0]));
            const float fy = fmaxf(fmaxf(0.0f, __fsub_rn(glo[1], hi.y)), __fsub_rn(lo.y, ghi[1]));
            const float fz = fmaxf(fmaxf(0.0f, __fsub_rn(glo[2], hi.z)), __fsub_rn(lo.z, ghi[2]));
            const float b2 = fmaf(fz, fz, fmaf(fy, fy, __fmul_rn(fx, fx)));
            open = b2 < A.rout2;
            if (MODE == WALK_LISTS) {
                const float ex = fmaxf(fmaxf(0.0f, __fsub_rn(glo[0], com.x)), __fsub_rn(com.x, ghi[0]));
                const float ey = fmaxf(fmaxf(0.0f, __fsub_rn(glo[1], com.y)), __fsub_rn(com.y, ghi[1]));
                const float ez = fmaxf(fmaxf(0.0f, __fsub_rn(glo[2], com.z)), __fsub_rn(com.z, ghi[2]));
                const float d2 = fmaf(ez, ez, fmaf(ey, ey, __fmul_rn(ex, ex)));
                const float u = __fadd_rn(s_lt[__float_as_int(hi.w)], lo.w);
                open = open || d2 < __fmul_rn(u, u);
            }
        }
        const bool inner = valid && open && link.y > 0;
        const bool leaf  = valid && open && link.y < 0;
        const bool acc   = MODE == WALK_LISTS && valid && !open;
        // children of opened internal cells go on the stack
        if (__any_sync(0xffffffffu, inner)) {
            int c = inner ? link.y : 0, x = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            const int total = __shfl_sync(0xffffffffu, x, 31);
            if (top + total > STACK_CAP + A.spill_cap) { overflow = 1; break; }
            const int w = top + x - c;
            if (top + total <= STACK_CAP) {                    // warp-uniform: everything stays in shared memory
#pragma unroll
                for (int k = 0; k < 8; ++k) if (k < c) S.stack[w + k] = link.x + k;
            } else {
                for (int k = 0; k < c; ++k) stack_put(S, spill, w + k, link.x + k);
            }
            top += total;
        }
        // accepted cells: their ids go on the particle-cell list
        if (MODE == WALK_LISTS) {
            const uint32_t m = __ballot_sync(0xffffffffu, acc);
            P3T_CHECK(fill_pc + __popc(m) <= 64);
            if (acc) S.pcid[fill_pc + __popc(m & lt_mask)] = node;
            fill_pc += __popc(m);
            npc += __popc(m);
            __syncwarp();
            list_flush(S.pcid, fill_pc, A.pcpool, pc_ptr, pc_end, lane, ovf);
        }
        // opened leaves: inclusive scan of their particle counts; particle k of this iteration's leaves
        // belongs to the first lane whose inclusive count exceeds k (binary search by shuffle)
        int lc_incl = leaf ? -link.y : 0, src_total = 0;
        if (__any_sync(0xffffffffu, leaf)) {
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, lc_incl, o); if (lane >= o) lc_incl += y; }
            src_total = __shfl_sync(0xffffffffu, lc_incl, 31);
        }
        const int lc_excl = lc_incl - (leaf ? -link.y : 0);
        npp += src_total;
        for (int k0 = 0; k0 < src_total; k0 += 32) {
            const int m = min(32, src_total - k0);
            const int k = k0 + lane;
            int pos = 0;
#pragma unroll
            for (int st = 16; st > 0; st >>= 1) {
                const int v = __shfl_sync(0xffffffffu, lc_incl, pos + st - 1);
                if (v <= k) pos += st;
            }
            pos = min(pos, 31);
            const int j = __shfl_sync(0xffffffffu, link.x, pos) + (k - __shfl_sync(0xffffffffu, lc_excl, pos));
            if (MODE == WALK_LISTS) {
                P3T_CHECK(fill_pp + m <= 64 && (lane >= m || (j >= 0 && j < A.n)));
                if (lane < m) S.ppid[fill_pp + lane] = j;
                fill_pp += m;
                __syncwarp();
                list_flush(S.ppid, fill_pp, A.pppool, pp_ptr, pp_end, lane, ovf);
            } else {
                // R10 neighbour predicate, bit-specified fp32, for the 32 particles of this round
                // only the particles within r_out of the group box can be anyone's neighbour: the box distance below is
                // built from the same monotone fp32 operations as R10's d2, so it never exceeds the d2 to a target
                // inside the box and the cull is exact
                bool keep = false; float4 p = make_float4(0, 0, 0, 0);
                if (lane < m) {
                    p = A.spm[j];
                    const float fx = fmaxf(fmaxf(0.0f, __fsub_rn(glo[0], p.x)), __fsub_rn(p.x, ghi[0]));
                    const float fy = fmaxf(fmaxf(0.0f, __fsub_rn(glo[1], p.y)), __fsub_rn(p.y, ghi[1]));
                    const float fz = fmaxf(fmaxf(0.0f, __fsub_rn(glo[2], p.z)), __fsub_rn(p.z, ghi[2]));
                    keep = fmaf(fz, fz, fmaf(fy, fy, __fmul_rn(fx, fx))) < A.rout2;
                }
                const uint32_t km = __ballot_sync(0xffffffffu, keep);
                if (keep) { const int q = __popc(km & lt_mask); C->x[q] = p.x; C->y[q] = p.y; C->z[q] = p.z; }
                const int ms = __popc(km);
                __syncwarp();
                // both target slots of the lane in one packed operation; d = x_i - x_j here, the exact negative of
                // R10's x_j - x_i, so d2 has the same bits.  Self (always met: its own leaf is opened) is counted
                // and taken off at the end, which spares the index test in the loop.
                const f2 TX = pk(tx[0], tx[1]), TY = pk(ty[0], ty[1]), TZ = pk(tz[0], tz[1]);
                for (int e = 0; e < ms; ++e) {
                    const float px = C->x[e], py = C->y[e], pz = C->z[e];
                    const f2 dx = sub2(TX, pk(px, px)), dy = sub2(TY, pk(py, py)), dz = sub2(TZ, pk(pz, pz));
                    const f2 d2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
                    cnt[0] += f2lo(d2) < A.rout2 ? 1 : 0;
                    cnt[1] += f2hi(d2) < A.rout2 ? 1 : 0;
                }
                __syncwarp();
            }
        }
        __syncwarp();
    }

    if (MODE == WALK_LISTS) {
        // tails, padded to the 32-entry boundary (the force kernel masks by n_pc / n_pp)
        if (fill_pc > 0) { fill_pc = 32; list_flush(S.pcid, fill_pc, A.pcpool, pc_ptr, pc_end, lane, ovf); }
        if (fill_pp > 0) { fill_pp = 32; list_flush(S.ppid, fill_pp, A.pppool, pp_ptr, pp_end, lane, ovf); }
        if (lane == 0) {
            A.glist[g] = make_uint4((uint32_t)(pc_begin >> 5), (uint32_t)npc, (uint32_t)(pp_begin >> 5), (uint32_t)npp);
            A.gnpp[g] = npp; A.gnpc[g] = npc;
            const unsigned long long c = (unsigned long long)(ge - gb);
            atomicAdd(&A.info->n_pp, c * npp); atomicAdd(&A.info->n_pc, c * npc);
            atomicAdd(&A.info->n_pp_list, (unsigned long long)npp); atomicAdd(&A.info->n_pc_list, (unsigned long long)npc);
            if (ovf) atomicOr(&A.info->pool_overflow, 1);
        }
        // Publish the group: the force kernel (running at the same time) waits for this word.  Every lane's list stores
        // precede the warp barrier, lane 0's release makes them visible with the state.  A group whose lists are
        // incomplete is marked failed and skipped by the force kernel; the host's repair pass (this kernel again,
        // larger pools, A.repair) redoes it.
        __syncwarp();
        if (lane == 0) {
            const bool failed = ovf || overflow;
            if (A.repair) {
                const int v = A.gready[g];
                if (v == A.base + G_FAILED && !failed) A.gready[g] = A.base + G_REDONE;
            } else {
                const int want = A.base + (failed ? G_FAILED : G_READY);
                int v = *(volatile int32_t*)&A.gready[g];
                while (!g_decided(v, A.base)) {                     // decided already: a force warp gave up on this group
                    const int old = cas_release_gpu(&A.gready[g], v, want);
                    if (old == v) break;
                    v = old;
                }
            }
        }
    } else {
#pragma unroll
        for (int s = 0; s < 2; ++s)
            if (tid[s] >= 0) A.nbcount[A.order[tid[s]]] = cnt[s] - (0.0f < A.rout2 ? 1 : 0);   // minus self (d2 = 0)
    }
    if (lane == 0 && overflow) atomicOr(&A.info->stack_overflow, 1);
}

template <int MODE>
__global__ void __launch_bounds__(WALK_THREADS) k_walk(walk_args A)
{
    __shared__ warp_smem smem[WALK_WARPS];
    __shared__ count_smem csm[MODE == WALK_COUNT ? WALK_WARPS : 1];
    __shared__ float s_lt[24];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (A.info->bad_input | A.info->node_overflow) return;       // nothing is written for an invalid build (the host reports it)
    if (threadIdx.x < 24) s_lt[threadIdx.x] = __fdiv_rn(ldexpf(A.info->side, -(int)threadIdx.x), A.theta);
    __syncthreads();
    warp_smem& S = smem[w];
    const long long wg = (long long)blockIdx.x * WALK_WARPS + w;
    int32_t* spill = A.spill + wg * SPILL_CAP;
    long long pc_ptr = wg * A.cap_pc, pp_ptr = wg * A.cap_pp;
    const long long pc_base = pc_ptr, pp_base = pp_ptr, pc_end = pc_ptr + A.cap_pc, pp_end = pp_ptr + A.cap_pp;
    const int g0 = A.info->shard_g0, ng = A.info->shard_g1;      // all groups unless the context is sharded (p3t_shard.cu)
    uint32_t* cursor = MODE == WALK_LISTS ? &A.info->group_cursor : &A.info->group_cursor2;
    for (;;) {
        int g = 0;
        if (lane == 0) g = g0 + (int)atomicAdd(cursor, 1u);
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g >= ng) break;
        walk_group<MODE>(A, S, &csm[MODE == WALK_COUNT ? w : 0], spill, g, A.gbegin[g], A.gbegin[g + 1], s_lt, pc_ptr, pc_end, pp_ptr, pp_end);
        __syncwarp();
    }
    if (MODE == WALK_LISTS && lane == 0) {
        atomicMax(&A.info->need_pc, (uint32_t)min(pc_ptr - pc_base, 0xffffffffll));
        atomicMax(&A.info->need_pp, (uint32_t)min(pp_ptr - pp_base, 0xffffffffll));
    }
}

// all cursors and counters of one force call (one launch, before the count walk, the list walk and the force kernel
// go to their streams)
__global__ void k_walk_reset(p3t_devinfo* info)
{
    info->group_cursor2 = 0; info->nb_total = 0ull; info->nb_max = 0;
    info->group_cursor = 0; info->group_cursor3 = 0;
    info->n_pp = info->n_pc = info->n_pp_list = info->n_pc_list = 0ull;
    info->pool_overflow = 0; info->need_pc = 0; info->need_pp = 0;
    info->nb_overflow = 0; info->spin_abort = 0;
    info->stack_overflow = 0;     // a condition of one force call (its theta), not of the tree: the next call may fit
}

static int walk_blocks(p3t_ctx* ctx, int mode, int* out, bool limit_by_n = true)
{
    int* per_sm = ctx->occ_walk;                             // per context: contexts may sit on different devices
    if (!per_sm[mode]) {
        if (mode == WALK_COUNT) P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[0], k_walk<WALK_COUNT>, WALK_THREADS, 0));
        else                    P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[1], k_walk<WALK_LISTS>, WALK_THREADS, 0));
        if (per_sm[mode] < 1) per_sm[mode] = 1;
    }
    // a persistent grid, but no more warps than there can be groups of >= 32 particles: every walker
    // warp owns a private region of the list pools, and idle warps would only inflate them
    const long long by_n = limit_by_n ? (ctx->n / 32 + WALK_WARPS - 1) / WALK_WARPS : (1ll << 40);
    const long long full = (long long)per_sm[mode] * ctx->num_sms;
    *out = (int)(by_n < 1 ? 1 : by_n < full ? by_n : full);
    return P3T_OK;
}

static void fill_args(p3t_ctx* ctx, walk_args& A, float r_out, float theta)
{
    A.spm = P<float4>(ctx->spm); A.order = P<uint32_t>(ctx->idx[0]);
    A.ncom = P<float4>(ctx->ncom); A.nlo = P<float4>(ctx->nlo); A.nhi = P<float4>(ctx->nhi); A.nlink = P<int2>(ctx->nlink);
    A.gbegin = P<int32_t>(ctx->gbegin); A.gnpp = P<int32_t>(ctx->gnpp); A.gnpc = P<int32_t>(ctx->gnpc);
    A.nbcount = P<int32_t>(ctx->nbcount);
    A.pcpool = P<int32_t>(ctx->pcpool); A.pppool = P<int32_t>(ctx->pppool); A.glist = P<uint4>(ctx->glist);
    A.cap_pc = ctx->pool_cap_pc; A.cap_pp = ctx->pool_cap_pp;
    A.spill = P<int32_t>(ctx->spill); A.info = INFO(ctx);
    volatile float ro2 = r_out * r_out;           // one fp32 product, as R10 states it
    A.rout2 = ro2; A.theta = theta; A.n = (int)ctx->n;
    A.gready = P<int32_t>(ctx->gready); A.base = 0; A.repair = 0;
    A.spill_cap = (ctx->test_fault & 2) ? 0 : SPILL_CAP;
}

int p3t_launch_walk_reset(p3t_ctx* ctx, cudaStream_t st)
{
    k_walk_reset<<<1, 1, 0, st>>>(INFO(ctx));
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
    return P3T_OK;
}

// a10, first half: neighbour counts per ORIGINAL id into ctx->nbcount
int p3t_launch_walk_count(p3t_ctx* ctx, float r_out, float theta, cudaStream_t st)
{
    int blocks, rc;
    if ((rc = walk_blocks(ctx, WALK_COUNT, &blocks))) return rc;
    walk_args A; fill_args(ctx, A, r_out, theta);
    A.spill = P<int32_t>(ctx->spill) + (size_t)ctx->walk_warps_max * SPILL_CAP;      // second half: the list walk may run at the same time
    k_walk<WALK_COUNT><<<blocks, WALK_THREADS, 0, st>>>(A);
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
    return P3T_OK;
}

// buffers of both walks: reserved before anything of the call is enqueued (a reallocation synchronises)
int p3t_walk_reserve(p3t_ctx* ctx, int ctas_per_sm)
{
    int blocks, rc;
    if ((rc = walk_blocks(ctx, WALK_LISTS, &blocks))) return rc;
    if (ctas_per_sm > 0 && blocks > ctas_per_sm * ctx->num_sms) blocks = ctas_per_sm * ctx->num_sms;
    const long long warps = (long long)blocks * WALK_WARPS;
    if ((rc = p3t_reserve(ctx, &ctx->spill, (size_t)ctx->walk_warps_max * 2 * SPILL_CAP * sizeof(int32_t)))) return rc;
    if (ctx->pool_cap_pc == 0 || warps != ctx->walk_list_warps) {
        // first call (or another share of the device): a guess from the group count (lists of the paper's workloads
        // hold 4-8 thousand cells and 1-3 thousand particles at theta = 0.4); corrected by the repair pass if too small.
        // A context that has measured its need keeps the total and spreads it over the new number of walker warps.
        const long long ng = (ctx->n + 31) / 32;
        long long tot_pc = ng * 6000, tot_pp = ng * 3000;
        if (ctx->pool_cap_pc != 0) { tot_pc = ctx->pool_cap_pc * ctx->walk_list_warps; tot_pp = ctx->pool_cap_pp * ctx->walk_list_warps; }
        ctx->pool_cap_pc = ((tot_pc / warps + 16384) + 31) & ~31ll;
        ctx->pool_cap_pp = ((tot_pp / warps + 16384) + 31) & ~31ll;
        ctx->walk_list_warps = warps;
    }
    if ((rc = p3t_reserve(ctx, &ctx->pcpool, (size_t)(warps * ctx->pool_cap_pc) * 4))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->pppool, (size_t)(warps * ctx->pool_cap_pp) * 4))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->glist, ((size_t)ctx->n + 1) * sizeof(uint4)))) return rc;
    return P3T_OK;
}

// a7: interaction lists (p3t_walk_reserve has sized the pools for this share of the device)
int p3t_launch_walk_lists(p3t_ctx* ctx, float r_out, float theta, cudaStream_t st, int base, int repair, int ctas_per_sm)
{
    int blocks, rc;
    if ((rc = p3t_walk_reserve(ctx, ctas_per_sm))) return rc;
    blocks = (int)(ctx->walk_list_warps / WALK_WARPS);
    walk_args A; fill_args(ctx, A, r_out, theta);
    A.base = base; A.repair = repair;
    k_walk<WALK_LISTS><<<blocks, WALK_THREADS, 0, st>>>(A);
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
    return P3T_OK;
}

int p3t_walk_init(p3t_ctx* ctx)
{
    int b0, b1, rc;
    if ((rc = walk_blocks(ctx, WALK_COUNT, &b0, false))) return rc;
    if ((rc = walk_blocks(ctx, WALK_LISTS, &b1, false))) return rc;
    ctx->walk_warps_max = (long long)(b0 > b1 ? b0 : b1) * WALK_WARPS;
    return P3T_OK;
}
