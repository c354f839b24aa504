// p3t_walk.cu -- steps a7-a11: group tree walk, particle-cell and
// particle-particle regular force with the cutoff of eq. 6 and neighbour-list
// emission fused in, scatter of the results to the caller's particle order.
//
//   F_R,i = sum_j m_j W(x_ij) (x_j - x_i) / r_ij^3,  W = 1 - K,  x = (r - r_in)/(r_out - r_in)
//   (eq. 1, 3, 4, 6, 8-10; attractive sign: DESIGN.md R1)
//
// One warp walks one target group (<= 64 particles, two target slots per lane).  Rules:
// DESIGN.md R-S7 (opening rule, bit-specified fp32), R-S8 (evaluation), R-S9 (accumulation),
// R10 (neighbour predicate, bit-specified fp32).
#include "p3t_internal.cuh"

#define WALK_WARPS   4                    // warps per CTA, each walks its own groups
#define WALK_THREADS (WALK_WARPS * 32)
#define STACK_CAP    512                  // per-warp node stack in shared memory; deeper entries spill
#define SPILL_CAP    8192                 // per-warp spill (global memory), entries
#define PC_TILE      32                   // cells evaluated per flush
#define PP_TILE      64                   // particles evaluated per flush

struct walk_consts {
    float rout2, rin2, r_in, inv_delta;   // inv_delta = 1 / (r_out - r_in)
    float psi_in;                          // psi(r_in), the constant regular pair potential inside r_in
    float k140;                            // 140 / (r_out - r_in)
    float s1;                              // S(1)
    float sc[6];                           // S(t) = t (sc0 + t (sc1 + ... t sc5))
    float rem;                             // c^3 (1+c)^3  (> 0)
    float c;                               // r_in / (r_out - r_in)
    float theta;
    int   pot_mode;
};

struct walk_args {
    const float4* spm; const uint32_t* order;
    const float4 *ncom, *nlo, *nhi, *nq0; const float2* nq1; const int2* nlink;
    const int32_t* gbegin;
    int32_t *gnpp, *gnpc;
    int32_t* nbcount;           // MODE 0 out: per ORIGINAL id
    const int64_t* nboff;       // MODE 1 in:  per ORIGINAL id
    int32_t* nbraw;             // MODE 1 out: unsorted rows
    float4* out;                // MODE 1 out: acc_pot, original order
    int32_t* spill;
    p3t_devinfo* info;
    walk_consts K;
};

struct warp_smem {
    int    stack[STACK_CAP];
    float4 pc_com[PC_TILE + 32];
    float4 pc_q0[PC_TILE + 32];
    float2 pc_q1[PC_TILE + 32];
    float4 pp_pos[PP_TILE + 32];
    int    pp_j[PP_TILE + 32];
};

__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// eq. 6, 0 < x < 1: W = x^4 (35 - 84 x + 70 x^2 - 20 x^3); evaluated through the
// symmetry W(x) = 1 - W(1 - x) above x = 1/2 so that fp32 Horner never cancels.
__device__ __forceinline__ float cutoff_W(float x)
{
    float t = x > 0.5f ? 1.0f - x : x;
    float t2 = t * t;
    float w = t2 * t2 * (35.0f + t * (-84.0f + t * (70.0f - 20.0f * t)));
    return x > 0.5f ? 1.0f - w : w;
}

// regular pair potential for r_in < r < r_out (R6): -W/r - (140/D) int_x^1 t^3(1-t)^3/(t+c) dt
__device__ __forceinline__ float cutoff_psi(const walk_consts& K, float x, float W, float rinv)
{
    float sx = x * (K.sc[0] + x * (K.sc[1] + x * (K.sc[2] + x * (K.sc[3] + x * (K.sc[4] + x * K.sc[5])))));
    float integral = (K.s1 - sx) - K.rem * __logf((1.0f + K.c) / (x + K.c));
    return -W * rinv - K.k140 * integral;
}

template <int NS> struct target {
    float x[NS], y[NS], z[NS];
    float ax[NS], ay[NS], az[NS], ph[NS];        // fp32 partial sums of the current tile
    double dax[NS], day[NS], daz[NS], dph[NS];   // fp64 masters (R-S9)
    int   id[NS];                                // sorted position of the target, -1 = no target
    long long cur[NS];                           // neighbour write cursor (MODE 1) / count (MODE 0)
};

template <int NS> __device__ __forceinline__ void fold(target<NS>& T)
{
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        T.dax[s] += (double)T.ax[s]; T.day[s] += (double)T.ay[s]; T.daz[s] += (double)T.az[s]; T.dph[s] += (double)T.ph[s];
        T.ax[s] = T.ay[s] = T.az[s] = T.ph[s] = 0.0f;
    }
}

// R-S8 particle-cell: monopole + traceless quadrupole, r = x_i - COM
//   phi = -M/R - (1/2) r.Q.r / R^5 ;  a = -M r/R^3 + Q.r/R^5 - (5/2)(r.Q.r) r/R^7
template <int NS> __device__ __forceinline__ void eval_pc(target<NS>& T, const warp_smem& S, int cnt)
{
#pragma unroll 2
    for (int e = 0; e < cnt; ++e) {
        const float4 cm = S.pc_com[e], q0 = S.pc_q0[e];
        const float2 q1 = S.pc_q1[e];
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const float rx = T.x[s] - cm.x, ry = T.y[s] - cm.y, rz = T.z[s] - cm.z;
            const float R2 = fmaf(rz, rz, fmaf(ry, ry, rx * rx));
            const float ri = rsqrt_approx(R2), ri2 = ri * ri;
            const float qx = fmaf(q1.x, rz, fmaf(q0.w, ry, q0.x * rx));      // (Q r)_x = xx rx + xy ry + xz rz
            const float qy = fmaf(q1.y, rz, fmaf(q0.y, ry, q0.w * rx));      // xy rx + yy ry + yz rz
            const float qz = fmaf(q0.z, rz, fmaf(q1.y, ry, q1.x * rx));      // xz rx + yz ry + zz rz
            const float rqr = fmaf(rz, qz, fmaf(ry, qy, rx * qx));
            const float ri3 = ri2 * ri, ri5 = ri3 * ri2;
            const float mono = cm.w * ri;                                      // M / R
            const float quad = 0.5f * rqr * ri5;                               // (1/2) rQr / R^5
            T.ph[s] -= mono + quad;
            const float cr = -(mono + 5.0f * quad) * ri2;                      // -(M/R^3 + (5/2) rQr/R^7)
            T.ax[s] += fmaf(cr, rx, qx * ri5);
            T.ay[s] += fmaf(cr, ry, qy * ri5);
            T.az[s] += fmaf(cr, rz, qz * ri5);
        }
    }
}

// R10 + eq. 6: particle-particle with cutoff; MODE 0 counts neighbours only, MODE 1 also emits
template <int NS, int MODE>
__device__ __forceinline__ void eval_pp(target<NS>& T, const warp_smem& S, int cnt, const walk_args& A)
{
    const walk_consts& K = A.K;
#pragma unroll 2
    for (int e = 0; e < cnt; ++e) {
        const float4 p = S.pp_pos[e];
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const float dx = __fsub_rn(p.x, T.x[s]), dy = __fsub_rn(p.y, T.y[s]), dz = __fsub_rn(p.z, T.z[s]);
            const float d2 = fmaf(dz, dz, fmaf(dy, dy, __fmul_rn(dx, dx)));
            if (d2 < K.rout2) {
                const int j = S.pp_j[e];
                if (T.id[s] >= 0 && j != T.id[s]) {                  // self excluded by index
                    if (MODE == 1) A.nbraw[T.cur[s]] = (int32_t)A.order[j];
                    T.cur[s]++;
                    if (MODE == 1) {
                        if (d2 > K.rin2) {
                            const float ri = rsqrt_approx(d2), r = d2 * ri;
                            const float x = fminf(fmaxf((r - K.r_in) * K.inv_delta, 0.0f), 1.0f);
                            const float W = cutoff_W(x);
                            const float f = p.w * W * ri * ri * ri;
                            T.ax[s] = fmaf(f, dx, T.ax[s]); T.ay[s] = fmaf(f, dy, T.ay[s]); T.az[s] = fmaf(f, dz, T.az[s]);
                            T.ph[s] += K.pot_mode == 0 ? p.w * cutoff_psi(K, x, W, ri) : -p.w * ri;
                        } else if (K.pot_mode == 0) {
                            T.ph[s] = fmaf(p.w, K.psi_in, T.ph[s]);    // inside r_in: constant psi(r_in), also r = 0 (R8)
                        } else if (d2 > 0.0f) {
                            T.ph[s] -= p.w * rsqrt_approx(d2);
                        }
                    }
                }
            } else if (MODE == 1) {
                const float ri = rsqrt_approx(d2);
                const float mr = p.w * ri, mr3 = mr * ri * ri;
                T.ph[s] -= mr;
                T.ax[s] = fmaf(mr3, dx, T.ax[s]); T.ay[s] = fmaf(mr3, dy, T.ay[s]); T.az[s] = fmaf(mr3, dz, T.az[s]);
            }
        }
    }
}

__device__ __forceinline__ int stack_get(const warp_smem& S, const int32_t* spill, int i)
{
    return i < STACK_CAP ? S.stack[i] : spill[i - STACK_CAP];
}
__device__ __forceinline__ void stack_put(warp_smem& S, int32_t* spill, int i, int v)
{
    if (i < STACK_CAP) S.stack[i] = v; else spill[i - STACK_CAP] = v;
}

template <int NS, int MODE>
__device__ void walk_group(const walk_args& A, warp_smem& S, int32_t* spill, int g, int gb, int ge,
                           const float* s_lt /* [24] fl(l/theta) per level */)
{
    const int lane = threadIdx.x & 31;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const walk_consts& K = A.K;
    target<NS> T;
    float glo[3] = { INFINITY, INFINITY, INFINITY }, ghi[3] = { -INFINITY, -INFINITY, -INFINITY };
    const float4 pfirst = A.spm[gb];
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        const int i = gb + s * 32 + lane;
        const bool v = i < ge;
        const float4 p = v ? A.spm[i] : pfirst;
        T.x[s] = p.x; T.y[s] = p.y; T.z[s] = p.z;
        T.ax[s] = T.ay[s] = T.az[s] = T.ph[s] = 0.0f;
        T.dax[s] = T.day[s] = T.daz[s] = T.dph[s] = 0.0;
        T.id[s] = v ? i : -1;
        T.cur[s] = 0;
        if (MODE == 1 && v) T.cur[s] = A.nboff[A.order[i]];
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

    int top = 1, npc = 0, npp = 0, fill_pc = 0, fill_pp = 0, overflow = 0;
    if (lane == 0) S.stack[0] = 0;
    __syncwarp();
    while (top > 0) {
        const int take = min(top, 32);
        top -= take;
        const bool valid = lane < take;
        int node = 0;
        if (valid) node = stack_get(S, spill, top + lane);
        bool open = false;
        int2 link = make_int2(0, 0);
        float4 com = make_float4(0, 0, 0, 0);
        if (valid) {
            com = A.ncom[node];
            const float4 lo = A.nlo[node], hi = A.nhi[node];
            link = A.nlink[node];
            // R-S7, every operation one fp32 rounding
            const float ex = fmaxf(fmaxf(0.0f, __fsub_rn(glo[0], com.x)), __fsub_rn(com.x, ghi[0]));
            const float ey = fmaxf(fmaxf(0.0f, __fsub_rn(glo[1], com.y)), __fsub_rn(com.y, ghi[1]));
            const float ez = fmaxf(fmaxf(0.0f, __fsub_rn(glo[2], com.z)), __fsub_rn(com.z, ghi[2]));
            const float fx = fmaxf(fmaxf(0.0f, __fsub_rn(glo[0], hi.x)), __fsub_rn(lo.x, ghi[0]));
            const float fy = fmaxf(fmaxf(0.0f, __fsub_rn(glo[1], hi.y)), __fsub_rn(lo.y, ghi[1]));
            const float fz = fmaxf(fmaxf(0.0f, __fsub_rn(glo[2], hi.z)), __fsub_rn(lo.z, ghi[2]));
            const float d2 = fmaf(ez, ez, fmaf(ey, ey, __fmul_rn(ex, ex)));
            const float b2 = fmaf(fz, fz, fmaf(fy, fy, __fmul_rn(fx, fx)));
            const float u = __fadd_rn(s_lt[__float_as_int(hi.w)], lo.w);
            const float rc2 = __fmul_rn(u, u);
            const bool near = b2 < K.rout2;
            open = MODE == 1 ? ((d2 < rc2) || near) : near;
        }
        const bool inner = valid && open && link.y > 0;
        const bool leaf  = valid && open && link.y < 0;
        const bool acc   = MODE == 1 && valid && !open;
        // children of opened internal cells go on the stack
        {
            int c = inner ? link.y : 0, x = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            const int total = __shfl_sync(0xffffffffu, x, 31);
            if (top + total > STACK_CAP + SPILL_CAP) { overflow = 1; break; }
            int w = top + x - c;
            for (int k = 0; k < c; ++k) stack_put(S, spill, w + k, link.x + k);
            top += total;
        }
        // accepted cells go on the particle-cell tile
        if (MODE == 1) {
            const uint32_t m = __ballot_sync(0xffffffffu, acc);
            if (acc) {
                const int w = fill_pc + __popc(m & lt_mask);
                S.pc_com[w] = com; S.pc_q0[w] = A.nq0[node]; S.pc_q1[w] = A.nq1[node];
            }
            fill_pc += __popc(m);
            npc += __popc(m);
        }
        // opened leaves: their particles go on the particle-particle tile
        uint32_t lm = __ballot_sync(0xffffffffu, leaf);
        __syncwarp();
        while (lm) {
            const int src = __ffs(lm) - 1;
            lm &= lm - 1;
            const int lb = __shfl_sync(0xffffffffu, link.x, src);
            const int lc = -__shfl_sync(0xffffffffu, link.y, src);
            npp += lc;
            for (int o = 0; o < lc; o += 32) {
                const int m = min(32, lc - o);
                if (lane < m) { S.pp_pos[fill_pp + lane] = A.spm[lb + o + lane]; S.pp_j[fill_pp + lane] = lb + o + lane; }
                fill_pp += m;
                __syncwarp();
                if (fill_pp >= PP_TILE) {
                    eval_pp<NS, MODE>(T, S, PP_TILE, A);
                    if (MODE == 1) fold(T);
                    __syncwarp();
                    const int rest = fill_pp - PP_TILE;
                    float4 tp; int tj;
                    if (lane < rest) { tp = S.pp_pos[PP_TILE + lane]; tj = S.pp_j[PP_TILE + lane]; }
                    __syncwarp();
                    if (lane < rest) { S.pp_pos[lane] = tp; S.pp_j[lane] = tj; }
                    fill_pp = rest;
                    __syncwarp();
                }
            }
        }
        if (MODE == 1 && fill_pc >= PC_TILE) {
            __syncwarp();
            eval_pc<NS>(T, S, PC_TILE);
            fold(T);
            __syncwarp();
            const int rest = fill_pc - PC_TILE;
            float4 a, b; float2 c;
            if (lane < rest) { a = S.pc_com[PC_TILE + lane]; b = S.pc_q0[PC_TILE + lane]; c = S.pc_q1[PC_TILE + lane]; }
            __syncwarp();
            if (lane < rest) { S.pc_com[lane] = a; S.pc_q0[lane] = b; S.pc_q1[lane] = c; }
            fill_pc = rest;
        }
        __syncwarp();
    }
    // tails
    __syncwarp();
    if (fill_pp > 0) { eval_pp<NS, MODE>(T, S, fill_pp, A); if (MODE == 1) fold(T); }
    if (MODE == 1 && fill_pc > 0) { eval_pc<NS>(T, S, fill_pc); fold(T); }
    __syncwarp();

    // a11: results to the caller's order
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        if (T.id[s] < 0) continue;
        const uint32_t orig = A.order[T.id[s]];
        if (MODE == 1) A.out[orig] = make_float4((float)T.dax[s], (float)T.day[s], (float)T.daz[s], (float)T.dph[s]);
        else A.nbcount[orig] = (int32_t)T.cur[s];
    }
    if (lane == 0) {
        if (MODE == 1) {
            A.gnpp[g] = npp; A.gnpc[g] = npc;
            const unsigned long long cnt = (unsigned long long)(ge - gb);
            atomicAdd(&A.info->n_pp, cnt * npp); atomicAdd(&A.info->n_pc, cnt * npc);
            atomicAdd(&A.info->n_pp_list, (unsigned long long)npp); atomicAdd(&A.info->n_pc_list, (unsigned long long)npc);
        }
        if (overflow) atomicOr(&A.info->stack_overflow, 1);
    }
}

template <int MODE>
__global__ void __launch_bounds__(WALK_THREADS) k_walk(walk_args A)
{
    __shared__ warp_smem smem[WALK_WARPS];
    __shared__ float s_lt[24];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x < 24) s_lt[threadIdx.x] = __fdiv_rn(ldexpf(A.info->side, -(int)threadIdx.x), A.K.theta);
    __syncthreads();
    warp_smem& S = smem[w];
    int32_t* spill = A.spill + (size_t)(blockIdx.x * WALK_WARPS + w) * SPILL_CAP;
    const int ng = A.info->n_groups;
    uint32_t* cursor = MODE == 1 ? &A.info->group_cursor : &A.info->group_cursor2;
    for (;;) {
        int g = 0;
        if (lane == 0) g = (int)atomicAdd(cursor, 1u);
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g >= ng) break;
        const int gb = A.gbegin[g], ge = A.gbegin[g + 1];
        if (ge - gb > 32) walk_group<2, MODE>(A, S, spill, g, gb, ge, s_lt);
        else              walk_group<1, MODE>(A, S, spill, g, gb, ge, s_lt);
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------
// a10  neighbour CSR: exclusive scan of the per-particle counts (original order) -> int64 offsets
// ---------------------------------------------------------------------------------------------
#define SCAN_TILE 4096

__global__ void __launch_bounds__(256) k_nb_blocksum(const int32_t* __restrict__ cnt, int n, long long* __restrict__ bsum,
                                                     p3t_devinfo* info)
{
    __shared__ long long s_sum[8];
    __shared__ int s_max[8];
    const int base = blockIdx.x * SCAN_TILE + threadIdx.x * 16;
    long long t = 0; int mx = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) { int i = base + k; int v = i < n ? cnt[i] : 0; t += v; mx = max(mx, v); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { t += __shfl_xor_sync(0xffffffffu, t, o); mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o)); }
    if ((threadIdx.x & 31) == 0) { s_sum[threadIdx.x >> 5] = t; s_max[threadIdx.x >> 5] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) { t += s_sum[k]; mx = max(mx, s_max[k]); }
        bsum[blockIdx.x] = t;
        atomicMax(&info->nb_max, mx);
    }
}

__global__ void __launch_bounds__(1024) k_nb_scansums(long long* __restrict__ bsum, int nb, long long* __restrict__ off_n,
                                                      p3t_devinfo* info)
{
    __shared__ long long s_w[32];
    __shared__ long long s_run;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_run = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nb; b0 += 1024) {
        const int b = b0 + threadIdx.x;
        long long v = b < nb ? bsum[b] : 0, x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { long long y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) s_w[w] = x;
        __syncthreads();
        long long add = s_run, tot = 0;
        for (int k = 0; k < 32; ++k) { long long t = s_w[k]; if (k < w) add += t; tot += t; }
        if (b < nb) bsum[b] = add + x - v;
        __syncthreads();
        if (threadIdx.x == 0) s_run += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) { *off_n = s_run; info->nb_total = (unsigned long long)s_run; }
}

__global__ void __launch_bounds__(256) k_nb_offsets(const int32_t* __restrict__ cnt, int n, const long long* __restrict__ bsum,
                                                    long long* __restrict__ off)
{
    __shared__ long long s_w[8];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int base = blockIdx.x * SCAN_TILE + threadIdx.x * 16;
    int v[16]; long long t = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) { int i = base + k; v[k] = i < n ? cnt[i] : 0; t += v[k]; }
    long long x = t;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { long long y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) s_w[w] = x;
    __syncthreads();
    long long run = bsum[blockIdx.x] + x - t;
    for (int k = 0; k < w; ++k) run += s_w[k];
#pragma unroll
    for (int k = 0; k < 16; ++k) { int i = base + k; if (i < n) off[i] = run; run += v[k]; }
}

// rows ascending in original id: rank sort (ids inside a row are distinct), out of place.
// Each lane sorts its own short row; rows longer than 16 are done by the whole warp.
__global__ void __launch_bounds__(256) k_nb_sortrows(const long long* __restrict__ off, const int32_t* __restrict__ raw,
                                                     int32_t* __restrict__ idx, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    long long b = 0; int len = 0;
    if (i < n) { b = off[i]; len = (int)(off[i + 1] - b); }
    if (len <= 16) {
        for (int a = 0; a < len; ++a) {
            const int v = raw[b + a]; int r = 0;
            for (int c = 0; c < len; ++c) r += raw[b + c] < v;
            idx[b + r] = v;
        }
    }
    uint32_t m = __ballot_sync(0xffffffffu, len > 16);
    while (m) {
        const int src = __ffs(m) - 1; m &= m - 1;
        const long long rb = __shfl_sync(0xffffffffu, b, src);
        const int rl = __shfl_sync(0xffffffffu, len, src);
        for (int a = lane; a < rl; a += 32) {
            const int v = raw[rb + a]; int r = 0;
            for (int c = 0; c < rl; ++c) r += raw[rb + c] < v;
            idx[rb + r] = v;
        }
    }
}

__global__ void k_force_reset(p3t_devinfo* info)
{
    info->group_cursor = 0; info->group_cursor2 = 0;
    info->n_pp = info->n_pc = info->n_pp_list = info->n_pc_list = 0ull;
    info->nb_total = 0ull; info->nb_max = 0;
}

// ---------------------------------------------------------------------------------------------
static void make_consts(walk_consts& K, float r_out, float r_in, float theta, int pot_mode)
{
    // fp32 thresholds exactly as DESIGN.md R10 states them: one fp32 product each
    volatile float ro2 = r_out * r_out, ri2 = r_in * r_in;
    K.rout2 = ro2; K.rin2 = ri2; K.r_in = r_in;
    const double D = (double)r_out - (double)r_in, c = (double)r_in / D, c1 = 1.0 + c;
    K.inv_delta = (float)(1.0 / D);
    K.k140 = (float)(140.0 / D);
    // t^3 (1-t)^3 = (t + c) (b5 t^5 + ... + b0) - c^3 (1+c)^3   (synthetic division at t = -c)
    const double b[6] = { c * c * c1 * c1 * c1, -c * c1 * c1 * c1, c1 * c1 * c1, -(3.0 + 3.0 * c + c * c), 3.0 + c, -1.0 };
    double s1 = 0.0;
    for (int k = 0; k < 6; ++k) { K.sc[k] = (float)(b[k] / (k + 1)); s1 += b[k] / (k + 1); }
    K.s1 = (float)s1;
    K.rem = (float)(c * c * c * c1 * c1 * c1);
    K.c = (float)c;
    // psi(r_in) = -(140/D) [ S(1) + rem ln((1+c)/c) ... ] with W(0) = 0; here the remainder enters with a minus sign
    K.psi_in = (float)(-(140.0 / D) * (s1 - c * c * c * c1 * c1 * c1 * log(c1 / c)));
    K.theta = theta;
    K.pot_mode = pot_mode;
}

int p3t_launch_force(p3t_ctx* ctx, float r_out, float r_in, float theta, int pot_mode, float4* acc_pot)
{
    const int n = (int)ctx->n;
    static int per_sm[2] = { 0, 0 };
    if (!per_sm[0]) {
        P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[0], k_walk<0>, WALK_THREADS, 0));
        P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[1], k_walk<1>, WALK_THREADS, 0));
        if (per_sm[0] < 1) per_sm[0] = 1;
        if (per_sm[1] < 1) per_sm[1] = 1;
    }
    const int blocks0 = per_sm[0] * ctx->num_sms, blocks1 = per_sm[1] * ctx->num_sms;
    const int maxblocks = blocks0 > blocks1 ? blocks0 : blocks1;
    int rc;
    if ((rc = p3t_reserve(ctx, &ctx->spill, (size_t)maxblocks * WALK_WARPS * SPILL_CAP * sizeof(int32_t)))) return rc;
    const int nsb = (n + SCAN_TILE - 1) / SCAN_TILE;
    if ((rc = p3t_reserve(ctx, &ctx->nbcount, (size_t)n * 4))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->nboff, ((size_t)n + 1) * 8))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->nbcur, (size_t)nsb * 8 + 64))) return rc;

    walk_args A;
    A.spm = P<float4>(ctx->spm); A.order = P<uint32_t>(ctx->idx[0]);
    A.ncom = P<float4>(ctx->ncom); A.nlo = P<float4>(ctx->nlo); A.nhi = P<float4>(ctx->nhi);
    A.nq0 = P<float4>(ctx->nq0); A.nq1 = P<float2>(ctx->nq1); A.nlink = P<int2>(ctx->nlink);
    A.gbegin = P<int32_t>(ctx->gbegin); A.gnpp = P<int32_t>(ctx->gnpp); A.gnpc = P<int32_t>(ctx->gnpc);
    A.nbcount = P<int32_t>(ctx->nbcount); A.nboff = P<int64_t>(ctx->nboff);
    A.nbraw = nullptr; A.out = acc_pot; A.spill = P<int32_t>(ctx->spill); A.info = INFO(ctx);
    make_consts(A.K, r_out, r_in, theta, pot_mode);

    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[4], ctx->stream));
    k_force_reset<<<1, 1, 0, ctx->stream>>>(INFO(ctx));
    // pass 1 (range search only): neighbour counts, so that the lists can be written in place
    k_walk<0><<<blocks0, WALK_THREADS, 0, ctx->stream>>>(A);
    k_nb_blocksum<<<nsb, 256, 0, ctx->stream>>>(A.nbcount, n, P<long long>(ctx->nbcur), INFO(ctx));
    k_nb_scansums<<<1, 1024, 0, ctx->stream>>>(P<long long>(ctx->nbcur), nsb, P<long long>(ctx->nboff) + n, INFO(ctx));
    k_nb_offsets<<<nsb, 256, 0, ctx->stream>>>(A.nbcount, n, P<long long>(ctx->nbcur), P<long long>(ctx->nboff));
    P3T_CUDA(ctx, cudaGetLastError());
    // the list buffers are sized from the total: the one host synchronisation of this call
    long long total = 0;
    P3T_CUDA(ctx, cudaMemcpyAsync(&total, P<long long>(ctx->nboff) + n, 8, cudaMemcpyDeviceToHost, ctx->stream));
    P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->nb_total_host = total;
    if ((rc = p3t_reserve(ctx, &ctx->nbidx, (size_t)total * 4 + 64))) return rc;
    p3t_buf* raw = &ctx->stage_out;      // unsorted rows share the host-staging scratch
    if ((rc = p3t_reserve(ctx, raw, (size_t)total * 4 + 64))) return rc;
    A.nbraw = P<int32_t>(*raw);
    // pass 2: walk + force + emission
    P3T_CUDA(ctx, cudaEventRecord(ctx->evw[0], ctx->stream));
    k_walk<1><<<blocks1, WALK_THREADS, 0, ctx->stream>>>(A);
    P3T_CUDA(ctx, cudaEventRecord(ctx->evw[1], ctx->stream));
    k_nb_sortrows<<<(n + 255) / 256, 256, 0, ctx->stream>>>(P<long long>(ctx->nboff), A.nbraw, P<int32_t>(ctx->nbidx), n);
    P3T_CUDA(ctx, cudaGetLastError());
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[5], ctx->stream));
    ctx->launches += 7;
    return P3T_OK;
}
