// p3t_irregular.cu -- SURVEY.md 8f NEXT-1: the irregular force, its time derivative (jerk) and the
// irregular potential of every particle over the neighbour list that p3t_regular_force emitted
// (eq. 1, 2, 5, 7; the paper's CUTOFF / cutoff0 routines, Table B2 :396-398).
//
// With d = x_j - x_i, v = xdot_j - xdot_i (attractive sign: DESIGN.md R1), r = |d|,
// x = (r - r_in)/(r_out - r_in), K = 1 - W (eq. 6):
//     F_I    = sum_{j in L(i)} m_j K d / r^3                                               (eq. 1)
//     Fdot_I = sum_{j in L(i)} m_j [ K ( v / r^3 - 3 (d.v) d / r^5 ) + Kdot d / r^3 ]      (eq. 2)
//     Kdot   = -W'(x) (d.v) / (r (r_out - r_in)),  W'(x) = 140 x^3 (1-x)^3                 (eq. 7)
//     phi_I  = sum_{j in L(i)} m_j ( -1/r - psi(r) )            (so that phi_I + phi_R = phi_Newton)
// Reading R2: eq. 2 / 7 are garbled in the text; Fdot_I is the exact time derivative of
// eq. 1.  Coincident pairs (r = 0, R8) are skipped.
//
// The lists are short (mean 2 entries at the paper's radii, up to ~500 in a King core): one thread
// per row up to 32 entries, one warp per longer row; terms in fp32 (IEEE sqrt and division, so that
// the r^-5 factor keeps 1e-7), sums in fp64.  HBM/L2-bound gather: 36 B per list entry.
#include "p3t_internal.cuh"
#include "p3t_cutoff.cuh"

// The integral I(x) = int_x^1 t^3 (1-t)^3 / (t + c) dt of the pair potential (R6) has a closed form
// that cancels (two terms of order 1 give 1e-2 .. 0): instead of evaluating it in fp64 with a log per list entry,
// the kernel interpolates a table made on the host in fp64 at every change of the radii: PSI_TAB intervals, cubic
// Hermite (the derivative -t^3 (1-t)^3 / (t + c) is exact), error h^4 max|4th derivative| / 384 < 1e-11.  Per
// interval two float4: (I_k hi, I_k lo, h I'_k, I_k+1 - I_k), (h I'_k+1, 0, 0, 0); the value is put together in fp64.
#define PSI_TAB 256

struct irr_args {
    const float4* spm; const int32_t* rank;     // sorted bodies, original id -> sorted position
    const uint32_t* order;                      // sorted position -> original id
    const float4* vel;                          // original order
    const int64_t* nboff; const int32_t* nbidx; // CSR, original ids
    float4 *acc, *jerk;                         // original order
    int n;
    const float4* psitab;                       // [PSI_TAB][2]
    const float4* pv;                           // [n][2]: position + mass, velocity; original order (k_irr_pack; PV only)
    walk_consts K;
};

struct irr_sum { double ax, ay, az, jx, jy, jz, ph; };

struct irr_src { float4 p, v; };

__device__ __forceinline__ void irr_term(const irr_args& A, const float4 pi, const float4 vi, const irr_src src, irr_sum& S)
{
    const walk_consts& K = A.K;
    const float4 pj = src.p, vj = src.v;
    const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if (!(r2 > 0.0f)) return;                                    // coincident pair (R8)
    const float vx = vj.x - vi.x, vy = vj.y - vi.y, vz = vj.z - vi.z;
    const float r = sqrtf(r2), ri = 1.0f / r, ri2 = ri * ri, ri3 = ri2 * ri;
    const float dv = fmaf(dz, vz, fmaf(dy, vy, dx * vx));
    const float m = pj.w;
    float Kc = 1.0f, Kdot = 0.0f, ph;
    if (r2 > K.rin2) {
        const float x = fminf(fmaxf((r - K.r_in) * K.inv_delta, 0.0f), 1.0f), y = 1.0f - x;
        Kc = cutoff_W(y);                                        // K(x) = 1 - W(x) = W(1 - x), no cancellation
        const float xy = x * y;
        Kdot = -140.0f * xy * xy * xy * dv * ri * K.inv_delta;   // -W'(x) xdot
        // -1/r - psi = -K/r + (140/D) int_x^1 t^3 (1-t)^3 / (t+c) dt = -cutoff_psi with W replaced by -K
        const float xs = x * (float)PSI_TAB;
        const int kt = min((int)xs, PSI_TAB - 1);
        const float t = xs - (float)kt, t2 = t * t, t3 = t2 * t;
        const float4 ta = __ldg(A.psitab + 2 * kt), tb = __ldg(A.psitab + 2 * kt + 1);
        const float dI = fmaf(t3 - t2, tb.x, fmaf(3.0f * t2 - 2.0f * t3, ta.w, (t3 - 2.0f * t2 + t) * ta.z));
        ph = (float)(K.dk140 * ((double)ta.x + (double)(ta.y + dI)) - (double)Kc * (double)ri);
    } else {
        ph = -ri - K.psi_in;
    }
    const float a = m * Kc * ri3;                                // m K / r^3
    const float b = m * (Kdot * ri3 - 3.0f * Kc * dv * ri3 * ri2);   // m ( Kdot / r^3 - 3 K (d.v) / r^5 )
    S.ax += (double)(a * dx); S.ay += (double)(a * dy); S.az += (double)(a * dz);
    S.jx += (double)fmaf(a, vx, b * dx); S.jy += (double)fmaf(a, vy, b * dy); S.jz += (double)fmaf(a, vz, b * dz);
    S.ph += (double)(m * ph);
}

// The entries first + k stride, k < cnt, of one row, in order.  The kernel is bound by the latency of the
// dependent gathers: they are staged over several iterations, so that every load issued in an iteration depends
// only on values that arrived during earlier ones (indices are clamped to the row, which keeps every staged load
// valid without predicates).  PV = false: index -> rank -> (position, velocity), four stages.  PV = true (lists
// with many entries per particle): position and velocity of a member come from one 32-byte record pv[j] in
// original order written by k_irr_pack, one sector per entry instead of three and one stage fewer.
template <bool PV>
__device__ __forceinline__ void irr_row(const irr_args& A, const float4 pi, const float4 vi, const int32_t* __restrict__ idx,
                                        int first, int cnt, int stride, irr_sum& S)
{
    if (cnt <= 0) return;
    const int last = cnt - 1;
    int j1 = idx[first], j2 = idx[first + min(1, last) * stride], j3 = idx[first + min(2, last) * stride];
    irr_src c1, c2;
    if (PV) {
        c1.p = A.pv[2 * (size_t)j1]; c1.v = A.pv[2 * (size_t)j1 + 1];
        c2.p = A.pv[2 * (size_t)j2]; c2.v = A.pv[2 * (size_t)j2 + 1];
#pragma unroll 1
        for (int k = 0; k < cnt; ++k) {
            const irr_src cur = c1;
            c1 = c2;
            c2.p = A.pv[2 * (size_t)j3]; c2.v = A.pv[2 * (size_t)j3 + 1];      // entry k + 2
            j3 = idx[first + min(k + 3, last) * stride];                       // entry k + 3
            irr_term(A, pi, vi, cur, S);
        }
    } else {
        int j4 = idx[first + min(3, last) * stride];
        int r1 = A.rank[j1], r2 = A.rank[j2], r3 = A.rank[j3];
        c1.p = A.spm[r1]; c1.v = A.vel[j1];
        c2.p = A.spm[r2]; c2.v = A.vel[j2];
#pragma unroll 1
        for (int k = 0; k < cnt; ++k) {
            const irr_src cur = c1;
            c1 = c2;
            c2.p = A.spm[r3]; c2.v = A.vel[j3];                    // entry k + 2
            r3 = A.rank[j4]; j3 = j4;                              // entry k + 3
            j4 = idx[first + min(k + 4, last) * stride];           // entry k + 4
            irr_term(A, pi, vi, cur, S);
        }
    }
}

// pv[j] = { x, y, z, m ; vx, vy, vz, - } of particle j, ORIGINAL order: coalesced reads of rank and vel, one gather
// of the sorted bodies, coalesced 32-byte writes
__global__ void __launch_bounds__(256) k_irr_pack(const float4* __restrict__ spm, const int32_t* __restrict__ rank,
                                                  const float4* __restrict__ vel, int n, float4* __restrict__ pv)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) { pv[2 * (size_t)j] = spm[rank[j]]; pv[2 * (size_t)j + 1] = vel[j]; }
}

template <bool PV>
__global__ void __launch_bounds__(256) k_irregular(irr_args A)
{
    // threads take the particles in Morton order: the rows of a warp are neighbours in space, so they
    // have similar lengths and share most of their entries (L1 hits on spm / vel / rank)
    const int sp = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    long long b = 0; int len = 0, i = 0;
    float4 pi = make_float4(0, 0, 0, 0), vi = pi;
    if (sp < A.n) { i = (int)A.order[sp]; b = A.nboff[i]; len = (int)(A.nboff[i + 1] - b); pi = A.spm[sp]; vi = A.vel[i]; }
    irr_sum S = { 0, 0, 0, 0, 0, 0, 0 };
    if (len <= 32) irr_row<PV>(A, pi, vi, A.nbidx + b, 0, len, 1, S);
    // Rows longer than a warp.  33 .. 256 entries: four rows at a time, eight lanes each -- a row of ~100 entries
    // gives a lane a dozen iterations, enough for the staged loads of irr_row to pay (with 32 lanes per row most of
    // the time went into the exposed first loads of every row).  Longer rows: all 32 lanes share the row.
    // Partial sums are reduced by shuffles in a fixed order.
    uint32_t m = __ballot_sync(0xffffffffu, len > 32 && len <= 256);
    const int grp = lane >> 3, sub = lane & 7;
    while (m) {
        // the grp-th set bit of m is this group's row (none: the group idles this round)
        uint32_t mm = m;
        for (int q = 0; q < grp; ++q) mm &= mm - 1;
        const int src = mm ? __ffs(mm) - 1 : -1;
        const int from = src < 0 ? lane : src;
        const long long rb = __shfl_sync(0xffffffffu, b, from);
        int rl = __shfl_sync(0xffffffffu, len, from);
        if (src < 0) rl = 0;
        float4 p, v;
        p.x = __shfl_sync(0xffffffffu, pi.x, from); p.y = __shfl_sync(0xffffffffu, pi.y, from);
        p.z = __shfl_sync(0xffffffffu, pi.z, from); p.w = 0.0f;
        v.x = __shfl_sync(0xffffffffu, vi.x, from); v.y = __shfl_sync(0xffffffffu, vi.y, from);
        v.z = __shfl_sync(0xffffffffu, vi.z, from); v.w = 0.0f;
        irr_sum R = { 0, 0, 0, 0, 0, 0, 0 };
        irr_row<PV>(A, p, v, A.nbidx + rb, sub, (rl - sub + 7) >> 3, 8, R);
        // which group worked on MY row (if it was one of this round's four)
        const int rank_in_m = __popc(m & ((1u << lane) - 1u));
        const bool mine = ((m >> lane) & 1u) && rank_in_m < 4;
        double* r = &R.ax;
#pragma unroll
        for (int c = 0; c < 7; ++c) {
#pragma unroll
            for (int o = 4; o > 0; o >>= 1) {
                int lo = __double2loint(r[c]), hi = __double2hiint(r[c]);
                lo = __shfl_xor_sync(0xffffffffu, lo, o); hi = __shfl_xor_sync(0xffffffffu, hi, o);
                r[c] += __hiloint2double(hi, lo);
            }
            int lo = __double2loint(r[c]), hi = __double2hiint(r[c]);
            lo = __shfl_sync(0xffffffffu, lo, mine ? 8 * rank_in_m : lane); hi = __shfl_sync(0xffffffffu, hi, mine ? 8 * rank_in_m : lane);
            if (mine) (&S.ax)[c] = __hiloint2double(hi, lo);
        }
        for (int q = 0; q < 4 && m; ++q) m &= m - 1;
    }
    m = __ballot_sync(0xffffffffu, len > 256);
    while (m) {
        const int src = __ffs(m) - 1; m &= m - 1;
        const long long rb = __shfl_sync(0xffffffffu, b, src);
        const int rl = __shfl_sync(0xffffffffu, len, src);
        float4 p, v;
        p.x = __shfl_sync(0xffffffffu, pi.x, src); p.y = __shfl_sync(0xffffffffu, pi.y, src);
        p.z = __shfl_sync(0xffffffffu, pi.z, src); p.w = 0.0f;
        v.x = __shfl_sync(0xffffffffu, vi.x, src); v.y = __shfl_sync(0xffffffffu, vi.y, src);
        v.z = __shfl_sync(0xffffffffu, vi.z, src); v.w = 0.0f;
        irr_sum R = { 0, 0, 0, 0, 0, 0, 0 };
        irr_row<PV>(A, p, v, A.nbidx + rb, lane, (rl - lane + 31) >> 5, 32, R);
        double* r = &R.ax;
#pragma unroll
        for (int c = 0; c < 7; ++c)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                int lo = __double2loint(r[c]), hi = __double2hiint(r[c]);
                lo = __shfl_xor_sync(0xffffffffu, lo, o); hi = __shfl_xor_sync(0xffffffffu, hi, o);
                r[c] += __hiloint2double(hi, lo);
            }
        if (lane == src) S = R;
    }
    if (sp < A.n) {
        A.acc[i]  = make_float4((float)S.ax, (float)S.ay, (float)S.az, (float)S.ph);
        A.jerk[i] = make_float4((float)S.jx, (float)S.jy, (float)S.jz, 0.0f);
    }
}

int p3t_launch_irregular(p3t_ctx* ctx, const float4* vel, float4* acc, float4* jerk)
{
    irr_args A;
    A.spm = P<float4>(ctx->spm); A.rank = P<int32_t>(ctx->rank); A.order = P<uint32_t>(ctx->idx[0]);
    A.vel = vel; A.nboff = P<int64_t>(ctx->nboff); A.nbidx = P<int32_t>(ctx->nbidx);
    A.acc = acc; A.jerk = jerk; A.n = (int)ctx->n;
    make_consts(A.K, ctx->r_out, ctx->r_in, ctx->theta, 0);
    if (!ctx->psitab.p || ctx->psitab_rout != ctx->r_out || ctx->psitab_rin != ctx->r_in) {
        int rc = p3t_reserve(ctx, &ctx->psitab, sizeof(ctx->psitab_host));
        if (rc) return rc;
        const walk_consts& K = A.K;
        double I[PSI_TAB + 1], dI[PSI_TAB + 1];
        for (int k = 0; k <= PSI_TAB; ++k) {
            const double x = (double)k / PSI_TAB;
            const double sx = x * (K.dsc[0] + x * (K.dsc[1] + x * (K.dsc[2] + x * (K.dsc[3] + x * (K.dsc[4] + x * K.dsc[5])))));
            // r_in = 0 (c = 0): the remainder term is exactly 0, and t^3 / (t + c) = t^2 also at t = 0
            I[k] = k == PSI_TAB ? 0.0 : (K.ds1 - sx) - (K.drem > 0.0 ? K.drem * (K.dlog1c - log(x + K.dc)) : 0.0);
            dI[k] = -(x + K.dc > 0.0 ? x * x * x / (x + K.dc) : 0.0) * (1.0 - x) * (1.0 - x) * (1.0 - x) / PSI_TAB;
        }
        float* h = ctx->psitab_host;
        for (int k = 0; k < PSI_TAB; ++k) {
            const float hi = (float)I[k];
            h[8 * k + 0] = hi; h[8 * k + 1] = (float)(I[k] - (double)hi); h[8 * k + 2] = (float)dI[k]; h[8 * k + 3] = (float)(I[k + 1] - I[k]);
            h[8 * k + 4] = (float)dI[k + 1]; h[8 * k + 5] = h[8 * k + 6] = h[8 * k + 7] = 0.0f;
        }
        P3T_CUDA(ctx, cudaMemcpyAsync(ctx->psitab.p, h, sizeof(ctx->psitab_host), cudaMemcpyHostToDevice, ctx->stream));
        P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));    // the host copy may be rewritten by the next call
        ctx->psitab_rout = ctx->r_out; ctx->psitab_rin = ctx->r_in;
    }
    A.psitab = P<float4>(ctx->psitab);
    // lists with four or more entries per particle: one pass packs position and velocity into 32-byte records
    const bool pv = ctx->nb_total_host >= 4 * ctx->n;
    A.pv = nullptr;
    if (pv) {
        int rc = p3t_reserve(ctx, &ctx->irrpv, (size_t)A.n * 32);
        if (rc) return rc;
        A.pv = P<float4>(ctx->irrpv);
    }
    P3T_CUDA(ctx, cudaEventRecord(ctx->evi[0], ctx->stream));
    if (pv) {
        k_irr_pack<<<(A.n + 255) / 256, 256, 0, ctx->stream>>>(A.spm, A.rank, vel, A.n, P<float4>(ctx->irrpv));
        k_irregular<true><<<(A.n + 255) / 256, 256, 0, ctx->stream>>>(A);
        ctx->launches += 1;
    } else {
        k_irregular<false><<<(A.n + 255) / 256, 256, 0, ctx->stream>>>(A);
    }
    P3T_CUDA(ctx, cudaGetLastError());
    P3T_CUDA(ctx, cudaEventRecord(ctx->evi[1], ctx->stream));
    ctx->launches += 1;
    return P3T_OK;
}
