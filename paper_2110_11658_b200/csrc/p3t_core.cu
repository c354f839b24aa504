// p3t_core.cu -- SURVEY.md 8f NEXT-3: core quantities by a sampled K-nearest-neighbour search
// (PAPER.md:134 section 2.5, :245 section 3.2.1: "a random sample of min(N, sqrt(5000 N)) particles,
// then ... a brute-force search for those particles' 6 nearest neighbours"; estimator: Casertano & Hut
// 1985 as cited there; conventions: DESIGN.md R17-R19).
//
// The paper's brute force is O(ns N); here the search is a K-NN query on the octree that the regular
// force already built: one thread per sample particle, depth-first with the children pushed farthest
// first, pruned by the fp32 distance from the particle to a cell's tight box.  That box distance uses
// the same monotone fp32 operation sequence as the pair distance (R10), so it never exceeds the
// distance to a particle of the cell and the pruning is exact: the neighbours are those of the brute
// force, under the order (fp32 d2, original index).
//   rho_i = (sum of the masses of the K-1 nearest) / (4 pi / 3 r_K^3)                (Casertano & Hut)
//   x_d = sum rho x / sum rho,  R_core^2 = sum rho^2 |x - x_d|^2 / sum rho^2,
//   rho_core = sum rho^2 / sum rho,  N_core = (N / ns) #{ sample : |x - x_d| < R_core }   (NBODY6)
#include "p3t_internal.cuh"
#include <math.h>

#define KNN_KMAX  16
#define KNN_STACK 192                     // <= 7 siblings left behind per level, 21 levels, + 8

struct knn_args {
    const float4* spm; const uint32_t* order; const int32_t* rank;
    const float4 *nlo, *nhi; const int2* nlink;
    const int32_t* sample; int ns, K;
    int32_t* nbr; float* d2k; double* rho;      // outputs (nbr may be NULL)
};

__device__ __forceinline__ float box_d2(const float4 lo, const float4 hi, const float4 p)
{
    const float fx = fmaxf(fmaxf(0.0f, __fsub_rn(lo.x, p.x)), __fsub_rn(p.x, hi.x));
    const float fy = fmaxf(fmaxf(0.0f, __fsub_rn(lo.y, p.y)), __fsub_rn(p.y, hi.y));
    const float fz = fmaxf(fmaxf(0.0f, __fsub_rn(lo.z, p.z)), __fsub_rn(p.z, hi.z));
    return fmaf(fz, fz, fmaf(fy, fy, __fmul_rn(fx, fx)));
}

__global__ void __launch_bounds__(128) k_knn(knn_args A)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= A.ns) return;
    const int K = A.K;
    const int i = A.sample[s], ps = A.rank[i];
    const float4 p = A.spm[ps];
    float bd[KNN_KMAX], bm[KNN_KMAX]; int bj[KNN_KMAX];
    for (int q = 0; q < K; ++q) { bd[q] = INFINITY; bj[q] = 0x7fffffff; bm[q] = 0.0f; }
    int stack[KNN_STACK]; float sb2[KNN_STACK];
    int top = 0;
    stack[top] = 0; sb2[top] = 0.0f; ++top;
    while (top > 0) {
        --top;
        if (sb2[top] > bd[K - 1]) continue;                        // the bound has shrunk since the push
        const int2 link = A.nlink[stack[top]];
        if (link.y < 0) {                                          // leaf: its particles
            for (int j = link.x; j < link.x - link.y; ++j) {
                if (j == ps) continue;                             // self excluded by index
                const float4 q = A.spm[j];
                const float dx = __fsub_rn(q.x, p.x), dy = __fsub_rn(q.y, p.y), dz = __fsub_rn(q.z, p.z);
                const float d2 = fmaf(dz, dz, fmaf(dy, dy, __fmul_rn(dx, dx)));      // R10
                if (d2 > bd[K - 1]) continue;
                const int oj = (int)A.order[j];
                if (d2 == bd[K - 1] && oj > bj[K - 1]) continue;   // ties by the smaller original index
                int w = K - 1;
                while (w > 0 && (d2 < bd[w - 1] || (d2 == bd[w - 1] && oj < bj[w - 1]))) {
                    bd[w] = bd[w - 1]; bj[w] = bj[w - 1]; bm[w] = bm[w - 1]; --w;
                }
                bd[w] = d2; bj[w] = oj; bm[w] = q.w;
            }
        } else {                                                   // internal: children, farthest pushed first
            float cb[8]; int nc = link.y;
            for (int c = 0; c < nc; ++c) cb[c] = box_d2(A.nlo[link.x + c], A.nhi[link.x + c], p);
            for (int r = 0; r < nc; ++r) {
                int best = -1; float bv = -1.0f;
                for (int c = 0; c < nc; ++c) if (cb[c] > bv) { bv = cb[c]; best = c; }
                if (best < 0) break;
                if (bv <= bd[K - 1] && top < KNN_STACK) { stack[top] = link.x + best; sb2[top] = bv; ++top; }
                cb[best] = -2.0f;
            }
        }
    }
    double m = 0.0;
    for (int q = 0; q < K; ++q) {
        if (A.nbr) A.nbr[(size_t)s * K + q] = bd[q] < INFINITY ? bj[q] : -1;
        if (q < K - 1 && bd[q] < INFINITY) m += (double)bm[q];
    }
    const bool full = bd[K - 1] < INFINITY;
    const double rk = full ? sqrt((double)bd[K - 1]) : 0.0;
    A.d2k[s] = bd[K - 1];
    A.rho[s] = rk > 0.0 ? m / (4.0 * M_PI / 3.0 * rk * rk * rk) : 0.0;
}

// ---- reductions over the sample: one block, fp64, fixed order (bit-reproducible) ----
#define CR_THREADS 1024
__device__ double block_sum(double v, double* s_w)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        int lo = __double2loint(v), hi = __double2hiint(v);
        lo = __shfl_xor_sync(0xffffffffu, lo, o); hi = __shfl_xor_sync(0xffffffffu, hi, o);
        v += __hiloint2double(hi, lo);
    }
    __syncthreads();
    if (lane == 0) s_w[w] = v;
    __syncthreads();
    double t = 0.0;
    for (int k = 0; k < CR_THREADS / 32; ++k) t += s_w[k];
    return t;
}

__global__ void __launch_bounds__(CR_THREADS) k_core_reduce(knn_args A, long long n, double* out)
{
    __shared__ double s_w[CR_THREADS / 32];
    double sr = 0, sr2 = 0, cx = 0, cy = 0, cz = 0;
    for (int s = threadIdx.x; s < A.ns; s += CR_THREADS) {
        const float4 p = A.spm[A.rank[A.sample[s]]];
        const double r = A.rho[s];
        sr += r; sr2 += r * r; cx += r * (double)p.x; cy += r * (double)p.y; cz += r * (double)p.z;
    }
    sr = block_sum(sr, s_w); sr2 = block_sum(sr2, s_w);
    cx = block_sum(cx, s_w) / sr; cy = block_sum(cy, s_w) / sr; cz = block_sum(cz, s_w) / sr;
    double q = 0;
    for (int s = threadIdx.x; s < A.ns; s += CR_THREADS) {
        const float4 p = A.spm[A.rank[A.sample[s]]];
        const double dx = (double)p.x - cx, dy = (double)p.y - cy, dz = (double)p.z - cz, r = A.rho[s];
        q += r * r * (dx * dx + dy * dy + dz * dz);
    }
    const double rc = sqrt(block_sum(q, s_w) / sr2);
    double inside = 0;
    for (int s = threadIdx.x; s < A.ns; s += CR_THREADS) {
        const float4 p = A.spm[A.rank[A.sample[s]]];
        const double dx = (double)p.x - cx, dy = (double)p.y - cy, dz = (double)p.z - cz;
        inside += (dx * dx + dy * dy + dz * dz) < rc * rc ? 1.0 : 0.0;
    }
    inside = block_sum(inside, s_w);
    if (threadIdx.x == 0) {
        out[0] = cx; out[1] = cy; out[2] = cz; out[3] = rc; out[4] = sr2 / sr;
        out[5] = inside * (double)n / (double)A.ns;
    }
}

int p3t_launch_core(p3t_ctx* ctx, int64_t ns, const int32_t* sample, int K, int32_t* nbr, float* d2k, double* rho, double* core_dev)
{
    knn_args A;
    A.spm = P<float4>(ctx->spm); A.order = P<uint32_t>(ctx->idx[0]); A.rank = P<int32_t>(ctx->rank);
    A.nlo = P<float4>(ctx->nlo); A.nhi = P<float4>(ctx->nhi); A.nlink = P<int2>(ctx->nlink);
    A.sample = sample; A.ns = (int)ns; A.K = K; A.nbr = nbr; A.d2k = d2k; A.rho = rho;
    P3T_CUDA(ctx, cudaEventRecord(ctx->evc[0], ctx->stream));
    k_knn<<<(unsigned)((ns + 127) / 128), 128, 0, ctx->stream>>>(A);
    k_core_reduce<<<1, CR_THREADS, 0, ctx->stream>>>(A, (long long)ctx->n, core_dev);
    P3T_CUDA(ctx, cudaGetLastError());
    P3T_CUDA(ctx, cudaEventRecord(ctx->evc[1], ctx->stream));
    ctx->launches += 2;
    return P3T_OK;
}
