// p3t_sort.cu -- steps a1-a3 of the hot path: bounding cube, Morton keys,
// stable LSD radix sort of (key, index), body permutation.  Rules: DESIGN.md R-S1..R-S3.
// The paper gives no detail of this stage ("the BONSAI library").
#include "p3t_internal.cuh"

// ---------------------------------------------------------------------------------------------
// a1  bounding cube (R-S1): lo_a = min x_a, ext = max_a fl32(hi_a - lo_a), side = 2^e, ext = f 2^e
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t f2ord(float f)      // order-preserving float -> uint
{
    uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t u)
{
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

__global__ void __launch_bounds__(256) k_cube(const float4* __restrict__ pm, int n, p3t_devinfo* info)
{
    float lo[3] = { INFINITY, INFINITY, INFINITY }, hi[3] = { -INFINITY, -INFINITY, -INFINITY };
    int bad = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float4 p = __ldg(pm + i);
        float v[3] = { p.x + 0.0f, p.y + 0.0f, p.z + 0.0f };              // -0 -> +0
        // finite test: |v| <= FLT_MAX is false for NaN and Inf
        // a negative mass is rejected too (cell masses could cancel); zero masses (tracers) are legal: R-S6a
        bad |= !(fabsf(p.x) <= 3.402823466e38f) | !(fabsf(p.y) <= 3.402823466e38f) |
               !(fabsf(p.z) <= 3.402823466e38f) | !(p.w >= 0.0f && p.w <= 3.402823466e38f);
#pragma unroll
        for (int a = 0; a < 3; ++a) { lo[a] = fminf(lo[a], v[a]); hi[a] = fmaxf(hi[a], v[a]); }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    __shared__ float s_lo[8][3], s_hi[8][3];
    __shared__ int s_bad[8];
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) {
        for (int a = 0; a < 3; ++a) { s_lo[w][a] = lo[a]; s_hi[w][a] = hi[a]; }
        s_bad[w] = bad;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) {
            for (int a = 0; a < 3; ++a) { lo[a] = fminf(lo[a], s_lo[k][a]); hi[a] = fmaxf(hi[a], s_hi[k][a]); }
            bad |= s_bad[k];
        }
        // minima are stored complemented so that one zero-initialised atomicMax serves all six
        for (int a = 0; a < 3; ++a) {
            atomicMax(&info->minmax[a], ~f2ord(lo[a]));
            atomicMax(&info->minmax[3 + a], f2ord(hi[a]));
        }
        if (bad) atomicOr(&info->bad_input, 1);
    }
}

// ---------------------------------------------------------------------------------------------
// a2  Morton keys (R-S2): g_a = min(2^B - 1, trunc(fl32(fl32(x_a - lo_a) * scale))), x highest
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t spread3(uint32_t v)   // bit k of v -> bit 3k (21 bits)
{
    uint64_t x = v & 0x1fffffu;
    x = (x | (x << 32)) & 0x001f00000000ffffull;
    x = (x | (x << 16)) & 0x001f0000ff0000ffull;
    x = (x | (x << 8))  & 0x100f00f00f00f00full;
    x = (x | (x << 4))  & 0x10c30c30c30c30c3ull;
    x = (x | (x << 2))  & 0x1249249249249249ull;
    return x;
}

__global__ void __launch_bounds__(256) k_keys(const float4* __restrict__ pm, int n, int B,
                                              p3t_devinfo* info, uint64_t* __restrict__ keys)
{
    float lo[3], ext = 0.0f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        lo[a] = ord2f(~info->minmax[a]);
        float hi = ord2f(info->minmax[3 + a]);
        ext = fmaxf(ext, __fsub_rn(hi, lo[a]));
    }
    float side = 1.0f;
    if (ext > 0.0f && ext <= 3.402823466e38f) { int e; (void)frexpf(ext, &e); side = ldexpf(1.0f, e); }
    const float scale = __fdiv_rn(ldexpf(1.0f, B), side);          // a power of two: exact
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        info->lo[0] = lo[0]; info->lo[1] = lo[1]; info->lo[2] = lo[2];
        info->side = side; info->scale = scale;
    }
    const uint32_t gmax = (1u << B) - 1u;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float4 p = __ldg(pm + i);
        uint32_t gx = min(gmax, __float2uint_rz(__fmul_rn(__fsub_rn(p.x, lo[0]), scale)));
        uint32_t gy = min(gmax, __float2uint_rz(__fmul_rn(__fsub_rn(p.y, lo[1]), scale)));
        uint32_t gz = min(gmax, __float2uint_rz(__fmul_rn(__fsub_rn(p.z, lo[2]), scale)));
        keys[i] = (spread3(gx) << 2) | (spread3(gy) << 1) | spread3(gz);
    }
}

// ---------------------------------------------------------------------------------------------
// a3  stable LSD radix sort (R-S3), 8-bit digits, three kernels per pass:
//     k_hist   per-tile digit counts            -> hist[digit][tile]
//     k_scan   exclusive scan of every digit row, row totals
//     k_scatter stable ranking inside the tile (warp match + per-warp counters) and scatter
// ---------------------------------------------------------------------------------------------
template <int ITEMS>
__global__ void __launch_bounds__(P3T_SORT_THREADS) k_hist(const uint64_t* __restrict__ keys, int n, int shift,
                                                           uint32_t* __restrict__ hist, int ntiles)
{
    __shared__ uint32_t h[P3T_RADIX];
    h[threadIdx.x] = 0;
    __syncthreads();
    const int base = blockIdx.x * (P3T_SORT_THREADS * ITEMS);
#pragma unroll 4
    for (int k = 0; k < ITEMS; ++k) {
        int i = base + k * P3T_SORT_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&h[(uint32_t)(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * ntiles + blockIdx.x] = h[threadIdx.x];
}

// one warp per digit row: in-place exclusive scan over the tiles, total -> totals[digit]
__global__ void __launch_bounds__(256) k_scan_rows(uint32_t* __restrict__ hist, int ntiles, uint32_t* __restrict__ totals)
{
    const int d = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    uint32_t* row = hist + (size_t)d * ntiles;
    uint32_t run = 0;
    for (int b0 = 0; b0 < ntiles; b0 += 32) {
        int b = b0 + lane;
        uint32_t v = b < ntiles ? row[b] : 0u, x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (b < ntiles) row[b] = run + x - v;
        run += __shfl_sync(0xffffffffu, x, 31);
    }
    if (lane == 0) totals[d] = run;
}

template <bool FIRST, int ITEMS>
__global__ void __launch_bounds__(P3T_SORT_THREADS) k_scatter(const uint64_t* __restrict__ kin, const uint32_t* __restrict__ vin,
                                                              uint64_t* __restrict__ kout, uint32_t* __restrict__ vout,
                                                              int n, int shift, const uint32_t* __restrict__ hist, int ntiles,
                                                              const uint32_t* __restrict__ totals)
{
    __shared__ uint32_t cnt[8][P3T_RADIX];
    __shared__ uint32_t s_scan[P3T_RADIX];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int k = 0; k < 8; ++k) cnt[k][threadIdx.x] = 0;
    // digit bases: exclusive scan of the 256 row totals
    {
        uint32_t v = totals[threadIdx.x], x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        s_scan[threadIdx.x] = x;                       // inclusive inside the warp
        __syncthreads();
        uint32_t add = 0;
        for (int k = 0; k < w; ++k) add += s_scan[k * 32 + 31];
        __syncthreads();
        s_scan[threadIdx.x] = add + x - v + hist[(size_t)threadIdx.x * ntiles + blockIdx.x];
    }
    __syncthreads();
    const int base = blockIdx.x * (P3T_SORT_THREADS * ITEMS) + w * (32 * ITEMS);
    uint64_t key[ITEMS];
    uint32_t rank[ITEMS];
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int i = base + r * 32 + lane;
        key[r] = i < n ? kin[i] : ~0ull;
    }
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int i = base + r * 32 + lane;
        uint32_t d = i < n ? ((uint32_t)(key[r] >> shift) & 255u) : 256u;
        uint32_t peers = __match_any_sync(0xffffffffu, d);
        int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (lane == leader && d < 256u) { old = cnt[w][d]; cnt[w][d] = old + __popc(peers); }
        old = __shfl_sync(0xffffffffu, old, leader);
        rank[r] = old + __popc(peers & lt);
        __syncwarp();
    }
    __syncthreads();
    {   // per digit: exclusive scan over the 8 warps, plus the tile's global offset
        uint32_t run = s_scan[threadIdx.x];
#pragma unroll
        for (int k = 0; k < 8; ++k) { uint32_t t = cnt[k][threadIdx.x]; cnt[k][threadIdx.x] = run; run += t; }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int i = base + r * 32 + lane;
        if (i < n) {
            uint32_t d = (uint32_t)(key[r] >> shift) & 255u;
            uint32_t pos = cnt[w][d] + rank[r];
            kout[pos] = key[r];
            vout[pos] = FIRST ? (uint32_t)i : vin[i];
        }
    }
}

__global__ void __launch_bounds__(256) k_permute(const float4* __restrict__ pm, const uint32_t* __restrict__ order,
                                                 int n, float4* __restrict__ spm, int32_t* __restrict__ rank)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { const uint32_t o = order[i]; spm[i] = __ldg(pm + o); rank[o] = i; }    // rank: original id -> sorted position
}

// ---------------------------------------------------------------------------------------------
int p3t_launch_cube_keys(p3t_ctx* ctx, const float4* pm)
{
    const int n = (int)ctx->n;
    int blocks = (n + 255) / 256;
    int cap = ctx->num_sms * 8;
    if (blocks > cap) blocks = cap;
    k_cube<<<blocks, 256, 0, ctx->stream>>>(pm, n, INFO(ctx));
    k_keys<<<blocks, 256, 0, ctx->stream>>>(pm, n, ctx->bits, INFO(ctx), P<uint64_t>(ctx->keys[0]));
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 2;
    return P3T_OK;
}

// Tiles of 2048 keys (8 per thread); 1024 below 2^18 particles, where the shorter serial chain of a block and
// the larger grid matter more than the size of the histogram (measured: sort 0.19 -> 0.12 ms at N = 2^14).
template <int ITEMS>
static int sort_passes(p3t_ctx* ctx)
{
    const int n = (int)ctx->n;
    const int tile = P3T_SORT_THREADS * ITEMS;
    const int ntiles = (n + tile - 1) / tile;
    const int passes = (3 * ctx->bits + P3T_RADIX_BITS - 1) / P3T_RADIX_BITS;     // 8 (63-bit) or 4 (30-bit)
    uint32_t* hist = P<uint32_t>(ctx->hist);
    uint32_t* totals = hist + (size_t)P3T_RADIX * ntiles;
    int cur = 0;
    for (int p = 0; p < passes; ++p) {
        const int shift = p * P3T_RADIX_BITS;
        uint64_t* kin = P<uint64_t>(ctx->keys[cur]);  uint64_t* kout = P<uint64_t>(ctx->keys[cur ^ 1]);
        uint32_t* vin = P<uint32_t>(ctx->idx[cur]);   uint32_t* vout = P<uint32_t>(ctx->idx[cur ^ 1]);
        k_hist<ITEMS><<<ntiles, P3T_SORT_THREADS, 0, ctx->stream>>>(kin, n, shift, hist, ntiles);
        k_scan_rows<<<P3T_RADIX / 8, 256, 0, ctx->stream>>>(hist, ntiles, totals);
        if (p == 0) k_scatter<true, ITEMS><<<ntiles, P3T_SORT_THREADS, 0, ctx->stream>>>(kin, vin, kout, vout, n, shift, hist, ntiles, totals);
        else        k_scatter<false, ITEMS><<<ntiles, P3T_SORT_THREADS, 0, ctx->stream>>>(kin, vin, kout, vout, n, shift, hist, ntiles, totals);
        cur ^= 1;
        ctx->launches += 3;
    }
    P3T_CUDA(ctx, cudaGetLastError());
    // an even number of passes leaves the result in buffer 0
    if (cur != 0) {
        p3t_buf t = ctx->keys[0]; ctx->keys[0] = ctx->keys[1]; ctx->keys[1] = t;
        t = ctx->idx[0]; ctx->idx[0] = ctx->idx[1]; ctx->idx[1] = t;
    }
    return P3T_OK;
}

int p3t_launch_sort(p3t_ctx* ctx)
{
    return ctx->n <= (1 << 18) ? sort_passes<P3T_SORT_ITEMS_MIN>(ctx) : sort_passes<8>(ctx);
}

int p3t_launch_permute(p3t_ctx* ctx, const float4* pm)
{
    const int n = (int)ctx->n;
    k_permute<<<(n + 255) / 256, 256, 0, ctx->stream>>>(pm, P<uint32_t>(ctx->idx[0]), n, P<float4>(ctx->spm), P<int32_t>(ctx->rank));
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
    return P3T_OK;
}
