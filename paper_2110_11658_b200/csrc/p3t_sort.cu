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

// k_keys also counts, for every radix pass, how many keys carry each digit (one read of the particles serves the
// keys and all the histograms of the sort below)
#define SORT_MAX_PASSES 8
__global__ void __launch_bounds__(256) k_keys(const float4* __restrict__ pm, int n, int B, int passes,
                                              p3t_devinfo* info, uint64_t* __restrict__ keys, uint32_t* __restrict__ ghist)
{
    __shared__ uint32_t s_hist[SORT_MAX_PASSES][P3T_RADIX];
    for (int k = 0; k < passes; ++k) s_hist[k][threadIdx.x] = 0;
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
    __syncthreads();
    const uint32_t gmax = (1u << B) - 1u;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float4 p = __ldg(pm + i);
        uint32_t gx = min(gmax, __float2uint_rz(__fmul_rn(__fsub_rn(p.x, lo[0]), scale)));
        uint32_t gy = min(gmax, __float2uint_rz(__fmul_rn(__fsub_rn(p.y, lo[1]), scale)));
        uint32_t gz = min(gmax, __float2uint_rz(__fmul_rn(__fsub_rn(p.z, lo[2]), scale)));
        const uint64_t key = (spread3(gx) << 2) | (spread3(gy) << 1) | spread3(gz);
        keys[i] = key;
        for (int k = 0; k < passes; ++k) atomicAdd(&s_hist[k][(uint32_t)(key >> (k * P3T_RADIX_BITS)) & 255u], 1u);
    }
    __syncthreads();
    for (int k = 0; k < passes; ++k) {
        const uint32_t c = s_hist[k][threadIdx.x];
        if (c) atomicAdd(&ghist[k * P3T_RADIX + threadIdx.x], c);
    }
}

// ---------------------------------------------------------------------------------------------
// a3  stable LSD radix sort (R-S3), 8-bit digits, ONE kernel per pass ("onesweep"): the digit totals of every pass are
//     known from k_keys, so a tile only needs the number of equal digits in the tiles before it.  Tiles take their
//     number from a ticket counter (a tile with a smaller number is always already running), rank their keys
//     (warp match + per-warp counters: stable), publish their 256 digit counts in one 64-bit word each
//     (flag | count) and look back over the earlier tiles' words until they meet an inclusive prefix
//     (decoupled look-back), publish their own inclusive prefix, and scatter.
//     status word: high half = 2 pass + 1 (count of this tile) or 2 pass + 2 (inclusive prefix), low half = value;
//     words of earlier passes have smaller flags, so the array is cleared once per sort, not per pass.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p)
{
    unsigned long long v; asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ void st_relaxed_u64(unsigned long long* p, unsigned long long v)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}

template <bool FIRST, int ITEMS>
__global__ void __launch_bounds__(P3T_SORT_THREADS) k_sort_pass(const uint64_t* __restrict__ kin, const uint32_t* __restrict__ vin,
                                                                uint64_t* __restrict__ kout, uint32_t* __restrict__ vout,
                                                                int n, int pass, const uint32_t* __restrict__ ghist,
                                                                unsigned long long* status, uint32_t* ticket)
{
    constexpr int TILE_KEYS = P3T_SORT_THREADS * ITEMS;
    __shared__ uint32_t cnt[8][P3T_RADIX];
    __shared__ uint32_t s_gbase[P3T_RADIX];          // where the tile's keys of digit d begin in the output
    __shared__ uint32_t s_lbase[P3T_RADIX];          // ... and in the tile's own sorted order
    __shared__ uint32_t s_wsum[8];
    __shared__ int s_tile;
    __shared__ uint64_t s_buf[TILE_KEYS];            // the tile in sorted order: keys, then (same space) values
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31, shift = pass * P3T_RADIX_BITS;
    if (threadIdx.x == 0) s_tile = (int)atomicAdd(&ticket[pass], 1u);
    for (int k = 0; k < 8; ++k) cnt[k][threadIdx.x] = 0;
    const uint32_t v_tot = ghist[pass * P3T_RADIX + threadIdx.x];
    __syncthreads();
    // all the tile's keys are requested before anything waits (the barrier below keeps the loads from sinking into
    // the ranking rounds, where each round would wait for its own load)
    const int tile = s_tile;
    const int base = tile * TILE_KEYS + w * (32 * ITEMS);
    uint64_t key[ITEMS];
    uint16_t rank[ITEMS];
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int i = base + r * 32 + lane;
        key[r] = i < n ? __ldcs(kin + i) : ~0ull;
    }
    // digit bases: exclusive scan of the 256 digit totals of this pass
    uint32_t dbase;
    {
        uint32_t v = v_tot, x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) s_wsum[w] = x;
        __syncthreads();
        uint32_t add = 0;
        for (int k = 0; k < w; ++k) add += s_wsum[k];
        dbase = add + x - v;
    }
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int i = base + r * 32 + lane;
        uint32_t d = i < n ? ((uint32_t)(key[r] >> shift) & 255u) : 256u;
        // lanes with the same digit: nine ballots, one per bit (match.any costs a round per distinct value in the warp)
        uint32_t peers = 0xffffffffu;
#pragma unroll
        for (int b = 0; b < 9; ++b) {
            const uint32_t m = __ballot_sync(0xffffffffu, (d >> b) & 1u);
            peers &= ((d >> b) & 1u) ? m : ~m;
        }
        int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (lane == leader && d < 256u) { old = cnt[w][d]; cnt[w][d] = old + __popc(peers); }
        old = __shfl_sync(0xffffffffu, old, leader);
        rank[r] = (uint16_t)(old + __popc(peers & lt));
        __syncwarp();
    }
    __syncthreads();
    {   // thread = digit: exclusive scan over the 8 warps, the tile's count, look-back over the earlier tiles
        uint32_t run = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) { uint32_t t = cnt[k][threadIdx.x]; cnt[k][threadIdx.x] = run; run += t; }
        const unsigned long long f_count = (unsigned long long)(2 * pass + 1) << 32, f_prefix = (unsigned long long)(2 * pass + 2) << 32;
        unsigned long long* mine = status + (size_t)tile * P3T_RADIX + threadIdx.x;
        if (tile > 0) st_relaxed_u64(mine, f_count | run);
        // the tile's own digit starts (exclusive scan of its 256 counts) while the earlier tiles publish
        uint32_t x = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        __syncthreads();                                  // s_wsum is free again (everybody has its dbase)
        if (lane == 31) s_wsum[w] = x;
        __syncthreads();
        uint32_t ladd = 0;
        for (int k = 0; k < w; ++k) ladd += s_wsum[k];
        s_lbase[threadIdx.x] = ladd + x - run;
        uint32_t excl = 0;
        if (tile > 0) {
            // look back over the earlier tiles, eight words in flight at a time (one L2 round trip per batch); a word
            // that is not there yet ends the batch and is polled again
            const unsigned long long fmin = (unsigned long long)(2 * pass + 1), fpre = (unsigned long long)(2 * pass + 2);
            int t = tile - 1;
            bool done = false;
            while (!done) {
                unsigned long long sv[8];
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    sv[j] = t - j >= 0 ? ld_relaxed_u64(status + (size_t)(t - j) * P3T_RADIX + threadIdx.x) : (fpre << 32);
                int used = 0;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    if (done || used < j) continue;                         // stopped at an earlier word of this batch
                    if ((sv[j] >> 32) < fmin) continue;                     // not published yet: poll again from here
                    excl += (uint32_t)sv[j];
                    used = j + 1;
                    if ((sv[j] >> 32) == fpre) done = true;
                }
                t -= used;
            }
        }
        st_relaxed_u64(mine, f_prefix | (unsigned long long)(excl + run));
        s_gbase[threadIdx.x] = dbase + excl;
    }
    __syncthreads();
    // The tile goes through shared memory in sorted order, so that a digit's run leaves as consecutive addresses
    // (8 or 16 keys per run on average: full sectors instead of one partial sector per key).
    const int tile_n = min(TILE_KEYS, n - tile * TILE_KEYS);
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int i = base + r * 32 + lane;
        if (i < n) {
            uint32_t d = (uint32_t)(key[r] >> shift) & 255u;
            P3T_CHECK(s_lbase[d] + cnt[w][d] + rank[r] < (uint32_t)tile_n);
            rank[r] = (uint16_t)(s_lbase[d] + cnt[w][d] + rank[r]);        // position in the tile's sorted order
            s_buf[rank[r]] = key[r];
        }
    }
    __syncthreads();
    uint32_t gpos[ITEMS];
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        const int e = r * P3T_SORT_THREADS + threadIdx.x;
        gpos[r] = 0;
        if (e < tile_n) {
            const uint64_t k = s_buf[e];
            const uint32_t d = (uint32_t)(k >> shift) & 255u;
            gpos[r] = s_gbase[d] + ((uint32_t)e - s_lbase[d]);
            P3T_CHECK(gpos[r] < (uint32_t)n);
            kout[gpos[r]] = k;
        }
    }
    __syncthreads();
    uint32_t* s_val = reinterpret_cast<uint32_t*>(s_buf);
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        int i = base + r * 32 + lane;
        if (i < n) s_val[rank[r]] = FIRST ? (uint32_t)i : vin[i];
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        const int e = r * P3T_SORT_THREADS + threadIdx.x;
        if (e < tile_n) vout[gpos[r]] = s_val[e];
    }
}

__global__ void __launch_bounds__(256) k_permute(const float4* __restrict__ pm, const uint32_t* __restrict__ order,
                                                 int n, float4* __restrict__ spm, int32_t* __restrict__ rank)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { const uint32_t o = order[i]; spm[i] = __ldg(pm + o); rank[o] = i; }    // rank: original id -> sorted position
}

// ---------------------------------------------------------------------------------------------
// layout of ctx->hist: digit totals [SORT_MAX_PASSES][256] u32 | tickets [SORT_MAX_PASSES] u32 (+ pad) | status [ntiles][256] u64
static inline size_t sort_status_offset() { return (size_t)SORT_MAX_PASSES * P3T_RADIX * 4 + 64; }
static inline int sort_tile(p3t_ctx* ctx) { return P3T_SORT_THREADS * (ctx->n <= (1 << 18) ? P3T_SORT_ITEMS_MIN : P3T_SORT_ITEMS_BIG); }
size_t p3t_sort_scratch_bytes(int64_t n)
{
    const size_t ntiles = ((size_t)n + P3T_SORT_TILE_MIN - 1) / P3T_SORT_TILE_MIN;
    return sort_status_offset() + ntiles * P3T_RADIX * 8;
}

int p3t_launch_cube_keys(p3t_ctx* ctx, const float4* pm)
{
    const int n = (int)ctx->n;
    int blocks = (n + 255) / 256;
    int cap = ctx->num_sms * 8;
    if (blocks > cap) blocks = cap;
    const int passes = (3 * ctx->bits + P3T_RADIX_BITS - 1) / P3T_RADIX_BITS;     // 8 (63-bit) or 4 (30-bit)
    const int tile = sort_tile(ctx), ntiles = (n + tile - 1) / tile;
    // digit totals, tickets and the look-back words of this sort: one clear
    P3T_CUDA(ctx, cudaMemsetAsync(ctx->hist.p, 0, sort_status_offset() + (size_t)ntiles * P3T_RADIX * 8, ctx->stream));
    k_cube<<<blocks, 256, 0, ctx->stream>>>(pm, n, INFO(ctx));
    k_keys<<<blocks, 256, 0, ctx->stream>>>(pm, n, ctx->bits, passes, INFO(ctx), P<uint64_t>(ctx->keys[0]), P<uint32_t>(ctx->hist));
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 2;
    return P3T_OK;
}

// Tiles of 2048 keys (8 per thread); 1024 below 2^18 particles, where the shorter serial chain of a block and
// the larger grid matter more (measured in round 1: sort 0.19 -> 0.12 ms at N = 2^14).
template <int ITEMS>
static int sort_passes(p3t_ctx* ctx)
{
    const int n = (int)ctx->n;
    const int tile = P3T_SORT_THREADS * ITEMS;
    const int ntiles = (n + tile - 1) / tile;
    const int passes = (3 * ctx->bits + P3T_RADIX_BITS - 1) / P3T_RADIX_BITS;     // 8 (63-bit) or 4 (30-bit)
    uint32_t* ghist = P<uint32_t>(ctx->hist);
    uint32_t* ticket = ghist + SORT_MAX_PASSES * P3T_RADIX;
    unsigned long long* status = (unsigned long long*)((char*)ctx->hist.p + sort_status_offset());
    int cur = 0;
    for (int p = 0; p < passes; ++p) {
        uint64_t* kin = P<uint64_t>(ctx->keys[cur]);  uint64_t* kout = P<uint64_t>(ctx->keys[cur ^ 1]);
        uint32_t* vin = P<uint32_t>(ctx->idx[cur]);   uint32_t* vout = P<uint32_t>(ctx->idx[cur ^ 1]);
        if (p == 0) k_sort_pass<true, ITEMS><<<ntiles, P3T_SORT_THREADS, 0, ctx->stream>>>(kin, vin, kout, vout, n, p, ghist, status, ticket);
        else        k_sort_pass<false, ITEMS><<<ntiles, P3T_SORT_THREADS, 0, ctx->stream>>>(kin, vin, kout, vout, n, p, ghist, status, ticket);
        cur ^= 1;
        ctx->launches += 1;
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
    return ctx->n <= (1 << 18) ? sort_passes<P3T_SORT_ITEMS_MIN>(ctx) : sort_passes<P3T_SORT_ITEMS_BIG>(ctx);
}

int p3t_launch_permute(p3t_ctx* ctx, const float4* pm)
{
    const int n = (int)ctx->n;
    k_permute<<<(n + 255) / 256, 256, 0, ctx->stream>>>(pm, P<uint32_t>(ctx->idx[0]), n, P<float4>(ctx->spm), P<int32_t>(ctx->rank));
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
    return P3T_OK;
}

// ---------------------------------------------------------------------------------------------
// p3t_morton_order_static (include/p3t.h): a1-a3 without a context and without any device allocation, for hosts
// that have given all device memory away (their own arena, a caching allocator), that cannot take the device-wide
// stall of cudaMalloc / cudaFree inside their step loop, or that run under a memory quota.  The kernels are the
// ones above, unchanged; what differs is where their scratch lives: in the fixed array below, which is part of the
// library image and so exists on every device that loads this code, for as long as the process runs.
//
// Layout of the array (all parts 256-byte aligned):
//   [ST_INFO]  p3t_devinfo: the cube's min/max words, bad_input, then lo / side / scale        (must start at zero)
//   [ST_SORT]  digit totals [8][256] u32 | tickets | look-back words [ntiles][256] u64        (must start at zero)
//   [ST_KEYS]  uint64[P3T_STATIC_MAX_N]: second key buffer of the ping-pong                    (fully written before read)
//   [ST_IDX]   uint32[P3T_STATIC_MAX_N]: second index buffer                                   (fully written before read)
// The caller's sorted_keys / order arrays are the first buffers: k_keys writes the unsorted keys there, and the
// number of passes is even (8 or 4), so the last pass lands there again.
// ---------------------------------------------------------------------------------------------
#include <mutex>
#include <stddef.h>

static constexpr size_t st_round(size_t b) { return (b + 255) / 256 * 256; }
static constexpr size_t ST_TILES = (P3T_STATIC_MAX_N + P3T_SORT_TILE_MIN - 1) / P3T_SORT_TILE_MIN;
static constexpr size_t ST_INFO = 0;
static constexpr size_t ST_SORT = st_round(sizeof(p3t_devinfo));
static constexpr size_t ST_SORT_HEAD = (size_t)SORT_MAX_PASSES * P3T_RADIX * 4 + 64;       // = sort_status_offset()
static constexpr size_t ST_KEYS = ST_SORT + st_round(ST_SORT_HEAD + ST_TILES * P3T_RADIX * 8);
static constexpr size_t ST_IDX = ST_KEYS + st_round((size_t)P3T_STATIC_MAX_N * 8);
static constexpr size_t ST_BYTES = ST_IDX + st_round((size_t)P3T_STATIC_MAX_N * 4);
static_assert(ST_BYTES == P3T_STATIC_SCRATCH_BYTES, "include/p3t.h states the size of the static scratch array");
static_assert(P3T_STATIC_MAX_N <= (1 << 18), "the static entry point uses the small sort tile only");
static_assert(offsetof(p3t_devinfo, lo) == 0 && offsetof(p3t_devinfo, side) == 12, "cube = the record's first 16 bytes");

// In host code this name is only a handle for cudaGetSymbolAddress; it is not an address a kernel can use.
static __device__ __align__(256) unsigned char g_static_scratch[ST_BYTES];

#define ST_MAX_DEVICES 64
static std::mutex g_static_mutex;
static unsigned char* g_static_ptr[ST_MAX_DEVICES];   // device address of g_static_scratch on each device (0 = not asked yet)
static int g_static_sms[ST_MAX_DEVICES];

// once per device, with that device current; allocates nothing
static int static_setup(int device, unsigned char** base, int* sms)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[device]) {
        void* p = nullptr; int s = 0;
        P3T_CUDA(nullptr, cudaGetSymbolAddress(&p, g_static_scratch));
        P3T_CUDA(nullptr, cudaDeviceGetAttribute(&s, cudaDevAttrMultiProcessorCount, device));
        if (!p || s < 1) return P3T_ECUDA;
        g_static_sms[device] = s;
        g_static_ptr[device] = (unsigned char*)p;
    }
    *base = g_static_ptr[device]; *sms = g_static_sms[device];
    return P3T_OK;
}

extern "C" int p3t_morton_order_static(int device, void* cuda_stream, int64_t n, const float* pos_mass, int key_bits,
                                       uint64_t* sorted_keys, uint32_t* order, float* cube, int32_t* bad_input)
{
    if (!pos_mass || !sorted_keys || !order || n < 1 || (key_bits != 30 && key_bits != 63)) return P3T_EINVAL;
    if (((uintptr_t)pos_mass & 15u) || ((uintptr_t)sorted_keys & 7u) || ((uintptr_t)order & 3u) ||
        ((uintptr_t)cube & 3u) || ((uintptr_t)bad_input & 3u)) return P3T_EINVAL;
    if (device < 0 || device >= ST_MAX_DEVICES) return P3T_EINVAL;
    if (n > P3T_STATIC_MAX_N) return P3T_ELIMIT;                     // the array is sized for P3T_STATIC_MAX_N: refuse, do not overrun
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device >= ndev) { (void)cudaGetLastError(); return P3T_EINVAL; }
    P3T_CUDA(nullptr, cudaSetDevice(device));
    unsigned char* base; int sms, rc;
    if ((rc = static_setup(device, &base, &sms)) != P3T_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int ni = (int)n, bits = key_bits / 3;
    const int passes = (3 * bits + P3T_RADIX_BITS - 1) / P3T_RADIX_BITS;         // 8 or 4: even
    const int ntiles = (ni + P3T_SORT_TILE_MIN - 1) / P3T_SORT_TILE_MIN;
    p3t_devinfo* info = (p3t_devinfo*)(base + ST_INFO);
    uint32_t* ghist = (uint32_t*)(base + ST_SORT);
    uint32_t* ticket = ghist + SORT_MAX_PASSES * P3T_RADIX;
    unsigned long long* status = (unsigned long long*)(base + ST_SORT + ST_SORT_HEAD);
    uint64_t* ktmp = (uint64_t*)(base + ST_KEYS);
    uint32_t* vtmp = (uint32_t*)(base + ST_IDX);
    // what the last call left behind goes: the cube record, the digit totals, the tickets and this call's look-back words
    P3T_CUDA(nullptr, cudaMemsetAsync(base, 0, ST_SORT + ST_SORT_HEAD + (size_t)ntiles * P3T_RADIX * 8, st));
    int blocks = (ni + 255) / 256;
    if (blocks > sms * 8) blocks = sms * 8;
    const float4* pm = (const float4*)pos_mass;
    k_cube<<<blocks, 256, 0, st>>>(pm, ni, info);
    k_keys<<<blocks, 256, 0, st>>>(pm, ni, bits, passes, info, sorted_keys, ghist);
    for (int p = 0; p < passes; ++p) {
        const uint64_t* kin = (p & 1) ? ktmp : sorted_keys;  uint64_t* kout = (p & 1) ? sorted_keys : ktmp;
        const uint32_t* vin = (p & 1) ? vtmp : order;        uint32_t* vout = (p & 1) ? order : vtmp;
        if (p == 0) k_sort_pass<true, P3T_SORT_ITEMS_MIN><<<ntiles, P3T_SORT_THREADS, 0, st>>>(kin, vin, kout, vout, ni, p, ghist, status, ticket);
        else        k_sort_pass<false, P3T_SORT_ITEMS_MIN><<<ntiles, P3T_SORT_THREADS, 0, st>>>(kin, vin, kout, vout, ni, p, ghist, status, ticket);
    }
    P3T_CUDA(nullptr, cudaGetLastError());
    if (cube) P3T_CUDA(nullptr, cudaMemcpyAsync(cube, &info->lo[0], 16, cudaMemcpyDeviceToDevice, st));
    if (bad_input) P3T_CUDA(nullptr, cudaMemcpyAsync(bad_input, &info->bad_input, 4, cudaMemcpyDeviceToDevice, st));
    return P3T_OK;
}
