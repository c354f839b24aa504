// p3t_shard.cu -- SURVEY.md 8e / 8f NEXT-4: the regular-force path split among the GPUs of a node.
// PAPER.md:277-291 names multi-GPU as future work; the path shards by TARGET GROUP with no data-path
// collective: every rank holds all bodies and builds the identical tree (the build is deterministic,
// 0.5 ms at N = 2^20: cheaper than exchanging it), walks the groups of one contiguous Morton range,
// and the ranks then exchange 16 B per particle of results (one all-gather, done by the caller with
// NCCL; paper_2110_11658_b200.shard).
//
// Cuts: rank r owns the groups whose first sorted particle lies in [cut_r, cut_{r+1}), where cut_r
// is the first group boundary at or after a nominal position -- r n / nranks, or the caller's own
// positions (cost-balanced from the previous step's list lengths).  Every rank computes all cuts, so
// that it can place the chunks it receives.
#include "p3t_internal.cuh"
#include <stdio.h>

__global__ void k_shard_range(const int32_t* __restrict__ gbegin, p3t_devinfo* info, const long long* __restrict__ nominal,
                              int rank, int nranks, int n, int32_t* __restrict__ cuts)
{
    const int r = threadIdx.x;
    if (r > nranks) return;
    const int ng = info->n_groups;
    long long c = nominal ? nominal[r] : (long long)r * n / nranks;
    if (r == 0) c = 0;
    if (r == nranks || c > n) c = n;
    if (c < 0) c = 0;
    int lo = 0, hi = ng;                                   // smallest g with gbegin[g] >= c (gbegin[ng] = n)
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (gbegin[mid] >= c) hi = mid; else lo = mid + 1; }
    cuts[r] = lo;
    cuts[nranks + 1 + r] = gbegin[lo];
    if (r == rank)     info->shard_g0 = lo;
    if (r == rank + 1) info->shard_g1 = lo;
}

// caller's cuts that are not ascending would give a rank a negative range: made monotone here
__global__ void k_shard_monotone(p3t_devinfo* info, int rank, int nranks, int32_t* __restrict__ cuts)
{
    if (threadIdx.x != 0) return;
    for (int r = 1; r <= nranks; ++r)
        if (cuts[r] < cuts[r - 1]) { cuts[r] = cuts[r - 1]; cuts[nranks + 1 + r] = cuts[nranks + 1 + r - 1]; }
    info->shard_g0 = cuts[rank]; info->shard_g1 = cuts[rank + 1];
}

int p3t_launch_shard_range(p3t_ctx* ctx)
{
    const int nr = ctx->shard_nranks;
    int rc;
    if ((rc = p3t_reserve(ctx, &ctx->shard_cuts, (size_t)2 * (nr + 1) * sizeof(int32_t)))) return rc;
    k_shard_range<<<1, 1024, 0, ctx->stream>>>(P<int32_t>(ctx->gbegin), INFO(ctx),
                                               ctx->shard_has_nominal ? P<long long>(ctx->shard_nominal) : nullptr,
                                               ctx->shard_rank, nr, (int)ctx->n, P<int32_t>(ctx->shard_cuts));
    if (ctx->shard_has_nominal) { k_shard_monotone<<<1, 32, 0, ctx->stream>>>(INFO(ctx), ctx->shard_rank, nr, P<int32_t>(ctx->shard_cuts)); ctx->launches += 1; }
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
    return P3T_OK;
}

// results of the owned particles, original order -> one contiguous chunk in sorted order, and back
__global__ void __launch_bounds__(256) k_shard_pack(const float4* __restrict__ src, const uint32_t* __restrict__ order,
                                                    const int32_t* __restrict__ cuts, int nranks, int rank, float4* __restrict__ dst)
{
    const int s0 = cuts[nranks + 1 + rank], s1 = cuts[nranks + 1 + rank + 1];
    for (int s = s0 + blockIdx.x * blockDim.x + threadIdx.x; s < s1; s += gridDim.x * blockDim.x) dst[s - s0] = src[order[s]];
}

__global__ void __launch_bounds__(256) k_shard_unpack(const float4* __restrict__ src, const uint32_t* __restrict__ order,
                                                      const int32_t* __restrict__ cuts, int nranks, int rank, float4* __restrict__ dst)
{
    const int s0 = cuts[nranks + 1 + rank], s1 = cuts[nranks + 1 + rank + 1];
    for (int s = s0 + blockIdx.x * blockDim.x + threadIdx.x; s < s1; s += gridDim.x * blockDim.x) dst[order[s]] = src[s - s0];
}

static int shard_ready(p3t_ctx* c)
{
    if (!c) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 1) { snprintf(c->err, sizeof(c->err), "shard call before p3t_build_tree"); return P3T_ESTATE; }
    if (c->shard_nranks < 2) { snprintf(c->err, sizeof(c->err), "context is not sharded (p3t_set_shard)"); return P3T_ESTATE; }
    return P3T_OK;
}

extern "C" int p3t_get_shard_cuts(p3t_ctx* c, int64_t* cuts_host, int32_t* group_cuts_host)
{
    int rc = shard_ready(c);
    if (rc) return rc;
    if (!cuts_host) return P3T_EINVAL;
    const int nr = c->shard_nranks;
    int32_t tmp[2 * (P3T_MAX_RANKS + 1)];
    P3T_CUDA(c, cudaSetDevice(c->device));
    P3T_CUDA(c, cudaMemcpyAsync(tmp, c->shard_cuts.p, (size_t)2 * (nr + 1) * 4, cudaMemcpyDeviceToHost, c->stream));
    P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int r = 0; r <= nr; ++r) { cuts_host[r] = tmp[nr + 1 + r]; if (group_cuts_host) group_cuts_host[r] = tmp[r]; }
    return P3T_OK;
}

extern "C" int p3t_shard_pack(p3t_ctx* c, const void* acc_pot, void* chunk)
{
    int rc = shard_ready(c);
    if (rc) return rc;
    if (!acc_pot || !chunk || (((uintptr_t)acc_pot | (uintptr_t)chunk) & 15u)) return P3T_EINVAL;
    P3T_CUDA(c, cudaSetDevice(c->device));
    const int blocks = (int)((c->n / c->shard_nranks + 255) / 256) + 1;
    k_shard_pack<<<blocks, 256, 0, c->stream>>>((const float4*)acc_pot, P<uint32_t>(c->idx[0]), P<int32_t>(c->shard_cuts),
                                               c->shard_nranks, c->shard_rank, (float4*)chunk);
    P3T_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return P3T_OK;
}

extern "C" int p3t_shard_unpack(p3t_ctx* c, int from_rank, const void* chunk, void* acc_pot)
{
    int rc = shard_ready(c);
    if (rc) return rc;
    if (!acc_pot || !chunk || (((uintptr_t)acc_pot | (uintptr_t)chunk) & 15u)) return P3T_EINVAL;
    if (from_rank < 0 || from_rank >= c->shard_nranks) return P3T_EINVAL;
    P3T_CUDA(c, cudaSetDevice(c->device));
    const int blocks = (int)((c->n / c->shard_nranks + 255) / 256) + 1;
    k_shard_unpack<<<blocks, 256, 0, c->stream>>>((const float4*)chunk, P<uint32_t>(c->idx[0]), P<int32_t>(c->shard_cuts),
                                                 c->shard_nranks, from_rank, (float4*)acc_pot);
    P3T_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return P3T_OK;
}
