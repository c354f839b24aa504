// p3t_api.cu -- the C-ABI of include/p3t.h: context, argument checks, buffer management,
// call sequencing, accessors.  All arithmetic of the method lives in p3t_sort/tree/walk.cu.
#include "p3t_internal.cuh"
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>

int p3t_fail_cuda(p3t_ctx* ctx, cudaError_t e, const char* what, int line)
{
    if (ctx) {
        snprintf(ctx->err, sizeof(ctx->err), "%s (%s) at line %d: %s", cudaGetErrorName(e), cudaGetErrorString(e), line, what);
        ctx->sticky = 1;
    }
    return e == cudaErrorMemoryAllocation ? P3T_ENOMEM : P3T_ECUDA;
}

int p3t_reserve(p3t_ctx* ctx, p3t_buf* b, size_t bytes)
{
    if (bytes <= b->bytes) return P3T_OK;
    if (b->p) { P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream)); P3T_CUDA(ctx, cudaFree(b->p)); b->p = nullptr; b->bytes = 0; }
    size_t want = bytes + bytes / 8 + 256;                 // a little head-room: lists grow slowly between steps
    cudaError_t e = cudaMalloc(&b->p, want);
    if (e != cudaSuccess) { b->p = nullptr; (void)cudaGetLastError(); return p3t_fail_cuda(ctx, e, "cudaMalloc", __LINE__); }
    b->bytes = want;
    return P3T_OK;
}

extern "C" {

const char* p3t_strerror(int code)
{
    switch (code) {
    case P3T_OK: return "ok";
    case P3T_EINVAL: return "invalid argument";
    case P3T_ESTATE: return "call out of order (build before force, force before neighbours)";
    case P3T_ENOMEM: return "out of device memory";
    case P3T_ECUDA: return "CUDA failure (see p3t_last_error)";
    case P3T_ERANGE: return "a neighbour row or list exceeds the capacity given";
    case P3T_ELIMIT: return "n exceeds P3T_STATIC_MAX_N, the capacity of the fixed scratch array of p3t_morton_order_static";
    default: return "unknown error code";
    }
}

const char* p3t_last_error(p3t_ctx* ctx) { return ctx ? ctx->err : ""; }

int p3t_create(p3t_ctx** out, int device, void* cuda_stream)
{
    if (!out) return P3T_EINVAL;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { (void)cudaGetLastError(); return P3T_EINVAL; }
    p3t_ctx* c = new (std::nothrow) p3t_ctx();
    if (!c) return P3T_ENOMEM;
    memset(c, 0, sizeof(*c));
    c->device = device; c->stream = (cudaStream_t)cuda_stream;
    c->nleaf = 16; c->ncrit = 64; c->order = 2; c->shard_nranks = 1;
    // Overlap on, 2 CTAs per SM for the walk beside the force kernel (measured 9.03 vs 9.06 ms at config 3), no fault
    // injection.  The library reads no environment variable; measurement and test knobs are set through
    // libp3t_diag.so (include/p3t_diag.h: p3t_diag_set_overlap, p3t_diag_set_fault).
    c->overlap = 1; c->walk_ctas_per_sm = 2; c->test_fault = 0;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, device);
    for (int k = 0; k < 6 && e == cudaSuccess; ++k) e = cudaEventCreate(&c->ev[k]);
    for (int k = 0; k < 4 && e == cudaSuccess; ++k) e = cudaEventCreate(&c->evw[k]);
    for (int k = 0; k < 2 && e == cudaSuccess; ++k) e = cudaEventCreate(&c->evi[k]);
    for (int k = 0; k < 2 && e == cudaSuccess; ++k) e = cudaEventCreate(&c->evc[k]);
    for (int k = 0; k < 2 && e == cudaSuccess; ++k) e = cudaEventCreate(&c->evo[k]);
    if (e != cudaSuccess) { delete c; (void)cudaGetLastError(); return P3T_ECUDA; }
    int rc = p3t_reserve(c, &c->info, sizeof(p3t_devinfo));
    if (rc == P3T_OK) rc = p3t_walk_init(c);
    if (rc != P3T_OK) { p3t_destroy(c); return rc; }
    *out = c;
    return P3T_OK;
}

int p3t_destroy(p3t_ctx* c)
{
    if (!c) return P3T_EINVAL;
    cudaSetDevice(c->device);
    p3t_force_abandon(c);                                    // a force call still in flight: drained, its overlap slot released
    cudaStreamSynchronize(c->stream);
    p3t_buf* bufs[] = { &c->keys[0], &c->keys[1], &c->idx[0], &c->idx[1], &c->spm, &c->rank, &c->hist, &c->nlevel, &c->nbegin, &c->nend,
                        &c->nfirst, &c->nnchild, &c->m64, &c->ncom, &c->nlo, &c->nhi, &c->nq0, &c->nq1, &c->nlink, &c->scan_tmp, &c->pcl, &c->plam, &c->nparent, &c->nfc, &c->ncount, &c->gsum,
                        &c->gflag, &c->gbegin, &c->gnpp, &c->gnpc, &c->nbcount, &c->nboff, &c->nbidx, &c->nbcur, &c->nbcnt, &c->part, &c->spill, &c->pcpool, &c->pppool, &c->glist,
                        &c->info, &c->stage_in, &c->stage_out, &c->core, &c->gready, &c->shard_nominal, &c->shard_cuts, &c->o64, &c->noct, &c->octcnt, &c->psitab, &c->irrpv };
    for (p3t_buf* b : bufs) if (b->p) cudaFree(b->p);
    for (int k = 0; k < 6; ++k) if (c->ev[k]) cudaEventDestroy(c->ev[k]);
    for (int k = 0; k < 4; ++k) if (c->evw[k]) cudaEventDestroy(c->evw[k]);
    for (int k = 0; k < 2; ++k) if (c->evi[k]) cudaEventDestroy(c->evi[k]);
    for (int k = 0; k < 2; ++k) if (c->evc[k]) cudaEventDestroy(c->evc[k]);
    for (int k = 0; k < 2; ++k) if (c->evo[k]) cudaEventDestroy(c->evo[k]);
    if (c->copy_stream) { cudaStreamSynchronize(c->copy_stream); cudaStreamDestroy(c->copy_stream); }
    if (c->walk_stream) {
        cudaStreamSynchronize(c->walk_stream); cudaStreamDestroy(c->walk_stream);
        cudaEventDestroy(c->ev_tree); cudaEventDestroy(c->ev_scan); cudaEventDestroy(c->ev_wdone);
    }
    (void)cudaGetLastError();
    delete c;
    return P3T_OK;
}

int p3t_set_tree_params(p3t_ctx* c, int nleaf, int ncrit)
{
    if (!c || nleaf < 1 || ncrit < nleaf || ncrit > P3T_MAX_NCRIT) return P3T_EINVAL;
    c->nleaf = nleaf; c->ncrit = ncrit;
    return P3T_OK;
}

int p3t_set_multipole_order(p3t_ctx* c, int order)
{
    if (!c || order < 1 || order > 3) return P3T_EINVAL;
    c->order = order;
    return P3T_OK;
}

int p3t_set_shard(p3t_ctx* c, int rank, int nranks, const int64_t* nominal_cuts)
{
    if (!c || nranks < 1 || nranks > P3T_MAX_RANKS || rank < 0 || rank >= nranks) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->pend.active) return P3T_ESTATE;
    c->shard_rank = rank; c->shard_nranks = nranks; c->shard_has_nominal = 0;
    if (nominal_cuts && nranks > 1) {
        P3T_CUDA(c, cudaSetDevice(c->device));
        int rc = p3t_reserve(c, &c->shard_nominal, (size_t)(nranks + 1) * 8);
        if (rc) return rc;
        P3T_CUDA(c, cudaMemcpyAsync(c->shard_nominal.p, nominal_cuts, (size_t)(nranks + 1) * 8, cudaMemcpyHostToDevice, c->stream));
        P3T_CUDA(c, cudaStreamSynchronize(c->stream));       // the caller's array may go away
        c->shard_has_nominal = 1;
    }
    c->state = 0;                                            // the shard takes effect at the next build
    return P3T_OK;
}

int p3t_build_tree(p3t_ctx* c, int64_t n, const float* pos_mass, int key_bits)
{
    if (!c || !pos_mass || n < 1 || n > P3T_MAX_N || (key_bits != 30 && key_bits != 63)) return P3T_EINVAL;
    if (((uintptr_t)pos_mass & 15u) != 0) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->pend.active) return P3T_ESTATE;                   // between p3t_regular_force_begin and _wait
    P3T_CUDA(c, cudaSetDevice(c->device));
    c->state = 0; c->nb_valid = 0; c->irr_done = 0; c->core_done = 0; c->oct_built = 0;
    c->n = n; c->key_bits = key_bits; c->bits = key_bits / 3;
    // hard bound on the cell count (data layout): leaves <= n, branching cells < n,
    // one-child chain cells <= levels * n / (nleaf + 1)
    int64_t cap = 2 * n + (int64_t)c->bits * (n / (c->nleaf + 1)) + 64;
    if (cap > 0x7fffff00ll) cap = 0x7fffff00ll;
    c->node_cap = cap;
    const size_t N = (size_t)n, C = (size_t)cap;
    const size_t ntiles = (N + P3T_SORT_TILE_MIN - 1) / P3T_SORT_TILE_MIN;
    int rc;
#define RES(buf, bytes) if ((rc = p3t_reserve(c, &c->buf, (bytes))) != P3T_OK) return rc
    RES(keys[0], N * 8); RES(keys[1], N * 8); RES(idx[0], N * 4); RES(idx[1], N * 4); RES(spm, N * 16); RES(rank, N * 4);
    RES(hist, p3t_sort_scratch_bytes(n));
    RES(nlevel, C * 4); RES(nbegin, C * 4); RES(nend, C * 4); RES(nfirst, C * 4); RES(nnchild, C * 4);
    RES(m64, C * 8 * M64_STRIDE);
    RES(ncom, C * 16); RES(nlo, C * 16); RES(nhi, C * 16); RES(nq0, C * 16); RES(nq1, C * 8); RES(nlink, C * 8);
    RES(scan_tmp, (size_t)22 * ((N + 255) / 256) * 4 + 64); RES(pcl, N + 64); RES(plam, N + 64);
    RES(nparent, C * 4); RES(nfc, C * 4); RES(ncount, C * 4); RES(gsum, ((N + 4095) / 4096 + 1) * 4);
    RES(gflag, N + 64); RES(gbegin, (N + 2) * 4); RES(gnpp, (N + 1) * 4); RES(gnpc, (N + 1) * 4);
#undef RES
    const float4* pm = (const float4*)pos_mass;
    P3T_CUDA(c, cudaEventRecord(c->ev[0], c->stream));
    P3T_CUDA(c, cudaMemsetAsync(c->info.p, 0, sizeof(p3t_devinfo), c->stream));
    if ((rc = p3t_launch_cube_keys(c, pm)) != P3T_OK) return rc;
    P3T_CUDA(c, cudaEventRecord(c->ev[2], c->stream));
    if ((rc = p3t_launch_sort(c)) != P3T_OK) return rc;
    P3T_CUDA(c, cudaEventRecord(c->ev[3], c->stream));
    if ((rc = p3t_launch_permute(c, pm)) != P3T_OK) return rc;
    if ((rc = p3t_launch_tree(c)) != P3T_OK) return rc;
    if (c->order == 3 && (rc = p3t_launch_octupoles(c)) != P3T_OK) return rc;
    P3T_CUDA(c, cudaEventRecord(c->ev[1], c->stream));
    c->state = 1;
    return P3T_OK;
}

static int force_check_args(p3t_ctx* c, float r_out, float r_in, float theta, int pot_mode, float r_buff,
                            float half_dt, float* vel, float* acc_pot)
{
    if (!c || !acc_pot) return P3T_EINVAL;
    if (!(r_in >= 0.0f) || !(r_in < r_out) || !(theta > 0.0f) || !isfinite(r_out) || !isfinite(theta)) return P3T_EINVAL;
    if (!(r_buff >= 0.0f) || !isfinite(r_buff) || !isfinite(half_dt)) return P3T_EINVAL;
    if (pot_mode != 0 && pot_mode != 1) return P3T_EINVAL;
    if (((uintptr_t)acc_pot & 15u) != 0 || ((uintptr_t)vel & 15u) != 0) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 1) return P3T_ESTATE;
    if (c->order == 3 && !c->oct_built) {
        snprintf(c->err, sizeof(c->err), "multipole order 3 needs a p3t_build_tree after p3t_set_multipole_order");
        return P3T_ESTATE;
    }
    P3T_CUDA(c, cudaSetDevice(c->device));
    c->nb_valid = 0; c->irr_done = 0;
    volatile float rl = r_out + r_buff;                        // one fp32 sum: the list radius of DESIGN.md section 10
    c->r_out = r_out; c->r_in = r_in; c->theta = theta; c->r_list = rl;
    return P3T_OK;
}

int p3t_regular_force_begin(p3t_ctx* c, float r_out, float r_in, float theta, int pot_mode, float r_buff,
                            float half_dt, float* vel, float* acc_pot)
{
    if (c && c->pend.active) return P3T_ESTATE;
    int rc = force_check_args(c, r_out, r_in, theta, pot_mode, r_buff, half_dt, vel, acc_pot);
    if (rc != P3T_OK) return rc;
    c->state = 1;                                            // no lists until the wait has returned
    if ((rc = p3t_force_begin(c, r_out, r_in, theta, pot_mode, (float4*)acc_pot, c->r_list, half_dt, (float4*)vel)) != P3T_OK) {
        (void)p3t_force_finish(c);                           // whatever was enqueued is drained before the error is returned
        return rc;
    }
    return P3T_OK;
}

int p3t_regular_force_wait(p3t_ctx* c)
{
    if (!c) return P3T_EINVAL;
    if (!c->pend.active) return P3T_ESTATE;
    P3T_CUDA(c, cudaSetDevice(c->device));
    int rc = p3t_force_finish(c);
    if (rc != P3T_OK) return rc;
    c->state = 2; c->nb_valid = 1;
    return P3T_OK;
}

int p3t_regular_force_ex(p3t_ctx* c, float r_out, float r_in, float theta, int pot_mode, float r_buff,
                         float half_dt, float* vel, float* acc_pot)
{
    int rc = p3t_regular_force_begin(c, r_out, r_in, theta, pot_mode, r_buff, half_dt, vel, acc_pot);
    if (rc != P3T_OK) return rc;
    return p3t_regular_force_wait(c);
}

int p3t_regular_force(p3t_ctx* c, float r_out, float r_in, float theta, int pot_mode, float* acc_pot)
{
    return p3t_regular_force_ex(c, r_out, r_in, theta, pot_mode, 0.0f, 0.0f, nullptr, acc_pot);
}

int p3t_irregular_force(p3t_ctx* c, const float* vel, float* acc_irr, float* jerk_irr)
{
    if (!c || !vel || !acc_irr || !jerk_irr) return P3T_EINVAL;
    if ((((uintptr_t)vel | (uintptr_t)acc_irr | (uintptr_t)jerk_irr) & 15u) != 0) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 2 || !c->nb_valid) return P3T_ESTATE;
    P3T_CUDA(c, cudaSetDevice(c->device));
    int rc = p3t_launch_irregular(c, (const float4*)vel, (float4*)acc_irr, (float4*)jerk_irr);
    if (rc != P3T_OK) return rc;
    c->irr_done = 1;
    return P3T_OK;
}

int p3t_core_quantities(p3t_ctx* c, int64_t ns, const int32_t* sample, int k, int32_t* nbr, float* d2k, double* rho,
                        double* core_out)
{
    if (!c || !sample || !d2k || !rho || !core_out || ns < 1 || ns > 0x7fffffff || k < 2 || k > 16) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 1) return P3T_ESTATE;
    if (c->n <= k) return P3T_EINVAL;                      // fewer than k other particles
    P3T_CUDA(c, cudaSetDevice(c->device));
    int rc = p3t_reserve(c, &c->core, 64);
    if (rc != P3T_OK) return rc;
    if ((rc = p3t_launch_core(c, ns, sample, k, nbr, d2k, rho, (double*)c->core.p)) != P3T_OK) return rc;
    c->core_done = 1;
    P3T_CUDA(c, cudaMemcpyAsync(core_out, c->core.p, 6 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    return P3T_OK;
}

static int sync_and_check(p3t_ctx* c, p3t_devinfo* h)
{
    P3T_CUDA(c, cudaSetDevice(c->device));
    P3T_CUDA(c, cudaMemcpyAsync(h, c->info.p, sizeof(p3t_devinfo), cudaMemcpyDeviceToHost, c->stream));
    P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    if (h->node_overflow || h->stack_overflow) {
        snprintf(c->err, sizeof(c->err), "internal capacity exceeded (node_overflow=%d stack_overflow=%d)", h->node_overflow, h->stack_overflow);
        return P3T_ECUDA;
    }
    if (h->bad_input) return P3T_EINVAL;
    return P3T_OK;
}

int p3t_get_stats(p3t_ctx* c, p3t_stats* out)
{
    if (!c || !out) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 1) return P3T_ESTATE;
    p3t_devinfo h;
    int rc = sync_and_check(c, &h);
    memset(out, 0, sizeof(*out));
    out->n = c->n; out->n_nodes = h.n_nodes; out->n_leaves = h.n_leaves; out->n_groups = h.n_groups;
    out->max_level = h.max_level; out->key_bits = c->key_bits;
    out->input_bad = h.bad_input;
    for (int a = 0; a < 3; ++a) out->cube_lo[a] = h.lo[a];
    out->cube_side = h.side;
    out->launches = c->launches;
    if (rc == P3T_ECUDA) return rc;
    (void)cudaEventElapsedTime(&out->ms_build, c->ev[0], c->ev[1]);
    (void)cudaEventElapsedTime(&out->ms_sort, c->ev[2], c->ev[3]);
    if (c->state >= 2) {
        out->n_pp = (int64_t)h.n_pp; out->n_pc = (int64_t)h.n_pc;
        out->n_pp_list = (int64_t)h.n_pp_list; out->n_pc_list = (int64_t)h.n_pc_list;
        out->nb_total = (int64_t)h.nb_total; out->nb_max = h.nb_max;
        (void)cudaEventElapsedTime(&out->ms_force, c->ev[4], c->ev[5]);
        (void)cudaEventElapsedTime(&out->ms_eval, c->evw[0], c->evw[1]);
        (void)cudaEventElapsedTime(&out->ms_walk, c->evw[2], c->evw[3]);
        if (c->walk_stream) (void)cudaEventElapsedTime(&out->ms_count, c->ev[4], c->ev_scan);
        if (c->irr_done) (void)cudaEventElapsedTime(&out->ms_irregular, c->evi[0], c->evi[1]);
        if (c->order == 3) (void)cudaEventElapsedTime(&out->ms_octupole, c->evo[0], c->evo[1]);
        out->force_flags = c->pend.flags;
    }
    if (c->core_done) {
        (void)cudaEventElapsedTime(&out->ms_core, c->evc[0], c->evc[1]);
    }
    (void)cudaGetLastError();
    return rc;
}

static int copy_out(p3t_ctx* c, void* dst, const void* src, size_t bytes)
{
    if (!dst || bytes == 0) return P3T_OK;
    P3T_CUDA(c, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDefault, c->stream));
    return P3T_OK;
}

int p3t_neighbours(p3t_ctx* c, const int64_t** offsets, const int32_t** indices, int64_t* total)
{
    if (!c) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 2 || !c->nb_valid) return P3T_ESTATE;
    p3t_devinfo h;
    int rc = sync_and_check(c, &h);
    if (rc != P3T_OK) return rc;
    if (offsets) *offsets = (const int64_t*)c->nboff.p;
    if (indices) *indices = (const int32_t*)c->nbidx.p;
    if (total) *total = (int64_t)h.nb_total;
    return P3T_OK;
}

int p3t_neighbours_copy(p3t_ctx* c, int64_t* offsets_out, int32_t* indices_out)
{
    const int64_t* off; const int32_t* idx; int64_t total;
    int rc = p3t_neighbours(c, &off, &idx, &total);
    if (rc != P3T_OK) return rc;
    if ((rc = copy_out(c, offsets_out, off, ((size_t)c->n + 1) * 8)) != P3T_OK) return rc;
    if ((rc = copy_out(c, indices_out, idx, (size_t)total * 4)) != P3T_OK) return rc;
    P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    return P3T_OK;
}

int p3t_neighbours_nbody6(p3t_ctx* c, int32_t lmax, int32_t* host_list)
{
    if (!c || !host_list || lmax < 0) return P3T_EINVAL;
    const int64_t* off; const int32_t* idx; int64_t total;
    int rc = p3t_neighbours(c, &off, &idx, &total);
    if (rc != P3T_OK) return rc;
    p3t_devinfo h;
    if ((rc = sync_and_check(c, &h)) != P3T_OK) return rc;
    if (h.nb_max > lmax) return P3T_ERANGE;
    const size_t n = (size_t)c->n;
    int64_t* ho = (int64_t*)malloc((n + 1) * 8);
    int32_t* hi = (int32_t*)malloc((size_t)total * 4 + 4);
    if (!ho || !hi) { free(ho); free(hi); return P3T_ENOMEM; }
    rc = p3t_neighbours_copy(c, ho, hi);
    if (rc == P3T_OK) {
        const size_t stride = (size_t)lmax + 1;
        for (size_t i = 0; i < n; ++i) {
            int32_t* row = host_list + i * stride;
            const int64_t b = ho[i], len = ho[i + 1] - b;
            row[0] = (int32_t)len;
            for (int64_t k = 0; k < len; ++k) row[1 + k] = hi[b + k] + 1;        // NBODY6 is 1-based
            for (size_t k = (size_t)len + 1; k < stride; ++k) row[k] = 0;
        }
    }
    free(ho); free(hi);
    return rc;
}

int p3t_step_host(p3t_ctx* c, int64_t n, const float* pos_mass_host, int key_bits,
                  float r_out, float r_in, float theta, int pot_mode,
                  float* acc_pot_host, int64_t* nb_offsets_host, int32_t* nb_indices_host,
                  int64_t nb_cap, int64_t* nb_total)
{
    if (!c || !pos_mass_host || !acc_pot_host || n < 1 || n > P3T_MAX_N) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->pend.active) return P3T_ESTATE;
    P3T_CUDA(c, cudaSetDevice(c->device));
    int rc;
    if ((rc = p3t_reserve(c, &c->stage_in, (size_t)n * 32)) != P3T_OK) return rc;     // pos_mass in, acc_pot out
    float* d_pm = (float*)c->stage_in.p;
    float* d_out = d_pm + (size_t)n * 4;
    P3T_CUDA(c, cudaMemcpyAsync(d_pm, pos_mass_host, (size_t)n * 16, cudaMemcpyHostToDevice, c->stream));
    if ((rc = p3t_build_tree(c, n, d_pm, key_bits)) != P3T_OK) return rc;
    if ((rc = force_check_args(c, r_out, r_in, theta, pot_mode, 0.0f, 0.0f, nullptr, d_out)) != P3T_OK) return rc;
    if ((rc = p3t_force_begin(c, r_out, r_in, theta, pot_mode, (float4*)d_out, c->r_list, 0.0f, nullptr)) != P3T_OK) { (void)p3t_force_finish(c); return rc; }
    // The CSR offsets and the entry count are final once the offset scan is through (ev_scan), long before the force
    // kernel ends: their copies go to a second stream and overlap it.  The host waits for that stream only.
    // From here to p3t_force_finish a call is in flight: every failure goes through p3t_force_finish (IN_FLIGHT), which
    // drains the stream and gives the device's overlap slot back -- a plain return would keep it for good.
#define IN_FLIGHT(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { (void)p3t_force_finish(c); return p3t_fail_cuda(c, e_, #call, __LINE__); } } while (0)
    if (!c->copy_stream) IN_FLIGHT(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    if (c->test_fault & 4) IN_FLIGHT(cudaErrorInvalidValue);          // tests: a CUDA failure with the call in flight
    p3t_devinfo h;
    IN_FLIGHT(cudaStreamWaitEvent(c->copy_stream, c->ev_scan, 0));
    if (nb_offsets_host) IN_FLIGHT(cudaMemcpyAsync(nb_offsets_host, c->nboff.p, ((size_t)n + 1) * 8, cudaMemcpyDeviceToHost, c->copy_stream));
    IN_FLIGHT(cudaMemcpyAsync(&h, c->info.p, sizeof(h), cudaMemcpyDeviceToHost, c->copy_stream));
    IN_FLIGHT(cudaStreamSynchronize(c->copy_stream));
    int64_t total = (int64_t)h.nb_total;
    const bool fits = total <= c->nb_cap && !h.bad_input;                 // else nothing was emitted: the repair pass of finish does it
    IN_FLIGHT(cudaMemcpyAsync(acc_pot_host, d_out, (size_t)n * 16, cudaMemcpyDeviceToHost, c->stream));
    int over = 0;
    if (nb_indices_host) {
        if (total > nb_cap) over = 1;
        else if (total > 0 && fits) IN_FLIGHT(cudaMemcpyAsync(nb_indices_host, c->nbidx.p, (size_t)total * 4, cudaMemcpyDeviceToHost, c->stream));
    }
#undef IN_FLIGHT
    if ((rc = p3t_force_finish(c)) != P3T_OK) return rc;            // synchronises the stream: the copies above are done
    c->state = 2; c->nb_valid = 1;
    if (c->pend.repaired || !fits) {                                // (first call of a context, normally) results changed after the copies
        P3T_CUDA(c, cudaMemcpyAsync(acc_pot_host, d_out, (size_t)n * 16, cudaMemcpyDeviceToHost, c->stream));
        if (nb_indices_host && !over && total > 0)
            P3T_CUDA(c, cudaMemcpyAsync(nb_indices_host, c->nbidx.p, (size_t)total * 4, cudaMemcpyDeviceToHost, c->stream));
        P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    if (nb_total) *nb_total = total;
    return over ? P3T_ERANGE : P3T_OK;
}

// ---- accessors ----
int p3t_get_keys(p3t_ctx* c, uint64_t* sorted_keys, uint32_t* order)
{
    if (!c) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 1) return P3T_ESTATE;
    int rc;
    if ((rc = copy_out(c, sorted_keys, c->keys[0].p, (size_t)c->n * 8)) != P3T_OK) return rc;
    if ((rc = copy_out(c, order, c->idx[0].p, (size_t)c->n * 4)) != P3T_OK) return rc;
    P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    return P3T_OK;
}

int p3t_get_nodes(p3t_ctx* c, int32_t* level, int32_t* begin, int32_t* end, int32_t* first_child, int32_t* n_child)
{
    if (!c) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 1) return P3T_ESTATE;
    p3t_devinfo h;
    int rc = sync_and_check(c, &h);
    if (rc != P3T_OK) return rc;
    const size_t b = (size_t)h.n_nodes * 4;
    if ((rc = copy_out(c, level, c->nlevel.p, b)) != P3T_OK) return rc;
    if ((rc = copy_out(c, begin, c->nbegin.p, b)) != P3T_OK) return rc;
    if ((rc = copy_out(c, end, c->nend.p, b)) != P3T_OK) return rc;
    if ((rc = copy_out(c, first_child, c->nfirst.p, b)) != P3T_OK) return rc;
    if ((rc = copy_out(c, n_child, c->nnchild.p, b)) != P3T_OK) return rc;
    P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    return P3T_OK;
}

int p3t_get_moments(p3t_ctx* c, float* com_m, float* quad, float* clo, float* chi, float* delta)
{
    if (!c) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 1) return P3T_ESTATE;
    p3t_devinfo h;
    int rc = sync_and_check(c, &h);
    if (rc != P3T_OK) return rc;
    const size_t nn = (size_t)h.n_nodes;
    // the walk's SoA packs delta and the level into the .w lanes: unpack on the host
    float4* t = (float4*)malloc(nn * 16 * 3 + nn * 8 + 16);
    if (!t) return P3T_ENOMEM;
    float4 *lo = t, *hi = t + nn, *q0 = t + 2 * nn; float2* q1 = (float2*)(t + 3 * nn);
    cudaError_t e = cudaMemcpyAsync(lo, c->nlo.p, nn * 16, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(hi, c->nhi.p, nn * 16, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(q0, c->nq0.p, nn * 16, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(q1, c->nq1.p, nn * 8, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess && com_m) e = cudaMemcpyAsync(com_m, c->ncom.p, nn * 16, cudaMemcpyDefault, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { free(t); return p3t_fail_cuda(c, e, "p3t_get_moments copies", __LINE__); }
    for (size_t k = 0; k < nn; ++k) {
        if (quad) { float* q = quad + 6 * k; q[0] = q0[k].x; q[1] = q0[k].y; q[2] = q0[k].z; q[3] = q0[k].w; q[4] = q1[k].x; q[5] = q1[k].y; }
        if (clo) { clo[3 * k] = lo[k].x; clo[3 * k + 1] = lo[k].y; clo[3 * k + 2] = lo[k].z; }
        if (chi) { chi[3 * k] = hi[k].x; chi[3 * k + 1] = hi[k].y; chi[3 * k + 2] = hi[k].z; }
        if (delta) delta[k] = lo[k].w;
    }
    free(t);
    return P3T_OK;
}

int p3t_get_groups(p3t_ctx* c, int32_t* begin, int32_t* end)
{
    if (!c) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 1) return P3T_ESTATE;
    p3t_devinfo h;
    int rc = sync_and_check(c, &h);
    if (rc != P3T_OK) return rc;
    const size_t b = (size_t)h.n_groups * 4;
    if ((rc = copy_out(c, begin, c->gbegin.p, b)) != P3T_OK) return rc;
    if ((rc = copy_out(c, end, (const int32_t*)c->gbegin.p + 1, b)) != P3T_OK) return rc;
    P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    return P3T_OK;
}

int p3t_get_list_lengths(p3t_ctx* c, int32_t* npp, int32_t* npc)
{
    if (!c) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 2) return P3T_ESTATE;
    p3t_devinfo h;
    int rc = sync_and_check(c, &h);
    if (rc != P3T_OK) return rc;
    const size_t b = (size_t)h.n_groups * 4;
    if ((rc = copy_out(c, npp, c->gnpp.p, b)) != P3T_OK) return rc;
    if ((rc = copy_out(c, npc, c->gnpc.p, b)) != P3T_OK) return rc;
    P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    return P3T_OK;
}

// eq. 20-25
int p3t_params_from_n(int64_t n, double sigma, double* tau, double* r_cut, double* r_buff, double* dt_reg, double* dt_max)
{
    if (n < 1 || !(sigma > 0.0)) return P3T_EINVAL;
    const double t = (1.0 / 128.0) * pow((double)n / 16384.0, -1.0 / 3.0);   // eq. 22
    double dt = 1.0;
    while (dt > t * (1.0 + 1e-12)) dt *= 0.5;                                 // eq. 23: largest 2^-k <= tau (reading R12)
    if (tau) *tau = t;
    if (r_cut) *r_cut = 4.0 * t;                                              // eq. 21
    if (r_buff) *r_buff = 3.0 * t * sigma;                                    // eq. 20
    if (dt_reg) *dt_reg = dt;
    if (dt_max) *dt_max = dt / 4.0;                                           // eq. 24-25
    return P3T_OK;
}

}  // extern "C"
