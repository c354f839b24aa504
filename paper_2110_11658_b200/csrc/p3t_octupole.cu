// p3t_octupole.cu -- SURVEY.md 8f NEXT-4: the octupole variant (p3t_set_multipole_order(ctx, 3)), a more
// accurate point on the accuracy-throughput curve.  The paper evaluates monopole + quadrupole;
// this adds the third-order term of the same Taylor expansion of 1/|r - d| for every ACCEPTED cell of the same
// interaction lists.  With the raw third moment T_abc = sum m d_a d_b d_c about the cell's centre of mass,
// r = x_i - COM, R = |r|:
//     t3 = T_abc r_a r_b r_c,  v_a = T_abc r_b r_c,  tau_a = T_bba,  u = tau.r
//     phi_3 = -(5/2) t3 / R^7 + (3/2) u / R^5
//     a_3   = (15/2) v / R^7 - (35/2) t3 r / R^9 - (3/2) tau / R^5 + (15/2) u r / R^7
// evaluated through the traceless form O = 5 T - sym(delta tau): phi_3 = -(1/2) O:rrr / R^7,
//     a_3 = (3/2) O:rr / R^7 - (7/2) (O:rrr) r / R^9   (identical, a third fewer operations).
// Two kernels, both outside the default path (which they leave untouched):
//   k_octupoles   third moments of every cell in fp64: leaves from their particles, internal cells by the
//                 parallel-axis rule, climbing with arrival counters like k_moments (p3t_tree.cu);
//   k_octupole_add  streams the particle-cell lists that k_walk wrote and adds the term to acc_pot.
// This is a first, plain version (scalar fp32, one warp per 32 targets, the data of 32 cells staged in shared
// memory): it is NOT tuned like k_force; DESIGN.md section 10 reports its time beside the default path's.
#include "p3t_internal.cuh"
#include <stdlib.h>

#define OCT_THREADS 128

struct oct_args {
    const float4* spm; const int32_t *nbegin, *nend, *nfirst, *nnchild, *nparent;
    const double* m64;          // [node][13] from k_moments: M, sum m x (3), Q (6), COM (3)
    double* o64;                // [node][11]: tr S, T (10: xxx yyy zzz xxy xxz xyy yyz xzz yzz xyz)
    float4* noct;               // [node][3]: the ten components of the traceless form, rounded once to fp32 (+ 2 x padding)
    int32_t* cnt;               // arrival counters, zeroed by the host side
    p3t_devinfo* info;
};

__device__ __forceinline__ void oct_store(const oct_args& A, int k, double tr, const double T[10])
{
    double* o = A.o64 + (size_t)k * 11;
    o[0] = tr;
#pragma unroll
    for (int q = 0; q < 10; ++q) o[1 + q] = T[q];
    // the force kernel reads the traceless form O_abc = 5 T_abc - (delta_ab tau_c + delta_ac tau_b + delta_bc tau_a),
    // tau_a = T_bba, with which phi_3 = -(1/2) O:rrr / R^7 and a_3 = (3/2) O:rr / R^7 - (7/2) (O:rrr) r / R^9
    // (O:rrr = 5 t3 - 3 R^2 u: the same term with a third fewer operations); made in fp64, rounded once
    const double tx = T[0] + T[5] + T[7], ty = T[3] + T[1] + T[8], tz = T[4] + T[6] + T[2];
    A.noct[(size_t)k * 3 + 0] = make_float4((float)(5.0 * T[0] - 3.0 * tx), (float)(5.0 * T[1] - 3.0 * ty), (float)(5.0 * T[2] - 3.0 * tz), (float)(5.0 * T[3] - ty));
    A.noct[(size_t)k * 3 + 1] = make_float4((float)(5.0 * T[4] - tz), (float)(5.0 * T[5] - tx), (float)(5.0 * T[6] - tz), (float)(5.0 * T[7] - tx));
    A.noct[(size_t)k * 3 + 2] = make_float4((float)(5.0 * T[8] - ty), (float)(5.0 * T[9]), 0.0f, 0.0f);
}

__global__ void __launch_bounds__(OCT_THREADS) k_octupoles(oct_args A)
{
    const int nn = A.info->n_nodes;
    int k = blockIdx.x * OCT_THREADS + threadIdx.x;
    if (k >= nn || A.info->node_overflow || A.nnchild[k] != 0) return;
    {
        const double* mk = A.m64 + (size_t)k * M64_STRIDE;
        const double c[3] = { mk[10], mk[11], mk[12] };
        double tr = 0.0, T[10] = { 0, 0, 0, 0, 0, 0, 0, 0, 0, 0 };
        for (int i = A.nbegin[k]; i < A.nend[k]; ++i) {
            const float4 p = A.spm[i];
            const double m = p.w, dx = p.x - c[0], dy = p.y - c[1], dz = p.z - c[2];
            tr += m * (dx * dx + dy * dy + dz * dz);
            T[0] += m * dx * dx * dx; T[1] += m * dy * dy * dy; T[2] += m * dz * dz * dz;
            T[3] += m * dx * dx * dy; T[4] += m * dx * dx * dz; T[5] += m * dx * dy * dy;
            T[6] += m * dy * dy * dz; T[7] += m * dx * dz * dz; T[8] += m * dy * dz * dz; T[9] += m * dx * dy * dz;
        }
        oct_store(A, k, tr, T);
    }
    for (;;) {
        const int p = A.nparent[k];
        if (p < 0) break;
        __threadfence();
        if (atomicAdd(&A.cnt[p], 1) + 1 < A.nnchild[p]) break;
        __threadfence();
        k = p;
        const double* mk = A.m64 + (size_t)k * M64_STRIDE;
        const double cm[3] = { mk[10], mk[11], mk[12] };
        double tr = 0.0, T[10] = { 0, 0, 0, 0, 0, 0, 0, 0, 0, 0 };
        const int fc = A.nfirst[k], nc = A.nnchild[k];
        for (int c = fc; c < fc + nc; ++c) {
            // parallel-axis rule, s = COM_c - COM: T_abc += T^c_abc + s_a S_bc + s_b S_ac + s_c S_ab + M_c s_a s_b s_c,
            // S = raw second moment of the child about its own COM = (Q + tr(S) 1) / 3
            const double* m = A.m64 + (size_t)c * M64_STRIDE;
            const double* o = A.o64 + (size_t)c * 11;
            const double Mc = m[0], sx = m[10] - cm[0], sy = m[11] - cm[1], sz = m[12] - cm[2];
            const double trc = __ldcg(o);
            const double Sxx = (m[4] + trc) / 3.0, Syy = (m[5] + trc) / 3.0, Szz = (m[6] + trc) / 3.0;
            const double Sxy = m[7] / 3.0, Sxz = m[8] / 3.0, Syz = m[9] / 3.0;
            tr += trc + Mc * (sx * sx + sy * sy + sz * sz);
            T[0] += __ldcg(o + 1) + 3.0 * sx * Sxx + Mc * sx * sx * sx;
            T[1] += __ldcg(o + 2) + 3.0 * sy * Syy + Mc * sy * sy * sy;
            T[2] += __ldcg(o + 3) + 3.0 * sz * Szz + Mc * sz * sz * sz;
            T[3] += __ldcg(o + 4) + 2.0 * sx * Sxy + sy * Sxx + Mc * sx * sx * sy;
            T[4] += __ldcg(o + 5) + 2.0 * sx * Sxz + sz * Sxx + Mc * sx * sx * sz;
            T[5] += __ldcg(o + 6) + sx * Syy + 2.0 * sy * Sxy + Mc * sx * sy * sy;
            T[6] += __ldcg(o + 7) + 2.0 * sy * Syz + sz * Syy + Mc * sy * sy * sz;
            T[7] += __ldcg(o + 8) + sx * Szz + 2.0 * sz * Sxz + Mc * sx * sz * sz;
            T[8] += __ldcg(o + 9) + sy * Szz + 2.0 * sz * Syz + Mc * sy * sz * sz;
            T[9] += __ldcg(o + 10) + sx * Syz + sy * Sxz + sz * Sxy + Mc * sx * sy * sz;
        }
        oct_store(A, k, tr, T);
    }
}

int p3t_launch_octupoles(p3t_ctx* ctx)
{
    int rc;
    const size_t C = (size_t)ctx->node_cap;
    if ((rc = p3t_reserve(ctx, &ctx->o64, C * 11 * sizeof(double)))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->noct, C * 3 * sizeof(float4)))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->octcnt, C * sizeof(int32_t)))) return rc;
    P3T_CUDA(ctx, cudaMemsetAsync(ctx->octcnt.p, 0, C * sizeof(int32_t), ctx->stream));
    oct_args A;
    A.spm = P<float4>(ctx->spm); A.nbegin = P<int32_t>(ctx->nbegin); A.nend = P<int32_t>(ctx->nend);
    A.nfirst = P<int32_t>(ctx->nfirst); A.nnchild = P<int32_t>(ctx->nnchild); A.nparent = P<int32_t>(ctx->nparent);
    A.m64 = P<double>(ctx->m64); A.o64 = P<double>(ctx->o64); A.noct = P<float4>(ctx->noct);
    A.cnt = P<int32_t>(ctx->octcnt); A.info = INFO(ctx);
    k_octupoles<<<(unsigned)((C + OCT_THREADS - 1) / OCT_THREADS), OCT_THREADS, 0, ctx->stream>>>(A);
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
    ctx->oct_built = 1;
    return P3T_OK;
}

// ---------------------------------------------------------------------------------------------
struct octadd_args {
    const float4* spm; const uint32_t* order;
    const float4 *ncom, *noct;
    const int32_t* gbegin; const uint4* glist; const int32_t* pcpool;
    float4 *out, *vel; float half_dt;
    p3t_devinfo* info;
    const int32_t* gready; int base, mode, evalall;      // the group filter of the force kernel (p3t_force.cu)
};

__global__ void __launch_bounds__(OCT_THREADS) k_octupole_add(octadd_args A)
{
    __shared__ float4 s_node[OCT_THREADS / 32][4][32];
    const int lane = threadIdx.x & 31;
    if (A.info->bad_input | A.info->node_overflow | A.info->stack_overflow) return;
    const int g0 = A.info->shard_g0, ng = A.info->shard_g1 - g0;
    const int nwarps = gridDim.x * (OCT_THREADS / 32);
    for (int c = blockIdx.x * (OCT_THREADS / 32) + (threadIdx.x >> 5); c < 2 * ng; c += nwarps) {
        const int g = g0 + (c >> 1);
        const int gb = A.gbegin[g], cnt = A.gbegin[g + 1] - gb, tb = 32 * (c & 1);
        if (tb >= cnt) continue;
        // the same groups as the force kernel of this pass (the term is ADDED: never twice to the same group)
        const int st = A.gready[g] - A.base;
        if (A.mode == 0 ? st != G_READY : !(st == G_REDONE || (A.evalall && st == G_READY))) continue;
        const bool kick = A.mode == 0 || st == G_REDONE;
        const int i = gb + tb + lane;
        const bool live = tb + lane < cnt;
        const float4 xi = A.spm[live ? i : gb];
        const uint4 gl = A.glist[g];
        const int32_t* list = A.pcpool + ((long long)gl.x << 5);
        const int npc = (int)gl.y;
        double ax = 0.0, ay = 0.0, az = 0.0, ph = 0.0;
        float4 (*S)[32] = s_node[threadIdx.x >> 5];
        for (int e0 = 0; e0 < npc; e0 += 32) {
            const int m = min(32, npc - e0);
            // the data of 32 cells go to shared memory, one cell per lane; the loop below reads them as broadcasts
            __syncwarp();
            if (lane < m) {
                const int node = list[e0 + lane];
                S[0][lane] = A.ncom[node];
                S[1][lane] = A.noct[(size_t)node * 3]; S[2][lane] = A.noct[(size_t)node * 3 + 1]; S[3][lane] = A.noct[(size_t)node * 3 + 2];
            }
            __syncwarp();
            float fx = 0.0f, fy = 0.0f, fz = 0.0f, fp = 0.0f;        // fp32 over <= 32 entries, folded into fp64 (R-S9)
#pragma unroll 2
            for (int q = 0; q < m; ++q) {
                const float4 cm = S[0][q], t0 = S[1][q], t1 = S[2][q], t2 = S[3][q];
                const float xxx = t0.x, yyy = t0.y, zzz = t0.z, xxy = t0.w, xxz = t1.x, xyy = t1.y, yyz = t1.z, xzz = t1.w, yzz = t2.x, xyz = t2.y;
                const float x = xi.x - cm.x, y = xi.y - cm.y, z = xi.z - cm.z;
                const float R2 = fmaf(z, z, fmaf(y, y, x * x));
                const float ri = rsqrtf(R2), ri2 = ri * ri, ri7 = ri2 * ri2 * ri2 * ri, ri9 = ri7 * ri2;
                const float x2 = x + x, y2 = y + y;
                const float xx = x * x, yy = y * y, zz = z * z, xy = x2 * y, xz = x2 * z, yz = y2 * z;
                const float wx = fmaf(xxx, xx, fmaf(xyy, yy, fmaf(xzz, zz, fmaf(xxy, xy, fmaf(xxz, xz, xyz * yz)))));
                const float wy = fmaf(xxy, xx, fmaf(yyy, yy, fmaf(yzz, zz, fmaf(xyy, xy, fmaf(xyz, xz, yyz * yz)))));
                const float wz = fmaf(xxz, xx, fmaf(yyz, yy, fmaf(zzz, zz, fmaf(xyz, xy, fmaf(xzz, xz, yzz * yz)))));
                const float o3 = fmaf(wz, z, fmaf(wy, y, wx * x));
                fp = fmaf(-0.5f * o3, ri7, fp);
                const float c1 = 1.5f * ri7, c2 = -3.5f * o3 * ri9;
                fx += fmaf(c2, x, c1 * wx);
                fy += fmaf(c2, y, c1 * wy);
                fz += fmaf(c2, z, c1 * wz);
            }
            ax += (double)fx; ay += (double)fy; az += (double)fz; ph += (double)fp;
        }
        if (live) {
            const uint32_t o = A.order[i];
            float4 r = A.out[o];
            const float dax = (float)ax, day = (float)ay, daz = (float)az;
            r.x += dax; r.y += day; r.z += daz; r.w += (float)ph;
            A.out[o] = r;
            if (A.vel && kick) {
                float4 v = A.vel[o];
                v.x = fmaf(A.half_dt, dax, v.x); v.y = fmaf(A.half_dt, day, v.y); v.z = fmaf(A.half_dt, daz, v.z);
                A.vel[o] = v;
            }
        }
    }
}

int p3t_launch_octupole_add(p3t_ctx* ctx, float4* acc_pot, float half_dt, float4* vel, int base, int mode, int evalall)
{
    octadd_args A;
    A.spm = P<float4>(ctx->spm); A.order = P<uint32_t>(ctx->idx[0]);
    A.ncom = P<float4>(ctx->ncom); A.noct = P<float4>(ctx->noct);
    A.gbegin = P<int32_t>(ctx->gbegin); A.glist = P<uint4>(ctx->glist); A.pcpool = P<int32_t>(ctx->pcpool);
    A.out = acc_pot; A.vel = vel; A.half_dt = half_dt; A.info = INFO(ctx);
    A.gready = P<int32_t>(ctx->gready); A.base = base; A.mode = mode; A.evalall = evalall;
    P3T_CUDA(ctx, cudaEventRecord(ctx->evo[0], ctx->stream));
    k_octupole_add<<<ctx->num_sms * 8, OCT_THREADS, 0, ctx->stream>>>(A);
    P3T_CUDA(ctx, cudaGetLastError());
    P3T_CUDA(ctx, cudaEventRecord(ctx->evo[1], ctx->stream));
    ctx->launches += 1;
    return P3T_OK;
}

// parity accessor: the fp32 third moments of every cell, [n_nodes][10]
extern "C" int p3t_get_octupoles(p3t_ctx* c, float* oct)
{
    if (!c || !oct) return P3T_EINVAL;
    if (c->sticky) return P3T_ECUDA;
    if (c->state < 1 || !c->oct_built) return P3T_ESTATE;
    P3T_CUDA(c, cudaSetDevice(c->device));
    p3t_devinfo h;
    P3T_CUDA(c, cudaMemcpyAsync(&h, c->info.p, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    P3T_CUDA(c, cudaStreamSynchronize(c->stream));
    const size_t nn = (size_t)h.n_nodes;
    double* t = (double*)malloc(nn * 88 + 16);
    if (!t) return P3T_ENOMEM;
    cudaError_t e = cudaMemcpyAsync(t, c->o64.p, nn * 88, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { free(t); return p3t_fail_cuda(c, e, "p3t_get_octupoles copy", __LINE__); }
    for (size_t k = 0; k < nn; ++k)
        for (int q = 0; q < 10; ++q) oct[10 * k + q] = (float)t[11 * k + 1 + q];
    free(t);
    return P3T_OK;
}
