// p3t_force.cu -- steps a8-a11: particle-cell and particle-particle regular force with
// the cutoff of eq. 6 and neighbour-list emission fused in, results
// scattered to the caller's particle order; plus the neighbour CSR bookkeeping (a10).
//
//   F_R,i = sum_j m_j W(x_ij) (x_j - x_i) / r_ij^3,  W = 1 - K,  x = (r - r_in)/(r_out - r_in)
//   (eq. 1, 3, 4, 6, 8-10; attractive sign: DESIGN.md R1)
//
// One warp evaluates one work item (up to 32 targets of one group, see `target` below) against the
// group's interaction lists that k_walk<WALK_LISTS> left in HBM.  32 list entries at a time are gathered
// (node / particle data, L2-resident) into a double-buffered structure-of-arrays tile in shared
// memory while the previous tile is being evaluated, so the FP32 pipe never waits for the walk.
// Rules: DESIGN.md R-S8 (evaluation), R-S9 (accumulation), R10 (neighbour predicate, bit-specified).
#include "p3t_internal.cuh"
#include "p3t_cutoff.cuh"
#include "p3t_f32x2.cuh"
#include <stdio.h>
#include <stdlib.h>
#include <math.h>

#define FORCE_WARPS   4
#define FORCE_THREADS (FORCE_WARPS * 32)
#define FORCE_CTAS_PER_SM 3               // a register cap (168), not the occupancy: ptxas takes 126 and 4 CTAs/SM are
                                          // resident; caps of 5 (102 regs) and 6 (80) measured 5 % and 8 % slower
#define TILE          32                  // list entries per tile
#define FAR_AWAY      1.0e18f             // position of the zero-mass padding entries of a tile

struct force_args {
    const float4* spm; const uint32_t* order;
    const float4 *ncom, *nq0; const float2* nq1;
    const int32_t* gbegin;
    const uint4* glist;
    const int32_t *pcpool, *pppool;
    const int64_t* nboff;       // per ORIGINAL id
    int32_t* nbraw;             // out: unsorted rows
    float4* out;                // out: acc_pot, original order
    int32_t* nbcnt;             // SPLIT: per sorted position, neighbours already written to the row (zeroed)
    double* part;               // SPLIT: partial sums [nseg][n][4], original order
    int nseg;                   // SPLIT: list segments per item
    int mp_order;               // 2: monopole + quadrupole (default); 1: monopole only
    int n;
    float4* vel;                // in/out (may be NULL): velocities, original order, kicked by half_dt * F_R (eq. 12)
    float half_dt;
    p3t_devinfo* info;
    int32_t* gready;            // per-group list state written by the walkers (p3t_internal.cuh: G_READY ...)
    int base;                   // epoch of the call
    int mode;                   // 0: the walkers run at the same time, wait for every group; 1: host repair pass
    int evalall;                // repair pass: every group again (the lists were not emitted), else only the redone ones
    long long nb_cap;           // capacity of nbraw in entries
    long long pc_size, pp_size; // entries of the list pools (P3T_CHECKS)
    walk_consts K;
};

// Per-warp list tiles, double-buffered, structure-of-arrays so that two (LDS.64) or four (LDS.128)
// consecutive entries arrive as the packed operands of the f32x2 instructions below.
// pc rows: 0-2 COM, 3 M, 4-9 MINUS the traceless quadrupole (xx yy zz xy xz yz).
struct __align__(16) tile_smem {
    float pc[2][10][TILE];
    float pp[2][4][TILE];       // x y z m
    int   ppj[2][TILE];         // sorted position of the source, -1 = padding
    int   nbrow[32];            // per target of the item: neighbours already written to its CSR row
};

__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// One work item = up to 32 targets of one group (see k_force; the items of a group stream the same
// lists).  An item with c <= 16 targets gives every target k = 2, 4 or 8 lanes
// ("parts"): lane = target * k + part, and part p evaluates the 4-entry blocks p, p + k, ... of every
// tile, so that a half-empty item costs half the time instead of idling half the lanes.  The parts
// of a target are summed by shuffles at the end.
//
// Every accumulator is a pair: .lo / e sums the even list entries, .hi / o the odd ones.  ph
// accumulates MINUS the potential of the far terms; the rare near-zone terms (cutoff branch) go to
// the scalar n* accumulators with their true sign.
struct target {
    float x, y, z;
    f2    ph;                                    // fp32 partial sums since the last fold
    float axe, aye, aze, axo, ayo, azo;          // scalar FFMAs: see pc_pair
    float nax, nay, naz, nph;
    double dax, day, daz, dph;                   // fp64 masters (R-S9)
    int   id;                                    // sorted position of the target, -1 = idle lane
    int   slot;                                  // index of the target inside the item (row of the neighbour cursor)
};

__device__ __forceinline__ void fold(target& T)
{
    T.dax += (double)((T.axe + T.axo) + T.nax);
    T.day += (double)((T.aye + T.ayo) + T.nay);
    T.daz += (double)((T.aze + T.azo) + T.naz);
    T.dph += (double)(T.nph - (f2lo(T.ph) + f2hi(T.ph)));
    T.ph = pk(0.0f, 0.0f);
    T.axe = T.aye = T.aze = T.axo = T.ayo = T.azo = 0.0f;
    T.nax = T.nay = T.naz = T.nph = 0.0f;
}

// R-S8 particle-cell, monopole + traceless quadrupole, two cells per packed operation.
// With d = COM - x_i (= -r), Q' = -Q (stored negated in the tile), R = |d|:
//   q' = d.Q'.d / R^5,  -phi = M/R - q'/2,  a = (M/R - (5/2) q') d / R^2 + (Q'.d) / R^5
// which is a = -M r/R^3 + Q.r/R^5 - (5/2)(r.Q.r) r/R^7 of R-S8.
__device__ __forceinline__ void pc_pair(target& T, f2 cx, f2 cy, f2 cz, f2 cm, f2 qxx, f2 qyy, f2 qzz, f2 qxy, f2 qxz, f2 qyz)
{
    const f2 mhalf = pk(-0.5f, -0.5f), m52 = pk(-2.5f, -2.5f);
    const f2 dx = sub2(cx, pk(T.x, T.x)), dy = sub2(cy, pk(T.y, T.y)), dz = sub2(cz, pk(T.z, T.z));
    const f2 R2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
    const f2 ri = pk(rsqrt_approx(f2lo(R2)), rsqrt_approx(f2hi(R2)));
    const f2 ri2 = mul2(ri, ri);
    const f2 qx = fma2(qxz, dz, fma2(qxy, dy, mul2(qxx, dx)));
    const f2 qy = fma2(qyz, dz, fma2(qyy, dy, mul2(qxy, dx)));
    const f2 qz = fma2(qzz, dz, fma2(qyz, dy, mul2(qxz, dx)));
    const f2 dqd = fma2(dz, qz, fma2(dy, qy, mul2(dx, qx)));
    const f2 ri3 = mul2(ri2, ri), ri5 = mul2(ri3, ri2);
    const f2 mono = mul2(cm, ri);
    const f2 q5 = mul2(dqd, ri5);
    T.ph = fma2(mhalf, q5, add2(T.ph, mono));
    const f2 cr = mul2(fma2(m52, q5, mono), ri2);
    // An FFMA2 with three distinct register-pair operands occupies the pipe for 3 cycles (measured:
    // operand bandwidth), two scalar FFMAs for 2: the accumulations are issued on the halves.
    const float crl = f2lo(cr), crh = f2hi(cr), r5l = f2lo(ri5), r5h = f2hi(ri5);
    T.axe = fmaf(f2lo(qx), r5l, fmaf(crl, f2lo(dx), T.axe)); T.axo = fmaf(f2hi(qx), r5h, fmaf(crh, f2hi(dx), T.axo));
    T.aye = fmaf(f2lo(qy), r5l, fmaf(crl, f2lo(dy), T.aye)); T.ayo = fmaf(f2hi(qy), r5h, fmaf(crh, f2hi(dy), T.ayo));
    T.aze = fmaf(f2lo(qz), r5l, fmaf(crl, f2lo(dz), T.aze)); T.azo = fmaf(f2hi(qz), r5h, fmaf(crh, f2hi(dz), T.azo));
}

// one tile of TILE cells; this lane takes the 4-entry blocks part, part + k, ...
__device__ __forceinline__ void eval_pc(target& T, const float (*pc)[TILE], int part, int k)
{
#pragma unroll 4
    for (int e = 4 * part; e < TILE; e += 4 * k) {
        ulonglong2 v[10];
#pragma unroll
        for (int r = 0; r < 10; ++r) v[r] = *reinterpret_cast<const ulonglong2*>(&pc[r][e]);
        pc_pair(T, v[0].x, v[1].x, v[2].x, v[3].x, v[4].x, v[5].x, v[6].x, v[7].x, v[8].x, v[9].x);
        pc_pair(T, v[0].y, v[1].y, v[2].y, v[3].y, v[4].y, v[5].y, v[6].y, v[7].y, v[8].y, v[9].y);
    }
}

// Monopole-only variant (SURVEY 8f NEXT-4, p3t_set_multipole_order(ctx, 1)): R-S8 with Q = 0,
// phi = -M/R, a = M d / R^3; 13 operations per pair instead of 33.
__device__ __forceinline__ void pc_pair_mono(target& T, f2 cx, f2 cy, f2 cz, f2 cm)
{
    const f2 dx = sub2(cx, pk(T.x, T.x)), dy = sub2(cy, pk(T.y, T.y)), dz = sub2(cz, pk(T.z, T.z));
    const f2 R2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
    const f2 ri = pk(rsqrt_approx(f2lo(R2)), rsqrt_approx(f2hi(R2)));
    const f2 mono = mul2(cm, ri);
    const f2 f = mul2(mono, mul2(ri, ri));
    T.ph = add2(T.ph, mono);
    const float fl = f2lo(f), fh = f2hi(f);
    T.axe = fmaf(fl, f2lo(dx), T.axe); T.axo = fmaf(fh, f2hi(dx), T.axo);
    T.aye = fmaf(fl, f2lo(dy), T.aye); T.ayo = fmaf(fh, f2hi(dy), T.ayo);
    T.aze = fmaf(fl, f2lo(dz), T.aze); T.azo = fmaf(fh, f2hi(dz), T.azo);
}
__device__ __forceinline__ void eval_pc_mono(target& T, const float (*pc)[TILE], int part, int k)
{
#pragma unroll 2
    for (int e = 4 * part; e < TILE; e += 4 * k) {
        ulonglong2 v[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) v[r] = *reinterpret_cast<const ulonglong2*>(&pc[r][e]);
        pc_pair_mono(T, v[0].x, v[1].x, v[2].x, v[3].x);
        pc_pair_mono(T, v[0].y, v[1].y, v[2].y, v[3].y);
    }
}

// Two sources per packed operation: the far zone (d2 >= r_out^2, W = 1, pure Newtonian) of the
// p-p list, branch-free.  d2 follows R10 bit for bit (sub, mul, fma, fma; all rn).  A near pair is
// (d2 < r_list^2, the neighbour search radius) masked out by replacing its d2 with +inf (rsqrt -> 0, every term exactly 0); the smallest d2 seen
// by the lane is returned so that the caller knows whether the tile needs the near pass.
__device__ __forceinline__ float pp_far_pair(target& T, f2 px, f2 py, f2 pz, f2 pm, float rlist2, float dmin)
{
    const f2 dx = sub2(px, pk(T.x, T.x)), dy = sub2(py, pk(T.y, T.y)), dz = sub2(pz, pk(T.z, T.z));
    const f2 d2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
    const float d2a = f2lo(d2), d2b = f2hi(d2);
    dmin = fminf(dmin, fminf(d2a, d2b));
    const f2 ri = pk(rsqrt_approx(d2a < rlist2 ? INFINITY : d2a), rsqrt_approx(d2b < rlist2 ? INFINITY : d2b));
    const f2 mri = mul2(pm, ri);
    const f2 f = mul2(mri, mul2(ri, ri));
    T.ph = add2(T.ph, mri);
    const float fl = f2lo(f), fh = f2hi(f);
    T.axe = fmaf(fl, f2lo(dx), T.axe); T.axo = fmaf(fh, f2hi(dx), T.axo);
    T.aye = fmaf(fl, f2lo(dy), T.aye); T.ayo = fmaf(fh, f2hi(dy), T.ayo);
    T.aze = fmaf(fl, f2lo(dz), T.aze); T.azo = fmaf(fh, f2hi(dz), T.azo);
    return dmin;
}

// R10 + eq. 6, near zone (d2 < r_out^2): neighbour emission and the cutoff-weighted pair term.
// Scalar pass over the 4-entry blocks in which the far pass saw this lane's target within r_out
// (bit mask), run only by warps that have such a block in the tile (about one tile in eight).  nbrow[slot] counts the entries already written
// to the target's CSR row (shared by the parts of a target).
__device__ __forceinline__ void pp_near_pass(target& T, const float (*pp)[TILE], const int* ppj, uint32_t nearblocks,
                                             long long rowbase, int* rowcnt, const force_args& A, bool emit)
{
    const walk_consts& K = A.K;
    while (nearblocks) {
        const int e0 = (__ffs(nearblocks) - 1) << 2;
        nearblocks &= nearblocks - 1;
#pragma unroll 1
        for (int e = e0; e < e0 + 4; ++e) {
            const float dx = __fsub_rn(pp[0][e], T.x), dy = __fsub_rn(pp[1][e], T.y), dz = __fsub_rn(pp[2][e], T.z);
            const float d2 = fmaf(dz, dz, fmaf(dy, dy, __fmul_rn(dx, dx)));
            if (d2 < K.rlist2) {
                const int j = ppj[e];
                if (T.id >= 0 && j != T.id) {                        // self excluded by index; idle lanes
                    if (emit) {
                        const int at = atomicAdd(rowcnt, 1);
                        P3T_CHECK(rowbase + at >= 0 && rowbase + at < A.nb_cap && rowbase + at < A.nboff[A.order[T.id] + 1]);
                        A.nbraw[rowbase + at] = (int32_t)A.order[j];
                    }
                    const float m = pp[3][e];
                    if (d2 >= K.rout2) {                               // buffer shell r_out <= r < r_list: on the list, wholly regular
                        const float ri = rsqrt_approx(d2), mr = m * ri, f = mr * ri * ri;
                        T.nax = fmaf(f, dx, T.nax); T.nay = fmaf(f, dy, T.nay); T.naz = fmaf(f, dz, T.naz);
                        T.nph -= mr;
                    } else if (d2 > K.rin2) {
                        const float ri = rsqrt_approx(d2), r = d2 * ri;
                        const float x = fminf(fmaxf((r - K.r_in) * K.inv_delta, 0.0f), 1.0f);
                        const float W = cutoff_W(x);
                        const float f = m * W * ri * ri * ri;
                        T.nax = fmaf(f, dx, T.nax); T.nay = fmaf(f, dy, T.nay); T.naz = fmaf(f, dz, T.naz);
                        T.nph += K.pot_mode == 0 ? m * cutoff_psi(K, x, W, ri) : -m * ri;
                    } else if (K.pot_mode == 0) {
                        T.nph = fmaf(m, K.psi_in, T.nph);              // inside r_in: constant psi(r_in), also r = 0 (R8)
                    } else if (d2 > 0.0f) {
                        T.nph -= m * rsqrt_approx(d2);
                    }
                }
            }
        }
    }
}

__device__ __forceinline__ void eval_pp(target& T, const float (*pp)[TILE], const int* ppj, int part, int k,
                                        long long rowbase, int* rowcnt, const force_args& A, bool emit)
{
    uint32_t nearblocks = 0;                     // bit b: this lane's target came within r_out of block b
#pragma unroll 2
    for (int e = 4 * part; e < TILE; e += 4 * k) {
        ulonglong2 v[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) v[r] = *reinterpret_cast<const ulonglong2*>(&pp[r][e]);
        float dmin = pp_far_pair(T, v[0].x, v[1].x, v[2].x, v[3].x, A.K.rlist2, INFINITY);
        dmin = pp_far_pair(T, v[0].y, v[1].y, v[2].y, v[3].y, A.K.rlist2, dmin);
        if (dmin < A.K.rlist2) nearblocks |= 1u << (e >> 2);
    }
    if (!__any_sync(0xffffffffu, nearblocks != 0)) return;
    pp_near_pass(T, pp, ppj, nearblocks, rowbase, rowcnt, A, emit);
}

// Software pipeline of the list stream: the ids of tile t+2 and the node / particle data of tile
// t+1 are in flight while tile t is evaluated; nothing is consumed before the evaluation is over
// (the quadrupole is negated on its way to shared memory, not at the load).
struct pc_regs { float4 c, q0; float2 q1; };
struct pp_regs { float4 p; int j; };

// list ids and the group record were written by another SM during this kernel: read them past L1 (a line of glist
// holds eight groups, some of them not yet published when the line is first fetched)
__device__ __forceinline__ int load_id(const int32_t* ids, int e, int n) { return e < n ? __ldcg(ids + e) : -1; }

__device__ __forceinline__ pc_regs gather_pc(const force_args& A, int id)
{
    pc_regs r;
    P3T_CHECK(id < A.info->n_nodes);
    if (id >= 0) { r.c = A.ncom[id]; r.q0 = A.nq0[id]; r.q1 = A.nq1[id]; }
    else {                                     // padding: a zero-mass cell far away contributes exactly 0
        r.c = make_float4(FAR_AWAY, FAR_AWAY, FAR_AWAY, 0.0f); r.q0 = make_float4(0, 0, 0, 0); r.q1 = make_float2(0, 0);
    }
    return r;
}
__device__ __forceinline__ void store_pc(float (*pc)[TILE], int lane, const pc_regs& r)
{
    pc[0][lane] = r.c.x; pc[1][lane] = r.c.y; pc[2][lane] = r.c.z; pc[3][lane] = r.c.w;
    pc[4][lane] = -r.q0.x; pc[5][lane] = -r.q0.y; pc[6][lane] = -r.q0.z; pc[7][lane] = -r.q0.w;
    pc[8][lane] = -r.q1.x; pc[9][lane] = -r.q1.y;
}
__device__ __forceinline__ pp_regs gather_pp(const force_args& A, int id)
{
    pp_regs r; r.j = id;
    P3T_CHECK(id < A.n);
    if (id >= 0) r.p = A.spm[id]; else r.p = make_float4(FAR_AWAY, FAR_AWAY, FAR_AWAY, 0.0f);
    return r;
}
__device__ __forceinline__ void store_pp(float (*pp)[TILE], int* ppj, int lane, const pp_regs& r)
{
    pp[0][lane] = r.p.x; pp[1][lane] = r.p.y; pp[2][lane] = r.p.z; pp[3][lane] = r.p.w; ppj[lane] = r.j;
}

__device__ __forceinline__ double shfl_xor_double(double v, int o)
{
    int lo = __double2loint(v), hi = __double2hiint(v);
    lo = __shfl_xor_sync(0xffffffffu, lo, o); hi = __shfl_xor_sync(0xffffffffu, hi, o);
    return __hiloint2double(hi, lo);
}

// targets [tb, te) (sorted positions, te - tb <= 32) of group g against the group's two lists.
// SPLIT (small problems, fewer items than resident warps): the item is shared by nseg warps, warp
// `seg` takes the tiles seg, seg + nseg, ... of both lists; the partial sums go to A.part and are
// added in segment order by k_force_final (bit-reproducible), the row cursors are global.
template <bool SPLIT, bool MONO>
__device__ void force_item(const force_args& A, tile_smem& S, int g, int tb, int te, int seg, int nseg, bool emit, bool kick)
{
    const int lane = threadIdx.x & 31;
    const int c = te - tb;
    const int kshift = c > 16 ? 0 : c > 8 ? 1 : c > 4 ? 2 : 3;     // k = 1, 2, 4, 8 lanes per target
    const int k = 1 << kshift, part = lane & (k - 1);
    target T;
    T.slot = lane >> kshift;
    const bool v = T.slot < c;
    const float4 p = A.spm[v ? tb + T.slot : tb];
    T.x = p.x; T.y = p.y; T.z = p.z;
    T.id = v ? tb + T.slot : -1;
    T.dax = T.day = T.daz = T.dph = 0.0;
    T.ph = pk(0.0f, 0.0f);
    T.axe = T.aye = T.aze = T.axo = T.ayo = T.azo = 0.0f;
    T.nax = T.nay = T.naz = T.nph = 0.0f;
    const uint32_t orig = v ? A.order[T.id] : 0u;
    const long long rowbase = v ? A.nboff[orig] : 0;
    int* rowcnt = SPLIT ? A.nbcnt + (v ? T.id : tb) : &S.nbrow[T.slot];
    if (!SPLIT) S.nbrow[lane] = 0;
    // Only lane 0 has read the group's state word with an acquire (group_state); the shuffle that hands the state to the
    // other lanes orders no memory.  This warp barrier does: every read of what the walker published for the group --
    // the list record below and the list entries after it -- comes behind it in every lane.
    __syncwarp();
    const uint4 rec = __ldcg(&A.glist[g]);
    // ---- a8: particle-cell list; a lane sees TILE / k cells per tile: fold every k tiles ----
    {
        const int32_t* ids = A.pcpool + ((long long)rec.x << 5);
        const int n = (int)rec.y, nt = (n + TILE - 1) / TILE;
        P3T_CHECK(((long long)rec.x << 5) + (long long)nt * TILE <= A.pc_size);
        if (seg < nt) {
            pc_regs r = gather_pc(A, load_id(ids, seg * TILE + lane, n));
            int idn = load_id(ids, (seg + nseg) * TILE + lane, n);
            store_pc(S.pc[0], lane, r);
            __syncwarp();
            for (int t = seg, it = 0; t < nt; t += nseg, ++it) {
                const bool more = t + nseg < nt;
                if (more) r = gather_pc(A, idn);
                idn = load_id(ids, (t + 2 * nseg) * TILE + lane, n);
                if (MONO) eval_pc_mono(T, S.pc[it & 1], part, k); else eval_pc(T, S.pc[it & 1], part, k);
                if (((it + 1) & (k - 1)) == 0) fold(T);
                if (more) store_pc(S.pc[(it + 1) & 1], lane, r);
                __syncwarp();
            }
            fold(T);
        }
    }
    // ---- a9: particle-particle list (cutoff, neighbour emission): fold every 2k tiles ----
    {
        const int32_t* ids = A.pppool + ((long long)rec.z << 5);
        const int n = (int)rec.w, nt = (n + TILE - 1) / TILE;
        P3T_CHECK(((long long)rec.z << 5) + (long long)nt * TILE <= A.pp_size);
        if (seg < nt) {
            pp_regs r = gather_pp(A, load_id(ids, seg * TILE + lane, n));
            int idn = load_id(ids, (seg + nseg) * TILE + lane, n);
            store_pp(S.pp[0], S.ppj[0], lane, r);
            __syncwarp();
            for (int t = seg, it = 0; t < nt; t += nseg, ++it) {
                const bool more = t + nseg < nt;
                const int b = it & 1;
                if (more) r = gather_pp(A, idn);
                idn = load_id(ids, (t + 2 * nseg) * TILE + lane, n);
                eval_pp(T, S.pp[b], S.ppj[b], part, k, rowbase, rowcnt, A, emit);
                if (((it + 1) & (2 * k - 1)) == 0) fold(T);
                if (more) store_pp(S.pp[b ^ 1], S.ppj[b ^ 1], lane, r);
                __syncwarp();
            }
            fold(T);
        }
    }
    // ---- the parts of a target are adjacent lanes: sum them (fixed order) ----
    for (int o = 1; o < k; o <<= 1) {
        T.dax += shfl_xor_double(T.dax, o); T.day += shfl_xor_double(T.day, o);
        T.daz += shfl_xor_double(T.daz, o); T.dph += shfl_xor_double(T.dph, o);
    }
    if (!(v && part == 0)) return;
    if (SPLIT) {
        double* q = A.part + ((size_t)seg * (size_t)A.n + orig) * 4;
        q[0] = T.dax; q[1] = T.day; q[2] = T.daz; q[3] = T.dph;
        return;
    }
    // ---- a11: results to the caller's order ----
    const float4 a = make_float4((float)T.dax, (float)T.day, (float)T.daz, (float)T.dph);
    A.out[orig] = a;
    if (A.vel && kick) {                        // eq. 12: xdot += (dt_reg / 2) F_R, one fma per component
        float4 u = A.vel[orig];
        u.x = fmaf(A.half_dt, a.x, u.x); u.y = fmaf(A.half_dt, a.y, u.y); u.z = fmaf(A.half_dt, a.z, u.z);
        A.vel[orig] = u;
    }
}

// SPLIT epilogue (a11): the segments of every particle in segment order, then the kick.  In the host's repair pass
// (A.mode 1) only the particles of redone groups are kicked, and -- unless every group was evaluated again (A.evalall) --
// only they are written: the result of a group that was complete after the first pass stays as it is (the octupole
// variant has already added its term to it, and p3t_launch_octupole_add visits the same set of groups as this kernel).
__global__ void __launch_bounds__(256) k_force_final(force_args A, int n, const int32_t* __restrict__ rank)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || (A.info->bad_input | A.info->node_overflow)) return;
    bool redone = true;
    if (A.mode == 1) {                                          // the group of particle i: last g with gbegin[g] <= rank[i]
        const int sp = rank[i];
        int lo = 0, hi = A.info->n_groups;
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (A.gbegin[mid] <= sp) lo = mid; else hi = mid; }
        const int st = A.gready[lo] - A.base;
        redone = st == G_REDONE;
        if (!(redone || (A.evalall && st == G_READY))) return;
    }
    double s[4] = { 0, 0, 0, 0 };
    for (int g = 0; g < A.nseg; ++g) {
        const double* q = A.part + ((size_t)g * n + i) * 4;
        s[0] += q[0]; s[1] += q[1]; s[2] += q[2]; s[3] += q[3];
    }
    const float4 a = make_float4((float)s[0], (float)s[1], (float)s[2], (float)s[3]);
    A.out[i] = a;
    const bool kick = A.vel != nullptr && redone;
    if (kick) {
        float4 u = A.vel[i];
        u.x = fmaf(A.half_dt, a.x, u.x); u.y = fmaf(A.half_dt, a.y, u.y); u.z = fmaf(A.half_dt, a.z, u.z);
        A.vel[i] = u;
    }
}

// State of group g's lists for the item a warp has drawn.  The list walk (k_walk<WALK_LISTS>) runs at the same time on
// the SM share the host left to it and publishes every group with a release; lane 0 waits here with an acquire.
// Returns base + G_READY / G_FAILED / G_REDONE.  A wait that lasts longer than any walk can (no walker is resident:
// another process holds the SMs) gives the group up -- it is marked failed, spin_abort makes every other waiting warp
// give up at once, and the host's repair pass redoes those groups -- so the kernel always terminates.
#define SPIN_TIMEOUT (1ll << 27)                 // SM cycles (~70 ms)
__device__ __forceinline__ int group_state(const force_args& A, int g)
{
    int v = ld_acquire_gpu(&A.gready[g]);
    if (A.mode == 1 || g_decided(v, A.base)) return v;
    const long long t0 = clock64();
    for (;;) {
        __nanosleep(200);
        v = ld_acquire_gpu(&A.gready[g]);
        if (g_decided(v, A.base)) return v;
        if (*(volatile int32_t*)&A.info->spin_abort || clock64() - t0 > SPIN_TIMEOUT) {
            *(volatile int32_t*)&A.info->spin_abort = 1;
            const int old = atomicCAS(&A.gready[g], v, A.base + G_FAILED);
            if (old == v) return A.base + G_FAILED;
            if (g_decided(old, A.base)) return old;            // the walker published in between
        }
    }
}

// Work items: the c <= 64 targets of a group are cut into chunks of 32, 32, 16 and c mod 16 targets
// (25 .. 31 left-over targets stay together), which run with k = 1, 1, 2 and 2 / 4 / 8 lanes per target: every chunk but the last fills its
// warp, and a chunk costs list length / k.  Persistent grid, dynamic
// scheduling; the chunks are handed out in four passes, k = 1 first and k = 8 last, so that the
// kernel ends on its cheapest items and the warps finish together.  The kernel is launched twice per call on the
// same cursor: on the SMs' share that the list walk leaves free, and again (behind the walk, in its stream) on the rest.
template <bool SPLIT, bool MONO>
__global__ void __launch_bounds__(FORCE_THREADS, FORCE_CTAS_PER_SM) k_force(force_args A)
{
    __shared__ tile_smem smem[FORCE_WARPS];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    tile_smem& S = smem[w];
    // an invalid build or a failed count walk (its offsets size the rows): nothing is written, the host reports it
    if (A.info->bad_input | A.info->node_overflow | A.info->stack_overflow) return;
    // the neighbour total is final (the offset scan precedes this kernel): rows are emitted only if they fit
    const bool emit = (long long)A.info->nb_total <= A.nb_cap;
    if (!emit && threadIdx.x == 0) A.info->nb_overflow = 1;
    const int ng = A.info->shard_g1 - A.info->shard_g0;          // all groups unless the context is sharded (p3t_shard.cu)
    // cursor ranges of the passes: [0, 2 ng) chunks 0-1 (k = 1), [2 ng, 3 ng) chunk 2 (k = 2), [3 ng, 4 ng) chunk 3 (the rest)
    for (;;) {
        int c = 0;
        if (lane == 0) c = (int)atomicAdd(&A.info->group_cursor3, 1u);
        c = __shfl_sync(0xffffffffu, c, 0);
        int seg = 0;
        if (SPLIT) { seg = c % A.nseg; c /= A.nseg; }          // the segments of an item are handed out together
        if (c >= 4 * ng) break;
        int g, j;
        if (c < 2 * ng)      { g = c >> 1; j = c & 1; }
        else if (c < 3 * ng) { g = c - 2 * ng; j = 2; }
        else                 { g = c - 3 * ng; j = 3; }
        g += A.info->shard_g0;
        const int gb = A.gbegin[g], n = A.gbegin[g + 1] - gb;
        const int full = n >> 5, r = n & 31;
        int tb, len;
        if (j < 2)       { tb = 32 * j;                len = j < full ? 32 : 0; }
        else if (j == 2) { tb = 32 * full;             len = r >= 25 ? r : (r & 16); }      // 25..31 left over: one k = 1 item costs the same as 16 + rest
        else             { tb = 32 * full + (r & 16);  len = r >= 25 ? 0 : (r & 15); }
        if (len == 0) continue;
        int st = 0;
        if (lane == 0) st = group_state(A, g) - A.base;
        st = __shfl_sync(0xffffffffu, st, 0);
        const bool run = A.mode == 0 ? st == G_READY : (st == G_REDONE || (A.evalall && st == G_READY));
        if (!run) continue;
        force_item<SPLIT, MONO>(A, S, g, gb + tb, gb + tb + len, seg, SPLIT ? A.nseg : 1, emit, A.mode == 0 || st == G_REDONE);
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

// Rows ascending in original id, out of place (ids inside a row are distinct).  Each lane rank-sorts its own short
// row (<= 16 entries); rows of 17 .. 32 are rank-sorted by the warp; longer rows (a King core has hundreds of
// entries per row, and the rank sort is quadratic) go through a bitonic network in the warp's shared memory, up
// to SORT_SMEM entries; beyond that the quadratic sort again (not met by the paper's workloads).
#define SORTROWS_THREADS 128
#define SORT_SMEM 2048
// LONG = false: no row is longer than 32 (the host knows the longest row): no shared memory, full occupancy.
template <bool LONG>
__global__ void __launch_bounds__(SORTROWS_THREADS) k_nb_sortrows(const long long* __restrict__ off, const int32_t* __restrict__ raw,
                                                                  int32_t* __restrict__ idx, int n, long long cap, const p3t_devinfo* info)
{
    __shared__ int32_t s_row[LONG ? SORTROWS_THREADS / 32 : 1][LONG ? SORT_SMEM : 1];
    const int i = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    if ((long long)info->nb_total > cap || (info->bad_input | info->node_overflow | info->stack_overflow)) return;   // nothing was emitted
    int32_t* s = s_row[LONG ? threadIdx.x >> 5 : 0];
    long long b = 0; int len = 0;
    if (i < n) { b = off[i]; len = (int)(off[i + 1] - b); P3T_CHECK(b >= 0 && len >= 0 && b + len <= cap); }
    if (len <= 16) {                              // the row in registers: one load per entry, then the quadratic rank
        int v[16];
#pragma unroll
        for (int a = 0; a < 16; ++a) v[a] = a < len ? raw[b + a] : 0x7fffffff;
#pragma unroll
        for (int a = 0; a < 16; ++a) {
            if (a < len) {
                int r = 0;
#pragma unroll
                for (int c = 0; c < 16; ++c) r += v[c] < v[a];
                idx[b + r] = v[a];
            }
        }
    }
    uint32_t m = __ballot_sync(0xffffffffu, len > 16);
    while (m) {
        const int src = __ffs(m) - 1; m &= m - 1;
        const long long rb = __shfl_sync(0xffffffffu, b, src);
        const int rl = __shfl_sync(0xffffffffu, len, src);
        if (!LONG || rl <= 32 || rl > SORT_SMEM) {
            for (int a = lane; a < rl; a += 32) {
                const int v = raw[rb + a]; int r = 0;
                for (int c = 0; c < rl; ++c) r += raw[rb + c] < v;
                idx[rb + r] = v;
            }
            continue;
        }
        int P = 64;
        while (P < rl) P <<= 1;
        for (int a = lane; a < P; a += 32) s[a] = a < rl ? raw[rb + a] : 0x7fffffff;
        __syncwarp();
        for (int k = 2; k <= P; k <<= 1)
            for (int j = k >> 1; j > 0; j >>= 1) {
                for (int t = lane; t < (P >> 1); t += 32) {
                    const int lo = 2 * t - (t & (j - 1)), hi = lo + j;        // the t-th pair of this stage
                    const int x = s[lo], y = s[hi];
                    const bool up = (lo & k) == 0;
                    if ((x > y) == up) { s[lo] = y; s[hi] = x; }
                }
                __syncwarp();
            }
        for (int a = lane; a < rl; a += 32) idx[rb + a] = s[a];
        __syncwarp();
    }
}


// ---------------------------------------------------------------------------------------------
// Host side of a7-a11.  One call = p3t_force_begin (everything enqueued, no host synchronisation) + p3t_force_finish
// (the call's one synchronisation, error report, repair of what an undersized buffer left out).
//
//   main stream:  reset | count walk, offset scan (a10) | k_force on (4 - w) CTAs per SM ............ | final, row sort
//   walk stream:        | k_walk<LISTS> on w CTAs per SM (a7) ........ | k_force again on those w CTAs |
//
// The force kernel is FP32-pipe-bound with issue slots to spare, the list walk is issue- and latency-bound with the
// FP32 pipe nearly idle: side by side on every SM the walk disappears behind the evaluation.  The force kernel draws
// groups in the order the walkers produce them and waits for a group's state word (group_state).
// Buffers whose size depends on the result (list pools, neighbour indices) are sized from the previous call with
// head-room; a call that outgrows them marks what it could not do (G_FAILED groups, nb_overflow) and p3t_force_finish
// redoes exactly that with larger buffers (normally only on the first call of a context).
// ---------------------------------------------------------------------------------------------
#include <atomic>
static std::atomic<int> g_overlap_owner[64];      // per device: one overlapped call at a time in this process (two force
                                                  // kernels waiting for two walks could fill the SMs and starve both walks)

static int force_streams(p3t_ctx* ctx)
{
    if (ctx->walk_stream) return P3T_OK;
    P3T_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->walk_stream, cudaStreamNonBlocking));
    P3T_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_tree, cudaEventDisableTiming));
    P3T_CUDA(ctx, cudaEventCreate(&ctx->ev_scan));                 // also the end of the count phase (p3t_stats::ms_count)
    P3T_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_wdone, cudaEventDisableTiming));
    return P3T_OK;
}

static void force_fill(p3t_ctx* ctx, force_args& A, int mode, int evalall)
{
    const p3t_pending& q = ctx->pend;
    A.spm = P<float4>(ctx->spm); A.order = P<uint32_t>(ctx->idx[0]);
    A.ncom = P<float4>(ctx->ncom); A.nq0 = P<float4>(ctx->nq0); A.nq1 = P<float2>(ctx->nq1);
    A.gbegin = P<int32_t>(ctx->gbegin); A.glist = P<uint4>(ctx->glist);
    A.pcpool = P<int32_t>(ctx->pcpool); A.pppool = P<int32_t>(ctx->pppool);
    A.nboff = P<int64_t>(ctx->nboff); A.nbraw = P<int32_t>(ctx->stage_out);      // unsorted rows
    A.out = q.acc_pot; A.info = INFO(ctx);
    make_consts(A.K, q.r_out, q.r_in, q.theta, q.pot_mode, q.r_list);
    A.vel = q.vel; A.half_dt = q.half_dt; A.mp_order = ctx->order;
    A.gready = P<int32_t>(ctx->gready); A.base = ctx->epoch; A.mode = mode; A.evalall = evalall; A.nb_cap = ctx->nb_cap;
    A.pc_size = (long long)(ctx->pcpool.bytes / 4); A.pp_size = (long long)(ctx->pppool.bytes / 4);
    A.n = (int)ctx->n; A.nbcnt = P<int32_t>(ctx->nbcnt); A.part = P<double>(ctx->part);
    // A problem with fewer work items (about 1.4 per 32 particles) than three per resident warp shares every item
    // among nseg warps (SPLIT), so that small N still fills the GPU.
    // (the nominal 4 CTAs per SM, not the occupancy ptxas happened to leave: nseg fixes the order of the partial sums,
    // so the bits of the result must not move with the register count of a build -- the -DP3T_CHECKS build has 3)
    const long long warps = 4ll * ctx->num_sms * FORCE_WARPS;
    const long long items = (long long)ctx->n / ctx->shard_nranks * 14 / 320 + 1;
    int nseg = 1;
    while (nseg < 8 && items * nseg < 3 * warps) nseg *= 2;
    A.nseg = nseg;
}

static void force_launch(const force_args& A, bool mono, int blocks, cudaStream_t st)
{
    if (A.nseg > 1) {
        if (mono) k_force<true, true><<<blocks, FORCE_THREADS, 0, st>>>(A);
        else      k_force<true, false><<<blocks, FORCE_THREADS, 0, st>>>(A);
    } else {
        if (mono) k_force<false, true><<<blocks, FORCE_THREADS, 0, st>>>(A);
        else      k_force<false, false><<<blocks, FORCE_THREADS, 0, st>>>(A);
    }
}

// what follows the force kernel on the main stream: SPLIT epilogue, octupole variant, row sort
static int force_tail(p3t_ctx* ctx, const force_args& A, int mode, int evalall)
{
    const int n = (int)ctx->n;
    int rc;
    if (A.nseg > 1) {
        k_force_final<<<(n + 255) / 256, 256, 0, ctx->stream>>>(A, n, P<int32_t>(ctx->rank));
        ctx->launches += 1;
    }
    P3T_CUDA(ctx, cudaEventRecord(ctx->evw[1], ctx->stream));
    if (ctx->order == 3 && (rc = p3t_launch_octupole_add(ctx, ctx->pend.acc_pot, ctx->pend.half_dt, ctx->pend.vel, ctx->epoch, mode, evalall))) return rc;
    // rows ascending (any variant sorts every row correctly; the hint only picks the faster one)
    if (ctx->nb_max_hint > 32) k_nb_sortrows<true><<<(n + SORTROWS_THREADS - 1) / SORTROWS_THREADS, SORTROWS_THREADS, 0, ctx->stream>>>(P<long long>(ctx->nboff), A.nbraw, P<int32_t>(ctx->nbidx), n, A.nb_cap, INFO(ctx));
    else                       k_nb_sortrows<false><<<(n + SORTROWS_THREADS - 1) / SORTROWS_THREADS, SORTROWS_THREADS, 0, ctx->stream>>>(P<long long>(ctx->nboff), A.nbraw, P<int32_t>(ctx->nbidx), n, A.nb_cap, INFO(ctx));
    P3T_CUDA(ctx, cudaGetLastError());
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[5], ctx->stream));
    ctx->launches += 1;
    return P3T_OK;
}

static int reserve_split(p3t_ctx* ctx, const force_args& A)
{
    if (A.nseg <= 1) return P3T_OK;
    int rc;
    if ((rc = p3t_reserve(ctx, &ctx->nbcnt, (size_t)ctx->n * 4))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->part, (size_t)A.nseg * ctx->n * 32))) return rc;
    return P3T_OK;
}

int p3t_force_begin(p3t_ctx* ctx, float r_out, float r_in, float theta, int pot_mode, float4* acc_pot,
                    float r_list, float half_dt, float4* vel)
{
    const int n = (int)ctx->n;
    int rc;
    if (!ctx->occ_force) {
        P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->occ_force, k_force<false, false>, FORCE_THREADS, 0));
        if (ctx->occ_force < 1) ctx->occ_force = 1;
    }
    if ((rc = force_streams(ctx))) return rc;
    p3t_pending& q = ctx->pend;
    q.r_out = r_out; q.r_in = r_in; q.theta = theta; q.r_list = r_list; q.half_dt = half_dt; q.pot_mode = pot_mode;
    q.acc_pot = acc_pot; q.vel = vel; q.active = 1; q.repaired = 0; q.flags = 0;
    // ---- every buffer before anything is enqueued (a reallocation synchronises the stream) ----
    const int nsb = (n + SCAN_TILE - 1) / SCAN_TILE;
    if ((rc = p3t_reserve(ctx, &ctx->nbcount, (size_t)n * 4))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->nboff, ((size_t)n + 1) * 8))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->nbcur, (size_t)nsb * 8 + 64))) return rc;
    if (ctx->gready.bytes < ((size_t)n + 2) * 4 || ctx->epoch > 0x3fffff00) {
        if ((rc = p3t_reserve(ctx, &ctx->gready, ((size_t)n + 2) * 4))) return rc;
        P3T_CUDA(ctx, cudaMemsetAsync(ctx->gready.p, 0, ctx->gready.bytes, ctx->stream));
        ctx->epoch = 0;
    }
    ctx->epoch += 4;
    if (ctx->nb_cap == 0) ctx->nb_cap = 4ll * n > (1ll << 20) ? 4ll * n : (1ll << 20);      // first call: a guess (mean row of 4)
    if (ctx->nb_total_host + ctx->nb_total_host / 4 + 4096 > ctx->nb_cap) ctx->nb_cap = ctx->nb_total_host + ctx->nb_total_host / 4 + 4096;
    if ((rc = p3t_reserve(ctx, &ctx->nbidx, (size_t)ctx->nb_cap * 4 + 64))) return rc;
    if ((rc = p3t_reserve(ctx, &ctx->stage_out, (size_t)ctx->nb_cap * 4 + 64))) return rc;
    // overlapped unless switched off, or another context of this process is in the middle of an overlapped call
    int overlapped = ctx->overlap && ctx->occ_force >= 2;
    if (overlapped) {
        int expect = 0;
        overlapped = g_overlap_owner[ctx->device & 63].compare_exchange_strong(expect, 1) ? 1 : 0;
    }
    q.overlapped = overlapped;
    if (overlapped) q.flags |= P3T_FF_OVERLAPPED;
    int wsm = overlapped ? ctx->walk_ctas_per_sm : 0;
    if (wsm >= ctx->occ_force) wsm = ctx->occ_force - 1;
    if ((rc = p3t_walk_reserve(ctx, wsm))) return rc;
    force_args A;
    force_fill(ctx, A, 0, 0);
    if ((rc = reserve_split(ctx, A))) return rc;
    A.nbcnt = P<int32_t>(ctx->nbcnt); A.part = P<double>(ctx->part);
    const bool mono = ctx->order < 2;
    cudaStream_t ms = ctx->stream, ws = overlapped ? ctx->walk_stream : ctx->stream;

    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[4], ms));
    if (ctx->shard_nranks > 1) {
        // a sharded context walks only its own groups: rows and list lengths of the others are empty
        P3T_CUDA(ctx, cudaMemsetAsync(ctx->nbcount.p, 0, (size_t)n * 4, ms));
        P3T_CUDA(ctx, cudaMemsetAsync(ctx->gnpp.p, 0, ((size_t)n + 1) * 4, ms));
        P3T_CUDA(ctx, cudaMemsetAsync(ctx->gnpc.p, 0, ((size_t)n + 1) * 4, ms));
    }
    if (A.nseg > 1) {
        P3T_CUDA(ctx, cudaMemsetAsync(ctx->nbcnt.p, 0, (size_t)n * 4, ms));
        P3T_CUDA(ctx, cudaMemsetAsync(ctx->part.p, 0, (size_t)A.nseg * n * 32, ms));   // a segment beyond a short list writes nothing
    }
    if ((rc = p3t_launch_walk_reset(ctx, ms))) return rc;
    if (ctx->test_fault & 1) P3T_CUDA(ctx, cudaMemsetAsync((char*)ctx->info.p + offsetof(p3t_devinfo, spin_abort), 1, 1, ms));
    // a7 on the walk stream, from now on
    if (overlapped) {
        P3T_CUDA(ctx, cudaEventRecord(ctx->ev_tree, ms));
        P3T_CUDA(ctx, cudaStreamWaitEvent(ws, ctx->ev_tree, 0));
        P3T_CUDA(ctx, cudaEventRecord(ctx->evw[2], ws));
        if ((rc = p3t_launch_walk_lists(ctx, r_list, theta, ws, ctx->epoch, 0, wsm))) return rc;
        P3T_CUDA(ctx, cudaEventRecord(ctx->evw[3], ws));
    }
    // a10, sizes: neighbour counts (range search only) -> CSR offsets, so that the lists can be written in place
    if ((rc = p3t_launch_walk_count(ctx, r_list, theta, ms))) return rc;
    k_nb_blocksum<<<nsb, 256, 0, ms>>>(P<int32_t>(ctx->nbcount), n, P<long long>(ctx->nbcur), INFO(ctx));
    k_nb_scansums<<<1, 1024, 0, ms>>>(P<long long>(ctx->nbcur), nsb, P<long long>(ctx->nboff) + n, INFO(ctx));
    k_nb_offsets<<<nsb, 256, 0, ms>>>(P<int32_t>(ctx->nbcount), n, P<long long>(ctx->nbcur), P<long long>(ctx->nboff));
    P3T_CUDA(ctx, cudaGetLastError());
    ctx->launches += 3;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev_scan, ms));
    if (!overlapped) {
        P3T_CUDA(ctx, cudaEventRecord(ctx->evw[2], ms));
        if ((rc = p3t_launch_walk_lists(ctx, r_list, theta, ms, ctx->epoch, 0, 0))) return rc;
        P3T_CUDA(ctx, cudaEventRecord(ctx->evw[3], ms));
    }
    // a8, a9, a11: the force kernel, on the SMs' share the walk leaves free; again behind the walk on the rest
    P3T_CUDA(ctx, cudaEventRecord(ctx->evw[0], ms));
    force_launch(A, mono, (ctx->occ_force - wsm) * ctx->num_sms, ms);
    ctx->launches += 1;
    if (overlapped) {
        P3T_CUDA(ctx, cudaStreamWaitEvent(ws, ctx->ev_scan, 0));
        force_launch(A, mono, wsm * ctx->num_sms, ws);
        ctx->launches += 1;
        P3T_CUDA(ctx, cudaEventRecord(ctx->ev_wdone, ws));
        P3T_CUDA(ctx, cudaStreamWaitEvent(ms, ctx->ev_wdone, 0));
    }
    P3T_CUDA(ctx, cudaGetLastError());
    return force_tail(ctx, A, 0, 0);
}

void p3t_force_abandon(p3t_ctx* ctx)
{
    p3t_pending& q = ctx->pend;
    if (q.active) { (void)cudaStreamSynchronize(ctx->stream); q.active = 0; }
    if (q.overlapped) { g_overlap_owner[ctx->device & 63].store(0); q.overlapped = 0; }
}

int p3t_force_finish(p3t_ctx* ctx)
{
    p3t_pending& q = ctx->pend;
    if (!q.active) return P3T_OK;
    q.active = 0;
    p3t_devinfo h;
    cudaError_t e = cudaMemcpyAsync(&h, ctx->info.p, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (q.overlapped) { g_overlap_owner[ctx->device & 63].store(0); q.overlapped = 0; }
    if (e != cudaSuccess) return p3t_fail_cuda(ctx, e, "force call", __LINE__);
    int rc;
    for (int attempt = 0;; ++attempt) {
        if (h.bad_input) return P3T_EINVAL;
        if (h.node_overflow || h.stack_overflow) {
            snprintf(ctx->err, sizeof(ctx->err), "internal capacity exceeded (node_overflow=%d stack_overflow=%d)", h.node_overflow, h.stack_overflow);
            return P3T_ECUDA;
        }
        ctx->nb_total_host = (long long)h.nb_total;
        ctx->nb_max_hint = h.nb_max;
        if (!h.pool_overflow && !h.nb_overflow && !h.spin_abort) break;
        if (attempt >= 4) { snprintf(ctx->err, sizeof(ctx->err), "list buffers still too small after %d repair passes", attempt); return P3T_ECUDA; }
        // ---- repair pass (stream order, no overlap): larger buffers, every list again, then only what is missing ----
        q.repaired = 1; q.flags |= P3T_FF_REPAIRED;
        if (h.spin_abort && !(ctx->test_fault & 1)) {
            // force warps waited ~70 ms for a walker that never became resident: this context stops overlapping
            // rather than paying that wait at every step (reported in p3t_stats::force_flags)
            q.flags |= P3T_FF_SPIN_ABORT; ctx->overlap = 0;
        }
        const int evalall = h.nb_overflow ? 1 : 0;
        if (h.pool_overflow) {
            ctx->pool_cap_pc = (((long long)h.need_pc + h.need_pc / 4 + 16384) + 31) & ~31ll;
            ctx->pool_cap_pp = (((long long)h.need_pp + h.need_pp / 4 + 16384) + 31) & ~31ll;
        }
        if (h.nb_overflow) {
            ctx->nb_cap = ctx->nb_total_host + ctx->nb_total_host / 4 + 4096;
            if ((rc = p3t_reserve(ctx, &ctx->nbidx, (size_t)ctx->nb_cap * 4 + 64))) return rc;
            if ((rc = p3t_reserve(ctx, &ctx->stage_out, (size_t)ctx->nb_cap * 4 + 64))) return rc;
        }
        const int wsm = ctx->overlap && ctx->occ_force >= 2 ? (ctx->walk_ctas_per_sm >= ctx->occ_force ? ctx->occ_force - 1 : ctx->walk_ctas_per_sm) : 0;
        if ((rc = p3t_launch_walk_reset(ctx, ctx->stream))) return rc;       // cursors and counters; nb_total / nb_max are restored below
        P3T_CUDA(ctx, cudaEventRecord(ctx->evw[2], ctx->stream));
        if ((rc = p3t_launch_walk_lists(ctx, q.r_list, q.theta, ctx->stream, ctx->epoch, 1, wsm))) return rc;
        P3T_CUDA(ctx, cudaEventRecord(ctx->evw[3], ctx->stream));
        p3t_devinfo h2;
        P3T_CUDA(ctx, cudaMemcpyAsync(&h2, ctx->info.p, sizeof(h2), cudaMemcpyDeviceToHost, ctx->stream));
        P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        h2.nb_total = h.nb_total; h2.nb_max = h.nb_max;
        P3T_CUDA(ctx, cudaMemcpyAsync((char*)ctx->info.p + offsetof(p3t_devinfo, nb_total), &h.nb_total, sizeof(h.nb_total), cudaMemcpyHostToDevice, ctx->stream));
        P3T_CUDA(ctx, cudaMemcpyAsync((char*)ctx->info.p + offsetof(p3t_devinfo, nb_max), &h.nb_max, sizeof(h.nb_max), cudaMemcpyHostToDevice, ctx->stream));
        if (h2.pool_overflow || h2.stack_overflow) { h2.nb_overflow = h.nb_overflow; h = h2; continue; }     // still too small: measured again
        force_args A;
        force_fill(ctx, A, 1, evalall);
        if ((rc = reserve_split(ctx, A))) return rc;
        A.nbcnt = P<int32_t>(ctx->nbcnt); A.part = P<double>(ctx->part);
        P3T_CUDA(ctx, cudaEventRecord(ctx->evw[0], ctx->stream));
        force_launch(A, ctx->order < 2, ctx->occ_force * ctx->num_sms, ctx->stream);
        ctx->launches += 1;
        P3T_CUDA(ctx, cudaGetLastError());
        if ((rc = force_tail(ctx, A, 1, evalall))) return rc;
        P3T_CUDA(ctx, cudaMemcpyAsync(&h, ctx->info.p, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
        P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return P3T_OK;
}
