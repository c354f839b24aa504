/* include/p3t.h -- C-ABI of the B200-native P3T regular-force library (libp3t.so).
 *
 * The library computes the data-parallel hot path of NBODY6+P3T (Arnold, Baumgardt & Wang,
 * arXiv:2110.11658; citations are /root/reference/PAPER.md:<line>): for every particle i
 *
 *     F_R,i = sum_{j != i} m_j (x_j - x_i) / |r_ij|^3 * (1 - K_ij)          (eq. 1, 3, 4)
 *
 * with the 7th-order cutoff K(x), x = (r - r_in)/(r_out - r_in) (eq. 6, 8-10; PAPER.md:52-66;
 * the paper's r_cut is called r_out here), evaluated with a Barnes-Hut octree with opening angle
 * theta, together with each particle's neighbour list { j != i : r_ij < r_out }
 * that the CPU Hermite/KS side consumes.  G = 1.
 * The readings taken where the paper is silent (sign of eq. 4, potential, opening rule, ...) are
 * listed in DESIGN.md (R-numbers).
 *
 * Conventions
 *  - Every call returns P3T_OK (0) or a negative error code; no exceptions, no exit, no stdout.
 *  - "DEVICE pointer": memory of the context's CUDA device.  "HOST pointer": ordinary host memory
 *    (pinned or pageable).  "ANY pointer": either one (copied with cudaMemcpyDefault).
 *  - Calls enqueue work on the context's stream and do NOT synchronise unless stated.  p3t_build_tree does not;
 *    p3t_regular_force / _ex synchronise once, at their end (see there); the accessors synchronise.
 *  - The library never frees caller memory and writes only to the output arguments named below.
 *  - One context per host thread; a context is bound to one device and one stream.
 *  - Every step runs in the library's CUDA kernels; there is no CPU fallback.
 */
#ifndef P3T_H
#define P3T_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define P3T_OK       0
#define P3T_EINVAL  -1   /* bad argument: n < 1, n > P3T_MAX_N, r_in < 0, r_in >= r_out, theta <= 0,
                            key_bits not 30/63, null pointer, NaN/Inf position or mass, negative mass
                            (found by the bounding-cube reduction of p3t_build_tree; reported by the next
                            synchronising call, p3t_regular_force included, which then writes nothing) */
#define P3T_ESTATE  -2   /* force before build, neighbours before force, ... */
#define P3T_ENOMEM  -3   /* device allocation failed */
#define P3T_ECUDA   -4   /* a CUDA call failed; sticky; text via p3t_last_error */
#define P3T_ERANGE  -5   /* p3t_neighbours_nbody6: a row is longer than lmax */

#define P3T_MAX_N   (1ll << 30)
#define P3T_MAX_NCRIT 64
#define P3T_MAX_RANKS 64   /* p3t_set_shard */

typedef struct p3t_ctx p3t_ctx;      /* opaque; owns all device scratch */

/* Sizes and timings of the last build / force call (p3t_get_stats synchronises the stream). */
typedef struct p3t_stats {
    int64_t n;               /* particles                                               */
    int64_t n_nodes;         /* octree cells                                            */
    int64_t n_leaves;
    int64_t n_groups;        /* target groups of the walk                               */
    int32_t max_level;
    int32_t key_bits;
    int64_t n_pp;            /* sum over targets of particle-particle terms evaluated   */
    int64_t n_pc;            /* sum over targets of particle-cell terms evaluated       */
    int64_t n_pp_list;       /* sum over groups of p-p list lengths                     */
    int64_t n_pc_list;       /* sum over groups of p-c list lengths                     */
    int64_t nb_total;        /* neighbour-list entries                                  */
    int32_t nb_max;          /* longest row                                             */
    int32_t input_bad;       /* 1 if the last build saw a NaN/Inf position or mass      */
    float   cube_lo[3];      /* bounding cube (DESIGN.md R-S1)                          */
    float   cube_side;
    float   ms_build;        /* CUDA-event time of the last p3t_build_tree (a1-a6)      */
    float   ms_force;        /* CUDA-event time of the last p3t_regular_force (a7-a11)  */
    float   ms_walk;         /* ... of its list-building tree walk kernel (a7), which runs beside the force kernel */
    float   ms_sort;         /* ... of the radix sort inside the last build             */
    float   ms_eval;         /* ... of the force kernel (a8, a9, a11), first launch to the end of the second */
    float   ms_count;        /* ... of the neighbour count walk + offset scan (a10)     */
    float   ms_irregular;    /* ... of the last p3t_irregular_force kernel (0 if none)  */
    float   ms_core;         /* ... of the last p3t_core_quantities kernels (0 if none)  */
    int64_t launches;        /* kernels this context has launched since p3t_create      */
    float   ms_octupole;     /* ... of the octupole add kernel of the last force (order 3; else 0) */
    int32_t force_flags;     /* how the last force call ran: P3T_FF_* bits                */
} p3t_stats;

#define P3T_FF_OVERLAPPED 1  /* the list walk ran beside the force kernel (the normal case; not when another context of the
                                process had an overlapped call in flight on the device, or after P3T_FF_SPIN_ABORT)          */
#define P3T_FF_REPAIRED   2  /* a buffer sized from the previous call was too small: part of the call was redone (normally
                                only the first call of a context; costs up to a second pass)                                */
#define P3T_FF_SPIN_ABORT 4  /* force warps stopped waiting for the list walk (~70 ms: no walker was resident, e.g. another
                                process filled the SMs); the call was repaired and the context runs its later calls without
                                the overlap, instead of paying that wait every step                                         */

/* Create a context on CUDA device `device`, enqueuing on `cuda_stream` (a cudaStream_t passed as
 * void*; NULL = the legacy default stream).  *out is set on success. */
int p3t_create(p3t_ctx** out, int device, void* cuda_stream);
int p3t_destroy(p3t_ctx* ctx);

/* Tree parameters (DESIGN.md R-S4/R-S5): a cell with more than nleaf particles is split;
 * target groups hold at most ncrit particles.  1 <= nleaf <= ncrit <= P3T_MAX_NCRIT.
 * Defaults 16 / 64.  Takes effect at the next build. */
int p3t_set_tree_params(p3t_ctx* ctx, int nleaf, int ncrit);

/* Multipole order of the particle-cell terms: 2 = monopole + quadrupole (default, north_star), 1 = monopole
 * only (a cheaper point on the accuracy-throughput curve: same walk and lists, the
 * quadrupole of the accepted cells left out), 3 = + octupole (a more accurate point: the third-order term of
 * the same Taylor expansion, from the raw third moments sum m d_a d_b d_c about each cell's centre of mass,
 * added for every accepted cell of the same lists).  Orders 1 and 2 take effect at the next
 * p3t_regular_force; order 3 needs the third moments, which p3t_build_tree computes when the order is 3:
 * p3t_regular_force returns P3T_ESTATE until the tree has been built with that order set. */
int p3t_set_multipole_order(p3t_ctx* ctx, int order);

/* Multi-GPU (PAPER.md:277-291 names it as future work): the path shards by target group
 * with no data-path collective.  Every rank calls p3t_build_tree with ALL n bodies (the build is
 * deterministic, so all ranks hold the identical tree) and p3t_regular_force then walks and evaluates only
 * the groups of this rank: those whose first sorted particle lies in [cut_rank, cut_rank+1), where cut_r is
 * the first group boundary at or after a nominal sorted position -- r n / nranks when nominal_cuts is NULL,
 * else nominal_cuts[r] (HOST int64[nranks + 1], copied; e.g. balanced by the previous step's list lengths).
 * In a sharded context p3t_regular_force writes acc_pot (and kicks vel) only for the owned particles --
 * the other entries are unspecified -- neighbour rows and list lengths of the other particles / groups
 * are empty, and the statistics count the own interactions.  nranks = 1 restores the whole path.
 * 1 <= nranks <= P3T_MAX_RANKS, 0 <= rank < nranks.  Takes effect at the next p3t_build_tree. */
int p3t_set_shard(p3t_ctx* ctx, int rank, int nranks, const int64_t* nominal_cuts);

/* The group-aligned cuts of ALL ranks after p3t_build_tree, identical on every rank: cuts_host[r]
 * (HOST int64[nranks + 1]) = first sorted position of rank r, cuts_host[nranks] = n; group_cuts_host
 * (HOST int32[nranks + 1], may be NULL) = the same as group indices.  Synchronises.  P3T_ESTATE if the
 * context is not sharded or not built. */
int p3t_get_shard_cuts(p3t_ctx* ctx, int64_t* cuts_host, int32_t* group_cuts_host);

/* The exchange step: p3t_shard_pack gathers the owned entries of a per-particle DEVICE float4[n] array in
 * original order (acc_pot of p3t_regular_force) into one contiguous DEVICE chunk of cuts[rank+1] - cuts[rank]
 * float4 in sorted order; p3t_shard_unpack scatters the chunk of rank from_rank (as received from it, e.g. by
 * an NCCL all-gather) back into original order.  After unpacking every rank's chunk the array is complete and
 * equal, bit for bit, to that of an unsharded context.  16-byte aligned pointers.  Do not synchronise. */
int p3t_shard_pack(p3t_ctx* ctx, const void* acc_pot, void* chunk);
int p3t_shard_unpack(p3t_ctx* ctx, int from_rank, const void* chunk, void* acc_pot);

/* Steps a1-a6: bounding cube, Morton keys (key_bits = 30 or 63), stable radix sort,
 * body permutation, canonical octree, monopole + traceless quadrupole moments, target groups.
 * pos_mass: DEVICE pointer, n x {x, y, z, m} fp32 (16-byte aligned), caller-owned, read-only;
 * it is copied (permuted) during the call and need not stay valid afterwards.
 * The paper names only "the BONSAI library" for this step. */
int p3t_build_tree(p3t_ctx* ctx, int64_t n, const float* pos_mass, int key_bits);

/* Steps a7-a11: group tree walk, particle-cell and particle-particle regular force with the cutoff
 * of eq. 6 and neighbour-list emission fused in.
 * acc_pot: DEVICE pointer, n x {ax, ay, az, phi} fp32, caller-owned, ORIGINAL particle order.
 * pot_mode 0: phi = regular potential (its gradient is -a; R6); 1: unsplit Newtonian
 * potential -sum m_j / r_ij.  Requires a prior build; theta, r_out, r_in may change between
 * calls without a rebuild.  Also produces the neighbour lists returned by p3t_neighbours.
 * r_in = 0 is legal (the cutoff then reaches down to r = 0); masses of 0 are legal (tracers; DESIGN.md R-S6a).
 * SYNCHRONISES the stream once, at its end: the whole call is enqueued first (the list walk runs on a second
 * stream of the context beside the force kernel and is joined back), then the host waits, so that on return
 * acc_pot, vel and the lists are complete and every error of the build or the walk is reported by THIS call:
 * P3T_EINVAL for NaN/Inf/negative input (nothing was written, vel is not kicked), P3T_ECUDA for an exceeded
 * internal capacity (walk stack, cell count: outputs unspecified).  List buffers sized by the previous call that
 * turn out too small are regrown and the missing part is redone inside the call (normally only the first call). */
int p3t_regular_force(p3t_ctx* ctx, float r_out, float r_in, float theta, int pot_mode, float* acc_pot);

/* p3t_regular_force with the neighbour search reaching r_list = r_out + r_buff
 * (PAPER.md:113, section 2.3: R_cut = R_s + R_buff; eq. 20, :156: r_buff = 3 tau sigma) and the leapfrog
 * half-kick of eq. 12 fused into the epilogue of the force kernel:
 *     L(i) = { j != i : r_ij < r_list },  r_list = fl32(r_out + r_buff)   (the cutoff stays at r_in, r_out:
 *     list members with r >= r_out contribute wholly to F_R and nothing to F_I);
 *     vel_i += half_dt * F_R,i   (one fma per component on the fp32 acceleration that is returned).
 * r_buff >= 0.  vel: DEVICE pointer, n x {vx, vy, vz, unused} fp32, ORIGINAL order, 16-byte aligned,
 * updated in place; NULL = no kick.  Everything else as p3t_regular_force (= r_buff 0, vel NULL). */
int p3t_regular_force_ex(p3t_ctx* ctx, float r_out, float r_in, float theta, int pot_mode, float r_buff,
                         float half_dt, float* vel, float* acc_pot);

/* The same call in two halves, for a host that has work of its own to do meanwhile: in the paper's loop (steps
 * (i)-(vi)) the CPU integrates the irregular forces between two regular steps, and Fig. 7
 * puts half of the wall time there.  p3t_regular_force_begin checks the arguments, enqueues the whole
 * call ("calls enqueue on the context's stream and do not synchronise") and returns;
 * p3t_regular_force_wait synchronises once, reports the errors listed above, redoes what an undersized buffer left
 * out, and only then are acc_pot, vel and the neighbour lists complete.  Between the two the caller must not touch
 * acc_pot / vel; a build, a step, a second begin or p3t_set_shard on this context returns P3T_ESTATE, and so do
 * the list accessors (the lists are not there yet); p3t_destroy is allowed and drains the call.
 * A begin that fails has drained whatever it had enqueued; no wait is needed (a wait with nothing pending returns
 * P3T_ESTATE).  p3t_regular_force_ex is exactly begin followed by wait. */
int p3t_regular_force_begin(p3t_ctx* ctx, float r_out, float r_in, float theta, int pot_mode, float r_buff,
                            float half_dt, float* vel, float* acc_pot);
int p3t_regular_force_wait(p3t_ctx* ctx);

/* core quantities by a sampled k-nearest-neighbour search (PAPER.md:134, :245:
 * "a random sample of min(N, sqrt(5000 N)) particles, then ... those particles' 6 nearest neighbours";
 * estimator of Casertano & Hut 1985 as cited there; R17-R19).  The search runs on the octree
 * of the last p3t_build_tree and returns exactly the brute-force neighbours under the order
 * (fp32 squared distance of R10, original index).
 * sample: DEVICE pointer, ns original ids (the caller draws the random sample); 2 <= k <= 16 (paper: 6).
 * nbr: DEVICE, ns x k int32 original ids, ascending in that order (may be NULL); d2k: DEVICE, ns fp32,
 * squared distance of the k-th neighbour; rho: DEVICE, ns fp64, (sum of the masses of the k-1 nearest) /
 * (4 pi / 3 r_k^3).  core_out: HOST double[6] = density centre sum rho x / sum rho (3), R_core =
 * sqrt(sum rho^2 |x - x_d|^2 / sum rho^2), rho_core = sum rho^2 / sum rho, N_core = (n / ns) x the
 * number of sample particles within R_core of the centre.  Requires a prior build.  Synchronises. */
int p3t_core_quantities(p3t_ctx* ctx, int64_t ns, const int32_t* sample, int k, int32_t* nbr, float* d2k, double* rho,
                        double* core_out);

/* irregular force, jerk and potential over the neighbour lists of the last
 * p3t_regular_force (same r_out, r_in), eq. 1, 2, 5, 7 (the paper's CUTOFF / cutoff0
 * routines, :396-398):  F_I = sum_{j in L(i)} m_j K d / r^3,  Fdot_I = its exact time derivative
 * (R2: eq. 2 / 7 are garbled in the text),  phi_I = sum m_j (-1/r - psi(r)), so that
 * F_I + F_R and phi_I + phi_R (pot_mode 0) are the unsplit Newtonian sums.
 * vel: DEVICE pointer, n x {vx, vy, vz, unused} fp32, ORIGINAL order, caller-owned, read-only.
 * acc_irr: DEVICE, n x {ax, ay, az, phi_I}; jerk_irr: DEVICE, n x {jx, jy, jz, 0}; ORIGINAL order.
 * All three 16-byte aligned.  P3T_ESTATE without a prior p3t_regular_force.  Does not synchronise. */
int p3t_irregular_force(p3t_ctx* ctx, const float* vel, float* acc_irr, float* jerk_irr);

/* Neighbour lists L(i) = { j != i : r_ij < r_out } of the last
 * p3t_regular_force, as CSR in ORIGINAL particle ids: offsets[n+1] (int64), indices[total]
 * (int32, 0-based, every row strictly ascending, self excluded; empty rows are legal,
 * PAPER.md:113).  The pointers are library-owned DEVICE pointers, valid until the next
 * force/build/destroy.  Synchronises the stream (total is returned on the host). */
int p3t_neighbours(p3t_ctx* ctx, const int64_t** offsets, const int32_t** indices, int64_t* total);

/* Same lists copied out: offsets_out[n+1], indices_out[total]: ANY pointers (either may be NULL). */
int p3t_neighbours_copy(p3t_ctx* ctx, int64_t* offsets_out, int32_t* indices_out);

/* NBODY6-style view "in a format compatible with NBODY6": HOST array
 * n x (lmax + 1) int32; row i = { count, 1-based ids ascending, zero padding }.
 * P3T_ERANGE if a row is longer than lmax (nothing is written then). */
int p3t_neighbours_nbody6(p3t_ctx* ctx, int32_t lmax, int32_t* host_list);

/* One whole regular-force step with HOST buffers (what the host integrator calls once per
 * dt_reg, steps (i)/(iv) of PAPER.md:89-94): copies pos_mass host->device, builds, evaluates,
 * and copies acc_pot[n x 4] and the neighbour CSR back.  nb_offsets[n+1] and nb_indices[nb_cap]
 * may be NULL (lists are then left on the device).  *nb_total receives the entry count; if it
 * exceeds nb_cap the indices are not copied and P3T_ERANGE is returned.  Synchronises. */
int p3t_step_host(p3t_ctx* ctx, int64_t n, const float* pos_mass_host, int key_bits,
                  float r_out, float r_in, float theta, int pot_mode,
                  float* acc_pot_host, int64_t* nb_offsets_host, int32_t* nb_indices_host,
                  int64_t nb_cap, int64_t* nb_total);

/* Steps a1-a3 (bounding cube, Morton keys, stable radix sort: the same kernels and rules as p3t_build_tree,
 * "the BONSAI library" of PAPER.md:117-119) for callers that must not allocate device memory.
 *
 * Who that is.  Every other call of this library takes a p3t_ctx, and a context gets its scratch from cudaMalloc
 * (p3t_create, then grow-only).  Some hosts of an N-body integrator cannot afford that: a code that has handed
 * the whole device to its own arena or to a framework's caching allocator has nothing left for the runtime to
 * hand out; a regular-step loop that also runs an irregular-force stream does not want cudaMalloc / cudaFree in
 * it, because both stall every stream of the device while they run; and a plug-in loaded into a process under a
 * fixed device-memory quota may simply be forbidden to grow.  Such a caller can still get the Morton order of its
 * particles (to reorder its own arrays for locality, or to feed its own tree) from this one call: it needs no
 * context and calls no cudaMalloc, cudaFree or other allocating routine, at the first call or any later one.
 *
 * How.  The scratch the sort needs (its digit totals, tile tickets and look-back words, the cube record and the
 * second buffer of the key / index ping-pong) lives in ONE fixed array inside the library image, 3 678 976 bytes
 * (P3T_STATIC_SCRATCH_BYTES), sized for P3T_STATIC_MAX_N = 262 144 particles (the paper's own range, N = 32k ...
 * 256k).  Every GPU on which the process uses this library holds that array from the moment the
 * library's code is loaded on it until the process exits, whether or not this call is ever made.
 *
 *   pos_mass     DEVICE, n x {x, y, z, m} fp32, 16-byte aligned, read-only           (input)
 *   sorted_keys  DEVICE uint64[n]: the Morton keys in ascending order                (output; also used as the
 *   order        DEVICE uint32[n]: sorted position -> original id, ties keep           first ping-pong buffer, so
 *                original order (stable)                                               both are required)
 *   cube         DEVICE float[4] = {lo_x, lo_y, lo_z, side} of the bounding cube      (output, may be NULL)
 *   bad_input    DEVICE int32[1]: 1 if a position or mass is NaN / Inf or a mass       (output, may be NULL)
 *                is negative (keys and order are then unspecified), else 0
 * Results equal, bit for bit, p3t_get_keys / p3t_stats::cube_* after p3t_build_tree on the same input.
 *
 * device / cuda_stream: as in p3t_create (the call makes `device` current, like every call of the library, and
 * enqueues on that stream; it does NOT synchronise).  All pointers must belong to `device`.
 *
 * First call on a device: the call looks up the device address of the array (cudaGetSymbolAddress) and the SM
 * count, once per device, and keeps them.  That set-up does not allocate, but it is not stream work: make the
 * first call on each device from ordinary host code, before any stream capture that is to contain later calls.
 *
 * Sharing: all calls on a device use the same array, and it keeps what the last call left there.  The call
 * clears, on the stream, the part that has to start at zero, so calls that follow one another on ONE stream (or
 * are ordered by events) are independent of each other.  Two calls whose GPU work overlaps -- different streams
 * without an event between them, or two host threads -- race on the array and return garbage; ordering them is
 * the caller's job.  The set-up itself is safe to race (it is serialised inside the library).
 *
 * Errors: P3T_EINVAL for a null or misaligned pointer, n < 1, key_bits not 30 / 63, or an unknown device;
 * P3T_ELIMIT for n > P3T_STATIC_MAX_N (nothing is enqueued; use a context, which has no such limit);
 * P3T_ECUDA if a CUDA call fails (no context, hence no p3t_last_error text: cudaGetLastError has the cause). */
#define P3T_ELIMIT  -6   /* p3t_morton_order_static: n exceeds the capacity of the library's fixed scratch array */
#define P3T_STATIC_MAX_N          (1 << 18)
#define P3T_STATIC_SCRATCH_BYTES  3678976
int p3t_morton_order_static(int device, void* cuda_stream, int64_t n, const float* pos_mass, int key_bits,
                            uint64_t* sorted_keys, uint32_t* order, float* cube, int32_t* bad_input);

/* ---- parity / debug accessors: synchronise; outputs are ANY pointers sized from p3t_get_stats ---- */
int p3t_get_stats(p3t_ctx* ctx, p3t_stats* out);
/* sorted Morton keys [n] (30-bit keys are widened to uint64) and order[n] (sorted position -> original id) */
int p3t_get_keys(p3t_ctx* ctx, uint64_t* sorted_keys, uint32_t* order);
/* nodes in breadth-first order (levels ascending, begin ascending inside a level), each [n_nodes];
 * first_child = -1 and n_child = 0 for a leaf */
int p3t_get_nodes(p3t_ctx* ctx, int32_t* level, int32_t* begin, int32_t* end,
                  int32_t* first_child, int32_t* n_child);
/* fp32 node data: com_m [n_nodes x 4], quad [n_nodes x 6] (xx yy zz xy xz yz, traceless),
 * clo / chi [n_nodes x 3] tight box, delta [n_nodes] = |COM - geometric centre| */
int p3t_get_moments(p3t_ctx* ctx, float* com_m, float* quad, float* clo, float* chi, float* delta);
/* octupole variant: fp32 raw third moments about the COM [n_nodes x 10], order xxx yyy zzz xxy xxz xyy yyz xzz yzz xyz;
 * P3T_ESTATE unless the tree was built with multipole order 3 */
int p3t_get_octupoles(p3t_ctx* ctx, float* oct);
/* target groups as ranges of sorted positions, each [n_groups], ascending */
int p3t_get_groups(p3t_ctx* ctx, int32_t* begin, int32_t* end);
/* per-group list lengths of the last force call: npp[n_groups], npc[n_groups] (int32) */
int p3t_get_list_lengths(p3t_ctx* ctx, int32_t* npp, int32_t* npc);

const char* p3t_strerror(int code);
const char* p3t_last_error(p3t_ctx* ctx);     /* text of the last CUDA failure ("" if none) */

/* Host helper, eq. 20-25: tau = (1/128)(N/2^14)^(-1/3), r_cut = 4 tau,
 * r_buff = 3 tau sigma, dt_reg = largest 2^-k <= tau, dt_max = dt_reg / 4.  Any output may be NULL. */
int p3t_params_from_n(int64_t n, double sigma, double* tau, double* r_cut, double* r_buff,
                      double* dt_reg, double* dt_max);

#ifdef __cplusplus
}
#endif
#endif
