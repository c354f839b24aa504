/* oracle/p3t_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the P3T regular-force path computes,
 * written from /root/reference/PAPER.md (Arnold, Baumgardt & Wang, arXiv:2110.11658).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load it.  It shares no code with the CUDA library under
 * paper_2110_11658_b200/csrc and neither includes the other.
 *
 * Part I   (p3t_oracle_direct.c)  plain definitions: cutoff K/W (eq. 6), pair potential psi,
 *          direct O(N^2) split sums (eq. 1, 3, 4), brute-force neighbour lists.
 *          (p3t_oracle_grid.c)    the same neighbour lists with a uniform cell grid for large N.
 * Part II  (p3t_oracle_tree.c)    a reference octree, step by step: cube, Morton keys, order,
 *          canonical topology, moments, sibling-run groups, opening rule, evaluation.
 *          The paper names only the library (Bonsai) and theta; every
 *          rule of Part II is a DESIGN.md reading (R-numbers cited at each function).
 *
 * Pins: tests/test_oracle_*.py (-m "not gpu").  Unpinned: the opening rule itself (a design
 * choice; pinned only through theta->0 == direct sum and the direct-sum error bound).
 */
#ifndef P3T_ORACLE_H
#define P3T_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- Part I ---- */
double p3t_o_W(double x);                                   /* 1 - K(x), eq. 6      */
double p3t_o_dW(double x);                                  /* polynomial of eq. 7  */
double p3t_o_psi(double r, double r_out, double r_in);      /* -dpsi/dr = W/r^2, psi(inf) = 0   */

/* Direct sums for nt targets (indices into the n particles; NULL = all, nt = n).
 * pos_mass: n x {x,y,z,m} fp32.  Outputs (any may be NULL): acc_reg[3nt], phi_reg[nt],
 * acc_irr[3nt], phi_newt[nt]; returns the number of coincident (r = 0, j != i) pairs seen. */
int64_t p3t_o_direct(int64_t n, const float* pos_mass, double r_out, double r_in,
                     int64_t nt, const int64_t* targets,
                     double* acc_reg, double* phi_reg, double* acc_irr, double* phi_newt);

/* eq. 1, 2, 5, 7: irregular acceleration, jerk and potential over the neighbour sphere r_ij < r_out
 * (SURVEY 8f NEXT-1).  vel: n x 4 fp32.  Outputs (any may be NULL): acc_irr[3nt], jerk_irr[3nt],
 * phi_irr[nt], abs_jerk[nt] (sum of |jerk term|), abs_newt[nt] (sum of the K = 1 term sizes).
 * Returns the number of coincident pairs skipped. */
int64_t p3t_o_irregular(int64_t n, const float* pos_mass, const float* vel, double r_out, double r_in,
                        int64_t nt, const int64_t* targets,
                        double* acc_irr, double* jerk_irr, double* phi_irr, double* abs_jerk, double* abs_newt);

/* the same sums with the candidates j of every target restricted to caller-given CSR rows that contain its
 * neighbour sphere (cand_off[nt + 1], cand_idx; NULL = every j): same predicate, same arithmetic per pair */
int64_t p3t_o_irregular_cand(int64_t n, const float* pos_mass, const float* vel, double r_out, double r_in,
                             int64_t nt, const int64_t* targets, const int64_t* cand_off, const int32_t* cand_idx,
                             double* acc_irr, double* jerk_irr, double* phi_irr, double* abs_jerk, double* abs_newt);

/* sampled K-nearest-neighbour densities (Casertano & Hut 1985) and the core
 * quantities built from them.  sample: ns original ids.  nbr[ns*K] (may be NULL),
 * d2k[ns] fp32, rho[ns] fp64.  out[6] = density centre (3), R_core, rho_core, N_core. */
void p3t_o_knn_density(int64_t n, const float* pos_mass, int64_t ns, const int32_t* sample, int K,
                       int32_t* nbr, float* d2k, double* rho);
void p3t_o_core_quantities(int64_t n, const float* pos_mass, int64_t ns, const int32_t* sample, const double* rho, double out[6]);

/* Brute-force neighbour rows for nt targets.  fp32_predicate = 1: the bit-spec predicate
 * (R10); 0: the fp64 "physics" predicate r_ij < r_out.  counts[nt] is always written;
 * if indices != NULL rows are written back to back (ascending j) and must hold sum(counts). */
int64_t p3t_o_neighbours(int64_t n, const float* pos_mass, float r_out, int fp32_predicate,
                         int64_t nt, const int64_t* targets, int64_t* counts, int32_t* indices);

/* The same lists (fp32 predicate of R10) with the candidates restricted by a uniform cell grid of edge
 * >= 1.001 r_out, independent of the octree (p3t_oracle_grid.c): for the sizes at which the
 * double loop above takes hours.  Same outputs; returns the total or -1 (allocation failure, r_out <= 0). */
int64_t p3t_o_neighbours_grid(int64_t n, const float* pos_mass, float r_out,
                              int64_t nt, const int64_t* targets, int64_t* counts, int32_t* indices);

/* ---- Part II ---- */
typedef struct p3t_o_tree p3t_o_tree;

p3t_o_tree* p3t_o_tree_build(int64_t n, const float* pos_mass, int key_bits, int nleaf, int ncrit);
void        p3t_o_tree_free(p3t_o_tree* t);

/* sizes: out[0]=n, [1]=n_nodes, [2]=n_leaves, [3]=max_level, [4]=n_groups, [5]=bits per axis */
void p3t_o_tree_sizes(const p3t_o_tree* t, int64_t out[6]);
void p3t_o_tree_cube(const p3t_o_tree* t, float lo[3], float* side);
void p3t_o_tree_keys(const p3t_o_tree* t, uint64_t* sorted_keys, uint32_t* order);
/* nodes in breadth-first order, levels ascending, begin ascending inside a level */
void p3t_o_tree_nodes(const p3t_o_tree* t, int32_t* level, int32_t* begin, int32_t* end,
                      int32_t* first_child, int32_t* n_child);
/* fp32-rounded node data: com_m[4], quad[6] (xx,yy,zz,xy,xz,yz; traceless), clo[3], chi[3], delta */
void p3t_o_tree_moments(const p3t_o_tree* t, float* com_m, float* quad, float* clo, float* chi, float* delta);
/* unrounded fp64 moments: mass, com[3], quad[6] */
void p3t_o_tree_moments64(const p3t_o_tree* t, double* mass, double* com, double* quad);
/* raw third moments about the COM per node [nn][10]: fp32-rounded and fp64 (either may be NULL) */
void p3t_o_tree_octupoles(const p3t_o_tree* t, float* foct, double* oct);
void p3t_o_tree_groups(const p3t_o_tree* t, int32_t* begin, int32_t* end, float* glo, float* ghi);

/* Tree force for ng groups (ids into the group list; NULL = all).  acc_pot: n x 4 fp64 in
 * ORIGINAL particle order, only the rows of the targets in those groups are written.
 * npp/npc (may be NULL): per requested group, particles on the p-p list / cells on the p-c list.
 * pot_mode 0: regular potential, 1: unsplit Newtonian.  abs_sum (may be NULL): n fp64, per target
 * the sum over its interactions of |a_ij| (conditioning of the sum; R15). */
void p3t_o_tree_force(const p3t_o_tree* t, float r_out, float r_in, float theta, int pot_mode,
                      int64_t ng, const int64_t* group_ids, double* acc_pot,
                      int64_t* npp, int64_t* npc, double* abs_sum);

/* the same with a neighbour search radius r_list >= r_out in the opening rule */
void p3t_o_tree_force_buffered(const p3t_o_tree* t, float r_list, float r_out, float r_in, float theta, int pot_mode,
                               int64_t ng, const int64_t* group_ids, double* acc_pot,
                               int64_t* npp, int64_t* npc, double* abs_sum);

/* the same with the multipole order chosen: 2 = monopole + quadrupole, 1 = monopole only, 3 = + octupole */
void p3t_o_tree_force_order(const p3t_o_tree* t, int order, float r_list, float r_out, float r_in, float theta, int pot_mode,
                            int64_t ng, const int64_t* group_ids, double* acc_pot,
                            int64_t* npp, int64_t* npc, double* abs_sum);

/* single particle-cell term (fp64) from fp32 node data: out = {ax, ay, az, phi} */
void p3t_o_pc_term(const double xi[3], const float com_m[4], const float quad[6], double out[4]);
/* octupole term of the same expansion, ADDED to out; T = raw third moment about the COM, order xxx yyy zzz xxy xxz xyy yyz xzz yzz xyz */
void p3t_o_pc_octupole(const double xi[3], const float com_m[4], const float T[10], double out[4]);
/* the fp32 opening test alone (R7): returns 1 = open */
int  p3t_o_open_test(const float glo[3], const float ghi[3], const float com[3], const float clo[3],
                     const float chi[3], float l, float delta, float theta, float r_out);
/* Morton key of integer grid coordinates (x highest) */
uint64_t p3t_o_interleave(uint32_t gx, uint32_t gy, uint32_t gz, int bits);

#ifdef __cplusplus
}
#endif
#endif
