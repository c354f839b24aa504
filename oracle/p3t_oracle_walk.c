/* oracle/p3t_oracle_walk.c -- TEST INFRASTRUCTURE (see p3t_oracle.h).
 * Part II continued: opening rule (R-S7) and evaluation (R-S8) of the reference octree.
 * Compile with -ffp-contract=off.
 */
#include "p3t_oracle_tree_priv.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

static inline float max3f(float a, float b, float c)
{
    float m = a > b ? a : b;
    return m > c ? m : c;
}

/* R-S7 opening rule.  Inputs are fp32 values; every operation is one IEEE fp32 rounding in this
 * order, no contraction except the explicit fmaf:
 *   e_a = max(0, glo_a - COM_a, COM_a - ghi_a);  d2 = fma(e_z, e_z, fma(e_y, e_y, e_x*e_x))
 *   f_a = max(0, glo_a - chi_a, clo_a - ghi_a);  b2 = fma(f_z, f_z, fma(f_y, f_y, f_x*f_x))
 *   u = fl(fl(l / theta) + delta);  open <=> d2 < fl(u*u)  OR  b2 < fl(r_out*r_out)
 * First clause: Barnes-Hut angle test with the Bonsai-style offset delta (theta).
 * Second clause: the "modification ... to populate the neighbour list": no cell
 * is accepted unless its particles all lie beyond r_out of every target in the group, so every
 * particle-cell term is wholly regular and all neighbours are met particle by particle. */
int p3t_o_open_test(const float glo[3], const float ghi[3], const float com[3], const float clo[3],
                    const float chi[3], float l, float delta, float theta, float r_out)
{
    float e[3], f[3];
    for (int a = 0; a < 3; ++a) {
        e[a] = max3f(0.0f, glo[a] - com[a], com[a] - ghi[a]);
        f[a] = max3f(0.0f, glo[a] - chi[a], clo[a] - ghi[a]);
    }
    float d2 = fmaf(e[2], e[2], fmaf(e[1], e[1], e[0] * e[0]));
    float b2 = fmaf(f[2], f[2], fmaf(f[1], f[1], f[0] * f[0]));
    float lt = l / theta;
    float u = lt + delta;
    float rc2 = u * u;
    float ro2 = r_out * r_out;
    return (d2 < rc2) || (b2 < ro2);
}

/* R-S8 particle-cell term: monopole + traceless quadrupole of a cell seen from x_i, fp64
 * arithmetic on the fp32-rounded node data.  r = x_i - COM, R = |r|:
 *   phi = -M/R - (1/2) r.Q.r / R^5
 *   a   = -M r/R^3 + Q.r/R^5 - (5/2) (r.Q.r) r / R^7                                     */
void p3t_o_pc_term(const double xi[3], const float com_m[4], const float q[6], double out[4])
{
    double r[3] = { xi[0] - (double)com_m[0], xi[1] - (double)com_m[1], xi[2] - (double)com_m[2] };
    double M = com_m[3];
    double R2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2], R = sqrt(R2);
    double Qr[3] = { (double)q[0] * r[0] + (double)q[3] * r[1] + (double)q[4] * r[2],
                     (double)q[3] * r[0] + (double)q[1] * r[1] + (double)q[5] * r[2],
                     (double)q[4] * r[0] + (double)q[5] * r[1] + (double)q[2] * r[2] };
    double rQr = r[0] * Qr[0] + r[1] * Qr[1] + r[2] * Qr[2];
    double R3 = R2 * R, R5 = R3 * R2, R7 = R5 * R2;
    out[3] = -M / R - 0.5 * rQr / R5;
    for (int a = 0; a < 3; ++a) out[a] = -M * r[a] / R3 + Qr[a] / R5 - 2.5 * rQr * r[a] / R7;
}

/* SURVEY 8f NEXT-4, octupole variant: the third-order term of the same Taylor expansion.  With the raw third
 * moment T_abc = sum m d_a d_b d_c about the COM (order xxx yyy zzz xxy xxz xyy yyz xzz yzz xyz), r = x_i - COM:
 *   1/|r - d| = ... + (5/2) (d.r)^3 / R^7 - (3/2) |d|^2 (d.r) / R^5 + O(d^4)
 *   t3 = T_abc r_a r_b r_c,  v_a = T_abc r_b r_c,  tau_a = T_bba,  u = tau.r
 *   phi_3 = -(5/2) t3 / R^7 + (3/2) u / R^5
 *   a_3   = -grad phi_3 = (15/2) v / R^7 - (35/2) t3 r / R^9 - (3/2) tau / R^5 + (15/2) u r / R^7
 * fp64 arithmetic on the fp32-rounded node data; ADDED to out. */
void p3t_o_pc_octupole(const double xi[3], const float com_m[4], const float T[10], double out[4])
{
    const double r[3] = { xi[0] - (double)com_m[0], xi[1] - (double)com_m[1], xi[2] - (double)com_m[2] };
    const double x = r[0], y = r[1], z = r[2];
    const double xxx = T[0], yyy = T[1], zzz = T[2], xxy = T[3], xxz = T[4], xyy = T[5], yyz = T[6], xzz = T[7], yzz = T[8], xyz = T[9];
    /* v_a = T_abc r_b r_c */
    const double v[3] = {
        xxx * x * x + xyy * y * y + xzz * z * z + 2.0 * (xxy * x * y + xxz * x * z + xyz * y * z),
        xxy * x * x + yyy * y * y + yzz * z * z + 2.0 * (xyy * x * y + xyz * x * z + yyz * y * z),
        xxz * x * x + yyz * y * y + zzz * z * z + 2.0 * (xyz * x * y + xzz * x * z + yzz * y * z) };
    const double tau[3] = { xxx + xyy + xzz, xxy + yyy + yzz, xxz + yyz + zzz };
    const double t3 = v[0] * x + v[1] * y + v[2] * z;
    const double u = tau[0] * x + tau[1] * y + tau[2] * z;
    const double R2 = x * x + y * y + z * z, R = sqrt(R2), R5 = R2 * R2 * R, R7 = R5 * R2, R9 = R7 * R2;
    out[3] += -2.5 * t3 / R7 + 1.5 * u / R5;
    for (int a = 0; a < 3; ++a) out[a] += 7.5 * v[a] / R7 - 17.5 * t3 * r[a] / R9 - 1.5 * tau[a] / R5 + 7.5 * u * r[a] / R7;
}

typedef struct { int32_t* v; int64_t n, cap; } ilist;
static void il_push(ilist* l, int32_t x)
{
    if (l->n == l->cap) { l->cap = l->cap ? 2 * l->cap : 4096; l->v = realloc(l->v, sizeof(int32_t) * l->cap); }
    l->v[l->n++] = x;
}

static void walk(const p3t_o_tree* t, int64_t g, int64_t node, float theta, float r_out, ilist* pc, ilist* pp)
{
    float l = t->side / (float)(1ull << t->level[node]);          /* power of two: exact */
    int open = p3t_o_open_test(t->glo + 3 * g, t->ghi + 3 * g, t->fcom_m + 4 * node, t->clo + 3 * node,
                               t->chi + 3 * node, l, t->delta[node], theta, r_out);
    if (!open) { il_push(pc, (int32_t)node); return; }             /* one p-c entry for the whole group */
    if (t->n_child[node] == 0) {                                   /* opened leaf: all its particles */
        for (int32_t i = t->begin[node]; i < t->end[node]; ++i) il_push(pp, i);
        return;
    }
    for (int c = 0; c < t->n_child[node]; ++c) walk(t, g, t->first_child[node] + c, theta, r_out, pc, pp);
}

void p3t_o_tree_force(const p3t_o_tree* t, float r_out_f, float r_in_f, float theta, int pot_mode,
                      int64_t ng, const int64_t* group_ids, double* acc_pot,
                      int64_t* npp, int64_t* npc, double* abs_sum)
{
    p3t_o_tree_force_buffered(t, r_out_f, r_out_f, r_in_f, theta, pot_mode, ng, group_ids, acc_pot, npp, npc, abs_sum);
}

/* SURVEY 8f NEXT-2, PAPER.md:113 (section 2.3, R_cut = R_s + R_buff) and eq. 20 (:156): the neighbour
 * search reaches r_list = r_out + r_buff >= r_out, so the second clause of the opening rule uses
 * r_list; the force itself is unchanged (cutoff between r_in and r_out). */
void p3t_o_tree_force_buffered(const p3t_o_tree* t, float r_list_f, float r_out_f, float r_in_f, float theta, int pot_mode,
                               int64_t ng, const int64_t* group_ids, double* acc_pot,
                               int64_t* npp, int64_t* npc, double* abs_sum)
{
    p3t_o_tree_force_order(t, 2, r_list_f, r_out_f, r_in_f, theta, pot_mode, ng, group_ids, acc_pot, npp, npc, abs_sum);
}

/* the variants for the accuracy-throughput curve.  order 2 = monopole + quadrupole
 * (north_star), order 1 = the same walk with the quadrupole of every accepted cell left out (R-S8 with Q = 0:
 * phi = -M/R, a = -M r/R^3), order 3 = the same walk with the octupole term of every accepted cell added. */
void p3t_o_tree_force_order(const p3t_o_tree* t, int order, float r_list_f, float r_out_f, float r_in_f, float theta, int pot_mode,
                            int64_t ng, const int64_t* group_ids, double* acc_pot,
                            int64_t* npp, int64_t* npc, double* abs_sum)
{
    static const float zero_quad[6] = { 0, 0, 0, 0, 0, 0 };
    const double r_out = r_out_f, r_in = r_in_f, D = r_out - r_in;
    const double psi_in = p3t_o_psi(r_in, r_out, r_in);
#pragma omp parallel
    {
        ilist pc = { 0, 0, 0 }, pp = { 0, 0, 0 };
#pragma omp for schedule(dynamic, 4)
        for (int64_t q = 0; q < ng; ++q) {
            int64_t g = group_ids ? group_ids[q] : q;
            pc.n = pp.n = 0;
            walk(t, g, 0, theta, r_list_f, &pc, &pp);
            if (npp) npp[q] = pp.n;
            if (npc) npc[q] = pc.n;
            for (int32_t i = t->gbegin[g]; i < t->gend[g]; ++i) {
                const float* pi = t->spm + 4 * (int64_t)i;
                double xi[3] = { pi[0], pi[1], pi[2] };
                double a[3] = { 0, 0, 0 }, phi = 0, asum = 0;
                for (int64_t k = 0; k < pc.n; ++k) {
                    double o[4];
                    p3t_o_pc_term(xi, t->fcom_m + 4 * (int64_t)pc.v[k], order >= 2 ? t->fquad + 6 * (int64_t)pc.v[k] : zero_quad, o);
                    if (order >= 3) p3t_o_pc_octupole(xi, t->fcom_m + 4 * (int64_t)pc.v[k], t->foct + 10 * (int64_t)pc.v[k], o);
                    a[0] += o[0]; a[1] += o[1]; a[2] += o[2]; phi += o[3];
                    asum += sqrt(o[0] * o[0] + o[1] * o[1] + o[2] * o[2]);
                }
                for (int64_t k = 0; k < pp.n; ++k) {
                    int32_t j = pp.v[k];
                    if (j == i) continue;                           /* self excluded by index */
                    const float* pj = t->spm + 4 * (int64_t)j;
                    double dx = pj[0] - xi[0], dy = pj[1] - xi[1], dz = pj[2] - xi[2], m = pj[3];
                    double r2 = dx * dx + dy * dy + dz * dz;
                    if (r2 == 0.0) { if (pot_mode == 0) phi += m * psi_in; continue; }   /* reading R8 */
                    double r = sqrt(r2), w, ps;
                    if (r >= r_out) { w = 1.0; ps = -1.0 / r; }
                    else if (r <= r_in) { w = 0.0; ps = psi_in; }
                    else { w = p3t_o_W((r - r_in) / D); ps = p3t_o_psi(r, r_out, r_in); }
                    double f = m * w / (r2 * r);
                    a[0] += f * dx; a[1] += f * dy; a[2] += f * dz;
                    phi += pot_mode == 0 ? m * ps : -m / r;
                    asum += fabs(f) * r;
                }
                int64_t orig = t->order[i];
                acc_pot[4 * orig] = a[0]; acc_pot[4 * orig + 1] = a[1]; acc_pot[4 * orig + 2] = a[2]; acc_pot[4 * orig + 3] = phi;
                if (abs_sum) abs_sum[orig] = asum;
            }
        }
        free(pc.v); free(pp.v);
    }
}
