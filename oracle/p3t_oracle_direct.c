/* oracle/p3t_oracle_direct.c -- TEST INFRASTRUCTURE (see p3t_oracle.h).
 * Part I: the plain definitions.  fp64 throughout; inputs are the fp32 arrays the GPU gets
 * (fp32 -> fp64 is exact).  Compile with -ffp-contract=off.
 */
#include "p3t_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* eq. 6: K = 1 - {0 | -20x^7 + 70x^6 - 84x^5 + 35x^4 | 1}; W := 1 - K is the
 * regular weight.  Reading R3: K = 1 inside r_in, 0 outside r_cut. */
double p3t_o_W(double x)
{
    if (x <= 0.0) return 0.0;
    if (x >= 1.0) return 1.0;
    double x2 = x * x, x4 = x2 * x2;
    return -20.0 * x4 * x2 * x + 70.0 * x4 * x2 - 84.0 * x4 * x + 35.0 * x4;
}

/* the polynomial of eq. 7: -140x^6 + 420x^5 - 420x^4 + 140x^3 (= dW/dx) */
double p3t_o_dW(double x)
{
    if (x <= 0.0 || x >= 1.0) return 0.0;
    double x3 = x * x * x;
    return -140.0 * x3 * x3 + 420.0 * x3 * x * x - 420.0 * x3 * x + 140.0 * x3;
}

/* Pair potential of the regular force: psi(r) = -int_r^inf W(x(s)) / s^2 ds, with
 * x = (s - r_in)/(r_out - r_in) (eq. 8-10).  The paper defines no potential
 * (reading R6); this is the antiderivative written in closed form:
 *   integrate by parts, W' = 140 t^3 (1-t)^3, s = D (t + c), D = r_out - r_in, c = r_in / D:
 *   psi = -W/r - (140/D) * int_x^1 t^3 (1-t)^3 / (t + c) dt
 * and the integrand is a degree-5 quotient q(t) plus rem/(t + c) (synthetic division).
 * For r < r_in the regular force vanishes, so psi is the constant psi(r_in).           */
double p3t_o_psi(double r, double r_out, double r_in)
{
    if (r >= r_out) return -1.0 / r;
    if (r < r_in) r = r_in;
    double D = r_out - r_in, c = r_in / D, x = (r - r_in) / D;
    /* t^3 (1-t)^3 = -t^6 + 3 t^5 - 3 t^4 + t^3 ; divide by (t + c): root -c */
    double p[7] = { -1.0, 3.0, -3.0, 1.0, 0.0, 0.0, 0.0 };   /* t^6 .. t^0 */
    double q[6], carry = 0.0;
    for (int k = 0; k < 6; ++k) { q[k] = p[k] + carry; carry = -c * q[k]; }   /* q: t^5 .. t^0 */
    double rem = p[6] + carry;
    /* S(t) = int_0^t q */
    double S1 = 0.0, Sx = 0.0;
    for (int k = 0; k < 6; ++k) {
        int pw = 6 - k;                   /* q[k] t^(5-k) integrates to q[k] t^(6-k)/(6-k) */
        S1 += q[k] / pw;
        Sx += q[k] * pow(x, pw) / pw;
    }
    /* r_in = 0 (c = 0): the remainder -c^3 (1+c)^3 is exactly 0 and so is its term (the limit of rem ln(1/x), x -> 0;
     * written out so that 0 * inf never appears) */
    double integral = (S1 - Sx) + (rem != 0.0 ? rem * log((1.0 + c) / (x + c)) : 0.0);
    /* r = 0 is reached only with r_in = 0: W(x)/r ~ 35 x^4 / r -> 0 */
    return -(r > 0.0 ? p3t_o_W(x) / r : 0.0) - (140.0 / D) * integral;
}

/* eq. 1, 3, 4, G = 1.  Reading R1: attractive gravity, so the vector in the
 * force on i is x_j - x_i (eq. 4 as printed, x_i - x_j, would repel).
 *   F_I,i = sum_j m_j K d / r^3      F_R,i = sum_j m_j d / r^3 - F_I,i = sum_j m_j W d / r^3
 * Coincident pairs (r = 0, j != i; reading R8): no force either way, phi_R gets m psi(r_in),
 * phi_N skips them; they are counted in the return value.                               */
int64_t p3t_o_direct(int64_t n, const float* pm, double r_out, double r_in,
                     int64_t nt, const int64_t* targets,
                     double* acc_reg, double* phi_reg, double* acc_irr, double* phi_newt)
{
    int64_t coincident = 0;
    const double D = r_out - r_in;
    const double psi_in = p3t_o_psi(r_in, r_out, r_in);
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : coincident)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        double xi = pm[4 * i], yi = pm[4 * i + 1], zi = pm[4 * i + 2];
        double ar[3] = { 0, 0, 0 }, ai[3] = { 0, 0, 0 }, pr = 0.0, pn = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double dx = pm[4 * j] - xi, dy = pm[4 * j + 1] - yi, dz = pm[4 * j + 2] - zi;
            double m = pm[4 * j + 3];
            double r2 = dx * dx + dy * dy + dz * dz;
            if (r2 == 0.0) { coincident++; pr += m * psi_in; continue; }
            double r = sqrt(r2);
            double newt = m / (r2 * r);
            pn -= m / r;
            if (r >= r_out) {                      /* wholly regular */
                ar[0] += newt * dx; ar[1] += newt * dy; ar[2] += newt * dz;
                pr -= m / r;
            } else if (r <= r_in) {                /* wholly irregular */
                ai[0] += newt * dx; ai[1] += newt * dy; ai[2] += newt * dz;
                pr += m * psi_in;
            } else {
                double W = p3t_o_W((r - r_in) / D), K = 1.0 - W;
                ar[0] += newt * W * dx; ar[1] += newt * W * dy; ar[2] += newt * W * dz;
                ai[0] += newt * K * dx; ai[1] += newt * K * dy; ai[2] += newt * K * dz;
                pr += m * p3t_o_psi(r, r_out, r_in);
            }
        }
        if (acc_reg) { acc_reg[3 * t] = ar[0]; acc_reg[3 * t + 1] = ar[1]; acc_reg[3 * t + 2] = ar[2]; }
        if (acc_irr) { acc_irr[3 * t] = ai[0]; acc_irr[3 * t + 1] = ai[1]; acc_irr[3 * t + 2] = ai[2]; }
        if (phi_reg) phi_reg[t] = pr;
        if (phi_newt) phi_newt[t] = pn;
    }
    return coincident;
}

/* Neighbour list L(i) = { j != i : r_ij < r_out } ("if |r_ij| > r_cut the force counts
 * wholly as part of F_R", :113; strict inequality, reading R4; self excluded by index).
 * fp32 predicate (reading R10), every operation one IEEE fp32 rounding, no contraction:
 *   dx = fl(x_j - x_i) ...;  d2 = fma(dz, dz, fma(dy, dy, fl(dx*dx)));  member <=> d2 < fl(r_out*r_out) */
int64_t p3t_o_neighbours(int64_t n, const float* pm, float r_out, int fp32_predicate,
                         int64_t nt, const int64_t* targets, int64_t* counts, int32_t* indices)
{
    const float rout2f = r_out * r_out;
    const double rout_d = (double)r_out;
    int64_t total = 0;
    /* pass 1: counts */
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : total)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        float xi = pm[4 * i], yi = pm[4 * i + 1], zi = pm[4 * i + 2];
        int64_t c = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            int member;
            if (fp32_predicate) {
                float dx = pm[4 * j] - xi, dy = pm[4 * j + 1] - yi, dz = pm[4 * j + 2] - zi;
                float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                member = d2 < rout2f;
            } else {
                double dx = (double)pm[4 * j] - xi, dy = (double)pm[4 * j + 1] - yi, dz = (double)pm[4 * j + 2] - zi;
                member = sqrt(dx * dx + dy * dy + dz * dz) < rout_d;
            }
            c += member;
        }
        counts[t] = c;
        total += c;
    }
    if (!indices) return total;
    int64_t* off = (int64_t*)malloc(sizeof(int64_t) * (size_t)(nt + 1));
    off[0] = 0;
    for (int64_t t = 0; t < nt; ++t) off[t + 1] = off[t] + counts[t];
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        float xi = pm[4 * i], yi = pm[4 * i + 1], zi = pm[4 * i + 2];
        int64_t w = off[t];
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            int member;
            if (fp32_predicate) {
                float dx = pm[4 * j] - xi, dy = pm[4 * j + 1] - yi, dz = pm[4 * j + 2] - zi;
                float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                member = d2 < rout2f;
            } else {
                double dx = (double)pm[4 * j] - xi, dy = (double)pm[4 * j + 1] - yi, dz = (double)pm[4 * j + 2] - zi;
                member = sqrt(dx * dx + dy * dy + dz * dz) < rout_d;
            }
            if (member) indices[w++] = (int32_t)j;
        }
    }
    free(off);
    return total;
}

/* eq. 1, 2, 5, 7: irregular acceleration and its time derivative (jerk) of
 * nt targets, summed over j != i with r_ij < r_out (the neighbour sphere; K = 0 beyond it).
 * With d = x_j - x_i, v = xdot_j - xdot_i (readings R1: attraction; eq. 5 with the same sign
 * convention), r = |d|, x = (r - r_in)/(r_out - r_in), K = 1 - W:
 *     F_I    = sum m_j K d / r^3                                                   (eq. 1)
 *     Fdot_I = sum m_j [ K ( v / r^3 - 3 (d.v) d / r^5 ) + Kdot d / r^3 ]          (eq. 2)
 *     Kdot   = dK/dt = -W'(x) xdot,   xdot = (d.v) / (r (r_out - r_in)),
 *     W'(x)  = 140 x^3 (1-x)^3 = the polynomial of eq. 7.
 * Reading R2: eq. 2 as printed has K multiplying only the first term and eq. 7 gives
 * K' the opposite sign; Fdot_I here is the exact time derivative of eq. 1 (pinned by finite
 * differences in tests/test_oracle_irregular.py).  Coincident pairs (r = 0, reading R8) are skipped
 * (a KS pair in the host code) and counted in the return value.
 * vel: n x 4 fp32 (vx, vy, vz, unused).  Outputs (any may be NULL): acc_irr[3 nt], jerk_irr[3 nt],
 * phi_irr[nt] = sum m_j (-1/r - psi(r)); conditioning of the sums: abs_jerk[nt] = sum of |jerk term|,
 * abs_newt[nt] = sum m_j (|v|/r^3 + 3 |d.v|/r^4), the size of the unweighted (K = 1) jerk terms. */
/* one pair of the sums above, added to the accumulators of target i; returns 1 if the pair is coincident */
typedef struct { double a[3], jk[3], phi, ab, an; } irr_acc;
static int irr_pair(const float* pm, const float* vel, double r_out, double r_in, int64_t i, int64_t j, irr_acc* S)
{
    const double D = r_out - r_in;
    const double d[3] = { (double)pm[4 * j] - pm[4 * i], (double)pm[4 * j + 1] - pm[4 * i + 1], (double)pm[4 * j + 2] - pm[4 * i + 2] };
    const double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    if (r2 >= r_out * r_out) return 0;
    if (r2 == 0.0) return 1;
    const double v[3] = { (double)vel[4 * j] - vel[4 * i], (double)vel[4 * j + 1] - vel[4 * i + 1], (double)vel[4 * j + 2] - vel[4 * i + 2] };
    const double m = pm[4 * j + 3], r = sqrt(r2), r3 = r2 * r, r5 = r3 * r2;
    const double dv = d[0] * v[0] + d[1] * v[1] + d[2] * v[2];
    const double x = (r - r_in) / D;
    const double K = 1.0 - p3t_o_W(x);
    const double Kdot = -p3t_o_dW(x) * dv / (r * D);
    double tn = 0.0;
    for (int c = 0; c < 3; ++c) {
        S->a[c] += m * K * d[c] / r3;
        const double term = m * (K * (v[c] / r3 - 3.0 * dv * d[c] / r5) + Kdot * d[c] / r3);
        S->jk[c] += term; tn += term * term;
    }
    S->ab += sqrt(tn);
    S->an += m * (sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]) / r3 + 3.0 * fabs(dv) / (r2 * r2));
    S->phi += m * (-1.0 / r - p3t_o_psi(r, r_out, r_in));
    return 0;
}

/* cand_off / cand_idx (may be NULL = every j): a caller-given SUPERSET of the neighbour sphere of every target,
 * as CSR rows over the nt targets (e.g. the rows of p3t_o_neighbours_grid at a radius a little above r_out).
 * The predicate r2 < r_out^2 and the arithmetic of every pair are the same either way; the candidates only
 * spare the O(N) scan per target at N = 2^20. */
int64_t p3t_o_irregular_cand(int64_t n, const float* pm, const float* vel, double r_out, double r_in,
                             int64_t nt, const int64_t* targets, const int64_t* cand_off, const int32_t* cand_idx,
                             double* acc_irr, double* jerk_irr, double* phi_irr, double* abs_jerk, double* abs_newt)
{
    int64_t coincident = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : coincident)
    for (int64_t t = 0; t < nt; ++t) {
        const int64_t i = targets ? targets[t] : t;
        irr_acc S;
        memset(&S, 0, sizeof(S));
        if (cand_off) {
            for (int64_t e = cand_off[t]; e < cand_off[t + 1]; ++e) {
                const int64_t j = cand_idx[e];
                if (j != i) coincident += irr_pair(pm, vel, r_out, r_in, i, j, &S);
            }
        } else {
            for (int64_t j = 0; j < n; ++j)
                if (j != i) coincident += irr_pair(pm, vel, r_out, r_in, i, j, &S);
        }
        for (int c = 0; c < 3; ++c) {
            if (acc_irr) acc_irr[3 * t + c] = S.a[c];
            if (jerk_irr) jerk_irr[3 * t + c] = S.jk[c];
        }
        if (phi_irr) phi_irr[t] = S.phi;
        if (abs_jerk) abs_jerk[t] = S.ab;
        if (abs_newt) abs_newt[t] = S.an;
    }
    return coincident;
}

int64_t p3t_o_irregular(int64_t n, const float* pm, const float* vel, double r_out, double r_in,
                        int64_t nt, const int64_t* targets,
                        double* acc_irr, double* jerk_irr, double* phi_irr, double* abs_jerk, double* abs_newt)
{
    return p3t_o_irregular_cand(n, pm, vel, r_out, r_in, nt, targets, NULL, NULL, acc_irr, jerk_irr, phi_irr, abs_jerk, abs_newt);
}

/* core quantities by a sampled 6-nearest-neighbour search (section 2.5,
 * :245 section 3.2.1: "takes a random sample of min(N, sqrt(5000 N)) particles, then performs a
 * brute-force search for those particles' 6 nearest neighbours"; the estimator is Casertano & Hut 1985,
 * which the paper cites and does not restate: readings R17-R19 of DESIGN.md).
 *
 * Step 1, per sample particle i (brute force over all j != i, by index):
 *   the K nearest neighbours under the order (d2, j), d2 the fp32 squared distance of R10
 *   (dx = fl(x_j - x_i) ..., d2 = fma(dz,dz,fma(dy,dy,fl(dx dx)))): an integer decision, so it is taken
 *   in the kernel's precision on both sides; ties by the smaller original index;
 *   rho_i = (sum of the masses of the K-1 nearest) / (4 pi / 3 r_K^3),  r_K = sqrt(d2_K) in fp64
 *   (Casertano & Hut's unbiased estimator: the K-th neighbour and the particle itself are left out).
 * Outputs: nbr[ns*K] original ids in ascending (d2, j), d2k[ns] fp32 d2 of the K-th, rho[ns] fp64. */
void p3t_o_knn_density(int64_t n, const float* pm, int64_t ns, const int32_t* sample, int K,
                       int32_t* nbr, float* d2k, double* rho)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t s = 0; s < ns; ++s) {
        const int64_t i = sample[s];
        const float xi = pm[4 * i], yi = pm[4 * i + 1], zi = pm[4 * i + 2];
        float bd[64]; int32_t bj[64];
        int cnt = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            const float dx = pm[4 * j] - xi, dy = pm[4 * j + 1] - yi, dz = pm[4 * j + 2] - zi;
            const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            if (cnt == K && !(d2 < bd[K - 1])) continue;          /* j ascending: an equal d2 never displaces */
            int p = cnt < K ? cnt++ : K - 1;
            while (p > 0 && d2 < bd[p - 1]) { bd[p] = bd[p - 1]; bj[p] = bj[p - 1]; --p; }
            bd[p] = d2; bj[p] = (int32_t)j;
        }
        double m = 0.0;
        for (int q = 0; q < K; ++q) { if (nbr) nbr[s * K + q] = q < cnt ? bj[q] : -1; if (q < K - 1 && q < cnt) m += (double)pm[4 * (int64_t)bj[q] + 3]; }
        const double rk = cnt == K ? sqrt((double)bd[K - 1]) : 0.0;
        if (d2k) d2k[s] = cnt == K ? bd[K - 1] : INFINITY;
        if (rho) rho[s] = rk > 0.0 ? m / (4.0 * M_PI / 3.0 * rk * rk * rk) : 0.0;
    }
}

/* Step 2, over the sample (fp64, index order): density centre, core radius, core density, core number
 * (NBODY6's conventions, reading R18):
 *   x_d = sum rho_i x_i / sum rho_i;  R_core^2 = sum rho_i^2 |x_i - x_d|^2 / sum rho_i^2;
 *   rho_core = sum rho_i^2 / sum rho_i;  N_core = (N / ns) * #{ sample i : |x_i - x_d| < R_core }  (R19).
 * out[6] = x_d (3), R_core, rho_core, N_core. */
void p3t_o_core_quantities(int64_t n, const float* pm, int64_t ns, const int32_t* sample, const double* rho, double out[6])
{
    double sr = 0, sr2 = 0, c[3] = { 0, 0, 0 };
    for (int64_t s = 0; s < ns; ++s) {
        const float* p = pm + 4 * (int64_t)sample[s];
        sr += rho[s]; sr2 += rho[s] * rho[s];
        for (int a = 0; a < 3; ++a) c[a] += rho[s] * (double)p[a];
    }
    for (int a = 0; a < 3; ++a) c[a] /= sr;
    double q = 0;
    for (int64_t s = 0; s < ns; ++s) {
        const float* p = pm + 4 * (int64_t)sample[s];
        double d2 = 0; for (int a = 0; a < 3; ++a) d2 += ((double)p[a] - c[a]) * ((double)p[a] - c[a]);
        q += rho[s] * rho[s] * d2;
    }
    const double rc = sqrt(q / sr2);
    int64_t inside = 0;
    for (int64_t s = 0; s < ns; ++s) {
        const float* p = pm + 4 * (int64_t)sample[s];
        double d2 = 0; for (int a = 0; a < 3; ++a) d2 += ((double)p[a] - c[a]) * ((double)p[a] - c[a]);
        inside += d2 < rc * rc;
    }
    out[0] = c[0]; out[1] = c[1]; out[2] = c[2]; out[3] = rc; out[4] = sr2 / sr; out[5] = (double)inside * (double)n / (double)ns;
}
