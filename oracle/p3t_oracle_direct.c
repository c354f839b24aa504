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
    double integral = (S1 - Sx) + rem * log((1.0 + c) / (x + c));
    return -p3t_o_W(x) / r - (140.0 / D) * integral;
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
