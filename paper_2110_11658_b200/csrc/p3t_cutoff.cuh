// p3t_cutoff.cuh -- the cutoff function of eq. 6 and the regular pair potential
// (R6) as device functions, with their host-side constants; shared by p3t_force.cu
// (regular force) and p3t_irregular.cu (irregular force and jerk).  Nothing here is shared with oracle/.
#pragma once
#include <math.h>

struct walk_consts {
    float rout2, rin2, r_in, inv_delta;   // inv_delta = 1 / (r_out - r_in)
    float rlist2;                          // neighbour search radius squared, r_list = r_out + r_buff >= r_out (NEXT-2)
    float psi_in;                          // psi(r_in), the constant regular pair potential inside r_in
    float k140;                            // 140 / (r_out - r_in)
    float s1;                              // S(1)
    float sc[6];                           // S(t) = t (sc0 + t (sc1 + ... t sc5))
    float rem;                             // c^3 (1+c)^3  (> 0)
    float c;                               // r_in / (r_out - r_in)
    double dk140, ds1, dsc[6], drem, dc;   // the same in fp64 (the table of p3t_irregular.cu)
    double dlog1c;                         // log(1 + c)
    float theta;
    int   pot_mode;
};


// eq. 6, 0 < x < 1: W = x^4 (35 - 84 x + 70 x^2 - 20 x^3); evaluated through the
// symmetry W(x) = 1 - W(1 - x) above x = 1/2 so that fp32 Horner never cancels.
__device__ __forceinline__ float cutoff_W(float x)
{
    float t = x > 0.5f ? 1.0f - x : x;
    float t2 = t * t;
    float w = t2 * t2 * (35.0f + t * (-84.0f + t * (70.0f - 20.0f * t)));
    return x > 0.5f ? 1.0f - w : w;
}

// regular pair potential for r_in < r < r_out (R6): -W/r - (140/D) int_x^1 t^3(1-t)^3/(t+c) dt
__device__ __forceinline__ float cutoff_psi(const walk_consts& K, float x, float W, float rinv)
{
    float sx = x * (K.sc[0] + x * (K.sc[1] + x * (K.sc[2] + x * (K.sc[3] + x * (K.sc[4] + x * K.sc[5])))));
    // r_in = 0: rem = 0 and its term is identically 0 (never 0 * log(1 / 0))
    float integral = (K.s1 - sx) - (K.rem > 0.0f ? K.rem * __logf((1.0f + K.c) / (x + K.c)) : 0.0f);
    return -W * rinv - K.k140 * integral;
}
// The closed form cancels: terms of order 1 give an integral of order 1e-2 .. 0 that is then multiplied
// by 140 / D ~ 3000, so in fp32 a pair's psi carries ~1e-5 of its Newtonian potential.  That is
// invisible in phi_R (dominated by the far field) but not in phi_I, which is made of near pairs only:
// the irregular path interpolates the integral from a table made in fp64 (p3t_irregular.cu).

static inline void make_consts(walk_consts& K, float r_out, float r_in, float theta, int pot_mode, float r_list = -1.0f)
{
    if (!(r_list >= r_out)) r_list = r_out;
    volatile float rl2 = r_list * r_list;
    K.rlist2 = rl2;
    // fp32 thresholds exactly as DESIGN.md R10 states them: one fp32 product each
    volatile float ro2 = r_out * r_out, ri2 = r_in * r_in;
    K.rout2 = ro2; K.rin2 = ri2; K.r_in = r_in;
    const double D = (double)r_out - (double)r_in, c = (double)r_in / D, c1 = 1.0 + c;
    K.inv_delta = (float)(1.0 / D);
    K.k140 = (float)(140.0 / D); K.dk140 = 140.0 / D;
    // t^3 (1-t)^3 = (t + c) (b5 t^5 + ... + b0) - c^3 (1+c)^3   (synthetic division at t = -c)
    const double b[6] = { c * c * c1 * c1 * c1, -c * c1 * c1 * c1, c1 * c1 * c1, -(3.0 + 3.0 * c + c * c), 3.0 + c, -1.0 };
    double s1 = 0.0;
    for (int k = 0; k < 6; ++k) { K.dsc[k] = b[k] / (k + 1); K.sc[k] = (float)K.dsc[k]; s1 += b[k] / (k + 1); }
    K.s1 = (float)s1; K.ds1 = s1;
    K.drem = c * c * c * c1 * c1 * c1; K.rem = (float)K.drem;
    K.c = (float)c; K.dc = c; K.dlog1c = log(c1);
    // psi(r_in) = -(140/D) [ S(1) + rem ln((1+c)/c) ... ] with W(0) = 0; here the remainder enters with a minus sign
    K.psi_in = (float)(-(140.0 / D) * (s1 - (c > 0.0 ? c * c * c * c1 * c1 * c1 * log(c1 / c) : 0.0)));   // r_in = 0: the remainder term is exactly 0
    K.theta = theta;
    K.pot_mode = pot_mode;
}


