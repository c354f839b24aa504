/* oracle/p3t_oracle_tree_priv.h -- TEST INFRASTRUCTURE (see p3t_oracle.h): the oracle tree record. */
#ifndef P3T_ORACLE_TREE_PRIV_H
#define P3T_ORACLE_TREE_PRIV_H
#include "p3t_oracle.h"
struct p3t_o_tree {
    int64_t n; int bits, nleaf, ncrit;
    float lo[3], side;
    uint64_t* keys; uint32_t* order; float* spm;             /* sorted keys, order, sorted bodies */
    int64_t nn, cap; int64_t n_leaves; int max_level;
    int32_t *level, *begin, *end, *first_child, *n_child; uint64_t* prefix;
    double *mass, *com, *quad;                                /* fp64 moments                */
    double *oct;                                              /* fp64 raw third moment [10]  */
    float *fcom_m, *fquad, *clo, *chi, *delta;                /* fp32-rounded node data      */
    float *foct;                                              /* fp32-rounded third moment   */
    int64_t ng, gcap; int32_t *gbegin, *gend; float *glo, *ghi;
};
#endif
