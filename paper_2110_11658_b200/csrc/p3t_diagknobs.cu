// p3t_diagknobs.cu -- measurement and fault-injection knobs of a context (include/p3t_diag.h), part of libp3t_diag.so.
// They used to be environment variables read by p3t_create; the product library now has no such switch.  The fields
// are written directly: this file and libp3t.so are compiled from the same p3t_internal.cuh.
#include "p3t_internal.cuh"
#include "p3t_diag.h"

extern "C" int p3t_diag_set_overlap(void* ctx, int overlap, int walk_ctas_per_sm)
{
    p3t_ctx* c = (p3t_ctx*)ctx;
    if (!c || (overlap != 0 && overlap != 1) || walk_ctas_per_sm > 16) return -1;
    if (c->pend.active) return -1;
    c->overlap = overlap;
    if (walk_ctas_per_sm > 0) c->walk_ctas_per_sm = walk_ctas_per_sm;
    return 0;
}

extern "C" int p3t_diag_set_fault(void* ctx, int bits)
{
    p3t_ctx* c = (p3t_ctx*)ctx;
    if (!c || bits < 0 || bits > 7) return -1;
    c->test_fault = bits;
    return 0;
}
