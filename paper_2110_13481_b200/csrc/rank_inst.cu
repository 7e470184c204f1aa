// Instantiates the rank-templated kernels for one rank (compile with -DDLR_RANK=<r>).
#include "rank_ops.h"

#ifndef DLR_RANK
#error "compile with -DDLR_RANK=<r>"
#endif
#define CAT2(a, b) a##b
#define CAT(a, b) CAT2(a, b)

namespace {
constexpr int R = DLR_RANK;
}

extern "C" const RankOps* CAT(dlr_rank_ops_, DLR_RANK)() {
    static const RankOps ops = {
        R,
        {
            launch_d1<R, R, D1_IN_REAL, D1_OP_NONE, D1_GRAM_NONE, D1_OUT_CPLX>,
            launch_d1<R, R, D1_IN_REAL, D1_OP_NONE, D1_GRAM_V, D1_OUT_CPLX>,
            launch_d1<R, R, D1_IN_REAL, D1_OP_NONE, D1_GRAM_E, D1_OUT_CPLX>,
            launch_d1<R, R, D1_IN_CPLX, D1_OP_NONLIN_E, D1_GRAM_NONE, D1_OUT_CPLX>,
            launch_d1<R, R, D1_IN_CPLX, D1_OP_NONLIN_V, D1_GRAM_NONE, D1_OUT_CPLX>,
            launch_d1<R, R, D1_IN_CPLX, D1_OP_NONE, D1_GRAM_PLAIN, D1_OUT_REAL>,
            launch_d1<R, R, D1_IN_CPLX, D1_OP_NONE, D1_GRAM_NONE, D1_OUT_REAL>,
            launch_d1<R, R, D1_IN_REAL, D1_OP_MATVEC, D1_GRAM_PLAIN, D1_OUT_REAL>,
            launch_d1<R, R, D1_IN_REAL, D1_OP_MATVEC, D1_GRAM_NONE, D1_OUT_REAL>,
            launch_d1<R, R, D1_IN_REAL, D1_OP_NONE, D1_GRAM_PLAIN, D1_OUT_NONE>,
            launch_d1<R, 1, D1_IN_REAL, D1_OP_MATVEC, D1_GRAM_NONE, D1_OUT_CPLX>,
        },
        {
            launch_d3<R, R, D3_FWD_STORE, false>,
            launch_d3<R, R, D3_FWD_STORE, true>,
            launch_d3<R, R, D3_FLOW_START, false>,
            launch_d3<R, R, D3_EULER_END, false>,
            launch_d3<R, R, D3_MID, false>,
            launch_d3<R, R, D3_END2, false>,
            launch_d3<R, R, D3_INV_ONLY, false>,
        }};
    return &ops;
}
