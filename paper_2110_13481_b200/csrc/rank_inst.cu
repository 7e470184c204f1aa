// Instantiates the rank-templated kernels for one rank (compile with -DDLR_RANK=<r>).
#include "rank_ops.h"

#ifndef DLR_RANK
#error "compile with -DDLR_RANK=<r>"
#endif
#define CAT2(a, b) a##b
#define CAT(a, b) CAT2(a, b)

namespace {
constexpr int R = DLR_RANK;

cudaError_t launch_chol_test(const CholArgs& ca, double* mat_out, cudaStream_t st) {
    k_chol_test<R><<<1, 32, 0, st>>>(ca, mat_out);
    return cudaGetLastError();
}

cudaError_t configure_rank() {
    cudaError_t e = cudaSuccess;
#define OPTIN(...) if (e == cudaSuccess) e = dlr_optin_smem(__VA_ARGS__)
    OPTIN(k_d1<R, R, D1_IN_REAL, D1_OP_MATVEC, D1_GRAM_PLAIN, D1_OUT_REAL>);
    OPTIN(k_d1<R, R, D1_IN_REAL, D1_OP_MATVEC, D1_GRAM_NONE, D1_OUT_REAL>);
    OPTIN(k_d1<R, R, D1_IN_REAL, D1_OP_NONE, D1_GRAM_PLAIN, D1_OUT_NONE>);
    OPTIN(k_d1<R, 1, D1_IN_REAL, D1_OP_MATVEC, D1_GRAM_NONE, D1_OUT_CPLX>);
    OPTIN(k_dir<R, 1, DOP_EXACT, DW_NONE>);
    OPTIN(k_dir<R, 2, DOP_EXACT, DW_NONE>);
    OPTIN(k_dir<R, 3, DOP_ETD1, DW_E>);
    OPTIN(k_dir<R, 3, DOP_ETD1, DW_V>);
    OPTIN(k_dir<R, 3, DOP_ETD2, DW_E>);
    OPTIN(k_dir<R, 3, DOP_ETD2, DW_V>);
    OPTIN(k_dir<R, 1, DOP_COEFF, DW_V>);
    OPTIN(k_dir<R, 1, DOP_COEFF, DW_E>);
    OPTIN(k_dir<R, 2, DOP_COEFF, DW_NONE>);
    OPTIN(k_dir<R, 3, DOP_COEFF, DW_NONE>);
    OPTIN(k_post<R>);
    OPTIN(k_apply<R, true>);
    OPTIN(k_apply<R, false>);
    if (e == cudaSuccess) e = configure_sub1<R>();
    OPTIN(k_lpred_sums<R>);
#undef OPTIN
    return e;
}
}  // namespace

extern "C" const RankOps* CAT(dlr_rank_ops_, DLR_RANK)() {
    static const RankOps ops = {
        R,
        configure_rank,
        {
            launch_d1<R, R, D1_IN_REAL, D1_OP_MATVEC, D1_GRAM_PLAIN, D1_OUT_REAL>,
            launch_d1<R, R, D1_IN_REAL, D1_OP_MATVEC, D1_GRAM_NONE, D1_OUT_REAL>,
            launch_d1<R, R, D1_IN_REAL, D1_OP_NONE, D1_GRAM_PLAIN, D1_OUT_NONE>,
            launch_d1<R, 1, D1_IN_REAL, D1_OP_MATVEC, D1_GRAM_NONE, D1_OUT_CPLX>,
        },
        {
            launch_dir<R, 1, DOP_EXACT, DW_NONE>,
            launch_dir<R, 2, DOP_EXACT, DW_NONE>,
            launch_dir<R, 3, DOP_ETD1, DW_E>,
            launch_dir<R, 3, DOP_ETD1, DW_V>,
            launch_dir<R, 3, DOP_ETD2, DW_E>,
            launch_dir<R, 3, DOP_ETD2, DW_V>,
            launch_dir<R, 1, DOP_COEFF, DW_V>,
            launch_dir<R, 1, DOP_COEFF, DW_E>,
            launch_dir<R, 2, DOP_COEFF, DW_NONE>,
            launch_dir<R, 3, DOP_COEFF, DW_NONE>,
        },
        launch_sub1<R>,
        sub1_occupancy<R>,
        {launch_apply<R, true>, launch_apply<R, false>},
        launch_cross<R>,
        launch_bug_s0<R>,
        launch_post<R>,
        launch_lpred<R>,
        launch_chol_test};
    return &ops;
}
