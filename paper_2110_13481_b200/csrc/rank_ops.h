// Per-rank kernel launch tables: the streaming kernels are templated on the rank r so that the per-point
// r-vectors live in registers; rank_inst.cu is compiled once per supported rank (-DDLR_RANK=r).
#pragma once
#include "kernels_d1.cuh"
#include "kernels_d2.cuh"
#include "kernels_d3.cuh"

enum {
    V1_FFT_PLAIN = 0,   // real -> half spectrum along dim 1
    V1_FFT_GRAMV,       // + C1 Gram with grid-velocity weights and column sums (rho_tilde)
    V1_FFT_GRAME,       // + D1 Gram with electric-field weights
    V1_MID_E,           // c2r -> sum_i diag(E_i) A M_i^T -> r2c     (K step, eq. (9))
    V1_MID_V,           // c2r -> sum_i diag(v_i) A M_i^T -> r2c     (L step, eq. (11); M_i = -D2_i)
    V1_INV_GRAM,        // c2r -> real, + plain Gram (first CholeskyQR Gram)
    V1_INV,             // c2r -> real
    V1_APPLY_GRAM,      // real -> A*Mat -> real, + plain Gram
    V1_APPLY,           // real -> A*Mat -> real
    V1_GRAM_ONLY,       // plain Gram of a real factor
    V1_RHO,             // real r columns -> (A p) one column -> half spectrum
    V1_COUNT
};
enum { V3_FWD = 0, V3_FWD_PGRAM, V3_START, V3_EULER_END, V3_MID, V3_END2, V3_INV, V3_COUNT };

struct RankOps {
    int R;
    cudaError_t (*d1[V1_COUNT])(const D1Args&, cudaStream_t);
    cudaError_t (*d3[V3_COUNT])(const D3Args&, cudaStream_t);
};

const RankOps* dlr_rank_ops(int R);      // nullptr if the rank is not compiled in
