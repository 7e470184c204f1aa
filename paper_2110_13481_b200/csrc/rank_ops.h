// Per-rank kernel launch tables: the streaming kernels are templated on the rank r so that the per-point
// r-vectors live in registers; rank_inst.cu is compiled once per supported rank (-DDLR_RANK=r).
#pragma once
#include "kernels_d1.cuh"
#include "kernels_d2.cuh"
#include "kernels_d3.cuh"
#include "kernels_dir.cuh"
#include "post.cuh"
#include "pass_sub1.cuh"
#include "pass_apply.cuh"
#include "pass_cross.cuh"

// row-tile kernels without a transform (CholeskyQR passes, density, initial-state check)
enum {
    V1_APPLY_GRAM = 0,  // real -> A*Mat -> real, + plain Gram
    V1_APPLY,           // real -> A*Mat -> real
    V1_GRAM_ONLY,       // plain Gram of a real factor
    V1_RHO,             // real r columns -> (A p) one column -> half spectrum (first pass of the Poisson solve)
    V1_COUNT
};
// directional passes (kernels_dir.cuh)
enum {
    VD_EXACT1 = 0,      // sub-flow along direction 1 (with the column mixing before and after)
    VD_EXACT2,          // sub-flow along direction 2
    VD_ETD1_E,          // third sub-flow, exponential Euler, field weights (K step)
    VD_ETD1_V,          //                                    velocity weights (L step)
    VD_ETD2_E,          // third sub-flow, ETD2RK
    VD_ETD2_V,
    VD_COEFF1_V,        // C coefficients: weighted Gram (+ rho_tilde) and Parseval sums along direction 1
    VD_COEFF1_E,        // D coefficients: same with field weights
    VD_COEFF2,          // Parseval sums along direction 2
    VD_COEFF3,          // Parseval sums along direction 3
    VD_COUNT
};

struct RankOps {
    int R;
    cudaError_t (*configure)();      // shared-memory opt-in of every kernel below on the current device (dlr_create)
    cudaError_t (*d1[V1_COUNT])(const D1Args&, cudaStream_t);
    cudaError_t (*dir[VD_COUNT])(const DirArgs&, cudaStream_t);
    cudaError_t (*sub1)(const Sub1Args&, int groups, int ctas, cudaStream_t);     // sub-flow 1, warp-autonomous (pass_sub1.cuh)
    int (*sub1_occ)(int log2n, int threads, size_t smem);                        // its resident CTAs per SM
    cudaError_t (*apply[2])(const ApplyArgs&, int ctas, cudaStream_t);          // A*Mat pass of CholeskyQR (pass_apply.cuh): [0] with Gram, [1] without
    cudaError_t (*cross)(const double* A, const double* B, long long N, double* partial, int ctas, cudaStream_t);   // pass_cross.cuh
    cudaError_t (*bug_s0)(const double* pm, int nm, const double* pn, int nn, double hx3, double hv3, double* S, cudaStream_t);
    cudaError_t (*post)(const PostArgs&, cudaStream_t);           // r x r work between two streaming phases (post.cuh)
    cudaError_t (*lpred)(const LpredArgs&, cudaStream_t);         // column sums of the predictor's L1 (post.cuh)
    cudaError_t (*chol_test)(const CholArgs&, double* mat_out, cudaStream_t);     // one CholeskyQR stage on its own (test hook)
};

const RankOps* dlr_rank_ops(int R);      // nullptr if the rank is not compiled in
