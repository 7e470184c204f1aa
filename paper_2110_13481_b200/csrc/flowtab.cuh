// Tables of one K- or L-flow (mode-mixing matrices, phases, phi functions): layout shared by the kernel that builds
// them (post.cuh) and the kernels that read them.
#pragma once
#include "common.cuh"

// ---------------------------------------------------------------------------------------------------------
// phi functions of a purely imaginary argument z = i*theta (reading R7): closed forms for |theta| >= 1,
// Taylor series below.
static __device__ const double DLR_INV_FACT[24] = {      // 1/k!, k = 1..24 (correctly rounded)
    1.0, 0.5, 0.16666666666666666, 0.041666666666666664,
    0.008333333333333333, 0.001388888888888889, 0.0001984126984126984, 2.48015873015873e-05,
    2.7557319223985893e-06, 2.755731922398589e-07, 2.505210838544172e-08, 2.08767569878681e-09,
    1.6059043836821613e-10, 1.1470745597729725e-11, 7.647163731819816e-13, 4.779477332387385e-14,
    2.8114572543455206e-15, 1.5619206968586225e-16, 8.22063524662433e-18, 4.110317623312165e-19,
    1.9572941063391263e-20, 8.896791392450574e-22, 3.868170170630684e-23, 1.6117375710961184e-24};
__device__ inline void phi12_imag(double th, double2& p1, double2& p2) {
    if (fabs(th) < 1.0) {
        // Horner in z = i th:  phi1 = sum z^m/(m+1)!,  phi2 = sum z^m/(m+2)!
        double2 s1 = make_double2(0.0, 0.0), s2 = s1;
        for (int m = 21; m >= 0; m--) {
            // s = s*z + coeff,  z = (0, th)
            s1 = make_double2(-s1.y * th + DLR_INV_FACT[m], s1.x * th);
            s2 = make_double2(-s2.y * th + DLR_INV_FACT[m + 1], s2.x * th);
        }
        p1 = s1; p2 = s2;
    } else {
        double sn, cs, sh, ch;
        sincos(th, &sn, &cs);
        sincos(0.5 * th, &sh, &ch);
        const double omc = 2.0 * sh * sh;      // 1 - cos(th)
        (void)cs; (void)ch;
        p1 = make_double2(sn / th, omc / th);
        p2 = make_double2(omc / (th * th), (th - sn) / (th * th));
    }
}

// Tables of one K- or L-flow (see D3Args).  Tm: 3 x [R][R] eigenvectors (columns), lam: 3 x [R];
// Sin: r x r column-major coupling matrix; transS = 0: A0 = Sin*T1 (K = X S), 1: A0 = Sin^T*T1 (L = V S^T).
// sgn = -1 (K equation (9)) or +1 (L equation (11)); tsub = length of sub-flows 1,2; t3 = length of sub-flow 3.
// M2c: 3 x [R][R] derivative coefficients; nl gets nlsign * M2c (matrices of the real-space term).
struct FlowTabPtrs {
    double* mats;   // 8 R^2: 0 Sin*T1, 1 T1^T T2, 2 T2^T T3, 3 T3^T, 4 T3, 5 T3^T T2, 6 T2^T T1, 7 T1^T  ([cin][cout])
    double* Q;      // 3 R^2: real-space term in the eigenbasis of direction 3, Q_i = T3^T nl_i^T T3, nl_i = nlsign * M2c_i
    double2 *ph1, *ph2, *ez, *f1, *f2a, *f2b;   // [n][R] each, by stored (bit-reversed) position
};

// 1D marginals of V and what the flow-free predictor L step needs of them (k_marginals, k_marg_reduce -> k_lpred_sums)
struct MargOut {
    double *M1, *M2, *M3;        // [R][n] marginals
    double2 *Ph1, *Ph2;          // [R][n] their DFTs (natural wavenumber order)
    double *s0, *mom3;           // [R]
    double2* Wv;                 // [n]
};
