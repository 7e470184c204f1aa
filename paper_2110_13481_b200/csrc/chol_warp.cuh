// One stage of (shifted) CholeskyQR done by ONE WARP in registers, in the prologue of the A*Mat pass that needs its
// result ("QR"; reading R12: any backward-stable QR).  Every CTA of the pass computes
// the same r x r factorisation from the same Gram sums (same instructions, same data: bit-identical), so no single-CTA
// kernel sits between two streaming passes; only CTA 0 writes the global by-products.
//
// Lane l holds column l of the unit-diagonal scaled Gram matrix; entries of other columns come by shuffle.  r <= 32.
//   gsum         : [P] upper pairs of A^T A, the final row of the producing pass (group_prereduce)
//   stage        : 0 adds `shift` to the scaled diagonal and clears the third-stage flag;
//                  1 decides whether a third stage is needed: with G scaled to unit diagonal, ||offdiag(G)||_F < 0.5
//                    implies ||G - I||_2 < 0.5, i.e. kappa(G) < 3 for every rank (a sufficient criterion), and then the
//                    factor after this stage is orthonormal to rounding level (CholeskyQR2 suffices for kappa(A)^2 u < 1):
//                    this stage is the last one;   2 is always the last one
//   mat (shared) : [cin][cout] matrix of the A*Mat pass = D U^-1 (times out_scale on the last stage)
//   Rtot (global, row-major, upper triangular) accumulates R_stage * Rtot with R_stage = U D^-1; on the last stage the
//   coupling matrix Sout (column-major) = Rtot * s_scale, or its transpose (transS: S = R^T for the L step, Fig. 1
//   line 40 transpose_inplace).
//   status[0] counts repaired pivots (QR fallbacks), status[2] the QRs that needed the third stage; qrflag[0] = 1 tells the
//   stage-2 launch to return at once.
// Returns (to all lanes) whether this stage is the last one.
#pragma once
#include "common.cuh"

struct CholArgs {
    const double* gsum;     // nullptr: no factorisation in this launch (the matrix is read from memory)
    int stage, transS;
    double shift, out_scale, s_scale;
    double* Rtot;
    double* Sout;
    int* status;
    int* qrflag;
};

template <int R>
__device__ __forceinline__ bool chol_warp(const CholArgs& ca, double* mat, bool writer) {
    static_assert(R <= 32, "one lane per column");
    constexpr unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int l = lane < R ? lane : R - 1;               // idle lanes mirror the last column (results unused)
    const int stage = ca.stage;
    // scaling to unit diagonal
    const double gd = ca.gsum[l * R - l * (l - 1) / 2];
    const double dsc_l = gd > 0.0 ? 1.0 / sqrt(gd) : 1.0, sg_l = gd > 0.0 ? sqrt(gd) : 1.0;
    double dsc[R], a[R];
#pragma unroll
    for (int i = 0; i < R; i++) dsc[i] = __shfl_sync(FULL, dsc_l, i);
    double f2 = 0.0;
#pragma unroll
    for (int i = 0; i < R; i++) {
        const int lo = i < l ? i : l, hi = i < l ? l : i;
        double g = ca.gsum[lo * R - lo * (lo - 1) / 2 + (hi - lo)] * dsc[i] * dsc_l;
        if (i == l && stage == 0) g += ca.shift;
        if (i != l && lane < R) f2 = fma(g, g, f2);
        a[i] = g;
    }
    f2 = warp_sum(f2);
    const bool skip = (stage == 1 && f2 < 0.25);         // NaN compares false: no skip
    const bool last = skip || stage == 2;
    // right-looking upper Cholesky G = U^T U; afterwards a[j] = U[j][l] for j <= l
    double dinv[R];
    int repaired = 0;
#pragma unroll
    for (int j = 0; j < R; j++) {
        double p = __shfl_sync(FULL, a[j], j);
        if (!(p > 1e-30)) { p = 1e-30; repaired++; }      // repaired pivot (counted as a QR fallback)
        double ri = rsqrt(p);
        ri = ri * fma(-0.5 * p * ri, ri, 1.5);            // one Newton step: rounding-level 1/sqrt(pivot)
        dinv[j] = ri;
        const double u = (l == j) ? p * ri : a[j] * ri;
        a[j] = u;
#pragma unroll
        for (int i = j + 1; i < R; i++) {
            const double uji = __shfl_sync(FULL, u, i);
            a[i] = fma(-uji, u, a[i]);                    // only entries i <= l are used later
        }
    }
    // inverse of U, column l:  b[l] = 1/U[l][l],  b[i] = -dinv[i] sum_{k = i+1..l} U[i][k] b[k]
    double b[R];
#pragma unroll
    for (int i = 0; i < R; i++) b[i] = (i == l) ? dinv[i] : 0.0;
#pragma unroll
    for (int i = R - 2; i >= 0; i--) {
        double s = 0.0;
#pragma unroll
        for (int k = i + 1; k < R; k++) {
            const double uik = __shfl_sync(FULL, a[i], k);     // U[i][k] (lane k, row i <= k)
            s = fma(uik, b[k], s);                             // b[k] = 0 for k > l
        }
        if (i < l) b[i] = -s * dinv[i];
    }
    const double osc = last ? ca.out_scale : 1.0;
    if (lane < R) {
#pragma unroll
        for (int i = 0; i < R; i++) mat[i * R + l] = dsc[i] * b[i] * osc;
    }
    if (writer) {
        // Rtot <- (U D^-1) Rtot, column l:  new[i][l] = sum_{k = i..l} U[i][k] sg[k] Rp[k][l]
        double rp[R];
#pragma unroll
        for (int k = 0; k < R; k++) rp[k] = (k <= l) ? (stage ? ca.Rtot[k * R + l] : (k == l ? 1.0 : 0.0)) * 1.0 : 0.0;
#pragma unroll
        for (int k = 0; k < R; k++) rp[k] *= __shfl_sync(FULL, sg_l, k);
#pragma unroll
        for (int i = 0; i < R; i++) {
            double s = 0.0;
#pragma unroll
            for (int k = i; k < R; k++) {
                const double uik = __shfl_sync(FULL, a[i], k);
                s = fma(uik, rp[k], s);                        // rp[k] = 0 for k > l
            }
            if (i > l) s = 0.0;
            if (lane < R) {
                ca.Rtot[i * R + l] = s;
                if (last) {
                    if (ca.transS) ca.Sout[l + R * i] = s * ca.s_scale;      // S = R^T
                    else ca.Sout[i + R * l] = s * ca.s_scale;                // S = R
                }
            }
        }
        if (lane == 0) {
            if (repaired) atomicAdd(ca.status, repaired);
            if (stage == 0) ca.qrflag[0] = 0;
            if (stage == 1) { ca.qrflag[0] = skip ? 1 : 0; if (!skip) atomicAdd(ca.status + 2, 1); }
        }
    }
    return last;
}

// one stage on its own (test hook: dlr_test_chol_decide)
template <int R>
__global__ void k_chol_test(const CholArgs ca, double* mat_out) {
    __shared__ double mat[R * R];
    chol_warp<R>(ca, mat, true);
    __syncwarp();
    for (int i = threadIdx.x; i < R * R; i += 32) mat_out[i] = mat[i];
}
