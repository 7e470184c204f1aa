// Small dense device kernels (r x r work, table building, reductions of per-CTA partial sums, diagnostics).
// All of it stays on the device so that one step needs no host round trip (the paper's own S step is 10x slower
// on the GPU than on the CPU because of tiny library calls).
// Matrix conventions: coefficient matrices C1,C2,D1,D2,T are row-major M[a*R+b]; S is column-major S[i + R*j]
// (the C ABI layout).
#pragma once
#include "common.cuh"

#define DLR_G1 32          // number of second-level partial rows
#define DLR_RMAXS 24       // largest rank the small kernels are dimensioned for

// ---------------------------------------------------------------------------------------------------------
// two-level deterministic reduction of per-CTA partial sums: out[g][v] = sum_{b in slice g} partial[b][v]
__global__ void k_reduce_partials(const double* __restrict__ partial, int nblocks, int nvals, double* __restrict__ out) {
    const int g = blockIdx.x;
    const int per = (nblocks + gridDim.x - 1) / gridDim.x;
    const int b0 = g * per, b1 = min(nblocks, b0 + per);
    for (int v = threadIdx.x; v < nvals; v += blockDim.x) {
        double s = 0.0;
        for (int b = b0; b < b1; b++) s += partial[(size_t)b * nvals + v];
        out[(size_t)g * nvals + v] = s;
    }
}

__device__ __forceinline__ double sum_g1(const double* p2, int nvals, int v) {
    double s = 0.0;
    for (int g = 0; g < DLR_G1; g++) s += p2[(size_t)g * nvals + v];
    return s;
}

// ---------------------------------------------------------------------------------------------------------
// coefficients from the reduced Gram sums.  gram: [DLR_G1][3P (+R)] (real-space, weights v_i or E_i),
// pgram: [DLR_G1][3 P2] (Parseval sums for the derivative coefficients).
//   M1_i = h^3 A^T diag(w_i) A (symmetric), M2_i = h^3 A^T d_i A (antisymmetric),
//   colsum = h^3 A^T 1 (rho_tilde of eq. (12)) if with_colsum.
__global__ void k_finalize_coeff(const double* gram, const double* pgram, int R, int with_colsum, double h3,
                                 double invN, double* M1, double* M2, double* colsum) {
    const int P = R * (R + 1) / 2, P2 = R * (R - 1) / 2;
    const int nv1 = 3 * P + (with_colsum ? R : 0), nv2 = 3 * P2;
    for (int idx = threadIdx.x; idx < 3 * R * R; idx += blockDim.x) {
        const int d = idx / (R * R), a = (idx / R) % R, b = idx % R;
        const int lo = min(a, b), hi = max(a, b);
        const int pe = lo * R - lo * (lo - 1) / 2 + (hi - lo);           // pair index of (lo <= hi)
        M1[idx] = h3 * sum_g1(gram, nv1, d * P + pe);
        double v = 0.0;
        if (a != b) {
            const int pe2 = lo * (R - 1) - lo * (lo - 1) / 2 + (hi - lo - 1);
            v = h3 * invN * sum_g1(pgram, nv2, d * P2 + pe2);
            if (a > b) v = -v;
        }
        M2[idx] = v;
    }
    if (with_colsum)
        for (int c = threadIdx.x; c < R; c += blockDim.x) colsum[c] = h3 * sum_g1(gram, nv1, 3 * P + c);
}

// ---------------------------------------------------------------------------------------------------------
// cyclic Jacobi eigen-decomposition of three symmetric r x r matrices (one warp each): Msym = T diag(lam) T^T
// (PAPER.md:260).  The input is symmetrised first (reading R5).
__global__ void k_eig3(const double* M1, int R, double* Tout, double* lam) {
    __shared__ double As[3][DLR_RMAXS][DLR_RMAXS + 1];
    __shared__ double Ts[3][DLR_RMAXS][DLR_RMAXS + 1];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (w >= 3) return;
    const double* Min = M1 + (size_t)w * R * R;
    double(*A)[DLR_RMAXS + 1] = As[w];
    double(*T)[DLR_RMAXS + 1] = Ts[w];
    for (int i = lane; i < R; i += 32)
        for (int j = 0; j < R; j++) {
            A[i][j] = 0.5 * (Min[i * R + j] + Min[j * R + i]);
            T[i][j] = i == j ? 1.0 : 0.0;
        }
    __syncwarp();
    double nrm = 0.0;
    for (int i = lane; i < R; i += 32)
        for (int j = 0; j < R; j++) nrm += A[i][j] * A[i][j];
    nrm = sqrt(warp_sum(nrm));
    for (int sweep = 0; sweep < 60; sweep++) {
        double off = 0.0;
        for (int i = lane; i < R; i += 32)
            for (int j = i + 1; j < R; j++) off += A[i][j] * A[i][j];
        off = sqrt(warp_sum(off));
        if (off <= 1e-16 * nrm || off == 0.0) break;
        for (int p = 0; p < R - 1; p++)
            for (int q = p + 1; q < R; q++) {
                const double apq = A[p][q];
                if (fabs(apq) <= 1e-20 * nrm) continue;          // warp-uniform
                const double theta = (A[q][q] - A[p][p]) / (2.0 * apq);
                const double t = fabs(theta) > 1e150 ? 0.5 / theta
                                                     : copysign(1.0, theta) / (fabs(theta) + sqrt(theta * theta + 1.0));
                const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
                __syncwarp();
                if (lane < R) {
                    const double aip = A[lane][p], aiq = A[lane][q];
                    A[lane][p] = c * aip - s * aiq;
                    A[lane][q] = s * aip + c * aiq;
                    const double tip = T[lane][p], tiq = T[lane][q];
                    T[lane][p] = c * tip - s * tiq;
                    T[lane][q] = s * tip + c * tiq;
                }
                __syncwarp();
                if (lane < R) {
                    const double api = A[p][lane], aqi = A[q][lane];
                    A[p][lane] = c * api - s * aqi;
                    A[q][lane] = s * api + c * aqi;
                }
                __syncwarp();
                if (lane == 0) { A[p][q] = 0.0; A[q][p] = 0.0; }
                __syncwarp();
            }
    }
    __syncwarp();
    for (int i = lane; i < R; i += 32) {
        lam[w * R + i] = A[i][i];
        for (int j = 0; j < R; j++) Tout[(size_t)w * R * R + i * R + j] = T[i][j];
    }
}

// ---------------------------------------------------------------------------------------------------------
// phi functions of a purely imaginary argument z = i*theta (reading R7): closed forms for |theta| >= 1,
// Taylor series below.
__device__ inline void phi12_imag(double th, double2& p1, double2& p2) {
    if (fabs(th) < 1.0) {
        // Horner in z = i th:  phi1 = sum z^m/(m+1)!,  phi2 = sum z^m/(m+2)!
        double2 s1 = make_double2(0.0, 0.0), s2 = s1;
        double f1 = 1.0, f2 = 1.0;             // 1/(m+1)!, 1/(m+2)! built on the fly
        double inv[24];
        double fac = 1.0;
        for (int m = 0; m < 24; m++) { fac *= (double)(m + 1); inv[m] = 1.0 / fac; }   // inv[m] = 1/(m+1)!
        (void)f1; (void)f2;
        for (int m = 21; m >= 0; m--) {
            // s = s*z + coeff,  z = (0, th)
            s1 = make_double2(-s1.y * th + inv[m], s1.x * th);
            s2 = make_double2(-s2.y * th + inv[m + 1], s2.x * th);
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
    double* mats;   // 8 R^2
    double* nl;     // 3 R^2
    double2 *ph1, *ph2, *ez, *f1, *f2a, *f2b;
};

__global__ void k_flow_tables(const double* Tm, const double* lam, const double* Sin, int transS, int R, GridDev g,
                              double sgn, double tsub, double t3, const double* M2c, double nlsign, FlowTabPtrs o) {
    const double* T1 = Tm;
    const double* T2 = Tm + R * R;
    const double* T3 = Tm + 2 * R * R;
    const int RR = R * R;
    for (int idx = threadIdx.x; idx < RR; idx += blockDim.x) {
        const int a = idx / R, b = idx % R;
        double m0 = 0, m1 = 0, m2 = 0, m5 = 0, m6 = 0;
        for (int k = 0; k < R; k++) {
            const double s_ak = transS ? Sin[k + R * a] : Sin[a + R * k];
            m0 = fma(s_ak, T1[k * R + b], m0);
            m1 = fma(T1[k * R + a], T2[k * R + b], m1);
            m2 = fma(T2[k * R + a], T3[k * R + b], m2);
            m5 = fma(T3[k * R + a], T2[k * R + b], m5);
            m6 = fma(T2[k * R + a], T1[k * R + b], m6);
        }
        o.mats[0 * RR + idx] = m0;
        o.mats[1 * RR + idx] = m1;
        o.mats[2 * RR + idx] = m2;
        o.mats[3 * RR + idx] = T3[b * R + a];
        o.mats[4 * RR + idx] = T3[idx];
        o.mats[5 * RR + idx] = m5;
        o.mats[6 * RR + idx] = m6;
        o.mats[7 * RR + idx] = T1[b * R + a];
        for (int d = 0; d < 3; d++) o.nl[d * RR + idx] = nlsign * M2c[d * RR + idx];
    }
    const int n = g.n, nh = g.nh;
    for (int idx = threadIdx.x; idx < nh * R; idx += blockDim.x) {
        const int k = idx / R, j = idx % R;
        double sn, cs;
        sincos(sgn * tsub * g.kt1[k] * lam[j], &sn, &cs);
        o.ph1[idx] = make_double2(cs, sn);
    }
    for (int idx = threadIdx.x; idx < n * R; idx += blockDim.x) {
        const int k = idx / R, j = idx % R;
        double sn, cs;
        sincos(sgn * tsub * g.kt2p[k] * lam[R + j], &sn, &cs);
        o.ph2[idx] = make_double2(cs, sn);
        const double th = sgn * t3 * g.kt2p[k] * lam[2 * R + j];
        sincos(th, &sn, &cs);
        o.ez[idx] = make_double2(cs, sn);
        double2 p1, p2;
        phi12_imag(th, p1, p2);
        o.f1[idx] = make_double2(t3 * p1.x, t3 * p1.y);
        o.f2a[idx] = make_double2(t3 * (p1.x - p2.x), t3 * (p1.y - p2.y));
        o.f2b[idx] = make_double2(t3 * p2.x, t3 * p2.y);
    }
}

// ---------------------------------------------------------------------------------------------------------
// S step: one classical RK4 step of eq. (10):  dS/dt = sum_i D2_i S C1_i^T - D1_i S C2_i^T
__global__ void k_sflow(double* S, int R, double t, const double* C1, const double* C2, const double* D1,
                        const double* D2) {
    __shared__ double Sc[DLR_RMAXS * DLR_RMAXS], Y[DLR_RMAXS * DLR_RMAXS], Kacc[DLR_RMAXS * DLR_RMAXS];
    __shared__ double Pm[3][DLR_RMAXS * DLR_RMAXS], Qm[3][DLR_RMAXS * DLR_RMAXS];
    const int RR = R * R;
    for (int i = threadIdx.x; i < RR; i += blockDim.x) { Sc[i] = S[i]; Y[i] = S[i]; Kacc[i] = 0.0; }
    __syncthreads();
    const double cw[4] = {1.0, 2.0, 2.0, 1.0}, cs[4] = {0.5, 0.5, 1.0, 0.0};
    for (int stage = 0; stage < 4; stage++) {
        // P_d = Y C1_d^T, Q_d = Y C2_d^T     (Y column-major: Y(a,k) = Y[a + R k])
        for (int idx = threadIdx.x; idx < 3 * RR; idx += blockDim.x) {
            const int d = idx / RR, a = (idx % RR) / R, b = idx % R;
            double p = 0, q = 0;
            for (int k = 0; k < R; k++) {
                const double y = Y[a + R * k];
                p = fma(y, C1[d * RR + b * R + k], p);
                q = fma(y, C2[d * RR + b * R + k], q);
            }
            Pm[d][a * R + b] = p;
            Qm[d][a * R + b] = q;
        }
        __syncthreads();
        double rhs_reg[4];      // each thread owns entries idx = tid + m*blockDim (R^2 <= 4*256)
        int m = 0;
        for (int idx = threadIdx.x; idx < RR; idx += blockDim.x, m++) {
            const int a = idx % R, b = idx / R;       // column-major entry (a,b)
            double r = 0;
            for (int d = 0; d < 3; d++)
                for (int k = 0; k < R; k++)
                    r += D2[d * RR + a * R + k] * Pm[d][k * R + b] - D1[d * RR + a * R + k] * Qm[d][k * R + b];
            rhs_reg[m] = r;
        }
        __syncthreads();
        m = 0;
        for (int idx = threadIdx.x; idx < RR; idx += blockDim.x, m++) {
            Kacc[idx] += cw[stage] * rhs_reg[m];
            Y[idx] = Sc[idx] + cs[stage] * t * rhs_reg[m];
        }
        __syncthreads();
    }
    for (int i = threadIdx.x; i < RR; i += blockDim.x) S[i] = Sc[i] + (t / 6.0) * Kacc[i];
}

// ---------------------------------------------------------------------------------------------------------
// One stage of (shifted) CholeskyQR on the reduced Gram sums (one warp).
//   gram: [DLR_G1][P] upper pairs of A^T A.   stage 0 adds `shift` to the unit-diagonal scaled Gram matrix.
//   apply[ci][co] : matrix for the next A*Mat pass (= D U^-1, times out_scale on the last stage)
//   Rtot (row-major, upper triangular) accumulates R_stage * Rtot.
//   On the last stage the coupling matrix is written: Sout column-major = Rtot*s_scale (transS=0) or its transpose.
__global__ void k_chol_stage(const double* gram, int R, int stage, int last, double shift, double out_scale,
                             double s_scale, int transS, double* apply, double* Rtot, double* Sout, int* status) {
    __shared__ double G[DLR_RMAXS][DLR_RMAXS + 1], U[DLR_RMAXS][DLR_RMAXS + 1], Ui[DLR_RMAXS][DLR_RMAXS + 1];
    __shared__ double dsc[DLR_RMAXS], Rn[DLR_RMAXS][DLR_RMAXS + 1];
    const int lane = threadIdx.x;
    const int P = R * (R + 1) / 2;
    if (lane < R) {
        const int l = lane;
        for (int a = 0; a < R; a++) {
            const int lo = min(a, l), hi = max(a, l);
            G[a][l] = sum_g1(gram, P, lo * R - lo * (lo - 1) / 2 + (hi - lo));
            U[a][l] = 0.0; Ui[a][l] = 0.0;
        }
    }
    __syncwarp();
    if (lane < R) {
        const double g = G[lane][lane];
        dsc[lane] = g > 0.0 ? 1.0 / sqrt(g) : 1.0;
    }
    __syncwarp();
    if (lane < R)
        for (int a = 0; a < R; a++) {
            G[a][lane] *= dsc[a] * dsc[lane];
            if (a == lane && stage == 0) G[a][lane] += shift;
        }
    __syncwarp();
    // upper Cholesky G = U^T U, lane = column
    for (int j = 0; j < R; j++) {
        if (lane == j) {
            double s = G[j][j];
            for (int k = 0; k < j; k++) s -= U[k][j] * U[k][j];
            if (!(s > 1e-30)) { s = 1e-30; atomicAdd(status, 1); }     // repaired pivot (counted as a QR fallback)
            U[j][j] = sqrt(s);
        }
        __syncwarp();
        if (lane > j && lane < R) {
            double s = G[j][lane];
            for (int k = 0; k < j; k++) s -= U[k][j] * U[k][lane];
            U[j][lane] = s / U[j][j];
        }
        __syncwarp();
    }
    // inverse of U (upper), lane = column l: U x = e_l
    if (lane < R) {
        const int l = lane;
        Ui[l][l] = 1.0 / U[l][l];
        for (int i = l - 1; i >= 0; i--) {
            double s = 0.0;
            for (int k = i + 1; k <= l; k++) s += U[i][k] * Ui[k][l];
            Ui[i][l] = -s / U[i][i];
        }
    }
    __syncwarp();
    if (lane < R) {
        const int l = lane;
        const double osc = last ? out_scale : 1.0;
        for (int a = 0; a < R; a++) apply[a * R + l] = dsc[a] * Ui[a][l] * osc;
        // R_stage = U D^-1 ;  Rtot <- R_stage * Rtot
        for (int a = 0; a < R; a++) {
            double s = 0.0;
            if (stage == 0) s = U[a][l] / dsc[l];
            else
                for (int k = a; k <= l; k++) s += (U[a][k] / dsc[k]) * Rtot[k * R + l];
            Rn[a][l] = (a <= l) ? s : 0.0;
        }
    }
    __syncwarp();
    if (lane < R) {
        const int l = lane;
        for (int a = 0; a < R; a++) {
            Rtot[a * R + l] = Rn[a][l];
            if (last) {
                if (transS) Sout[l + R * a] = Rn[a][l] * s_scale;      // S = R^T
                else Sout[a + R * l] = Rn[a][l] * s_scale;             // S = R
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// vectors for the charge density: out[c] = scale * sum_j S(c,j) vec[j]   (use_S) or scale * vec[c]
__global__ void k_rho_vec(const double* S, const double* vec, int R, int use_S, double scale, double* out) {
    const int c = threadIdx.x;
    if (c >= R) return;
    double s = 0.0;
    if (use_S == 2) for (int j = 0; j < R; j++) s += S[c + R * j] * vec[5 * j];      // vec = column moments, stride 5
    else if (use_S) for (int j = 0; j < R; j++) s += S[c + R * j] * vec[j];
    else s = vec[c];
    out[c] = scale * s;
}

// ---------------------------------------------------------------------------------------------------------
// diagnostics
// column sums with weights {1, w1, w2, w3, |w|^2} (w = grid coordinate): out[c*5+m]; one CTA per column
__global__ void k_colmoments(const double* A, GridDev g, double* out) {
    __shared__ double red[5][32];
    const int c = blockIdx.x, n = g.n;
    const double* col = A + (size_t)c * g.N;
    double s[5] = {0, 0, 0, 0, 0};
    for (long long I = threadIdx.x; I < g.N; I += blockDim.x) {
        const int i1 = (int)(I % n), i2 = (int)((I / n) % n), i3 = (int)(I / ((long long)n * n));
        const double w1 = g.lo + g.h * i1, w2 = g.lo + g.h * i2, w3 = g.lo + g.h * i3, a = col[I];
        s[0] += a; s[1] += a * w1; s[2] += a * w2; s[3] += a * w3; s[4] += a * (w1 * w1 + w2 * w2 + w3 * w3);
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int m = 0; m < 5; m++) { s[m] = warp_sum(s[m]); if (lane == 0) red[m][w] = s[m]; }
    __syncthreads();
    if (threadIdx.x < 5) {
        double t = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); i++) t += red[threadIdx.x][i];
        out[c * 5 + threadIdx.x] = t;
    }
}

// sum of squares of nvals doubles -> out[0] (single CTA, fixed order)
__global__ void k_sumsq(const double* a, long long nvals, double* out) {
    __shared__ double red[32];
    double s = 0.0;
    for (long long i = threadIdx.x; i < nvals; i += blockDim.x) s = fma(a[i], a[i], s);
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); i++) t += red[i];
        out[0] = t;
    }
}

// moments from the column moments; res: mass, mom1..3, kinetic, s_fro, nonfinite
__global__ void k_moments_final(const double* mx, const double* mv, const double* S, int R, double hx3, double hv3,
                                double* res) {
    if (threadIdx.x != 0) return;
    double out[5] = {0, 0, 0, 0, 0}, fro = 0.0;
    int bad = 0;
    for (int i = 0; i < R; i++)
        for (int j = 0; j < R; j++) {
            const double s = S[i + R * j];
            if (!isfinite(s)) bad = 1;
            fro += s * s;
            for (int m = 0; m < 5; m++) out[m] += hx3 * mx[i * 5] * s * hv3 * mv[j * 5 + m];
        }
    res[0] = out[0]; res[1] = out[1]; res[2] = out[2]; res[3] = out[3]; res[4] = 0.5 * out[4];
    res[5] = sqrt(fro); res[6] = (double)bad;
}

__global__ void k_probes(const double* X, const double* S, const double* V, long long Nx, long long Nv, int R, int np,
                         const long long* ix, const long long* iv, double* f) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    double s = 0.0;
    for (int i = 0; i < R; i++) {
        double t = 0.0;
        for (int j = 0; j < R; j++) t += S[i + R * j] * V[(size_t)j * Nv + iv[p]];
        s += X[(size_t)i * Nx + ix[p]] * t;
    }
    f[p] = s;
}
