// Small dense device kernels (r x r work, table building, reductions of per-CTA partial sums, diagnostics).
// All of it stays on the device so that one step needs no host round trip (the paper's own S step is 10x slower
// on the GPU than on the CPU because of tiny library calls).
// Matrix conventions: coefficient matrices C1,C2,D1,D2,T are row-major M[a*R+b]; S is column-major S[i + R*j]
// (the C ABI layout).
#pragma once
#include "common.cuh"
#include "flowtab.cuh"

#define DLR_G1 32          // number of second-level partial rows
#define DLR_RMAXS 24       // largest rank the small kernels are dimensioned for
#define DLR_SMALL_THREADS 512   // CTA size of the single-CTA r x r kernels (also the width of their inline reductions)

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

// CTA-wide deterministic reduction of per-CTA partial rows, done by the consumer kernel itself (no separate
// reduction launch):  out[v] = sum_b partial[b * stride + off + v],  v < nvals <= blockDim.x.
// Thread (g, v) sums the rows b = g, g+G, ... (coalesced in v), then the G group sums are added in fixed order.
// out: shared [nvals]; tmp: shared [blockDim.x].  Ends with a __syncthreads().
__device__ __forceinline__ void cta_reduce_rows(const double* __restrict__ partial, int nblocks, int stride, int off,
                                                int nvals, double* out, double* tmp) {
    const int nth = blockDim.x, tid = threadIdx.x;
    const int G = nth / nvals;                     // >= 1
    const int g = tid / nvals, v = tid - g * nvals;
    if (g < G) {
        const double* p = partial + off + v;
        double s[8] = {0, 0, 0, 0, 0, 0, 0, 0};          // eight loads in flight per thread, fixed summation order
        int b = g;
        for (; b + 7 * G < nblocks; b += 8 * G) {
#pragma unroll
            for (int u = 0; u < 8; u++) s[u] += p[(size_t)(b + u * G) * stride];
        }
        for (; b < nblocks; b += G) s[0] += p[(size_t)b * stride];
        tmp[g * nvals + v] = ((s[0] + s[1]) + (s[2] + s[3])) + ((s[4] + s[5]) + (s[6] + s[7]));
    }
    __syncthreads();
    if (tid < nvals) {
        double s = 0.0;
        for (int gg = 0; gg < G; gg++) s += tmp[gg * nvals + tid];
        out[tid] = s;
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------------------------
// First half of a coefficient set + its eigen-decompositions, one CTA per direction d (grid = 3):
//   M1_d = h^3 A^T diag(w_d) A from the real-space Gram partial sums of the dimension-1 pass,
//   colsum = h^3 A^T 1 (rho_tilde of eq. (12); CTA 0, if with_colsum),
//   M1_d (symmetrised, reading R5) = T diag(lam) T^T by cyclic Jacobi with ROUND-ROBIN pair ordering:
//   every round rotates R/2 disjoint pairs at once, A <- J^T A J and T <- T J entry-wise from the previous
//   buffer (two barriers per round instead of a serial chain of R(R-1)/2 rotations per sweep).
// partial: [nblocks][3P (+R)], entry e of direction d at d*P + e, column sums at 3P + c.
#define DLR_EIG_THREADS 256
#ifndef DLR_EIG_TOL2
#define DLR_EIG_TOL2 1e-20
#endif
__global__ void __launch_bounds__(DLR_EIG_THREADS)
k_coeff1_eig(const double* partial, int nblocks, int R, int with_colsum, double h3, double* M1, double* colsum,
             double* Tout, double* lam, int warm, int* status) {
    __shared__ double As[2][DLR_RMAXS][DLR_RMAXS + 1], Ts[2][DLR_RMAXS][DLR_RMAXS + 1];
    __shared__ double red[DLR_RMAXS * (DLR_RMAXS + 1) / 2], tmp[DLR_EIG_THREADS];
    __shared__ double alpha[DLR_RMAXS], beta[DLR_RMAXS], sq[DLR_RMAXS];
    __shared__ int part[DLR_RMAXS];
    __shared__ double s_nrm2, s_off2;
    const int d = blockIdx.x, tid = threadIdx.x, nth = blockDim.x;
    const int P = R * (R + 1) / 2, nv = 3 * P + (with_colsum ? R : 0), RR = R * R;
    if (d == 0 && with_colsum) {
        cta_reduce_rows(partial, nblocks, nv, 3 * P, R, red, tmp);
        if (tid < R) colsum[tid] = h3 * red[tid];
        __syncthreads();
    }
    cta_reduce_rows(partial, nblocks, nv, d * P, P, red, tmp);
    for (int idx = tid; idx < RR; idx += nth) {
        const int i = idx / R, j = idx - i * R;
        const int lo = min(i, j), hi = max(i, j);
        const double v = h3 * red[lo * R - lo * (lo - 1) / 2 + (hi - lo)];     // symmetric by construction
        As[0][i][j] = v;
        Ts[0][i][j] = i == j ? 1.0 : 0.0;
        M1[(size_t)d * RR + idx] = v;
    }
    __syncthreads();
    if (warm) {
        // warm start: the matrix changes little between consecutive solves, so the previous eigenvectors Tp (still in
        // Tout) almost diagonalise it: iterate on Tp^T A Tp and accumulate the rotations onto Tp (2-3 sweeps instead
        // of ~8).  T diag(lam) T^T is gauge-free, so the result is as valid as a cold start.
        for (int idx = tid; idx < RR; idx += nth) Ts[0][idx / R][idx % R] = Tout[(size_t)d * RR + idx];
        __syncthreads();
        for (int idx = tid; idx < RR; idx += nth) {            // B = A Tp
            const int i = idx / R, j = idx - i * R;
            double acc = 0.0;
            for (int k = 0; k < R; k++) acc = fma(As[0][i][k], Ts[0][k][j], acc);
            As[1][i][j] = acc;
        }
        __syncthreads();
        for (int idx = tid; idx < RR; idx += nth) {            // A' = Tp^T B, upper part mirrored
            const int i = idx / R, j = idx - i * R;
            if (i <= j) {
                double acc = 0.0;
                for (int k = 0; k < R; k++) acc = fma(Ts[0][k][i], As[1][k][j], acc);
                As[0][i][j] = acc;
                As[0][j][i] = acc;
            }
        }
        __syncthreads();
    }
    if (tid < 32) {
        double nr = 0.0;
        for (int idx = tid; idx < RR; idx += 32) { const double v = As[0][idx / R][idx % R]; nr += v * v; }
        nr = warp_sum(nr);
        if (tid == 0) s_nrm2 = nr;
    }
    __syncthreads();
    const double nrm2 = s_nrm2;
    const int m = R + (R & 1), half = m >> 1;
    int cur = 0;
    bool converged = false;
    for (int sweep = 0; sweep < 40; sweep++) {
        double myoff = 0.0;                                     // sum of apq^2 met by this thread's pairs
        for (int r = 0; r < m - 1; r++) {
            if (tid < half) {
                int p = tid == 0 ? m - 1 : (r + tid) % (m - 1);
                int q = (r + m - 1 - tid) % (m - 1);
                if (p > q) { const int t = p; p = q; q = t; }
                if (q >= R) {                                   // paired with the padding index: untouched
                    alpha[p] = 1.0; beta[p] = 0.0; part[p] = p;
                } else {
                    const double apq = As[cur][p][q];
                    myoff += apq * apq;
                    double c = 1.0, sn = 0.0;
                    if (apq * apq > 1e-40 * nrm2) {
                        // tan of the rotation angle, t = sgn(theta) / (|theta| + sqrt(theta^2 + 1)) with
                        // theta = (aqq - app) / (2 apq), written so that the dependent chain is two rsqrt and one divide:
                        // t = 2 apq sgn(d) / (|d| + sqrt(d^2 + 4 apq^2)),  c = 1 / sqrt(1 + t^2),  s = t c
                        const double d = As[cur][q][q] - As[cur][p][p], x2 = 2.0 * apq;
                        const double hh = fma(d, d, x2 * x2);
                        double r = rsqrt(hh);
                        r = r * fma(-0.5 * hh * r, r, 1.5);            // Newton step: rounding-level 1/sqrt
                        const double t = copysign(x2, x2 * d) / (fabs(d) + hh * r);
                        const double tt = fma(t, t, 1.0);
                        double rc = rsqrt(tt);
                        rc = rc * fma(-0.5 * tt * rc, rc, 1.5);
                        c = rc;
                        sn = t * rc;
                    }
                    alpha[p] = c; beta[p] = -sn; part[p] = q;   // new column p = c a_p - s a_q
                    alpha[q] = c; beta[q] = sn; part[q] = p;    // new column q = s a_p + c a_q
                }
            }
            __syncthreads();
            const int nxt = cur ^ 1;
            for (int idx = tid; idx < RR; idx += nth) {
                const int i = idx / R, j = idx - i * R;
                const int pi = part[i], pj = part[j];
                const double ai = alpha[i], bi = beta[i], aj = alpha[j], bj = beta[j];
                double v = ai * (aj * As[cur][i][j] + bj * As[cur][i][pj]) + bi * (aj * As[cur][pi][j] + bj * As[cur][pi][pj]);
                if (pi == j && i != j && (bi != 0.0)) v = 0.0;  // the rotated pair's off-diagonal entry is annihilated
                As[nxt][i][j] = v;
                Ts[nxt][i][j] = aj * Ts[cur][i][j] + bj * Ts[cur][i][pj];
            }
            cur = nxt;
            __syncthreads();
        }
        if (tid < DLR_RMAXS) sq[tid] = tid < half ? myoff : 0.0;
        __syncthreads();
        if (tid == 0) {
            double o = 0.0;
            for (int k = 0; k < half; k++) o += sq[k];
            s_off2 = o;
        }
        __syncthreads();
        // Converged when the off-diagonal norm MET in this sweep (before its rotations) is <= 1e-10 ||A||_F: cyclic Jacobi
        // converges quadratically, so after the rotations of this sweep it is at rounding level (<= ~1e-20 ||A||_F^2 / gap);
        // waiting until a sweep meets <= 1e-16 ||A||_F costs one more full sweep for nothing
        if (s_off2 <= DLR_EIG_TOL2 * nrm2) { converged = true; break; }
    }
    if (!converged && tid == 0) atomicAdd(status + 3, 1);      // sweep cap hit: reported as dlr_moments_t.eig_unconverged
    if (warm) {
        // one Newton-Schulz step T <- T (3 I - T^T T) / 2 keeps the accumulated T orthogonal to rounding level no matter
        // how many steps it has been carried along
        const int oth = cur ^ 1;
        for (int idx = tid; idx < RR; idx += nth) {            // G = T^T T
            const int i = idx / R, j = idx - i * R;
            double acc = 0.0;
            for (int k = 0; k < R; k++) acc = fma(Ts[cur][k][i], Ts[cur][k][j], acc);
            Ts[oth][i][j] = acc;
        }
        __syncthreads();
        for (int idx = tid; idx < RR; idx += nth) {            // T (1.5 I - 0.5 G), into the free half of As
            const int i = idx / R, j = idx - i * R;
            double acc = 0.0;
            for (int k = 0; k < R; k++) acc = fma(Ts[cur][i][k], Ts[oth][k][j], acc);
            As[oth][i][j] = 1.5 * Ts[cur][i][j] - 0.5 * acc;
        }
        __syncthreads();
        for (int idx = tid; idx < RR; idx += nth) {
            const int i = idx / R, j = idx - i * R;
            Tout[(size_t)d * RR + idx] = As[oth][i][j];
            if (i == j) lam[d * R + i] = As[cur][i][i];
        }
        return;
    }
    for (int idx = tid; idx < RR; idx += nth) {
        const int i = idx / R, j = idx - i * R;
        Tout[(size_t)d * RR + idx] = Ts[cur][i][j];
        if (i == j) lam[d * R + i] = As[cur][i][i];
    }
}

// ---------------------------------------------------------------------------------------------------------
// column sums of a flow result from the per-CTA sums of its last pass: out[c] = sum_b part[b][c]
__global__ void __launch_bounds__(DLR_SMALL_THREADS) k_colsum_reduce(const double* part, int nblocks, int R, double* out) {
    __shared__ double red[DLR_RMAXS], tmp[DLR_SMALL_THREADS];
    cta_reduce_rows(part, nblocks, R, 0, R, red, tmp);
    if (threadIdx.x < R) out[threadIdx.x] = red[threadIdx.x];
}

// ---------------------------------------------------------------------------------------------------------
// diagnostics
// column sums with weights {1, w1, w2, w3, |w|^2} (w = grid coordinate), two levels, fixed order:
//   k_colmoments: grid (R, DLR_MCH); CTA (c, ch) sums a contiguous range of rows (lines along i1) of column c,
//   one warp per row -> part[(c*DLR_MCH + ch)*5 + m];   k_colmoments_sum adds the DLR_MCH chunks -> out[c*5 + m].
#define DLR_MCH 32
__global__ void __launch_bounds__(256) k_colmoments(const double* A, GridDev g, double* part) {
    __shared__ double red[5][8];
    const int c = blockIdx.x, ch = blockIdx.y, n = g.n, lg = g.log2n;
    const int rows = n << lg;                                   // n^2 rows of n points
    const int per = (rows + DLR_MCH - 1) / DLR_MCH;
    const int r0 = ch * per, r1 = min(rows, r0 + per);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const double* col = A + (size_t)c * g.N;
    double s[5] = {0, 0, 0, 0, 0};
    for (int q = r0 + w; q < r1; q += nw) {
        const int i2 = q & (n - 1), i3 = q >> lg;
        const double w2 = g.lo + g.h * i2, w3 = g.lo + g.h * i3, w23 = w2 * w2 + w3 * w3;
        const double* row = col + ((size_t)q << lg);
        double t0 = 0.0, t1 = 0.0, t4 = 0.0;
        for (int i1 = lane; i1 < n; i1 += 32) {
            const double w1 = g.lo + g.h * i1, a = row[i1];
            t0 += a; t1 += a * w1; t4 += a * (w1 * w1);
        }
        s[0] += t0; s[1] += t1; s[2] += t0 * w2; s[3] += t0 * w3; s[4] += t4 + t0 * w23;
    }
    for (int m = 0; m < 5; m++) { s[m] = warp_sum(s[m]); if (lane == 0) red[m][w] = s[m]; }
    __syncthreads();
    if (threadIdx.x < 5) {
        double t = 0.0;
        for (int i = 0; i < nw; i++) t += red[threadIdx.x][i];
        part[((size_t)c * DLR_MCH + ch) * 5 + threadIdx.x] = t;
    }
}

__global__ void k_colmoments_sum(const double* partx, const double* partv, int R, double* mx, double* mv) {
    for (int idx = threadIdx.x; idx < 2 * R * 5; idx += blockDim.x) {
        const int which = idx / (R * 5), e = idx - which * R * 5, c = e / 5, m = e - c * 5;
        const double* p = (which ? partv : partx) + (size_t)c * DLR_MCH * 5 + m;
        double t = 0.0;
        for (int ch = 0; ch < DLR_MCH; ch++) t += p[ch * 5];
        (which ? mv : mx)[e] = t;
    }
}

// partial sums of squares of nvals doubles -> out[blockIdx.x] (fixed order; k_moments_final adds the DLR_ECH parts)
#define DLR_ECH 64
__global__ void __launch_bounds__(256) k_sumsq(const double* a, long long nvals, double* out) {
    __shared__ double red[8];
    const long long per = (nvals + gridDim.x - 1) / gridDim.x;
    const long long i0 = (long long)blockIdx.x * per, i1 = min(nvals, i0 + per);
    double s = 0.0;
    for (long long i = i0 + threadIdx.x; i < i1; i += blockDim.x) s = fma(a[i], a[i], s);
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); i++) t += red[i];
        out[blockIdx.x] = t;
    }
}

// moments from the column moments; res: mass, mom1..3, kinetic, s_fro, nonfinite, sum |E|^2
__global__ void k_moments_final(const double* mx, const double* mv, const double* S, int R, double hx3, double hv3,
                                const double* epart, double* res) {
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
    double es = 0.0;
    for (int i = 0; i < DLR_ECH; i++) es += epart[i];
    res[0] = out[0]; res[1] = out[1]; res[2] = out[2]; res[3] = out[3]; res[4] = 0.5 * out[4];
    res[5] = sqrt(fro); res[6] = (double)bad; res[7] = es;
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

// ---------------------------------------------------------------------------------------------------------
// Predictor L step of Algorithm 2 without the flow.  Line 2 of Algorithm 2 needs of L1 only its column sums
// (rho = -X (L^T omega_v), eq. (13)).  Every operation of the Lie L-flow is linear and separable:
// the exact sub-flow along direction d preserves the marginal sums over the other directions and acts on the marginal
// along d as the same 1D shift; the exponential-Euler stage changes the total only by t * sum_points N(m), and
// N(m) = sum_i v_i o (m Q_i) needs the first moments sum_points v_i m only.  So the column sums of L1 follow from the three
// 1D marginals of V (3 n r numbers), n-point DFTs and r x r products - mathematically the same numbers as the full flow.
//
// k_marginals: grid (n, R): CTA (i3, c) sums the plane (i1, i2) of column c:  p1[(c n + i3) n + i1] = sum_i2 A,
//              p2[(c n + i3) n + i2] = sum_i1 A.   k_marg_reduce: M1[c][i1], M2[c][i2] = sums over i3; M3[c][i3] = sum_i2 p2.
__global__ void __launch_bounds__(256) k_marginals(const double* A, GridDev g, double* p1, double* p2) {
    __shared__ double cs[8][256];
    const int n = g.n, lg = g.log2n, i3 = blockIdx.x, c = blockIdx.y;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const double* plane = A + (size_t)c * g.N + ((size_t)i3 << (2 * lg));
    double col[8] = {0, 0, 0, 0, 0, 0, 0, 0};                    // column sums of this warp's rows, i1 = lane + 32 k
    double* row2 = p2 + ((size_t)c * n + i3) * n;
    for (int i2 = w; i2 < n; i2 += nw) {
        const double* row = plane + ((size_t)i2 << lg);
        double rs = 0.0;
#pragma unroll
        for (int k = 0; k < 8; k++) {
            const int i1 = lane + 32 * k;
            if (i1 < n) { const double v = row[i1]; col[k] += v; rs += v; }
        }
        rs = warp_sum(rs);
        if (lane == 0) row2[i2] = rs;
    }
#pragma unroll
    for (int k = 0; k < 8; k++) cs[w][lane + 32 * k] = col[k];
    __syncthreads();
    for (int i1 = threadIdx.x; i1 < n; i1 += blockDim.x) {
        double s = 0.0;
        for (int ww = 0; ww < nw; ww++) s += cs[ww][i1];
        p1[((size_t)c * n + i3) * n + i1] = s;
    }
}

// grid (R, 3): CTA (c, which).  which 0, 1: M[c][i] = sum_k p[(c n + k) n + i] (coalesced in i, four k-groups per i);
// which 2: M3[c][i3] = sum_i2 p2[(c n + i3) n + i2] (one warp per row, lanes along i2).
// Then what k_lpred_sums needs of the marginals and does not depend on the coupling matrix (so it runs here, on the
// side branch, long before the predictor's S step):  which 0, 1: Ph[c][k] = sum_i M[c][i] e^{-2 pi i ik/n} (n-point DFT
// by its definition), which 0 also s0[c] = sum_i M1[c][i];  which 2: mom3[c] = sum_i v(i) M3[c][i], and CTA (0, 2) the
// grid constant Wv[k] = sum_i v(i) e^{+2 pi i ik/n}.
__global__ void __launch_bounds__(256) k_marg_reduce(const double* p1, const double* p2, GridDev g, MargOut o) {
    __shared__ double red[256];
    __shared__ double Ms[256];
    __shared__ double2 twf[256];
    const int n = g.n, c = blockIdx.x, which = blockIdx.y, tid = threadIdx.x;
    for (int m = tid; m < n; m += blockDim.x) {              // exp(-2 pi i m / n), full circle
        const double2 w = m < (n >> 1) ? g.tw[m] : g.tw[m - (n >> 1)];
        twf[m] = m < (n >> 1) ? w : make_double2(-w.x, -w.y);
    }
    if (which < 2) {
        const double* p = (which == 0 ? p1 : p2) + (size_t)c * n * n;
        double* M = (which == 0 ? o.M1 : o.M2) + (size_t)c * n;
        const int ng = max(1, (int)blockDim.x / n);              // k-groups
        for (int i0 = 0; i0 < n; i0 += blockDim.x) {
            const int i = i0 + (tid % n), kg = tid / n;
            double s = 0.0;
            if (i < n && kg < ng)
                for (int k = kg; k < n; k += ng) s += p[(size_t)k * n + i];
            red[tid] = s;
            __syncthreads();
            if (tid < n && i0 + tid < n) {
                double t = 0.0;
                for (int gq = 0; gq < ng; gq++) t += red[gq * n + tid];
                M[i0 + tid] = t;
                Ms[i0 + tid] = t;
            }
            __syncthreads();
        }
        double2* Ph = (which == 0 ? o.Ph1 : o.Ph2) + (size_t)c * n;
        for (int k = tid; k < n; k += blockDim.x) {
            double2 fh = make_double2(0.0, 0.0);
            for (int i = 0; i < n; i++) {
                const double2 w = twf[(i * k) & (n - 1)];
                fh.x = fma(Ms[i], w.x, fh.x);
                fh.y = fma(Ms[i], w.y, fh.y);
            }
            Ph[k] = fh;
        }
        if (which == 0 && tid == 0) {
            double a = 0.0;
            for (int i = 0; i < n; i++) a += Ms[i];
            o.s0[c] = a;
        }
    } else {
        const int lane = tid & 31, w = tid >> 5, nw = blockDim.x >> 5;
        for (int i = w; i < n; i += nw) {
            const double* row = p2 + ((size_t)c * n + i) * n;
            double s = 0.0;
            for (int k = lane; k < n; k += 32) s += row[k];
            s = warp_sum(s);
            if (lane == 0) { o.M3[(size_t)c * n + i] = s; Ms[i] = s; }
        }
        __syncthreads();
        if (tid == 0) {
            double b = 0.0;
            for (int i = 0; i < n; i++) b = fma(g.lo + g.h * i, Ms[i], b);
            o.mom3[c] = b;
        }
        if (c == 0) {
            for (int k = tid; k < n; k += blockDim.x) {
                double2 s = make_double2(0.0, 0.0);
                for (int i = 0; i < n; i++) {
                    const double2 wv = twf[(i * k) & (n - 1)];
                    const double v = g.lo + g.h * i;
                    s.x = fma(v, wv.x, s.x);
                    s.y = fma(v, -wv.y, s.y);                     // conjugate: e^{+...}
                }
                o.Wv[k] = s;
            }
        }
    }
}
