// The r x r work between two streaming phases in ONE launch of five independent CTAs (rank-templated: every inner loop
// over the rank is unrolled, the operands sit in shared memory):
//   CTA 0: do_m2 : derivative coefficients M2_i = h^3 A^T d_i A (antisymmetric) from the totals of the
//                  1D Parseval sums of the three coefficient passes (pgram[d][P2], entry (a<b));
//          do_s  : S step, one classical RK4 step of eq. (10):
//                  dS/dt = sum_i D2_i S C1_i^T - D1_i S C2_i^T;
//          do_tab: mats[0] = Sin T1 (K = X S) or Sin^T T1 (L = V S^T) with the NEW S;
//   CTA 1: do_tab: the other mode-mixing matrices (products of the eigenvector matrices of C1_i^T / D1_i^T)
//                  and the real-space term in the eigenbasis of direction 3, Q_i = T3^T nl_i^T T3 (eqs. (9), (11), (16));
//   CTA 2, 3: do_tab: phases exp(s i t k~ lambda_j) of the exact sub-flows 1 and 2 (eqs. (17), (18));
//   CTA 4: do_tab: e^z, t phi1, t (phi1 - phi2), t phi2 of the exponential Runge-Kutta stage (eq. (19), reading R8).
// The paper's own S step is latency-bound on the GPU (0.65 ms); here the whole launch is ~6 us.
#pragma once
#include "flowtab.cuh"

#define DLR_POST_THREADS 512

struct PostArgs {
    int R, do_m2, do_s, do_tab;
    const double* pgram[3]; double m2scale; double* M2;
    double* S; double ts; const double *C1, *C2, *D1, *D2;
    double ssign;           // +1: eq. (10) as printed (the backward sub-flow of the projector splitting); -1: the forward Galerkin
                            // S step of the unconventional integrator (oracle.S_flow_forward)
    const double *Tm, *lam, *Sin; int transS; GridDev g; double sgn, tsub, t3; const double* M2c; double nlsign;
    FlowTabPtrs o;
};

__host__ __device__ constexpr int post_smem_doubles(int R) { return 21 * R * R + 8; }

template <int R>
__global__ void __launch_bounds__(DLR_POST_THREADS) k_post(const PostArgs a) {
    pdl_wait();
    pdl_trigger();
    constexpr int RR = R * R, P2 = R * (R - 1) / 2;
    extern __shared__ double psm[];
    const int tid = threadIdx.x, nth = blockDim.x;
    const int job = blockIdx.x;

    // antisymmetric M2_d from the packed upper sums, entry idx = i * R + j
    const auto m2_entry = [&](int d, int idx) {
        const int i = idx / R, j = idx - i * R;
        if (i == j) return 0.0;
        const int lo = i < j ? i : j, hi = i < j ? j : i;
        const double v = a.m2scale * a.pgram[d][lo * (R - 1) - lo * (lo - 1) / 2 + (hi - lo - 1)];
        return i > j ? -v : v;
    };
    (void)P2;

    if (job == 0) {
        double* C1 = psm;                 // [3][RR] each: C1, C2, D1, D2 (row-major M[a * R + b])
        double* C2 = C1 + 3 * RR;
        double* D1 = C2 + 3 * RR;
        double* D2 = D1 + 3 * RR;
        double* Sc = D2 + 3 * RR;         // S at the start of the step (column-major, like S)
        double* Y = Sc + RR;              // stage value
        double* Pm = Y + RR;              // [3][RR]: Y C1_d^T (row-major [a][b])
        double* Qm = Pm + 3 * RR;         // [3][RR]: Y C2_d^T
        double* T1s = Qm + 3 * RR;        // [RR]
        if (a.do_s) {
            for (int i = tid; i < 3 * RR; i += nth) { C1[i] = a.C1[i]; C2[i] = a.C2[i]; D1[i] = a.D1[i]; D2[i] = a.D2[i]; }
        }
        if (a.do_m2) {
            for (int i = tid; i < 3 * RR; i += nth) {
                const double v = m2_entry(i / RR, i % RR);
                a.M2[i] = v;
                if (a.do_s) { if (a.M2 == a.C2) C2[i] = v; else if (a.M2 == a.D2) D2[i] = v; }
            }
        }
        if (a.do_tab) for (int i = tid; i < RR; i += nth) T1s[i] = a.Tm[i];
        if (a.do_s || a.do_tab) {
            const double* Ssrc = a.do_s ? a.S : a.Sin;
            for (int i = tid; i < RR; i += nth) { const double s = Ssrc[i]; Sc[i] = s; Y[i] = s; }
        }
        __syncthreads();
        if (a.do_s) {
            const double t = a.ts;
            double kacc = 0.0;                                  // entry idx (one per thread; RR <= blockDim.x)
            const double cw[4] = {1.0, 2.0, 2.0, 1.0}, cs[4] = {0.5, 0.5, 1.0, 0.0};
#pragma unroll 1
            for (int stage = 0; stage < 4; stage++) {
                if (tid < RR) {
                    const int aa = tid / R, b = tid - aa * R;
                    double p[3] = {0, 0, 0}, q[3] = {0, 0, 0};
#pragma unroll
                    for (int k = 0; k < R; k++) {
                        const double y = Y[aa + R * k];
#pragma unroll
                        for (int d = 0; d < 3; d++) {
                            p[d] = fma(y, C1[d * RR + b * R + k], p[d]);
                            q[d] = fma(y, C2[d * RR + b * R + k], q[d]);
                        }
                    }
#pragma unroll
                    for (int d = 0; d < 3; d++) { Pm[d * RR + tid] = p[d]; Qm[d * RR + tid] = q[d]; }
                }
                __syncthreads();
                double rhs = 0.0;
                if (tid < RR) {
                    const int aa = tid % R, b = tid / R;        // column-major entry (aa, b)
                    double r0 = 0.0, r1 = 0.0, r2 = 0.0;
#pragma unroll
                    for (int k = 0; k < R; k++) {
                        r0 = fma(D2[0 * RR + aa * R + k], Pm[0 * RR + k * R + b], r0);
                        r1 = fma(D2[1 * RR + aa * R + k], Pm[1 * RR + k * R + b], r1);
                        r2 = fma(D2[2 * RR + aa * R + k], Pm[2 * RR + k * R + b], r2);
                        r0 = fma(-D1[0 * RR + aa * R + k], Qm[0 * RR + k * R + b], r0);
                        r1 = fma(-D1[1 * RR + aa * R + k], Qm[1 * RR + k * R + b], r1);
                        r2 = fma(-D1[2 * RR + aa * R + k], Qm[2 * RR + k * R + b], r2);
                    }
                    rhs = a.ssign * ((r0 + r1) + r2);
                    kacc = fma(cw[stage], rhs, kacc);
                    Y[tid] = stage < 3 ? fma(cs[stage] * t, rhs, Sc[tid]) : fma(t / 6.0, kacc, Sc[tid]);
                }
                __syncthreads();
            }
            if (tid < RR) a.S[tid] = Y[tid];
        }
        if (a.do_tab && tid < RR) {
            // mats[0][a][b] = sum_k S(a,k) T1[k][b]  (transS: S(k,a));  S column-major, the NEW S when do_s
            const bool same = (a.Sin == a.S) || !a.do_s;
            const int aa = tid / R, b = tid - aa * R;
            double m0 = 0.0;
#pragma unroll
            for (int k = 0; k < R; k++) {
                const double s = same ? (a.transS ? Y[k + R * aa] : Y[aa + R * k])
                                      : (a.transS ? a.Sin[k + R * aa] : a.Sin[aa + R * k]);
                m0 = fma(s, T1s[k * R + b], m0);
            }
            a.o.mats[tid] = m0;
        }
        return;
    }
    if (!a.do_tab) return;
    if (job == 1) {
        double* T1 = psm;
        double* T2 = T1 + RR;
        double* T3 = T2 + RR;
        double* nls = T3 + RR;            // [3][RR]
        double* tmpm = nls + 3 * RR;      // [3][RR]: nl_i^T T3
        for (int i = tid; i < 3 * RR; i += nth) psm[i] = a.Tm[i];
        const bool local_m2 = a.do_m2 && a.M2c == a.M2;          // CTA 0 is writing M2 right now: rebuild it here
        for (int i = tid; i < 3 * RR; i += nth) nls[i] = local_m2 ? m2_entry(i / RR, i % RR) : a.M2c[i];
        __syncthreads();
        if (tid < RR) {
            const int aa = tid / R, b = tid - aa * R;
            double m1 = 0, m2 = 0, m5 = 0, m6 = 0;
#pragma unroll
            for (int k = 0; k < R; k++) {
                m1 = fma(T1[k * R + aa], T2[k * R + b], m1);
                m2 = fma(T2[k * R + aa], T3[k * R + b], m2);
                m5 = fma(T3[k * R + aa], T2[k * R + b], m5);
                m6 = fma(T2[k * R + aa], T1[k * R + b], m6);
            }
            a.o.mats[1 * RR + tid] = m1;
            a.o.mats[2 * RR + tid] = m2;
            a.o.mats[3 * RR + tid] = T3[b * R + aa];
            a.o.mats[4 * RR + tid] = T3[tid];
            a.o.mats[5 * RR + tid] = m5;
            a.o.mats[6 * RR + tid] = m6;
            a.o.mats[7 * RR + tid] = T1[b * R + aa];
        }
        // N(A) T3 = sum_i diag(w_i) (A T3) (T3^T nl_i^T T3):  Q_i = nlsign T3^T (M2c_i^T T3)
        for (int idx = tid; idx < 3 * RR; idx += nth) {
            const int d = idx / RR, e = idx - d * RR, pp = e / R, b = e - pp * R;
            double t = 0.0;
#pragma unroll
            for (int qq = 0; qq < R; qq++) t = fma(nls[d * RR + qq * R + pp], T3[qq * R + b], t);
            tmpm[idx] = t;
        }
        __syncthreads();
        for (int idx = tid; idx < 3 * RR; idx += nth) {
            const int d = idx / RR, e = idx - d * RR, aa = e / R, b = e - aa * R;
            double q = 0.0;
#pragma unroll
            for (int pp = 0; pp < R; pp++) q = fma(T3[pp * R + aa], tmpm[d * RR + pp * R + b], q);
            a.o.Q[idx] = a.nlsign * q;
        }
        return;
    }
    // phase / phi tables, by stored (bit-reversed) position k and column j
    const int n = a.g.n;
    if (job == 2 || job == 3) {
        const double* lam = a.lam + (job - 2) * R;
        double2* ph = job == 2 ? a.o.ph1 : a.o.ph2;
        const double f = a.sgn * a.tsub;
        for (int idx = tid; idx < n * R; idx += nth) {
            const int k = idx / R, j = idx - k * R;
            double sn, cs;
            sincos(f * a.g.kt2p[k] * lam[j], &sn, &cs);
            ph[idx] = make_double2(cs, sn);
        }
        return;
    }
    {
        const double* lam = a.lam + 2 * R;
        const double t3 = a.t3;
        for (int idx = tid; idx < n * R; idx += nth) {
            const int k = idx / R, j = idx - k * R;
            const double th = a.sgn * t3 * a.g.kt2p[k] * lam[j];
            double sn, cs;
            sincos(th, &sn, &cs);
            a.o.ez[idx] = make_double2(cs, sn);
            double2 p1, p2;
            phi12_imag(th, p1, p2);
            a.o.f1[idx] = make_double2(t3 * p1.x, t3 * p1.y);
            a.o.f2a[idx] = make_double2(t3 * (p1.x - p2.x), t3 * (p1.y - p2.y));
            a.o.f2b[idx] = make_double2(t3 * p2.x, t3 * p2.y);
        }
    }
}

template <int R>
inline cudaError_t launch_post(const PostArgs& a, cudaStream_t st) {
    static_assert(R * R <= DLR_POST_THREADS, "one thread per matrix entry");
    return dlr_launch(k_post<R>, a.do_tab ? 5 : 1, DLR_POST_THREADS, post_smem_doubles(R) * sizeof(double), st, a);
}

// ---------------------------------------------------------------------------------------------------------
// Predictor L step of Algorithm 2 without the flow.  Line 2 of Algorithm 2 needs of L1 only its column sums
// (rho = -X (L^T omega_v), eq. (13)).  Every operation of the Lie L-flow is linear and separable:
// the exact sub-flow along direction d preserves the marginal sums over the other directions and acts on the marginal
// along d as the same 1D shift; the exponential-Euler stage changes the total only by t * sum_points N(m), and
// N(m) = sum_i v_i o (m Q_i) needs the first moments sum_points v_i m only.  So the column sums of L1 follow from the three
// 1D marginals of V (3 n r numbers), n-point DFTs and r x r products - mathematically the same numbers as the full flow.
// The DFTs of the marginals do not depend on the coupling matrix and are done beside the coefficient passes
// (k_marg_reduce); here only the mixing with the matrices of the L-flow (built by k_post from the predictor's S) is left:
//   nu_d[c] = (1/n) Re sum_k ph_d[k][c] W_k sum_k' Ph_d[k'][k] B_d[k'][c],   B_1 = A0,  B_2 = A0 A1.
// Single CTA.  zsum[c] = sum_points L1_c (no h^3 weight).
struct LpredArgs {
    MargOut m;
    FlowTabPtrs tb;
    GridDev g;
    double t3;
    double* zsum;
};

__host__ __device__ constexpr size_t lpred_smem_bytes(int R, int n) { return (size_t)(8 * R * R + 2 * R * n + 8 * R + 8) * 8; }

template <int R>
__global__ void __launch_bounds__(DLR_POST_THREADS) k_lpred_sums(const LpredArgs a) {
    pdl_wait();
    pdl_trigger();
    constexpr int RR = R * R;
    extern __shared__ double psm[];
    const int n = a.g.n, lg = a.g.log2n, tid = threadIdx.x, nth = blockDim.x;
    double* msm = psm;                  // [7][RR]: A0, A1, A2, A3, Q1..3
    double* B1 = msm + 7 * RR;          // [RR] A0 A1
    double* parts = B1 + RR;            // [2][R][n]
    double* vec = parts + 2 * R * n;    // 8 x [R]
    for (int i = tid; i < 4 * RR; i += nth) msm[i] = a.tb.mats[i];
    for (int i = tid; i < 3 * RR; i += nth) msm[4 * RR + i] = a.tb.Q[i];
    __syncthreads();
    const double* A0 = msm;
    const double* A1 = msm + RR;
    const double* A2 = msm + 2 * RR;
    const double* A3 = msm + 3 * RR;
    const double* Qs = msm + 4 * RR;
    if (tid < RR) {
        const int aa = tid / R, b = tid - aa * R;
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < R; k++) s = fma(A0[aa * R + k], A1[k * R + b], s);
        B1[tid] = s;
    }
    __syncthreads();
    for (int idx = tid; idx < 2 * R * n; idx += nth) {
        const int d = idx / (R * n), e = idx - d * R * n, c = e / n, k = e - c * n;
        const double2* Ph = (d == 0 ? a.m.Ph1 : a.m.Ph2) + k;
        const double* B = (d == 0 ? A0 : B1) + c;
        double2 fh = make_double2(0.0, 0.0);
#pragma unroll
        for (int kk = 0; kk < R; kk++) {
            const double2 p = Ph[(size_t)kk * n];
            const double bb = B[kk * R];
            fh.x = fma(p.x, bb, fh.x);
            fh.y = fma(p.y, bb, fh.y);
        }
        const int ep = (int)(__brev((unsigned)k) >> (32 - lg));           // stored position of wavenumber index k
        const double2 ph = (d == 0 ? a.tb.ph1 : a.tb.ph2)[(size_t)ep * R + c];
        parts[idx] = cmul(cmul(ph, fh), a.m.Wv[k]).x;
    }
    __syncthreads();
    double *s0 = vec, *mom3 = vec + R, *nu1 = vec + 2 * R, *nu2 = vec + 3 * R, *ta = vec + 4 * R, *tb2 = vec + 5 * R,
           *acc = vec + 6 * R, *tmpv = vec + 7 * R;
    {
        const int lane = tid & 31, w = tid >> 5, nw = nth >> 5;
        for (int row = w; row < 2 * R; row += nw) {
            double s = 0.0;
            for (int k = lane; k < n; k += 32) s += parts[row * n + k];
            s = warp_sum(s);
            if (lane == 0) (row < R ? nu1 : nu2)[row < R ? row : row - R] = s / (double)n;
        }
        if (tid < R) { s0[tid] = a.m.s0[tid]; mom3[tid] = a.m.mom3[tid]; }
    }
    __syncthreads();
    if (tid >= 32) return;
    // r-vector chain (row vector times matrix, [cin][cout]) by one warp
    const auto vm = [&](const double* v, const double* Mx, double* out) {
        double s = 0.0;
        if (tid < R) {
#pragma unroll
            for (int k = 0; k < R; k++) s = fma(v[k], Mx[k * R + tid], s);
        }
        __syncwarp();
        if (tid < R) out[tid] = s;
        __syncwarp();
    };
    vm(s0, A0, ta); vm(ta, A1, tb2); vm(tb2, A2, acc);          // acc = sum_points m
    vm(mom3, A0, ta); vm(ta, A1, tb2); vm(tb2, A2, mom3);       // mu_3
    vm(nu2, A2, ta);                                            // mu_2 -> ta
    vm(nu1, A1, tb2); vm(tb2, A2, nu1);                         // mu_1
    if (tid < R) {
        double gsum = 0.0;
#pragma unroll
        for (int k = 0; k < R; k++)
            gsum += nu1[k] * Qs[k * R + tid] + ta[k] * Qs[RR + k * R + tid] + mom3[k] * Qs[2 * RR + k * R + tid];
        tmpv[tid] = acc[tid] + a.t3 * gsum;
    }
    __syncwarp();
    vm(tmpv, A3, a.zsum);
}

template <int R>
inline cudaError_t launch_lpred(const LpredArgs& a, cudaStream_t st) {
    return dlr_launch(k_lpred_sums<R>, 1, DLR_POST_THREADS, lpred_smem_bytes(R, a.g.n), st, a);
}
