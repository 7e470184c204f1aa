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
    const double *Tm, *lam, *Sin; int transS; GridDev g; double sgn, tsub, t3; const double* M2c; double nlsign;
    FlowTabPtrs o;
};

__host__ __device__ constexpr int post_smem_doubles(int R) { return 21 * R * R + 8; }

template <int R>
__global__ void __launch_bounds__(DLR_POST_THREADS) k_post(const PostArgs a) {
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
                    rhs = (r0 + r1) + r2;
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
    k_post<R><<<a.do_tab ? 5 : 1, DLR_POST_THREADS, post_smem_doubles(R) * sizeof(double), st>>>(a);
    return cudaGetLastError();
}
