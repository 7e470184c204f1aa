// Dimension-3 pass: a tile of pencils along k3 of ALL columns sits in shared memory; forward FFT along k3 completes
// the 3D transform, the Fourier-space part of the K/L flow is applied mode by mode across the columns
// (exact directional sub-flows, eqs. (14),(15),(17),(18); exponential Runge-Kutta stages of
// eq. (19)), and the inverse FFT along k3 starts the way back - one read and one write of the data.
#pragma once
#include "common.cuh"

enum {
    D3_FWD_STORE = 0,   // FFT3 -> store spectrum (factor transform), optional Parseval Gram for C2/D2
    D3_FLOW_START = 1,  // spectrum in (no FFT) -> sub-flows 1,2 -> eigenbasis of sub-flow 3; mbuf = e^z M; out = state for N()
    D3_EULER_END = 2,   // FFT3 of N(A) -> exponential Euler -> IFFT3
    D3_MID = 3,         // FFT3 of N(A) -> first ETD2RK stage, keeps the combination needed by the second -> IFFT3
    D3_END2 = 4,        // FFT3 of N(A_a) -> second ETD2RK stage -> sub-flows 2,1 -> IFFT3
    D3_POISSON = 5,     // FFT3 of rho -> E_hat (3 columns) -> IFFT3
    D3_INV_ONLY = 6     // spectrum in -> IFFT3 (tests)
};

struct D3Args {
    GridDev g;
    const double2* in;    // RIN columns, stride NC
    double2* out;         // ROUT columns (may alias in)
    double2* mbuf;        // R columns
    const double* mats;   // 8 x [R][R], [cin][cout]:  0 Sin*T1, 1 T1^T T2, 2 T2^T T3, 3 T3^T, 4 T3, 5 T3^T T2, 6 T2^T T1, 7 T1^T
    const double2* ph1;   // [nh][R] phases of sub-flow 1 by k1
    const double2* ph2;   // [n][R]  phases of sub-flow 2 by stored k2'
    const double2* ez;    // [n][R]  exp(z) of sub-flow 3 by stored k3'
    const double2* f1;    // [n][R]  t*phi1(z)
    const double2* f2;    // [n][R]  MID: t*(phi1-phi2)(z);  END2: t*phi2(z)
    double* partial;      // Parseval Gram partial sums [gridDim.x][3*R(R-1)/2]
    double* zero_out;     // optional [R]: real part of the k = 0 mode of the result (before the inverse transform)
    double e_scale;
    int T;                // pencils per CTA
    int skip_store;       // EULER_END: only zero_out is wanted
    int threads;          // CTA size (0 = DLR_THREADS); must be a multiple of T
};

__host__ inline size_t d3_smem_bytes(int n, int RMAX, int T, int nmat) {
    const int LP = (RMAX * T) | 1;
    return (size_t)n * LP * 16 + (size_t)(n / 2) * 16 + (size_t)nmat * 8 + 16;
}

template <int R>
__device__ __forceinline__ void matvec_c(double2 (&x)[R], const double* A) {     // x <- x * A, A[cin][cout]
    double2 y[R];
#pragma unroll
    for (int co = 0; co < R; co++) {
        double2 acc = make_double2(0.0, 0.0);
#pragma unroll
        for (int ci = 0; ci < R; ci++) {
            const double m = A[ci * R + co];
            acc.x = fma(m, x[ci].x, acc.x);
            acc.y = fma(m, x[ci].y, acc.y);
        }
        y[co] = acc;
    }
#pragma unroll
    for (int c = 0; c < R; c++) x[c] = y[c];
}

template <int R>
__device__ __forceinline__ void phase_c(double2 (&x)[R], const double2* ph) {
#pragma unroll
    for (int c = 0; c < R; c++) x[c] = cmul(x[c], __ldg(ph + c));
}

template <int RIN, int ROUT, int FOP, bool PGRAM>
__global__ void __launch_bounds__(DLR_THREADS, ((RIN > ROUT ? RIN : ROUT) <= 10 ? 2 : 1)) k_d3(const D3Args a) {
    constexpr int RMAX = RIN > ROUT ? RIN : ROUT;
    constexpr int R = RIN;
    constexpr int NMAT = (FOP == D3_FWD_STORE || FOP == D3_POISSON || FOP == D3_INV_ONLY) ? 0 : 4 * R * R;
    const int n = a.g.n, nh = a.g.nh, lg = a.g.log2n, T = a.T;
    const int lt = __ffs(T) - 1;                                 // T is a power of two
    const int LP = (RMAX * T) | 1;
    const int plane = nh * n;                                    // pencils per column (<= 129 * 256)
    const int p0 = (int)blockIdx.x * T;
    const int tw_ = min(T, plane - p0);                          // valid pencils in this tile
    const FastDiv fnh = make_fastdiv((unsigned)nh);
    extern __shared__ double2 smem2[];
    double2* z = smem2;
    double2* tw = z + (size_t)n * LP;
    double* mats = (double*)(tw + n / 2);
    const int tid = threadIdx.x, nth = blockDim.x;
    for (int i = tid; i < n / 2; i += nth) tw[i] = a.g.tw[i];
    if (NMAT) {
        // the four matrices this variant uses, in order of use
        const int m0 = FOP == D3_FLOW_START ? 0 : 4;
        const int sel[4] = {m0, FOP == D3_FLOW_START ? 1 : (FOP == D3_END2 ? 5 : 3), FOP == D3_FLOW_START ? 2 : 6,
                            FOP == D3_FLOW_START ? 3 : 7};
        for (int i = tid; i < 4 * R * R; i += nth) mats[i] = a.mats[sel[i / (R * R)] * R * R + i % (R * R)];
    }
    // ---- load
    {
        const int items = RIN * n * T;
        for (int w = tid; w < items; w += nth) {
            const int t = w & (T - 1), rest = w >> lt;
            const int e = rest & (n - 1), c = rest >> lg;
            z[(size_t)e * LP + c * T + t] =
                t < tw_ ? a.in[(size_t)c * a.g.NC + (size_t)e * plane + p0 + t] : make_double2(0.0, 0.0);
        }
    }
    __syncthreads();
    if (FOP != D3_FLOW_START && FOP != D3_INV_ONLY) fft_lines<false>(z, LP, RIN * T, a.g.log2n, tw, 1);

    // ---- Parseval Gram: C2_i[a][b] = (h^3/N) sum_k wgt(k1) kt_i (Im a Re b - Re a Im b), a<b
    if (PGRAM) {
        constexpr int P2 = R * (R - 1) / 2;
        const int warp = tid >> 5, lane = tid & 31, nwarp = nth >> 5;
        double* part = a.partial + (size_t)blockIdx.x * 3 * P2;
        const int items = n * T;
        for (int en = warp; en < P2; en += nwarp) {
            int ca = 0, rem = en;
            while (rem >= R - 1 - ca) { rem -= R - 1 - ca; ca++; }
            const int cb = ca + 1 + rem;
            double s0 = 0.0, s1 = 0.0, s2 = 0.0;
            for (int w = lane; w < items; w += 32) {
                const int t = w & (T - 1), e = w >> lt;
                if (t >= tw_) continue;
                const int p = p0 + t;
                const int k2 = (int)fdiv((unsigned)p, fnh), k1 = p - k2 * nh;
                const double2 za = z[(size_t)e * LP + ca * T + t], zb = z[(size_t)e * LP + cb * T + t];
                double q = za.y * zb.x - za.x * zb.y;
                if (k1 != 0 && k1 != nh - 1) q *= 2.0;
                s0 = fma(__ldg(a.g.kt1 + k1), q, s0);
                s1 = fma(__ldg(a.g.kt2p + k2), q, s1);
                s2 = fma(__ldg(a.g.kt2p + e), q, s2);
            }
            s0 = warp_sum(s0); s1 = warp_sum(s1); s2 = warp_sum(s2);
            if (lane == 0) { part[en] = s0; part[P2 + en] = s1; part[2 * P2 + en] = s2; }
        }
    }

    // ---- mode-wise operation across the columns
    if (FOP != D3_FWD_STORE) {
        const int items = FOP == D3_INV_ONLY ? 0 : n * T;
        // blockDim is a multiple of T, so a thread keeps its pencil t (and with it k1, k2) over the whole loop
        const int t = tid & (T - 1);
        const int p = p0 + t;
        const int k2 = (int)fdiv((unsigned)p, fnh), k1 = p - k2 * nh;
        for (int w = tid; w < items; w += nth) {
            const int e = w >> lt;
            if (t >= tw_) continue;
            double2* zp = z + (size_t)e * LP + t;
            if (FOP == D3_POISSON) {
                const double2 rho = zp[0];
                const double k2sum = __ldg(a.g.ksq1 + k1) + __ldg(a.g.ksq2p + k2) + __ldg(a.g.ksq2p + e);
                const double inv = k2sum > 0.0 ? a.e_scale / k2sum : 0.0;
                const double2 phi = make_double2(rho.x * inv, rho.y * inv);
                const double kk[3] = {__ldg(a.g.kt1 + k1), __ldg(a.g.kt2p + k2), __ldg(a.g.kt2p + e)};
#pragma unroll
                for (int d = 0; d < 3; d++) zp[d * T] = make_double2(phi.y * kk[d], -phi.x * kk[d]);   // -i k phi
                continue;
            }
            double2 x[R];
#pragma unroll
            for (int c = 0; c < R; c++) x[c] = zp[c * T];
            const size_t gofs = (size_t)e * plane + p0 + t;
            if (FOP == D3_FLOW_START) {
                matvec_c<R>(x, mats);
                phase_c<R>(x, a.ph1 + (size_t)k1 * R);
                matvec_c<R>(x, mats + R * R);
                phase_c<R>(x, a.ph2 + (size_t)k2 * R);
                matvec_c<R>(x, mats + 2 * R * R);
#pragma unroll
                for (int c = 0; c < R; c++)
                    a.mbuf[(size_t)c * a.g.NC + gofs] = cmul(x[c], __ldg(a.ez + (size_t)e * R + c));
                matvec_c<R>(x, mats + 3 * R * R);
            } else {
                matvec_c<R>(x, mats);                                    // G = F(N) T3
                if (FOP == D3_EULER_END) {
#pragma unroll
                    for (int c = 0; c < R; c++)
                        x[c] = cadd(a.mbuf[(size_t)c * a.g.NC + gofs], cmul(x[c], __ldg(a.f1 + (size_t)e * R + c)));
                    matvec_c<R>(x, mats + R * R);
                } else if (FOP == D3_MID) {
#pragma unroll
                    for (int c = 0; c < R; c++) {
                        const double2 mb = a.mbuf[(size_t)c * a.g.NC + gofs];
                        a.mbuf[(size_t)c * a.g.NC + gofs] = cadd(mb, cmul(x[c], __ldg(a.f2 + (size_t)e * R + c)));
                        x[c] = cadd(mb, cmul(x[c], __ldg(a.f1 + (size_t)e * R + c)));
                    }
                    matvec_c<R>(x, mats + R * R);
                } else {  // D3_END2
#pragma unroll
                    for (int c = 0; c < R; c++)
                        x[c] = cadd(a.mbuf[(size_t)c * a.g.NC + gofs], cmul(x[c], __ldg(a.f2 + (size_t)e * R + c)));
                    matvec_c<R>(x, mats + R * R);
                    phase_c<R>(x, a.ph2 + (size_t)k2 * R);
                    matvec_c<R>(x, mats + 2 * R * R);
                    phase_c<R>(x, a.ph1 + (size_t)k1 * R);
                    matvec_c<R>(x, mats + 3 * R * R);
                }
            }
            if (a.zero_out != nullptr && e == 0 && p == 0) {
#pragma unroll
                for (int c = 0; c < R; c++) a.zero_out[c] = x[c].x;
            }
#pragma unroll
            for (int c = 0; c < R; c++) zp[c * T] = x[c];
        }
        if (FOP == D3_EULER_END && a.skip_store) return;
        __syncthreads();
        fft_lines<true>(z, LP, ROUT * T, a.g.log2n, tw, 1);
    } else {
        __syncthreads();
    }
    // ---- store
    {
        const int items = ROUT * n * T;
        for (int w = tid; w < items; w += nth) {
            const int t = w & (T - 1), rest = w >> lt;
            const int e = rest & (n - 1), c = rest >> lg;
            if (t < tw_) a.out[(size_t)c * a.g.NC + (size_t)e * plane + p0 + t] = z[(size_t)e * LP + c * T + t];
        }
    }
}

template <int RIN, int ROUT, int FOP, bool PGRAM>
inline cudaError_t launch_d3(const D3Args& a, cudaStream_t st) {
    constexpr int RMAX = RIN > ROUT ? RIN : ROUT;
    constexpr int NMAT = (FOP == D3_FWD_STORE || FOP == D3_POISSON || FOP == D3_INV_ONLY) ? 0 : 4 * RIN * RIN;
    auto kern = k_d3<RIN, ROUT, FOP, PGRAM>;
    const size_t sm = d3_smem_bytes(a.g.n, RMAX, a.T, NMAT);
    static size_t configured = 0;
    if (sm > configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return e;
        configured = sm;
    }
    const long long plane = (long long)a.g.nh * a.g.n;
    const unsigned grid = (unsigned)((plane + a.T - 1) / a.T);
    kern<<<grid, a.threads > 0 ? a.threads : DLR_THREADS, sm, st>>>(a);
    return cudaGetLastError();
}
