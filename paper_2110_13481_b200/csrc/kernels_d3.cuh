// Dimension-3 pass of the single-column 3D FFT of the Poisson solve: a tile of pencils along k3
// sits in shared memory; the forward FFT along k3 completes the 3D transform of rho, the Poisson symbol and the
// gradient are applied mode by mode (E_hat = -i k~ rho_hat / |k|^2, readings R4, R6), and the inverse FFT along k3
// starts the way back - one read and one write of the data.
// (The K/L flows do not use this kernel: their sub-flows are the directional passes of kernels_dir.cuh.)
#pragma once
#include "common.cuh"

enum {
    D3_FWD_STORE = 0,   // FFT3 -> store the spectrum (test hook)
    D3_POISSON = 5,     // FFT3 of rho -> E_hat (3 columns) -> IFFT3
    D3_INV_ONLY = 6     // spectrum in -> IFFT3 (test hook)
};

struct D3Args {
    GridDev g;
    const double2* in;    // RIN columns, stride NC
    double2* out;         // ROUT columns (may alias in)
    double e_scale;
    int T;                // pencils per CTA (power of two)
    int threads;          // CTA size (0 = DLR_THREADS); must be a multiple of T
};

__host__ inline size_t d3_smem_bytes(int n, int RMAX, int T, int nmat) {
    const int LP = (RMAX * T) | 1;
    return (size_t)n * LP * 16 + (size_t)(n / 2) * 16 + (size_t)nmat * 8 + 16;
}

template <int RIN, int ROUT, int FOP, bool UNUSED>
__global__ void __launch_bounds__(DLR_THREADS, 2) k_d3(const D3Args a) {
    pdl_wait();
    pdl_trigger();
    constexpr int RMAX = RIN > ROUT ? RIN : ROUT;
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
    const int tid = threadIdx.x, nth = blockDim.x;
    for (int i = tid; i < n / 2; i += nth) tw[i] = a.g.tw[i];
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
    if (FOP != D3_INV_ONLY) fft_lines<false>(z, LP, RIN * T, lg, tw, 1);
    // ---- Poisson symbol and gradient, mode by mode
    if (FOP == D3_POISSON) {
        // blockDim is a multiple of T, so a thread keeps its pencil t (and with it k1, k2) over the whole loop
        const int t = tid & (T - 1);
        const int p = p0 + t;
        const int k2 = (int)fdiv((unsigned)p, fnh), k1 = p - k2 * nh;
        for (int w = tid; w < n * T; w += nth) {
            const int e = w >> lt;
            if (t >= tw_) continue;
            double2* zp = z + (size_t)e * LP + t;
            const double2 rho = zp[0];
            const double k2sum = __ldg(a.g.ksq1 + k1) + __ldg(a.g.ksq2p + k2) + __ldg(a.g.ksq2p + e);
            const double inv = k2sum > 0.0 ? a.e_scale / k2sum : 0.0;
            const double2 phi = make_double2(rho.x * inv, rho.y * inv);
            const double kk[3] = {__ldg(a.g.kt1 + k1), __ldg(a.g.kt2p + k2), __ldg(a.g.kt2p + e)};
#pragma unroll
            for (int d = 0; d < 3; d++) zp[d * T] = make_double2(phi.y * kk[d], -phi.x * kk[d]);   // -i k phi
        }
    }
    if (FOP != D3_FWD_STORE) {
        __syncthreads();
        fft_lines<true>(z, LP, ROUT * T, lg, tw, 1);
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

template <int RIN, int ROUT, int FOP, bool UNUSED>
inline cudaError_t launch_d3(const D3Args& a, cudaStream_t st) {
    constexpr int RMAX = RIN > ROUT ? RIN : ROUT;
    auto kern = k_d3<RIN, ROUT, FOP, UNUSED>;
    const size_t sm = d3_smem_bytes(a.g.n, RMAX, a.T, 0);
    const long long plane = (long long)a.g.nh * a.g.n;
    const unsigned grid = (unsigned)((plane + a.T - 1) / a.T);
    return dlr_launch(kern, grid, a.threads > 0 ? a.threads : DLR_THREADS, sm, st, a);
}
