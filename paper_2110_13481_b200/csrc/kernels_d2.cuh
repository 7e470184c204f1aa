// Dimension-2 pass: in-place complex FFT (forward: natural -> bit-reversed positions; inverse: the transpose)
// along k2 of the half spectrum Ah[c][k3'][k2][k1].  Columns are independent here, so a CTA takes NB (column, k3)
// slabs and a chunk of T2 consecutive k1 (contiguous in memory).
#pragma once
#include "common.cuh"

struct D2Args {
    GridDev g;
    double2* data;       // ncols columns, stride NC
    int ncols;
    int T2, NB, nchunks; // k1 chunk width, slabs per CTA, ceil(nh / T2)
};

__host__ inline size_t d2_smem_bytes(int n, int T2, int NB) {
    const int LP = (T2 * NB) | 1;
    return (size_t)n * LP * 16 + (size_t)(n / 2) * 16 + 16;
}

template <bool INV>
__global__ void __launch_bounds__(DLR_THREADS) k_d2(const D2Args a) {
    const int n = a.g.n, nh = a.g.nh, T2 = a.T2, NB = a.NB;
    const int nlines = T2 * NB, LP = nlines | 1;
    extern __shared__ double2 smem2[];
    double2* z = smem2;
    double2* tw = z + (size_t)n * LP;
    const int tid = threadIdx.x, nth = blockDim.x;
    const int chunk = blockIdx.x % a.nchunks;
    const long long slab0 = (long long)(blockIdx.x / a.nchunks) * NB;
    const long long nslab = (long long)a.ncols * n;
    const int k10 = chunk * T2;
    const int kw = min(T2, nh - k10);
    for (int i = tid; i < n / 2; i += nth) tw[i] = a.g.tw[i];
    const int items = NB * n * T2;
    for (int w = tid; w < items; w += nth) {
        const int ko = w % T2, rest = w / T2;
        const int k2 = rest % n, sb = rest / n;
        const long long slab = slab0 + sb;
        if (ko < kw && slab < nslab) {
            const long long c = slab / n, k3 = slab % n;
            z[(size_t)k2 * LP + sb * T2 + ko] = a.data[c * a.g.NC + (k3 * n + k2) * nh + k10 + ko];
        } else {
            z[(size_t)k2 * LP + sb * T2 + ko] = make_double2(0.0, 0.0);
        }
    }
    __syncthreads();
    fft_lines<INV>(z, LP, nlines, a.g.log2n, tw, 1);
    for (int w = tid; w < items; w += nth) {
        const int ko = w % T2, rest = w / T2;
        const int k2 = rest % n, sb = rest / n;
        const long long slab = slab0 + sb;
        if (ko < kw && slab < nslab) {
            const long long c = slab / n, k3 = slab % n;
            a.data[c * a.g.NC + (k3 * n + k2) * nh + k10 + ko] = z[(size_t)k2 * LP + sb * T2 + ko];
        }
    }
}

template <bool INV>
inline cudaError_t launch_d2(const D2Args& a, cudaStream_t st) {
    auto kern = k_d2<INV>;
    const size_t sm = d2_smem_bytes(a.g.n, a.T2, a.NB);
    static size_t configured = 0;
    if (sm > configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        if (e != cudaSuccess) return e;
        configured = sm;
    }
    const long long nslab = (long long)a.ncols * a.g.n;
    const unsigned grid = (unsigned)(a.nchunks * ((nslab + a.NB - 1) / a.NB));
    kern<<<grid, DLR_THREADS, sm, st>>>(a);
    return cudaGetLastError();
}
