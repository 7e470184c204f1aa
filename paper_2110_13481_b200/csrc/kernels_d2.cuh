// Dimension-2 pass: in-place complex FFT (forward: natural -> bit-reversed positions; inverse: the transpose)
// along k2 of the half spectrum Ah[c][k3'][k2][k1].  Columns are independent here, so a CTA takes NB (column, k3)
// slabs and a chunk of T2 consecutive k1 (contiguous in memory).
// Index arithmetic: n is a power of two (shifts); T2 is not (n/2+1 is odd) -> FastDiv; slab decoding is hoisted
// out of the element loops.
#pragma once
#include "common.cuh"

struct D2Args {
    GridDev g;
    double2* data;       // ncols columns, stride NC
    int ncols;
    int T2, NB, nchunks; // k1 chunk width, slabs per CTA, ceil(nh / T2)
    int threads;         // CTA size
};

__host__ inline size_t d2_smem_bytes(int n, int T2, int NB) {
    const int LP = (T2 * NB) | 1;
    return (size_t)n * LP * 16 + (size_t)(n / 2) * 16 + 16;
}

template <bool INV>
__global__ void __launch_bounds__(DLR_THREADS, 3) k_d2(const D2Args a) {
    pdl_wait();
    pdl_trigger();
    const int n = a.g.n, nh = a.g.nh, lg = a.g.log2n, T2 = a.T2, NB = a.NB;
    const int nlines = T2 * NB, LP = nlines | 1;
    extern __shared__ double2 smem2[];
    double2* z = smem2;
    double2* tw = z + (size_t)n * LP;
    const int tid = threadIdx.x, nth = blockDim.x;
    const FastDiv fch = make_fastdiv((unsigned)a.nchunks), fT2 = make_fastdiv((unsigned)T2);
    const int cb = (int)fdiv(blockIdx.x, fch);
    const int chunk = (int)blockIdx.x - cb * a.nchunks;
    const int slab0 = cb * NB;
    const int nslab = a.ncols << lg;
    const int k10 = chunk * T2;
    const int kw = min(T2, nh - k10);
    for (int i = tid; i < n / 2; i += nth) tw[i] = a.g.tw[i];
    const int per = n * T2;                                    // elements of one slab chunk (k2, ko)
    for (int sb = 0; sb < NB; sb++) {
        const int slab = slab0 + sb;
        const bool live = slab < nslab;
        const int c = slab >> lg, k3 = slab & (n - 1);
        const double2* src = a.data + (size_t)c * a.g.NC + ((size_t)k3 << lg) * nh + k10;
        double2* dst = z + sb * T2;
        for (int w = tid; w < per; w += nth) {
            const int k2 = (int)fdiv((unsigned)w, fT2);
            const int ko = w - k2 * T2;
            dst[(size_t)k2 * LP + ko] = (live && ko < kw) ? src[(size_t)k2 * nh + ko] : make_double2(0.0, 0.0);
        }
    }
    __syncthreads();
    fft_lines<INV>(z, LP, nlines, lg, tw, 1);
    for (int sb = 0; sb < NB; sb++) {
        const int slab = slab0 + sb;
        if (slab >= nslab) break;
        const int c = slab >> lg, k3 = slab & (n - 1);
        double2* out = a.data + (size_t)c * a.g.NC + ((size_t)k3 << lg) * nh + k10;
        const double2* srcz = z + sb * T2;
        for (int w = tid; w < per; w += nth) {
            const int k2 = (int)fdiv((unsigned)w, fT2);
            const int ko = w - k2 * T2;
            if (ko < kw) out[(size_t)k2 * nh + ko] = srcz[(size_t)k2 * LP + ko];
        }
    }
}

template <bool INV>
inline cudaError_t launch_d2(const D2Args& a, cudaStream_t st) {
    auto kern = k_d2<INV>;
    const size_t sm = d2_smem_bytes(a.g.n, a.T2, a.NB);
    const long long nslab = (long long)a.ncols * a.g.n;
    const unsigned grid = (unsigned)(a.nchunks * ((nslab + a.NB - 1) / a.NB));
    return dlr_launch(kern, grid, a.threads > 0 ? a.threads : DLR_THREADS, sm, st, a);
}
