// Cross-Gram matrix of two factors, G[a][b] = sum_points A_a B_b (r x r, NOT symmetric), on the fp64 tensor cores: the
// change-of-basis matrices M = <X1, X0>, N = <V1, V0> of the unconventional integrator (the paper's reference [4], named
// in PAPER.md:29, 288; oracle.step_bug).  Read-only streaming pass over both factors; fragments come straight from global
// memory (lane -> column 8 I + (lane >> 2), point 4 g + (lane & 3): 32-byte runs per column).  Every CTA writes one
// partial r x r block; k_bug_s0 adds them in index order (bit-reproducible) and forms S~ = M S0 N^T.
#pragma once
#include "gram_mma.cuh"

#define DLR_CROSS_THREADS 256

template <int R>
__global__ void __launch_bounds__(DLR_CROSS_THREADS) k_cross(const double* __restrict__ A, const double* __restrict__ B,
                                                             long long N, double* __restrict__ partial) {
    constexpr int NB = GramShape<R>::NB;
    __shared__ double scratch[(DLR_CROSS_THREADS / 32) * 64];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
    const int ci = lane >> 2, k = lane & 3;
    double acc[NB][NB][2];
#pragma unroll
    for (int I = 0; I < NB; I++)
#pragma unroll
        for (int J = 0; J < NB; J++) acc[I][J][0] = acc[I][J][1] = 0.0;
    const long long ngroups = N >> 2;                                   // 4 points per MMA (N = n^3 is a multiple of 512)
    for (long long g = (long long)blockIdx.x * nwarp + warp; g < ngroups; g += (long long)gridDim.x * nwarp) {
        const long long p = 4 * g + k;
        double fa[NB], fb[NB];
#pragma unroll
        for (int I = 0; I < NB; I++) {
            const int col = 8 * I + ci;
            fa[I] = col < R ? A[(size_t)col * N + p] : 0.0;
            fb[I] = col < R ? B[(size_t)col * N + p] : 0.0;
        }
#pragma unroll
        for (int I = 0; I < NB; I++)
#pragma unroll
            for (int J = 0; J < NB; J++) dmma884(acc[I][J], fa[I], fb[J]);
    }
    // accumulator of block (I, J): lane holds C[lane >> 2][2 (lane & 3) + {0, 1}]; cross-warp sums in fixed order
    double* part = partial + (size_t)blockIdx.x * R * R;
#pragma unroll
    for (int I = 0; I < NB; I++)
#pragma unroll
        for (int J = 0; J < NB; J++) {
            double* dst = scratch + warp * 64 + (lane >> 2) * 8 + 2 * (lane & 3);
            dst[0] = acc[I][J][0];
            dst[1] = acc[I][J][1];
            __syncthreads();
            if (tid < 64) {
                double s = 0.0;
                for (int w = 0; w < nwarp; w++) s += scratch[w * 64 + tid];
                const int a = 8 * I + (tid >> 3), b = 8 * J + (tid & 7);
                if (a < R && b < R) part[a * R + b] = s;
            }
            __syncthreads();
        }
}

// S~ = M S0 N^T with M = hx3 * sum_cta pm, N = hv3 * sum_cta pn (row-major [new][old]); S column-major, in place.
template <int R>
__global__ void __launch_bounds__(512) k_bug_s0(const double* pm, int nm, const double* pn, int nn, double hx3, double hv3,
                                               double* S) {
    constexpr int RR = R * R;
    __shared__ double M[RR], Nm[RR], S0[RR], T[RR];
    const int tid = threadIdx.x;
    if (tid < RR) {
        double s = 0.0;
        for (int b = 0; b < nm; b++) s += pm[(size_t)b * RR + tid];
        M[tid] = hx3 * s;
        s = 0.0;
        for (int b = 0; b < nn; b++) s += pn[(size_t)b * RR + tid];
        Nm[tid] = hv3 * s;
        S0[tid] = S[tid];
    }
    __syncthreads();
    if (tid < RR) {                                   // T(a, j) = sum_i M[a][i] S0(i, j), stored column-major like S
        const int a = tid % R, j = tid / R;
        double s = 0.0;
#pragma unroll
        for (int i = 0; i < R; i++) s = fma(M[a * R + i], S0[i + R * j], s);
        T[tid] = s;
    }
    __syncthreads();
    if (tid < RR) {                                   // S~(a, b) = sum_j T(a, j) N[b][j]
        const int a = tid % R, b = tid / R;
        double s = 0.0;
#pragma unroll
        for (int j = 0; j < R; j++) s = fma(T[a + R * j], Nm[b * R + j], s);
        S[tid] = s;
    }
}

template <int R>
inline cudaError_t launch_cross(const double* A, const double* B, long long N, double* partial, int ctas, cudaStream_t st) {
    k_cross<R><<<(unsigned)ctas, DLR_CROSS_THREADS, 0, st>>>(A, B, N, partial);
    return cudaGetLastError();
}
template <int R>
inline cudaError_t launch_bug_s0(const double* pm, int nm, const double* pn, int nn, double hx3, double hv3, double* S,
                                 cudaStream_t st) {
    k_bug_s0<R><<<1, 512, 0, st>>>(pm, nm, pn, nn, hx3, hv3, S);
    return cudaGetLastError();
}
