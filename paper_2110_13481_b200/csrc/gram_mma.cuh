// Gram-type sums over a shared-memory tile on the fp64 tensor cores (mma.sync m8n8k4, DMMA).
// The coefficient matrices of PAPER.md:150-166 and the Gram matrix of the QR are contractions G = Y^T diag(w) Y with
// M = N = r and K = number of grid points: the one place on the path where a contraction is dense enough for MMA.
// One warp-per-entry sweep re-reads every value ~r times through the shared-memory pipe, which is what bounds the
// pass kernels (profiles/); as an MMA every value is read once per block of 8 columns.
//
// Tile layout (both pass families): element (e, l) of column c is the double2  z[e * LPZ + c * CS + l]  holding two
// grid points (.x, .y); items w = e * CS + l, CS a power of two.  A group = 2 consecutive items = 4 points = the K
// extent of one MMA.  Fragment of column block I (columns 8I .. 8I+7):  lane -> column 8I + (lane >> 2), point
// (lane & 3); the same register serves as the A operand (row-major 8x4) and as the B operand (col-major 4x8).
// Accumulator of block pair (I <= J): lane holds C[lane >> 2][2 (lane & 3) + {0, 1}].
#pragma once
#include "common.cuh"

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1])
                 : "d"(a), "d"(b));
}

template <int R>
struct GramShape {
    static constexpr int NB = (R + 7) / 8;             // column blocks
    static constexpr int NTP = NB * (NB + 1) / 2;      // block pairs I <= J
    __host__ __device__ static constexpr int tp(int I, int J) { return I * NB - I * (I - 1) / 2 + (J - I); }
};

// Real-space Gram sums: acc[d][tp] += sum_points w_d Y_I^T Y_J  (NW = 1: plain, w = 1;  NW = 3: the three weights
// returned by wf(e, l, w0, w1, w2) as double2 (.x, .y = the two points of the item)).  COLSUM: cs[I] += Y_I^T 1.
template <int R, int NW, bool COLSUM, class WF>
__device__ __forceinline__ void gram_mma_accum(const double2* z, int LPZ, int CS, int lCS, int nitems, WF wf,
                                               double (&acc)[NW][GramShape<R>::NTP][2],
                                               double (&cs)[GramShape<R>::NB][2]) {
    constexpr int NB = GramShape<R>::NB;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    const int ci = lane >> 2, k = lane & 3, comp = k & 1;
    for (int g = warp; g < (nitems >> 1); g += nwarp) {
        const int w = 2 * g + (k >> 1);
        const int l = w & (CS - 1), e = w >> lCS;
        const double* base = (const double*)(z + (size_t)e * LPZ + l) + comp;
        double frag[NB];
#pragma unroll
        for (int I = 0; I < NB; I++) {
            const int col = 8 * I + ci;
            frag[I] = col < R ? base[(size_t)col * CS * 2] : 0.0;
        }
        double wd[3] = {1.0, 1.0, 1.0};
        if (NW == 3) {
            double2 w0, w1, w2;
            wf(e, l, w0, w1, w2);
            wd[0] = comp ? w0.y : w0.x; wd[1] = comp ? w1.y : w1.x; wd[2] = comp ? w2.y : w2.x;
        }
#pragma unroll
        for (int I = 0; I < NB; I++) {
#pragma unroll
            for (int J = I; J < NB; J++) {
#pragma unroll
                for (int d = 0; d < NW; d++)
                    dmma884(acc[d][GramShape<R>::tp(I, J)], NW == 3 ? frag[I] * wd[d] : frag[I], frag[J]);
            }
            if (COLSUM) dmma884(cs[I], frag[I], 1.0);
        }
    }
}

// Parseval sums of a derivative coefficient on a transformed tile (kt = odd-derivative wavenumber by stored position):
// acc[tp] += sum_items kt(e) (Im Z_I^T Re Z_J - Re Z_I^T Im Z_J);  K extent = 4 consecutive items.
template <int R>
__device__ __forceinline__ void parseval_mma_accum(const double2* z, int LPZ, int CS, int lCS, int nitems,
                                                   const double* __restrict__ kt, double (&acc)[GramShape<R>::NTP][2]) {
    constexpr int NB = GramShape<R>::NB;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    const int ci = lane >> 2, k = lane & 3;
    for (int g = warp; g < (nitems >> 2); g += nwarp) {
        const int w = 4 * g + k;
        const int l = w & (CS - 1), e = w >> lCS;
        const double kk = __ldg(kt + e);
        const double2* base = z + (size_t)e * LPZ + l;
        double2 frag[NB];
#pragma unroll
        for (int I = 0; I < NB; I++) {
            const int col = 8 * I + ci;
            frag[I] = col < R ? base[(size_t)col * CS] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int I = 0; I < NB; I++) {
#pragma unroll
            for (int J = I; J < NB; J++) {
                dmma884(acc[GramShape<R>::tp(I, J)], kk * frag[I].y, frag[J].x);
                dmma884(acc[GramShape<R>::tp(I, J)], -kk * frag[I].x, frag[J].y);
            }
        }
    }
}

// Cross-warp reduction of NACC accumulator tiles through shared scratch (capacity cap doubles, may be the tile itself
// once it is no longer needed; the caller has synchronised).  acc is addressed as a flat array of NACC x 2 doubles.
// emit(a, pos, value) is called once per accumulator a and tile position pos = i * 8 + j with the CTA-wide sum.
template <int NACC, class EMIT>
__device__ __forceinline__ void mma_tiles_reduce(const double* acc_flat, double* scratch, int cap, EMIT emit) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    const int per = nwarp * 64;
    int ch = cap / per;
    if (ch < 1) ch = 1;
    if (ch > NACC) ch = NACC;
    const int pos0 = (lane >> 2) * 8 + 2 * (lane & 3);
    for (int a0 = 0; a0 < NACC; a0 += ch) {
        const int na = min(ch, NACC - a0);
#pragma unroll
        for (int a = 0; a < NACC; a++) {
            if (a >= a0 && a < a0 + na) {
                double* dst = scratch + ((size_t)(a - a0) * nwarp + warp) * 64 + pos0;
                dst[0] = acc_flat[2 * a];
                dst[1] = acc_flat[2 * a + 1];
            }
        }
        __syncthreads();
        for (int idx = threadIdx.x; idx < na * 64; idx += blockDim.x) {
            const int a = idx >> 6, pos = idx & 63;
            const double* src = scratch + (size_t)a * nwarp * 64 + pos;
            double s = 0.0;
            for (int wv = 0; wv < nwarp; wv++) s += src[wv * 64];
            emit(a0 + a, pos, s);
        }
        __syncthreads();
    }
}

// index of the upper pair (ca <= cb) in the packed row of R (R + 1) / 2 entries
__host__ __device__ inline int upper_pair_index(int R, int ca, int cb) { return ca * R - ca * (ca - 1) / 2 + (cb - ca); }
