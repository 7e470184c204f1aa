// A * Mat pass of CholeskyQR (the QR after every K and L step; reading R12):
//     out = A Mat,   [Gram sums of out for the next stage],
// a point-wise product across the r columns.  No transform, so the tile needs no transposition: a chunk of C consecutive
// grid points is r contiguous runs of C doubles (one per column) and moves with bulk asynchronous copies (TMA,
// cp.async.bulk + mbarrier, tma.cuh).  One persistent CTA per SM walks over its chunks with a ring of S stages:
//     producer warp:  bulk loads of chunk k + S - 1  |  all threads: wait for chunk k, out = x Mat IN PLACE (a thread owns
//     its points in every column)  |  producer warp: bulk stores of chunk k  |  all warps: Gram of chunk k on the fp64 MMA
// so loads, arithmetic and stores of different chunks overlap.
// The r x r factorisation that yields Mat is done by warp 0 in the prologue, while the first loads are in flight
// (chol_warp.cuh); Mat may also be given.
#pragma once
#include "chol_warp.cuh"
#include "gram_mma.cuh"
#include "tma.cuh"

struct ApplyArgs {
    long long N;               // points per column
    const double* in;          // N x R
    double* out;               // N x R (never aliases in)
    double* out_alt;           // destination if stage 1 turns out to be the last stage (the basis)
    const double* mat;         // [R][R] ([cin][cout]) when ch.gsum == nullptr
    CholArgs ch;               // ch.gsum != nullptr: Mat is this CholeskyQR stage; a stage-2 launch returns at once when
                               //   ch.qrflag[0] != 0; stage 1 that is the last one writes out_alt and skips the Gram
    double* partial;           // [grid][P] Gram partial rows, or nullptr
    double *partial2, *partialF;
    unsigned* grp_cnt;
    int C, S;                  // chunk length (multiple of 64, divides N), stages
};

#define DLR_APPLY_THREADS 256
__host__ __device__ constexpr int apply_cs(int C) { return C + 4; }            // column stride: spreads the MMA fragment loads
__host__ inline size_t apply_smem_bytes(int R, int C, int S) {
    return (size_t)S * R * apply_cs(C) * 8 + (size_t)R * R * 8 + 8 * 16 + 64;
}

template <int R, bool GRAM>
__global__ void __launch_bounds__(DLR_APPLY_THREADS, 1) k_apply(const ApplyArgs a) {
    extern __shared__ double2 smem2[];
    constexpr int RR = R * R, P = R * (R + 1) / 2;
    constexpr int NTP = GramShape<R>::NTP, NB = GramShape<R>::NB;
    const int C = a.C, S = a.S, CS = apply_cs(C);
    const int tid = threadIdx.x, nth = blockDim.x;
    double* stage0 = (double*)smem2;                               // [S][R][CS]
    double* mat = stage0 + (size_t)S * R * CS;                     // [RR]
    uint64_t* full = (uint64_t*)(mat + RR);                        // [S] (<= 8)
    __shared__ int s_last;
    const bool chol = a.ch.gsum != nullptr;
    if (tid == 32) {
        for (int s = 0; s < a.S; s++) mbar_init(full + s, 1);
        mbar_fence_init();
    }
    pdl_wait();
    if (chol && a.ch.stage == 2 && a.ch.qrflag[0] != 0) return;   // third stage not needed

    const long long nchunks = a.N / C;
    const int nloc = (int)((nchunks - blockIdx.x + gridDim.x - 1) / gridDim.x);     // chunks of this CTA
    const uint32_t col_bytes = (uint32_t)C * 8, stage_bytes = col_bytes * R;
    const auto chunk_of = [&](int it) { return (long long)blockIdx.x + (long long)it * gridDim.x; };
    // producer = warp 1 (warp 0 factorises): lane c issues the copies of column c, so the r bulk operations of a stage go out
    // with one instruction each instead of one after the other; every lane tracks its own bulk groups
    const int pl = tid - 32;                                        // lane in the producer warp (0 <= pl < 32 there)
    const bool is_prod = pl >= 0 && pl < 32;
    const auto issue_load = [&](int it) {                           // whole producer warp
        const int s = it % S;
        if (pl == 0) mbar_arrive_expect_tx(full + s, stage_bytes);
        __syncwarp();
        if (pl < R)
            bulk_g2s(stage0 + (size_t)s * R * CS + (size_t)pl * CS, a.in + chunk_of(it) * C + (size_t)pl * a.N, col_bytes, full + s);
    };
    __syncthreads();
    if (is_prod) {
        const int pre = nloc < S - 1 ? nloc : S - 1;
        for (int it = 0; it < pre; it++) issue_load(it);
    }
    if (chol) {
        if (tid < 32) {
            const bool last = chol_warp<R>(a.ch, mat, blockIdx.x == 0);
            if (tid == 0) s_last = last ? 1 : 0;
        }
    } else {
        for (int i = tid; i < RR; i += nth) mat[i] = a.mat[i];
    }
    __syncthreads();
    double* out = a.out;
    bool want_gram = GRAM && a.partial != nullptr;
    if (chol && a.ch.stage == 1 && s_last) { out = a.out_alt; want_gram = false; }     // this pass is the last one

    double gacc[NTP][2];
#pragma unroll
    for (int t = 0; t < NTP; t++) gacc[t][0] = gacc[t][1] = 0.0;
    const int warp = tid >> 5, lane = tid & 31, nwarp = nth >> 5;

    for (int it = 0; it < nloc; it++) {
        const int s = it % S;
        double* st = stage0 + (size_t)s * R * CS;
        mbar_wait(full + s, (uint32_t)((it / S) & 1));
        // out = x Mat in place: thread p2 owns points 2 p2, 2 p2 + 1 of every column
        for (int p2 = tid; p2 < (C >> 1); p2 += nth) {
            double2* px = (double2*)st + p2;
            double2 x[R];
#pragma unroll
            for (int c = 0; c < R; c++) x[c] = px[(size_t)c * (CS >> 1)];
#pragma unroll
            for (int co = 0; co < R; co++) {
                double2 acc = make_double2(0.0, 0.0);
#pragma unroll
                for (int ci = 0; ci < R; ci++) {
                    const double m = mat[ci * R + co];
                    acc.x = fma(m, x[ci].x, acc.x);
                    acc.y = fma(m, x[ci].y, acc.y);
                }
                px[(size_t)co * (CS >> 1)] = acc;
            }
        }
        fence_proxy_async();                                        // the bulk stores below read what was just written
        __syncthreads();                                            // also: every warp is done with the Gram of chunk it - 1
        if (is_prod) {
            if (pl < R) bulk_s2g(out + chunk_of(it) * C + (size_t)pl * a.N, st + (size_t)pl * CS, col_bytes);
            bulk_commit();
            if (it + S - 1 < nloc) {
                bulk_wait_read<1>();                                // this lane's store of chunk it - 1 has read its stage
                __syncwarp();                                       // ... and so have the other lanes'
                issue_load(it + S - 1);                             // into stage (it - 1) % S
            }
        }
        if (want_gram) {
            // Gram of the output chunk: fragment = column 8 I + (lane >> 2), point 4 g + (lane & 3)
            const int ci = lane >> 2, k = lane & 3;
            for (int g = warp; g < (C >> 2); g += nwarp) {
                const double* base = st + 4 * g + k;
                double frag[NB];
#pragma unroll
                for (int I = 0; I < NB; I++) {
                    const int col = 8 * I + ci;
                    frag[I] = col < R ? base[(size_t)col * CS] : 0.0;
                }
#pragma unroll
                for (int I = 0; I < NB; I++)
#pragma unroll
                    for (int J = I; J < NB; J++) dmma884(gacc[GramShape<R>::tp(I, J)], frag[I], frag[J]);
            }
        }
    }
    pdl_trigger();
    if (is_prod) bulk_wait_read<0>();                               // every store has read its stage
    __syncthreads();
    if (want_gram) {
        double* part = a.partial + (size_t)blockIdx.x * P;
        mma_tiles_reduce<NTP>(&gacc[0][0], stage0, S * R * CS, [&](int ai, int pos, double v) {
            const int i = pos >> 3, j = pos & 7;
            int I = 0, tp = ai;
            while (tp >= NB - I) { tp -= NB - I; I++; }
            const int ca = 8 * I + i, cb = 8 * (I + tp) + j;
            if (ca <= cb && cb < R) part[upper_pair_index(R, ca, cb)] = v;
        });
        group_prereduce(a.partial, P, a.grp_cnt, a.partial2, a.partialF);
    }
    if (is_prod) bulk_wait_all<0>();                                // the stores are complete before the CTA exits
}

template <int R, bool GRAM>
inline cudaError_t launch_apply(const ApplyArgs& a, int ctas, cudaStream_t st) {
    return dlr_launch(k_apply<R, GRAM>, (unsigned)ctas, DLR_APPLY_THREADS, apply_smem_bytes(R, a.C, a.S), st, a);
}
