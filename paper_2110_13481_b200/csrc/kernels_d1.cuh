// Row-tile pass: a tile of grid rows (lines along i1) of ALL columns sits in shared memory in real space.  Used for
//   * the A*R^-1 passes of CholeskyQR (real in -> A*Mat -> Gram of the result on the fp64 tensor cores -> real out),
//   * the Gram check of dlr_set_initial,
//   * the first and last pass of the single-column 3D FFT of the Poisson solve: rho = A p followed by the real-to-complex
//     transform along dim 1 into the half spectrum, and the complex-to-real inverse of the three field components.
// A real row of n doubles is handled as n/2 complex numbers z[j] = a[2j] + i a[2j+1] (half-length complex FFT
// + split/merge step), so the real data never needs a repacking pass.
// (The K/L flows and the coefficient sums use the directional passes of kernels_dir.cuh.)
#pragma once
#include "common.cuh"
#include "gram_mma.cuh"
#include "chol_warp.cuh"

enum { D1_IN_REAL = 0, D1_IN_CPLX = 1 };
enum { D1_OP_NONE = 0, D1_OP_MATVEC = 1 };
enum { D1_GRAM_NONE = 0, D1_GRAM_PLAIN = 1 };
enum { D1_OUT_NONE = 0, D1_OUT_REAL = 1, D1_OUT_CPLX = 2, D1_OUT_BOTH = 3 };

struct D1Args {
    GridDev g;
    const double* in_real;     // RIN columns, stride N
    const double2* in_cplx;    // RIN columns, stride NC
    double* out_real;          // ROUT columns
    double2* out_cplx;         // ROUT columns
    const double* mat;         // MATVEC: [RIN][ROUT]
    double* partial;           // [gridDim.x][nvals] Gram partial sums
    double* partial2;          // [groups][nvals] group sums (see group_prereduce), or nullptr
    double* partialF;          // [nvals] their sum (the row a consumer reads), or nullptr
    unsigned* grp_cnt;         // group counters
    CholArgs ch;               // MATVEC with ch.gsum != nullptr: the matrix is the CholeskyQR stage of chol_warp.cuh, done by
                               //   warp 0 of every CTA.  Stage 1 that turns out to be the last one writes out_alt (the
                               //   basis) without a Gram; a stage-2 launch returns at once when ch.qrflag[0] != 0
    double* out_alt;
    double scale;              // applied to the data after a complex input (2/N for an inverse transform)
    int T;                     // rows per CTA (power of two dividing n^2)
    int threads;               // CTA size (0 = DLR_THREADS)
    // charge-density vector of eqs. (12)/(13) (ROUT = 1, MATVEC): if rho_vec != nullptr the CTA forms
    // mat[i] = rho_scale * sum_j rho_S[i + RIN j] rho_vec[j * rho_stride]   (rho_S column-major r x r), or
    // mat[i] = rho_scale * rho_vec[i * rho_stride] when rho_S == nullptr, instead of reading `mat`.
    const double* rho_S;
    const double* rho_vec;
    int rho_stride;
    double rho_scale;
};

__host__ __device__ inline int d1_gram_nvals(int R, int kind) {
    const int P = R * (R + 1) / 2;
    return kind == D1_GRAM_PLAIN ? P : 0;
}

// double2 elements of the tile region: at least the scratch of the cross-warp MMA reduction (64 doubles per warp)
__host__ __device__ inline int d1_zelems(int M, int LP) {
    const int need = (DLR_THREADS / 32) * 64 / 2;
    return M * LP > need ? M * LP : need;
}

__host__ inline size_t d1_smem_bytes(int n, int RMAX, int T, bool needE, int nmat) {
    const int M = n / 2;
    const int LP = (RMAX * T) | 1;
    size_t b = (size_t)d1_zelems(M, LP) * 16 + (size_t)M * 16 + (size_t)nmat * 8;
    (void)needE;
    return b + 16;
}

template <int RIN, int ROUT, int IN_MODE, int OP, int GRAM, int OUT_MODE>
__global__ void __launch_bounds__(DLR_THREADS, ((RIN > ROUT ? RIN : ROUT) <= 16 ? 2 : 1)) k_d1(const D1Args a) {
    pdl_wait();
    pdl_trigger();
    constexpr int RMAX = RIN > ROUT ? RIN : ROUT;
    constexpr int NMAT = OP == D1_OP_MATVEC ? RIN * ROUT : 0;
    const int n = a.g.n, M = n >> 1, lg = a.g.log2n, logM = lg - 1, T = a.T;
    const int lt = __ffs(T) - 1;                              // log2(T)
    const int nlines = RMAX * T, LP = nlines | 1;
    const long long q0 = (long long)blockIdx.x * T;          // first row (q = i2 + n*i3)
    extern __shared__ double2 smem2[];
    double2* z = smem2;                                       // [M][LP]
    double2* tw = z + d1_zelems(M, LP);                       // [M]  exp(-2 pi i k/n), k < n/2
    double* mat = (double*)(tw + M);                          // [NMAT]
    const int tid = threadIdx.x, nth = blockDim.x;
    double* out_real = a.out_real;
    bool want_gram = true;
    constexpr bool CHOL = (OP == D1_OP_MATVEC && RIN == ROUT && RIN > 3);
    __shared__ int s_chol_last;
    bool chol = false;
    if constexpr (CHOL) {
        chol = a.ch.gsum != nullptr;
        if (chol && a.ch.stage == 2 && a.ch.qrflag[0] != 0) return;       // third stage not needed
    }

    for (int i = tid; i < M; i += nth) tw[i] = a.g.tw[i];
    if (chol) {
        if constexpr (CHOL) {
            if (tid < 32) {
                const bool last = chol_warp<RIN>(a.ch, mat, blockIdx.x == 0);
                if (tid == 0) s_chol_last = last ? 1 : 0;
            }
        }
    } else if (OP == D1_OP_MATVEC && ROUT == 1 && a.rho_vec != nullptr) {
        for (int i = tid; i < RIN; i += nth) {
            double sacc = 0.0;
            if (a.rho_S != nullptr)
                for (int j = 0; j < RIN; j++) sacc = fma(a.rho_S[i + RIN * j], a.rho_vec[(size_t)j * a.rho_stride], sacc);
            else
                sacc = a.rho_vec[(size_t)i * a.rho_stride];
            mat[i] = a.rho_scale * sacc;
        }
    } else {
        for (int i = tid; i < NMAT; i += nth) mat[i] = a.mat[i];
    }
    if (IN_MODE == D1_IN_CPLX) __syncthreads();               // tw needed by the merge step below

    // ------------------------------------------------------------------ load
    if (IN_MODE == D1_IN_REAL) {
        const int cnt = T * M;
        // warp 0 is busy with the factorisation: the other warps load the tile meanwhile
        const int ltid = chol ? tid - 32 : tid, lnth = chol ? nth - 32 : nth;
        if (ltid >= 0) {
            for (int c = 0; c < RIN; c++) {
                const double2* src = (const double2*)(a.in_real + (size_t)c * a.g.N) + q0 * M;
                for (int i = ltid; i < cnt; i += lnth) {
                    const int t = i >> logM, j = i & (M - 1);
                    z[(size_t)j * LP + c * T + t] = src[i];
                }
            }
        }
        __syncthreads();
        if (chol && a.ch.stage == 1 && s_chol_last) { out_real = a.out_alt; want_gram = false; }   // last stage: no Gram
    } else {
        // half-spectrum row Ah[0..M] -> Z[k] = Ze[k] + i Zo[k] at bit-reversed positions, then inverse FFT
        const int nk = (M >> 1) + 1, nh = a.g.nh;
        const FastDiv fnk = make_fastdiv((unsigned)nk);
        const int items = RIN * T * nk;
        for (int w = tid; w < items; w += nth) {
            const int line = (int)fdiv((unsigned)w, fnk), k = w - line * nk;
            const int c = line >> lt, t = line & (T - 1);
            const double2* row = a.in_cplx + (size_t)c * a.g.NC + (q0 + t) * nh;
            const double2 A = row[k], Bc = cconj(row[M - k]);
            const double2 ze = make_double2(0.5 * (A.x + Bc.x), 0.5 * (A.y + Bc.y));
            const double2 df = make_double2(0.5 * (A.x - Bc.x), 0.5 * (A.y - Bc.y));
            const double2 zo = cmulc(df, tw[k]);                        // 1/2 conj(w^k) (A[k] - conj A[M-k])
            z[(size_t)brev(k, logM) * LP + line] = make_double2(ze.x - zo.y, ze.y + zo.x);        // Ze + i Zo
            if (k != 0 && k != M - k)
                z[(size_t)brev(M - k, logM) * LP + line] = make_double2(ze.x + zo.y, -ze.y + zo.x);  // conj(Ze) + i conj(Zo)
        }
        __syncthreads();
        fft_lines<true>(z, LP, RIN * T, logM, tw, 2);
    }

    // ------------------------------------------------------------------ point-wise operation across columns
    if (OP != D1_OP_NONE || IN_MODE == D1_IN_CPLX) {
        const int items = M * T;
        for (int w = tid; w < items; w += nth) {
            const int t = w & (T - 1), j = w >> lt;
            double2* p = z + (size_t)j * LP + t;
            double2 x[RIN];
#pragma unroll
            for (int c = 0; c < RIN; c++) {
                x[c] = p[c * T];
                if (IN_MODE == D1_IN_CPLX) { x[c].x *= a.scale; x[c].y *= a.scale; }
            }
            if (OP == D1_OP_NONE) {
#pragma unroll
                for (int c = 0; c < RIN; c++) p[c * T] = x[c];
            } else if (OP == D1_OP_MATVEC) {
#pragma unroll
                for (int co = 0; co < ROUT; co++) {
                    double2 acc = make_double2(0.0, 0.0);
#pragma unroll
                    for (int ci = 0; ci < RIN; ci++) {
                        const double m = mat[ci * ROUT + co];
                        acc.x = fma(m, x[ci].x, acc.x);
                        acc.y = fma(m, x[ci].y, acc.y);
                    }
                    p[co * T] = acc;
                }
            }
        }
        __syncthreads();
    }

    // ------------------------------------------------------------------ Gram accumulation (ROUT columns)
    constexpr int NTPg = GramShape<ROUT>::NTP;
    double gacc[1][NTPg][2];
    double gcs[GramShape<ROUT>::NB][2];
    if (GRAM == D1_GRAM_PLAIN && want_gram) {
        // plain Gram matrix of the output on the fp64 tensor cores (gram_mma.cuh); reduced across warps after the store
#pragma unroll
        for (int t = 0; t < NTPg; t++) gacc[0][t][0] = gacc[0][t][1] = 0.0;
        gram_mma_accum<ROUT, 1, false>(z, LP, T, lt, M * T, [](int, int, double2&, double2&, double2&) {}, gacc, gcs);
    }

    // ------------------------------------------------------------------ store
    // (the group sums of the Gram rows are formed after the store so that the fence covers only small data)
    if (OUT_MODE & D1_OUT_REAL) {
        const int cnt = T * M;
        for (int c = 0; c < ROUT; c++) {
            double2* dst = (double2*)(out_real + (size_t)c * a.g.N) + q0 * M;
            for (int i = tid; i < cnt; i += nth) {
                const int t = i >> logM, j = i & (M - 1);
                dst[i] = z[(size_t)j * LP + c * T + t];
            }
        }
    }
    if (OUT_MODE & D1_OUT_CPLX) {
        __syncthreads();
        fft_lines<false>(z, LP, ROUT * T, logM, tw, 2);
        const int nk = (M >> 1) + 1, nh = a.g.nh;
        const FastDiv fnk = make_fastdiv((unsigned)nk);
        const int items = ROUT * T * nk;
        for (int w = tid; w < items; w += nth) {
            const int line = (int)fdiv((unsigned)w, fnk), k = w - line * nk;
            const int c = line >> lt, t = line & (T - 1);
            double2* row = a.out_cplx + (size_t)c * a.g.NC + (q0 + t) * nh;
            const double2 Zk = z[(size_t)brev(k, logM) * LP + line];
            const double2 Zm = cconj(z[(size_t)brev((M - k) & (M - 1), logM) * LP + line]);
            const double2 ze = make_double2(0.5 * (Zk.x + Zm.x), 0.5 * (Zk.y + Zm.y));
            const double2 zo = make_double2(0.5 * (Zk.y - Zm.y), -0.5 * (Zk.x - Zm.x));      // -(i/2)(Zk - conj Z[M-k])
            const double2 wz = cmul(zo, tw[k]);
            row[k] = cadd(ze, wz);
            if (k != M - k) row[M - k] = cconj(csub(ze, wz));
        }
    }
    if (GRAM == D1_GRAM_PLAIN && want_gram) {
        constexpr int P = ROUT * (ROUT + 1) / 2;
        __syncthreads();                                        // the store has read the tile: it becomes scratch
        double* part = a.partial + (size_t)blockIdx.x * P;
        mma_tiles_reduce<NTPg>(&gacc[0][0][0], (double*)z, 2 * d1_zelems(M, LP), [&](int ai, int pos, double v) {
            constexpr int NB = GramShape<ROUT>::NB;
            int I = 0, tp = ai;
            while (tp >= NB - I) { tp -= NB - I; I++; }
            const int ca = 8 * I + (pos >> 3), cb = 8 * (I + tp) + (pos & 7);
            if (ca <= cb && cb < ROUT) part[upper_pair_index(ROUT, ca, cb)] = v;
        });
    }
    if (GRAM != D1_GRAM_NONE && want_gram && a.partial2 != nullptr)
        group_prereduce(a.partial, d1_gram_nvals(ROUT, GRAM), a.grp_cnt, a.partial2, a.partialF);
}

template <int RIN, int ROUT, int IN_MODE, int OP, int GRAM, int OUT_MODE>
inline cudaError_t launch_d1(const D1Args& a, cudaStream_t st) {
    constexpr int RMAX = RIN > ROUT ? RIN : ROUT;
    constexpr int NMAT = OP == D1_OP_MATVEC ? RIN * ROUT : 0;
    auto kern = k_d1<RIN, ROUT, IN_MODE, OP, GRAM, OUT_MODE>;
    const size_t sm = d1_smem_bytes(a.g.n, RMAX, a.T, false, (NMAT + 1) & ~1);
    const unsigned grid = (unsigned)(((long long)a.g.n * a.g.n) / a.T);
    return dlr_launch(kern, grid, a.threads > 0 ? a.threads : DLR_THREADS, sm, st, a);
}
