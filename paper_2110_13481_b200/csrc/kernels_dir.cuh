// Directional passes.  Every sub-flow of the K/L step involves the wavenumber of ONE direction only (eqs. (14)-(19),
// PAPER.md:246-270 use the partial transforms F_{x_i}), so no 3D transform is ever formed: a pass loads a tile that
// holds complete lines along its direction for ALL columns, transforms along that direction in shared memory, applies
// the sub-flow, transforms back and stores REAL data - one read and one write of the factor per sub-flow.
//
//   DOP_EXACT : [A <- A*Min] -> FFT_d -> * exp(s i t k~_d lambda_j) -> IFFT_d -> [A <- A*Mout]      eqs. (14),(15),(17),(18)
//   DOP_ETD1/2: third sub-flow in the eigenbasis of direction 3, exponential Euler / ETD2RK (eq. (19), reading R8);
//               both stages, including the real-space term N(A) (eqs. (9),(11),(16)), happen inside the tile
//   DOP_COEFF : read only: weighted Gram in real space (C1/D1, rho_tilde) and, after FFT_d, the 1D Parseval sums of
//               the derivative coefficients  M2_d[a][b] = h^3 A_a^T d_d A_b = (h^3/n) sum k~ (Im a Re b - Re a Im b)
//
// Real lines are transformed two at a time as one complex line z = u + i v: all multipliers used here are conjugate
// symmetric in k (k~ = 0 at Nyquist, reading R4), so Re and Im stay separate lines without any split step.
//   direction 1: u, v = two consecutive grid rows of the same column (tile = 2L consecutive rows)
//   direction 2, 3: a double2 of the array (grid points i1 = 2j, 2j+1) already is such a pair (tile = L double2 along i1
//                   x all points of the line x all columns)
// Shared layout z[e][line], line = c*L + l fastest (conflict-free butterflies, warp-uniform twiddles); after the
// forward (decimation-in-frequency) transform element e holds the wavenumber of bit-reversed position e, and all
// tables are stored in that order.
#pragma once
#include "common.cuh"
#include "fft_reg.cuh"
#include "gram_mma.cuh"

enum { DOP_EXACT = 0, DOP_ETD1 = 1, DOP_ETD2 = 2, DOP_COEFF = 3 };
enum { DW_NONE = 0, DW_E = 1, DW_V = 2 };

struct DirArgs {
    GridDev g;
    const double* in;      // N x R real, column stride N
    double* out;           // N x R real (may alias in)
    const double* E;       // [3][N] electric field (DW_E)
    const double* min_;    // [R][R] ([cin][cout]) applied at load, or nullptr
    const double* mout;    // [R][R] applied before the store, or nullptr
    const double* Q;       // 3 x [R][R]: real-space term in the eigenbasis, G = sum_i w_i o (m Q_i)
    const double2* ph;     // [n][R] EXACT: phases by stored position
    const double2 *ez, *f1, *f2a, *f2b;   // [n][R] ETD: e^z, t phi1, t (phi1 - phi2), t phi2
    double* gram;          // per-CTA partial sums: plain Gram of the OUTPUT (EXACT/ETD), weighted Gram of the INPUT (COEFF)
    double* pgram;         // COEFF: per-CTA Parseval partial sums [grid][R(R-1)/2]
    double* colsum;        // per-CTA column sums of the output [grid][R], or nullptr
    double *gram2, *pgram2, *colsum2;   // group sums of the three (see group_prereduce)
    double *gramF, *pgramF, *colsumF;   // and their totals: the single row a consumer reads
    unsigned* grp_cnt;     // group counters: [0..) gram, [DLR_CNT_STRIDE..) pgram, [2 DLR_CNT_STRIDE..) colsum
    int L;                 // packed lines per column in a tile (power of two)
    int store;             // write `out`
    int threads;           // CTA size (0 = DLR_THREADS)
};

template <int DOP, int DW>
__host__ __device__ inline bool dir_ereg(int n, int L, int threads) {
    return (DOP == DOP_ETD1 || DOP == DOP_ETD2) && DW == DW_E && n * L <= threads;
}

__host__ __device__ inline int dir_tiles(int n, int L) { return (n * n / 2) / L; }     // same count for all directions

// double2 elements of the tile region: at least the scratch of the cross-warp MMA reduction (64 doubles per warp)
__host__ __device__ inline int dir_zelems(int n, int LP) {
    const int need = (DLR_THREADS / 32) * 64 / 2;
    return n * LP > need ? n * LP : need;
}

// r x r matrices in shared memory: row stride padded to an even number of doubles so that the coefficients of two
// neighbouring output columns come with ONE 128-bit load (one LDS per four FMAs instead of one per two)
__host__ __device__ constexpr int mat_rs(int R) { return (R + 1) & ~1; }
__host__ __device__ constexpr int mat_ms(int R) { return R * mat_rs(R); }

// row stride of the tile (double2 units): the point-wise phases (thread <-> (e, l), l fastest) read rows e, e+1, ... of
// L consecutive double2 each within a quarter warp, the FFT phases consecutive lines of one row: a stride = L (mod 8)
// puts the 8 / L rows of a quarter warp on different banks (any odd stride for L = 1, any stride for L >= 8)
__host__ __device__ inline int dir_lpz(int lines, int L) {
    if (L >= 8) return lines | 1;
    return lines + (((L - lines) % 8) + 8) % 8;
}

__host__ inline size_t dir_smem_bytes(int n, int R, int L, int nbuf, int nmat, bool needE) {
    const int LP = dir_lpz(nbuf * R * L, L);
    size_t b = (size_t)dir_zelems(n, LP) * 16 + (size_t)nmat * mat_ms(R) * 8;
    if (needE) b += (size_t)3 * n * L * 16;
    return b + 16;
}

// tile position
struct DirGeom {
    int n, lg, M, L, lL;
    int q0;          // DIR 1: first row
    int ia;          // DIR 2: i3 of the tile;  DIR 3: i2 of the tile
    int j0;          // DIR 2, 3: first double2 along i1
    double lo, h;
};

// global double2 index (within one column) of tile element (e, l); DIR 1 returns the index of row u (row v is + M)
template <int DIR>
__device__ __forceinline__ size_t dir_index(const DirGeom& gm, int e, int l) {
    if (DIR == 1) return (size_t)(gm.q0 + 2 * l) * gm.M + e;                      // e = double2 index j along the row
    if (DIR == 2) return ((size_t)((gm.ia << gm.lg) + e)) * gm.M + gm.j0 + l;     // (i3*n + i2)*M + j
    return ((size_t)((e << gm.lg) + gm.ia)) * gm.M + gm.j0 + l;                   // (i3*n + i2)*M + j
}

// weights of the three real-space terms at the two grid points packed in element (e, l): .x for Re, .y for Im
template <int DIR, int DW>
__device__ __forceinline__ void dir_weights(const DirGeom& gm, const double2* Et, int e, int l, double2& w0,
                                            double2& w1, double2& w2) {
    if (DW == DW_E) {
        const int nL = gm.n * gm.L;
        const double2* p = Et + e * gm.L + l;
        w0 = p[0]; w1 = p[nL]; w2 = p[2 * nL];
    } else {
        if (DIR == 1) {
            const int q = gm.q0 + 2 * l, i2 = q & (gm.n - 1), i3 = q >> gm.lg;
            const double x1 = gm.lo + gm.h * e;
            w0 = make_double2(x1, x1);
            w1 = make_double2(gm.lo + gm.h * i2, gm.lo + gm.h * (i2 + 1));
            const double x3 = gm.lo + gm.h * i3;
            w2 = make_double2(x3, x3);
        } else {
            const int i1 = 2 * (gm.j0 + l);
            w0 = make_double2(gm.lo + gm.h * i1, gm.lo + gm.h * (i1 + 1));
            const double xe = gm.lo + gm.h * e, xa = gm.lo + gm.h * gm.ia;
            if (DIR == 2) { w1 = make_double2(xe, xe); w2 = make_double2(xa, xa); }
            else { w1 = make_double2(xa, xa); w2 = make_double2(xe, xe); }
        }
    }
}

// The loop over output-column pairs of the streamed r x r products stays ROLLED: a thread runs these bodies once or twice
// per tile, so unrolled code is fetched once per use (ncu: 17 % of the stall samples of the third sub-flow were
// instruction-fetch stalls with 4100 instructions of straight-line code); x[] is indexed by the unrolled inner loop only.
#ifdef DLR_CO_UNROLLED
#define DLR_CO_LOOP _Pragma("unroll")
#else
#define DLR_CO_LOOP _Pragma("unroll 1")
#endif

// copy a dense [R][R] matrix into the padded layout (pads zeroed); all threads of the CTA
template <int R>
__device__ __forceinline__ void mat_stage(double* dst, const double* __restrict__ src) {
    constexpr int RS = mat_rs(R);
    for (int i = threadIdx.x; i < R * RS; i += blockDim.x) {
        const int ci = i / RS, co = i - ci * RS;
        dst[i] = co < R ? src[ci * R + co] : 0.0;
    }
}

template <int R>
__device__ __forceinline__ void dir_matvec(double2 (&x)[R], const double* A) {     // x <- x * A, A[cin][cout] (padded)
    constexpr int RS = mat_rs(R);
    double2 y[R];
#pragma unroll
    for (int co = 0; co < R; co += 2) {
        double2 a0 = make_double2(0.0, 0.0), a1 = a0;
#pragma unroll
        for (int ci = 0; ci < R; ci++) {
            const double2 m = *(const double2*)(A + ci * RS + co);
            a0.x = fma(m.x, x[ci].x, a0.x); a0.y = fma(m.x, x[ci].y, a0.y);
            a1.x = fma(m.y, x[ci].x, a1.x); a1.y = fma(m.y, x[ci].y, a1.y);
        }
        y[co] = a0;
        if (co + 1 < R) y[co + 1] = a1;
    }
#pragma unroll
    for (int c = 0; c < R; c++) x[c] = y[c];
}

// out[co * stride] = (x A)[co], streamed out two components at a time (x is fully in registers, so out may alias the
// place x was loaded from): no second r-vector in registers
template <int R>
__device__ __forceinline__ void dir_matvec_store(const double2 (&x)[R], const double* A, double2* out, int stride) {
    constexpr int RS = mat_rs(R);
DLR_CO_LOOP
    for (int co = 0; co < R; co += 2) {
        double2 a0 = make_double2(0.0, 0.0), a1 = a0;
#pragma unroll
        for (int ci = 0; ci < R; ci++) {
            const double2 m = *(const double2*)(A + ci * RS + co);
            a0.x = fma(m.x, x[ci].x, a0.x); a0.y = fma(m.x, x[ci].y, a0.y);
            a1.x = fma(m.y, x[ci].x, a1.x); a1.y = fma(m.y, x[ci].y, a1.y);
        }
        out[co * stride] = a0;
        if (co + 1 < R) out[(co + 1) * stride] = a1;
    }
}

// real-space term in the eigenbasis: g = sum_i w_i o (m Q_i), component co written to gout[co * stride]
// (streamed out two components at a time: only m stays in registers); Q = three padded matrices
template <int R>
__device__ __forceinline__ void dir_nonlin(const double2 (&m)[R], double2* gout, int stride, const double* Q, double2 w0,
                                           double2 w1, double2 w2) {
    constexpr int RS = mat_rs(R), MS = mat_ms(R);
DLR_CO_LOOP
    for (int co = 0; co < R; co += 2) {
        double2 s0 = make_double2(0.0, 0.0), s1 = s0, s2 = s0, t0 = s0, t1 = s0, t2 = s0;
#pragma unroll
        for (int ci = 0; ci < R; ci++) {
            const double2 q0 = *(const double2*)(Q + ci * RS + co), q1 = *(const double2*)(Q + MS + ci * RS + co),
                          q2 = *(const double2*)(Q + 2 * MS + ci * RS + co);
            s0.x = fma(q0.x, m[ci].x, s0.x); s0.y = fma(q0.x, m[ci].y, s0.y);
            s1.x = fma(q1.x, m[ci].x, s1.x); s1.y = fma(q1.x, m[ci].y, s1.y);
            s2.x = fma(q2.x, m[ci].x, s2.x); s2.y = fma(q2.x, m[ci].y, s2.y);
            t0.x = fma(q0.y, m[ci].x, t0.x); t0.y = fma(q0.y, m[ci].y, t0.y);
            t1.x = fma(q1.y, m[ci].x, t1.x); t1.y = fma(q1.y, m[ci].y, t1.y);
            t2.x = fma(q2.y, m[ci].x, t2.x); t2.y = fma(q2.y, m[ci].y, t2.y);
        }
        gout[co * stride] = make_double2(fma(w0.x, s0.x, fma(w1.x, s1.x, w2.x * s2.x)),
                                         fma(w0.y, s0.y, fma(w1.y, s1.y, w2.y * s2.y)));
        if (co + 1 < R)
            gout[(co + 1) * stride] = make_double2(fma(w0.x, t0.x, fma(w1.x, t1.x, w2.x * t2.x)),
                                                   fma(w0.y, t0.y, fma(w1.y, t1.y, w2.y * t2.y)));
    }
}

// Real-space phase of the exponential Runge-Kutta stages:
//   x = scale * src [* Min, written back to src];  dst = N'(x) = sum_i w_i o (x Q_i)          (src, dst: column 0 of (e, l))
// (measured at 64^3, r = 10: inlined 72.3 us per ETD2RK launch, as one shared non-inlined copy 75.1: the call passes
// its arguments through the stack)
template <int R, int DIR, int DW>
__device__ __forceinline__ void etd_realspace(double2* z, int LPZ, int pitems, int src_off, int dst_off, double scale,
                                           const double* min_, const double* Q, const DirGeom gm, const double2* Et,
                                           const bool wreg_on, const double2 (&wreg)[3]) {
    const int L = gm.L, lL = gm.lL;
    for (int w = threadIdx.x; w < pitems; w += blockDim.x) {
        const int l = w & (L - 1), e = w >> lL;
        double2* p = z + (size_t)e * LPZ + l;
        double2 x[R];
#pragma unroll
        for (int c = 0; c < R; c++) { x[c] = p[src_off + c * L]; x[c].x *= scale; x[c].y *= scale; }
        if (min_ != nullptr) {
            dir_matvec_store<R>(x, min_, p + src_off, L);
#pragma unroll
            for (int c = 0; c < R; c++) x[c] = p[src_off + c * L];       // this thread's own stores
        }
        double2 w0 = wreg[0], w1 = wreg[1], w2 = wreg[2];                // the thread's own point (field weights in registers)
        if (!wreg_on) dir_weights<DIR, DW>(gm, Et, e, l, w0, w1, w2);
        dir_nonlin<R>(x, p + dst_off, L, Q, w0, w1, w2);                 // x is fully in registers: dst may be src
    }
    __syncthreads();
}

// emit functions for mma_tiles_reduce: accumulator index a and tile position pos -> entry of the partial row
template <int R>
__device__ __forceinline__ void tp_decode(int tp, int& I, int& J) {
    constexpr int NB = GramShape<R>::NB;
    I = 0;
    while (tp >= NB - I) { tp -= NB - I; I++; }
    J = I + tp;
}

template <int R, int DIR, int DOP, int DW>
__global__ void __launch_bounds__(((DOP == DOP_EXACT && DIR == 2) || ((DOP == DOP_ETD1 || DOP == DOP_ETD2) && R > 10)) ? 2 * DLR_THREADS : DLR_THREADS,
                                  ((DOP == DOP_EXACT && DIR == 2) ? (R <= 10 ? 2 : 1)
                                   : (DOP == DOP_COEFF && DW == DW_NONE) ? (R <= 10 ? 3 : (R <= 16 ? 2 : 1))
                                   : (DOP == DOP_COEFF || DOP == DOP_EXACT) ? (R <= 16 ? 2 : 1)
                                   : (R <= 10 ? 2 : 1)))
k_dir(const DirArgs a) {
    constexpr bool ETD = (DOP == DOP_ETD1 || DOP == DOP_ETD2);
    constexpr bool MIX = ETD || (DOP == DOP_EXACT && DIR == 1);   // column mixing exists only in these passes: the
                                                                  // direction-2 sub-flow keeps a small register budget
    constexpr int NBUF = ETD ? 2 : 1;
    constexpr int NMAT = ETD ? 5 : 2;
    constexpr int MS = mat_ms(R);
    const int n = a.g.n, lg = a.g.log2n, M = n >> 1, L = a.L;
    const int lL = __ffs(L) - 1;
    const int nl = R * L, LPZ = dir_lpz(NBUF * nl, L);
    extern __shared__ double2 smem2[];
    double2* z = smem2;                                        // [n][LPZ]
    double* mats = (double*)(z + dir_zelems(n, LPZ));          // [NMAT] padded matrices: Min, Mout, Q0, Q1, Q2
    double2* Et = (double2*)(mats + NMAT * MS);                // [3][n][L]
    const int tid = threadIdx.x, nth = blockDim.x;
    DirGeom gm;
    gm.n = n; gm.lg = lg; gm.M = M; gm.L = L; gm.lL = lL; gm.lo = a.g.lo; gm.h = a.g.h;
    gm.q0 = 0; gm.ia = 0; gm.j0 = 0;
    if (DIR == 1) {
        gm.q0 = (int)blockIdx.x * 2 * L;
    } else {
        const int ltp = (lg - 1) - lL;                         // log2 of tiles per plane (M / L)
        gm.ia = (int)blockIdx.x >> ltp;
        gm.j0 = ((int)blockIdx.x & ((1 << ltp) - 1)) << lL;
    }
    pdl_wait();
    const size_t N2 = (size_t)(a.g.N >> 1);
    const double invn = 1.0 / (double)n;
    // Field weights of the third sub-flow: with at most one tile point per thread they stay in registers for both
    // evaluations of the real-space term and the tile needs no field rows in shared memory (64^3, r = 10: 103 -> 91 KB per
    // CTA, which leaves the two resident CTAs an L1 large enough for the e^z / phi tables they read in Fourier space)
    const bool ereg = dir_ereg<DOP, DW>(n, L, (int)nth);
    double2 wreg[3] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0), make_double2(0.0, 0.0)};

    // Passes without point-wise work across the columns before the transform (direction-2 sub-flow, Parseval-only
    // coefficient passes) feed the first FFT group straight from global memory (and the sub-flow writes its last inverse
    // group straight back): two round trips through shared memory instead of four.  Needs a transform of >= 2 groups.
    constexpr bool GLOBAL_FFT = (DOP == DOP_EXACT && DIR == 2) || (DOP == DOP_COEFF && DW == DW_NONE && DIR != 1);
    const bool gfft = GLOBAL_FFT && lg >= 4;
    const auto gidx = [&](int e, int l) { return dir_index<DIR>(gm, e, l); };
    const FastDiv fnl = make_fastdiv((unsigned)nl);
    if (gfft) {
        if (lg == 4) fft_first_from_global<2>((const double2*)a.in, N2, gidx, z, LPZ, fnl, lg, L, lL);
        else fft_first_from_global<3>((const double2*)a.in, N2, gidx, z, LPZ, fnl, lg, L, lL);
    }
    // ------------------------------------------------------------------ load
    if (!gfft) {
        const double2* in2 = (const double2*)a.in;
        if (DIR == 1) {
            const int lM = lg - 1, items = nl << lM;
            for (int w = tid; w < items; w += nth) {
                const int j = w & (M - 1), line = w >> lM;
                const int c = line >> lL, l = line & (L - 1);
                const double2* p = in2 + (size_t)c * N2 + dir_index<1>(gm, j, l);
                const double2 ra = p[0], rb = p[M];
                z[(size_t)(2 * j) * LPZ + line] = make_double2(ra.x, rb.x);
                z[(size_t)(2 * j + 1) * LPZ + line] = make_double2(ra.y, rb.y);
            }
        } else {
            const int items = nl << lg;
            for (int w = tid; w < items; w += nth) {
                const int l = w & (L - 1), e = (w >> lL) & (n - 1), c = w >> (lL + lg);
                cp_async16(z + (size_t)e * LPZ + c * L + l, in2 + (size_t)c * N2 + dir_index<DIR>(gm, e, l));
            }
        }
        if (DW == DW_E && ereg) {
            if (tid < (n << lL)) {
                const int l = tid & (L - 1), e = tid >> lL;
#pragma unroll
                for (int d = 0; d < 3; d++) wreg[d] = ((const double2*)(a.E + (size_t)d * a.g.N))[dir_index<DIR>(gm, e, l)];
            }
        } else if (DW == DW_E) {
            for (int d = 0; d < 3; d++) {
                const double2* e2 = (const double2*)(a.E + (size_t)d * a.g.N);
                double2* Ed = Et + (size_t)d * n * L;
                if (DIR == 1) {
                    const int lM = lg - 1, items = L << lM;
                    for (int w = tid; w < items; w += nth) {
                        const int j = w & (M - 1), l = w >> lM;
                        const double2* p = e2 + dir_index<1>(gm, j, l);
                        const double2 ra = p[0], rb = p[M];
                        Ed[(2 * j) * L + l] = make_double2(ra.x, rb.x);
                        Ed[(2 * j + 1) * L + l] = make_double2(ra.y, rb.y);
                    }
                } else {
                    const int items = L << lg;
                    for (int w = tid; w < items; w += nth) {
                        const int l = w & (L - 1), e = w >> lL;
                        cp_async16(Ed + e * L + l, e2 + dir_index<DIR>(gm, e, l));
                    }
                }
            }
        }
    }
    // the mixing matrices are staged while the asynchronous copies of the tile (directions 2, 3) are in flight
    if (MIX && a.min_ != nullptr) mat_stage<R>(mats, a.min_);
    if (MIX && a.mout != nullptr) mat_stage<R>(mats + MS, a.mout);
    if (ETD) { mat_stage<R>(mats + 2 * MS, a.Q); mat_stage<R>(mats + 3 * MS, a.Q + R * R); mat_stage<R>(mats + 4 * MS, a.Q + 2 * R * R); }
    cp_async_wait_all();
    __syncthreads();
    pdl_trigger();                                            // one tile per CTA: every CTA of the grid has started by now
    const int pitems = n << lL;                               // tile points (e, l)

    if (DOP == DOP_COEFF) {
        // -------------------------------------------------------------- coefficients (read only), on the fp64 MMA
        constexpr int NB = GramShape<R>::NB, NTP = GramShape<R>::NTP;
        constexpr int P = R * (R + 1) / 2, P2 = R * (R - 1) / 2;
        constexpr bool WG = (DW != DW_NONE);
        constexpr int NACCW = WG ? 3 * NTP + (DW == DW_V ? NB : 0) : 1;
        struct { double acc[3][NTP][2]; double cs[NB][2]; } gw;
        if (WG && a.gram != nullptr) {
#pragma unroll
            for (int d = 0; d < 3; d++)
#pragma unroll
                for (int t = 0; t < NTP; t++) gw.acc[d][t][0] = gw.acc[d][t][1] = 0.0;
#pragma unroll
            for (int I = 0; I < NB; I++) gw.cs[I][0] = gw.cs[I][1] = 0.0;
            gram_mma_accum<R, 3, DW == DW_V>(z, LPZ, L, lL, pitems,
                [&](int e, int l, double2& w0, double2& w1, double2& w2) { dir_weights<DIR, DW>(gm, Et, e, l, w0, w1, w2); },
                gw.acc, gw.cs);
            __syncthreads();
        }
        fft_lines_c<false>(z, LPZ, nl, lg, false, gfft);       // (the first group is already done when fed from global)
        double pacc[NTP][2];
#pragma unroll
        for (int t = 0; t < NTP; t++) pacc[t][0] = pacc[t][1] = 0.0;
        parseval_mma_accum<R>(z, LPZ, L, lL, pitems, a.g.kt2p, pacc);
        __syncthreads();                                        // the tile is free: it becomes the reduction scratch
        double* scratch = (double*)z;
        const int cap = 2 * dir_zelems(n, LPZ);
        if (WG && a.gram != nullptr) {
            constexpr int NV = 3 * P + (DW == DW_V ? R : 0);
            double* part = a.gram + (size_t)blockIdx.x * NV;
            mma_tiles_reduce<NACCW>(&gw.acc[0][0][0], scratch, cap, [&](int ai, int pos, double v) {
                const int i = pos >> 3, j = pos & 7;
                if (ai < 3 * NTP) {
                    const int d = ai / NTP;
                    int I, J;
                    tp_decode<R>(ai - d * NTP, I, J);
                    const int ca = 8 * I + i, cb = 8 * J + j;
                    if (ca <= cb && cb < R) part[d * P + upper_pair_index(R, ca, cb)] = v;
                } else {
                    const int c = 8 * (ai - 3 * NTP) + i;
                    if (j == 0 && c < R) part[3 * P + c] = v;
                }
            });
        }
        {
            double* part = a.pgram + (size_t)blockIdx.x * P2;
            mma_tiles_reduce<NTP>(&pacc[0][0], scratch, cap, [&](int ai, int pos, double v) {
                const int i = pos >> 3, j = pos & 7;
                int I, J;
                tp_decode<R>(ai, I, J);
                const int ca = 8 * I + i, cb = 8 * J + j;
                if (ca < cb && cb < R) part[ca * (R - 1) - ca * (ca - 1) / 2 + (cb - ca - 1)] = v;
            });
        }
        if (WG && a.gram != nullptr) {
            constexpr int NV = 3 * P + (DW == DW_V ? R : 0);
            group_prereduce(a.gram, NV, a.grp_cnt, a.gram2, a.gramF);
        }
        group_prereduce(a.pgram, P2, a.grp_cnt + DLR_CNT_STRIDE, a.pgram2, a.pgramF);
        return;
    }

    if (DOP == DOP_EXACT) {
        // -------------------------------------------------------------- exact directional sub-flow
        if (MIX && a.min_ != nullptr) {
            for (int w = tid; w < pitems; w += nth) {
                const int l = w & (L - 1), e = w >> lL;
                double2* p = z + (size_t)e * LPZ + l;
                double2 x[R];
#pragma unroll
                for (int c = 0; c < R; c++) x[c] = p[c * L];
                dir_matvec_store<R>(x, mats, p, L);
            }
            __syncthreads();
        }
        fft_lines_c<false>(z, LPZ, nl, lg, true, gfft);
        {
            const double2* ph = a.ph;
            fft_mid(z, LPZ, nl, lg, [&](double2& v, int e, int line) {
                double2 f = __ldg(ph + (size_t)e * R + (line >> lL));
                f.x *= invn; f.y *= invn;
                v = cmul(v, f);
            });
        }
        fft_lines_c<true>(z, LPZ, nl, lg, true, gfft);
        if (gfft) {                                           // last inverse group straight to global memory: done
            if (lg == 4) fft_last_to_global<2>(z, LPZ, fnl, lg, L, lL, (double2*)a.out, N2, gidx);
            else fft_last_to_global<3>(z, LPZ, fnl, lg, L, lL, (double2*)a.out, N2, gidx);
            return;
        }
        if (MIX && a.mout != nullptr) {
            for (int w = tid; w < pitems; w += nth) {
                const int l = w & (L - 1), e = w >> lL;
                double2* p = z + (size_t)e * LPZ + l;
                double2 x[R];
#pragma unroll
                for (int c = 0; c < R; c++) x[c] = p[c * L];
                dir_matvec_store<R>(x, mats + MS, p, L);
            }
            __syncthreads();
        }
    }

    if (ETD) {
        // -------------------------------------------------------------- third sub-flow, exponential Runge-Kutta
        const double* Q = mats + 2 * MS;
        // m = A Min,  g0 = N'(m)
        etd_realspace<R, DIR, DW>(z, LPZ, pitems, 0, nl, 1.0, a.min_ != nullptr ? mats : nullptr, Q, gm, Et, ereg, wreg);
        // Fourier-space stages fused into the middle FFT group (fft_mid2): the spectra of m and g0 never make a round
        // trip through shared memory.  a = e^z M^ + t phi1 G0^  (stage-1 state);  ETD2RK keeps  e^z M^ + t (phi1 - phi2) G0^
        // in buffer A (spectral) and adds t phi2 G1^ to it after the second evaluation of the real-space term.
        fft_lines_c<false>(z, LPZ, 2 * nl, lg, true);
        if (DOP == DOP_ETD1) {
            fft_mid2<true, true, true, false, true, false>(z, nl, LPZ, nl, lg, [&](double2& av, double2& bv, int e, int line) {
                const int c = line >> lL;
                av = cadd(cmul(av, __ldg(a.ez + (size_t)e * R + c)), cmul(bv, __ldg(a.f1 + (size_t)e * R + c)));
            });
            fft_lines_c<true>(z, LPZ, nl, lg, true);
        } else {
            fft_mid2<true, true, false, true, true, true>(z, nl, LPZ, nl, lg, [&](double2& av, double2& bv, int e, int line) {
                const int c = line >> lL;
                const double2 em = cmul(av, __ldg(a.ez + (size_t)e * R + c));
                const double2 ah = cadd(em, cmul(bv, __ldg(a.f1 + (size_t)e * R + c)));
                av = cadd(em, cmul(bv, __ldg(a.f2a + (size_t)e * R + c)));
                bv = ah;                                      // inverse-transformed for N'(a)
            });
            fft_lines_c<true>(z + nl, LPZ, nl, lg, true);
            etd_realspace<R, DIR, DW>(z, LPZ, pitems, nl, nl, invn, nullptr, Q, gm, Et, ereg, wreg);      // g1 = N'(a), in place
            fft_lines_c<false>(z + nl, LPZ, nl, lg, true);
            fft_mid2<false, true, true, false, true, false>(z, nl, LPZ, nl, lg, [&](double2& av, double2& bv, int e, int line) {
                av = cadd(av, cmul(bv, __ldg(a.f2b + (size_t)e * R + (line >> lL))));
            });
            fft_lines_c<true>(z, LPZ, nl, lg, true);
        }
        for (int w = tid; w < pitems; w += nth) {             // scale of the inverse transform, back to the output basis
            const int l = w & (L - 1), e = w >> lL;
            double2* p = z + (size_t)e * LPZ + l;
            double2 x[R];
#pragma unroll
            for (int c = 0; c < R; c++) { x[c] = p[c * L]; x[c].x *= invn; x[c].y *= invn; }
            if (a.mout != nullptr) dir_matvec_store<R>(x, mats + MS, p, L);
            else {
#pragma unroll
                for (int c = 0; c < R; c++) p[c * L] = x[c];
            }
        }
        __syncthreads();
    }

    // ------------------------------------------------------------------ sums of the output, store
    constexpr int NTPo = GramShape<R>::NTP;
    double gacc[1][NTPo][2];
    double gcs[GramShape<R>::NB][2];
    if (a.gram != nullptr) {
#pragma unroll
        for (int t = 0; t < NTPo; t++) gacc[0][t][0] = gacc[0][t][1] = 0.0;
        gram_mma_accum<R, 1, false>(z, LPZ, L, lL, pitems, [](int, int, double2&, double2&, double2&) {}, gacc, gcs);
    }
    if (a.colsum != nullptr) {
        const int warp = tid >> 5, lane = tid & 31, nwarp = nth >> 5;
        for (int c = warp; c < R; c += nwarp) {
            double s = 0.0;
            for (int w = lane; w < pitems; w += 32) {
                const double2 v = z[(size_t)(w >> lL) * LPZ + c * L + (w & (L - 1))];
                s += v.x + v.y;
            }
            s = warp_sum(s);
            if (lane == 0) a.colsum[(size_t)blockIdx.x * R + c] = s;
        }
    }
    if (a.store) {
        double2* out2 = (double2*)a.out;
        if (DIR == 1) {
            const int lM = lg - 1, items = nl << lM;
            for (int w = tid; w < items; w += nth) {
                const int j = w & (M - 1), line = w >> lM;
                const int c = line >> lL, l = line & (L - 1);
                const double2 za = z[(size_t)(2 * j) * LPZ + line], zb = z[(size_t)(2 * j + 1) * LPZ + line];
                double2* p = out2 + (size_t)c * N2 + dir_index<1>(gm, j, l);
                p[0] = make_double2(za.x, zb.x);
                p[M] = make_double2(za.y, zb.y);
            }
        } else {
            const int items = nl << lg;
            for (int w = tid; w < items; w += nth) {
                const int l = w & (L - 1), e = (w >> lL) & (n - 1), c = w >> (lL + lg);
                out2[(size_t)c * N2 + dir_index<DIR>(gm, e, l)] = z[(size_t)e * LPZ + c * L + l];
            }
        }
    }
    if (a.gram != nullptr) {
        constexpr int P = R * (R + 1) / 2;
        __syncthreads();                                        // the store has read the tile: it becomes scratch
        double* part = a.gram + (size_t)blockIdx.x * P;
        mma_tiles_reduce<NTPo>(&gacc[0][0][0], (double*)z, 2 * dir_zelems(n, LPZ), [&](int ai, int pos, double v) {
            const int i = pos >> 3, j = pos & 7;
            int I, J;
            tp_decode<R>(ai, I, J);
            const int ca = 8 * I + i, cb = 8 * J + j;
            if (ca <= cb && cb < R) part[upper_pair_index(R, ca, cb)] = v;
        });
        group_prereduce(a.gram, P, a.grp_cnt, a.gram2, a.gramF);
    }
    if (a.colsum != nullptr) group_prereduce(a.colsum, R, a.grp_cnt + 2 * DLR_CNT_STRIDE, a.colsum2, a.colsumF);
}

template <int R, int DIR, int DOP, int DW>
inline cudaError_t launch_dir(const DirArgs& a, cudaStream_t st) {
    constexpr bool ETD = (DOP == DOP_ETD1 || DOP == DOP_ETD2);
    auto kern = k_dir<R, DIR, DOP, DW>;
    const int threads = a.threads > 0 ? a.threads : DLR_THREADS;
    const size_t sm = dir_smem_bytes(a.g.n, R, a.L, ETD ? 2 : 1, ETD ? 5 : 2, DW == DW_E && !dir_ereg<DOP, DW>(a.g.n, a.L, threads));
    return dlr_launch(kern, (unsigned)dir_tiles(a.g.n, a.L), threads, sm, st, a);
}
