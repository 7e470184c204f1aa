// Shared-memory FFT over many lines, register butterflies (used by the directional passes).
// Same data layout and ordering as fft_lines in common.cuh (s[elem * LP + line], forward = decimation in frequency,
// natural order in -> bit-reversed order out; inverse = its transpose, unnormalised), but
//   * a group of G <= 3 levels is one true radix-2^G butterfly: the internal twiddles are the hard-coded 8th roots of
//     unity, only the 2^G - 1 external twiddles w_B^(j f) are looked up,
//   * the external twiddles come from CONSTANT memory (twiddles.cuh), not from shared memory: the shared-memory data
//     pipe is what bounds these kernels (ncu: l1tex 72-87 % of peak, profiles/), and a 128-bit twiddle load costs as
//     much of it as a data load,
//   * fft_mid runs the last forward group, a point-wise operation on the spectrum and the first inverse group in
//     registers: the spectrum never makes a round trip through shared memory.
#pragma once
#include "common.cuh"
#include "twiddles.cuh"

// v * w_8^k (forward) or v * conj(w_8^k) (inverse), k = 0..3 known at compile time after unrolling
__device__ __forceinline__ double2 mul_w8(double2 v, int k, bool inv) {
    const double h = 0.70710678118654752440;
    if (k == 0) return v;
    if (k == 1) return inv ? make_double2((v.x - v.y) * h, (v.x + v.y) * h) : make_double2((v.x + v.y) * h, (v.y - v.x) * h);
    if (k == 2) return inv ? make_double2(-v.y, v.x) : make_double2(v.y, -v.x);
    return inv ? make_double2(-(v.x + v.y) * h, (v.x - v.y) * h) : make_double2((v.y - v.x) * h, -(v.x + v.y) * h);
}

// DFT of size 2^G in registers: forward natural -> bit-reversed positions, inverse bit-reversed -> natural
template <int G, bool INV>
__device__ __forceinline__ void bfly(double2 (&a)[1 << G]) {
    constexpr int R = 1 << G;
    if (!INV) {
#pragma unroll
        for (int lv = 0; lv < G; lv++) {
            const int hq = R >> (lv + 1);
#pragma unroll
            for (int q = 0; q < R; q++) {
                if ((q & hq) == 0) {
                    const int k8 = ((q & (hq - 1)) << lv) * (8 / R);
                    const double2 u = a[q], v = a[q + hq];
                    a[q] = cadd(u, v);
                    a[q + hq] = mul_w8(csub(u, v), k8 & 3, false);
                }
            }
        }
    } else {
#pragma unroll
        for (int lv = G - 1; lv >= 0; lv--) {
            const int hq = R >> (lv + 1);
#pragma unroll
            for (int q = 0; q < R; q++) {
                if ((q & hq) == 0) {
                    const int k8 = ((q & (hq - 1)) << lv) * (8 / R);
                    const double2 u = a[q], t = mul_w8(a[q + hq], k8 & 3, true);
                    a[q] = cadd(u, t);
                    a[q + hq] = csub(u, t);
                }
            }
        }
    }
}

__host__ __device__ constexpr int brev_small(int q, int G) {
    int r = 0;
    for (int i = 0; i < G; i++) r |= ((q >> i) & 1) << (G - 1 - i);
    return r;
}

// exp(-2 pi i ex / B) with B = 2^logB, 0 <= ex < B
__device__ __forceinline__ double2 tw_const(int ex, int logB) {
    int idx = ex << (8 - logB);                 // DLR_TWN = 256
    const bool neg = idx >= DLR_TWN / 2;
    if (neg) idx -= DLR_TWN / 2;
    const double2 w = c_tw[idx];
    return neg ? make_double2(-w.x, -w.y) : w;
}

// one group of G levels starting at level lev0 of a 2^logM-point transform, over nl.d lines
// Not inlined: a directional pass calls the radix groups from up to ten places and a thread runs each call for two or
// three items, so inlined copies are fetched from the instruction cache for a single use each (third sub-flow at 64^3,
// r = 10: 10.4 K -> 6.1 K instructions, 81 -> 76 us per launch).
#ifdef DLR_FFT_INLINE
#define DLR_FFT_INL __forceinline__
#else
#define DLR_FFT_INL __noinline__
#endif
template <int G, bool INV>
__device__ DLR_FFT_INL void fft_group_c(double2* s, int LP, FastDiv nl, int logM, int lev0) {
    constexpr int R = 1 << G;
    const int nlines = (int)nl.d;
    const int logst = logM - lev0 - G, st = 1 << logst, logB = logM - lev0;
    const int items = (1 << (logM - G)) * nlines;
    for (int w = threadIdx.x; w < items; w += blockDim.x) {
        const int it = (int)fdiv((unsigned)w, nl);
        const int line = w - it * nlines;
        const int j = it & (st - 1), b = it >> logst;
        double2* p = s + (size_t)((b << logB) + j) * LP + line;
        const size_t es = (size_t)st * LP;
        double2 a[R];
#pragma unroll
        for (int q = 0; q < R; q++) a[q] = p[q * es];
        if (!INV) {
            bfly<G, false>(a);
            if (logst > 0) {
#pragma unroll
                for (int q = 1; q < R; q++) a[q] = cmul(a[q], tw_const(j * brev_small(q, G), logB));
            }
        } else {
            if (logst > 0) {
#pragma unroll
                for (int q = 1; q < R; q++) a[q] = cmulc(a[q], tw_const(j * brev_small(q, G), logB));
            }
            bfly<G, true>(a);
        }
#pragma unroll
        for (int q = 0; q < R; q++) p[q * es] = a[q];
    }
}

// last forward group + point-wise operation f(value, stored position e, line) + first inverse group, in registers
template <int G, class F>
__device__ __forceinline__ void fft_mid_group(double2* s, int LP, FastDiv nl, int logM, F f) {
    constexpr int R = 1 << G;
    const int nlines = (int)nl.d;
    const int items = (1 << (logM - G)) * nlines;
    for (int w = threadIdx.x; w < items; w += blockDim.x) {
        const int b = (int)fdiv((unsigned)w, nl);
        const int line = w - b * nlines;
        double2* p = s + (size_t)(b << G) * LP + line;
        double2 a[R];
#pragma unroll
        for (int q = 0; q < R; q++) a[q] = p[(size_t)q * LP];
        bfly<G, false>(a);
#pragma unroll
        for (int q = 0; q < R; q++) f(a[q], (b << G) + q, line);
        bfly<G, true>(a);
#pragma unroll
        for (int q = 0; q < R; q++) p[(size_t)q * LP] = a[q];
    }
}

// all groups of the forward (or inverse) transform; skip_last omits the LAST forward group / the FIRST inverse group
// (they are done by fft_mid).  Every group ends with a __syncthreads().
template <bool INV>
__device__ __forceinline__ void fft_lines_c(double2* s, int LP, int nlines, int logM, bool skip_last,
                                            bool skip_first = false) {
    int g[3], ng;
    fft_plan(logM, g, ng);
    const FastDiv nl = make_fastdiv((unsigned)nlines);
    int lev[3];
    lev[0] = 0;
    lev[1] = g[0];
    lev[2] = g[0] + g[1];
    for (int ii = 0; ii < ng; ii++) {
        const int i = INV ? ng - 1 - ii : ii;
        if (skip_last && i == ng - 1) continue;
        if (skip_first && i == 0) continue;
        switch (g[i]) {
            case 1: fft_group_c<1, INV>(s, LP, nl, logM, lev[i]); break;
            case 2: fft_group_c<2, INV>(s, LP, nl, logM, lev[i]); break;
            default: fft_group_c<3, INV>(s, LP, nl, logM, lev[i]); break;
        }
        __syncthreads();
    }
}

template <class F>
__device__ __forceinline__ void fft_mid(double2* s, int LP, int nlines, int logM, F f) {
    int g[3], ng;
    fft_plan(logM, g, ng);
    const FastDiv nl = make_fastdiv((unsigned)nlines);
    switch (g[ng - 1]) {
        case 1: fft_mid_group<1>(s, LP, nl, logM, f); break;
        case 2: fft_mid_group<2>(s, LP, nl, logM, f); break;
        default: fft_mid_group<3>(s, LP, nl, logM, f); break;
    }
    __syncthreads();
}

// Two-buffer variant of fft_mid for the exponential Runge-Kutta passes: lines `line` of buffer A (s) and of buffer B
// (s + boff) are processed together.  FA / FB: run the last forward group on A / B first (otherwise the data already
// is in that state);  f(a, b, stored position e, line) combines the two spectra element by element;  IA / IB: run
// the first inverse group on A / B afterwards;  SA / SB: store A / B back.
template <int G, bool FA, bool FB, bool IA, bool IB, bool SA, bool SB, class F>
__device__ __forceinline__ void fft_mid2_group(double2* s, int boff, int LP, FastDiv nl, int logM, F f) {
    constexpr int R = 1 << G;
    const int nlines = (int)nl.d;
    const int items = (1 << (logM - G)) * nlines;
    for (int w = threadIdx.x; w < items; w += blockDim.x) {
        const int b = (int)fdiv((unsigned)w, nl);
        const int line = w - b * nlines;
        double2* p = s + (size_t)(b << G) * LP + line;
        double2 a[R], bb[R];
#pragma unroll
        for (int q = 0; q < R; q++) { a[q] = p[(size_t)q * LP]; bb[q] = p[(size_t)q * LP + boff]; }
        if (FA) bfly<G, false>(a);
        if (FB) bfly<G, false>(bb);
#pragma unroll
        for (int q = 0; q < R; q++) f(a[q], bb[q], (b << G) + q, line);
        if (IA) bfly<G, true>(a);
        if (IB) bfly<G, true>(bb);
#pragma unroll
        for (int q = 0; q < R; q++) {
            if (SA) p[(size_t)q * LP] = a[q];
            if (SB) p[(size_t)q * LP + boff] = bb[q];
        }
    }
}

template <bool FA, bool FB, bool IA, bool IB, bool SA, bool SB, class F>
__device__ __forceinline__ void fft_mid2(double2* s, int boff, int LP, int nlines, int logM, F f) {
    int g[3], ng;
    fft_plan(logM, g, ng);
    const FastDiv nl = make_fastdiv((unsigned)nlines);
    switch (g[ng - 1]) {
        case 1: fft_mid2_group<1, FA, FB, IA, IB, SA, SB>(s, boff, LP, nl, logM, f); break;
        case 2: fft_mid2_group<2, FA, FB, IA, IB, SA, SB>(s, boff, LP, nl, logM, f); break;
        default: fft_mid2_group<3, FA, FB, IA, IB, SA, SB>(s, boff, LP, nl, logM, f); break;
    }
    __syncthreads();
}

// First forward group fed from GLOBAL memory and last inverse group writing to GLOBAL memory (passes whose tile needs no
// point-wise work across columns before / after the transform: the direction-2 sub-flow, the Parseval-only coefficient
// passes): the tile makes two round trips through shared memory instead of four.  IDX(e, l) = global double2 index
// (within one column) of tile element (e, l); column stride N2; line = c * L + l.  Only for transforms of >= 2 groups.
template <int G, class IDX>
__device__ __forceinline__ void fft_first_from_global(const double2* __restrict__ in2, size_t N2, IDX idx, double2* s,
                                                      int LP, FastDiv nl, int logM, int L, int lL) {
    constexpr int R = 1 << G;
    const int nlines = (int)nl.d;
    const int logst = logM - G, st = 1 << logst;
    const int items = st * nlines;
    for (int w = threadIdx.x; w < items; w += blockDim.x) {
        const int j = (int)fdiv((unsigned)w, nl);
        const int line = w - j * nlines;
        const int c = line >> lL, l = line & (L - 1);
        const double2* src = in2 + (size_t)c * N2;
        double2 a[R];
#pragma unroll
        for (int q = 0; q < R; q++) a[q] = src[idx(j + q * st, l)];
        bfly<G, false>(a);
#pragma unroll
        for (int q = 1; q < R; q++) a[q] = cmul(a[q], tw_const(j * brev_small(q, G), logM));
        double2* p = s + (size_t)j * LP + line;
#pragma unroll
        for (int q = 0; q < R; q++) p[(size_t)q * st * LP] = a[q];
    }
}

template <int G, class IDX>
__device__ __forceinline__ void fft_last_to_global(const double2* s, int LP, FastDiv nl, int logM, int L, int lL,
                                                   double2* __restrict__ out2, size_t N2, IDX idx) {
    constexpr int R = 1 << G;
    const int nlines = (int)nl.d;
    const int logst = logM - G, st = 1 << logst;
    const int items = st * nlines;
    for (int w = threadIdx.x; w < items; w += blockDim.x) {
        const int j = (int)fdiv((unsigned)w, nl);
        const int line = w - j * nlines;
        const int c = line >> lL, l = line & (L - 1);
        const double2* p = s + (size_t)j * LP + line;
        double2 a[R];
#pragma unroll
        for (int q = 0; q < R; q++) a[q] = p[(size_t)q * st * LP];
#pragma unroll
        for (int q = 1; q < R; q++) a[q] = cmulc(a[q], tw_const(j * brev_small(q, G), logM));
        bfly<G, true>(a);
        double2* dst = out2 + (size_t)c * N2;
#pragma unroll
        for (int q = 0; q < R; q++) dst[idx(j + q * st, l)] = a[q];
    }
}

// the groups between the first and the last one (only transforms of three groups have one); ends with a barrier
template <bool INV>
__device__ __forceinline__ void fft_middle_groups_c(double2* s, int LP, int nlines, int logM) {
    int g[3], ng;
    fft_plan(logM, g, ng);
    if (ng < 3) return;
    const FastDiv nl = make_fastdiv((unsigned)nlines);
    if (g[1] == 2) fft_group_c<2, INV>(s, LP, nl, logM, g[0]);
    else fft_group_c<3, INV>(s, LP, nl, logM, g[0]);
    __syncthreads();
}
