// Line transforms for the warp-autonomous pass kernels (pass_*.cuh).
//
// A UNIT is the smallest piece of a factor on which a directional sub-flow of section 4 of the paper
// is closed: complete grid lines along one direction, for all columns the operation couples.  One thread GROUP (a warp,
// or a few warps with their own named barrier) owns a unit from load to store and synchronises only with itself, so the
// groups of an SM drift apart and the loads of one overlap the butterflies and stores of the others - no CTA-wide
// barrier, no tail of half-filled waves.
//
// Shared-memory layout of a unit (double2 = one complex element = two real grid points, reading R4 keeps them separate):
//     z[c * CP + (e + (e >> PS)) * L + l]        c column, e element along the line, l < L packed line of the column
// - l fastest: the point-wise phases across columns (mixing, real-space term; thread <-> point (e, l)) and the butterfly
//   phases (thread <-> (l, j)) both touch runs of consecutive 16-byte words;
// - one pad element per 2^PS elements, PS = log2 of the radix of the LAST forward group: the stride between the blocks of
//   that group (elements 2^PS apart) then falls on different banks, every other group reads runs of >= 8 words.
// Forward = decimation in frequency, natural order in -> bit-reversed order out; inverse = its transpose, unnormalised:
// the same convention as fft_reg.cuh, all tables by stored position.  External twiddles come from a small
// shared-memory table ordered [q][j] (consecutive lanes = consecutive j: conflict-free), built once per CTA.
#pragma once
#include "common.cuh"
#include "fft_reg.cuh"

struct Grp {                      // thread group of one unit
    int tid, nth, bar;            // rank in the group, size (multiple of 32), named barrier id (1..15; unused for a warp)
    __device__ __forceinline__ void sync() const {
        if (nth == 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(nth) : "memory");
    }
};

struct WPlan {                    // radix groups of a 2^logM-point transform
    int g[3], ng, ps;             // log2 radices (forward order), count, pad shift
    int st[3], logst[3], logB[3]; // per group: stride between its registers, log2 of it, log2 of its block size
    int toff[3];                  // offset of the group's twiddle table (double2 units); groups with st = 1 have none
    int tlen;                     // total table length
};

__host__ __device__ constexpr WPlan wf_plan(int logM) {
    WPlan p{};
    p.g[0] = p.g[1] = p.g[2] = 0;
    switch (logM) {
        case 1: p.g[0] = 1; p.ng = 1; break;
        case 2: p.g[0] = 2; p.ng = 1; break;
        case 3: p.g[0] = 3; p.ng = 1; break;
        case 4: p.g[0] = 2; p.g[1] = 2; p.ng = 2; break;
        case 5: p.g[0] = 3; p.g[1] = 2; p.ng = 2; break;
        case 6: p.g[0] = 3; p.g[1] = 3; p.ng = 2; break;
        case 7: p.g[0] = 2; p.g[1] = 3; p.g[2] = 2; p.ng = 3; break;     // block stride of the middle group = 32
        default: p.g[0] = 3; p.g[1] = 3; p.g[2] = 2; p.ng = 3; break;
    }
    p.ps = p.g[p.ng - 1];
    int lev = 0, off = 0;
    for (int i = 0; i < 3; i++) {
        p.st[i] = p.logst[i] = p.logB[i] = p.toff[i] = 0;
        if (i >= p.ng) continue;
        p.logB[i] = logM - lev;
        p.logst[i] = logM - lev - p.g[i];
        p.st[i] = 1 << p.logst[i];
        p.toff[i] = off;
        if (p.logst[i] > 0) off += ((1 << p.g[i]) - 1) << p.logst[i];
        lev += p.g[i];
    }
    p.tlen = off;
    return p;
}

__host__ __device__ constexpr int wf_padded(int n, int ps) { return n + (n >> ps); }

// twiddle tables of all groups: T_i[(q - 1) * st + j] = exp(-2 pi i j brev(q) / B_i), built once by the host
// (wf_host_tables) and copied from global memory by the whole CTA (coalesced: one latency); the caller synchronises
template <int LG>
__device__ __forceinline__ void wf_load_tables(double2* tab, const double2* __restrict__ gtab) {
    constexpr WPlan p = wf_plan(LG);
    for (int w = threadIdx.x; w < p.tlen; w += blockDim.x) tab[w] = gtab[w];
}

// host: the tables of wf_plan(logM) into out[0 .. tlen)
inline void wf_host_tables(int logM, double2* out) {
    const WPlan p = wf_plan(logM);
    const long double PI = 3.14159265358979323846264338327950288L;
    for (int i = 0; i < p.ng; i++) {
        if (p.logst[i] == 0) continue;
        const int G = p.g[i], cnt = ((1 << G) - 1) << p.logst[i];
        for (int w = 0; w < cnt; w++) {
            const int q = (w >> p.logst[i]) + 1, j = w & (p.st[i] - 1);
            int br = 0;
            for (int b = 0; b < G; b++) br |= ((q >> b) & 1) << (G - 1 - b);
            const long double ang = -2.0L * PI * (long double)(j * br) / (long double)(1 << p.logB[i]);
            out[p.toff[i] + w] = make_double2((double)cosl(ang), (double)sinl(ang));
        }
    }
}

struct ZL {
    int L, lL, CP, ps;
    __device__ __forceinline__ int at(int c, int e, int l) const { return c * CP + ((e + (e >> ps)) << lL) + l; }
    __device__ __forceinline__ int row(int e) const { return (e + (e >> ps)) << lL; }
};

// One radix group on shared memory, all lines of the unit (ncol columns x L lines).  Items: l fastest, then the
// butterfly index within the line, then the column.
template <int G, bool INV>
__device__ __forceinline__ void wf_group(double2* z, const ZL& zl, int ncol, int logM, int logst, int logB,
                                         const double2* __restrict__ tw, const Grp& gp) {
    constexpr int R = 1 << G;
    const int st = 1 << logst, lipl = logM - G;          // items per line = 2^lipl
    const int items = (ncol << lipl) << zl.lL;
    for (int w = gp.tid; w < items; w += gp.nth) {
        const int l = w & (zl.L - 1), t = (w >> zl.lL) & ((1 << lipl) - 1), c = w >> (zl.lL + lipl);
        const int j = t & (st - 1), b = t >> logst;
        const int e0 = (b << logB) + j;
        double2* base = z + c * zl.CP + l;
        double2 a[R];
#pragma unroll
        for (int q = 0; q < R; q++) a[q] = base[zl.row(e0 + (q << logst))];
        if (!INV) {
            bfly<G, false>(a);
            if (logst > 0) {
#pragma unroll
                for (int q = 1; q < R; q++) a[q] = cmul(a[q], tw[((q - 1) << logst) + j]);
            }
        } else {
            if (logst > 0) {
#pragma unroll
                for (int q = 1; q < R; q++) a[q] = cmulc(a[q], tw[((q - 1) << logst) + j]);
            }
            bfly<G, true>(a);
        }
#pragma unroll
        for (int q = 0; q < R; q++) base[zl.row(e0 + (q << logst))] = a[q];
    }
}

// first forward group fed by ld(c, e, l) (global memory or a staging buffer) instead of the unit
template <int G, class LD>
__device__ __forceinline__ void wf_first(double2* z, const ZL& zl, int ncol, int logM, const double2* __restrict__ tw,
                                         const Grp& gp, LD ld) {
    constexpr int R = 1 << G;
    const int logst = logM - G, st = 1 << logst;
    const int items = (ncol << logst) << zl.lL;
    for (int w = gp.tid; w < items; w += gp.nth) {
        const int l = w & (zl.L - 1), j = (w >> zl.lL) & (st - 1), c = w >> (zl.lL + logst);
        double2 a[R];
#pragma unroll
        for (int q = 0; q < R; q++) a[q] = ld(c, j + (q << logst), l);
        bfly<G, false>(a);
        if (logst > 0) {
#pragma unroll
            for (int q = 1; q < R; q++) a[q] = cmul(a[q], tw[((q - 1) << logst) + j]);
        }
        double2* base = z + c * zl.CP + l;
#pragma unroll
        for (int q = 0; q < R; q++) base[zl.row(j + (q << logst))] = a[q];
    }
}

// last inverse group (the transpose of the first forward one) handing its results to st_(c, e, l, value)
template <int G, class ST>
__device__ __forceinline__ void wf_last(const double2* z, const ZL& zl, int ncol, int logM,
                                        const double2* __restrict__ tw, const Grp& gp, ST st_) {
    constexpr int R = 1 << G;
    const int logst = logM - G, st = 1 << logst;
    const int items = (ncol << logst) << zl.lL;
    for (int w = gp.tid; w < items; w += gp.nth) {
        const int l = w & (zl.L - 1), j = (w >> zl.lL) & (st - 1), c = w >> (zl.lL + logst);
        const double2* base = z + c * zl.CP + l;
        double2 a[R];
#pragma unroll
        for (int q = 0; q < R; q++) a[q] = base[zl.row(j + (q << logst))];
        if (logst > 0) {
#pragma unroll
            for (int q = 1; q < R; q++) a[q] = cmulc(a[q], tw[((q - 1) << logst) + j]);
        }
        bfly<G, true>(a);
#pragma unroll
        for (int q = 0; q < R; q++) st_(c, j + (q << logst), l, a[q]);
    }
}

// last forward group + point-wise f(value, stored position e, column c) + first inverse group, in registers
template <int G, class F>
__device__ __forceinline__ void wf_mid(double2* z, const ZL& zl, int ncol, int logM, const Grp& gp, F f) {
    constexpr int R = 1 << G;
    const int lipl = logM - G;
    const int items = (ncol << lipl) << zl.lL;
    for (int w = gp.tid; w < items; w += gp.nth) {
        const int l = w & (zl.L - 1), b = (w >> zl.lL) & ((1 << lipl) - 1), c = w >> (zl.lL + lipl);
        double2* base = z + c * zl.CP + l;
        double2 a[R];
#pragma unroll
        for (int q = 0; q < R; q++) a[q] = base[zl.row((b << G) + q)];
        bfly<G, false>(a);
#pragma unroll
        for (int q = 0; q < R; q++) f(a[q], (b << G) + q, c);
        bfly<G, true>(a);
#pragma unroll
        for (int q = 0; q < R; q++) base[zl.row((b << G) + q)] = a[q];
    }
}

// the forward group strictly between the first and the last (only three-group plans have one), then a group sync;
// and its inverse.  LG = log2 of the transform length: the plan is a compile-time constant.
template <int LG, bool INV>
__device__ __forceinline__ void wf_middle(double2* z, const ZL& zl, int ncol, const double2* tab, const Grp& gp) {
    constexpr WPlan p = wf_plan(LG);
    if constexpr (p.ng == 3) {
        wf_group<p.g[1], INV>(z, zl, ncol, LG, p.logst[1], p.logB[1], tab + p.toff[1], gp);
        gp.sync();
    }
}
