// Shared device-side definitions of the DLR hot path (sm_100a, fp64).
// Data layouts:
//   real factor      A[c][i3][i2][i1]            column stride N = n^3, i1 fastest (the C ABI's column-major N x r)
//   half spectrum    Ah[c][k3'][k2'][k1]         column stride NC = (n/2+1) n^2 complex; k1 = 0..n/2 in natural
//                    order, k2', k3' are BIT-REVERSED positions (decimation-in-frequency forward transforms leave
//                    them there; decimation-in-time inverses consume them; all wavenumber tables are built in
//                    stored-position order, so no kernel ever reorders data).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define DLR_THREADS 256

struct GridDev {
    int n, nh, log2n;        // points per dimension, n/2+1, log2(n)
    long long N, NC;         // n^3, nh*n*n
    double lo, h, h3;        // left extreme, spacing, h^3
    const double* kt1;       // [nh]  odd-derivative wavenumber by k1 (0 at Nyquist)            (reading R4)
    const double* kt2p;      // [n]   same, by stored (bit-reversed) position in dims 2,3
    const double* ksq1;      // [nh]  true k^2 by k1
    const double* ksq2p;     // [n]   true k^2 by stored position
    const double2* tw;       // [n/2] exp(-2 pi i k / n)
    const double2* wtab;     // twiddle tables of the radix groups of wf_plan(log2n), see wfft.cuh (built by the host)
};

// Opt a kernel in to the whole dynamic shared memory of an SM of the CURRENT device.  cudaFuncSetAttribute is state
// of (function, device), not of a context: every dlr_create does this once for all kernels it may launch (idempotent,
// same value from every context and thread), so the library keeps no process-wide "already configured" flags.
template <class K>
inline cudaError_t dlr_optin_smem(K kern) {
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, kern);
    if (e != cudaSuccess) return e;
    int dev = 0, optin = 0;
    e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes);
    // (no carve-out preference: the driver sizes L1 from what a launch needs; the phase/phi tables are read through L1)
    return e;
}

// ---------------------------------------------------------------- programmatic dependent launch
// Every kernel of the step is launched with programmatic stream serialisation (dlr_launch): the next kernel of the stream
// may become resident while this one drains, so its launch latency and whatever it does before pdl_wait() (twiddle
// tables that dlr_create wrote: nothing a kernel of the step produces) overlap the tail of its predecessor.  pdl_wait()
// returns once the preceding kernel of the stream has completed and its writes are visible; EVERY kernel calls it before
// its first access to step data (also before overwriting what an earlier kernel reads), which keeps the chain transitive.
// pdl_trigger() only moves the point at which the successor may become resident; correctness never depends on it.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() {
#ifndef DLR_PDL_NO_TRIGGER
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
}

// 16-byte asynchronous copy global -> shared (LDGSTS): a thread can have all the elements of its tile share in flight at once
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory"); }

extern thread_local int g_dlr_pdl;      // set by the issuing entry point of api.cu for the duration of a call (0 = plain launches)

template <class... KA, class... A>
inline cudaError_t dlr_launch(void (*kern)(KA...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, A&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = g_dlr_pdl ? 1 : 0;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KA(args)...);
}

// ---------------------------------------------------------------- complex helpers
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) {   // a * conj(b)
    return make_double2(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -a.x * b.y));
}
__device__ __forceinline__ double2 cconj(double2 a) { return make_double2(a.x, -a.y); }

// ---------------------------------------------------------------- shared-memory FFT over many lines
// Lines live in shared memory as s[elem * LP + line] (line index fastest => consecutive threads touch
// consecutive 16-byte words: conflict-free in every stage, twiddles are warp-uniform).
// Forward = decimation in frequency, natural order in -> bit-reversed order out, kernel exp(-2 pi i jk/M).
// Inverse = the exact transpose: bit-reversed in -> natural out, conjugate twiddles, unnormalised.
// tw[] holds exp(-2 pi i k / TWN), k < TWN/2, with TWN = M * twmul.
// Exact unsigned division by a runtime constant without a hardware divide (the streaming loops index with
// non-power-of-two line counts such as n/2+1):  q = floor(w / d) = umulhi(w, ceil(2^32 / d)), exact for w*d < 2^32.
struct FastDiv { unsigned d, m; };
__host__ __device__ inline FastDiv make_fastdiv(unsigned d) {
    FastDiv f;
    f.d = d;
    f.m = d <= 1 ? 0u : (unsigned)((0x100000000ull + d - 1) / d);
    return f;
}
__device__ __forceinline__ unsigned fdiv(unsigned w, FastDiv f) { return f.d == 1 ? w : __umulhi(w, f.m); }

template <int G, bool INV>
__device__ __forceinline__ void fft_group(double2* s, int LP, FastDiv nl, int logM, int lev0, const double2* tw,
                                          int twmul) {
    constexpr int R = 1 << G;
    const int nlines = (int)nl.d;
    const int logst = logM - lev0 - G;        // log2 of the element stride between the R registers
    const int st = 1 << logst;
    const int logB = logM - lev0;             // block size at the first (coarsest) level of the group
    const int items = (1 << (logM - G)) * nlines;
    for (int w = threadIdx.x; w < items; w += blockDim.x) {
        const int it = (int)fdiv((unsigned)w, nl);
        const int line = w - it * nlines;
        const int j = it & (st - 1);
        const int b = it >> logst;
        double2* p = s + (size_t)((b << logB) + j) * LP + line;
        double2 a[R];
#pragma unroll
        for (int q = 0; q < R; q++) a[q] = p[(size_t)q * st * LP];
        if (!INV) {
#pragma unroll
            for (int lv = 0; lv < G; lv++) {
                const int hq = R >> (lv + 1);
                const int mul = twmul << (lev0 + lv);      // M/(2h) * twmul with 2h = B >> lv
#pragma unroll
                for (int q = 0; q < R; q++) {
                    if ((q & hq) == 0) {
                        const int pos = j + (q & (hq - 1)) * st;
                        double2 u = a[q], v = a[q + hq];
                        a[q] = cadd(u, v);
                        a[q + hq] = cmul(csub(u, v), tw[pos * mul]);
                    }
                }
            }
        } else {
#pragma unroll
            for (int lv = G - 1; lv >= 0; lv--) {
                const int hq = R >> (lv + 1);
                const int mul = twmul << (lev0 + lv);
#pragma unroll
                for (int q = 0; q < R; q++) {
                    if ((q & hq) == 0) {
                        const int pos = j + (q & (hq - 1)) * st;
                        double2 u = a[q];
                        double2 t = cmulc(a[q + hq], tw[pos * mul]);
                        a[q] = cadd(u, t);
                        a[q + hq] = csub(u, t);
                    }
                }
            }
        }
#pragma unroll
        for (int q = 0; q < R; q++) p[(size_t)q * st * LP] = a[q];
    }
}

// level grouping for log2(M) = 2..8 (each group = one pass over shared memory)
__device__ __forceinline__ void fft_plan(int logM, int g[3], int& ng) {
    switch (logM) {
        case 1: g[0] = 1; ng = 1; break;
        case 2: g[0] = 2; ng = 1; break;
        case 3: g[0] = 3; ng = 1; break;
        case 4: g[0] = 2; g[1] = 2; ng = 2; break;
        case 5: g[0] = 3; g[1] = 2; ng = 2; break;
        case 6: g[0] = 3; g[1] = 3; ng = 2; break;
        case 7: g[0] = 3; g[1] = 2; g[2] = 2; ng = 3; break;
        default: g[0] = 3; g[1] = 3; g[2] = 2; ng = 3; break;
    }
}

template <bool INV>
__device__ __forceinline__ void fft_lines(double2* s, int LP, int nlines, int logM, const double2* tw, int twmul) {
    int g[3], ng;
    fft_plan(logM, g, ng);
    const FastDiv nl = make_fastdiv((unsigned)nlines);
    int lev[3];
    lev[0] = 0;
    lev[1] = g[0];
    lev[2] = g[0] + g[1];
    for (int ii = 0; ii < ng; ii++) {
        const int i = INV ? ng - 1 - ii : ii;
        switch (g[i]) {
            case 1: fft_group<1, INV>(s, LP, nl, logM, lev[i], tw, twmul); break;
            case 2: fft_group<2, INV>(s, LP, nl, logM, lev[i], tw, twmul); break;
            default: fft_group<3, INV>(s, LP, nl, logM, lev[i], tw, twmul); break;
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------- three-level deterministic partial sums
// A producer CTA writes its partial row rows[blockIdx.x][0..nvals); the LAST CTA to finish of every group of DLR_GRP
// consecutive CTAs then adds the group's rows in index order into rows2[group][0..nvals), and the last GROUP to finish
// adds the group sums in index order into final_row[0..nvals) (if not nullptr).  The result does not depend on which
// CTA does it, so the sums stay bit-reproducible; a consumer reads one row.  counters[group] and the grid-level counter
// counters[DLR_CNT_STRIDE - 1] must be 0 on entry and are 0 again on exit (atomicInc wraps).
#define DLR_GRP 16
#define DLR_CNT_STRIDE 4096
__host__ __device__ inline int dlr_groups(int nblocks) { return (nblocks + DLR_GRP - 1) / DLR_GRP; }

__device__ __forceinline__ void group_prereduce(const double* rows, int nvals, unsigned* counters, double* rows2,
                                                double* final_row = nullptr) {
    __shared__ int s_last;
    __syncthreads();                                           // the partial row of this CTA is written (CTA scope) ...
    const int grp = (int)blockIdx.x / DLR_GRP, first = grp * DLR_GRP;
    const int cnt = min(DLR_GRP, (int)gridDim.x - first);
    if (threadIdx.x == 0) {
        __threadfence();                                       // ... and ordered device-wide before the counter moves: ONE
        s_last = (atomicInc(counters + grp, (unsigned)(cnt - 1)) == (unsigned)(cnt - 1));   // fence per CTA (cumulative
    }                                                          // over the barrier), not one per thread (ncu: 7-14 % of
    __syncthreads();                                           // the stall samples of the coefficient passes were membar)
    if (!s_last) return;
    __threadfence();
    for (int v = threadIdx.x; v < nvals; v += blockDim.x) {
        const double* p = rows + (size_t)first * nvals + v;
        double s = 0.0;
        for (int b = 0; b < cnt; b++) s += __ldcg(p + (size_t)b * nvals);     // L2 (other CTAs wrote these)
        rows2[(size_t)grp * nvals + v] = s;
    }
    if (final_row == nullptr) return;
    const int ngrp = dlr_groups((int)gridDim.x);
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = (atomicInc(counters + DLR_CNT_STRIDE - 1, (unsigned)(ngrp - 1)) == (unsigned)(ngrp - 1));
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int v = threadIdx.x; v < nvals; v += blockDim.x) {
        const double* p = rows2 + v;
        double s = 0.0;
        for (int g = 0; g < ngrp; g++) s += __ldcg(p + (size_t)g * nvals);
        final_row[v] = s;
    }
}

__device__ __forceinline__ int brev(int k, int logM) { return (int)(__brev((unsigned)k) >> (32 - logM)); }

// ---------------------------------------------------------------- warp-owned Gram accumulation
// Each warp owns a contiguous range of the output entries; for every entry it sweeps all points of the
// tile (lane-strided), reduces by shuffles and lane 0 writes the partial: no atomics, fixed order.
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
