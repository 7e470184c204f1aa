// Sub-flow along direction 1 with the changes of eigenbasis before and after it (eqs. (14), (17)):
//     A  <-  F_1^-1 [ ((F_1 A) Min) o exp(s i t k~_1 lambda_j) Mout ]
// The column mixing commutes with the transform along x1, so both mixing matrices act in Fourier space, in the same
// point-wise phase as the phase factors: the first radix group reads global memory straight into registers, the last
// inverse group writes its registers straight back, and a unit makes four round trips through shared memory.
// A unit = NL packed lines (2 NL consecutive grid rows: row u is the real part, row u + 1 the imaginary part of one
// complex line, reading R4 keeps them separate) of ALL r columns, owned by one warp (or a small group with its own
// named barrier) from load to store: no CTA-wide barrier inside the loop over units (wfft.cuh).
// Optionally the Gram matrix of the OUTPUT (the first Gram of the CholeskyQR that follows the flow) is accumulated on
// the fp64 tensor cores from the spectrum (Parseval along x1: sum_x u u' + v v' = n sum_k Re(Z conj Z')).
#pragma once
#include "wfft.cuh"
#include "gram_mma.cuh"
#include "kernels_dir.cuh"

struct Sub1Args {
    GridDev g;
    const double* in;      // N x R real
    double* out;           // N x R real (may alias in)
    const double* min_;    // [R][R] ([cin][cout]) or nullptr
    const double* mout;    // [R][R] or nullptr
    const double2* ph;     // [n][R] phases by stored position
    int NL;                // packed lines per column in a unit (power of two)
    int wpu;               // warps per unit
    double* gram;          // per-CTA partial rows of the Gram matrix of the output [grid][R (R + 1) / 2], or nullptr
    double *gram2, *gramF; // group sums and total (group_prereduce)
    unsigned* grp_cnt;
};

__host__ __device__ constexpr int sub1_rp(int R) { return R | 1; }
__host__ inline size_t sub1_unit_elems(int n, int R, int NL) {
    return (size_t)wf_padded(n, wf_plan(31 - __builtin_clz(n)).ps) * NL * R;
}
__host__ inline size_t sub1_smem_bytes(int n, int R, int NL, int groups) {
    const WPlan p = wf_plan(31 - __builtin_clz(n));
    size_t units = sub1_unit_elems(n, R, NL) * groups;
    const size_t need = (size_t)groups * 8 * 64 / 2;          // scratch of the cross-warp MMA reduction (8 warps max per group set)
    if (units < need) units = need;
    return ((size_t)p.tlen + (size_t)n * sub1_rp(R) + (size_t)(2 * mat_ms(R)) / 2 + 1 + units) * 16;
}

template <int R, int LG>
__global__ void __launch_bounds__(256, (R <= 10 ? 2 : 1)) k_sub1(const Sub1Args a) {
    extern __shared__ double2 smem2[];
    constexpr int n = 1 << LG, lg = LG;
    constexpr WPlan p = wf_plan(LG);
    constexpr int MS = mat_ms(R), RP = sub1_rp(R);
    constexpr int NTP = GramShape<R>::NTP, NB = GramShape<R>::NB;
    const int NL = a.NL, lNL = __ffs(NL) - 1;
    double2* tab = smem2;                                   // twiddle tables
    double2* phs = tab + p.tlen;                            // [n][RP] phases times 1/n
    double* mats = (double*)(phs + n * RP);                 // Min, Mout
    double2* zbase = (double2*)(mats + 2 * MS) + 1;
    const int gsz = a.wpu << 5;
    const int grp = (int)threadIdx.x / gsz, ngrp = (int)blockDim.x / gsz;
    ZL zl;
    zl.L = NL; zl.lL = lNL; zl.ps = p.ps; zl.CP = wf_padded(n, p.ps) << lNL;
    double2* z = zbase + (size_t)grp * R * zl.CP;
    wf_load_tables<LG>(tab, a.g.wtab);                      // written by dlr_create: may precede pdl_wait()
    pdl_wait();
    const double invn = 1.0 / (double)n;
    for (int i = threadIdx.x; i < n * R; i += blockDim.x) {
        const int e = i / R, c = i - e * R;
        const double2 f = a.ph[i];
        phs[e * RP + c] = make_double2(f.x * invn, f.y * invn);
    }
    const bool has_min = a.min_ != nullptr, has_mout = a.mout != nullptr;
    if (has_min) mat_stage<R>(mats, a.min_);
    if (has_mout) mat_stage<R>(mats + MS, a.mout);
    __syncthreads();
    Grp gp;
    gp.tid = (int)threadIdx.x - grp * gsz; gp.nth = gsz; gp.bar = 1 + grp;
    const int nunits = (n * n / 2) >> lNL;
    const size_t N = (size_t)a.g.N;
    double gacc[NTP][2];
#pragma unroll
    for (int t = 0; t < NTP; t++) gacc[t][0] = gacc[t][1] = 0.0;
    const bool want_gram = a.gram != nullptr;

    for (int u = blockIdx.x * ngrp + grp; u < nunits; u += gridDim.x * ngrp) {
        const size_t row0 = (size_t)u * 2 * NL;              // first grid row of the unit
        const auto ld = [&](int c, int e, int l) {
            const double* pr = a.in + (size_t)c * N + ((row0 + 2 * l) << lg) + e;
            return make_double2(pr[0], pr[n]);
        };
        const auto st = [&](int c, int e, int l, double2 v) {
            double* pr = a.out + (size_t)c * N + ((row0 + 2 * l) << lg) + e;
            pr[0] = v.x;
            pr[n] = v.y;
        };
        wf_first<p.g[0]>(z, zl, R, lg, tab + p.toff[0], gp, ld);
        gp.sync();
        wf_middle<LG, false>(z, zl, R, tab, gp);
        if constexpr (p.ng >= 2) {
            wf_group<p.g[p.ng - 1], false>(z, zl, R, lg, 0, p.g[p.ng - 1], tab, gp);
            gp.sync();
        }
        // point-wise across the columns, in Fourier space: mixing in, phases, mixing out
        {
            const int items = n << lNL;
            for (int w = gp.tid; w < items; w += gp.nth) {
                const int l = w & (NL - 1), e = w >> lNL;
                double2* pz = z + zl.row(e) + l;
                double2 x[R];
#pragma unroll
                for (int c = 0; c < R; c++) x[c] = pz[c * zl.CP];
                if (has_min) dir_matvec<R>(x, mats);
                const double2* pp = phs + e * RP;
#pragma unroll
                for (int c = 0; c < R; c++) x[c] = cmul(x[c], pp[c]);
                if (has_mout) dir_matvec_store<R>(x, mats + MS, pz, zl.CP);
                else {
#pragma unroll
                    for (int c = 0; c < R; c++) pz[c * zl.CP] = x[c];
                }
            }
            gp.sync();
        }
        if (want_gram) {
            // Gram of the output from its spectrum: acc += sum over the unit of Y_I^T Y_J, both components of every element
            const int lane = threadIdx.x & 31, wig = gp.tid >> 5, nwg = gp.nth >> 5;
            const int ci = lane >> 2, k = lane & 3, comp = k & 1;
            const int items = n << lNL;
            for (int g = wig; g < (items >> 1); g += nwg) {
                const int w = 2 * g + (k >> 1);
                const int l = w & (NL - 1), e = w >> lNL;
                const double* base = (const double*)(z + zl.row(e) + l) + comp;
                double frag[NB];
#pragma unroll
                for (int I = 0; I < NB; I++) {
                    const int col = 8 * I + ci;
                    frag[I] = col < R ? base[(size_t)col * zl.CP * 2] : 0.0;
                }
#pragma unroll
                for (int I = 0; I < NB; I++)
#pragma unroll
                    for (int J = I; J < NB; J++) dmma884(gacc[GramShape<R>::tp(I, J)], frag[I], frag[J]);
            }
            gp.sync();      // every warp of the group has read the unit before the inverse transform rewrites it (two-warp units!)
        }
        if constexpr (p.ng >= 2) {
            wf_group<p.g[p.ng - 1], true>(z, zl, R, lg, 0, p.g[p.ng - 1], tab, gp);
            gp.sync();
        }
        wf_middle<LG, true>(z, zl, R, tab, gp);
        wf_last<p.g[0]>(z, zl, R, lg, tab + p.toff[0], gp, st);
        gp.sync();                                            // the unit is free for the next one
    }
    pdl_trigger();
    if (want_gram) {
        constexpr int P = R * (R + 1) / 2;
        __syncthreads();                                      // every unit is done: the buffers become reduction scratch
        double* part = a.gram + (size_t)blockIdx.x * P;
        const int cap = R * zl.CP * ngrp * 2;
        mma_tiles_reduce<NTP>(&gacc[0][0], (double*)zbase, cap > (int)(blockDim.x >> 5) * 64 ? cap : (int)(blockDim.x >> 5) * 64,
                              [&](int ai, int pos, double v) {
            const int i = pos >> 3, j = pos & 7;
            int I, J;
            tp_decode<R>(ai, I, J);
            const int ca = 8 * I + i, cb = 8 * J + j;
            if (ca <= cb && cb < R) part[upper_pair_index(R, ca, cb)] = v * (double)n;      // Parseval along x1
        });
        group_prereduce(a.gram, P, a.grp_cnt, a.gram2, a.gramF);
    }
}

template <int R, int LG>
inline cudaError_t launch_sub1_lg(const Sub1Args& a, int groups, int ctas, cudaStream_t st) {
    const size_t sm = sub1_smem_bytes(1 << LG, R, a.NL, groups);
    return dlr_launch(k_sub1<R, LG>, (unsigned)ctas, groups * a.wpu * 32, sm, st, a);
}

template <int R>
inline cudaError_t launch_sub1(const Sub1Args& a, int groups, int ctas, cudaStream_t st) {
    switch (a.g.log2n) {
        case 3: return launch_sub1_lg<R, 3>(a, groups, ctas, st);
        case 4: return launch_sub1_lg<R, 4>(a, groups, ctas, st);
        case 5: return launch_sub1_lg<R, 5>(a, groups, ctas, st);
        case 6: return launch_sub1_lg<R, 6>(a, groups, ctas, st);
        case 7: return launch_sub1_lg<R, 7>(a, groups, ctas, st);
        case 8: return launch_sub1_lg<R, 8>(a, groups, ctas, st);
        default: return cudaErrorInvalidValue;
    }
}

template <int R>
inline cudaError_t configure_sub1() {
    cudaError_t e = dlr_optin_smem(k_sub1<R, 3>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub1<R, 4>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub1<R, 5>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub1<R, 6>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub1<R, 7>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub1<R, 8>);
    return e;
}

// resident CTAs per SM of the variant for this grid size
template <int R>
inline int sub1_occupancy(int log2n, int threads, size_t sm) {
    int k = 0;
    cudaError_t e = cudaErrorInvalidValue;
    switch (log2n) {
        case 3: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub1<R, 3>, threads, sm); break;
        case 4: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub1<R, 4>, threads, sm); break;
        case 5: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub1<R, 5>, threads, sm); break;
        case 6: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub1<R, 6>, threads, sm); break;
        case 7: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub1<R, 7>, threads, sm); break;
        case 8: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub1<R, 8>, threads, sm); break;
    }
    return (e == cudaSuccess && k > 0) ? k : 1;
}
