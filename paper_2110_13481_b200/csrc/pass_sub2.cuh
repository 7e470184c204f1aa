// Sub-flow along direction 2 in the eigenbasis of C1_2 / D1_2 (eqs. (15), (18)):
//     A_j  <-  F_2^-1 [ exp(s i t k~_2 lambda_j) F_2 A_j ]        for every column j on its own
// The columns do not couple here (the change of eigenbasis sits in the passes before and after), so a unit is tiny:
// L = 4 packed lines (64 bytes along i1) x n points along i2 of ONE column at one i3 - one warp, 4-18 KB of shared
// memory, no barrier but __syncwarp.  The first radix group reads global memory straight into registers and the last
// inverse group writes its registers straight back: two round trips through shared memory per element.
// grid = (CTAs per column, r): the warps of a CTA share the column's n phases and the twiddle tables.
#pragma once
#include "wfft.cuh"

struct Sub2Args {
    GridDev g;
    const double* in;      // N x R real
    double* out;           // N x R real (may alias in)
    const double2* ph;     // [n][R] phases by stored position
    int R, L;              // columns, packed lines per unit (power of two <= n/2)
    int wpu;               // warps per unit (1: a warp owns a unit; 2, 4: a group with its own named barrier)
};

__host__ inline size_t sub2_unit_elems(int n, int L) { return (size_t)wf_padded(n, wf_plan(31 - __builtin_clz(n)).ps) * L; }
__host__ inline size_t sub2_smem_bytes(int n, int L, int groups) {
    const WPlan p = wf_plan(31 - __builtin_clz(n));
    return ((size_t)p.tlen + n + sub2_unit_elems(n, L) * groups) * 16;
}

template <int LG>
__global__ void __launch_bounds__(256) k_sub2(const Sub2Args a) {
    extern __shared__ double2 smem2[];
    constexpr int n = 1 << LG, lg = LG, M = n >> 1;
    constexpr WPlan p = wf_plan(LG);
    const int L = a.L, lL = __ffs(L) - 1;
    double2* tab = smem2;                       // twiddle tables
    double2* phs = tab + p.tlen;                // [n] phases of this CTA's column, times 1/n
    const int gsz = a.wpu << 5;                 // threads per group
    const int c = blockIdx.y, warp = (int)threadIdx.x / gsz, nwarp = (int)blockDim.x / gsz;   // group index, groups per CTA
    ZL zl;
    zl.L = L; zl.lL = lL; zl.ps = p.ps; zl.CP = 0;
    const int ne = wf_padded(n, p.ps) << lL;
    double2* z = phs + n + (size_t)warp * ne;
    wf_load_tables<LG>(tab, a.g.wtab);           // written by dlr_create: may precede pdl_wait()
    pdl_wait();
    const double invn = 1.0 / (double)n;
    for (int e = threadIdx.x; e < n; e += blockDim.x) {
        const double2 f = a.ph[(size_t)e * a.R + c];
        phs[e] = make_double2(f.x * invn, f.y * invn);
    }
    __syncthreads();
    Grp gp;
    gp.tid = (int)threadIdx.x - warp * gsz; gp.nth = gsz; gp.bar = 1 + warp;
    const int ljb = (lg - 1) - lL;              // log2 of units per plane (M / L)
    const int nunits = n << ljb;                // per column
    const size_t N2 = (size_t)(a.g.N >> 1);
    const double2* in2 = (const double2*)a.in + (size_t)c * N2;
    double2* out2 = (double2*)a.out + (size_t)c * N2;
    for (int u = blockIdx.x * nwarp + warp; u < nunits; u += gridDim.x * nwarp) {
        const int i3 = u >> ljb, j0 = (u & ((1 << ljb) - 1)) << lL;
        const size_t base = ((size_t)i3 << lg) * M + j0;       // (i3 n + e) M + j0 + l
        const auto ld = [&](int, int e, int l) { return in2[base + (size_t)e * M + l]; };
        const auto st = [&](int, int e, int l, double2 v) { out2[base + (size_t)e * M + l] = v; };
        const auto phase = [&](double2& v, int e, int) { v = cmul(v, phs[e]); };
        if constexpr (p.ng == 1) {
            // n <= 8: the whole transform is one register butterfly
            for (int l = gp.tid; l < L; l += gp.nth) {
                double2 x[8];
#pragma unroll
                for (int q = 0; q < 8; q++) x[q] = q < n ? ld(0, q, l) : make_double2(0.0, 0.0);
                bfly<3, false>(x);
#pragma unroll
                for (int q = 0; q < 8; q++) phase(x[q], q, 0);
                bfly<3, true>(x);
#pragma unroll
                for (int q = 0; q < 8; q++) st(0, q, l, x[q]);
            }
        } else {
            wf_first<p.g[0]>(z, zl, 1, lg, tab + p.toff[0], gp, ld);
            gp.sync();
            wf_middle<LG, false>(z, zl, 1, tab, gp);
            wf_mid<p.g[p.ng - 1]>(z, zl, 1, lg, gp, phase);
            gp.sync();
            wf_middle<LG, true>(z, zl, 1, tab, gp);
            wf_last<p.g[0]>(z, zl, 1, lg, tab + p.toff[0], gp, st);
            gp.sync();                              // the unit is free for the next one
        }
    }
    pdl_trigger();
}

inline cudaError_t launch_sub2(const Sub2Args& a, int groups, int ctas_per_col, cudaStream_t st) {
    const size_t sm = sub2_smem_bytes(a.g.n, a.L, groups);
    const int warps = groups * a.wpu;
    const dim3 grid((unsigned)ctas_per_col, (unsigned)a.R);
    switch (a.g.log2n) {
        case 3: return dlr_launch(k_sub2<3>, grid, warps * 32, sm, st, a);
        case 4: return dlr_launch(k_sub2<4>, grid, warps * 32, sm, st, a);
        case 5: return dlr_launch(k_sub2<5>, grid, warps * 32, sm, st, a);
        case 6: return dlr_launch(k_sub2<6>, grid, warps * 32, sm, st, a);
        case 7: return dlr_launch(k_sub2<7>, grid, warps * 32, sm, st, a);
        case 8: return dlr_launch(k_sub2<8>, grid, warps * 32, sm, st, a);
        default: return cudaErrorInvalidValue;
    }
}

// resident CTAs per SM of the variant for this grid size (registers and shared memory)
inline int sub2_occupancy(int log2n, int warps, size_t sm) {
    int k = 0;
    cudaError_t e = cudaErrorInvalidValue;
    switch (log2n) {
        case 3: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub2<3>, warps * 32, sm); break;
        case 4: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub2<4>, warps * 32, sm); break;
        case 5: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub2<5>, warps * 32, sm); break;
        case 6: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub2<6>, warps * 32, sm); break;
        case 7: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub2<7>, warps * 32, sm); break;
        case 8: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k, k_sub2<8>, warps * 32, sm); break;
    }
    return (e == cudaSuccess && k > 0) ? k : 1;
}

inline cudaError_t configure_sub2() {
    cudaError_t e = dlr_optin_smem(k_sub2<3>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub2<4>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub2<5>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub2<6>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub2<7>);
    if (e == cudaSuccess) e = dlr_optin_smem(k_sub2<8>);
    return e;
}
