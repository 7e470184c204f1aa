// C ABI of include/dlr.h: context, workspace carving, and the orchestration of one step of Algorithm 2
// / Algorithm 1 as a fixed sequence of kernels on one stream, replayed as a
// CUDA graph.  No CPU fallback anywhere: every stage is a kernel launch.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/dlr.h"
#include "rank_ops.h"
#include "small.cuh"
#include "pass_sub2.cuh"

extern "C" {
const RankOps* dlr_rank_ops_5();
const RankOps* dlr_rank_ops_8();
const RankOps* dlr_rank_ops_10();
const RankOps* dlr_rank_ops_15();
const RankOps* dlr_rank_ops_20();
}

const RankOps* dlr_rank_ops(int R) {
    switch (R) {
        case 5: return dlr_rank_ops_5();
        case 8: return dlr_rank_ops_8();
        case 10: return dlr_rank_ops_10();
        case 15: return dlr_rank_ops_15();
        case 20: return dlr_rank_ops_20();
        default: return nullptr;
    }
}

thread_local int g_dlr_pdl = 0;     // common.cuh: dlr_launch sets the programmatic-serialisation attribute while this is 1

namespace {

struct HostGrid {
    GridDev g;
    int T1;               // rows per CTA in dimension-1 passes (rank columns)
    int T1s;              // same for the 1..3 column field passes
    int T3, T3s;          // pencils per CTA in dimension-3 passes
    int T2, NB2, nch2;    // dimension-2 pass tiling
    int thr1, thr2, thr3; // CTA sizes of the three pass families
    int Lx, Le, Lc;       // directional passes: packed lines per column for EXACT, ETD and COEFF tiles
    int thrx, thre, thrc; // CTA sizes of the EXACT, ETD and COEFF directional passes
    int Lc2, thrc2;       // the Parseval-only coefficient passes (directions 2, 3)
    int thrx2;            // CTA size of the direction-2 sub-flow (register-light: up to 512 threads)
};

struct FlowTab {
    FlowTabPtrs p;
};

#define DLR_CROSS_CTAS 148
struct Sub2Cfg { int L, groups, wpu, ctas; };      // launch shape of the direction-2 sub-flow (pass_sub2.cuh)
struct ApplyCfg { int C, S, ctas; };              // chunk length, stages and grid of the A*Mat pass (pass_apply.cuh)
struct Sub1Cfg { int use, NL, groups, wpu, ctas; };  // launch shape of the direction-1 sub-flow (pass_sub1.cuh); use = 0: CTA-tile kernel

struct Phase {
    const char* name;
    cudaEvent_t ev;
};

}  // namespace

struct dlr_ctx {
    dlr_config cfg;
    int R;
    int dev;                      // device of the workspace: every entry point runs under it (DevGuard)
    int nsm;                      // its number of SMs (persistent grids)
    cudaStream_t st, cap_st;
    cudaStream_t side;            // side branch: the coefficient/eigen kernel overlaps the dim-2/3 passes of its transform
    cudaEvent_t ev_fork, ev_join;
    cudaEvent_t ev_mfork;             // marginals of V on the side branch (joined by the coefficient set's join)
    cudaEvent_t ev_ffork, ev_fjoin;   // field solve on the side stream, joined before the first pass that reads E
    bool field_pending;
    bool tc_warm, td_warm;            // TC / TD hold a previous eigen-decomposition (warm start of the Jacobi solves)
    double bytes_acc, bytes_step;     // algorithmic bytes of the factor-sized passes issued by the current / last step
    const RankOps* ops;
    HostGrid gx, gv;
    Sub2Cfg s2x, s2v;
    Sub1Cfg s1x, s1v;
    ApplyCfg apx, apv;
    // big buffers
    double *X, *X1, *V, *S, *Sp;     // X1: the predictor basis of Algorithm 2 (X itself stays X0 until the first K step)
    double2* Eh;
    double *KL, *Q1, *W, *E;
    double* Em;                   // field of the diagnostics (dlr_moments): c->E stays the field used last by dlr_step
    double *partial, *partialP[3], *partialC, *partial2a;
    double *margp1, *margp2;                 // marginals of V: partial planes of k_marginals
    MargOut marg;                            // M1, M2, M3 ([r][n_v] each), their DFTs and moments (k_marg_reduce)
    double *gram2, *pgram2[3], *colsum2;     // group sums of the per-CTA partial rows (group_prereduce)
    double *gramF, *pgramF[3], *colsumF;     // and their totals (one row each): what the consumers read
    unsigned* grp_cnt;                       // 3 x DLR_CNT_STRIDE group counters, zero between kernels
    // small buffers
    double *crossM, *crossN;      // per-CTA partial blocks of <X1, X0>, <V1, V0> (unconventional integrator)
    double *C1, *C2, *D1, *D2, *rho_t, *TC, *lamC, *TD, *lamD, *apply, *Rtot, *zsum, *mx, *mv, *mxp, *mvp, *mres, *esum;
    int* status;
    long long *pix, *piv;
    double* pf;
    int probe_cap;
    int pdl;                      // programmatic dependent launch for the kernels of a step (see dlr_create)
    FlowTab ft;
    double* small_end;
    bool has_state, vh_valid, profiling;
    int prof_level;               // 1: events between phases; 2: an event after every launch
    int launches, count_launches;
    cudaGraphExec_t graph;
    double graph_tau;
    cudaError_t last_err;
    std::string last_err_msg;
    std::vector<Phase> phases;
    std::vector<float> phase_ms;
    std::vector<const char*> phase_names;
    size_t partial_cap;
};

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// programmatic dependent launch (common.cuh) is on while dlr_step issues or captures a step, off in every other entry point
struct PdlScope {
    explicit PdlScope(int on) { g_dlr_pdl = on; }
    ~PdlScope() { g_dlr_pdl = 0; }
};

// every entry point that touches the device runs with the context's device current and restores the caller's
struct DevGuard {
    int prev;
    bool switched;
    explicit DevGuard(int dev) : prev(-1), switched(false) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DevGuard() { if (switched) cudaSetDevice(prev); }
};

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
int ilog2(int n) { int l = 0; while ((1 << l) < n) l++; return l; }
int brev_host(int k, int bits) { int r = 0; for (int i = 0; i < bits; i++) if (k & (1 << i)) r |= 1 << (bits - 1 - i); return r; }

// ---- tiling choices (shared-memory budget: <= ~110 KB so that two CTAs fit an SM when the problem allows) ----
const size_t SMEM_TARGET = 110 * 1024, SMEM_MAX = 227 * 1024;

int choose_T1(int n, int RMAX, bool needE, int nmat) {
    const long long rows = (long long)n * n;
    int best = 1;
    for (int T = 1; T <= rows && T <= 64; T *= 2) {
        const size_t sm = d1_smem_bytes(n, RMAX, T, needE, nmat);
        if (sm > SMEM_TARGET && T > 1) break;
        if (rows / T >= 148 || T <= 4) best = T;     // measured: larger tiles win as long as every SM gets one
    }
    while (best > 1 && d1_smem_bytes(n, RMAX, best, needE, nmat) > SMEM_MAX) best /= 2;
    return best;
}

int choose_T3(int n, int RMAX, int nmat) {
    int best = 1;
    for (int T = 1; T <= 16; T *= 2) {
        const size_t sm = d3_smem_bytes(n, RMAX, T, nmat);
        if (sm <= SMEM_TARGET || (T <= 2 && sm <= SMEM_MAX)) best = T;
    }
    return best;
}

// Tuning overrides for experiments, compiled in only with -DDLR_ENABLE_TUNE (never in the product build):
// DLR_TUNE="t1=8,t3=4,nb2=1,smem2=48,thr1=256,thr2=256,thr3=128" (all optional).
// Values are validated by the callers (powers of two, shared-memory limits); unknown keys are ignored.
int tune(const char* key, int dflt) {
#ifndef DLR_ENABLE_TUNE
    (void)key;
    return dflt;                              // product builds: fixed tile rules, no environment dependence
#endif
    const char* e = getenv("DLR_TUNE");
    if (!e) return dflt;
    const std::string s(e), k = std::string(key) + "=";
    size_t pos = 0;
    while ((pos = s.find(k, pos)) != std::string::npos) {
        if (pos == 0 || s[pos - 1] == ',') return atoi(s.c_str() + pos + k.size());
        pos += k.size();
    }
    return dflt;
}

int valid_threads(int t) { return (t == 64 || t == 128 || t == 256) ? t : DLR_THREADS; }

void choose_T2(int n, int nh, int& T2, int& NB, int& nch) {
    const size_t target = (size_t)tune("smem2", 48) * 1024;
    int lines = (int)(target / ((size_t)n * 16));
    if (lines > 255) lines = 255;
    if (lines < 1) lines = 1;
    nch = (nh + lines - 1) / lines;
    T2 = (nh + nch - 1) / nch;
    NB = lines / T2;
    const int nbo = tune("nb2", 0);
    if (nbo > 0) NB = nbo;
    if (NB < 1) NB = 1;
    if (NB > 16) NB = 16;
    while (NB > 1 && d2_smem_bytes(n, T2, NB) > SMEM_MAX) NB--;
}

// packed lines per column of a directional tile: the largest power of two <= lmax whose tile fits the target
int choose_L(int n, int R, int nbuf, int nmat, bool needE, size_t target, int lmax) {
    int best = 1;
    for (int L = 1; L <= lmax && L <= n / 2; L *= 2)
        if (dir_smem_bytes(n, R, L, nbuf, nmat, needE) <= target) best = L;
    return best;
}

struct Carver {
    char* base;
    size_t off;
    template <class Tp>
    Tp* take(size_t count) {
        off = align_up(off, 256);
        Tp* p = base ? (Tp*)(base + off) : nullptr;
        off += count * sizeof(Tp);
        return p;
    }
};

int check_cfg(const dlr_config* c) {
    if (!c) return DLR_ERR_INVALID;
    for (int d = 1; d < 3; d++)
        if (c->n_x[d] != c->n_x[0] || c->n_v[d] != c->n_v[0]) return DLR_ERR_UNSUPPORTED;
    const int nx = c->n_x[0], nv = c->n_v[0];
    if (!is_pow2(nx) || !is_pow2(nv) || nx < 8 || nv < 8 || nx > 256 || nv > 256) return DLR_ERR_UNSUPPORTED;
    if (!dlr_rank_ops(c->rank)) return DLR_ERR_UNSUPPORTED;
    if (c->order != 1 && c->order != 2) return DLR_ERR_INVALID;
    if ((c->flags & ~(uint32_t)(DLR_FLAG_PREDICTOR_L_FLOW | DLR_FLAG_UNCONVENTIONAL)) != 0) return DLR_ERR_INVALID;
    if ((c->flags & DLR_FLAG_UNCONVENTIONAL) && c->order != 1) return DLR_ERR_INVALID;
    for (int d = 0; d < 3; d++) {
        if (!(c->x_hi[d] > c->x_lo[d]) || !(c->v_hi[d] > c->v_lo[d])) return DLR_ERR_INVALID;
        if (c->x_lo[d] != c->x_lo[0] || c->x_hi[d] != c->x_hi[0] || c->v_lo[d] != c->v_lo[0] || c->v_hi[d] != c->v_hi[0])
            return DLR_ERR_UNSUPPORTED;     // cubic boxes only (all configs of BASELINE.json)
    }
    return DLR_OK;
}

size_t grid_table_doubles(int n) { return (size_t)(2 * (n / 2 + 1) + 2 * n + n) + 8; }

// carve the workspace; with base == nullptr only measures
size_t carve(dlr_ctx* c, char* base) {
    const int R = c->R;
    const long long Nx = c->gx.g.N, Nv = c->gv.g.N, NCx = c->gx.g.NC;
    const long long Nmax = Nx > Nv ? Nx : Nv;
    Carver cv{base, 0};
    c->X = cv.take<double>((size_t)Nx * R);
    c->X1 = cv.take<double>((size_t)Nx * R);
    c->V = cv.take<double>((size_t)Nv * R);
    c->KL = cv.take<double>((size_t)Nmax * R);
    c->Q1 = cv.take<double>((size_t)Nmax * R);
    c->W = cv.take<double>((size_t)Nmax * R);
    c->E = cv.take<double>((size_t)3 * Nx);
    c->Em = cv.take<double>((size_t)3 * Nx);
    c->Eh = cv.take<double2>((size_t)3 * NCx);
    // per-CTA partial sums: the largest producer is a dimension-1 pass with the weighted Gram
    const int nvmax = 3 * R * (R + 1) / 2 + R;
    size_t blocks = 0;
    for (const HostGrid* hg : {&c->gx, &c->gv}) {
        size_t b1 = (size_t)hg->g.n * hg->g.n / hg->T1;
        size_t bd = (size_t)dir_tiles(hg->g.n, 1);            // directional tiles at L = 1 (the most there can be)
        bd = std::max(std::max(bd / hg->Lx, bd / hg->Lc2), std::max(bd / hg->Le, bd / hg->Lc));
        blocks = std::max(blocks, std::max(b1, bd));
        blocks = std::max(blocks, std::min((size_t)dir_tiles(hg->g.n, 1), (size_t)2048));   // persistent grids (pass_sub1.cuh)
    }
    c->partial_cap = blocks * nvmax;
    c->partial = cv.take<double>(c->partial_cap);
    for (int d = 0; d < 3; d++) c->partialP[d] = cv.take<double>(blocks * (size_t)(R * (R - 1) / 2));   // Parseval sums
    c->partialC = cv.take<double>(blocks * (size_t)R);                                                  // column sums
    const size_t groups = (size_t)dlr_groups((int)blocks) + 1;
    c->gram2 = cv.take<double>(groups * nvmax);
    for (int d = 0; d < 3; d++) c->pgram2[d] = cv.take<double>(groups * (size_t)(R * (R - 1) / 2));
    c->colsum2 = cv.take<double>(groups * (size_t)R);
    c->gramF = cv.take<double>(nvmax);
    for (int d = 0; d < 3; d++) c->pgramF[d] = cv.take<double>((size_t)(R * (R - 1) / 2));
    c->colsumF = cv.take<double>(R);
    c->grp_cnt = cv.take<unsigned>(3 * DLR_CNT_STRIDE);
    {
        const size_t nv = (size_t)c->gv.g.n;
        c->margp1 = cv.take<double>((size_t)R * nv * nv);
        c->margp2 = cv.take<double>((size_t)R * nv * nv);
        c->marg.M1 = cv.take<double>((size_t)R * nv); c->marg.M2 = cv.take<double>((size_t)R * nv);
        c->marg.M3 = cv.take<double>((size_t)R * nv);
        c->marg.Ph1 = cv.take<double2>((size_t)R * nv); c->marg.Ph2 = cv.take<double2>((size_t)R * nv);
        c->marg.s0 = cv.take<double>(R); c->marg.mom3 = cv.take<double>(R);
        c->marg.Wv = cv.take<double2>(nv);
    }
    c->partial2a = cv.take<double>((size_t)DLR_G1 * nvmax);
    const int RR = R * R;
    c->S = cv.take<double>(RR); c->Sp = cv.take<double>(RR);
    c->C1 = cv.take<double>(3 * RR); c->C2 = cv.take<double>(3 * RR);
    c->D1 = cv.take<double>(3 * RR); c->D2 = cv.take<double>(3 * RR);
    c->rho_t = cv.take<double>(R);
    c->TC = cv.take<double>(3 * RR); c->lamC = cv.take<double>(3 * R);
    c->TD = cv.take<double>(3 * RR); c->lamD = cv.take<double>(3 * R);
    c->apply = cv.take<double>(RR); c->Rtot = cv.take<double>(RR);
    c->crossM = cv.take<double>((size_t)DLR_CROSS_CTAS * RR); c->crossN = cv.take<double>((size_t)DLR_CROSS_CTAS * RR);
    c->zsum = cv.take<double>(R);
    c->mx = cv.take<double>(5 * R); c->mv = cv.take<double>(5 * R); c->mres = cv.take<double>(8);
    c->mxp = cv.take<double>((size_t)5 * R * DLR_MCH); c->mvp = cv.take<double>((size_t)5 * R * DLR_MCH); c->esum = cv.take<double>(DLR_ECH);
    c->status = cv.take<int>(4);
    c->probe_cap = 4096;
    // Programmatic dependent launch pays where a pass is short (L2-resident factors: 64^3, r = 10: 1.029 -> 1.009 ms/step);
    // with HBM-resident factors the early-resident CTAs of the next pass only take slots (128^3, r = 15: 11.43 -> 11.51 ms)
    c->pdl = tune("pdl", 8.0 * (double)std::max(c->gx.g.N, c->gv.g.N) * c->R <= 64.0 * 1024 * 1024 ? 1 : 0);
    c->pix = cv.take<long long>(c->probe_cap); c->piv = cv.take<long long>(c->probe_cap); c->pf = cv.take<double>(c->probe_cap);
    const int nmax = std::max(c->gx.g.n, c->gv.g.n);
    c->ft.p.mats = cv.take<double>(8 * RR);
    c->ft.p.Q = cv.take<double>(3 * RR);
    c->ft.p.ph1 = cv.take<double2>((size_t)nmax * R);
    c->ft.p.ph2 = cv.take<double2>((size_t)nmax * R);
    c->ft.p.ez = cv.take<double2>((size_t)nmax * R);
    c->ft.p.f1 = cv.take<double2>((size_t)nmax * R);
    c->ft.p.f2a = cv.take<double2>((size_t)nmax * R);
    c->ft.p.f2b = cv.take<double2>((size_t)nmax * R);
    // grid tables
    for (HostGrid* hg : {&c->gx, &c->gv}) {
        const int n = hg->g.n, nh = hg->g.nh;
        double* t = cv.take<double>(grid_table_doubles(n));
        hg->g.kt1 = t; hg->g.ksq1 = t ? t + nh : nullptr;
        hg->g.kt2p = t ? t + 2 * nh : nullptr; hg->g.ksq2p = t ? t + 2 * nh + n : nullptr;
        double2* tw = cv.take<double2>(n / 2);
        hg->g.tw = tw;
        hg->g.wtab = cv.take<double2>((size_t)wf_plan(hg->g.log2n).tlen + 1);
    }
    return align_up(cv.off, 256);
}

void setup_grid(HostGrid& hg, int n, double lo, double hi, int R) {
    hg.g.n = n; hg.g.nh = n / 2 + 1; hg.g.log2n = ilog2(n);
    hg.g.N = (long long)n * n * n; hg.g.NC = (long long)hg.g.nh * n * n;
    hg.g.lo = lo; hg.g.h = (hi - lo) / n; hg.g.h3 = hg.g.h * hg.g.h * hg.g.h;
    hg.T1 = choose_T1(n, R, true, 3 * R * R);
    hg.T1s = choose_T1(n, 3, false, 4);
    hg.T3 = choose_T3(n, R, 4 * R * R);
    hg.T3s = choose_T3(n, 3, 0);
    { const int v = tune("t1s", 0); if (is_pow2(v) && v <= n * n) hg.T1s = v; }
    { const int v = tune("t3s", 0); if (is_pow2(v) && v <= 16) hg.T3s = v; }
    const int t1 = tune("t1", 0), t3 = tune("t3", 0);
    if (is_pow2(t1) && t1 <= n * n && d1_smem_bytes(n, R, t1, true, 3 * R * R) <= SMEM_MAX) hg.T1 = t1;
    if (is_pow2(t3) && t3 <= 16 && d3_smem_bytes(n, R, t3, 4 * R * R) <= SMEM_MAX) hg.T3 = t3;
    choose_T2(n, hg.g.nh, hg.T2, hg.NB2, hg.nch2);
    hg.thr1 = valid_threads(tune("thr1", DLR_THREADS));
    hg.thr2 = valid_threads(tune("thr2", DLR_THREADS));
    hg.thr3 = valid_threads(tune("thr3", DLR_THREADS));
    auto dthreads = [](int t) { return (t >= 64 && t <= DLR_THREADS && t % 32 == 0) ? t : DLR_THREADS; };
    hg.thrx = dthreads(tune("thrx", DLR_THREADS));
    // third sub-flow above rank 10: one CTA per SM (register budget), so 512 threads (128 registers each) instead of 256
    { const int t = tune("thre", R > 10 ? 2 * DLR_THREADS : DLR_THREADS);
      hg.thre = (t >= 64 && t <= (R > 10 ? 2 : 1) * DLR_THREADS && t % 32 == 0) ? t : DLR_THREADS; }
    { const int t = tune("thrx2", 0); hg.thrx2 = (t >= 64 && t <= 2 * DLR_THREADS && t % 32 == 0) ? t : 0; }
    hg.thrc = dthreads(tune("thrc", DLR_THREADS));
    const int lmax = 8;
    hg.Lx = choose_L(n, R, 1, 2, false, (size_t)tune("smx", 96) * 1024, lmax);
    hg.Le = choose_L(n, R, 2, 5, true, (size_t)tune("sme", 110) * 1024, lmax);
    hg.Lc = choose_L(n, R, 1, 2, true, (size_t)tune("smc", 110) * 1024, lmax);
    // a tile with a single packed line per column means 16-byte strided segments in directions 2 and 3: measured at
    // configs 4 and 5 it pays to give such a tile all of the shared memory (one CTA per SM) to reach two lines
    const size_t smem_all = SMEM_MAX - 1024;
    if (hg.Lx < 2) hg.Lx = choose_L(n, R, 1, 2, false, smem_all, 2);
    if (hg.Le < 2) hg.Le = choose_L(n, R, 2, 5, true, smem_all, 2);
    if (hg.Lc < 2) hg.Lc = choose_L(n, R, 1, 2, true, smem_all, 2);
    const int lx = tune("lx", 0), le = tune("le", 0), lc = tune("lc", 0);
    if (is_pow2(lx) && lx <= n / 2 && dir_smem_bytes(n, R, lx, 1, 2, false) <= SMEM_MAX) hg.Lx = lx;
    if (is_pow2(le) && le <= n / 2 && dir_smem_bytes(n, R, le, 2, 5, true) <= SMEM_MAX) hg.Le = le;
    if (is_pow2(lc) && lc <= n / 2 && dir_smem_bytes(n, R, lc, 1, 2, true) <= SMEM_MAX) hg.Lc = lc;
    // Parseval-only passes (no weighted Gram): at 64^3, r = 10 half-size tiles with 192 threads, three CTAs per SM, read the
    // factor in 22.6 / 20.6 us (directions 2 / 3) against 23.7 / 22.6 with the tiles of the first pass (which wants them
    // large: 42.6 us at L = 8, 52.9 at L = 4)
    hg.Lc2 = hg.Lc; hg.thrc2 = hg.thrc;
    if (n == 64 && R <= 10 && hg.Lc == 8 && tune("lc", 0) == 0 && tune("thrc", 0) == 0) { hg.Lc2 = 4; hg.thrc2 = 192; }
    if (hg.thrx2 == 0) {
        // the direction-2 sub-flow is register-light (up to 512 threads per CTA): 320 threads when the butterfly items of
        // an FFT group (n/8 per line) then divide evenly, e.g. 640 items at n = 64, r = 10, 8 lines per column
        const int items = (n / 8) * R * hg.Lx;
        hg.thrx2 = (n >= 8 && items % 320 == 0) ? 320 : DLR_THREADS;
    }
}

cudaError_t upload_tables(dlr_ctx* c, HostGrid& hg, double lo, double hi) {
    const int n = hg.g.n, nh = hg.g.nh, lg = hg.g.log2n;
    const double L = hi - lo, PI = 3.14159265358979323846264338327950288;
    std::vector<double> t(grid_table_doubles(n), 0.0);
    for (int k = 0; k < nh; k++) {
        const double kk = 2.0 * PI * k / L;
        t[k] = (k == n / 2) ? 0.0 : kk;           // odd-derivative wavenumber, zero at Nyquist (R4)
        t[nh + k] = kk * kk;                      // true k^2
    }
    for (int e = 0; e < n; e++) {
        const int f = brev_host(e, lg);
        const int m = f < n / 2 ? f : f - n;
        const double kk = 2.0 * PI * m / L;
        t[2 * nh + e] = (f == n / 2) ? 0.0 : kk;
        t[2 * nh + n + e] = kk * kk;
    }
    cudaError_t e = cudaMemcpyAsync((void*)hg.g.kt1, t.data(), t.size() * sizeof(double), cudaMemcpyHostToDevice, c->st);
    if (e != cudaSuccess) return e;
    std::vector<double2> tw(n / 2);
    for (int k = 0; k < n / 2; k++) {
        const long double a = -2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)n;
        tw[k] = make_double2((double)cosl(a), (double)sinl(a));
    }
    e = cudaMemcpyAsync((void*)hg.g.tw, tw.data(), tw.size() * sizeof(double2), cudaMemcpyHostToDevice, c->st);
    if (e != cudaSuccess) return e;
    std::vector<double2> wt((size_t)wf_plan(lg).tlen + 1);
    wf_host_tables(lg, wt.data());
    e = cudaMemcpyAsync((void*)hg.g.wtab, wt.data(), wt.size() * sizeof(double2), cudaMemcpyHostToDevice, c->st);
    if (e != cudaSuccess) return e;
    return cudaStreamSynchronize(c->st);
}

// ---------------------------------------------------------------------------------------------------------
// launch helpers.  Every launch goes through CK so that the first failure is latched and counted.
#define CK(expr)                                                      \
    do {                                                              \
        cudaError_t _e = (expr);                                      \
        if (_e != cudaSuccess && c->last_err == cudaSuccess) {        \
            c->last_err = _e;                                         \
            c->last_err_msg = std::string(#expr) + ": " + cudaGetErrorString(_e); \
        }                                                             \
        c->count_launches++;                                          \
        if (c->prof_level == 2) launch_mark(c, #expr);                \
    } while (0)

void launch_mark(dlr_ctx* c, const char* name);

void phase_mark(dlr_ctx* c, const char* name) {
    if (!c->profiling || (c->prof_level == 2 && strcmp(name, "start") != 0)) return;
    Phase p;
    p.name = name;
    cudaEventCreate(&p.ev);
    cudaEventRecord(p.ev, c->st);
    c->phases.push_back(p);
}

void launch_mark(dlr_ctx* c, const char* name) {
    Phase p;
    p.name = name;
    cudaEventCreate(&p.ev);
    cudaEventRecord(p.ev, c->st);
    c->phases.push_back(p);
}

void run_d2(dlr_ctx* c, const HostGrid& hg, double2* data, int ncols, bool inv) {
    D2Args a;
    a.g = hg.g; a.data = data; a.ncols = ncols; a.T2 = hg.T2; a.NB = hg.NB2; a.nchunks = hg.nch2; a.threads = hg.thr2;
    if (inv) CK(launch_d2<true>(a, c->st)); else CK(launch_d2<false>(a, c->st));
}

D1Args d1args(dlr_ctx* c, const HostGrid& hg) {
    D1Args a;
    memset(&a, 0, sizeof(a));
    a.g = hg.g; a.T = hg.T1; a.scale = 2.0 / (double)hg.g.N; a.threads = hg.thr1;
    a.partial2 = c->gram2; a.partialF = c->gramF; a.grp_cnt = c->grp_cnt;
    return a;
}

D3Args d3args(dlr_ctx* c, const HostGrid& hg) {
    D3Args a;
    memset(&a, 0, sizeof(a));
    a.g = hg.g; a.T = hg.T3; a.e_scale = c->cfg.e_scale; a.threads = hg.thr3;
    return a;
}

void reduce_partials(dlr_ctx* c, int nblocks, int nvals, double* out2) {
    k_reduce_partials<<<DLR_G1, 256, 0, c->st>>>(c->partial, nblocks, nvals, out2);
    CK(cudaGetLastError());
}

int d1_blocks(const HostGrid& hg) { return (int)((long long)hg.g.n * hg.g.n / hg.T1); }
int d3_blocks(const HostGrid& hg) { return (int)(((long long)hg.g.nh * hg.g.n + hg.T3 - 1) / hg.T3); }

// algorithmic bytes: one real factor (N x r doubles) read or written counts B = 8 N r; the field adds 8 N per component
double fac_bytes(dlr_ctx* c, const HostGrid& hg) { return 8.0 * (double)hg.g.N * c->R; }

DirArgs dirargs(dlr_ctx* c, const HostGrid& hg) {
    DirArgs a;
    memset(&a, 0, sizeof(a));
    a.g = hg.g; a.threads = hg.thrx;
    a.gram2 = c->gram2; a.colsum2 = c->colsum2; a.grp_cnt = c->grp_cnt;
    a.gramF = c->gramF; a.colsumF = c->colsumF;
    return a;
}
int dir_blocks(const HostGrid& hg, int L) { return dir_tiles(hg.g.n, L); }

// sub-flow along direction 2 (pass_sub2.cuh): one warp per unit, as many resident warps as the SM holds
void setup_sub2(dlr_ctx* c, const HostGrid& hg, Sub2Cfg& sc) {
    // measured at 64^3, r = 10 (B200): 128-byte segments (L = 8) and small CTAs (4 groups) win: 14.4 us per pass
    // against 18.4 (L = 4, 8 warps) and 19.1 for the CTA-tile kernel of round 1.  Larger n: keep a unit near 10 KB
    // per warp (L = 4, and two warps per unit at n = 256)
    const int n = hg.g.n, M = n / 2;
    sc.L = n <= 64 ? std::min(M, 8) : 4;
    sc.wpu = n >= 256 ? 2 : 1;
    sc.groups = n >= 256 ? 2 : (n <= 64 ? 5 : 4); // measured at 256^3, r = 20: 2123 -> 1956 us per pass with two 2-warp groups;
                                                  // at 64^3, r = 10 (us per pass): 2 groups 19.0, 3: 15.5, 4: 15.6, 5: 15.1, 8: 17.0
    { const int l = tune("s2l", 0); if (is_pow2(l) && l <= M) sc.L = l; }
    { const int w = tune("s2w", 0); if (w >= 1 && w <= 8) sc.groups = w; }
    { const int w = tune("s2u", 0); if (w == 1 || w == 2 || w == 4) sc.wpu = w; }
    while (sc.groups > 1 && sub2_smem_bytes(n, sc.L, sc.groups) > SMEM_MAX - 1024) sc.groups /= 2;
    const int per_sm = sub2_occupancy(hg.g.log2n, sc.groups * sc.wpu, sub2_smem_bytes(n, sc.L, sc.groups));
    const int units = n * (M / sc.L);
    const int want = (c->nsm * per_sm + c->R - 1) / c->R;                 // CTAs per column to fill the device once
    sc.ctas = std::max(1, std::min(want, (units + sc.groups - 1) / sc.groups));
}
cudaError_t run_sub2(dlr_ctx* c, const HostGrid& hg, const double* in, double* out, const double2* ph) {
    const Sub2Cfg& sc = (&hg == &c->gx) ? c->s2x : c->s2v;
    Sub2Args a;
    a.g = hg.g; a.in = in; a.out = out; a.ph = ph; a.R = c->R; a.L = sc.L; a.wpu = sc.wpu;
    return launch_sub2(a, sc.groups, sc.ctas, c->st);
}

// sub-flow along direction 1 with both changes of basis (pass_sub1.cuh): one warp per unit of NL packed lines of all
// columns.  Units above 48 KB (n = 256 at the larger ranks) stay with the CTA-tile kernel k_dir<r,1,EXACT>.
void setup_sub1(dlr_ctx* c, const HostGrid& hg, Sub1Cfg& sc) {
    const int n = hg.g.n, R = c->R;
    sc.NL = n >= 64 ? 1 : 64 / n;
    { const int l = tune("s1l", 0); if (is_pow2(l) && l <= n * n / 2) sc.NL = l; }
    const size_t unit = sub1_unit_elems(n, R, sc.NL) * 16;
    sc.wpu = unit <= 24 * 1024 ? 1 : 2;
    { const int w = tune("s1u", 0); if (w == 1 || w == 2 || w == 4) sc.wpu = w; }
    sc.use = unit <= (size_t)tune("s1max", 48) * 1024 && tune("s1", 1) != 0;
    sc.groups = 8 / sc.wpu;
    { const int w = tune("s1w", 0); if (w >= 1 && w <= 8 / sc.wpu) sc.groups = w; }
    // up to rank 10 two CTAs share an SM (110 KB each); above, one CTA owns it (register budget): more units per CTA
    // (128^3, r = 15: 365 -> 332 us per pass)
    const size_t target = (size_t)tune("s1sm", R > 10 ? 200 : 110) * 1024;
    while (sc.groups > 1 && sub1_smem_bytes(n, R, sc.NL, sc.groups) > target) sc.groups--;
    if (sub1_smem_bytes(n, R, sc.NL, sc.groups) > SMEM_MAX - 1024) sc.use = 0;
    if (!sc.use) return;
    const int units = (n * n / 2) / sc.NL;
    // Every warp (group) owns whole units and all warps of the single wave run in step, so the pass lasts as long as the
    // SM with the most units: one group fewer per CTA can spread the units evenly (64^3, r = 10: 2048 units as 256 CTAs of
    // 8 warps put 16 on 108 SMs and 8 on the others; 293 CTAs of 7 warps put 14 on each: 30.1 -> 28.1 us per pass)
    const auto plan = [&](int g, int& ctas) {
        const int per_sm = c->ops->sub1_occ(hg.g.log2n, g * sc.wpu * 32, sub1_smem_bytes(n, R, sc.NL, g));
        ctas = std::max(1, std::min(c->nsm * per_sm, (units + g - 1) / g));
        const int upw = (units + ctas * g - 1) / (ctas * g);
        return ((ctas + c->nsm - 1) / c->nsm) * g * upw;           // units of the busiest SM
    };
    int ctas_a = 1, ctas_b = 1;
    const int cost_a = plan(sc.groups, ctas_a);
    sc.ctas = ctas_a;
    if (sc.groups > 2 && tune("s1w", 0) == 0 && plan(sc.groups - 1, ctas_b) < cost_a) { sc.groups--; sc.ctas = ctas_b; }
}
cudaError_t run_sub1(dlr_ctx* c, const HostGrid& hg, const DirArgs& d) {
    const Sub1Cfg& sc = (&hg == &c->gx) ? c->s1x : c->s1v;
    if (!sc.use) return c->ops->dir[VD_EXACT1](d, c->st);
    Sub1Args a;
    a.g = hg.g; a.in = d.in; a.out = d.out; a.min_ = d.min_; a.mout = d.mout; a.ph = d.ph; a.NL = sc.NL; a.wpu = sc.wpu;
    a.gram = d.gram; a.gram2 = d.gram2; a.gramF = d.gramF; a.grp_cnt = d.grp_cnt;
    return c->ops->sub1(a, sc.groups, sc.ctas, c->st);
}

// Coefficient set of a factor A (N x r, real):  kind = 1: C coefficients (weights v_i, + rho_tilde);  2: D coefficients
// (weights E_i).  Three read-only passes, one per direction: the first also accumulates the real-space weighted Gram
// (M1 = C1 or D1, colsum), each leaves the 1D Parseval sums of its derivative coefficient in c->partialP[d] for
// post(..., do_m2).  M1, its eigen-decomposition (T, lam) and colsum are final when this returns (in stream order).
void coeffs(dlr_ctx* c, const HostGrid& hg, const double* A, int kind, double* M1, double* colsum, double* T, double* lam) {
    const int R = c->R;
    DirArgs a = dirargs(c, hg);
    a.in = A; a.E = c->E; a.L = hg.Lc; a.gram = c->partial; a.pgram = c->partialP[0]; a.pgram2 = c->pgram2[0]; a.pgramF = c->pgramF[0];
    a.threads = hg.thrc;
    CK(c->ops->dir[kind == 1 ? VD_COEFF1_V : VD_COEFF1_E](a, c->st));
    c->bytes_acc += 3.0 * fac_bytes(c, hg) + (kind == 2 ? 24.0 * (double)hg.g.N : 0.0);
    // fork: M1 and its eigen-decomposition need only the Gram sums of the pass above; they run beside the two
    // remaining passes (under stream capture this becomes a parallel branch of the step graph)
    CK(cudaEventRecord(c->ev_fork, c->st));
    CK(cudaStreamWaitEvent(c->side, c->ev_fork, 0));
    k_coeff1_eig<<<3, DLR_EIG_THREADS, 0, c->side>>>(c->gramF, 1, R, kind == 1, hg.g.h3, M1, colsum, T, lam,
                                                     (kind == 1 ? c->tc_warm : c->td_warm) ? 1 : 0, c->status);
    CK(cudaGetLastError());
    (kind == 1 ? c->tc_warm : c->td_warm) = true;
    CK(cudaEventRecord(c->ev_join, c->side));
    c->count_launches -= 3;                         // the three event calls above are not kernel launches
    a.gram = nullptr; a.E = nullptr;
    a.L = hg.Lc2; a.threads = hg.thrc2;
    a.pgram = c->partialP[1]; a.pgram2 = c->pgram2[1]; a.pgramF = c->pgramF[1];
    CK(c->ops->dir[VD_COEFF2](a, c->st));
    a.pgram = c->partialP[2]; a.pgram2 = c->pgram2[2]; a.pgramF = c->pgramF[2];
    CK(c->ops->dir[VD_COEFF3](a, c->st));
    CK(cudaStreamWaitEvent(c->st, c->ev_join, 0));  // join before anything reads M1, T, lam, colsum
    c->count_launches -= 1;
}

// 1D marginals of V for the flow-free predictor L step (k_lpred_sums): one light read-only pass and a reduction.
// Called right BEFORE the C coefficients of V are computed (V changes only at the L-step QR): the two kernels go to the
// side stream, run beside the first coefficient pass, and are covered by the join at the end of coeffs() (the Jacobi
// kernel follows them on the same stream).
void marginals_V(dlr_ctx* c) {
    const HostGrid& hg = c->gv;
    const int n = hg.g.n, R = c->R;
    CK(cudaEventRecord(c->ev_mfork, c->st));
    CK(cudaStreamWaitEvent(c->side, c->ev_mfork, 0));
    c->count_launches -= 2;
    k_marginals<<<dim3(n, R), 256, 0, c->side>>>(c->V, hg.g, c->margp1, c->margp2);
    CK(cudaGetLastError());
    k_marg_reduce<<<dim3(R, 3), 256, 0, c->side>>>(c->margp1, c->margp2, hg.g, c->marg);
    CK(cudaGetLastError());
    c->bytes_acc += fac_bytes(c, hg);
}

// Column sums of the predictor's L1 (all that line 2 of Algorithm 2 needs of it) from the marginals of V and the tables
// of the L-flow that post() has just built.
void lpred_sums(dlr_ctx* c, double t3) {
    LpredArgs a;
    a.m = c->marg; a.tb = c->ft.p; a.g = c->gv.g; a.t3 = t3; a.zsum = c->zsum;
    CK(c->ops->lpred(a, c->st));
}

// The r x r work between two streaming phases, one launch (see k_post).
struct PostM2 { const HostGrid* hg; double* M2; };
struct PostS { double* S; double t; double sign; };      // sign: +1 eq. (10) as printed, -1 the forward Galerkin S step
struct PostTab { const HostGrid* hg; const double *T, *lam, *Sin; int transS; double sgn, tsub, t3; const double* M2c; double nlsign; };
void post(dlr_ctx* c, const PostM2* m2, const PostS* sf, const PostTab* tb) {
    PostArgs a;
    memset(&a, 0, sizeof(a));
    a.R = c->R;
    if (m2) {
        a.do_m2 = 1;
        for (int d = 0; d < 3; d++) a.pgram[d] = c->pgramF[d];             // the totals of the three coefficient passes
        a.m2scale = m2->hg->g.h3 / (double)m2->hg->g.n; a.M2 = m2->M2;     // 1D Parseval: sum_x u dv = (1/n) sum_k ...
    }
    a.ssign = 1.0;
    if (sf) { a.do_s = 1; a.S = sf->S; a.ts = sf->t; a.ssign = sf->sign; a.C1 = c->C1; a.C2 = c->C2; a.D1 = c->D1; a.D2 = c->D2; }
    if (tb) {
        a.do_tab = 1; a.Tm = tb->T; a.lam = tb->lam; a.Sin = tb->Sin; a.transS = tb->transS; a.g = tb->hg->g;
        a.sgn = tb->sgn; a.tsub = tb->tsub; a.t3 = tb->t3; a.M2c = tb->M2c; a.nlsign = tb->nlsign; a.o = c->ft.p;
    }
    CK(c->ops->post(a, c->st));
}

// Electric field from rho = A * p (p holds the minus sign and the quadrature weight): eqs. (12)/(13) + Poisson
// (PAPER.md:180-190):  r2c -> FFT2 -> FFT3, E_hat = -i kt phi_hat, back -> E (3 x N_x real).
// p = scale * S vec (S != nullptr; vec has element stride vstride) or scale * vec is formed inside the first pass.
void field(dlr_ctx* c, const double* A, const double* S, const double* vec, int vstride, double scale, double* Eout = nullptr) {
    if (Eout == nullptr) Eout = c->E;
    const HostGrid& hg = c->gx;
    D1Args a = d1args(c, hg);
    a.in_real = A; a.out_cplx = c->Eh; a.rho_S = S; a.rho_vec = vec; a.rho_stride = vstride; a.rho_scale = scale;
    CK(c->ops->d1[V1_RHO](a, c->st));
    c->bytes_acc += fac_bytes(c, hg) + 24.0 * (double)hg.g.N;      // read the basis, write E (spectra stay in L2)
    run_d2(c, hg, c->Eh, 1, false);
    D3Args b = d3args(c, hg);
    b.in = c->Eh; b.out = c->Eh; b.T = hg.T3s;
    CK((launch_d3<1, 3, D3_POISSON, false>(b, c->st)));
    run_d2(c, hg, c->Eh, 3, true);
    D1Args e = d1args(c, hg);
    e.T = hg.T1s; e.in_cplx = c->Eh; e.out_real = Eout;
    CK((launch_d1<3, 3, D1_IN_CPLX, D1_OP_NONE, D1_GRAM_NONE, D1_OUT_REAL>(e, c->st)));
}

// The same solve as a side branch: sub-flows 1 and 2 of the K step that follows do not read E, so the five small
// kernels of the Poisson solve run beside them; field_join() is called before the first pass that needs E.
void field_fork(dlr_ctx* c, const double* A, const double* S, const double* vec, int vstride, double scale) {
    CK(cudaEventRecord(c->ev_ffork, c->st));
    CK(cudaStreamWaitEvent(c->side, c->ev_ffork, 0));
    cudaStream_t main_st = c->st;
    c->st = c->side;
    field(c, A, S, vec, vstride, scale);
    c->st = main_st;
    CK(cudaEventRecord(c->ev_fjoin, c->side));
    c->count_launches -= 3;
    c->field_pending = true;
}
void field_join(dlr_ctx* c) {
    if (!c->field_pending) return;
    CK(cudaStreamWaitEvent(c->st, c->ev_fjoin, 0));
    c->count_launches -= 1;
    c->field_pending = false;
}

void setup_apply(dlr_ctx* c, const HostGrid& hg, ApplyCfg& ac) {
    // A*Mat pass of the QR (pass_apply.cuh): chunks of 512 points (4 KB per column and bulk copy) and as many stages as fit
    // into ~190 KB, at least two.  Measured: 64^3, r = 10: 512 x 4 stages 20.5 us per pass, 256 x 8: 22, 128 x 8: 35 (per-chunk
    // barrier and copy issue), 1024 x 2: 21.5; HBM-resident shapes want the larger copies even with few stages:
    // 128^3, r = 15: 512 x 3 stages 113 us against 167 for 256 x 6; 256^3, r = 20: 512 x 2 stages -20 % against 256 x 4
    const int R = c->R;
    ac.C = hg.g.N % 512 == 0 ? 512 : 256;
    { const int v = tune("apc", 0); if (v >= 64 && v % 64 == 0 && hg.g.N % v == 0) ac.C = v; }
    const size_t stage = (size_t)R * apply_cs(ac.C) * 8;
    ac.S = (int)std::max<size_t>(2, std::min<size_t>(8, (190 * 1024) / stage));
    { const int v = tune("aps", 0); if (v >= 2 && v <= 8) ac.S = v; }
    while (ac.S > 2 && apply_smem_bytes(R, ac.C, ac.S) > SMEM_MAX - 1024) ac.S--;
    ac.ctas = (int)std::min<long long>(c->nsm, hg.g.N / ac.C);
}

// shifted CholeskyQR3 of KL (N x r) -> orthonormal basis (h^3 B^T B = I) into `basis`, coupling matrix into Sout
// (transS: S = R^T for the L step, Fig. 1 line 40 transpose_inplace).
// The total of the Gram sums of KL must already be in c->gramF (written by the last pass of the flow).  Three A*Mat
// passes (bulk-copy pipeline, pass_apply.cuh); the r x r factorisation of each stage happens in the prologue of its own pass (chol_warp.cuh).  Stage 1
// decides on the device whether the third is needed (only while kappa(K) >~ 1e7, i.e. the first few steps): if not it
// writes the basis itself and the stage-2 launch returns at once.
void qr(dlr_ctx* c, const HostGrid& hg, double* basis, double* Sout, int transS) {
    const int R = c->R;
    const ApplyCfg& ac = (&hg == &c->gx) ? c->apx : c->apv;
    double* src[3] = {c->KL, c->Q1, c->KL};
    double* dst[3] = {c->Q1, c->KL, basis};
    for (int stage = 0; stage < 3; stage++) {
        ApplyArgs a;
        memset(&a, 0, sizeof(a));
        a.N = hg.g.N; a.in = src[stage]; a.out = dst[stage]; a.out_alt = basis;
        a.partial = c->partial; a.partial2 = c->gram2; a.partialF = c->gramF; a.grp_cnt = c->grp_cnt;
        a.C = ac.C; a.S = ac.S;
        a.ch.gsum = c->gramF; a.ch.stage = stage; a.ch.transS = transS;
        a.ch.shift = 64.0 * R * 2.220446049250313e-16;
        a.ch.out_scale = 1.0 / sqrt(hg.g.h3); a.ch.s_scale = sqrt(hg.g.h3);
        a.ch.Rtot = c->Rtot; a.ch.Sout = Sout; a.ch.status = c->status; a.ch.qrflag = c->status + 1;
        if (stage < 2) c->bytes_acc += 2.0 * fac_bytes(c, hg);     // the third stage is skipped in steady state: not counted
        CK(c->ops->apply[stage < 2 ? 0 : 1](a, ac.ctas, c->st));
    }
}

// K- or L-flow of section 4 of the factor `src` (X or V; the product with the coupling matrix is
// folded into the first column-mixing matrix).  order 1: Lie + exponential Euler = 3 directional passes;
// order 2: Strang + ETD2RK = 5 passes (1, 2, 3, 2, 1).  Result: real factor in c->KL with its Gram sums in c->partial,
// or (zero_only) only the column sums of the result (without the h^3 weight) in c->zsum.
void flow(dlr_ctx* c, const HostGrid& hg, const double* src, bool is_L, int order, bool zero_only) {
    const RankOps* ops = c->ops;
    const int RR = c->R * c->R;
    const double* mats = c->ft.p.mats;
    DirArgs a = dirargs(c, hg);
    a.store = 1; a.L = hg.Lx;
    // sub-flow 1:  A <- src (Sin T1), phases, then into the eigenbasis of direction 2
    a.in = src; a.out = c->W; a.min_ = mats + 0 * RR; a.mout = mats + 1 * RR; a.ph = c->ft.p.ph1;
    CK(run_sub1(c, hg, a));
    c->bytes_acc += (order == 1 ? (zero_only ? 5.0 : 6.0) : 10.0) * fac_bytes(c, hg) + (is_L ? 0.0 : 24.0 * (double)hg.g.N);
    // sub-flow 2
    a.in = c->W; a.min_ = nullptr; a.mout = nullptr; a.ph = c->ft.p.ph2;
    CK(run_sub2(c, hg, c->W, c->W, c->ft.p.ph2));
    // sub-flow 3 in the eigenbasis of direction 3 (the first pass of a K flow that reads the electric field)
    field_join(c);
    DirArgs e = dirargs(c, hg);
    e.threads = hg.thre; e.L = hg.Le; e.in = c->W; e.E = c->E; e.min_ = mats + 2 * RR; e.Q = c->ft.p.Q;
    e.ez = c->ft.p.ez; e.f1 = c->ft.p.f1; e.f2a = c->ft.p.f2a; e.f2b = c->ft.p.f2b;
    if (order == 1) {
        e.mout = mats + 3 * RR;                      // T3^T: back to the original basis
        if (zero_only) { e.store = 0; e.colsum = c->partialC; }
        else { e.store = 1; e.out = c->KL; e.gram = c->partial; }
        CK(ops->dir[is_L ? VD_ETD1_V : VD_ETD1_E](e, c->st));
        if (zero_only) {
            k_colsum_reduce<<<1, DLR_SMALL_THREADS, 0, c->st>>>(c->colsumF, 1, c->R, c->zsum);
            CK(cudaGetLastError());
        }
        return;
    }
    e.mout = mats + 5 * RR; e.store = 1; e.out = c->W;          // T3^T T2
    CK(ops->dir[is_L ? VD_ETD2_V : VD_ETD2_E](e, c->st));
    CK(run_sub2(c, hg, c->W, c->W, c->ft.p.ph2));                // sub-flow 2, second half
    a.out = c->KL; a.min_ = mats + 6 * RR; a.mout = mats + 7 * RR; a.ph = c->ft.p.ph1; a.gram = c->partial;
    CK(run_sub1(c, hg, a));                                      // sub-flow 1, second half, + Gram of the result
}

// One step of the unconventional integrator (DLR_FLAG_UNCONVENTIONAL; oracle.step_bug, the paper's reference [4] named in
// PAPER.md:29, 288).  Reuses the Lie flows, the QR and the coefficient passes of Algorithm 1; new: the cross-Gram passes
// M = <X1, X0>, N = <V1, V0> and the forward S step.  X1 goes to c->X1, V1 to c->W, and both are copied over X, V once
// the old bases are no longer needed.
void issue_step_bug(dlr_ctx* c, double tau) {
    const HostGrid &gx = c->gx, &gv = c->gv;
    const int R = c->R;
    phase_mark(c, "start");
    c->bytes_acc = 0.0;
    if (!c->vh_valid) {
        coeffs(c, gv, c->V, 1, c->C1, c->rho_t, c->TC, c->lamC);
        const PostM2 m2C{&gv, c->C2};
        post(c, &m2C, nullptr, nullptr);
    }
    phase_mark(c, "C coefficients (V0)");
    field_fork(c, c->X, c->S, c->rho_t, 1, -1.0);                  // E0, eq. (12)
    // K step from (X0, S0) -> X1 (the triangular factor is not used)
    {
        const PostTab tb{&gx, c->TC, c->lamC, c->S, 0, -1.0, tau, tau, c->C2, 1.0};
        post(c, nullptr, nullptr, &tb);
    }
    flow(c, gx, c->X, false, 1, false);
    qr(c, gx, c->X1, c->Sp, 0);
    phase_mark(c, "K step + QR");
    const int cx = (int)std::min<long long>(DLR_CROSS_CTAS, gx.g.N / 1024), cv = (int)std::min<long long>(DLR_CROSS_CTAS, gv.g.N / 1024);
    const int ncx = std::max(1, cx), ncv = std::max(1, cv);
    CK(c->ops->cross(c->X1, c->X, gx.g.N, c->crossM, ncx, c->st));
    c->bytes_acc += 2.0 * fac_bytes(c, gx);
    // L step from (V0, S0) with the coefficients of the OLD basis X0 -> V1
    coeffs(c, gx, c->X, 2, c->D1, nullptr, c->TD, c->lamD);
    {
        const PostM2 m2D{&gx, c->D2};
        const PostTab tb{&gv, c->TD, c->lamD, c->S, 1, +1.0, tau, tau, c->D2, -1.0};
        post(c, &m2D, nullptr, &tb);
    }
    flow(c, gv, c->V, true, 1, false);
    qr(c, gv, c->W, c->Sp, 1);
    phase_mark(c, "L step + QR");
    CK(c->ops->cross(c->W, c->V, gv.g.N, c->crossN, ncv, c->st));
    c->bytes_acc += 2.0 * fac_bytes(c, gv);
    CK(c->ops->bug_s0(c->crossM, ncx, c->crossN, ncv, gx.g.h3, gv.g.h3, c->S, c->st));     // S~ = M S0 N^T
    // the new bases replace the old ones
    CK(cudaMemcpyAsync(c->X, c->X1, (size_t)gx.g.N * R * sizeof(double), cudaMemcpyDeviceToDevice, c->st));
    CK(cudaMemcpyAsync(c->V, c->W, (size_t)gv.g.N * R * sizeof(double), cudaMemcpyDeviceToDevice, c->st));
    c->bytes_acc += 2.0 * fac_bytes(c, gx) + 2.0 * fac_bytes(c, gv);
    // Galerkin S step forward in time with the coefficients of X1, V1 (E0 still in c->E)
    coeffs(c, gv, c->V, 1, c->C1, c->rho_t, c->TC, c->lamC);
    {
        const PostM2 m2C{&gv, c->C2};
        post(c, &m2C, nullptr, nullptr);
    }
    coeffs(c, gx, c->X, 2, c->D1, nullptr, c->TD, c->lamD);
    {
        const PostM2 m2D{&gx, c->D2};
        const PostS sf{c->S, tau, -1.0};
        post(c, &m2D, &sf, nullptr);
    }
    phase_mark(c, "S step (Galerkin)");
    c->vh_valid = true;                                   // C(V1) are the next step's coefficients
    c->bytes_step = c->bytes_acc;
}

// one step, issued on c->st (directly or under stream capture)
void issue_step(dlr_ctx* c, double tau) {
    if (c->cfg.flags & DLR_FLAG_UNCONVENTIONAL) { issue_step_bug(c, tau); return; }
    const int order = c->cfg.order;
    const double tp = order == 2 ? 0.5 * tau : tau;     // step size of the Algorithm-1 part
    const HostGrid &gx = c->gx, &gv = c->gv;
    double* Sp = order == 2 ? c->Sp : c->S;             // the predictor of Algorithm 2 works on a scratch S
    const PostM2 m2C{&gv, c->C2}, m2D{&gx, c->D2};
    phase_mark(c, "start");
    c->bytes_acc = 0.0;
    // ---- Algorithm 1, line 1: C coefficients from V0 (kept from the previous step's line 10 when valid)
    if (!c->vh_valid) {
        marginals_V(c);
        coeffs(c, gv, c->V, 1, c->C1, c->rho_t, c->TC, c->lamC);
        post(c, &m2C, nullptr, nullptr);
    }
    phase_mark(c, "C coefficients (V0)");
    // ---- line 2: K0 = X0 S0 is never formed (the product with S0 is folded into the flow).  In Algorithm 2 the
    //      predictor basis X1 goes to its own buffer: the corrector's first K step starts from X0 again.
    double* Xp = order == 2 ? c->X1 : c->X;
    // ---- line 3: E0 from K0 and V0, eq. (12): rho = -X0 (S0 rho_tilde)
    field_fork(c, c->X, c->S, c->rho_t, 1, -1.0);
    phase_mark(c, "electric field E0");
    // ---- line 4: K step (Lie, exponential Euler) of length tp with E0;  line 5: QR -> X1, S1
    {
        const PostTab tb{&gx, c->TC, c->lamC, c->S, 0, -1.0, tp, tp, c->C2, 1.0};
        post(c, nullptr, nullptr, &tb);
    }
    flow(c, gx, c->X, false, 1, false);
    phase_mark(c, "K step (predictor)");
    qr(c, gx, Xp, Sp, 0);
    phase_mark(c, "QR K (predictor)");
    // ---- line 6: D coefficients from X1 and E0;  line 7: S step;  lines 8-9: L0 = V0 S2^T, tables of the L step
    coeffs(c, gx, Xp, 2, c->D1, nullptr, c->TD, c->lamD);
    phase_mark(c, "D coefficients (predictor)");
    {
        const PostS sf{Sp, tp, 1.0};
        const PostTab tb{&gv, c->TD, c->lamD, Sp, 1, +1.0, tp, tp, c->D2, -1.0};
        post(c, &m2D, &sf, &tb);
    }
    phase_mark(c, "S step (predictor)");
    if (order == 1) {
        flow(c, gv, c->V, true, 1, false);
        phase_mark(c, "L step");
        qr(c, gv, c->V, c->S, 1);                 // line 10: V1, S3 = R^T
        phase_mark(c, "QR L");
        c->vh_valid = false;
        c->bytes_step = c->bytes_acc;
        return;
    }
    // only rho(L1) = L1^T omega_v is needed (eq. (13)): no flow, see k_lpred_sums.  DLR_FLAG_PREDICTOR_L_FLOW runs the
    // Lie flow of Algorithm 1 line 9 literally instead (A/B check of the marginal-based shortcut)
    if (c->cfg.flags & DLR_FLAG_PREDICTOR_L_FLOW) flow(c, gv, c->V, true, 1, true);
    else lpred_sums(c, tp);
    phase_mark(c, "L step (predictor)");
    // ---- Algorithm 2, line 2: E^{1/2} from X1 and L1, eq. (13)
    field_fork(c, Xp, nullptr, c->zsum, 1, -gv.g.h3);
    phase_mark(c, "electric field E1/2");
    // ---- line 3: K step (Strang, ETD2RK) of length tau/2 from K0 = X0 S0 with E^{1/2};  line 4: QR -> X2, S3
    {
        const PostTab tb{&gx, c->TC, c->lamC, c->S, 0, -1.0, 0.25 * tau, 0.5 * tau, c->C2, 1.0};
        post(c, nullptr, nullptr, &tb);
    }
    flow(c, gx, c->X, false, 2, false);
    phase_mark(c, "first K step");
    qr(c, gx, c->X, c->S, 0);
    phase_mark(c, "QR K (first)");
    // ---- line 5: D coefficients from X2 and E^{1/2};  line 6: S step;  tables of the L step (L = V0 S4^T)
    coeffs(c, gx, c->X, 2, c->D1, nullptr, c->TD, c->lamD);
    phase_mark(c, "D coefficients");
    {
        const PostS sf{c->S, 0.5 * tau, 1.0};
        const PostTab tb{&gv, c->TD, c->lamD, c->S, 1, +1.0, 0.5 * tau, tau, c->D2, -1.0};
        post(c, &m2D, &sf, &tb);
    }
    phase_mark(c, "first S step");
    // ---- lines 7-9: L step (Strang) of length tau, QR -> V1, S5 = R^T
    flow(c, gv, c->V, true, 2, false);
    phase_mark(c, "L step");
    qr(c, gv, c->V, c->S, 1);
    phase_mark(c, "QR L");
    // ---- line 10: C coefficients from V1 (they are also the next step's line-1 coefficients);  line 11: S step;
    //      tables of the second K step (K3 = X2 S6)
    marginals_V(c);
    coeffs(c, gv, c->V, 1, c->C1, c->rho_t, c->TC, c->lamC);
    phase_mark(c, "C coefficients");
    {
        const PostS sf{c->S, 0.5 * tau, 1.0};
        const PostTab tb{&gx, c->TC, c->lamC, c->S, 0, -1.0, 0.25 * tau, 0.5 * tau, c->C2, 1.0};
        post(c, &m2C, &sf, &tb);
    }
    phase_mark(c, "second S step");
    // ---- lines 12-14: K step (Strang) of length tau/2, QR -> X3, S7
    flow(c, gx, c->X, false, 2, false);
    phase_mark(c, "second K step");
    qr(c, gx, c->X, c->S, 0);
    phase_mark(c, "QR K (second)");
    c->vh_valid = true;
    c->bytes_step = c->bytes_acc;
}

int fail(dlr_ctx* c, cudaError_t e, const char* what) {
    if (c && c->last_err == cudaSuccess) {
        c->last_err = e;
        c->last_err_msg = std::string(what) + ": " + cudaGetErrorString(e);
    }
    return DLR_ERR_CUDA;
}

}  // namespace

// =========================================================================================================
extern "C" {

const char* dlr_strerror(int code) {
    switch (code) {
        case DLR_OK: return "ok";
        case DLR_ERR_INVALID: return "invalid argument";
        case DLR_ERR_UNSUPPORTED: return "unsupported grid size or rank";
        case DLR_ERR_WORKSPACE: return "workspace too small or misaligned";
        case DLR_ERR_CUDA: return "CUDA error";
        case DLR_ERR_NOT_ORTHONORMAL: return "initial factors are not orthonormal";
        case DLR_ERR_NO_STATE: return "no state set";
        case DLR_ERR_TOO_LARGE: return "size exceeds the static device scratch (DLR_NOALLOC_MAX_PROBES)";
        default: return "unknown error";
    }
}

const char* dlr_last_cuda_error(dlr_ctx* c) { return c ? c->last_err_msg.c_str() : ""; }

int dlr_clear_error(dlr_ctx* c) {
    if (!c) return DLR_ERR_INVALID;
    DevGuard guard(c->dev);
    cudaGetLastError();                        // drop a non-sticky runtime error, if any
    c->last_err = cudaSuccess;
    c->last_err_msg.clear();
    c->field_pending = false;
    if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }      // a failed capture may have left it stale
    c->has_state = false;                      // the state may be half-updated: dlr_set_initial must follow
    c->vh_valid = false;
    return DLR_OK;
}

// shared-memory opt-in of every kernel this context may launch, on the current (= the context's) device
static cudaError_t configure_kernels(dlr_ctx* c) {
    cudaError_t e = c->ops->configure();
#define OPTIN(...) if (e == cudaSuccess) e = dlr_optin_smem(__VA_ARGS__)
    OPTIN(k_d2<true>);
    OPTIN(k_d2<false>);
    OPTIN(k_d3<1, 3, D3_POISSON, false>);
    OPTIN(k_d3<3, 3, D3_FWD_STORE, false>);
    OPTIN(k_d3<3, 3, D3_INV_ONLY, false>);
    OPTIN(k_d1<3, 3, D1_IN_CPLX, D1_OP_NONE, D1_GRAM_NONE, D1_OUT_REAL>);
    OPTIN(k_d1<3, 3, D1_IN_REAL, D1_OP_NONE, D1_GRAM_NONE, D1_OUT_CPLX>);
    if (e == cudaSuccess) e = configure_sub2();
#undef OPTIN
    return e;
}

static void init_grids(dlr_ctx* c) {
    setup_grid(c->gx, c->cfg.n_x[0], c->cfg.x_lo[0], c->cfg.x_hi[0], c->R);
    setup_grid(c->gv, c->cfg.n_v[0], c->cfg.v_lo[0], c->cfg.v_hi[0], c->R);
}

int dlr_workspace_bytes(const dlr_config* cfg, size_t* bytes) {
    if (!bytes) return DLR_ERR_INVALID;
    int rc = check_cfg(cfg);
    if (rc != DLR_OK) return rc;
    dlr_ctx tmp{};
    tmp.cfg = *cfg; tmp.R = cfg->rank;
    init_grids(&tmp);
    *bytes = carve(&tmp, nullptr);
    return DLR_OK;
}

int dlr_create(const dlr_config* cfg, void* d_workspace, size_t bytes, void* cuda_stream, dlr_ctx** out) {
    if (!out || !d_workspace) return DLR_ERR_INVALID;
    int rc = check_cfg(cfg);
    if (rc != DLR_OK) return rc;
    if (((uintptr_t)d_workspace & 255) != 0) return DLR_ERR_WORKSPACE;
    dlr_ctx* c = new dlr_ctx{};
    c->cfg = *cfg; c->R = cfg->rank; c->st = (cudaStream_t)cuda_stream; c->ops = dlr_rank_ops(cfg->rank);
    c->last_err = cudaSuccess;
    init_grids(c);
    const size_t need = carve(c, (char*)d_workspace);
    if (need > bytes) { delete c; return DLR_ERR_WORKSPACE; }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) { delete c; return DLR_ERR_CUDA; }
    // the context lives on the device that owns the workspace, whatever the caller's current device is
    cudaPointerAttributes pa;
    e = cudaPointerGetAttributes(&pa, d_workspace);
    if (e != cudaSuccess || pa.type != cudaMemoryTypeDevice) { cudaGetLastError(); delete c; return DLR_ERR_WORKSPACE; }
    c->dev = pa.device;
    DevGuard guard(c->dev);
    if (cudaDeviceGetAttribute(&c->nsm, cudaDevAttrMultiProcessorCount, c->dev) != cudaSuccess || c->nsm < 1) c->nsm = 148;
    e = configure_kernels(c);
    if (e != cudaSuccess) { delete c; return DLR_ERR_CUDA; }
    setup_sub2(c, c->gx, c->s2x);
    setup_sub2(c, c->gv, c->s2v);
    setup_apply(c, c->gx, c->apx);
    setup_apply(c, c->gv, c->apv);
    setup_sub1(c, c->gx, c->s1x);
    setup_sub1(c, c->gv, c->s1v);
    e = cudaStreamCreateWithFlags(&c->cap_st, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_mfork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_ffork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_fjoin, cudaEventDisableTiming);
    if (e != cudaSuccess) { dlr_destroy(c); return DLR_ERR_CUDA; }
    e = upload_tables(c, c->gx, cfg->x_lo[0], cfg->x_hi[0]);
    if (e == cudaSuccess) e = upload_tables(c, c->gv, cfg->v_lo[0], cfg->v_hi[0]);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->status, 0, 4 * sizeof(int), c->st);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->grp_cnt, 0, 3 * DLR_CNT_STRIDE * sizeof(unsigned), c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    if (e != cudaSuccess) { dlr_destroy(c); return DLR_ERR_CUDA; }      // releases the streams and events created above
    *out = c;
    return DLR_OK;
}

void dlr_destroy(dlr_ctx* c) {
    if (!c) return;
    DevGuard guard(c->dev);
    if (c->graph) cudaGraphExecDestroy(c->graph);
    if (c->cap_st) cudaStreamDestroy(c->cap_st);
    if (c->side) cudaStreamDestroy(c->side);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->ev_mfork) cudaEventDestroy(c->ev_mfork);
    if (c->ev_ffork) cudaEventDestroy(c->ev_ffork);
    if (c->ev_fjoin) cudaEventDestroy(c->ev_fjoin);
    for (auto& p : c->phases) cudaEventDestroy(p.ev);
    delete c;
}

static int gram_check(dlr_ctx* c, const HostGrid& hg, const double* A) {
    const int R = c->R, P = R * (R + 1) / 2;
    D1Args a = d1args(c, hg);
    a.in_real = A; a.partial = c->partial;
    CK(c->ops->d1[V1_GRAM_ONLY](a, c->st));
    reduce_partials(c, d1_blocks(hg), P, c->partial2a);
    std::vector<double> h((size_t)DLR_G1 * P);
    cudaError_t e = cudaMemcpyAsync(h.data(), c->partial2a, h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    if (e != cudaSuccess) return fail(c, e, "gram_check");
    if (c->last_err != cudaSuccess) return DLR_ERR_CUDA;
    int idx = 0;
    for (int a1 = 0; a1 < R; a1++)
        for (int b = a1; b < R; b++, idx++) {
            double s = 0.0;
            for (int g = 0; g < DLR_G1; g++) s += h[(size_t)g * P + idx];
            if (!(fabs(s * hg.g.h3 - (a1 == b ? 1.0 : 0.0)) <= 1e-10)) return DLR_ERR_NOT_ORTHONORMAL;
        }
    return DLR_OK;
}

int dlr_set_initial(dlr_ctx* c, const double* X, const double* S, const double* V, int on_device) {
    if (!c || !X || !S || !V) return DLR_ERR_INVALID;
    DevGuard guard(c->dev);
    const cudaMemcpyKind k = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    const int R = c->R;
    cudaError_t e = cudaMemcpyAsync(c->X, X, (size_t)c->gx.g.N * R * sizeof(double), k, c->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->V, V, (size_t)c->gv.g.N * R * sizeof(double), k, c->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->S, S, (size_t)R * R * sizeof(double), k, c->st);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->status, 0, 4 * sizeof(int), c->st);
    if (e != cudaSuccess) return fail(c, e, "dlr_set_initial copy");
    c->vh_valid = false;
    c->has_state = false;
    c->tc_warm = c->td_warm = false;
    int rc = gram_check(c, c->gx, c->X);
    if (rc == DLR_OK) rc = gram_check(c, c->gv, c->V);
    if (rc != DLR_OK) return rc;
    c->has_state = true;
    return DLR_OK;
}

int dlr_step(dlr_ctx* c, double tau) {
    if (!c) return DLR_ERR_INVALID;
    DevGuard guard(c->dev);
    if (!c->has_state) return DLR_ERR_NO_STATE;
    if (c->last_err != cudaSuccess) return DLR_ERR_CUDA;
    PdlScope pdl(c->profiling ? 0 : c->pdl);      // profiling records events between the launches: plain launches
    if (c->profiling || !c->vh_valid) {
        // first step after set_initial (it also computes the C coefficients of V0) or profiling: direct launches
        for (auto& p : c->phases) cudaEventDestroy(p.ev);
        c->phases.clear();
        c->count_launches = 0;
        issue_step(c, tau);
        return c->last_err == cudaSuccess ? DLR_OK : DLR_ERR_CUDA;
    }
    if (!c->graph || c->graph_tau != tau) {
        if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }
        // warm every kernel's attributes outside capture is unnecessary: they were all launched by the first step
        cudaGraph_t g;
        // capture on a private stream (the caller's may be the legacy default stream, which cannot capture);
        // the instantiated graph is then launched on the caller's stream
        cudaStream_t user = c->st;
        cudaError_t e = cudaStreamBeginCapture(c->cap_st, cudaStreamCaptureModeThreadLocal);
        if (e != cudaSuccess) return fail(c, e, "begin capture");
        c->count_launches = 0;
        c->st = c->cap_st;
        issue_step(c, tau);
        c->st = user;
        e = cudaStreamEndCapture(c->cap_st, &g);
        if (e != cudaSuccess) return fail(c, e, "end capture");
        if (c->last_err != cudaSuccess) { cudaGraphDestroy(g); return DLR_ERR_CUDA; }
        c->launches = c->count_launches;
        e = cudaGraphInstantiate(&c->graph, g, 0);
        cudaGraphDestroy(g);
        if (e != cudaSuccess) return fail(c, e, "graph instantiate");
        c->graph_tau = tau;
    }
    cudaError_t e = cudaGraphLaunch(c->graph, c->st);
    if (e != cudaSuccess) return fail(c, e, "graph launch");
    return DLR_OK;
}

int dlr_run(dlr_ctx* c, double tau, int nsteps) {
    for (int i = 0; i < nsteps; i++) {
        int rc = dlr_step(c, tau);
        if (rc != DLR_OK) return rc;
    }
    return DLR_OK;
}

int dlr_launches_per_step(dlr_ctx* c) { return c ? (c->launches ? c->launches : c->count_launches) : 0; }

double dlr_bytes_per_step(dlr_ctx* c) {
    // algorithmic bytes of the factor-sized passes one step issues: every read or write of an
    // N x r factor counts 8 N r, the field 8 N per component; r x r work and L2-resident single-column spectra are not
    // counted.  Valid after the first dlr_step.
    return c ? c->bytes_step : 0.0;
}

int dlr_set_profiling(dlr_ctx* c, int on) {
    if (!c) return DLR_ERR_INVALID;
    c->profiling = on != 0;
    c->prof_level = on;
    return DLR_OK;
}

int dlr_get_phase_times(dlr_ctx* c, int cap, float* ms, const char** names) {
    if (!c) return 0;
    DevGuard guard(c->dev);
    cudaStreamSynchronize(c->st);
    int n = 0;
    for (size_t i = 1; i < c->phases.size() && n < cap; i++, n++) {
        float t = 0.f;
        cudaEventElapsedTime(&t, c->phases[i - 1].ev, c->phases[i].ev);
        if (ms) ms[n] = t;
        if (names) names[n] = c->phases[i].name;
    }
    return n;
}

int dlr_moments(dlr_ctx* c, dlr_moments_t* out, int n_probe, const int64_t* probe_ix, const int64_t* probe_iv,
                double* f_probe) {
    if (!c || !out) return DLR_ERR_INVALID;
    DevGuard guard(c->dev);
    if (!c->has_state) return DLR_ERR_NO_STATE;
    if (n_probe < 0 || n_probe > c->probe_cap || (n_probe > 0 && (!probe_ix || !probe_iv || !f_probe))) return DLR_ERR_INVALID;
    const int R = c->R;
    k_colmoments<<<dim3(R, DLR_MCH), 256, 0, c->st>>>(c->X, c->gx.g, c->mxp);
    CK(cudaGetLastError());
    k_colmoments<<<dim3(R, DLR_MCH), 256, 0, c->st>>>(c->V, c->gv.g, c->mvp);
    CK(cudaGetLastError());
    k_colmoments_sum<<<1, 256, 0, c->st>>>(c->mxp, c->mvp, R, c->mx, c->mv);
    CK(cudaGetLastError());
    // electric energy: E from eq. (12) on the current factors.  rho_tilde = h_v^3 V^T 1 = h_v^3 * mv[:,0]
    // (into the diagnostics' own field buffer: dlr_get_field keeps returning the field dlr_step used last)
    field(c, c->X, c->S, c->mv, 5, -c->gv.g.h3, c->Em);
    k_sumsq<<<DLR_ECH, 256, 0, c->st>>>(c->Em, 3 * c->gx.g.N, c->esum);
    CK(cudaGetLastError());
    k_moments_final<<<1, 32, 0, c->st>>>(c->mx, c->mv, c->S, R, c->gx.g.h3, c->gv.g.h3, c->esum, c->mres);
    CK(cudaGetLastError());
    if (n_probe > 0) {
        cudaError_t e = cudaMemcpyAsync(c->pix, probe_ix, n_probe * sizeof(int64_t), cudaMemcpyHostToDevice, c->st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(c->piv, probe_iv, n_probe * sizeof(int64_t), cudaMemcpyHostToDevice, c->st);
        if (e != cudaSuccess) return fail(c, e, "probe upload");
        k_probes<<<(n_probe + 127) / 128, 128, 0, c->st>>>(c->X, c->S, c->V, c->gx.g.N, c->gv.g.N, R, n_probe, c->pix, c->piv, c->pf);
        CK(cudaGetLastError());
    }
    double res[8];
    int st[4];
    cudaError_t e = cudaMemcpyAsync(res, c->mres, 8 * sizeof(double), cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(st, c->status, 4 * sizeof(int), cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess && n_probe > 0) e = cudaMemcpyAsync(f_probe, c->pf, n_probe * sizeof(double), cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    if (e != cudaSuccess) return fail(c, e, "dlr_moments");
    if (c->last_err != cudaSuccess) return DLR_ERR_CUDA;
    out->mass = res[0];
    out->momentum[0] = res[1]; out->momentum[1] = res[2]; out->momentum[2] = res[3];
    out->kinetic_energy = res[4];
    out->s_fro = res[5];
    out->nonfinite = res[6] != 0.0;
    out->electric_energy = 0.5 * c->gx.g.h3 * res[7];
    out->qr_fallbacks = st[0];
    out->qr_third_stage = st[2];
    out->eig_unconverged = st[3];
    return DLR_OK;
}

int dlr_get_factors(dlr_ctx* c, double* X, double* S, double* V, int on_device) {
    if (!c) return DLR_ERR_INVALID;
    DevGuard guard(c->dev);
    if (!c->has_state) return DLR_ERR_NO_STATE;
    const cudaMemcpyKind k = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    const int R = c->R;
    cudaError_t e = cudaSuccess;
    if (X) e = cudaMemcpyAsync(X, c->X, (size_t)c->gx.g.N * R * sizeof(double), k, c->st);
    if (e == cudaSuccess && V) e = cudaMemcpyAsync(V, c->V, (size_t)c->gv.g.N * R * sizeof(double), k, c->st);
    if (e == cudaSuccess && S) e = cudaMemcpyAsync(S, c->S, (size_t)R * R * sizeof(double), k, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    if (e != cudaSuccess) return fail(c, e, "dlr_get_factors");
    return c->last_err == cudaSuccess ? DLR_OK : DLR_ERR_CUDA;
}

int dlr_get_field(dlr_ctx* c, double* E, int on_device) {
    if (!c || !E) return DLR_ERR_INVALID;
    DevGuard guard(c->dev);
    cudaError_t e = cudaMemcpyAsync(E, c->E, (size_t)3 * c->gx.g.N * sizeof(double),
                                    on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    return e == cudaSuccess ? DLR_OK : fail(c, e, "dlr_get_field");
}

int dlr_test_fft_roundtrip(dlr_ctx* c, int which, int ncols, const double* d_in, double* d_out, double* d_spec) {
    if (!c || !d_in || !d_out || !d_spec) return DLR_ERR_INVALID;
    DevGuard guard(c->dev);
    if (ncols != 3) return DLR_ERR_UNSUPPORTED;
    const HostGrid& hg = which ? c->gv : c->gx;
    if (hg.g.NC > c->gx.g.NC) return DLR_ERR_UNSUPPORTED;      // the scratch spectrum is sized for the x grid
    double2* spec = (double2*)d_spec;
    D1Args a = d1args(c, hg);
    a.in_real = d_in; a.out_cplx = spec; a.T = hg.T1s;
    D3Args b = d3args(c, hg);
    b.in = spec; b.out = spec; b.T = hg.T3s;
    D1Args e = d1args(c, hg);
    e.in_cplx = spec; e.out_real = d_out; e.T = hg.T1s;
    CK((launch_d1<3, 3, D1_IN_REAL, D1_OP_NONE, D1_GRAM_NONE, D1_OUT_CPLX>(a, c->st)));
    run_d2(c, hg, spec, ncols, false);
    CK((launch_d3<3, 3, D3_FWD_STORE, false>(b, c->st)));
    cudaError_t er = cudaStreamSynchronize(c->st);
    if (er != cudaSuccess) return fail(c, er, "fft forward");
    // the inverse consumes a copy so that d_spec keeps the forward transform for inspection
    double2* tmp = c->Eh;
    er = cudaMemcpyAsync(tmp, spec, (size_t)ncols * hg.g.NC * sizeof(double2), cudaMemcpyDeviceToDevice, c->st);
    if (er != cudaSuccess) return fail(c, er, "fft copy");
    b.in = tmp; b.out = tmp; e.in_cplx = tmp;
    CK((launch_d3<3, 3, D3_INV_ONLY, false>(b, c->st)));
    run_d2(c, hg, tmp, ncols, true);
    CK((launch_d1<3, 3, D1_IN_CPLX, D1_OP_NONE, D1_GRAM_NONE, D1_OUT_REAL>(e, c->st)));
    er = cudaStreamSynchronize(c->st);
    if (er != cudaSuccess) return fail(c, er, "fft inverse");
    return c->last_err == cudaSuccess ? DLR_OK : DLR_ERR_CUDA;
}

int dlr_test_chol_decide(dlr_ctx* c, const double* gram_upper, int* third_stage_needed) {
    if (!c || !gram_upper || !third_stage_needed) return DLR_ERR_INVALID;
    DevGuard guard(c->dev);
    const int R = c->R, P = R * (R + 1) / 2;
    int st_before[4], st_after[4];
    cudaError_t e = cudaMemcpyAsync(c->gram2, gram_upper, P * sizeof(double), cudaMemcpyHostToDevice, c->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(st_before, c->status, sizeof(st_before), cudaMemcpyDeviceToHost, c->st);
    if (e != cudaSuccess) return fail(c, e, "dlr_test_chol_decide");
    // stage 1 of the CholeskyQR of a factor whose once-orthogonalised Gram matrix is gram_upper (the total row)
    CholArgs ca;
    ca.gsum = c->gram2; ca.stage = 1; ca.transS = 0; ca.shift = 0.0; ca.out_scale = 1.0; ca.s_scale = 1.0;
    ca.Rtot = c->Rtot; ca.Sout = c->Sp; ca.status = c->status; ca.qrflag = c->status + 1;
    CK(c->ops->chol_test(ca, c->apply, c->st));
    e = cudaMemcpyAsync(st_after, c->status, sizeof(st_after), cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->status, st_before, sizeof(st_before), cudaMemcpyHostToDevice, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    if (e != cudaSuccess) return fail(c, e, "dlr_test_chol_decide");
    *third_stage_needed = st_after[1] ? 0 : 1;
    return c->last_err == cudaSuccess ? DLR_OK : DLR_ERR_CUDA;
}

int dlr_test_dir_pass(dlr_ctx* c, int which, int kind, const double* d_in, double* d_out, const double* min_,
                      const double* mout, const double* tabs, const double* Q, const double* d_E) {
    if (!c || !d_in || !d_out || !tabs || kind < 0 || kind > 3) return DLR_ERR_INVALID;
    if (kind >= 2 && (!Q || (which == 0 && !d_E))) return DLR_ERR_INVALID;
    DevGuard guard(c->dev);
    const HostGrid& hg = which ? c->gv : c->gx;
    const int R = c->R, RR = R * R, n = hg.g.n, lg = hg.g.log2n;
    const int ntab = kind < 2 ? 1 : 4;
    // tables arrive in natural wavenumber order [tab][k][column] (complex); the kernels index them by stored position
    std::vector<double2> t((size_t)ntab * n * R);
    const double2* src = (const double2*)tabs;
    for (int q = 0; q < ntab; q++)
        for (int e = 0; e < n; e++)
            for (int j = 0; j < R; j++) t[((size_t)q * n + e) * R + j] = src[((size_t)q * n + brev_host(e, lg)) * R + j];
    double2* dst[4] = {kind < 2 ? c->ft.p.ph1 : c->ft.p.ez, c->ft.p.f1, c->ft.p.f2a, c->ft.p.f2b};
    cudaError_t e = cudaSuccess;
    for (int q = 0; q < ntab && e == cudaSuccess; q++)
        e = cudaMemcpyAsync(dst[q], t.data() + (size_t)q * n * R, (size_t)n * R * sizeof(double2), cudaMemcpyHostToDevice, c->st);
    if (e == cudaSuccess && min_) e = cudaMemcpyAsync(c->ft.p.mats, min_, RR * sizeof(double), cudaMemcpyHostToDevice, c->st);
    if (e == cudaSuccess && mout) e = cudaMemcpyAsync(c->ft.p.mats + RR, mout, RR * sizeof(double), cudaMemcpyHostToDevice, c->st);
    if (e == cudaSuccess && Q) e = cudaMemcpyAsync(c->ft.p.Q, Q, 3 * RR * sizeof(double), cudaMemcpyHostToDevice, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);          // the staging vector goes out of scope below
    if (e != cudaSuccess) return fail(c, e, "dlr_test_dir_pass");
    DirArgs a = dirargs(c, hg);
    a.in = d_in; a.out = d_out; a.store = 1;
    a.min_ = min_ ? c->ft.p.mats : nullptr; a.mout = mout ? c->ft.p.mats + RR : nullptr;
    if (kind < 2) {
        a.L = hg.Lx; a.ph = c->ft.p.ph1;
        if (kind == 1) CK(run_sub2(c, hg, d_in, d_out, c->ft.p.ph1));
        else CK(run_sub1(c, hg, a));
    } else {
        a.threads = hg.thre; a.L = hg.Le; a.E = d_E; a.Q = c->ft.p.Q;
        a.ez = c->ft.p.ez; a.f1 = c->ft.p.f1; a.f2a = c->ft.p.f2a; a.f2b = c->ft.p.f2b;
        const int v = kind == 2 ? (which ? VD_ETD1_V : VD_ETD1_E) : (which ? VD_ETD2_V : VD_ETD2_E);
        CK(c->ops->dir[v](a, c->st));
    }
    e = cudaStreamSynchronize(c->st);
    if (e != cudaSuccess) return fail(c, e, "dlr_test_dir_pass");
    c->vh_valid = false;                 // the flow tables were overwritten: the next step rebuilds everything
    if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }
    return c->last_err == cudaSuccess ? DLR_OK : DLR_ERR_CUDA;
}

}  // extern "C"
