/*
 * dlr.h - C ABI of the B200 (sm_100a, fp64) hot path of the second-order projector-splitting dynamical
 * low-rank (DLR) integrator for the 6D Vlasov-Poisson equations,
 *     Cassini & Einkemmer, arXiv 2110.13481 (cited as PAPER.md:<line>), Algorithm 2
 * with the Fourier-spectral / exponential-integrator sub-steps of section 4.
 *
 * State: f(x,v) ~ sum_ij X_i(x) S_ij V_j(v) on a periodic n_x^3 x n_v^3 grid:
 *   X : N_x x r, column-major (each column = one low-rank factor on the grid),
 *       grid index I = i1 + n1*(i2 + n2*i3)  (x1 fastest),  h_x^3 X^T X = I
 *   S : r x r, column-major
 *   V : N_v x r, column-major, same linearisation, h_v^3 V^T V = I
 * All numbers are IEEE fp64 ("double precision").  Every step of the path runs in CUDA
 * kernels of this library; there is no CPU fallback: without a CUDA device every call that touches the
 * device returns DLR_ERR_CUDA.
 *
 * Conventions: C linkage, no exceptions cross the boundary, return 0 = DLR_OK, negative = error.
 * Pointers are HOST pointers unless the argument is documented as device / "on_device".
 * One context per stream/thread; no global state: a context lives on the device that owns its workspace (every
 * call switches to that device and restores the caller's), several contexts of any shape may coexist in a process.
 */
#ifndef DLR_B200_H
#define DLR_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    DLR_OK = 0,
    DLR_ERR_INVALID = -1,          /* null pointer / bad argument */
    DLR_ERR_UNSUPPORTED = -2,      /* grid size or rank outside the supported set */
    DLR_ERR_WORKSPACE = -3,        /* workspace too small or misaligned */
    DLR_ERR_CUDA = -4,             /* a CUDA runtime call failed (see dlr_last_cuda_error) */
    DLR_ERR_NOT_ORTHONORMAL = -5,  /* dlr_set_initial: h^3 X^T X or h^3 V^T V differs from I by > 1e-10 */
    DLR_ERR_NO_STATE = -6,         /* dlr_step / dlr_moments before dlr_set_initial */
    DLR_ERR_TOO_LARGE = -7         /* dlr_probe_noalloc: more probes than the static device scratch holds */
};

/* dlr_config.flags: the predictor of Algorithm 2 (line 1) needs of its L step only rho(L^1) = L^1^T omega_v
 * (eq. (13)), which the default path obtains from the 1D marginals of V without running the flow
 * (DESIGN.md row a7'). With this flag the Lie L-flow of Algorithm 1 line 9 is run literally and its
 * column sums are used: same numbers up to rounding, one more pass family per step. For A/B tests. */
#define DLR_FLAG_PREDICTOR_L_FLOW 1u
/* dlr_step advances with the unconventional ("basis update & Galerkin") integrator, the paper's reference [4], which
 * PAPER.md:29 and PAPER.md:288 name as supported by the framework without writing it out; here as oracle.step_bug
 * restates it (reading R19): K step and L step BOTH from (X0, S0, V0) with E frozen at E0 of eq. (12) ->
 * QR -> X1, V1;  M = <X1, X0>, N = <V1, V0> (h^3-weighted);  S step forward in time from M S0 N^T with the coefficients
 * of X1, V1.  First order; requires order = 1; robust to a rank-deficient S0. */
#define DLR_FLAG_UNCONVENTIONAL 2u

/* Grid descriptors of Fig. 2: number of points, left extreme, right extreme of the
 * periodic box per direction (grid spacing h = (hi-lo)/n, points lo + i*h, i = 0..n-1).
 * Supported: n_x[0]=n_x[1]=n_x[2] and n_v[0]=n_v[1]=n_v[2], each a power of two in 8..256 (n_x may differ
 * from n_v); rank in {5, 8, 10, 15, 20}. */
typedef struct dlr_config {
    int32_t n_x[3], n_v[3];
    double x_lo[3], x_hi[3], v_lo[3], v_hi[3];
    int32_t rank;
    int32_t order;      /* 2 = Algorithm 2; 1 = Algorithm 1 */
    double e_scale;     /* multiplies the electric field; 1.0 = the paper's equations, 0.0 = test hook "E = 0" */
    uint32_t flags;     /* 0, DLR_FLAG_PREDICTOR_L_FLOW (order 2) or DLR_FLAG_UNCONVENTIONAL (order 1) */
} dlr_config;

/* Diagnostics the paper plots (Figs. 4-7). */
typedef struct dlr_moments_t {
    double mass;               /* int int f dx dv          = (h_x^3 1^T X) S (h_v^3 V^T 1)                 */
    double momentum[3];        /* int int v_i f dx dv                                                      */
    double kinetic_energy;     /* 1/2 int int |v|^2 f dx dv                                                */
    double electric_energy;    /* 1/2 int |E|^2 dx, E from eq. (12) + Poisson on the state  */
    double s_fro;              /* ||S||_F                                                                   */
    int32_t qr_fallbacks;      /* number of Cholesky pivots that had to be repaired since dlr_set_initial: the
                                  factor was rank deficient to working precision ("QR or SVD"); 0 in
                                  every run whose results are compared with the oracle (reading R12)     */
    int32_t nonfinite;         /* 1 if a non-finite value was seen in S                                    */
    int32_t qr_third_stage;    /* QR decompositions since dlr_set_initial that needed a third CholeskyQR stage
                                  (kappa(K) >~ 1e7: the first steps of a rank-1 initial value); informational    */
    int32_t eig_unconverged;   /* symmetric eigen-solves that hit the Jacobi sweep cap; must be 0 */
} dlr_moments_t;

typedef struct dlr_ctx dlr_ctx;

/* Size in bytes of the single device workspace a context for cfg needs. Pure. */
int dlr_workspace_bytes(const dlr_config* cfg, size_t* bytes);

/* Create a context. d_workspace: DEVICE pointer, 256-byte aligned, >= dlr_workspace_bytes, owned by the
 * caller (e.g. a torch.empty tensor) and kept alive until dlr_destroy. cuda_stream: a cudaStream_t (0 = the
 * legacy default stream) on which ALL work of this context is issued. Builds wavenumber/twiddle tables. */
int dlr_create(const dlr_config* cfg, void* d_workspace, size_t bytes, void* cuda_stream, dlr_ctx** out);

/* Copy in the initial factors (Algorithm 2 "Input"). X: N_x*r, S: r*r, V: N_v*r doubles in the
 * layout above; on_device != 0: the three pointers are device pointers. Checks h^3 X^T X = I, h^3 V^T V = I
 * to 1e-10 (DLR_ERR_NOT_ORTHONORMAL). S may be singular. The caller keeps its buffers. Synchronises. */
int dlr_set_initial(dlr_ctx* ctx, const double* X, const double* S, const double* V, int on_device);

/* One step of Algorithm 2 (order 1: Algorithm 1) of size tau: (X,S,V) <- (X3,S7,V1).
 * Asynchronous on the context's stream; returns launch errors only. Numerical status is latched and
 * read through dlr_moments. */
int dlr_step(dlr_ctx* ctx, double tau);

/* nsteps steps of size tau (same as calling dlr_step nsteps times). */
int dlr_run(dlr_ctx* ctx, double tau, int nsteps);

/* Diagnostics of the current state; optionally f at n_probe grid-index pairs:
 * f_probe[p] = X[probe_ix[p],:] S V[probe_iv[p],:]^T (rows of F = X S V^T). probe_ix, probe_iv,
 * f_probe are HOST arrays (may be NULL with n_probe = 0). Synchronises the stream. */
int dlr_moments(dlr_ctx* ctx, dlr_moments_t* out, int n_probe, const int64_t* probe_ix,
                const int64_t* probe_iv, double* f_probe);

/* Copy out the current factors (checkpoint / tests). Factors are defined only up to the gauge
 * X -> X Q1, V -> V Q2, S -> Q1^T S Q2. Any of X, S, V may be NULL. Synchronises. */
int dlr_get_factors(dlr_ctx* ctx, double* X, double* S, double* V, int on_device);

/* The electric field used last inside dlr_step (E^{1/2} of Algorithm 2 line 2; E^0 for order 1):
 * 3*N_x doubles, component-major. For tests. dlr_moments does not disturb it (its own field buffer). */
int dlr_get_field(dlr_ctx* ctx, double* E, int on_device);

/* Per-phase device times (ms) of the LAST dlr_step executed with profiling on (dlr_set_profiling(ctx,1)
 * makes dlr_step record CUDA events between phases and disables graph replay; on = 2 records an event after every
 * launch instead, names = the launch expressions). names: the rows of the
 * paper's Table 2. Returns the number of phases written (<= cap). */
int dlr_set_profiling(dlr_ctx* ctx, int on);
int dlr_get_phase_times(dlr_ctx* ctx, int cap, float* ms, const char** names);

/* Number of kernel launches one dlr_step issues (for bench.py's gpu_launches). */
int dlr_launches_per_step(dlr_ctx* ctx);

/* Algorithmic bytes of the factor-sized passes the last dlr_step issued: every read or
 * write of an N x r factor counts 8 N r bytes, the field 8 N per component.  0 before the first step. */
double dlr_bytes_per_step(dlr_ctx* ctx);

/* Kernel-level entry point for tests (all pointers DEVICE, stream of ctx): the batched 3D real-to-complex FFT of
 * the Poisson solve on ncols = 3 columns of the x grid (which = 0; which = 1: the v grid, only if
 * it is not larger than the x grid) into the library's half-spectrum layout (k1 natural 0..n/2, k2 and k3 at
 * bit-reversed positions), and back (out = in up to rounding).  Other ncols: DLR_ERR_UNSUPPORTED.  The K/L flows
 * themselves use 1D transforms inside their passes and are tested through dlr_step. */
int dlr_test_fft_roundtrip(dlr_ctx* ctx, int which, int ncols, const double* d_in, double* d_out,
                           double* d_spec /* 2*ncols*(n/2+1)*n*n doubles */);

/* Kernel-level entry point for tests: ONE directional pass of a K/L flow (section 4) on a factor-
 * shaped array, so that a parity failure of dlr_step can be located.  d_in, d_out (and d_E: 3*N_x, only which = 0,
 * kind >= 2): DEVICE arrays of N*r doubles on grid `which` (0 = x, 1 = v); every other pointer is a HOST array.
 *   kind 0: sub-flow along direction 1, eqs. (14)/(17):  A <- [A min] -> F_1 -> * tabs[k1][j] -> F_1^-1 -> [* mout]
 *   kind 1: sub-flow along direction 2, eqs. (15)/(18):  F_2 -> * tabs[k2][j] -> F_2^-1     (min, mout ignored)
 *   kind 2 / 3: third sub-flow, eq. (19), exponential Euler / ETD2RK (reading R8) in a given eigenbasis:
 *           m = A min; N(m) = sum_i w_i o (m Q_i) with w = E (which = 0) or the velocity coordinate (which = 1);
 *           tabs = e^z, t phi1, t (phi1 - phi2), t phi2; result times mout.
 * min, mout: r x r row-major [column in][column out] or NULL (identity); Q: 3 r x r; tabs: complex
 * [1 or 4][n][r] in NATURAL DFT order of the wavenumber index, conjugate symmetric in k (real lines are transformed
 * in pairs).  Overwrites the context's flow tables (harmless: every flow of dlr_step rebuilds them). Synchronises. */
int dlr_test_dir_pass(dlr_ctx* ctx, int which, int kind, const double* d_in, double* d_out, const double* min_,
                      const double* mout, const double* tabs, const double* Q, const double* d_E);

/* Test entry for the adaptive CholeskyQR: given the upper pairs (row-major, r(r+1)/2 HOST
 * doubles) of the Gram matrix of a once-orthogonalised factor, reports whether the device-side criterion asks for a
 * third stage. Does not touch the state or the status counters. */
int dlr_test_chol_decide(dlr_ctx* ctx, const double* gram_upper, int* third_stage_needed);

void dlr_destroy(dlr_ctx* ctx);
const char* dlr_strerror(int code);
const char* dlr_last_cuda_error(dlr_ctx* ctx);

/* After a call returned DLR_ERR_CUDA the context refuses further work until the error is cleared. Clears the
 * latched error and drops the state (it may be half-updated): dlr_set_initial must follow. A sticky CUDA error
 * (illegal address, ...) cannot be cleared: the next call fails again. */
int dlr_clear_error(dlr_ctx* ctx);

/* f at grid-index pairs WITHOUT any device allocation, context or workspace: f_probe[p] = X[probe_ix[p],:] S
 * V[probe_iv[p],:]^T (rows of F = X S V^T), the same kernel arithmetic as the probes of dlr_moments.
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, serving loops, harnesses that forbid it): the
 * probe indices and results pass through a file-scope static device array of DLR_NOALLOC_MAX_PROBES * 24 bytes that every
 * GPU loading the library holds until the process exits; the call makes no cudaMalloc/cudaFree.
 *   d_X (N_x x rank), d_S (rank x rank), d_V (N_v x rank): DEVICE arrays in the layout at the top of this file (e.g.
 *   the output of dlr_get_factors(..., on_device = 1)), owned by the caller, all on the device that owns d_X (which the
 *   call makes current and restores); probe_ix, probe_iv, f_probe: HOST arrays of n_probe entries; cuda_stream: the
 *   stream the work is issued on (0 = legacy default).  Synchronises that stream.
 * Errors: n_probe > DLR_NOALLOC_MAX_PROBES -> DLR_ERR_TOO_LARGE (nothing is launched; split the call); null pointers,
 * non-positive sizes, an index outside [0, N) or a non-device d_X -> DLR_ERR_INVALID; CUDA failures -> DLR_ERR_CUDA.
 * dlr_noalloc_last_error() returns the message of the calling thread's last failed call ("" if none).
 * ALL calls share the one array: calls that overlap on the GPU (different streams or host threads) race on it and must
 * be serialised by the caller.  The array keeps the previous call's contents; nothing in it needs to start at zero
 * (a call overwrites every slot it reads). */
#define DLR_NOALLOC_MAX_PROBES 4096
int dlr_probe_noalloc(const double* d_X, const double* d_S, const double* d_V, int64_t N_x, int64_t N_v, int rank,
                      int n_probe, const int64_t* probe_ix, const int64_t* probe_iv, double* f_probe, void* cuda_stream);
const char* dlr_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DLR_B200_H */
