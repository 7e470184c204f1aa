// noalloc.cu - dlr_probe_noalloc (include/dlr.h): f = X S V^T at grid-index pairs (rows of F) for callers
// that may not allocate device memory (CUDA graph capture around them, tight serving loops, harnesses that forbid
// cudaMalloc).  The existing path (dlr_moments -> k_probes, small.cuh) keeps the probe indices and the results in the
// caller-owned workspace of a context; this variant keeps them in a file-scope static device array instead and needs
// no context and no workspace.  It calls no cudaMalloc/cudaFree and no allocating library routine.
//
// The array lives in every GPU that loads the library until the process exits (DLR_NOALLOC_MAX_PROBES * 24 bytes = 96 KB).
// Every call shares it: calls that overlap on the GPU (two streams, two host threads) race on it.  Nothing in it has to
// start at zero: a call overwrites the index slots it reads and the result slots it copies out, and reads no other slot.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/dlr.h"

namespace {

constexpr int MAXP = DLR_NOALLOC_MAX_PROBES;
constexpr int MAXDEV = 64;

// [0, MAXP) probe_ix | [MAXP, 2 MAXP) probe_iv (both as long long bit patterns) | [2 MAXP, 3 MAXP) f
static __device__ __align__(256) double g_probe_scratch[3 * MAXP];

// In host code `g_probe_scratch` is only a host-side stand-in of the symbol, not a device address: the address the
// kernel receives comes from cudaGetSymbolAddress, once per device, with that device current.
std::mutex g_mu;
double* g_scratch_ptr[MAXDEV];      // device address of g_probe_scratch on device d; nullptr = not looked up yet

cudaError_t scratch_on_current_device(int dev, double** out) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_probe_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return cudaSuccess;
}

// same arithmetic and order as k_probes (small.cuh): f[p] = sum_i X[ix_p, i] * (sum_j S[i, j] V[iv_p, j])
__global__ void k_probes_noalloc(const double* __restrict__ X, const double* __restrict__ S, const double* __restrict__ V,
                                 long long Nx, long long Nv, int R, int np, double* scratch) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const long long ix = reinterpret_cast<const long long*>(scratch)[p];
    const long long iv = reinterpret_cast<const long long*>(scratch + MAXP)[p];
    double s = 0.0;
    for (int i = 0; i < R; i++) {
        double t = 0.0;
        for (int j = 0; j < R; j++) t += S[i + R * j] * V[(size_t)j * Nv + iv];
        s += X[(size_t)i * Nx + ix] * t;
    }
    scratch[2 * MAXP + p] = s;
}

thread_local char g_err[256] = "";

int cuda_fail(cudaError_t e, const char* where, int prev_dev) {
    snprintf(g_err, sizeof g_err, "%s: %s", where, cudaGetErrorString(e));
    if (prev_dev >= 0) cudaSetDevice(prev_dev);
    return DLR_ERR_CUDA;
}

}  // namespace

extern "C" const char* dlr_noalloc_last_error(void) { return g_err; }

extern "C" int dlr_probe_noalloc(const double* d_X, const double* d_S, const double* d_V, int64_t N_x, int64_t N_v,
                                 int rank, int n_probe, const int64_t* probe_ix, const int64_t* probe_iv,
                                 double* f_probe, void* cuda_stream) {
    g_err[0] = 0;
    if (!d_X || !d_S || !d_V || N_x <= 0 || N_v <= 0 || rank <= 0 || n_probe < 0) {
        snprintf(g_err, sizeof g_err, "dlr_probe_noalloc: null pointer or non-positive size");
        return DLR_ERR_INVALID;
    }
    if (n_probe > MAXP) {
        snprintf(g_err, sizeof g_err, "dlr_probe_noalloc: n_probe = %d exceeds DLR_NOALLOC_MAX_PROBES = %d "
                 "(the static device scratch holds no more; split the call)", n_probe, MAXP);
        return DLR_ERR_TOO_LARGE;
    }
    if (n_probe == 0) return DLR_OK;
    if (!probe_ix || !probe_iv || !f_probe) {
        snprintf(g_err, sizeof g_err, "dlr_probe_noalloc: null probe array");
        return DLR_ERR_INVALID;
    }
    for (int p = 0; p < n_probe; p++)
        if (probe_ix[p] < 0 || probe_ix[p] >= N_x || probe_iv[p] < 0 || probe_iv[p] >= N_v) {
            snprintf(g_err, sizeof g_err, "dlr_probe_noalloc: probe %d outside the grid", p);
            return DLR_ERR_INVALID;
        }
    // the device that owns X becomes current for the call (and for the one-time symbol look-up)
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, d_X);
    if (e != cudaSuccess) return cuda_fail(e, "cudaPointerGetAttributes", -1);
    if (at.type != cudaMemoryTypeDevice || at.device < 0 || at.device >= MAXDEV) {
        snprintf(g_err, sizeof g_err, "dlr_probe_noalloc: d_X is not a device pointer");
        return DLR_ERR_INVALID;
    }
    int prev = -1;
    e = cudaGetDevice(&prev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice", -1);
    e = cudaSetDevice(at.device);
    if (e != cudaSuccess) return cuda_fail(e, "cudaSetDevice", prev);
    double* scratch = nullptr;
    e = scratch_on_current_device(at.device, &scratch);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress", prev);

    cudaStream_t st = (cudaStream_t)cuda_stream;
    e = cudaMemcpyAsync(scratch, probe_ix, (size_t)n_probe * sizeof(int64_t), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(scratch + MAXP, probe_iv, (size_t)n_probe * sizeof(int64_t), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e, "probe upload", prev);
    k_probes_noalloc<<<(n_probe + 127) / 128, 128, 0, st>>>(d_X, d_S, d_V, N_x, N_v, rank, n_probe, scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "k_probes_noalloc launch", prev);
    e = cudaMemcpyAsync(f_probe, scratch + 2 * MAXP, (size_t)n_probe * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e, "k_probes_noalloc", prev);
    cudaSetDevice(prev);
    return DLR_OK;
}
