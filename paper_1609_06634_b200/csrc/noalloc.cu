// noalloc.cu -- the one entry point of the library that allocates nothing (include/bioem.h, "Allocation-free entry point"):
// Eq. 10 on caller-supplied device arrays, for callers that may not call cudaMalloc (code under CUDA graph
// capture, tight serving loops).  The existing path, bioem_get_ensemble_log_posterior, allocates its three work arrays per
// call and runs one thread block; this variant runs one thread per image over the whole GPU and keeps its work array --
// the per-image inner log-sums -- in a file-scope device array of fixed size, which every GPU that loads the library holds
// until the process exits (BIOEM_NOALLOC_MAX_IMG doubles = 512 KiB).
//
// The array's NAME is a device symbol: in host code it is a host-side stand-in, not a device address, and must never be
// passed to a kernel.  Host code takes its address once per device with cudaGetSymbolAddress (prepare() below, with that
// device current) and passes that pointer; device code could name the array directly.
//
// Every call shares the array and finds the previous call's contents in it.  Nothing in it has to start at zero: a call
// writes entries [0, n_img) in its first kernel and reads exactly those in its second, on the same stream.  Two calls whose
// kernels overlap on the GPU (different streams, or two host threads) race on it.
#include "../../include/bioem.h"
#include "common.cuh"

#include <math_constants.h>

#include <cmath>
#include <cstdio>
#include <mutex>

namespace {

constexpr int MAX_DEVICES = 64;

static __device__ __align__(256) double g_noalloc_scratch[BIOEM_NOALLOC_MAX_IMG];

std::mutex g_mu;
double *g_scratch_addr[MAX_DEVICES] = {};           // device address of g_noalloc_scratch on each device, once taken
thread_local char g_err[256] = "";

int fail(int code, const char *what, cudaError_t e = cudaSuccess)
{
    if (e != cudaSuccess)
        std::snprintf(g_err, sizeof g_err, "%s: %s", what, cudaGetErrorString(e));
    else
        std::snprintf(g_err, sizeof g_err, "%s", what);
    return code;
}

// Restores the caller's current device on every way out.
struct DeviceGuard {
    int prev = -1;
    cudaError_t enter(int device)
    {
        cudaError_t e = cudaGetDevice(&prev);
        if (e != cudaSuccess) { prev = -1; return e; }
        return device == prev ? cudaSuccess : cudaSetDevice(device);
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Inner sum of Eq. 10 for one image per thread: log sum_m w_m P_m,omega, max-shifted.  The log-weights are formed once per
// block in shared memory (w = 0 -> -inf: the model drops out; w < 0 -> NaN, which reaches the outputs).
__global__ void __launch_bounds__(256) k_ens_inner(const double *logp, const double *w, int n_img, int n_model, double *inner, double *per_image)
{
    __shared__ double lw[BIOEM_NOALLOC_MAX_MODEL];
    for (int m = threadIdx.x; m < n_model; m += 256) lw[m] = log(w ? w[m] : 1.0 / (double)n_model);
    __syncthreads();
    const int img = blockIdx.x * 256 + threadIdx.x;
    if (img >= n_img) return;
    const double *lp = logp + (size_t)img * n_model;
    double M = -CUDART_INF;
    bool bad = false;
    for (int m = 0; m < n_model; ++m) {
        const double t = lp[m] + lw[m];
        bad |= (t != t);
        M = fmax(M, t);
    }
    double v = M;
    if (bad) {
        v = CUDART_NAN;
    } else if (M != -CUDART_INF) {
        double S = 0.0;
        for (int m = 0; m < n_model; ++m) S += exp(lp[m] + lw[m] - M);
        v = M + log(S);
    }
    inner[img] = v;
    if (per_image) per_image[img] = v;
}

// Outer sum of Eq. 10 in the order of the existing path (finalize.cu, k_ensemble): thread i adds images i, i + 256, ... in
// order, then a fixed tree over the 256 partial sums -- so the total has the same rounding as that path's.
__global__ void __launch_bounds__(256) k_ens_outer(const double *inner, int n_img, double *total)
{
    __shared__ double sh[256];
    double acc = 0.0;
    for (int img = threadIdx.x; img < n_img; img += 256) acc += inner[img];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int st = 128; st >= 1; st >>= 1) {
        if ((int)threadIdx.x < st) sh[threadIdx.x] += sh[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = sh[0];
}

// Set-up, once per device, with that device current: the device address of the file-scope array.
int prepare(int device, double **out)
{
    if (device < 0 || device >= MAX_DEVICES) return fail(BIOEM_EBADARG, "noalloc: device index out of range");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[device]) {
        DeviceGuard guard;
        cudaError_t e = guard.enter(device);
        if (e != cudaSuccess) return fail(BIOEM_ECUDA, "noalloc: cudaSetDevice", e);
        double *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, g_noalloc_scratch);
        if (e != cudaSuccess || !ptr) return fail(BIOEM_ECUDA, "noalloc: cudaGetSymbolAddress", e);
        g_scratch_addr[device] = ptr;
    }
    if (out) *out = g_scratch_addr[device];
    return BIOEM_OK;
}

}  // namespace

extern "C" {

const char *bioem_noalloc_last_error(void) { return g_err; }

int bioem_noalloc_prepare(int device) { return prepare(device, nullptr); }

int bioem_ensemble_log_posterior_noalloc(int device, void *cuda_stream, int n_img, int n_model, const double *log_p, const double *weights,
                                         double *out_total, double *out_per_image)
{
    if (!log_p || !out_total) return fail(BIOEM_EBADARG, "ensemble_log_posterior_noalloc: log_p and out_total must not be NULL");
    if (n_img < 1 || n_model < 1) return fail(BIOEM_EBADARG, "ensemble_log_posterior_noalloc: n_img and n_model must be >= 1");
    if (n_img > BIOEM_NOALLOC_MAX_IMG || n_model > BIOEM_NOALLOC_MAX_MODEL) {
        std::snprintf(g_err, sizeof g_err,
                      "ensemble_log_posterior_noalloc: n_img = %d, n_model = %d exceed the fixed work array (at most %d images, %d models); "
                      "use bioem_get_ensemble_log_posterior",
                      n_img, n_model, BIOEM_NOALLOC_MAX_IMG, BIOEM_NOALLOC_MAX_MODEL);
        return BIOEM_EUNSUPPORTED;
    }
    double *scratch = nullptr;
    int rc = prepare(device, &scratch);
    if (rc) return rc;
    DeviceGuard guard;
    cudaError_t e = guard.enter(device);
    if (e != cudaSuccess) return fail(BIOEM_ECUDA, "ensemble_log_posterior_noalloc: cudaSetDevice", e);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    k_ens_inner<<<(unsigned)((n_img + 255) / 256), 256, 0, st>>>(log_p, weights, n_img, n_model, scratch, out_per_image);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BIOEM_ECUDA, "ensemble_log_posterior_noalloc: k_ens_inner", e);
    k_ens_outer<<<1, 256, 0, st>>>(scratch, n_img, out_total);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BIOEM_ECUDA, "ensemble_log_posterior_noalloc: k_ens_outer", e);
    return BIOEM_OK;
}

}  // extern "C"
