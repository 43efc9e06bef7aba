// pf_noalloc.cu -- pf_relax_noalloc (include/pf_noalloc.h): row N5 (Table 2 step 5) for callers
// that cannot allocate.  No grid, no cudaMalloc: the scratch of the reduction is the file-scope device array below.
//
// The array's NAME is a device symbol.  In host code it is only a stand-in (handing it to a kernel would pass a host
// address: a fault, or on systems where the GPU reaches host memory, silently the wrong memory).  The host obtains the
// device address once per device with cudaGetSymbolAddress, with that device current, and passes it to the kernels.
#include "../../include/pf_noalloc.h"
#include "pf_launch.h"

#include <mutex>

namespace pf {

void set_create_error(const char* msg);      // pf_api.cu: the message pf_last_error(NULL) returns

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_CHUNK = 4096;                                    // nodes per block
constexpr long long NA_MAX_BLOCKS = PF_NOALLOC_MAX_N / NA_CHUNK;  // 65 536
static_assert(NA_MAX_BLOCKS * NA_CHUNK == PF_NOALLOC_MAX_N, "the maximum is a whole number of blocks");

// One partial maximum per block; 512 KB per GPU that loads the library, held until the process exits.  Shared by all
// calls on the device; keeps the last call's contents; every call overwrites the entries it reads.
static __device__ __align__(256) double g_noalloc_partial[NA_MAX_BLOCKS];

// Block b: nodes [b * NA_CHUNK, (b + 1) * NA_CHUNK).  Same statements as k_relax of pf_pointwise.cu.
__global__ void __launch_bounds__(NA_THREADS)
k_relax_partial(long long n, double w, double w1, const double* __restrict__ phi0, double* __restrict__ phi,
                double* __restrict__ partial) {
    __shared__ double ms[32];
    double d = 0.0;
    const long long base = (long long)blockIdx.x * NA_CHUNK;
#pragma unroll 4
    for (int k = threadIdx.x; k < NA_CHUNK; k += NA_THREADS) {
        const long long i = base + k;
        if (i < n) {
            const double p0 = phi0[i];
            const double pn = add(mul(w, p0), mul(w1, phi[i]));
            phi[i] = pn;
            d = max_abs(d, sub(pn, p0));
        }
    }
    for (int s = 16; s > 0; s >>= 1) d = max_abs(d, __shfl_xor_sync(0xffffffffu, d, s));
    if ((threadIdx.x & 31) == 0) ms[threadIdx.x >> 5] = d;
    __syncthreads();
    if (threadIdx.x < 32) {
        d = threadIdx.x < NA_THREADS / 32 ? ms[threadIdx.x] : 0.0;
        for (int s = 16; s > 0; s >>= 1) d = max_abs(d, __shfl_xor_sync(0xffffffffu, d, s));
        if (threadIdx.x == 0) partial[blockIdx.x] = d;
    }
}

// One block: the maximum of the nblk partial results (a NaN is kept, max_abs) to the caller's output.
__global__ void __launch_bounds__(1024)
k_relax_final(int nblk, const double* __restrict__ partial, double* __restrict__ out) {
    __shared__ double ms[32];
    double d = 0.0;
    for (int b = threadIdx.x; b < nblk; b += blockDim.x) d = max_abs(d, partial[b]);
    for (int s = 16; s > 0; s >>= 1) d = max_abs(d, __shfl_xor_sync(0xffffffffu, d, s));
    if ((threadIdx.x & 31) == 0) ms[threadIdx.x >> 5] = d;
    __syncthreads();
    if (threadIdx.x < 32) {
        d = ms[threadIdx.x];
        for (int s = 16; s > 0; s >>= 1) d = max_abs(d, __shfl_xor_sync(0xffffffffu, d, s));
        if (threadIdx.x == 0) *out = d;
    }
}

// Device address of the scratch, looked up once per device (with that device current).
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mutex;
double* g_na_addr[NA_MAX_DEVICES] = {nullptr};

cudaError_t scratch_address(double** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_partial);       // the current device's copy of the array
        if (e != cudaSuccess) return e;
        g_na_addr[dev] = static_cast<double*>(p);
    }
    *out = g_na_addr[dev];
    return cudaSuccess;
}

int na_fail(int code, const char* msg) {
    set_create_error(msg);
    return code;
}

}  // namespace
}  // namespace pf

extern "C" int pf_relax_noalloc(long long n, double omega_pf, const double* phi0, double* phi, double* incr_out,
                                void* cuda_stream) {
    using namespace pf;
    if (n < 0) return na_fail(PF_ERR_ARG, "pf_relax_noalloc: n < 0");
    if (n > PF_NOALLOC_MAX_N)
        return na_fail(PF_ERR_ARG, "pf_relax_noalloc: n exceeds PF_NOALLOC_MAX_N = 2^28 nodes (the fixed scratch of the "
                                   "no-allocation entry point holds one partial result per 4096 nodes; use pf_solve_pf)");
    if (!incr_out || (n > 0 && (!phi0 || !phi))) return na_fail(PF_ERR_ARG, "pf_relax_noalloc: NULL pointer");
    if (!(omega_pf >= 0.0 && omega_pf < 1.0)) return na_fail(PF_ERR_ARG, "pf_relax_noalloc: omega_PF must be in [0,1)");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return na_fail(PF_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
    }
    double* partial = nullptr;
    cudaError_t e = scratch_address(&partial);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return na_fail(PF_ERR_CUDA, cudaGetErrorString(e));
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int nblk = (int)((n + NA_CHUNK - 1) / NA_CHUNK);
    if (nblk > 0) {
        ++g_launch_count;
        k_relax_partial<<<nblk, NA_THREADS, 0, s>>>(n, omega_pf, 1.0 - omega_pf, phi0, phi, partial);
    }
    ++g_launch_count;
    k_relax_final<<<1, 1024, 0, s>>>(nblk, partial, incr_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(PF_ERR_CUDA, cudaGetErrorString(e));
    return PF_OK;
}
