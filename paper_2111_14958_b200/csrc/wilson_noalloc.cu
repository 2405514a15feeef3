// wilson_noalloc.cu — wd_norm2_noalloc: the paper's dot-product kernel <a,a> for callers that cannot
// call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation).
//
// wd_norm2 (wilson_cg.cu) keeps the scratch of its grid reduction -- one fp64 partial per CTA and the ticket counter --
// in buffers that wd_create allocates.  This entry point needs no context and allocates NOTHING: the same scratch lives
// in a file-scope __device__ array of fixed size (every GPU that loads the library holds these 128.25 KB until the
// process exits).  The caller passes the input field and the device address of the result; the call only enqueues a
// 256-byte memset and one kernel on the caller's stream.
//
// The array's name is, in host code, a host-side stand-in and not a device address: the address the kernel is given
// comes from cudaGetSymbolAddress, asked once per device with that device current (na_scratch_ptr below).
//
// Every call shares the array.  It keeps the last call's contents: the ticket counter, which must start at zero, is
// cleared on the caller's stream in front of every launch; the partials are all overwritten before they are read.
// Two calls that overlap on the GPU (different streams, or two processes' worth of threads on one device through this
// library instance) race on it: callers serialise their calls per device.
#include "../../include/wilson_cg.h"
#include "wilson_kernels.cuh"

#include <cstdio>
#include <mutex>

using namespace wd;

namespace {

// CTA b sums the vectors [b * NA_CHUNK, (b + 1) * NA_CHUNK): the number of partials, hence the order of every addition,
// depends on the field size only -- the result is bit-identical on any GPU (wd_norm2's grid follows the SM count).
constexpr int NA_PER_THREAD = 16;
constexpr size_t NA_CHUNK = (size_t)VEC_NT * NA_PER_THREAD;      // 4096 128-bit vectors per CTA
constexpr size_t NA_MAX_PARTIALS = 16384;                         // 128 KB of fp64 partials
constexpr size_t NA_HEADER = 256;                                 // ticket counter, padded to the alignment
constexpr size_t NA_SCRATCH_BYTES = NA_HEADER + NA_MAX_PARTIALS * sizeof(double);
constexpr size_t NA_MAX_VECS = NA_MAX_PARTIALS * NA_CHUNK;        // 67 108 864 vectors of 128 bits = 1 GiB of field

static __device__ __align__(256) unsigned char na_scratch[NA_SCRATCH_BYTES];

template <typename real>
__global__ void __launch_bounds__(VEC_NT)
norm2_noalloc_kernel(const typename Field<real>::svec *__restrict__ a, size_t n, int V, int padded,
                     unsigned char *scratch, double *result)
{
    using svec = typename Field<real>::svec;
    unsigned int *counter = reinterpret_cast<unsigned int *>(scratch);
    double *partials = reinterpret_cast<double *>(scratch + NA_HEADER);
    const size_t base = (size_t)blockIdx.x * NA_CHUNK + threadIdx.x;
    double local = 0.0;
#pragma unroll 4
    for (int k = 0; k < NA_PER_THREAD; ++k) {
        const size_t i = base + (size_t)k * VEC_NT;
        if (i < n && real_site<Field<real>::NSP>(i, V, padded)) local += vnorm2<svec>(__ldg(a + i));
    }
    double total;
    if (grid_sum<VEC_NT>(local, partials, counter, &total)) *result = total;
}

thread_local char na_error[256] = "";

int na_fail(int code, const char *msg)
{
    snprintf(na_error, sizeof na_error, "%s", msg);
    return code;
}
int na_fail_cuda(const char *what, cudaError_t e)
{
    snprintf(na_error, sizeof na_error, "wd_norm2_noalloc: %s: %s", what, cudaGetErrorString(e));
    return WD_ERR_CUDA;
}

// device address of na_scratch on the CURRENT device, asked once per device
int na_scratch_ptr(unsigned char **out)
{
    static std::mutex mu;
    static unsigned char *ptr[WD_MAXDEV] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail_cuda("cudaGetDevice", e);
    if (dev < 0 || dev >= WD_MAXDEV) return na_fail(WD_ERR_ARG, "wd_norm2_noalloc: device ordinal beyond the library's table");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        unsigned char *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, na_scratch);
        if (e != cudaSuccess) return na_fail_cuda("cudaGetSymbolAddress(na_scratch)", e);
        if (!p) return na_fail(WD_ERR_CUDA, "wd_norm2_noalloc: cudaGetSymbolAddress returned a null address");
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return WD_OK;
}

size_t na_vecs(int precision, size_t vpad) { return (size_t)(precision == 32 ? 6 : 12) * vpad; }

}  // namespace

extern "C" const char *wd_noalloc_last_error(void) { return na_error; }

extern "C" size_t wd_noalloc_max_sites(int precision)
{
    if (precision != 32 && precision != 64) return 0;
    // largest V whose padded field has at most NA_MAX_VECS vectors, and whose site index fits the kernels' int
    const size_t v = NA_MAX_VECS / (precision == 32 ? 6 : 12);
    const size_t cap = (size_t)2147483647 / SB * SB;
    return (v < cap ? v : cap) / SB * SB;
}

extern "C" int wd_noalloc_prepare(void)
{
    unsigned char *p;
    return na_scratch_ptr(&p);
}

extern "C" int wd_norm2_noalloc(int precision, size_t n_sites, const void *a_native, double *result_dev,
                                void *cuda_stream)
{
    if (precision != 32 && precision != 64) return na_fail(WD_ERR_PRECISION, "wd_norm2_noalloc: precision must be 32 or 64");
    if (!a_native || !result_dev) return na_fail(WD_ERR_ARG, "wd_norm2_noalloc: NULL argument");
    if (n_sites == 0) return na_fail(WD_ERR_DIMS, "wd_norm2_noalloc: n_sites is 0");
    if (n_sites > wd_noalloc_max_sites(precision)) {
        snprintf(na_error, sizeof na_error,
                 "wd_norm2_noalloc: %zu sites exceed the static scratch (%zu partials of %zu vectors: at most %zu sites in "
                 "fp%d); use wd_norm2 with a context", n_sites, NA_MAX_PARTIALS, NA_CHUNK, wd_noalloc_max_sites(precision),
                 precision);
        return WD_ERR_DIMS;
    }
    unsigned char *scratch = nullptr;
    const int rc = na_scratch_ptr(&scratch);
    if (rc != WD_OK) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const size_t vpad = (n_sites + SB - 1) / SB * SB;
    const size_t n = na_vecs(precision, vpad);
    const unsigned int grid = (unsigned int)((n + NA_CHUNK - 1) / NA_CHUNK);
    const int padded = vpad != n_sites;
    // the ticket counter must start at zero whatever an earlier (possibly failed) call left behind
    cudaError_t e = cudaMemsetAsync(scratch, 0, NA_HEADER, stream);
    if (e != cudaSuccess) return na_fail_cuda("cudaMemsetAsync", e);
    if (precision == 32)
        norm2_noalloc_kernel<float><<<grid, VEC_NT, 0, stream>>>((const float4 *)a_native, n, (int)n_sites, padded, scratch, result_dev);
    else
        norm2_noalloc_kernel<double><<<grid, VEC_NT, 0, stream>>>((const double2 *)a_native, n, (int)n_sites, padded, scratch, result_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail_cuda("kernel launch", e);
    na_error[0] = 0;
    return WD_OK;
}
