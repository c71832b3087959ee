// unitarity_noalloc.cu — gf_unitarity_noalloc (include/gf.h): Eq. (33) on a caller-owned link buffer,
// for callers that must not allocate.
//
// Who this is for.  gf_unitarity works on a context, and a context owns a second copy of the configuration plus its
// reduction buffers (gf_create allocates them) and, on top of that, takes and returns two scratch buffers with
// cudaMalloc / cudaFree on every call (cudaFree waits for the whole device).  Some users of the library cannot afford
// either: a lattice code whose own fields already fill the HBM of the GPU (the paper's 64^3 x 256 configuration in
// double is 39 GB, and it sits next to propagators and solver workspaces) and that only wants to watch |1 - det U| of
// ITS buffer; code that runs inside a memory pool with a fixed budget, where a cudaMalloc behind the pool's back fails
// or fragments it; a monitoring step between kernels of other streams that a device-wide cudaFree would stall.
// This entry point takes the caller's device buffer, needs no context, and gets, keeps and gives back no memory:
// the per-block partial sums, the only scratch the measurement needs, live in the file-scope array below, which is
// part of the loaded library image.
//
// The price, stated in gf.h as well: the array has a fixed size, so one call covers at most
// GF_UNITARITY_NOALLOC_MAX_LINKS links; every GPU that loads libgf.so holds the 2 MiB until the process exits; and
// all calls on one device share the array, so two calls whose kernels can run at the same time (different streams,
// different host threads) overwrite each other's partial sums — order them on one stream or with events.
//
// The kernel is the per-link part of unitarity_kernel (aux_kernels.cuh) for links in the host layout of gf.h
// (18 reals per link, row major, re/im innermost), not for the parity-split device store of a context.  Nothing of
// the existing code path is touched.
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/gf.h"

namespace {

constexpr int NA_THREADS = 256;          // threads per CTA
constexpr int NA_LINKS_PER_THREAD = 8;
constexpr int NA_LINKS_PER_CTA = NA_THREADS * NA_LINKS_PER_THREAD;                                  // 2048
constexpr int64_t NA_MAX_CTAS = (int64_t)GF_UNITARITY_NOALLOC_MAX_LINKS / NA_LINKS_PER_CTA;         // 131072
constexpr int NA_MAX_DEVICES = 64;

// The scratch: (sum, max) of |1 - det U| per CTA of the first kernel.  2 * 131072 doubles = 2 MiB per GPU.
// HOST code must never pass this name to a kernel: on the host it is a stand-in symbol, not a device address.
// scratch_of_current_device() below asks the runtime for the real address, once per device.
static __device__ __align__(256) double g_na_scratch[2 * NA_MAX_CTAS];

std::mutex g_na_mutex;
double* g_na_scratch_addr[NA_MAX_DEVICES];   // device address of g_na_scratch on device i, nullptr = not yet asked

// |1 - det U| of one link, 18 reals in double (the formula of unitarity_kernel)
__device__ __forceinline__ double det_deviation(const double (&m)[18]) {
#define NA_RE(i, j) m[((i) * 3 + (j)) * 2]
#define NA_IM(i, j) m[((i) * 3 + (j)) * 2 + 1]
    double dr = 0.0, di = 0.0;   // det = sum_j U_0j (U_1a U_2b - U_1b U_2a), (j, a, b) cyclic
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int a = (j + 1) % 3, b = (j + 2) % 3;
        const double cr = NA_RE(1, a) * NA_RE(2, b) - NA_IM(1, a) * NA_IM(2, b) - (NA_RE(1, b) * NA_RE(2, a) - NA_IM(1, b) * NA_IM(2, a));
        const double ci = NA_RE(1, a) * NA_IM(2, b) + NA_IM(1, a) * NA_RE(2, b) - (NA_RE(1, b) * NA_IM(2, a) + NA_IM(1, b) * NA_RE(2, a));
        dr += NA_RE(0, j) * cr - NA_IM(0, j) * ci;
        di += NA_RE(0, j) * ci + NA_IM(0, j) * cr;
    }
#undef NA_RE
#undef NA_IM
    return sqrt((1.0 - dr) * (1.0 - dr) + di * di);
}

// 18 reals of link i from the caller's buffer, widened to double; 16-byte (double) / 8-byte (float) loads
__device__ __forceinline__ void load_link(const double* __restrict__ p, int64_t i, double (&m)[18]) {
    const double2* q = reinterpret_cast<const double2*>(p + i * 18);
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const double2 v = __ldg(q + k);
        m[2 * k] = v.x; m[2 * k + 1] = v.y;
    }
}
__device__ __forceinline__ void load_link(const float* __restrict__ p, int64_t i, double (&m)[18]) {
    const float2* q = reinterpret_cast<const float2*>(p + i * 18);
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const float2 v = __ldg(q + k);
        m[2 * k] = (double)v.x; m[2 * k + 1] = (double)v.y;
    }
}

// (sum, max) over the CTA, fixed order; valid in thread 0
__device__ __forceinline__ void cta_sum_max(double& s, double& mx) {
    __shared__ double ss[32], sm[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s += __shfl_down_sync(0xffffffffu, s, o);
        mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    }
    if (lane == 0) { ss[w] = s; sm[w] = mx; }
    __syncthreads();
    if (w == 0) {
        s = lane < nw ? ss[lane] : 0.0;
        mx = lane < nw ? sm[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            s += __shfl_down_sync(0xffffffffu, s, o);
            mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
        }
    }
}

// CTA b covers links [b * 2048, (b + 1) * 2048): thread t takes b * 2048 + k * 256 + t, k = 0..7.
// scratch[2 b] = sum, scratch[2 b + 1] = max of |1 - det U| over the CTA's links: every slot the second kernel reads
// is written here in the same call, so nothing has to be cleared between calls.
template <class E>
__global__ void __launch_bounds__(NA_THREADS) unitarity_noalloc_kernel(const E* __restrict__ links, int64_t n_links,
                                                                      double* __restrict__ scratch) {
    const int64_t base = (int64_t)blockIdx.x * NA_LINKS_PER_CTA + threadIdx.x;
    double s = 0.0, mx = 0.0;
#pragma unroll 2
    for (int k = 0; k < NA_LINKS_PER_THREAD; ++k) {
        const int64_t i = base + (int64_t)k * NA_THREADS;
        if (i < n_links) {
            double m[18];
            load_link(links, i, m);
            const double dev = det_deviation(m);
            s += dev;
            mx = fmax(mx, dev);
        }
    }
    cta_sum_max(s, mx);
    if (threadIdx.x == 0) {
        scratch[2 * (int64_t)blockIdx.x] = s;
        scratch[2 * (int64_t)blockIdx.x + 1] = mx;
    }
}

// one CTA: result[0] = (sum of the n_ctas sums) / n_links, result[1] = max of the n_ctas maxima (n_links = 0: both 0)
__global__ void __launch_bounds__(1024) unitarity_noalloc_reduce_kernel(const double* __restrict__ scratch, int n_ctas,
                                                                        int64_t n_links, double* __restrict__ result) {
    double s = 0.0, mx = 0.0;
    for (int k = threadIdx.x; k < n_ctas; k += blockDim.x) {
        s += scratch[2 * (int64_t)k];
        mx = fmax(mx, scratch[2 * (int64_t)k + 1]);
    }
    cta_sum_max(s, mx);
    if (threadIdx.x == 0) {
        result[0] = n_links > 0 ? s / (double)n_links : 0.0;
        result[1] = mx;
    }
}

int na_fail(char* errbuf, int errbuf_len, int code, const char* fmt, ...) {
    if (errbuf && errbuf_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, (size_t)errbuf_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// Set-up, once per device, with that device current: the device address of g_na_scratch.  No allocation: the array
// came with the library image.  (The runtime may load the image onto the device at this point if nothing of libgf.so
// ran there before; that is why the first call on a device belongs before a stream capture.)
cudaError_t scratch_of_current_device(double** out, int* device) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    *device = dev;
    if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_na_scratch);
        if (e != cudaSuccess) return e;
        g_na_scratch_addr[dev] = static_cast<double*>(p);
    }
    *out = g_na_scratch_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int gf_unitarity_noalloc(const void* links_device, int elem_bytes, int64_t n_links, double* result_device,
                                    void* cuda_stream, char* errbuf, int errbuf_len) {
    if (errbuf && errbuf_len > 0) errbuf[0] = 0;
    // argument checks first: none of them touches the device
    if (elem_bytes != 4 && elem_bytes != 8)
        return na_fail(errbuf, errbuf_len, GF_EINVAL, "gf_unitarity_noalloc: elem_bytes = %d, must be 4 (float) or 8 (double)", elem_bytes);
    if (n_links < 0) return na_fail(errbuf, errbuf_len, GF_EINVAL, "gf_unitarity_noalloc: n_links = %lld < 0", (long long)n_links);
    if (n_links > (int64_t)GF_UNITARITY_NOALLOC_MAX_LINKS)
        return na_fail(errbuf, errbuf_len, GF_EINVAL,
                       "gf_unitarity_noalloc: n_links = %lld exceeds GF_UNITARITY_NOALLOC_MAX_LINKS = %lld (the fixed scratch array "
                       "holds one partial sum per %d links; measure the buffer in pieces of at most that many links and combine "
                       "the averages and maxima, or use gf_unitarity on a context)",
                       (long long)n_links, (long long)GF_UNITARITY_NOALLOC_MAX_LINKS, NA_LINKS_PER_CTA);
    if (!result_device) return na_fail(errbuf, errbuf_len, GF_EINVAL, "gf_unitarity_noalloc: result_device is NULL");
    if (n_links > 0 && !links_device) return na_fail(errbuf, errbuf_len, GF_EINVAL, "gf_unitarity_noalloc: links_device is NULL");
    if (((uintptr_t)links_device & (uintptr_t)(2 * elem_bytes - 1)) || ((uintptr_t)result_device & 7u))
        return na_fail(errbuf, errbuf_len, GF_EINVAL, "gf_unitarity_noalloc: links_device must be aligned to %d bytes and result_device to 8",
                       2 * elem_bytes);

    double* scratch = nullptr;
    int dev = -1;
    cudaError_t e = scratch_of_current_device(&scratch, &dev);
    if (e != cudaSuccess)
        return na_fail(errbuf, errbuf_len, GF_ECUDA, "gf_unitarity_noalloc: address of the scratch array on device %d: %s", dev,
                       cudaGetErrorString(e));

    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const int n_ctas = (int)((n_links + NA_LINKS_PER_CTA - 1) / NA_LINKS_PER_CTA);
    if (n_ctas > 0) {
        if (elem_bytes == 8)
            unitarity_noalloc_kernel<double><<<(unsigned)n_ctas, NA_THREADS, 0, stream>>>((const double*)links_device, n_links, scratch);
        else
            unitarity_noalloc_kernel<float><<<(unsigned)n_ctas, NA_THREADS, 0, stream>>>((const float*)links_device, n_links, scratch);
        e = cudaGetLastError();
        if (e != cudaSuccess)
            return na_fail(errbuf, errbuf_len, GF_ECUDA, "gf_unitarity_noalloc: launch of unitarity_noalloc_kernel: %s", cudaGetErrorString(e));
    }
    unitarity_noalloc_reduce_kernel<<<1, 1024, 0, stream>>>(scratch, n_ctas, n_links, result_device);
    e = cudaGetLastError();
    if (e != cudaSuccess)
        return na_fail(errbuf, errbuf_len, GF_ECUDA, "gf_unitarity_noalloc: launch of unitarity_noalloc_reduce_kernel: %s", cudaGetErrorString(e));
    return GF_OK;
}
