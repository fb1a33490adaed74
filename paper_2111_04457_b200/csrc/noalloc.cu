// noalloc.cu — bq_field_norm2_noalloc (include/bq.h): |a|^2 of an internal-layout field without any device allocation.
//
// Who this is for.  Every other reduction of this library keeps its per-CTA partial sums and its arrival counter in
// memory that the handle gets from cudaMalloc (blas.cu: blas_ctx_reserve; hop_kernels.cuh: hop_partials).  Some programs
// that embed the library must not, or cannot, allocate at the moment they need a norm:
//   * a host framework that has handed the whole device to its own caching allocator (PyTorch with a memory fraction,
//     an inference server with a fixed arena): a cudaMalloc from a plug-in library fails, or fragments the arena;
//   * code running while another thread of the process captures a stream in the global capture mode, where cudaMalloc is
//     a prohibited call and invalidates that capture;
//   * latency-critical loops (a monitor that checks a residual norm every step) in which cudaMalloc / cudaFree would
//     synchronise the whole device.
// For them the scratch lives in the library image itself: a file-scope __device__ array below, of fixed size, which
// every GPU that loads libbq.so holds from module load until the process exits (BQ_NOALLOC_SCRATCH_BYTES = 128 KiB + 256 B).
//
// The kernel is a variant of k_norm2 (blas.cu) — same work items and per-thread arithmetic (blas.cuh Item<PREC>: fp64
// accumulation for fp64 storage, fp32 per thread then fp64 across threads for fp32 / half storage), but every CTA owns a
// fixed run of 1024 sites and one slot of the scratch, so the scratch bounds the field size: at most
// BQ_NOALLOC_MAX_SITES = 16384 x 1024 sites.  No thread-block cluster, no handle, no workspace.
//
// The array's name means two different things.  In device code `noalloc_scratch` is the array.  In host code it is only
// the host-side shadow the runtime uses as a lookup key: passing it to a kernel would hand the kernel a host address (a
// fault, or on systems where the GPU can reach host memory a silent write to the wrong place).  The host therefore asks
// for the device address with cudaGetSymbolAddress — once per device, with that device current, since every device has
// its own copy — and passes that pointer to the kernel.
#include <mutex>

#include "blas.cuh"

namespace {

constexpr int NA_BLOCK = 256;
constexpr int NA_SITES_PER_CTA = 1024;
constexpr int NA_MAX_CTAS = 16384;
constexpr int NA_TICKET_DOUBLES = 32;   // the arrival counter sits in a 256-byte slot of its own behind the partial sums
constexpr int NA_MAX_DEVICES = 64;

static_assert((long long)NA_MAX_CTAS * NA_SITES_PER_CTA == BQ_NOALLOC_MAX_SITES, "bq.h states the limit");
static_assert((NA_MAX_CTAS + NA_TICKET_DOUBLES) * sizeof(double) == BQ_NOALLOC_SCRATCH_BYTES, "bq.h states the footprint");

// [0, NA_MAX_CTAS): one partial sum per CTA;  [NA_MAX_CTAS]: the arrival counter (first 4 bytes of its slot).
// Shared by every call on this device; holds whatever the previous call left there.
static __device__ __align__(256) double noalloc_scratch[NA_MAX_CTAS + NA_TICKET_DOUBLES];

template <int PREC> __global__ void __launch_bounds__(NA_BLOCK) k_norm2_noalloc(long long nsites, const void* __restrict__ a,
                                                                                 double* scratch, double* __restrict__ result) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = I::FLAT ? 4 : 1;
    constexpr int PER_SITE = PREC == BQ_FP64 ? 12 : (PREC == BQ_FP32 ? 6 : 1);   // work items per site, as Item<PREC>::count
    constexpr int ITEMS_PER_CTA = NA_SITES_PER_CTA * PER_SITE;
    const int n = (int)(nsites * PER_SITE);   // < 2^31: nsites <= 2^24, PER_SITE <= 12
    const int begin = blockIdx.x * ITEMS_PER_CTA;
    const int end = min(begin + ITEMS_PER_CTA, n);
    C acc = 0;
    for (int i0 = begin + threadIdx.x; i0 < end; i0 += NA_BLOCK * UNR) {
        C v[UNR][2 * I::NC];
#pragma unroll
        for (int u = 0; u < UNR; u++) I::load_or_zero(a, (int)nsites, i0 + u * NA_BLOCK, end, v[u]);
#pragma unroll
        for (int u = 0; u < UNR; u++)
#pragma unroll
            for (int k = 0; k < 2 * I::NC; k++) acc = mad(v[u][k], v[u][k], acc);
    }

    // CTA sum in fp64, fixed order: lanes by shuffle, warps in index order
    __shared__ double s_warp[NA_BLOCK / 32];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double w = warp_sum((double)acc);
    if (lane == 0) s_warp[warp] = w;
    __syncthreads();
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + NA_MAX_CTAS);
    if (threadIdx.x == 0) {
        double s = 0;
#pragma unroll
        for (int k = 0; k < NA_BLOCK / 32; k++) s += s_warp[k];
        scratch[blockIdx.x] = s;
        __threadfence();
        s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;

    // the CTA that arrived last adds the partial sums, again in a fixed order
    __threadfence();
    double t = 0;
    for (unsigned int c = threadIdx.x; c < gridDim.x; c += NA_BLOCK) t += __ldcg(scratch + c);
    t = warp_sum(t);
    if (lane == 0) s_warp[warp] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0;
#pragma unroll
        for (int k = 0; k < NA_BLOCK / 32; k++) s += s_warp[k];
        *result = s;
        *ticket = 0;   // the host clears it before every launch as well; see bq_field_norm2_noalloc
    }
}

// device address of noalloc_scratch on each device of this process, looked up on the first call made with that device current
std::mutex g_mutex;
double* g_scratch[NA_MAX_DEVICES] = {};

bq_status fail(char* err, size_t errlen, bq_status st, const char* what, const char* detail = nullptr) {
    if (err && errlen) snprintf(err, errlen, detail ? "bq_field_norm2_noalloc: %s: %s" : "bq_field_norm2_noalloc: %s", what, detail);
    return st;
}

}   // namespace

extern "C" bq_status bq_field_norm2_noalloc(const void* a, long long nsites, bq_prec prec, double* result, void* stream, char* err,
                                            size_t errlen) {
    if (err && errlen) err[0] = 0;
    if (!a || !result) return fail(err, errlen, BQ_EINVAL, "NULL field or result pointer");
    if (prec != BQ_FP64 && prec != BQ_FP32 && prec != BQ_HALF) return fail(err, errlen, BQ_EINVAL, "prec must be BQ_FP64, BQ_FP32 or BQ_HALF");
    if (nsites < 0 || nsites % 8) return fail(err, errlen, BQ_EINVAL, "nsites must be a non-negative multiple of 8 (the layout's tile)");
    if (nsites > BQ_NOALLOC_MAX_SITES) {
        if (err && errlen)
            snprintf(err, errlen,
                     "bq_field_norm2_noalloc: %lld sites exceed BQ_NOALLOC_MAX_SITES = %lld, the most the fixed in-library scratch covers "
                     "(one slot per 1024 sites); reduce the field in pieces, or use a call that owns a workspace",
                     nsites, (long long)BQ_NOALLOC_MAX_SITES);
        return BQ_EINVAL;
    }
    if (((uintptr_t)a & 15) || ((uintptr_t)result & 7)) return fail(err, errlen, BQ_EINVAL, "field must be 16-byte and result 8-byte aligned");

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(err, errlen, BQ_ECUDA, "cudaGetDevice", cudaGetErrorString(e));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(err, errlen, BQ_EINVAL, "device ordinal beyond the 64 this entry point keeps addresses for");
    double* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if (!g_scratch[dev]) {
            // set-up, once per device: `noalloc_scratch` in host code is not a device address (see the file header)
            double* p = nullptr;
            e = cudaGetSymbolAddress((void**)&p, noalloc_scratch);
            if (e != cudaSuccess || !p) return fail(err, errlen, BQ_ECUDA, "cudaGetSymbolAddress(noalloc_scratch)", cudaGetErrorString(e));
            g_scratch[dev] = p;
        }
        scratch = g_scratch[dev];
    }

    const cudaStream_t s = (cudaStream_t)stream;
    // the arrival counter must start at zero whatever an earlier (possibly failed) call left in the shared array; the partial
    // sums need no clearing: slots [0, grid) are all written before the last CTA reads them
    e = cudaMemsetAsync(scratch + NA_MAX_CTAS, 0, NA_TICKET_DOUBLES * sizeof(double), s);
    if (e != cudaSuccess) return fail(err, errlen, BQ_ECUDA, "cudaMemsetAsync(arrival counter)", cudaGetErrorString(e));
    const unsigned int grid = nsites ? (unsigned int)((nsites + NA_SITES_PER_CTA - 1) / NA_SITES_PER_CTA) : 1u;
    if (prec == BQ_FP64) k_norm2_noalloc<BQ_FP64><<<grid, NA_BLOCK, 0, s>>>(nsites, a, scratch, result);
    else if (prec == BQ_FP32) k_norm2_noalloc<BQ_FP32><<<grid, NA_BLOCK, 0, s>>>(nsites, a, scratch, result);
    else k_norm2_noalloc<BQ_HALF><<<grid, NA_BLOCK, 0, s>>>(nsites, a, scratch, result);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(err, errlen, BQ_ECUDA, "kernel launch", cudaGetErrorString(e));
    return BQ_OK;
}
