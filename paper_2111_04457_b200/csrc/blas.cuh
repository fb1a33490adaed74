// blas.cuh — fused BLAS-1 building blocks for the solver.
//
// Work items.  fp64 / fp32 vectors are treated as flat arrays of 16-byte chunks (1 resp. 2 complex numbers):
// perfectly coalesced, trivially few registers.  Half-storage vectors carry one fp32 norm per site, so there the
// work item is a site (12 complex numbers): mantissas are rescaled on load and renormalised on store.
//
// Reductions.  Per thread in the compute type (fp64, or fp32 for fp32/half storage: BASELINE.json config 5
// "fp32 reductions"), then in fp64: warp shuffle -> shared memory -> thread-block cluster (distributed shared
// memory: rank 0 of each 4-CTA cluster reads its peers' block sums) -> one partial per cluster in global memory
// -> the last cluster to arrive (atomic ticket) adds the partials in index order and runs the finaliser, which
// updates the solver's device-resident scalars.  The order of every addition is fixed, so results are bitwise
// reproducible and no scalar ever visits the host inside an iteration.
#pragma once

#include <cooperative_groups.h>

#include "layout.cuh"

namespace cg = cooperative_groups;

constexpr int BLAS_BLOCK = 256;
constexpr int BLAS_CLUSTER = 4;
#ifndef BLAS_CTAS_PER_SM
#define BLAS_CTAS_PER_SM 4  // grid = SMs x this (persistent-style, grid-stride loops)
#endif

template <int PREC> struct Item;
template <> struct Item<BQ_FP64> {
    using C = double;
    static constexpr int NC = 1;
    static constexpr bool FLAT = true;   // items are independent 16-byte chunks: several per thread per trip (blas.cu)
    __host__ __device__ static int count(int Vh) { return 12 * Vh; }
    __device__ static void load_or_zero(const void* b, int Vh, int i, int n, C* v, int off = 0) {
        if (i < n) load(b, Vh, i + off, v);
        else v[0] = v[1] = 0;
    }
    __device__ static void load(const void* b, int, int i, C* v) {
        const double2 d = reinterpret_cast<const double2*>(b)[i];
        v[0] = d.x; v[1] = d.y;
    }
    __device__ static void store(void* b, int, int i, const C* v) { reinterpret_cast<double2*>(b)[i] = make_double2(v[0], v[1]); }
};
template <> struct Item<BQ_FP32> {
    using C = float;
    static constexpr int NC = 2;
    static constexpr bool FLAT = true;
    __host__ __device__ static int count(int Vh) { return 6 * Vh; }
    __device__ static void load_or_zero(const void* b, int Vh, int i, int n, C* v, int off = 0) {
        if (i < n) load(b, Vh, i + off, v);
        else v[0] = v[1] = v[2] = v[3] = 0;
    }
    __device__ static void load(const void* b, int, int i, C* v) {
        const float4 d = reinterpret_cast<const float4*>(b)[i];
        v[0] = d.x; v[1] = d.y; v[2] = d.z; v[3] = d.w;
    }
    __device__ static void store(void* b, int, int i, const C* v) { reinterpret_cast<float4*>(b)[i] = make_float4(v[0], v[1], v[2], v[3]); }
};
template <> struct Item<BQ_HALF> {
    using C = float;
    static constexpr int NC = 12;
    static constexpr bool FLAT = false;  // a site is already 52 bytes in 4 requests
    __host__ __device__ static int count(int Vh) { return Vh; }
    __device__ static void load_or_zero(const void* b, int Vh, int i, int n, C* v, int off = 0) {
        if (i < n) load(b, Vh, i + off, v);
        else {
#pragma unroll
            for (int k = 0; k < 24; k++) v[k] = 0;
        }
    }
    __device__ static void load(const void* b, int Vh, int i, C* v) { load_spinor<BQ_HALF>(b, Vh, i, v); }
    __device__ static void store(void* b, int Vh, int i, const C* v) { store_spinor<BQ_HALF>(b, Vh, i, v); }
    // The same load in two steps — request the packed words, unpack later — so that a kernel with several operands can
    // put all its requests in flight before the first conversion (k_final: 5 operands, 22 requests per site).
    struct Raw { uint4 q[3]; float n; };
    __device__ static void load_raw(const void* b, int Vh, int i, Raw& r) {
        using A = SpinorAddr<BQ_HALF>;
        const char* c = static_cast<const char*>(b);
#pragma unroll
        for (int k = 0; k < 3; k++) r.q[k] = *reinterpret_cast<const uint4*>(c + A::word(Vh, i, k));
        r.n = *reinterpret_cast<const float*>(c + A::tail(Vh, i));
    }
    __device__ static void unpack(const Raw& r, C* v) {
#pragma unroll
        for (int k = 0; k < 3; k++) unpack8(r.q[k], v + 8 * k);
#pragma unroll
        for (int k = 0; k < 24; k++) v[k] = __fmul_rn(v[k], r.n);   // as load_spinor
    }
    // what a load of the just-stored item would return: v -> fp16(v/n) * n, n = max|v|
    __device__ static void requantize(C* v) {
        float n = 0.f;
#pragma unroll
        for (int k = 0; k < 24; k++) n = fmaxf(n, fabsf(v[k]));
        const float inv = n > 0.f ? 1.0f / n : 0.f;
#pragma unroll
        for (int k = 0; k < 24; k++) v[k] = __half2float(__float2half_rn(v[k] * inv)) * n;
    }
};

// Device-resident solver state (one per handle).  Complex scalars are (re, im).
struct SolverScalars {
    double rho[2], alpha[2], omega[2], beta[2];
    double rhat_v[2], ts[2], tt;
    double r2;         // |r|^2 of the running (recursive) residual
    double stop2;      // stop when r2 <= stop2
    double red[4];     // plain reduction results (norm2, cdot, ...)
    double scale;      // outer loop: 1/|r| of the fp64 residual (0 if r == 0)
    double rnorm;      // outer loop: |r| of the fp64 residual
    int done;          // 0 running, 1 converged, 2 breakdown
    int iters;         // completed iterations
    int cg;            // 1: the state belongs to a CG on the normal equations (rho = |r_N|^2, real alpha and beta)
};

struct RedBuf {
    double* partials;        // [rhs][clusters][4]
    unsigned int* ticket;    // [rhs]
    int pstride;             // doubles of partials per right-hand side
};

// Batched (multi-rhs) launches: gridDim.y = right-hand sides; blockIdx.y selects the operand fields, the BiCGStab state
// sc[rhs] and the reduction scratch of that right-hand side.  gridDim.y = 1 is the plain case.  The fields of one operand
// are `stride` ITEMS apart (16-byte chunks for fp64 / fp32 vectors, sites for half-storage vectors and for the site-wise
// conversion kernels) and are reached through the item index, i + blockIdx.y * stride, NOT by offsetting the pointer
// parameters: with offset pointers ptxas no longer issued the 5 loads of k_final ahead of the arithmetic (2 instead of 5
// requests in flight per thread: 115 -> 211 us).  Item indices stay below 2^31 (checked by the callers).
__device__ __forceinline__ RedBuf rhs_redbuf(RedBuf rb) {
    rb.partials += (size_t)blockIdx.y * rb.pstride;
    rb.ticket += blockIdx.y;
    return rb;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// v[NRED]: this thread's partial sums.  fin(red) runs in exactly one thread of the grid with the full sums.
// Must be called by every thread of every block of a kernel launched with cluster size BLAS_CLUSTER.
template <int NRED, class Fin> __device__ __forceinline__ void grid_reduce(double* v, const RedBuf& rb, Fin fin) {
    __shared__ double s_warp[NRED][BLAS_BLOCK / 32];
    __shared__ double s_blk[NRED];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NRED; k++) {
        const double w = warp_sum(v[k]);
        if (lane == 0) s_warp[k][warp] = w;
    }
    __syncthreads();
    if (threadIdx.x < NRED) {
        double a = 0;
#pragma unroll
        for (int w = 0; w < BLAS_BLOCK / 32; w++) a += s_warp[threadIdx.x][w];
        s_blk[threadIdx.x] = a;
    }
    cg::cluster_group cl = cg::this_cluster();
    cl.sync();
    const unsigned int ncl = gridDim.x / BLAS_CLUSTER;
    if (cl.block_rank() == 0 && threadIdx.x < NRED) {
        double a = s_blk[threadIdx.x];
        for (unsigned int r = 1; r < BLAS_CLUSTER; r++) a += *cl.map_shared_rank(&s_blk[threadIdx.x], r);
        rb.partials[(size_t)(blockIdx.x / BLAS_CLUSTER) * NRED + threadIdx.x] = a;
        __threadfence();
    }
    cl.sync();   // peers' shared memory must stay alive until rank 0 has read it
    if (cl.block_rank() != 0) return;
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int t = atomicAdd(rb.ticket, 1u);
        s_last = (t == ncl - 1);
    }
    __syncthreads();
    if (!s_last || warp != 0) return;
    __threadfence();
    double red[NRED];
#pragma unroll
    for (int k = 0; k < NRED; k++) {
        double a = 0;
        for (unsigned int c = lane; c < ncl; c += 32) a += __ldcg(rb.partials + (size_t)c * NRED + k);
        red[k] = warp_sum(a);
    }
    if (lane == 0) {
        fin(red);
        *rb.ticket = 0;
        __threadfence();
    }
}

// complex helpers on (re, im) pairs
__device__ __forceinline__ void cdiv(const double* a, const double* b, double* q);

// Finalisers of the two inner products of a BiCGStab iteration, shared by the stand-alone reduction kernels
// (blas.cu) and by the hop kernel's fused reduction epilogues (hop.cu).
// (v)   r = <rhat, v>:            alpha = rho / <rhat, v>
__device__ __forceinline__ void fin_alpha(SolverScalars* sc, const double* r) {
    sc->rhat_v[0] = r[0];
    sc->rhat_v[1] = r[1];
    if (r[0] == 0.0 && r[1] == 0.0) {
        if (!sc->done) sc->done = 2;
    } else {
        cdiv(sc->rho, r, sc->alpha);
    }
}
// (iii) r = (<t,s>, <t,t>):       omega = <t,s> / <t,t>
__device__ __forceinline__ void fin_omega(SolverScalars* sc, const double* r) {
    sc->ts[0] = r[0]; sc->ts[1] = r[1]; sc->tt = r[2];
    if (r[2] == 0.0) {
        if (!sc->done) sc->done = 2;
    } else if (sc->cg) {
        // CG on M^dag M (out = q = M p, z = p): alpha = |r_N|^2 / <p, M^dag M p> = rho / |q|^2
        sc->alpha[0] = sc->rho[0] / r[2];
        sc->alpha[1] = 0;
    } else {
        sc->omega[0] = r[0] / r[2];
        sc->omega[1] = r[1] / r[2];
    }
}

template <typename C> __device__ __forceinline__ void cfma(C* y, C ar, C ai, const C* x) {   // y += a x
    const C xr = x[0], xi = x[1];
    y[0] = mad(-ai, xi, mad(ar, xr, y[0]));
    y[1] = mad(ai, xr, mad(ar, xi, y[1]));
}
__device__ __forceinline__ void cdiv(const double* a, const double* b, double* q) {   // q = a / b
    const double d = b[0] * b[0] + b[1] * b[1];
    q[0] = (a[0] * b[0] + a[1] * b[1]) / d;
    q[1] = (a[1] * b[0] - a[0] * b[1]) / d;
}
__device__ __forceinline__ void cmuld(const double* a, const double* b, double* q) {
    const double r = a[0] * b[0] - a[1] * b[1], i = a[0] * b[1] + a[1] * b[0];
    q[0] = r; q[1] = i;
}
