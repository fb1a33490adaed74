// bench_hooks.cu — the benchmark hooks of include/bq_test.h (bq_bench_kernel, bq_bench_kernel_multi): device time of ONE internal
// kernel of the hot path, or of one whole inner BiCGStab iteration as the solver enqueues it.  Not part of the product boundary
// and not on any solve path: they only launch what hop.cu / blas.cu / solve.cu already launch, on scratch vectors of their own,
// bracketed by CUDA events on the solver's stream.
#include <math.h>
#include <stdlib.h>

#include "blas.cuh"
#include "blas_api.h"

// solve.cu
bq_status bq_solver_blas(bq_lattice* lat, BlasCtx** ctx, SolverScalars** host_mirror);
void bq_solver_drop_graphs(bq_lattice* lat);
void bq_solver_set_scalars(SolverScalars* sc, double ar, double ai, double wr, double wi, cudaStream_t s);

static bq_status schur(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw, int prec, int recon,
                       cudaStream_t s, const HopRed* red = nullptr, int nrhs = 0) {
    return bq_schur_red(lat, out, in, tmp, kappa, csw, prec, recon, s, red, nrhs);
}

// scratch filler of bq_bench_kernel: finite, non-zero, site- and component-dependent values in [-0.5, 0.5)
template <int PREC> __global__ void k_bench_fill(int Vh, void* f, unsigned int seed) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= Vh) return;
    typename Prec<PREC>::comp v[24];
#pragma unroll
    for (int i = 0; i < 24; i++) {
        unsigned int x = (unsigned int)h * 24u + i + seed * 0x9E3779B9u;
        x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
        v[i] = (typename Prec<PREC>::comp)((x >> 8) * (1.0f / 16777216.0f) - 0.5f);
    }
    store_spinor<PREC>(f, Vh, h, v);
}
static void bench_fill(int prec, int Vh, void* f, unsigned int seed, cudaStream_t s) {
    const int grid = (Vh + 127) / 128;
    if (prec == BQ_FP64) k_bench_fill<BQ_FP64><<<grid, 128, 0, s>>>(Vh, f, seed);
    else if (prec == BQ_FP32) k_bench_fill<BQ_FP32><<<grid, 128, 0, s>>>(Vh, f, seed);
    else k_bench_fill<BQ_HALF><<<grid, 128, 0, s>>>(Vh, f, seed);
}

// ---------------------------------------------------------------------------------------------------
// bq_bench_kernel: device time of one internal kernel of the hot path, measured with CUDA events over `reps`
// back-to-back launches that rotate over `nsets` sets of scratch vectors (so that consecutive launches do not find
// their operands in L2).  Benchmark hook only: contents of the scratch vectors are irrelevant.
// ---------------------------------------------------------------------------------------------------
extern "C" bq_status bq_bench_kernel(bq_lattice* lat, int which, bq_prec prec, bq_recon recon, double csw, double kappa, int reps,
                                     int nsets, double* us_per_launch, double* bytes_per_launch) {
    if (!lat) return BQ_EINVAL;
    if (!us_per_launch || !bytes_per_launch || reps < 1 || nsets < 1 || nsets > 16) return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel: bad arguments");
    if (prec != BQ_FP64 && prec != BQ_FP32 && prec != BQ_HALF) return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel: bad precision");
    if (recon != BQ_RECON18 && recon != BQ_RECON12) return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel: bad recon");
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "bq_bench_kernel: no gauge field loaded");
    BlasCtx* w = nullptr;
    SolverScalars* mirror = nullptr;
    BQ_TRY(bq_solver_blas(lat, &w, &mirror));
    const BlasCtx& c = *w;
    cudaStream_t s = c.stream;
    const Geom& g = lat->g;
    const size_t fb = field_bytes_one_parity(g, prec);
    const size_t xb = field_bytes_one_parity(g, prec == BQ_HALF ? BQ_FP32 : prec);   // solution accumulator of k_final
    const bool clover = csw != 0.0;
    const void *cl = nullptr, *cli = nullptr;
    const size_t cb = (size_t)g.Vh * CLOVER_REALS * prec_real_bytes(prec);
    if (clover) {
        BQ_TRY(bq_clover_build(lat, csw, kappa));
        BQ_TRY(bq_get_clover(lat, prec, 0, &cl));
        BQ_TRY(bq_get_clover(lat, prec, 1, &cli));
    }
    const void* gauge = nullptr;
    BQ_TRY(bq_get_gauge(lat, prec, recon, &gauge));
    // scratch: per set 7 vectors of the storage precision + 1 accumulator
    constexpr int NV = 7;
    char* pool = nullptr;
    const size_t set_bytes = NV * fb + xb;
    BQ_CUDA(lat, cudaMalloc(&pool, set_bytes * nsets));
    // finite non-zero contents: an exactly zero inner product would set the solver's breakdown flag and make the
    // following kernels exit early
    for (int set = 0; set < nsets; set++) {
        for (int i = 0; i < NV; i++) bench_fill(prec, g.Vh, pool + (size_t)set * set_bytes + (size_t)i * fb, 1 + set * 8 + i, s);
        bench_fill(prec == BQ_HALF ? BQ_FP32 : prec, g.Vh, pool + (size_t)set * set_bytes + (size_t)NV * fb, 100 + set, s);
    }
    bq_solver_set_scalars(c.sc, 0.5, 0.1, 0.5, -0.1, s);
    BQ_CHECK_LAUNCH(lat);
    const double spin_b = (double)spinor_site_bytes(prec), link_b = (double)link_reals(recon) * prec_real_bytes(prec);
    const double clov_b = (double)CLOVER_REALS * prec_real_bytes(prec), acc_b = (double)spinor_site_bytes(prec == BQ_HALF ? BQ_FP32 : prec);
    double bytes = 0;
    bq_status st = BQ_OK;
    auto vec = [&](int set, int i) { return static_cast<void*>(pool + (size_t)set * set_bytes + (size_t)i * fb); };
    auto accv = [&](int set) { return static_cast<void*>(pool + (size_t)set * set_bytes + (size_t)NV * fb); };
    auto launch = [&](int set) -> bq_status {
        void *v0 = vec(set, 0), *v1 = vec(set, 1), *v2 = vec(set, 2), *v3 = vec(set, 3), *v4 = vec(set, 4), *v5 = vec(set, 5);
        switch (which) {
            case BQ_K_HOP: bytes = 8 * link_b + 2 * spin_b; return bq_hop(lat, v0, v1, nullptr, -kappa, 0, prec, recon, nullptr, 0, s);
            case BQ_K_HOP_XPAY: bytes = 8 * link_b + 3 * spin_b; return bq_hop(lat, v0, v1, v2, kappa, 0, prec, recon, nullptr, 0, s);
            case BQ_K_HOP_CLOVINV:
                if (!clover) return bq_set_error(lat, BQ_ENOCLOVER, "bq_bench_kernel: clover kernels need csw != 0");
                bytes = 8 * link_b + 2 * spin_b + clov_b;
                return bq_hop(lat, v0, v1, nullptr, -kappa, 1, prec, recon, static_cast<const char*>(cli) + cb, 1, s);
            case BQ_K_HOP_CLOV_XPAY:
                if (!clover) return bq_set_error(lat, BQ_ENOCLOVER, "bq_bench_kernel: clover kernels need csw != 0");
                bytes = 8 * link_b + 3 * spin_b + clov_b;
                return bq_hop(lat, v0, v1, v2, kappa, 0, prec, recon, cl, 2, s);
            case BQ_K_SCHUR:
                bytes = 2 * (8 * link_b + 2 * spin_b) + spin_b + (clover ? 2 * clov_b : 0);
                return schur(lat, v0, v1, v2, kappa, csw, prec, recon, s);
            case BQ_K_NORM2: bytes = spin_b; return blas_norm2(lat, c, prec, v0);
            case BQ_K_P_UPDATE: bytes = 4 * spin_b; return bicg_p_update(lat, c, prec, v0, v1, v2);
            case BQ_K_ALPHA: bytes = 2 * spin_b; return bicg_alpha(lat, c, prec, v0, v1);
            case BQ_K_S_UPDATE: bytes = 3 * spin_b; return bicg_s_update(lat, c, prec, v0, v1, v2);
            case BQ_K_OMEGA: bytes = 2 * spin_b; return bicg_omega(lat, c, prec, v0, v1);
            case BQ_K_FINAL: bytes = 5 * spin_b + 2 * acc_b; return bicg_final(lat, c, prec, v0, v1, v2, v3, accv(set), v4);
            case BQ_K_HOP_XPAY_ALPHA: {
                bytes = 8 * link_b + 4 * spin_b + (clover ? clov_b : 0);
                const HopRed red{1, v3, c.sc};
                return bq_hop(lat, v0, v1, v2, kappa, 0, prec, recon, clover ? cl : nullptr, clover ? 2 : 0, s, &red);
            }
            case BQ_K_HOP_XPAY_OMEGA: {
                bytes = 8 * link_b + 3 * spin_b + (clover ? clov_b : 0);
                const HopRed red{2, nullptr, c.sc};
                return bq_hop(lat, v0, v1, v2, kappa, 0, prec, recon, clover ? cl : nullptr, clover ? 2 : 0, s, &red);
            }
            case BQ_K_BICG_ITER_UNFUSED:
            case BQ_K_BICG_ITER: {
                // one whole inner iteration (same order as inner_bicgstab): p-update, M^ (+ <rhat,v>), s-update,
                // M^ (+ <t,s>, <t,t>), final; the UNFUSED form runs the two inner products as separate kernels
                const bool fused = which == BQ_K_BICG_ITER;
                const double schur_b = 2 * (8 * link_b + 2 * spin_b) + spin_b + (clover ? 2 * clov_b : 0);
                bytes = 2 * schur_b + (4 + 3 + 5) * spin_b + 2 * acc_b + (fused ? 1 : 4) * spin_b;
                void* v6 = vec(set, 6);
                const HopRed red_alpha{1, v3, c.sc}, red_omega{2, nullptr, c.sc};
                BQ_TRY(bicg_p_update(lat, c, prec, v0, v1, v2));
                BQ_TRY(schur(lat, v2, v1, v6, kappa, csw, prec, recon, s, fused ? &red_alpha : nullptr));
                if (!fused) BQ_TRY(bicg_alpha(lat, c, prec, v3, v2));
                BQ_TRY(bicg_s_update(lat, c, prec, v0, v2, v4));
                BQ_TRY(schur(lat, v5, v4, v6, kappa, csw, prec, recon, s, fused ? &red_omega : nullptr));
                if (!fused) BQ_TRY(bicg_omega(lat, c, prec, v5, v4));
                return bicg_final(lat, c, prec, v1, v4, v5, v3, accv(set), v0);
            }
            default: return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel: unknown kernel id %d", which);
        }
    };
    for (int i = 0; i < nsets && st == BQ_OK; i++) st = launch(i);      // warm-up: one launch per set
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    if (st == BQ_OK) {
        cudaEventRecord(e0, s);
        for (int i = 0; i < reps && st == BQ_OK; i++) st = launch(i % nsets);
        cudaEventRecord(e1, s);
    }
    cudaError_t e = cudaStreamSynchronize(s);
    float ms = 0;
    if (st == BQ_OK && e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(pool);
    if (st != BQ_OK) return st;
    if (e != cudaSuccess) return bq_set_error(lat, BQ_ECUDA, "bq_bench_kernel: %s", cudaGetErrorString(e));
    *us_per_launch = (double)ms * 1e3 / reps;
    *bytes_per_launch = bytes * (double)g.Vh;
    return BQ_OK;
}

// ---------------------------------------------------------------------------------------------------
// bq_bench_kernel_multi: the same measurement for the multi-rhs kernels.  Algorithmic bytes per launch: links and
// clover blocks once, spinors once per right-hand side.
// ---------------------------------------------------------------------------------------------------
extern "C" bq_status bq_bench_kernel_multi(bq_lattice* lat, int which, bq_prec prec, bq_recon recon, double csw, double kappa,
                                           int nrhs, int reps, int nsets, double* us_per_launch, double* bytes_per_launch) {
    if (!lat) return BQ_EINVAL;
    if (!us_per_launch || !bytes_per_launch || reps < 1 || nsets < 1 || nsets > 16 || nrhs < 1)
        return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel_multi: bad arguments");
    if (prec != BQ_FP64 && prec != BQ_FP32 && prec != BQ_HALF) return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel_multi: bad precision");
    if (recon != BQ_RECON18 && recon != BQ_RECON12) return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel_multi: bad recon");
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "bq_bench_kernel_multi: no gauge field loaded");
    if ((double)nrhs * 2.0 * 12.0 * lat->g.Vh >= 2147483648.0) return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel_multi: batch too large");
    const Geom& g = lat->g;
    cudaStream_t s = 0;
    const size_t fb = field_bytes_one_parity(g, prec);
    const bool clover = csw != 0.0;
    const void *cl = nullptr, *cli = nullptr;
    const size_t cb = (size_t)g.Vh * CLOVER_REALS * prec_real_bytes(prec);
    if (clover) {
        BQ_TRY(bq_clover_build(lat, csw, kappa));
        BQ_TRY(bq_get_clover(lat, prec, 0, &cl));
        BQ_TRY(bq_get_clover(lat, prec, 1, &cli));
    }
    const void* gauge = nullptr;
    BQ_TRY(bq_get_gauge(lat, prec, recon, &gauge));
    const bool iter = which == BQ_K_BICG_ITER;
    const int NV = iter ? 8 : 3;     // per set: out, in, z/tmp (+ the BiCGStab vectors) — each an array of nrhs fields
    const size_t xb = field_bytes_one_parity(g, prec == BQ_HALF ? BQ_FP32 : prec);
    BlasCtx* w = nullptr;
    if (iter) {
        SolverScalars* mirror = nullptr;
        BQ_TRY(bq_solver_blas(lat, &w, &mirror));
        bq_solver_drop_graphs(lat);
        BQ_TRY(blas_ctx_reserve(lat, w, nrhs));
        w->nrhs = nrhs; w->stride = fb; w->xstride = xb; w->stride64 = field_bytes_one_parity(g, BQ_FP64);
        s = w->stream;
        for (int k = 0; k < nrhs; k++) {
            bq_solver_set_scalars(w->sc + k, 0.5, 0.1, 0.5, -0.1, s);
            BQ_CHECK_LAUNCH(lat);
        }
    }
    char* pool = nullptr;
    const size_t vec_bytes = (fb > xb ? fb : xb) * nrhs, set_bytes = NV * vec_bytes;
    BQ_CUDA(lat, cudaMalloc(&pool, set_bytes * nsets));
    for (int set = 0; set < nsets; set++)
        for (int i = 0; i < NV; i++)
            for (int k = 0; k < nrhs; k++)
                bench_fill(i == 7 && prec == BQ_HALF ? BQ_FP32 : prec, g.Vh,
                           pool + (size_t)set * set_bytes + (size_t)i * vec_bytes + (size_t)k * (i == 7 ? xb : fb), 1 + set * 256 + i * 16 + k, s);
    const double spin_b = (double)spinor_site_bytes(prec), link_b = (double)link_reals(recon) * prec_real_bytes(prec);
    const double clov_b = (double)CLOVER_REALS * prec_real_bytes(prec);
    double bytes = 0;
    bq_status st = BQ_OK;
    const HopMulti m{nrhs, fb, fb, fb, fb};
    auto launch = [&](int set) -> bq_status {
        void *v0 = pool + (size_t)set * set_bytes, *v1 = pool + (size_t)set * set_bytes + vec_bytes, *v2 = pool + (size_t)set * set_bytes + 2 * vec_bytes;
        switch (which) {
            case BQ_K_HOP: bytes = 8 * link_b + nrhs * 2 * spin_b; return bq_hop(lat, v0, v1, nullptr, -kappa, 0, prec, recon, nullptr, 0, s, nullptr, &m);
            case BQ_K_HOP_XPAY: bytes = 8 * link_b + nrhs * 3 * spin_b; return bq_hop(lat, v0, v1, v2, kappa, 0, prec, recon, nullptr, 0, s, nullptr, &m);
            case BQ_K_HOP_CLOVINV:
                if (!clover) return bq_set_error(lat, BQ_ENOCLOVER, "bq_bench_kernel_multi: clover kernels need csw != 0");
                bytes = 8 * link_b + clov_b + nrhs * 2 * spin_b;
                return bq_hop(lat, v0, v1, nullptr, -kappa, 1, prec, recon, static_cast<const char*>(cli) + cb, 1, s, nullptr, &m);
            case BQ_K_HOP_CLOV_XPAY:
                if (!clover) return bq_set_error(lat, BQ_ENOCLOVER, "bq_bench_kernel_multi: clover kernels need csw != 0");
                bytes = 8 * link_b + clov_b + nrhs * 3 * spin_b;
                return bq_hop(lat, v0, v1, v2, kappa, 0, prec, recon, cl, 2, s, nullptr, &m);
            case BQ_K_SCHUR:
                bytes = 2 * (8 * link_b + nrhs * 2 * spin_b) + nrhs * spin_b + (clover ? 2 * clov_b : 0);
                return bq_schur_red(lat, v0, v1, v2, kappa, csw, prec, recon, s, nullptr, nrhs);
            case BQ_K_BICG_ITER: {
                // one whole batched inner iteration as bq_solve_multi runs it (7 launches + 2 one-CTA-per-rhs finalisers)
                const BlasCtx& c = *w;
                char* base = pool + (size_t)set * set_bytes;
                void *r = base, *p = base + vec_bytes, *v = base + 2 * vec_bytes, *rhat = base + 3 * vec_bytes, *sv = base + 4 * vec_bytes,
                     *t = base + 5 * vec_bytes, *tmp = base + 6 * vec_bytes, *x = base + 7 * vec_bytes;
                const double schur_b = 2 * (8 * link_b + nrhs * 2 * spin_b) + nrhs * spin_b + (clover ? 2 * clov_b : 0);
                const double acc_b = (double)spinor_site_bytes(prec == BQ_HALF ? BQ_FP32 : prec);
                bytes = 2 * schur_b + nrhs * ((4 + 3 + 5 + 1) * spin_b + 2 * acc_b);
                const HopRed red_alpha{1, rhat, c.sc}, red_omega{2, nullptr, c.sc};
                BQ_TRY(bicg_p_update(lat, c, prec, r, p, v));
                BQ_TRY(bq_schur_red(lat, v, p, tmp, kappa, csw, prec, recon, s, &red_alpha, nrhs));
                BQ_TRY(bicg_s_update(lat, c, prec, r, v, sv));
                BQ_TRY(bq_schur_red(lat, t, sv, tmp, kappa, csw, prec, recon, s, &red_omega, nrhs));
                return bicg_final(lat, c, prec, p, sv, t, rhat, x, r);
            }
            default: return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel_multi: unsupported kernel id %d", which);
        }
    };
    for (int i = 0; i < nsets && st == BQ_OK; i++) st = launch(i);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    if (st == BQ_OK) {
        cudaEventRecord(e0, s);
        for (int i = 0; i < reps && st == BQ_OK; i++) st = launch(i % nsets);
        cudaEventRecord(e1, s);
    }
    cudaError_t e = cudaStreamSynchronize(s);
    float ms = 0;
    if (st == BQ_OK && e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(pool);
    if (w) w->nrhs = 1;
    if (st != BQ_OK) return st;
    if (e != cudaSuccess) return bq_set_error(lat, BQ_ECUDA, "bq_bench_kernel_multi: %s", cudaGetErrorString(e));
    *us_per_launch = (double)ms * 1e3 / reps;
    *bytes_per_launch = bytes * (double)g.Vh;
    return BQ_OK;
}
