// solve.cu — bq_solve: even-odd preconditioned BiCGStab with a mixed-precision defect-correction outer loop
// (the paper's `invert(x, b, nconv, diff)` of a "mixed precision solver").
//
//   b^_e = b_e + kappa H_eo A_oo^-1 b_o                                  (A10, fp64)
//   outer:  r = b^_e - M^ x_e (fp64) ; stop if |r| <= tol |b| ; r_lo = convert(r/|r|)          (A9)
//           inner BiCGStab  M^ e = r_lo  in fp64 / fp32 / half storage, e0 = 0               (A8)
//           x_e += |r| e
//   x_o = A_oo^-1 (b_o + kappa H_oe x_e)                                 (A10, fp64)
//   M^ = A_ee - kappa^2 H_eo A_oo^-1 H_oe                                (A7; A = 1 for Wilson)
//
// All BiCGStab scalars live in device memory (SolverScalars) and are produced by the reduction kernels'
// finalisers; the host only polls the {done, iters, r2} triple every `check_every` iterations.
#include <math.h>
#include <stdlib.h>

#include "blas.cuh"
#include "blas_api.h"

struct SolverWork {
    BlasCtx blas;
    bool blas_ok;
    // fp64, full lattice [even | odd]
    void *b, *x;
    // fp64, one parity
    void *bhat, *r, *t, *tmp;
    // inner precision, one parity
    int inner_prec;
    void *irhat, *ir, *ip, *iv, *is, *it, *itmp, *ie;
    SolverScalars* h_sc;   // pinned host mirror
    cudaEvent_t ev0, ev1;
};

static void free_inner(SolverWork* w) {
    void** v[] = {&w->irhat, &w->ir, &w->ip, &w->iv, &w->is, &w->it, &w->itmp, &w->ie};
    for (void** p : v) {
        if (*p) cudaFree(*p);
        *p = nullptr;
    }
    w->inner_prec = -1;
}

void bq_solver_free(bq_lattice* lat) {
    SolverWork* w = lat->work;
    if (!w) return;
    free_inner(w);
    void** v[] = {&w->b, &w->x, &w->bhat, &w->r, &w->t, &w->tmp};
    for (void** p : v) {
        if (*p) cudaFree(*p);
        *p = nullptr;
    }
    if (w->blas_ok) blas_ctx_destroy(&w->blas);
    if (w->h_sc) cudaFreeHost(w->h_sc);
    if (w->ev0) cudaEventDestroy(w->ev0);
    if (w->ev1) cudaEventDestroy(w->ev1);
    free(w);
    lat->work = nullptr;
}

static bq_status get_work(bq_lattice* lat, int inner_prec, SolverWork** out) {
    const Geom& g = lat->g;
    if (!lat->work) {
        SolverWork* w = static_cast<SolverWork*>(calloc(1, sizeof(SolverWork)));
        if (!w) return bq_set_error(lat, BQ_ENOMEM, "solver workspace: host allocation failed");
        w->inner_prec = -1;
        lat->work = w;
        BQ_TRY(blas_ctx_create(lat, &w->blas));
        w->blas_ok = true;
        const size_t fb = field_bytes_one_parity(g, BQ_FP64);
        BQ_CUDA(lat, cudaMalloc(&w->b, 2 * fb));
        BQ_CUDA(lat, cudaMalloc(&w->x, 2 * fb));
        BQ_CUDA(lat, cudaMalloc(&w->bhat, fb));
        BQ_CUDA(lat, cudaMalloc(&w->r, fb));
        BQ_CUDA(lat, cudaMalloc(&w->t, fb));
        BQ_CUDA(lat, cudaMalloc(&w->tmp, fb));
        BQ_CUDA(lat, cudaMallocHost(&w->h_sc, sizeof(SolverScalars)));
        BQ_CUDA(lat, cudaEventCreate(&w->ev0));
        BQ_CUDA(lat, cudaEventCreate(&w->ev1));
    }
    SolverWork* w = lat->work;
    if (w->inner_prec != inner_prec) {
        free_inner(w);
        const size_t fb = field_bytes_one_parity(g, inner_prec);
        void** v[] = {&w->irhat, &w->ir, &w->ip, &w->iv, &w->is, &w->it, &w->itmp};
        for (void** p : v) BQ_CUDA(lat, cudaMalloc(p, fb));
        // solution accumulator of the inner solve: fp32 when the inner storage is half
        BQ_CUDA(lat, cudaMalloc(&w->ie, field_bytes_one_parity(g, inner_prec == BQ_HALF ? BQ_FP32 : inner_prec)));
        w->inner_prec = inner_prec;
    }
    *out = w;
    return BQ_OK;
}

__global__ void k_set_bicg_scalars(SolverScalars* sc, double ar, double ai, double wr, double wi) {
    sc->alpha[0] = ar; sc->alpha[1] = ai;
    sc->omega[0] = wr; sc->omega[1] = wi;
    sc->rho[0] = 1; sc->rho[1] = 0;
    sc->done = 0; sc->iters = 0; sc->stop2 = -1.0;
}

// out_e = M^ in_e in precision prec (tmp: odd scratch)
static bq_status schur(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw, int prec, int recon,
                       cudaStream_t s, const HopRed* red = nullptr) {
    return bq_schur_red(lat, out, in, tmp, kappa, csw, prec, recon, s, red);
}

static bq_status poll(bq_lattice* lat, SolverWork* w) {
    BQ_CUDA(lat, cudaMemcpyAsync(w->h_sc, w->blas.sc, sizeof(SolverScalars), cudaMemcpyDeviceToHost, w->blas.stream));
    BQ_CUDA(lat, cudaStreamSynchronize(w->blas.stream));
    return BQ_OK;
}

// Inner BiCGStab on M^ e = ir (e0 = 0), stop when |r|^2 <= stop2 or after max_iter iterations.
// On return w->h_sc holds the final device state.  Textbook van der Vorst recurrences (reading O4).
static bq_status inner_bicgstab(bq_lattice* lat, SolverWork* w, double kappa, double csw, int prec, int recon, double stop2,
                                int max_iter, int check_every) {
    const BlasCtx& c = w->blas;
    cudaStream_t s = c.stream;
    const size_t fb = field_bytes_one_parity(lat->g, prec);
    const size_t eb = field_bytes_one_parity(lat->g, prec == BQ_HALF ? BQ_FP32 : prec);
    BQ_CUDA(lat, cudaMemsetAsync(w->ie, 0, eb, s));
    BQ_CUDA(lat, cudaMemsetAsync(w->ip, 0, fb, s));
    BQ_CUDA(lat, cudaMemsetAsync(w->iv, 0, fb, s));
    BQ_CUDA(lat, cudaMemcpyAsync(w->irhat, w->ir, fb, cudaMemcpyDeviceToDevice, s));
    BQ_TRY(bicg_init(lat, c, prec, w->ir, stop2));
    int launched = 0;
    // the two inner products on v and t ride on the second hop of M^ (hop.cu, RED epilogues): 7 kernels per iteration
    const HopRed red_alpha{1, w->irhat, c.sc}, red_omega{2, nullptr, c.sc};
    for (;;) {
        const int batch = (max_iter - launched) < check_every ? (max_iter - launched) : check_every;
        for (int k = 0; k < batch; k++) {
            BQ_TRY(bicg_p_update(lat, c, prec, w->ir, w->ip, w->iv));                          // p = r + beta (p - omega v)
            BQ_TRY(schur(lat, w->iv, w->ip, w->itmp, kappa, csw, prec, recon, s, &red_alpha)); // v = M^ p; alpha = rho/<rhat,v>
            BQ_TRY(bicg_s_update(lat, c, prec, w->ir, w->iv, w->is));                          // s = r - alpha v
            BQ_TRY(schur(lat, w->it, w->is, w->itmp, kappa, csw, prec, recon, s, &red_omega)); // t = M^ s; omega = <t,s>/<t,t>
            BQ_TRY(bicg_final(lat, c, prec, w->ip, w->is, w->it, w->irhat, w->ie, w->ir));
        }
        launched += batch;
        BQ_TRY(poll(lat, w));
        if (w->h_sc->done || launched >= max_iter) break;
    }
    return BQ_OK;
}

extern "C" bq_status bq_solve(bq_lattice* lat, const double* b, double* x, double kappa, double tol, const bq_solve_opts* opts,
                              bq_solve_info* info) {
    if (!lat) return BQ_EINVAL;
    if (info) {
        info->status = BQ_EINVAL; info->outer_cycles = 0; info->inner_iters = 0; info->restarts = 0;
        info->true_rel_residual = NAN; info->seconds = 0;
    }
    if (!b || !x) return bq_set_error(lat, BQ_EINVAL, "bq_solve: b or x is NULL");
    if (!(tol > 0.0) || !isfinite(tol)) return bq_set_error(lat, BQ_EINVAL, "bq_solve: tol must be positive");
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "bq_solve: no gauge field loaded");
    bq_solve_opts o;
    if (opts) o = *opts;
    else { o.inner_prec = BQ_FP32; o.recon = BQ_RECON18; o.csw = 0; o.inner_tol = 0; o.max_inner = 0; o.max_outer = 0; o.check_every = 0; o.stream = nullptr; }
    if (o.inner_prec != BQ_FP64 && o.inner_prec != BQ_FP32 && o.inner_prec != BQ_HALF) return bq_set_error(lat, BQ_EINVAL, "bq_solve: bad inner_prec");
    if (o.recon != BQ_RECON18 && o.recon != BQ_RECON12) return bq_set_error(lat, BQ_EINVAL, "bq_solve: bad recon");
    if (o.stream) return bq_set_error(lat, BQ_EINVAL, "bq_solve: opts->stream must be NULL");
    const int prec = o.inner_prec;
    const double inner_tol = o.inner_tol > 0 ? o.inner_tol : (prec == BQ_HALF ? 5e-2 : 1e-5);
    const int max_inner = o.max_inner > 0 ? o.max_inner : (prec == BQ_HALF ? 100 : 1000);
    const int max_outer = o.max_outer > 0 ? o.max_outer : 50;
    const int check_every = o.check_every > 0 ? o.check_every : 8;
    const double csw = o.csw;
    const bool clover = csw != 0.0;

    SolverWork* w = nullptr;
    BQ_TRY(get_work(lat, prec, &w));
    const BlasCtx& c = w->blas;
    cudaStream_t s = c.stream;
    const Geom& g = lat->g;
    const size_t fb64 = field_bytes_one_parity(g, BQ_FP64);
    char* bb = static_cast<char*>(w->b);
    char* xx = static_cast<char*>(w->x);
    const void *cl64 = nullptr, *cli64 = nullptr;
    const size_t cb64 = (size_t)g.Vh * CLOVER_REALS * sizeof(double);
    if (clover) {
        BQ_TRY(bq_clover_build(lat, csw, kappa));
        BQ_TRY(bq_get_clover(lat, BQ_FP64, 0, &cl64));
        BQ_TRY(bq_get_clover(lat, BQ_FP64, 1, &cli64));
    }

    BQ_CUDA(lat, cudaEventRecord(w->ev0, s));
    // ---- import b and x0 (canonical, host or device) through a device staging buffer ----
    {
        const size_t nb = (size_t)g.V * 24 * sizeof(double);
        double* stage = nullptr;
        BQ_CUDA(lat, cudaMalloc(&stage, nb));
        cudaError_t e = cudaMemcpyAsync(stage, b, nb, cudaMemcpyDefault, s);
        bq_status st = BQ_OK;
        if (e == cudaSuccess) st = bq_field_import(lat, w->b, stage, BQ_FULL, BQ_FP64, s);
        if (e == cudaSuccess && st == BQ_OK) e = cudaMemcpyAsync(stage, x, nb, cudaMemcpyDefault, s);
        if (e == cudaSuccess && st == BQ_OK) st = bq_field_import(lat, w->x, stage, BQ_FULL, BQ_FP64, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        cudaFree(stage);
        if (e != cudaSuccess) return bq_set_error(lat, BQ_ECUDA, "bq_solve: import failed: %s", cudaGetErrorString(e));
        BQ_TRY(st);
    }
    // |b|^2 over the full lattice (two parities)
    double bnorm2 = 0;
    for (int p = 0; p < 2; p++) {
        BQ_TRY(blas_norm2(lat, c, BQ_FP64, bb + p * fb64));
        BQ_TRY(poll(lat, w));
        bnorm2 += w->h_sc->red[0];
    }
    const double bnorm = sqrt(bnorm2);
    bq_status result = BQ_OK;
    int outer = 0, inner_total = 0, restarts = 0;
    if (bnorm == 0.0) {
        BQ_CUDA(lat, cudaMemsetAsync(w->x, 0, 2 * fb64, s));
    } else {
        // ---- b^_e = b_e + kappa H_eo A_oo^-1 b_o ----
        const void* bo = bb + fb64;
        if (clover) {
            BQ_TRY(bq_clover_mul(lat, w->tmp, bo, static_cast<const char*>(cli64) + cb64, BQ_FP64, s));
            bo = w->tmp;
        }
        BQ_TRY(bq_hop(lat, w->bhat, bo, bb, kappa, 0, BQ_FP64, BQ_RECON18, nullptr, 0, s));
        const double target = tol * bnorm;
        double prev_rnorm = INFINITY;
        int stalled = 0;
        for (;;) {
            // r = b^_e - M^ x_e in fp64
            BQ_TRY(schur(lat, w->t, xx, w->tmp, kappa, csw, BQ_FP64, BQ_RECON18, s));
            BQ_TRY(outer_residual(lat, c, w->bhat, w->t, w->r));
            BQ_TRY(poll(lat, w));
            const double rnorm = sqrt(w->h_sc->r2);
            if (!(rnorm == rnorm)) { result = bq_set_error(lat, BQ_EBREAKDOWN, "bq_solve: residual is NaN"); break; }
            if (rnorm <= target) break;
            if (outer >= max_outer) { result = bq_set_error(lat, BQ_ENOTCONVERGED, "bq_solve: max_outer reached, |r|/|b| = %.3e", rnorm / bnorm); break; }
            if (rnorm > 0.5 * prev_rnorm) {
                if (++stalled >= 4) { result = bq_set_error(lat, BQ_ENOTCONVERGED, "bq_solve: stalled at |r|/|b| = %.3e", rnorm / bnorm); break; }
            } else stalled = 0;
            prev_rnorm = rnorm;
            outer++;
            // normalised low-precision right-hand side and inner stopping threshold
            BQ_TRY(outer_to_low(lat, c, prec, w->r, w->ir));
            double rel = (prec == BQ_FP64) ? 0.9 * target / rnorm : fmax(inner_tol, 0.5 * target / rnorm);
            BQ_TRY(inner_bicgstab(lat, w, kappa, csw, prec, o.recon, rel * rel, max_inner, check_every));
            inner_total += w->h_sc->iters;
            if (w->h_sc->done == 2) restarts++;   // breakdown: the next outer cycle restarts from the true residual
            if (w->h_sc->done == 2 && w->h_sc->iters == 0 && restarts > 3) {
                result = bq_set_error(lat, BQ_EBREAKDOWN, "bq_solve: BiCGStab breakdown (rho or <rhat,v> or <t,t> = 0)");
                break;
            }
            // x_e += |r| e   (|r| = sc->rnorm, written by outer_residual; the inner loop does not touch it)
            BQ_TRY(outer_accumulate(lat, c, prec == BQ_HALF ? BQ_FP32 : prec, w->ie, xx));
        }
        // ---- x_o = A_oo^-1 (b_o + kappa H_oe x_e) ----
        BQ_TRY(bq_hop(lat, xx + fb64, xx, bb + fb64, kappa, 1, BQ_FP64, BQ_RECON18, nullptr, 0, s));
        if (clover) BQ_TRY(bq_clover_mul(lat, xx + fb64, xx + fb64, static_cast<const char*>(cli64) + cb64, BQ_FP64, s));
    }
    // ---- true residual |b - D x| / |b| on the full lattice, fp64 ----
    double true_rel = 0.0;
    if (bnorm > 0.0) {
        // reuse: t (even) and tmp (odd) are one-parity buffers; compute per parity
        double r2 = 0;
        for (int p = 0; p < 2; p++) {
            const void* clp = clover ? static_cast<const char*>(cl64) + p * cb64 : nullptr;
            BQ_TRY(bq_hop(lat, w->t, xx + (1 - p) * fb64, xx + p * fb64, -kappa, p, BQ_FP64, BQ_RECON18, clp, clover ? 2 : 0, s));
            BQ_TRY(outer_residual(lat, c, bb + p * fb64, w->t, w->r));
            BQ_TRY(poll(lat, w));
            r2 += w->h_sc->r2;
        }
        true_rel = sqrt(r2) / bnorm;
    }
    // ---- export x ----
    {
        const size_t nb = (size_t)g.V * 24 * sizeof(double);
        double* stage = nullptr;
        BQ_CUDA(lat, cudaMalloc(&stage, nb));
        bq_status st = bq_field_export(lat, stage, w->x, BQ_FULL, BQ_FP64, s);
        cudaError_t e = cudaSuccess;
        if (st == BQ_OK) e = cudaMemcpyAsync(x, stage, nb, cudaMemcpyDefault, s);
        if (e == cudaSuccess) e = cudaEventRecord(w->ev1, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        cudaFree(stage);
        if (e != cudaSuccess) return bq_set_error(lat, BQ_ECUDA, "bq_solve: export failed: %s", cudaGetErrorString(e));
        BQ_TRY(st);
    }
    float ms = 0;
    cudaEventElapsedTime(&ms, w->ev0, w->ev1);
    if (info) {
        info->status = result;
        info->outer_cycles = (prec == BQ_FP64) ? 0 : outer;
        info->inner_iters = inner_total;
        info->restarts = (prec == BQ_FP64) ? (outer > 0 ? outer - 1 : 0) + restarts : restarts;
        info->true_rel_residual = true_rel;
        info->seconds = ms * 1e-3;
    }
    return result;
}

// ---------------------------------------------------------------------------------------------------
// BLAS-1 test / benchmark entry points
// ---------------------------------------------------------------------------------------------------
static bq_status blas_entry(bq_lattice* lat, int prec, SolverWork** w) {
    if (!lat) return BQ_EINVAL;
    if (prec != BQ_FP64 && prec != BQ_FP32 && prec != BQ_HALF) return bq_set_error(lat, BQ_EINVAL, "bad precision");
    return get_work(lat, lat->work && lat->work->inner_prec >= 0 ? lat->work->inner_prec : BQ_FP32, w);
}

extern "C" bq_status bq_blas_norm2(bq_lattice* lat, const void* a, bq_prec prec, double* result) {
    SolverWork* w = nullptr;
    BQ_TRY(blas_entry(lat, prec, &w));
    if (!a || !result) return bq_set_error(lat, BQ_EINVAL, "bq_blas_norm2: NULL argument");
    BQ_TRY(blas_norm2(lat, w->blas, prec, a));
    BQ_TRY(poll(lat, w));
    *result = w->h_sc->red[0];
    return BQ_OK;
}

extern "C" bq_status bq_blas_cdot(bq_lattice* lat, const void* a, const void* b, bq_prec prec, double* result) {
    SolverWork* w = nullptr;
    BQ_TRY(blas_entry(lat, prec, &w));
    if (!a || !b || !result) return bq_set_error(lat, BQ_EINVAL, "bq_blas_cdot: NULL argument");
    BQ_TRY(blas_cdot(lat, w->blas, prec, a, b));
    BQ_TRY(poll(lat, w));
    result[0] = w->h_sc->red[0];
    result[1] = w->h_sc->red[1];
    return BQ_OK;
}

extern "C" bq_status bq_blas_caxpy(bq_lattice* lat, const double* alpha, const void* x, void* y, bq_prec prec) {
    SolverWork* w = nullptr;
    BQ_TRY(blas_entry(lat, prec, &w));
    if (!alpha || !x || !y) return bq_set_error(lat, BQ_EINVAL, "bq_blas_caxpy: NULL argument");
    return blas_caxpy(lat, w->blas, prec, alpha[0], alpha[1], x, y);
}

extern "C" bq_status bq_blas_bicg_update(bq_lattice* lat, const double* alpha, const double* omega, const void* p, const void* s,
                                         const void* t, const void* rhat, void* x, void* r, bq_prec prec, double* r_norm2,
                                         double* rhat_r) {
    SolverWork* w = nullptr;
    BQ_TRY(blas_entry(lat, prec, &w));
    if (!alpha || !omega || !p || !s || !t || !rhat || !x || !r || !r_norm2 || !rhat_r)
        return bq_set_error(lat, BQ_EINVAL, "bq_blas_bicg_update: NULL argument");
    k_set_bicg_scalars<<<1, 1, 0, w->blas.stream>>>(w->blas.sc, alpha[0], alpha[1], omega[0], omega[1]);
    BQ_CHECK_LAUNCH(lat);
    BQ_TRY(bicg_final(lat, w->blas, prec, p, s, t, rhat, x, r));
    BQ_TRY(poll(lat, w));
    *r_norm2 = w->h_sc->r2;
    rhat_r[0] = w->h_sc->rho[0];
    rhat_r[1] = w->h_sc->rho[1];
    return BQ_OK;
}

extern "C" bq_status bq_schur_apply_dots(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw,
                                         bq_prec prec, bq_recon recon, const void* w_vec, double* dots) {
    SolverWork* w = nullptr;
    BQ_TRY(blas_entry(lat, prec, &w));
    if (!dots) return bq_set_error(lat, BQ_EINVAL, "bq_schur_apply_dots: dots is NULL");
    const HopRed red{w_vec ? 1 : 2, w_vec, w->blas.sc};
    k_set_bicg_scalars<<<1, 1, 0, w->blas.stream>>>(w->blas.sc, 1, 0, 1, 0);   // rho = 1: alpha = 1 / <w, out>
    BQ_CHECK_LAUNCH(lat);
    BQ_TRY(bq_schur_red(lat, out, in, tmp, kappa, csw, prec, recon, w->blas.stream, &red));
    BQ_TRY(poll(lat, w));
    if (w_vec) {
        dots[0] = w->h_sc->rhat_v[0];
        dots[1] = w->h_sc->rhat_v[1];
    } else {
        dots[0] = w->h_sc->ts[0];
        dots[1] = w->h_sc->ts[1];
        dots[2] = w->h_sc->tt;
    }
    return BQ_OK;
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
    SolverWork* w = nullptr;
    BQ_TRY(get_work(lat, lat->work && lat->work->inner_prec >= 0 ? lat->work->inner_prec : BQ_FP32, &w));
    const BlasCtx& c = w->blas;
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
    k_set_bicg_scalars<<<1, 1, 0, s>>>(c.sc, 0.5, 0.1, 0.5, -0.1);
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
                if (!clover) return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel: clover kernels need csw != 0");
                bytes = 8 * link_b + 2 * spin_b + clov_b;
                return bq_hop(lat, v0, v1, nullptr, -kappa, 1, prec, recon, static_cast<const char*>(cli) + cb, 1, s);
            case BQ_K_HOP_CLOV_XPAY:
                if (!clover) return bq_set_error(lat, BQ_EINVAL, "bq_bench_kernel: clover kernels need csw != 0");
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
