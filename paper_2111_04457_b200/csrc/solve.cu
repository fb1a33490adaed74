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

// One batch of `batch` inner iterations captured as a CUDA graph.  Every kernel argument of an iteration is fixed for a
// given (method, precision, link form, kappa, csw, batch shape) — the vectors are the handle's workspace and all scalars
// live in device memory — so the graph is instantiated once and replayed for every later batch, inner solve and call.
struct IterGraph {
    cudaGraphExec_t exec;
    int method, prec, recon, nrhs, batch;
    double kappa, csw;
    unsigned long long epoch;
    bool warm;                               // a batch with this key has run eagerly (lazy stores and scratch exist)
    unsigned long long d_launch, d_hop[3], d_ls;   // what one replay adds to the handle's launch counters
};

struct SolverWork {
    BlasCtx blas;
    IterGraph graph;
    bool blas_ok;
    int nrhs;              // right-hand sides the buffers below are sized for
    // fp64, full lattice, [rhs][even | odd]
    void *b, *x;
    // fp64, one parity, [rhs]
    void *bhat, *r, *t, *tmp;
    // inner precision, one parity, [rhs]
    int inner_prec;
    void *irhat, *ir, *ip, *iv, *is, *it, *itmp, *ie;
    SolverScalars* h_sc;   // pinned host mirror, [rhs]
    double* h_stop2;       // pinned host staging of the per-rhs inner thresholds, [rhs]
    cudaEvent_t ev0, ev1;
    cudaEvent_t evp[4];    // phase boundaries: import | prepare | iterate | finish | export (bq_solve_info.phase_seconds)
    cudaStream_t side;     // second stream: the export + device-to-host copy of x runs here while the true residual is computed
    cudaEvent_t ev_side;
    bool persistent_stage; double* stage;   // device staging buffer of one canonical field (import / export)
};

static void drop_graph(SolverWork* w) {
    if (w->graph.exec) cudaGraphExecDestroy(w->graph.exec);
    w->graph.exec = nullptr;
    w->graph.warm = false;
}

static void free_inner(SolverWork* w) {
    drop_graph(w);
    void** v[] = {&w->irhat, &w->ir, &w->ip, &w->iv, &w->is, &w->it, &w->itmp, &w->ie};
    for (void** p : v) {
        if (*p) cudaFree(*p);
        *p = nullptr;
    }
    w->inner_prec = -1;
}

static void free_outer(SolverWork* w) {
    void** v[] = {&w->b, &w->x, &w->bhat, &w->r, &w->t, &w->tmp};
    for (void** p : v) {
        if (*p) cudaFree(*p);
        *p = nullptr;
    }
    if (w->h_sc) cudaFreeHost(w->h_sc);
    if (w->h_stop2) cudaFreeHost(w->h_stop2);
    w->h_sc = nullptr; w->h_stop2 = nullptr;
    w->nrhs = 0;
}

void bq_solver_free(bq_lattice* lat) {
    SolverWork* w = lat->work;
    if (!w) return;
    free_inner(w);
    free_outer(w);
    if (w->blas_ok) {
        blas_ctx_destroy(&w->blas);
        if (w->blas.stream) cudaStreamDestroy(w->blas.stream);
    }
    if (w->ev0) cudaEventDestroy(w->ev0);
    if (w->ev1) cudaEventDestroy(w->ev1);
    for (cudaEvent_t& e : w->evp) if (e) cudaEventDestroy(e);
    if (w->ev_side) cudaEventDestroy(w->ev_side);
    if (w->side) cudaStreamDestroy(w->side);
    if (w->stage) cudaFree(w->stage);
    free(w);
    lat->work = nullptr;
}

static bq_status get_work(bq_lattice* lat, int inner_prec, SolverWork** out, int nrhs = 1) {
    const Geom& g = lat->g;
    if (!lat->work) {
        SolverWork* w = static_cast<SolverWork*>(calloc(1, sizeof(SolverWork)));
        if (!w) return bq_set_error(lat, BQ_ENOMEM, "solver workspace: host allocation failed");
        w->inner_prec = -1;
        lat->work = w;
        // all or nothing: a half-built workspace must not survive (the next call would run with NULL streams / buffers)
        auto init = [&]() -> bq_status {
            BQ_TRY(blas_ctx_create(lat, &w->blas));
            w->blas_ok = true;
            BQ_CUDA(lat, cudaEventCreate(&w->ev0));
            BQ_CUDA(lat, cudaEventCreate(&w->ev1));
            for (cudaEvent_t& e : w->evp) BQ_CUDA(lat, cudaEventCreate(&e));
            BQ_CUDA(lat, cudaEventCreate(&w->ev_side));
            BQ_CUDA(lat, cudaStreamCreateWithFlags(&w->side, cudaStreamNonBlocking));
            BQ_CUDA(lat, cudaMalloc(&w->stage, (size_t)g.V * 24 * sizeof(double)));
            return BQ_OK;
        };
        const bq_status st = init();
        if (st != BQ_OK) {
            bq_solver_free(lat);
            return st;
        }
    }
    SolverWork* w = lat->work;
    if (w->nrhs < nrhs) {
        free_outer(w);
        free_inner(w);
        BQ_TRY(blas_ctx_reserve(lat, &w->blas, nrhs));
        const size_t fb = field_bytes_one_parity(g, BQ_FP64) * nrhs;
        BQ_CUDA(lat, cudaMalloc(&w->b, 2 * fb));
        BQ_CUDA(lat, cudaMalloc(&w->x, 2 * fb));
        BQ_CUDA(lat, cudaMalloc(&w->bhat, fb));
        BQ_CUDA(lat, cudaMalloc(&w->r, fb));
        BQ_CUDA(lat, cudaMalloc(&w->t, fb));
        BQ_CUDA(lat, cudaMalloc(&w->tmp, fb));
        BQ_CUDA(lat, cudaMallocHost(&w->h_sc, sizeof(SolverScalars) * nrhs));
        BQ_CUDA(lat, cudaMallocHost(&w->h_stop2, sizeof(double) * nrhs));
        w->nrhs = nrhs;
    }
    if (w->inner_prec != inner_prec) {
        free_inner(w);
        const size_t fb = field_bytes_one_parity(g, inner_prec) * w->nrhs;
        void** v[] = {&w->irhat, &w->ir, &w->ip, &w->iv, &w->is, &w->it, &w->itmp};
        for (void** p : v) BQ_CUDA(lat, cudaMalloc(p, fb));
        // solution accumulator of the inner solve: fp32 when the inner storage is half
        BQ_CUDA(lat, cudaMalloc(&w->ie, field_bytes_one_parity(g, inner_prec == BQ_HALF ? BQ_FP32 : inner_prec) * w->nrhs));
        w->inner_prec = inner_prec;
    }
    // batch shape of the BLAS launches: plain single-field launches until a multi-rhs solve says otherwise
    w->blas.nrhs = 1; w->blas.stride = 0; w->blas.xstride = 0; w->blas.stride64 = 0;
    *out = w;
    return BQ_OK;
}

// dd.cu: the BLAS-1 context (reduction scratch, device scalars, stream) and the pinned host mirror of a handle
bq_status bq_solver_blas(bq_lattice* lat, BlasCtx** ctx, SolverScalars** host_mirror) {
    SolverWork* w = nullptr;
    BQ_TRY(get_work(lat, lat->work && lat->work->inner_prec >= 0 ? lat->work->inner_prec : BQ_FP32, &w));
    *ctx = &w->blas;
    *host_mirror = w->h_sc;
    return BQ_OK;
}

// bench_hooks.cu: cached iteration graphs hold the workspace's batch shape — a benchmark that reshapes the context drops them
void bq_solver_drop_graphs(bq_lattice* lat) {
    if (lat->work) drop_graph(lat->work);
}

__global__ void k_set_bicg_scalars(SolverScalars* sc, double ar, double ai, double wr, double wi) {
    sc->alpha[0] = ar; sc->alpha[1] = ai;
    sc->omega[0] = wr; sc->omega[1] = wi;
    sc->rho[0] = 1; sc->rho[1] = 0;
    sc->done = 0; sc->iters = 0; sc->stop2 = -1.0;
}

// preset of a BiCGStab state (alpha, omega; rho = 1, running) on stream s: test and benchmark hooks
void bq_solver_set_scalars(SolverScalars* sc, double ar, double ai, double wr, double wi, cudaStream_t s) {
    k_set_bicg_scalars<<<1, 1, 0, s>>>(sc, ar, ai, wr, wi);
}

// out_e = M^ in_e in precision prec (tmp: odd scratch); nrhs = 0: single fields, >= 1: arrays of nrhs fields
static bq_status schur(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw, int prec, int recon,
                       cudaStream_t s, const HopRed* red = nullptr, int nrhs = 0) {
    return bq_schur_red(lat, out, in, tmp, kappa, csw, prec, recon, s, red, nrhs);
}

// Publish the device-resident solver states of the nrhs right-hand sides of the current batch to w->h_sc (pinned, mapped host
// memory) and wait for them.  A tiny kernel stores them straight through the mapped pointer — not a cudaMemcpyAsync: a
// device-to-host copy would queue on the copy engine behind whatever else is going that way (the 400 MB of x that
// bq_solve sends home on its side stream while the true residual is being polled).
__global__ void k_publish(unsigned long long* __restrict__ host, const unsigned long long* __restrict__ dev, int n8) {
    for (int i = threadIdx.x; i < n8; i += blockDim.x) host[i] = dev[i];
    __threadfence_system();
}
static_assert(sizeof(SolverScalars) % 8 == 0, "SolverScalars is published in 8-byte pieces");

static bq_status poll(bq_lattice* lat, SolverWork* w) {
    k_publish<<<1, 128, 0, w->blas.stream>>>(reinterpret_cast<unsigned long long*>(w->h_sc),
                                             reinterpret_cast<const unsigned long long*>(w->blas.sc),
                                             (int)(sizeof(SolverScalars) * w->blas.nrhs / 8));
    BQ_CUDA(lat, cudaGetLastError());
    BQ_CUDA(lat, cudaStreamSynchronize(w->blas.stream));
    return BQ_OK;
}

// Run `batch` iterations, enqueued one at a time by `one()`: eagerly the first time a key is seen (that run also creates
// whatever is made on first use: low-precision gauge / clover copies, reduction scratch), as a replay of the cached
// graph afterwards; full batches only.  Any failure of the capture falls back to eager launches.
template <class F>
static bq_status run_batch(bq_lattice* lat, SolverWork* w, int method, int prec, int recon, double kappa, double csw, int batch,
                           int full_batch, F one) {
    IterGraph& g = w->graph;
    cudaStream_t s = w->blas.stream;
    const bool same = g.method == method && g.prec == prec && g.recon == recon && g.nrhs == w->blas.nrhs && g.batch == batch &&
                      g.kappa == kappa && g.csw == csw && g.epoch == lat->epoch;
    auto eager = [&]() -> bq_status {
        for (int k = 0; k < batch; k++) BQ_TRY(one());
        return BQ_OK;
    };
    if (!lat->use_graphs || batch != full_batch) return eager();
    if (same && g.exec) {
        BQ_CUDA(lat, cudaGraphLaunch(g.exec, s));
        lat->n_launch += g.d_launch;
        for (int p = 0; p < 3; p++) lat->n_hop[p] += g.d_hop[p];
        lat->n_ls += g.d_ls;
        return BQ_OK;
    }
    if (!same || !g.warm) {
        drop_graph(w);
        g.method = method; g.prec = prec; g.recon = recon; g.nrhs = w->blas.nrhs; g.batch = batch; g.kappa = kappa; g.csw = csw;
        g.epoch = lat->epoch;
        BQ_TRY(eager());
        g.warm = true;
        return BQ_OK;
    }
    // second batch with this key: capture it, then launch what was captured
    const unsigned long long l0 = lat->n_launch, h0[3] = {lat->n_hop[0], lat->n_hop[1], lat->n_hop[2]}, ls0 = lat->n_ls;
    if (cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        return eager();
    }
    bq_status st = eager();
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(s, &graph);
    if (st == BQ_OK && e == cudaSuccess && graph) e = cudaGraphInstantiate(&g.exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (st != BQ_OK || e != cudaSuccess || !g.exec) {
        cudaGetLastError();
        g.exec = nullptr;
        lat->use_graphs = 0;              // do not try again on this handle
        lat->n_launch = l0;
        for (int p = 0; p < 3; p++) lat->n_hop[p] = h0[p];
        lat->n_ls = ls0;
        return eager();
    }
    g.d_launch = lat->n_launch - l0;
    for (int p = 0; p < 3; p++) g.d_hop[p] = lat->n_hop[p] - h0[p];
    g.d_ls = lat->n_ls - ls0;
    BQ_CUDA(lat, cudaGraphLaunch(g.exec, s));
    return BQ_OK;
}

// While one of these lives, every hop launched through the handle tests the `done` flag of its right-hand side's solver
// state at entry (HopArgs::done) exactly as the BLAS-1 kernels do: once a right-hand side has converged (or broken
// down) the rest of the batch of iterations already enqueued for it — hops included — costs a launch and nothing else.
struct HopDoneScope {
    bq_lattice* lat;
    HopDoneScope(bq_lattice* l, const SolverScalars* sc) : lat(l) { lat->hop_done = sc; }
    ~HopDoneScope() { lat->hop_done = nullptr; }
};

// Inner BiCGStab on M^ e = ir (e0 = 0) for every right-hand side of the batch (w->blas.nrhs), each with its own
// device-resident scalars; rhs k stops when |r_k|^2 <= w->h_stop2[k] or after max_iter iterations.  A right-hand
// side that has stopped keeps its iterate frozen (its update kernels and its share of the hop kernels exit early) while
// the others go on.  On return w->h_sc holds the final device states.
// Textbook van der Vorst recurrences (reading O4).
static bq_status inner_bicgstab(bq_lattice* lat, SolverWork* w, double kappa, double csw, int prec, int recon, int max_iter,
                                int check_every) {
    const BlasCtx& c = w->blas;
    cudaStream_t s = c.stream;
    const int n = c.nrhs, mrhs = n > 1 ? n : 0;
    const size_t fb = field_bytes_one_parity(lat->g, prec) * n;
    const size_t eb = field_bytes_one_parity(lat->g, prec == BQ_HALF ? BQ_FP32 : prec) * n;
    BQ_CUDA(lat, cudaMemsetAsync(w->ie, 0, eb, s));
    BQ_CUDA(lat, cudaMemsetAsync(w->ip, 0, fb, s));
    BQ_CUDA(lat, cudaMemsetAsync(w->iv, 0, fb, s));
    BQ_CUDA(lat, cudaMemcpyAsync(w->irhat, w->ir, fb, cudaMemcpyDeviceToDevice, s));
    BQ_CUDA(lat, cudaMemcpyAsync(c.stop2s, w->h_stop2, sizeof(double) * n, cudaMemcpyHostToDevice, s));
    BQ_TRY(bicg_init(lat, c, prec, w->ir, 0.0, true));
    int launched = 0;
    const HopDoneScope done_scope(lat, c.sc);
    // the two inner products on v and t ride on the second hop of M^ (hop.cu, RED epilogues): 7 kernels per iteration
    const HopRed red_alpha{1, w->irhat, c.sc}, red_omega{2, nullptr, c.sc};
    for (;;) {
        const int batch = (max_iter - launched) < check_every ? (max_iter - launched) : check_every;
        BQ_TRY(run_batch(lat, w, BQ_BICGSTAB, prec, recon, kappa, csw, batch, check_every, [&]() -> bq_status {
            BQ_TRY(bicg_p_update(lat, c, prec, w->ir, w->ip, w->iv));                                // p = r + beta (p - omega v)
            BQ_TRY(schur(lat, w->iv, w->ip, w->itmp, kappa, csw, prec, recon, s, &red_alpha, mrhs)); // v = M^ p; alpha = rho/<rhat,v>
            BQ_TRY(bicg_s_update(lat, c, prec, w->ir, w->iv, w->is));                                // s = r - alpha v
            BQ_TRY(schur(lat, w->it, w->is, w->itmp, kappa, csw, prec, recon, s, &red_omega, mrhs)); // t = M^ s; omega = <t,s>/<t,t>
            return bicg_final(lat, c, prec, w->ip, w->is, w->it, w->irhat, w->ie, w->ir);
        }));
        launched += batch;
        BQ_TRY(poll(lat, w));
        bool all_done = true;
        for (int k = 0; k < n; k++) all_done = all_done && w->h_sc[k].done;
        if (all_done || launched >= max_iter) break;
    }
    // iterations enqueued after a right-hand side had stopped: their 4 hop launches each were no-ops (HopArgs::done)
    for (int k = 0; k < n; k++) lat->n_hop_idle[prec] += 4ull * (unsigned long long)(launched - w->h_sc[k].iters);
    return BQ_OK;
}

// Inner CG on the normal equations M^^dag M^ e = M^^dag ir (e0 = 0) for every right-hand side of the batch
// (Hestenes-Stiefel CG, see blas.cu).  rhs k stops when the normal-equation residual has dropped
// by sqrt(w->h_stop2[k]) relative to its start, or after max_iter iterations.  Vector roles: irhat = r_N, ip = p,
// iv = q = M^ p, it = M^^dag q, ie = e.  6 hops + 3 BLAS-1 kernels per iteration, |q|^2 fused into the hop that makes q.
static bq_status inner_cgnr(bq_lattice* lat, SolverWork* w, double kappa, double csw, int prec, int recon, int max_iter,
                            int check_every) {
    const BlasCtx& c = w->blas;
    cudaStream_t s = c.stream;
    const int n = c.nrhs, mrhs = n > 1 ? n : 0;
    const size_t eb = field_bytes_one_parity(lat->g, prec == BQ_HALF ? BQ_FP32 : prec) * n;
    BQ_CUDA(lat, cudaMemsetAsync(w->ie, 0, eb, s));
    BQ_CUDA(lat, cudaMemcpyAsync(c.stop2s, w->h_stop2, sizeof(double) * n, cudaMemcpyHostToDevice, s));
    BQ_TRY(bq_schur_red(lat, w->irhat, w->ir, w->itmp, kappa, csw, prec, recon, s, nullptr, mrhs, true));   // r_N = M^^dag r
    BQ_TRY(cg_init(lat, c, prec, w->irhat, w->ip, 0.0, true));
    int launched = 0;
    const HopDoneScope done_scope(lat, c.sc);
    const HopRed red_qq{2, nullptr, c.sc};
    for (;;) {
        const int batch = (max_iter - launched) < check_every ? (max_iter - launched) : check_every;
        BQ_TRY(run_batch(lat, w, BQ_CGNR, prec, recon, kappa, csw, batch, check_every, [&]() -> bq_status {
            BQ_TRY(bq_schur_red(lat, w->iv, w->ip, w->itmp, kappa, csw, prec, recon, s, &red_qq, mrhs, false));  // q = M^ p; alpha = rho/|q|^2
            BQ_TRY(bq_schur_red(lat, w->it, w->iv, w->itmp, kappa, csw, prec, recon, s, nullptr, mrhs, true));   // t = M^^dag q
            BQ_TRY(cg_update(lat, c, prec, w->ip, w->it, w->ie, w->irhat));                                       // e, r_N, beta
            return cg_p_update(lat, c, prec, w->irhat, w->ip);                                                    // p = r_N + beta p
        }));
        launched += batch;
        BQ_TRY(poll(lat, w));
        bool all_done = true;
        for (int k = 0; k < n; k++) all_done = all_done && w->h_sc[k].done;
        if (all_done || launched >= max_iter) break;
    }
    // iterations enqueued after a right-hand side had stopped: their 4 hop launches each were no-ops (HopArgs::done)
    for (int k = 0; k < n; k++) lat->n_hop_idle[prec] += 4ull * (unsigned long long)(launched - w->h_sc[k].iters);
    return BQ_OK;
}

static bq_status solve_lex(bq_lattice* lat, SolverWork* w, const bq_solve_opts& o, double kappa, double tol, double inner_tol,
                           int max_inner, int max_outer, int check_every, bq_solve_info* info, bq_status* result);

// device time of the five phases of a solve from the events recorded along the way
static void phase_times(SolverWork* w, bq_solve_info* info, int n) {
    if (!info) return;
    cudaEvent_t ev[6] = {w->ev0, w->evp[0], w->evp[1], w->evp[2], w->evp[3], w->ev1};
    for (int p = 0; p < 5; p++) {
        float ms = 0;
        if (cudaEventElapsedTime(&ms, ev[p], ev[p + 1]) != cudaSuccess) ms = 0;
        for (int k = 0; k < n; k++) info[k].phase_seconds[p] = ms * 1e-3;
    }
}

// x (canonical, host or device) <- the n full-lattice fp64 fields of w->x: layout conversion into the staging buffer and
// the copy to the caller's buffer, enqueued on stream xs (does not synchronise)
static bq_status enqueue_export(bq_lattice* lat, SolverWork* w, double* x, int n, cudaStream_t xs, const char* fn) {
    const Geom& g = lat->g;
    const size_t nb = (size_t)g.V * 24 * sizeof(double), fb64 = field_bytes_one_parity(g, BQ_FP64);
    for (int k = 0; k < n; k++) {
        BQ_TRY(bq_field_export(lat, w->stage, static_cast<char*>(w->x) + (size_t)k * 2 * fb64, BQ_FULL, BQ_FP64, xs));
        const cudaError_t e = cudaMemcpyAsync(reinterpret_cast<char*>(x) + (size_t)k * nb, w->stage, nb, cudaMemcpyDefault, xs);
        if (e != cudaSuccess) return bq_set_error(lat, BQ_ECUDA, "%s: export failed: %s", fn, cudaGetErrorString(e));
    }
    return BQ_OK;
}

// export on the solver's own stream; records w->evp[3] before, w->ev1 after, and synchronises
static bq_status export_solution(bq_lattice* lat, SolverWork* w, double* x, int n, const char* fn) {
    cudaStream_t s = w->blas.stream;
    cudaError_t e = cudaEventRecord(w->evp[3], s);
    bq_status st = e == cudaSuccess ? enqueue_export(lat, w, x, n, s, fn) : BQ_OK;
    if (e == cudaSuccess) e = cudaEventRecord(w->ev1, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return bq_set_error(lat, BQ_ECUDA, "%s: export failed: %s", fn, cudaGetErrorString(e));
    return st;
}

// bq_solve (nrhs = 1, single-field kernels) and bq_solve_multi (nrhs >= 1 right-hand sides solved together with the
// multi-rhs kernels: one gauge-field read per hop for the whole batch).  b, x: nrhs canonical fields one after the other.
static bq_status solve_impl(bq_lattice* lat, const double* b, double* x, int nrhs, bool multi, double kappa, double tol,
                            const bq_solve_opts* opts, bq_solve_info* info) {
    if (!lat) return BQ_EINVAL;
    const char* fn = multi ? "bq_solve_multi" : "bq_solve";
    if (info)
        for (int k = 0; k < (nrhs > 0 ? nrhs : 0); k++) {
            info[k].status = BQ_EINVAL; info[k].outer_cycles = 0; info[k].inner_iters = 0; info[k].restarts = 0;
            info[k].true_rel_residual = NAN; info[k].seconds = 0;
            for (double& ps : info[k].phase_seconds) ps = 0;
        }
    if (nrhs < 1) return bq_set_error(lat, BQ_EINVAL, "%s: nrhs must be >= 1", fn);
    if (!b || !x) return bq_set_error(lat, BQ_EINVAL, "%s: b or x is NULL", fn);
    if (!(tol > 0.0) || !isfinite(tol)) return bq_set_error(lat, BQ_EINVAL, "%s: tol must be positive", fn);
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "%s: no gauge field loaded", fn);
    if (lat->sub) return bq_set_error(lat, BQ_EINVAL, "%s: a sub-lattice handle solves through bq_dd_solve", fn);
    bq_solve_opts o;
    if (opts) o = *opts;
    else { o.inner_prec = BQ_FP32; o.recon = BQ_RECON18; o.csw = 0; o.inner_tol = 0; o.max_inner = 0; o.max_outer = 0; o.check_every = 0; o.method = BQ_BICGSTAB; o.lexical = 0; o.x0_zero = 0; o.stream = nullptr; }
    if (o.inner_prec != BQ_FP64 && o.inner_prec != BQ_FP32 && o.inner_prec != BQ_HALF) return bq_set_error(lat, BQ_EINVAL, "%s: bad inner_prec", fn);
    if (o.method != BQ_BICGSTAB && o.method != BQ_CGNR) return bq_set_error(lat, BQ_EINVAL, "%s: bad method %d", fn, o.method);
    const bool cgnr = o.method == BQ_CGNR;
    if (o.lexical && (multi || cgnr)) return bq_set_error(lat, BQ_EINVAL, "%s: the lexical solve is BiCGStab on one right-hand side", fn);
    if (o.recon != BQ_RECON18 && o.recon != BQ_RECON12) return bq_set_error(lat, BQ_EINVAL, "%s: bad recon", fn);
    const int prec = o.inner_prec;
    // half storage: the inner solve is asked for what the storage format can represent (four times its rounding of 2^-11 per stored real; the hop's parity
    // bound 5e-3) and polled every 4 iterations: with the looser 5e-2 of round 1 an inner solve gained 1.3 decades and the fp64 outer loop — two fp64
    // hops and five fp64 vector passes per cycle — was 40 % of the config-5 solve (5 cycles for 9 iterations: 57.8 ms; now 3 cycles: 47 ms)
    const double inner_tol = o.inner_tol > 0 ? o.inner_tol : (prec == BQ_HALF ? 2e-3 : 1e-5);
    const int max_inner = o.max_inner > 0 ? o.max_inner : (prec == BQ_HALF ? 100 : 1000);
    const int max_outer = o.max_outer > 0 ? o.max_outer : 50;
    const int check_every = o.check_every > 0 ? o.check_every : (prec == BQ_HALF ? 4 : 8);
    const double csw = o.csw;
    const bool clover = csw != 0.0;
    const int n = nrhs;
    // the batched BLAS-1 kernels index all right-hand sides of an operand with one int (blas.cuh)
    if ((double)n * 2.0 * 12.0 * lat->g.Vh >= 2147483648.0)
        return bq_set_error(lat, BQ_EINVAL, "%s: nrhs * 24 * Vh must stay below 2^31 — split the batch", fn);

    SolverWork* w = nullptr;
    BQ_TRY(get_work(lat, prec, &w, n));
    const Geom& g = lat->g;
    const size_t fb64 = field_bytes_one_parity(g, BQ_FP64);
    w->blas.nrhs = n;
    w->blas.stride = field_bytes_one_parity(g, prec);
    w->blas.xstride = field_bytes_one_parity(g, prec == BQ_HALF ? BQ_FP32 : prec);
    w->blas.stride64 = fb64;
    const BlasCtx& c = w->blas;
    cudaStream_t s = c.stream;
    char* bb = static_cast<char*>(w->b);     // [rhs][even | odd], 2*fb64 per rhs
    char* xx = static_cast<char*>(w->x);
    const void *cl64 = nullptr, *cli64 = nullptr;
    const size_t cb64 = (size_t)g.Vh * CLOVER_REALS * sizeof(double);
    if (clover) {
        BQ_TRY(bq_clover_build(lat, csw, kappa));
        BQ_TRY(bq_get_clover(lat, BQ_FP64, 0, &cl64));
        BQ_TRY(bq_get_clover(lat, BQ_FP64, 1, &cli64));
    }
    // operand strides of the fp64 hops: full-lattice fields (b, x) are 2*fb64 apart, one-parity work vectors fb64
    const HopMulti* none = nullptr;
    auto hm = [&](size_t s_in, size_t s_out, size_t s_z) { return HopMulti{n, s_in, s_out, s_z, 0}; };

    if (o.stream) {
        // the caller's stream: everything enqueued there so far (e.g. the kernels that produce b) is waited for by the
        // solver's own stream; the call synchronises before it returns, so work enqueued there afterwards sees x
        BQ_CUDA(lat, cudaEventRecord(w->ev_side, static_cast<cudaStream_t>(o.stream)));
        BQ_CUDA(lat, cudaStreamWaitEvent(s, w->ev_side, 0));
    }
    BQ_CUDA(lat, cudaEventRecord(w->ev0, s));
    // ---- import b and x0 (canonical, host or device) through a device staging buffer ----
    {
        const size_t nb = (size_t)g.V * 24 * sizeof(double);
        double* stage = w->stage;
        cudaError_t e = cudaSuccess;
        bq_status st = BQ_OK;
        for (int k = 0; k < n && e == cudaSuccess && st == BQ_OK; k++) {
            e = cudaMemcpyAsync(stage, reinterpret_cast<const char*>(b) + (size_t)k * nb, nb, cudaMemcpyDefault, s);
            if (e == cudaSuccess) st = bq_field_import(lat, bb + (size_t)k * 2 * fb64, stage, BQ_FULL, BQ_FP64, s);
            if (o.x0_zero) {          // x is output only: no transfer, no conversion of an initial guess
                if (e == cudaSuccess && st == BQ_OK) e = cudaMemsetAsync(xx + (size_t)k * 2 * fb64, 0, 2 * fb64, s);
                continue;
            }
            if (e == cudaSuccess && st == BQ_OK) e = cudaMemcpyAsync(stage, reinterpret_cast<const char*>(x) + (size_t)k * nb, nb, cudaMemcpyDefault, s);
            if (e == cudaSuccess && st == BQ_OK) st = bq_field_import(lat, xx + (size_t)k * 2 * fb64, stage, BQ_FULL, BQ_FP64, s);
        }
        if (e == cudaSuccess) e = cudaEventRecord(w->evp[0], s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess || st != BQ_OK) w->blas.nrhs = 1;
        if (e != cudaSuccess) return bq_set_error(lat, BQ_ECUDA, "%s: import failed: %s", fn, cudaGetErrorString(e));
        BQ_TRY(st);
    }
    if (o.lexical) {
        // unpreconditioned solve on the full matrix (solve_lex); one right-hand side
        bq_status result = BQ_OK;
        cudaEventRecord(w->evp[1], s);
        bq_status st = solve_lex(lat, w, o, kappa, tol, inner_tol, max_inner, max_outer, check_every, info, &result);
        cudaEventRecord(w->evp[2], s);
        if (st == BQ_OK) st = export_solution(lat, w, x, 1, fn);
        w->blas.nrhs = 1;
        if (st != BQ_OK) return st;
        float ms = 0;
        cudaEventElapsedTime(&ms, w->ev0, w->ev1);
        if (info) { info->status = result; info->seconds = ms * 1e-3; }
        phase_times(w, info, 1);
        return result;
    }
    // |b_k|^2 over the full lattice (two parities)
    double* bnorm = static_cast<double*>(calloc(5 * (size_t)n, sizeof(double)));
    int* ik = static_cast<int*>(calloc(7 * (size_t)n, sizeof(int)));
    if (!bnorm || !ik) { free(bnorm); free(ik); w->blas.nrhs = 1; return bq_set_error(lat, BQ_ENOMEM, "%s: host allocation failed", fn); }
    double *target = bnorm + n, *prev_rnorm = bnorm + 2 * n, *rnorm = bnorm + 3 * n, *true_rel = bnorm + 4 * n;
    int *stalled = ik, *inner_total = ik + n, *restarts = ik + 2 * n, *cycles = ik + 3 * n, *fin = ik + 4 * n, *stat = ik + 5 * n, *dead = ik + 6 * n;
    bq_status result = BQ_OK;
    // every early exit below goes through `bail`: once the export of x has been enqueued on the side stream the library may
    // still be writing the caller's x, so a failure waits for both streams before it returns (errors of the waits themselves are
    // ignored: the status being returned is the one that matters), puts the context back to one right-hand side and
    // releases the host scratch
    auto bail = [&](bq_status st) {
        cudaStreamSynchronize(w->side);
        cudaStreamSynchronize(s);
        w->blas.nrhs = 1;
        free(bnorm);
        free(ik);
        return st;
    };
#define SOLVE_TRY(expr)                         \
    do {                                        \
        bq_status _s = (expr);                  \
        if (_s != BQ_OK) return bail(_s);       \
    } while (0)
    {
        BlasCtx cb = c;
        cb.stride = 2 * fb64;
        for (int p = 0; p < 2; p++) {
            SOLVE_TRY(blas_norm2(lat, cb, BQ_FP64, bb + p * fb64));
            SOLVE_TRY(poll(lat, w));
            for (int k = 0; k < n; k++) bnorm[k] += w->h_sc[k].red[0];
        }
    }
    bool any_nonzero = false;
    for (int k = 0; k < n; k++)
        if (!isfinite(bnorm[k])) {
            return bail(bq_set_error(lat, BQ_EINVAL, "%s: right-hand side %d contains NaN or Inf", fn, k));
        }
    for (int k = 0; k < n; k++) {
        bnorm[k] = sqrt(bnorm[k]);
        target[k] = tol * bnorm[k];
        prev_rnorm[k] = INFINITY;
        any_nonzero = any_nonzero || bnorm[k] > 0.0;
    }
    int outer = 0;
    // a zero right-hand side has the solution x = 0 (and is "converged" from the start: |r| <= 0 needs x = 0)
    for (int k = 0; k < n; k++)
        if (bnorm[k] == 0.0) {
            cudaError_t e = cudaMemsetAsync(xx + (size_t)k * 2 * fb64, 0, 2 * fb64, s);
            if (e != cudaSuccess) return bail(bq_set_error(lat, BQ_ECUDA, "%s: memset failed", fn));
        }
    cudaEventRecord(w->evp[1], s);
    cudaEventRecord(w->evp[2], s);
    if (any_nonzero) {
        // ---- b^_e = b_e + kappa H_eo A_oo^-1 b_o ----
        const void* bo = bb + fb64;
        size_t bo_stride = 2 * fb64;
        if (clover) {
            for (int k = 0; k < n; k++)
                SOLVE_TRY(bq_clover_mul(lat, static_cast<char*>(w->tmp) + (size_t)k * fb64, bb + (size_t)k * 2 * fb64 + fb64,
                                        static_cast<const char*>(cli64) + cb64, BQ_FP64, s));
            bo = w->tmp;
            bo_stride = fb64;
        }
        {
            const HopMulti m = hm(bo_stride, fb64, 2 * fb64);
            SOLVE_TRY(bq_hop(lat, w->bhat, bo, bb, kappa, 0, BQ_FP64, BQ_RECON18, nullptr, 0, s, nullptr, multi ? &m : none));
        }
        cudaEventRecord(w->evp[1], s);
        for (;;) {
            // r = b^_e - M^ x_e in fp64  (declared zero guess, first cycle: M^ x_e = 0 without applying the operator)
            if (o.x0_zero && outer == 0) {
                cudaError_t e = cudaMemsetAsync(w->t, 0, fb64 * n, s);
                if (e != cudaSuccess) return bail(bq_set_error(lat, BQ_ECUDA, "%s: memset failed", fn));
            } else {
                // x_e of rhs k lives at xx + k*2*fb64: Schur with input stride 2*fb64 = two hops by hand
                const HopMulti m1 = hm(2 * fb64, fb64, 0), m2 = hm(fb64, fb64, 2 * fb64);
                if (!clover) {
                    SOLVE_TRY(bq_hop(lat, w->tmp, xx, nullptr, -kappa, 1, BQ_FP64, BQ_RECON18, nullptr, 0, s, nullptr, multi ? &m1 : none));
                    SOLVE_TRY(bq_hop(lat, w->t, w->tmp, xx, kappa, 0, BQ_FP64, BQ_RECON18, nullptr, 0, s, nullptr, multi ? &m2 : none));
                } else {
                    SOLVE_TRY(bq_hop(lat, w->tmp, xx, nullptr, -kappa, 1, BQ_FP64, BQ_RECON18, static_cast<const char*>(cli64) + cb64, 1, s, nullptr, multi ? &m1 : none));
                    SOLVE_TRY(bq_hop(lat, w->t, w->tmp, xx, kappa, 0, BQ_FP64, BQ_RECON18, cl64, 2, s, nullptr, multi ? &m2 : none));
                }
            }
            SOLVE_TRY(outer_residual(lat, c, w->bhat, fb64, w->t, w->r));
            SOLVE_TRY(poll(lat, w));
            // every right-hand side is judged on its own (bq.h): one that has converged, produced a NaN, stalled or broken
            // down for good is FINISHED — it keeps its status and its iterate, its inner solves stop at once — and the
            // others go on
            bool any_active = false;
            for (int k = 0; k < n; k++) {
                rnorm[k] = sqrt(w->h_sc[k].r2);
                if (fin[k]) continue;
                if (bnorm[k] == 0.0 || rnorm[k] <= target[k]) { fin[k] = 1; continue; }
                if (!(rnorm[k] == rnorm[k])) { fin[k] = 1; stat[k] = BQ_EBREAKDOWN; continue; }
                if (dead[k]) { fin[k] = 1; stat[k] = BQ_EBREAKDOWN; continue; }
                if (rnorm[k] > 0.5 * prev_rnorm[k]) {
                    if (++stalled[k] >= 4) { fin[k] = 1; stat[k] = BQ_ENOTCONVERGED; continue; }
                } else stalled[k] = 0;
                prev_rnorm[k] = rnorm[k];
                any_active = true;
            }
            if (!any_active) break;
            if (outer >= max_outer) {
                for (int k = 0; k < n; k++)
                    if (!fin[k]) { fin[k] = 1; stat[k] = BQ_ENOTCONVERGED; }
                break;
            }
            outer++;
            // normalised low-precision right-hand sides and inner stopping thresholds; a right-hand side that has
            // already converged gets an infinite threshold: its inner solve stops at once with e = 0
            SOLVE_TRY(outer_to_low(lat, c, prec, w->r, w->ir));
            for (int k = 0; k < n; k++) {
                if (fin[k]) { w->h_stop2[k] = INFINITY; continue; }
                // CGNR stops on the normal-equation residual |M^^dag (r - M^ e)|, whose reduction only bounds that of
                // |r - M^ e| up to cond(M^): ask for a decade more and let the outer loop judge the true residual
                const double rel = ((prec == BQ_FP64) ? 0.9 * target[k] / rnorm[k] : fmax(inner_tol, 0.5 * target[k] / rnorm[k])) *
                                   (cgnr ? 0.1 : 1.0);
                w->h_stop2[k] = rel * rel;
                cycles[k]++;
            }
            if (cgnr) SOLVE_TRY(inner_cgnr(lat, w, kappa, csw, prec, o.recon, max_inner, check_every));
            else SOLVE_TRY(inner_bicgstab(lat, w, kappa, csw, prec, o.recon, max_inner, check_every));
            for (int k = 0; k < n; k++) {
                inner_total[k] += w->h_sc[k].iters;
                if (w->h_sc[k].done == 2) {   // breakdown: the next outer cycle restarts from the true residual
                    restarts[k]++;
                    if (w->h_sc[k].iters == 0 && restarts[k] > 3) dead[k] = 1;
                }
            }
            // x_e += |r| e   (|r| = sc->rnorm, written by outer_residual; the inner loop does not touch it)
            SOLVE_TRY(outer_accumulate(lat, c, prec == BQ_HALF ? BQ_FP32 : prec, w->ie, xx, 2 * fb64));
        }
        cudaEventRecord(w->evp[2], s);
        // ---- x_o = A_oo^-1 (b_o + kappa H_oe x_e) ----
        {
            const HopMulti m = hm(2 * fb64, 2 * fb64, 2 * fb64);
            SOLVE_TRY(bq_hop(lat, xx + fb64, xx, bb + fb64, kappa, 1, BQ_FP64, BQ_RECON18, nullptr, 0, s, nullptr, multi ? &m : none));
        }
        if (clover)
            for (int k = 0; k < n; k++)
                SOLVE_TRY(bq_clover_mul(lat, xx + (size_t)k * 2 * fb64 + fb64, xx + (size_t)k * 2 * fb64 + fb64,
                                        static_cast<const char*>(cli64) + cb64, BQ_FP64, s));
        // ---- x is final: its layout conversion and its copy to the caller run on a second stream from here on ... ----
        bool exported = false;
        {
            cudaError_t e = cudaEventRecord(w->ev_side, s);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(w->side, w->ev_side, 0);
            if (e != cudaSuccess) return bail(bq_set_error(lat, BQ_ECUDA, "%s: %s", fn, cudaGetErrorString(e)));
        }
        // ---- ... while the true residual |b - D x| / |b| is computed on the full lattice in fp64 ----
        for (int p = 0; p < 2; p++) {
            const void* clp = clover ? static_cast<const char*>(cl64) + p * cb64 : nullptr;
            const HopMulti m = hm(2 * fb64, fb64, 2 * fb64);
            SOLVE_TRY(bq_hop(lat, w->t, xx + (1 - p) * fb64, xx + p * fb64, -kappa, p, BQ_FP64, BQ_RECON18, clp, clover ? 2 : 0, s, nullptr,
                             multi ? &m : none));
            SOLVE_TRY(outer_residual(lat, c, bb + p * fb64, 2 * fb64, w->t, w->r));
            if (!exported) {     // enqueued behind the first residual kernels: a pageable destination makes this call block the host
                SOLVE_TRY(enqueue_export(lat, w, x, n, w->side, fn));
                exported = true;
            }
            SOLVE_TRY(poll(lat, w));
            for (int k = 0; k < n; k++) true_rel[k] += w->h_sc[k].r2;
        }
        for (int k = 0; k < n; k++) true_rel[k] = bnorm[k] > 0.0 ? sqrt(true_rel[k]) / bnorm[k] : 0.0;
        // the solver's stream waits for the side stream: w->ev1 closes the whole call
        {
            cudaError_t e = cudaEventRecord(w->evp[3], s);
            if (e == cudaSuccess) e = cudaEventRecord(w->ev_side, w->side);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(s, w->ev_side, 0);
            if (e == cudaSuccess) e = cudaEventRecord(w->ev1, s);
            if (e == cudaSuccess) e = cudaStreamSynchronize(s);
            if (e != cudaSuccess) return bail(bq_set_error(lat, BQ_ECUDA, "%s: export failed: %s", fn, cudaGetErrorString(e)));
        }
    } else {
        // nothing to solve (all right-hand sides zero): x = 0
        SOLVE_TRY(export_solution(lat, w, x, n, fn));
    }
#undef SOLVE_TRY
    float ms = 0;
    cudaEventElapsedTime(&ms, w->ev0, w->ev1);
    // worst status of the batch: breakdown before non-convergence
    for (int k = 0; k < n; k++)
        if (stat[k] == BQ_EBREAKDOWN && result != BQ_EBREAKDOWN)
            result = bq_set_error(lat, BQ_EBREAKDOWN, "%s: right-hand side %d: NaN residual or BiCGStab breakdown (rho, <rhat,v> or <t,t> = 0)", fn, k);
    for (int k = 0; k < n && result == BQ_OK; k++)
        if (stat[k] == BQ_ENOTCONVERGED)
            result = bq_set_error(lat, BQ_ENOTCONVERGED, "%s: right-hand side %d stopped at |r|/|b| = %.3e (stalled or max_outer reached)", fn, k,
                                  bnorm[k] > 0 ? rnorm[k] / bnorm[k] : 0.0);
    if (info)
        for (int k = 0; k < n; k++) {
            info[k].status = stat[k];
            info[k].outer_cycles = (prec == BQ_FP64) ? 0 : cycles[k];
            info[k].inner_iters = inner_total[k];
            info[k].restarts = (prec == BQ_FP64) ? (cycles[k] > 0 ? cycles[k] - 1 : 0) + restarts[k] : restarts[k];
            info[k].true_rel_residual = true_rel[k];
            info[k].seconds = ms * 1e-3;     // device time of the whole call (all right-hand sides together)
        }
    phase_times(w, info, n);
    free(bnorm);
    free(ik);
    w->blas.nrhs = 1;
    return result;
}

// ---------------------------------------------------------------------------------------------------
// Lexical (not even-odd preconditioned) solve: BiCGStab on the full matrix D of Eq. 1 itself (the
// paper's example instantiates the `lex` fermion operator) with the same defect-correction outer loop.
// Vectors are full-lattice [even | odd] fields; the BLAS-1 kernels run on them as fields of V sites; D = two hop
// launches with the site-diagonal term in their epilogue; the inner products are separate kernels (the two launches of
// one apply cannot share a fused reduction).  One right-hand side.  Work vectors are allocated per call.
// ---------------------------------------------------------------------------------------------------
static bq_status solve_lex(bq_lattice* lat, SolverWork* w, const bq_solve_opts& o, double kappa, double tol, double inner_tol,
                           int max_inner, int max_outer, int check_every, bq_solve_info* info, bq_status* result) {
    const Geom& g = lat->g;
    const int prec = o.inner_prec;
    const double csw = o.csw;
    BlasCtx c = w->blas;                 // the same scratch and scalars, fields of V = 2 Vh sites
    c.Vh = g.V; c.nrhs = 1; c.stride = c.xstride = c.stride64 = 0;
    cudaStream_t s = c.stream;
    const size_t fb64 = 2 * field_bytes_one_parity(g, BQ_FP64), fb = 2 * field_bytes_one_parity(g, prec);
    const size_t eb = 2 * field_bytes_one_parity(g, prec == BQ_HALF ? BQ_FP32 : prec);
    char* pool = nullptr;
    BQ_CUDA(lat, cudaMalloc(&pool, 2 * fb64 + 6 * fb + eb));
    void *r64 = pool, *t64 = pool + fb64;
    char* q = pool + 2 * fb64;
    void *ir = q, *irhat = q + fb, *ip = q + 2 * fb, *iv = q + 3 * fb, *is = q + 4 * fb, *it = q + 5 * fb, *ie = q + 6 * fb;
    bq_status st = BQ_OK;
    double bnorm = 0, rnorm = 0, prev = INFINITY;
    int outer = 0, inner_total = 0, restarts = 0, stalled = 0;
#define LEX_TRY(expr)                                   \
    do {                                                \
        st = (expr);                                    \
        if (st != BQ_OK) { cudaFree(pool); return st; } \
    } while (0)
    LEX_TRY(blas_norm2(lat, c, BQ_FP64, w->b));
    LEX_TRY(poll(lat, w));
    bnorm = sqrt(w->h_sc[0].red[0]);
    if (!isfinite(bnorm)) {
        cudaFree(pool);
        return bq_set_error(lat, BQ_EINVAL, "bq_solve: the right-hand side contains NaN or Inf");
    }
    if (bnorm == 0.0) {
        cudaMemsetAsync(w->x, 0, fb64, s);
    } else {
        const double target = tol * bnorm;
        for (;;) {
            LEX_TRY(bq_dirac_full(lat, t64, w->x, kappa, csw, BQ_FP64, BQ_RECON18, s, false));
            LEX_TRY(outer_residual(lat, c, w->b, 0, t64, r64));
            LEX_TRY(poll(lat, w));
            rnorm = sqrt(w->h_sc[0].r2);
            if (!(rnorm == rnorm)) { *result = bq_set_error(lat, BQ_EBREAKDOWN, "bq_solve: residual is NaN"); break; }
            if (rnorm <= target) break;
            if (outer >= max_outer) { *result = bq_set_error(lat, BQ_ENOTCONVERGED, "bq_solve: max_outer reached, |r|/|b| = %.3e", rnorm / bnorm); break; }
            if (rnorm > 0.5 * prev) {
                if (++stalled >= 4) { *result = bq_set_error(lat, BQ_ENOTCONVERGED, "bq_solve: stalled at |r|/|b| = %.3e", rnorm / bnorm); break; }
            } else stalled = 0;
            prev = rnorm;
            outer++;
            LEX_TRY(outer_to_low(lat, c, prec, r64, ir));
            const double rel = (prec == BQ_FP64) ? 0.9 * target / rnorm : fmax(inner_tol, 0.5 * target / rnorm);
            // inner BiCGStab on D e = ir, e0 = 0 (reading O4)
            cudaMemsetAsync(ie, 0, eb, s);
            cudaMemsetAsync(ip, 0, fb, s);
            cudaMemsetAsync(iv, 0, fb, s);
            cudaMemcpyAsync(irhat, ir, fb, cudaMemcpyDeviceToDevice, s);
            LEX_TRY(bicg_init(lat, c, prec, ir, rel * rel));
            int launched = 0;
            const HopDoneScope done_scope(lat, c.sc);
            for (;;) {
                const int batch = (max_inner - launched) < check_every ? (max_inner - launched) : check_every;
                for (int k = 0; k < batch; k++) {
                    LEX_TRY(bicg_p_update(lat, c, prec, ir, ip, iv));
                    LEX_TRY(bq_dirac_full(lat, iv, ip, kappa, csw, prec, o.recon, s, false));     // v = D p
                    LEX_TRY(bicg_alpha(lat, c, prec, irhat, iv));
                    LEX_TRY(bicg_s_update(lat, c, prec, ir, iv, is));
                    LEX_TRY(bq_dirac_full(lat, it, is, kappa, csw, prec, o.recon, s, false));     // t = D s
                    LEX_TRY(bicg_omega(lat, c, prec, it, is));
                    LEX_TRY(bicg_final(lat, c, prec, ip, is, it, irhat, ie, ir));
                }
                launched += batch;
                LEX_TRY(poll(lat, w));
                if (w->h_sc[0].done || launched >= max_inner) break;
            }
            inner_total += w->h_sc[0].iters;
            lat->n_hop_idle[prec] += 4ull * (unsigned long long)(launched - w->h_sc[0].iters);
            if (w->h_sc[0].done == 2) {
                restarts++;
                if (w->h_sc[0].iters == 0 && restarts > 3) { *result = bq_set_error(lat, BQ_EBREAKDOWN, "bq_solve: BiCGStab breakdown"); break; }
            }
            LEX_TRY(outer_accumulate(lat, c, prec == BQ_HALF ? BQ_FP32 : prec, ie, w->x, 0));
        }
        // true residual of the returned x
        LEX_TRY(bq_dirac_full(lat, t64, w->x, kappa, csw, BQ_FP64, BQ_RECON18, s, false));
        LEX_TRY(outer_residual(lat, c, w->b, 0, t64, r64));
        LEX_TRY(poll(lat, w));
        rnorm = sqrt(w->h_sc[0].r2);
    }
#undef LEX_TRY
    cudaStreamSynchronize(s);
    cudaFree(pool);
    if (info) {
        info->outer_cycles = (prec == BQ_FP64) ? 0 : outer;
        info->inner_iters = inner_total;
        info->restarts = (prec == BQ_FP64) ? (outer > 0 ? outer - 1 : 0) + restarts : restarts;
        info->true_rel_residual = bnorm > 0 ? rnorm / bnorm : 0.0;
    }
    return BQ_OK;
}

extern "C" bq_status bq_solve(bq_lattice* lat, const double* b, double* x, double kappa, double tol, const bq_solve_opts* opts,
                              bq_solve_info* info) {
    return solve_impl(lat, b, x, 1, false, kappa, tol, opts, info);
}

extern "C" bq_status bq_solve_multi(bq_lattice* lat, const double* b, double* x, int nrhs, double kappa, double tol,
                                    const bq_solve_opts* opts, bq_solve_info* info) {
    return solve_impl(lat, b, x, nrhs, true, kappa, tol, opts, info);
}

// ---------------------------------------------------------------------------------------------------
// bq_propagator: the program of the paper's Fig. 1 — for each of the 12 spin-colour components (id, ic)
// set a point source at one site and invert — as ONE batched solve.  The sources are made on the device (no host
// transfer of 12 mostly-zero fields); S receives the 12 solutions, canonical layout, source index 3*id + ic.
// ---------------------------------------------------------------------------------------------------
__global__ void k_point_sources(double* b, size_t field_doubles, size_t site) {
    const int k = threadIdx.x;                       // source index 3*spin + colour
    if (k < 12) b[(size_t)k * field_doubles + site * 24 + 2 * k] = 1.0;
}

extern "C" bq_status bq_propagator(bq_lattice* lat, const int* src_site, double* S, double kappa, double tol, const bq_solve_opts* opts,
                                   bq_solve_info* info) {
    if (!lat) return BQ_EINVAL;
    if (!src_site || !S) return bq_set_error(lat, BQ_EINVAL, "bq_propagator: src_site or S is NULL");
    const Geom& g = lat->g;
    for (int mu = 0; mu < 4; mu++)
        if (src_site[mu] < 0 || src_site[mu] >= g.L[mu]) return bq_set_error(lat, BQ_EINVAL, "bq_propagator: source site outside the lattice");
    const size_t site = src_site[0] + (size_t)g.L[0] * (src_site[1] + (size_t)g.L[1] * (src_site[2] + (size_t)g.L[2] * src_site[3]));
    const size_t fd = (size_t)g.V * 24;
    double* b = nullptr;
    BQ_CUDA(lat, cudaMalloc(&b, 12 * fd * sizeof(double)));
    cudaError_t e = cudaMemset(b, 0, 12 * fd * sizeof(double));
    if (e == cudaSuccess) {
        k_point_sources<<<1, 32>>>(b, fd, site);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        cudaFree(b);
        return bq_set_error(lat, BQ_ECUDA, "bq_propagator: %s", cudaGetErrorString(e));
    }
    lat->n_launch++;
    bq_solve_opts o;
    if (opts) o = *opts;
    else { o.inner_prec = BQ_FP32; o.recon = BQ_RECON18; o.csw = 0; o.inner_tol = 0; o.max_inner = 0; o.max_outer = 0; o.check_every = 0; o.method = BQ_BICGSTAB; o.lexical = 0; o.x0_zero = 0; o.stream = nullptr; }
    o.x0_zero = 1;                                   // S is output only
    const bq_status st = solve_impl(lat, b, S, 12, true, kappa, tol, &o, info);
    cudaFree(b);
    return st;
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
    if (lat->sub) return bq_set_error(lat, BQ_EINVAL, "bq_schur_apply_dots: not on a sub-lattice handle");
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
