// blas_api.h — host launchers of the fused BLAS-1 kernels (blas.cu), used by the solver (solve.cu).
#pragma once

#include "bq_internal.h"

struct SolverScalars;

struct BlasCtx {
    int Vh;
    int grid;                 // blocks per launch and right-hand side (multiple of the cluster size)
    double* partials;         // reduction scratch, [cap][pstride]
    unsigned int* ticket;     // [cap]
    SolverScalars* sc;        // device-resident solver states, [cap]
    double* stop2s;           // per-rhs stopping thresholds of bicg_init, [cap]
    int pstride, cap;
    cudaStream_t stream;
    // batch shape of the launches made through this context: nrhs right-hand sides (gridDim.y), operand fields
    // `stride` bytes apart (vectors of the call's storage precision), `xstride` (the solution accumulator of bicg_final /
    // the e operand of outer_accumulate), `stride64` (fp64 one-parity work vectors of the outer loop)
    int nrhs;
    size_t stride, xstride, stride64;
};

bq_status blas_ctx_create(bq_lattice* lat, BlasCtx* ctx);
bq_status blas_ctx_reserve(bq_lattice* lat, BlasCtx* ctx, int nrhs);
void blas_ctx_destroy(BlasCtx* ctx);
static inline BlasCtx blas_single(const BlasCtx& c) { BlasCtx o = c; o.nrhs = 1; return o; }

// --- generic (results land in sc->red[], no host sync) ---
bq_status blas_norm2(bq_lattice* lat, const BlasCtx& c, int prec, const void* a);                  // red[0] = |a|^2
bq_status blas_cdot(bq_lattice* lat, const BlasCtx& c, int prec, const void* a, const void* b);    // red[0..1] = <a,b>
bq_status blas_caxpy(bq_lattice* lat, const BlasCtx& c, int prec, double ar, double ai, const void* x, void* y);

// --- BiCGStab steps; scalars read from / written to c.sc ---
// set stop2 and reset the state; then r2 = |r|^2, rho = <rhat,r> = r2 (rhat == r), beta = rho, alpha = omega = 1
// per_rhs_stop2: thresholds from c.stop2s[rhs] (device) instead of `stop2`
bq_status bicg_init(bq_lattice* lat, const BlasCtx& c, int prec, const void* r, double stop2, bool per_rhs_stop2 = false);
bq_status bicg_p_update(bq_lattice* lat, const BlasCtx& c, int prec, const void* r, void* p, const void* v);
bq_status bicg_alpha(bq_lattice* lat, const BlasCtx& c, int prec, const void* rhat, const void* v);
bq_status bicg_s_update(bq_lattice* lat, const BlasCtx& c, int prec, const void* r, const void* v, void* s);
bq_status bicg_omega(bq_lattice* lat, const BlasCtx& c, int prec, const void* t, const void* s);
// x += alpha p + omega s ; r = s - omega t ; r2, rho', beta ; iters++ ; convergence / breakdown flag.
// For prec == BQ_HALF the accumulator x is an fp32 field (site layout), everything else half storage.
bq_status bicg_final(bq_lattice* lat, const BlasCtx& c, int prec, const void* p, const void* s, const void* t, const void* rhat,
                     void* x, void* r);

// --- CG on the normal equations M^dag M e = M^dag r; scalars in c.sc (rho = |r_N|^2) ---
// p = r_N; rho = |r_N|^2; stop2 = rel2 * rho (rel2 from c.stop2s[rhs] when per_rhs_rel2); marks the state as CG
bq_status cg_init(bq_lattice* lat, const BlasCtx& c, int prec, const void* rn, void* p, double rel2, bool per_rhs_rel2 = false);
// x += alpha p ; r_N -= alpha t ; rho' = |r_N|^2 ; beta = rho'/rho ; iters++ ; convergence flag   (x: as in bicg_final)
bq_status cg_update(bq_lattice* lat, const BlasCtx& c, int prec, const void* p, const void* t, void* x, void* rn);
// p = r_N + beta p
bq_status cg_p_update(bq_lattice* lat, const BlasCtx& c, int prec, const void* rn, void* p);

// --- outer (fp64) loop ---
// r = b - t (fp64); sc->r2 = red[0] = |r|^2; sc->scale = 1/|r| (0 if r == 0)
// b: fields bstride bytes apart (the full-lattice b of the true-residual check, or b^_e); t, r: c.stride64 apart
bq_status outer_residual(bq_lattice* lat, const BlasCtx& c, const void* b, size_t bstride, const void* t, void* r);
// lo = convert(r * sc->scale) into precision prec_lo (site-wise; half: per-site norm)
bq_status outer_to_low(bq_lattice* lat, const BlasCtx& c, int prec_lo, const void* r64, void* lo);
// x64 += |r| * e_lo   (|r| = sqrt(sc->r2)); e_prec = precision of e (fp32 accumulator when the inner solver is half)
bq_status outer_accumulate(bq_lattice* lat, const BlasCtx& c, int e_prec, const void* e, void* x64, size_t x64stride);
