// bq_internal.h — shared declarations of the CUDA implementation behind include/bq.h.
// Product code: shares nothing with oracle/ (the gamma-matrix algebra is hard-wired as spin projections
// in hop.cuh, typed in independently from SURVEY.md Appendix A.2).
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "bq.h"
#include "bq_test.h"

// ---------------------------------------------------------------------------------------------------
// Geometry.  Half index h = xh + Lxh*(y + Ly*(z + Lz*t)), xh = x >> 1.
// ---------------------------------------------------------------------------------------------------
struct Geom {
    int L[4];   // Lx, Ly, Lz, Lt
    int Lxh;    // Lx / 2
    int Vh;     // sites per parity
    int V;      // all sites
};

// reals per site / per link in each store
constexpr int SPINOR_REALS = 24;
constexpr int CLOVER_REALS = 72;  // 2 blocks x (6 real diagonal + 15 complex off-diagonal)
__host__ __device__ constexpr int link_reals(int recon) { return recon == BQ_RECON12 ? 12 : 18; }

__host__ __device__ constexpr size_t prec_real_bytes(int prec) { return prec == BQ_FP64 ? 8 : (prec == BQ_FP32 ? 4 : 2); }
// bytes per site of a spinor in precision prec (half: 48 B mantissas + 4 B norm)
__host__ __device__ constexpr size_t spinor_site_bytes(int prec) { return prec == BQ_FP64 ? 192 : (prec == BQ_FP32 ? 96 : 52); }

struct SolverWork;
struct SolverScalars;

struct bq_lattice {
    Geom g;
    double bc[8];            // 4 x (re, im)
    int bc_nontrivial[4];    // phase != 1 in that direction
    double* U_canon;         // device copy of the canonical fp64 gauge field (kept for the clover build)
    void* gauge[3][2];       // [prec][recon]: [parity][mu][link planes over Vh]
    bool have_gauge;
    // clover: [prec][inverse]: [parity][72 reals as planes over Vh]; fp64 always built first
    void* clover[3][2];
    bool have_clover;
    double clover_csw, clover_kappa;
    // domain decomposition (dd.cu; opt-in): a sub-lattice of a process grid.  sub == 0 for ordinary handles.
    int sub, grid[4], coords[4];
    void* dd;                // DdBufs: face buffers, side stream
    SolverWork* work;
    int* d_flag;             // device int scratch (singular-clover flag etc.)
    double* hop_partials;    // per-CTA partial sums of the hop kernel's fused reduction epilogues (lazily allocated)
    size_t hop_partials_cap; // doubles allocated there
    unsigned long long epoch;  // bumped whenever gauge or clover stores are freed: cached CUDA graphs of the solver hold their addresses
    int use_graphs;          // solver: replay the batches of inner iterations as CUDA graphs (default 1; env BQ_GRAPH=0 disables)
    int mrhs_patch;          // multi-rhs hop: 1 = patch mapping where the geometry allows (default), 0 = plain (env BQ_MRHS_PATCH)
    int hop_pdl;             // single-rhs hop: programmatic dependent launch when Vh <= this (default 262144; env BQ_PDL = 0 off, or a bound)
    int mrhs_ls;             // multi-rhs hop: 2 = link-stationary kernels (default): hop_ls.cuh for fp32 / half storage, the direction-split
                             // hop_lsp.cuh for fp64 with >= 8 right-hand sides; 1 = hop_ls.cuh only; 3 = hop_lsp.cuh wherever it applies;
                             // 0 = off (env BQ_MRHS_LS)
    int hop_small;           // single-rhs hop, fp32: the uncapped-register build of the kernel when Vh <= this (default 2 x SMs x 128 = 37888: every CTA resident at once; env BQ_HOP_SMALL)
    const SolverScalars* hop_done;   // set by the solver around its inner iterations: hop launches test these `done` flags (HopArgs::done)
    unsigned long long n_launch;      // kernels launched through this handle
    unsigned long long n_hop[3];      // hop applications (per right-hand side) per storage precision
    unsigned long long n_ls;          // launches of the link-stationary multi-rhs hop kernels (hop_ls.cuh, hop_lsp.cuh)
    unsigned long long n_lsp;         // of n_ls: direct (not graph-replayed) launches of the direction-split kernel (hop_lsp.cuh)
    unsigned long long n_hop_idle[3]; // of n_hop: applications enqueued in a batch of solver iterations after their right-hand side had
                                      // stopped — the kernel returned at entry (HopArgs::done), no flop was executed
    char err[512];
};

// ---------------------------------------------------------------------------------------------------
// Error plumbing
// ---------------------------------------------------------------------------------------------------
bq_status bq_set_error(bq_lattice* lat, bq_status s, const char* fmt, ...);

#define BQ_CUDA(lat, expr)                                                                              \
    do {                                                                                                \
        cudaError_t _e = (expr);                                                                        \
        if (_e != cudaSuccess)                                                                          \
            return bq_set_error((lat), _e == cudaErrorMemoryAllocation ? BQ_ENOMEM : BQ_ECUDA,          \
                                "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
    } while (0)

// after every kernel launch: count it (bq_get_counters) and pick up launch errors
#define BQ_CHECK_LAUNCH(lat)                 \
    do {                                     \
        (lat)->n_launch++;                   \
        BQ_CUDA((lat), cudaGetLastError());  \
    } while (0)

#define BQ_TRY(expr)                  \
    do {                                \
        bq_status _s = (expr);          \
        if (_s != BQ_OK) return _s;     \
    } while (0)

// ---------------------------------------------------------------------------------------------------
// Internal entry points shared between translation units
// ---------------------------------------------------------------------------------------------------
// gauge store of (prec, recon), built on first use from the fp64 18-real store
bq_status bq_get_gauge(bq_lattice* lat, int prec, int recon, const void** out);
// clover blocks of (prec, inverse), built on first use; requires bq_clover_build to have run
bq_status bq_clover_build(bq_lattice* lat, double csw, double kappa);
bq_status bq_get_clover(bq_lattice* lat, int prec, int inverse, const void** out);

// Hop with epilogue:  out_p = scale * H_{p,1-p} in  [+ z]   (z == nullptr: no xpay).
// Clover epilogues (cl != nullptr, 72-real blocks of parity p in precision prec):
//   cl_mode 1: out = scale * C (H in) [+ z]          (C = A^-1 blocks: the "A_oo^-1 H_oe" step)
//   cl_mode 2: out = C z + scale * H in               (C = A blocks: the "A_ee x - kappa^2 H ..." step)
// Fused reduction epilogue (xpay forms only), accumulated on the values before they are rounded to storage:
//   mode 1: <w, out> -> sc->rhat_v, sc->alpha = sc->rho / <w, out>;   mode 2: <out, z>, <out, out> -> sc->ts, tt, omega
struct HopRed {
    int mode;
    const void* w;
    SolverScalars* sc;
};
// Multi-rhs form: every operand is an array of nrhs one-parity fields, s_* bytes apart; red->sc is an array of nrhs
// SolverScalars (one BiCGStab state per right-hand side).
struct HopMulti {
    int nrhs;
    size_t s_in, s_out, s_z, s_w;
};
bq_status bq_hop(bq_lattice* lat, void* out, const void* in, const void* z, double scale, int out_parity, int prec,
                 int recon, const void* cl, int cl_mode, cudaStream_t stream, const HopRed* red = nullptr,
                 const HopMulti* multi = nullptr, bool dag = false /* hop of D^dagger: H^dag in place of H */);
// out_e = M^ in_e (see bq_schur_apply) with an optional fused reduction on out in the second hop
bq_status bq_schur_red(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw, int prec, int recon,
                       cudaStream_t stream, const HopRed* red, int nrhs = 0 /* 0: single field; >= 1: arrays of nrhs fields */,
                       bool dag = false /* M^^dagger = A_ee - kappa^2 H^dag_eo A_oo^-1 H^dag_oe */);
// out = D in (dag: D^dagger in) on the whole lattice, [even | odd] buffers; csw = 0: Wilson
bq_status bq_dirac_full(bq_lattice* lat, void* out, const void* in, double kappa, double csw, int prec, int recon,
                        cudaStream_t stream, bool dag);
// out = C in on one parity (site-diagonal clover multiply)
bq_status bq_clover_mul(bq_lattice* lat, void* out, const void* in, const void* cl, int prec, cudaStream_t stream);

void bq_solver_free(bq_lattice* lat);
void bq_dd_free(bq_lattice* lat);

static inline size_t field_bytes_one_parity(const Geom& g, int prec) { return (size_t)g.Vh * spinor_site_bytes(prec); }
