/* bq.h — C-ABI boundary of the B200-native even-odd Wilson(-clover) Dirac operator and its
 * mixed-precision BiCGStab (hot path of arXiv 2111.04457, "Bridge++ 2.0").
 *
 * Citations: PAPER.md:N = /root/reference/PAPER.md line N; SURVEY §x = /root/repo/SURVEY.md.
 *
 * The paper states the problem as a 4-D lattice x_mu = 1..L_mu with SU(3) link variables
 * U_mu(x) and a fermion vector of 3 colour x 4 spinor complex components per site, on which the fermion
 * matrix of Eq. 1 acts:
 *
 *   D_{x,y} = [1 + F(x)] d_{x,y} - kappa sum_mu [ (1 - g_mu) U_mu(x) d_{x+mu,y} + (1 + g_mu) U_mu^dag(x-mu) d_{x-mu,y} ]
 *
 * with a boundary condition "imposed in each direction", and the linear equation D x = b
 * solved by a mixed-precision solver (Fig. 1: set_config(U), set_mode("D"),
 * invert(x, b, nconv, diff)).  Everything below runs on ONE GPU in hand-written CUDA kernels; there is
 * no CPU fallback: every entry point returns BQ_ECUDA when no device is usable.
 *
 * ---------------------------------------------------------------------------------------------
 * Canonical (caller-side) layouts — all fp64, complex = (re, im) interleaved, C-contiguous:
 *   site    s = x + Lx*(y + Ly*(z + Lz*t)), 0-based (the paper counts from 1); mu = 0..3 = x,y,z,t
 *   spinor  psi[s][spin 0..3][colour 0..2][re,im]                     24 doubles per site
 *   gauge   U[s][mu][row 0..2][col 0..2][re,im]                        72 doubles per site; U_mu(x) as in Eq. 1,
 *                                                                      row = colour index of the result
 * Gamma matrices: Euclidean Dirac representation: g_k = [[0,-i s_k],[+i s_k,0]],
 * g_4 = diag(1,1,-1,-1).
 *
 * Internal (device-side) field layout, produced by bq_field_import and consumed by the apply calls:
 * even-odd (checkerboard), site-vectorised, tiled structure of arrays.  parity p = (x+y+z+t)&1, half index
 * h = (x>>1) + (Lx/2)*(y + Ly*(z + Lz*t)), Vh = V/2 (a multiple of 8).  A site's S bytes are cut into 16-byte
 * words (word k = reals [k*W, (k+1)*W) of the site's 24, W = 16/sizeof(real)); sites are grouped in tiles of 8
 * consecutive half indices; inside a tile, word k of the 8 sites is one contiguous 128-byte plane:
 *     address(h, k) = base + (h >> 3)*8*S + k*128 + (h & 7)*16
 *   BQ_FP64: 12 words of double2               S = 192   (Vh*192 bytes)
 *   BQ_FP32:  6 words of float4                S =  96   (Vh* 96 bytes)
 *   BQ_HALF:  3 words of 8 x fp16 mantissas v_i/n, then a 4-byte fp32 n = max_i|v_i|   S = 52   (Vh*52 bytes)
 * so a warp of 32 consecutive h reads four whole 128-byte lines per load.  A BQ_FULL buffer is the even block
 * followed by the odd block.  bq_field_bytes gives the sizes.  Buffers must be 16-byte aligned.
 * A multi-right-hand-side buffer (the *_multi calls) is nrhs such fields one after the other.
 *
 * Ownership: the caller (PyTorch in this repo) allocates and frees every field buffer and passes raw
 * DEVICE pointers; the library never keeps them after the call returns.  The handle owns its gauge
 * copies, clover blocks and solver workspace.  Calls on one handle must not run concurrently.
 * Unless a `stream` argument says otherwise, work is enqueued on the CUDA legacy default stream and
 * the call returns without synchronising (bq_solve and bq_gauge_load synchronise before returning).  The solver (and
 * the test / benchmark hooks of bq_test.h) run on a stream the handle owns — a blocking stream, i.e. ordered with the legacy
 * default stream exactly as the legacy stream is with itself — because batches of solver iterations are replayed as
 * CUDA graphs and the legacy stream cannot be captured.
 *
 * Environment switches.  Six variables are read (bq_lattice_create; BQ_LS_BRICK at the first multi-rhs launch) — measurement
 * A/B switches of the kernels' launch strategy kept for the tables in DESIGN.md; none changes a result (every variant
 * computes the same bits), the defaults are the measured best, and a production build needs none of them:
 *   BQ_GRAPH=0        solver: launch the batches of inner iterations eagerly instead of replaying CUDA graphs
 *   BQ_PDL=0|<Vh>     single-rhs hop: programmatic dependent launch off, or only when Vh <= the bound (default 262144)
 *   BQ_HOP_SMALL=<Vh> single-rhs fp32 hop: uncapped-register build when Vh <= the bound (default 2 x SMs x 128)
 *   BQ_MRHS_LS=0..3   multi-rhs hop: 0 = per-(site, rhs) kernel only, 1 = link-stationary kernel for fp32 / half only,
 *                     2 (default) = that + the direction-split fp64 kernel from 8 right-hand sides on, 3 = direction-split wherever it applies
 *   BQ_MRHS_PATCH=0   multi-rhs per-(site, rhs) kernel: plain instead of patch thread mapping
 *   BQ_LS_BRICK=y,z,t link-stationary kernels: cap of the launch-order brick (default 4,4,4; 1,1,1 = lexicographic)
 * ---------------------------------------------------------------------------------------------
 */
#ifndef BQ_H
#define BQ_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bq_lattice bq_lattice; /* opaque: geometry, boundary phases, gauge copies, clover, workspaces */

typedef enum {
    BQ_OK = 0,
    BQ_EINVAL = 1,           /* NULL pointer, bad enum, |phase| != 1, non-positive tolerance ...            */
    BQ_EODD_EXTENT = 2,      /* an extent is odd or < 2 (checkerboard needs even L_mu)                    */
    BQ_ENOGAUGE = 3,         /* apply / solve before bq_gauge_load                                        */
    BQ_ENOCLOVER = 4,        /* a clover kernel was asked for but no clover term exists (csw = 0 / not built) */
    BQ_ESINGULAR_CLOVER = 5, /* a 6x6 clover block is not positive definite (Cholesky failed)             */
    BQ_ECUDA = 6,            /* CUDA runtime error or no device; text in bq_last_error                    */
    BQ_ENOMEM = 7,           /* device allocation failed                                                  */
    BQ_ENOTCONVERGED = 8,    /* solver hit max_inner / max_outer; x holds the best iterate                */
    BQ_EBREAKDOWN = 9        /* BiCGStab breakdown (rho, <rhat,v> or <t,t> = 0) that a restart did not cure */
} bq_status;

typedef enum { BQ_FP64 = 0, BQ_FP32 = 1, BQ_HALF = 2 } bq_prec;
/* BQ_EVEN: out_e = -kappa H_eo in_o;  BQ_ODD: out_o = -kappa H_oe in_e;  BQ_FULL: out = D in (Eq. 1, F = 0). */
typedef enum { BQ_EVEN = 0, BQ_ODD = 1, BQ_FULL = 2 } bq_parity;
/* 18 reals per link, or rows 0,1 only (12 reals) with row 2 = conj(row0 x row1) rebuilt in registers. */
typedef enum { BQ_RECON18 = 0, BQ_RECON12 = 1 } bq_recon;
/* Operator modes of the paper's interface, set_mode("D"), ("Ddag"), ("DdagD"). */
typedef enum { BQ_MODE_D = 0, BQ_MODE_DDAG = 1, BQ_MODE_DDAGD = 2 } bq_mode;

/* Lattice handle.  bc_phase = 4 x (re, im): psi(x + L_mu mu^) = phi_mu psi(x), |phi_mu| = 1
 * ("a boundary condition ... is imposed in each direction"; reading S3: the phase multiplies the
 * forward hop that wraps, its conjugate the backward hop that wraps; it is never folded into the links).
 * NULL means periodic in x,y,z and antiperiodic in t.  Extents must be even and >= 2, V < 2^31. */
bq_status bq_lattice_create(int Lx, int Ly, int Lz, int Lt, const double* bc_phase, bq_lattice** out);
bq_status bq_lattice_destroy(bq_lattice* lat);

/* Static text for a status, and the handle's last error message (valid until the next call on it). */
const char* bq_status_string(bq_status s);
const char* bq_last_error(const bq_lattice* lat);

/* set_config: hand the link field to the operator.  U: canonical fp64 layout, 72*V doubles,
 * HOST or DEVICE pointer (detected).  Copies: the caller may free U afterwards.  Builds the fp64 even-odd
 * SoA gauge store; fp32 / half and 12-real copies are made on first use.  Invalidates any cached clover term.
 * U is assumed to be SU(3); it is not checked (BQ_RECON12 silently relies on it).  Synchronises. */
bq_status bq_gauge_load(bq_lattice* lat, const double* U);

/* Bytes of an internal-layout field of one parity (BQ_EVEN / BQ_ODD) or of the full lattice (BQ_FULL). */
bq_status bq_field_bytes(const bq_lattice* lat, bq_prec prec, bq_parity parity, size_t* bytes);

/* Layout conversion at the interface (source and solution stay in the caller's layout
 * and are rearranged "to respect coalesced access" on entry).  canonical: DEVICE pointer, 24*V doubles (the whole
 * lattice, whatever `parity` says); internal: DEVICE buffer of bq_field_bytes(prec, parity).
 * import: picks the sites of `parity` (or both), converts fp64 -> prec with round-to-nearest-even; for BQ_HALF
 *         n = max|v_i| per site, mantissas fp16(v_i/n), an all-zero site stores n = 0 and zero mantissas.
 * export: writes the sites of `parity` into `canonical` and leaves the other parity's entries untouched. */
bq_status bq_field_import(bq_lattice* lat, void* internal, const double* canonical, bq_parity parity, bq_prec prec,
                          void* stream);
bq_status bq_field_export(bq_lattice* lat, double* canonical, const void* internal, bq_parity parity, bq_prec prec,
                          void* stream);

/* Hopping term of Eq. 1 on internal-layout fields; F = 0 (the "Wilson matrix"):
 *   BQ_EVEN: out (even sites) = -kappa sum_mu [(1-g_mu) U_mu(x) in(x+mu) + (1+g_mu) U_mu^dag(x-mu) in(x-mu)], in = odd field
 *   BQ_ODD : the same with the parities exchanged
 *   BQ_FULL: out = D in = in - kappa H in, both parities (in, out: [even | odd] buffers)
 * in and out must not overlap.  One kernel launch per parity on `stream` (a cudaStream_t, NULL = legacy default
 * stream); no host synchronisation.  Errors: BQ_ENOGAUGE, BQ_EINVAL, BQ_ECUDA (launch error). */
bq_status bq_wilson_apply(bq_lattice* lat, void* out, const void* in, double kappa, bq_parity parity, bq_prec prec,
                          bq_recon recon, void* stream);

/* Clover term 1 + F(x) of Eq. 1 — "a 12x12 Hermitian matrix made of the link variables"; formula from
 * BASELINE.json config 4 / SURVEY O2:  A(x) = 1 - csw*kappa sum_{mu<nu} sigma_mu_nu (x) F_mu_nu(x),
 * F_mu_nu = (Q - Q^dag)/(8i), Q = the four plaquette leaves at x (trace part NOT removed, S5).
 * Stored per site as two Hermitian 6x6 chirality blocks (72 reals).
 * The first call for a given (csw, kappa) after bq_gauge_load builds the blocks and their inverses (Cholesky in
 * fp64) and caches them; out == NULL && in == NULL means "build only".
 *   out(x) = A(x) in(x)   (inverse = 0)   or   A(x)^-1 in(x)   (inverse = 1),   x of `parity` (BQ_FULL: all sites).
 * in/out: internal-layout DEVICE buffers of precision `prec`; out may equal in.  The apply is one kernel launch on `stream`
 * (a cudaStream_t, NULL = legacy default stream), no host synchronisation; a build synchronises.
 * Errors: BQ_ENOGAUGE, BQ_ESINGULAR_CLOVER (build), BQ_EINVAL, BQ_ECUDA. */
bq_status bq_clover_apply(bq_lattice* lat, double csw, double kappa, void* out, const void* in, bq_parity parity,
                          int inverse, bq_prec prec, void* stream);

/* Full Wilson-clover matrix of Eq. 1 on the whole lattice, internal layout ([even | odd] buffers):
 *   out = D in = A in - kappa H in;   csw = 0 gives the Wilson matrix. */
bq_status bq_dirac_apply(bq_lattice* lat, void* out, const void* in, double kappa, double csw, bq_prec prec,
                         bq_recon recon, void* stream);

/* Even-odd preconditioned (Schur complement) operator on even-site fields:
 *   out_e = A_ee in_e - kappa^2 H_eo A_oo^-1 H_oe in_e      (A = 1 when csw = 0).
 * tmp: caller-provided scratch field of one parity (same precision).  in, out, tmp must not overlap. */
bq_status bq_schur_apply(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw,
                         bq_prec prec, bq_recon recon, void* stream);

/* The operator in the paper's three modes, full lattice, internal layout:
 *   BQ_MODE_D: out = D in;   BQ_MODE_DDAG: out = D^dagger in;   BQ_MODE_DDAGD: out = D^dagger D in.
 * D^dagger = g5 D g5: the same hop kernel with the projectors (1 -+ g_mu) exchanged (a compile-time variant that
 * renames registers; links, phases and traffic are those of D); the clover term is Hermitian.
 * tmp: scratch field of the full lattice, needed (and must be distinct) for BQ_MODE_DDAGD only. */
bq_status bq_dirac_apply_mode(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw, bq_mode mode,
                              bq_prec prec, bq_recon recon, void* stream);
/* The even-odd Schur operator in the same modes: M^, M^^dagger = A_ee - kappa^2 H^dag_eo A_oo^-1 H^dag_oe, M^^dagger M^.
 * tmp: one-parity scratch; tmp2: a second one, BQ_MODE_DDAGD only. */
bq_status bq_schur_apply_mode(bq_lattice* lat, void* out, const void* in, void* tmp, void* tmp2, double kappa, double csw,
                              bq_mode mode, bq_prec prec, bq_recon recon, void* stream);

/* Multi-right-hand-side forms (the paper's use case is the 12 spin-colour sources of one
 * propagator on one gauge field): the same operators applied to nrhs fields in ONE launch per hop, so
 * that every link is fetched from HBM once for all right-hand sides (compulsory traffic per site and rhs: 8/nrhs links
 * + 2 spinors).  in / out / tmp: nrhs internal-layout fields one after the other (rhs k at byte offset
 * k * bq_field_bytes(prec, parity)); results equal nrhs separate single-field calls bit for bit. */
bq_status bq_wilson_apply_multi(bq_lattice* lat, void* out, const void* in, int nrhs, double kappa, bq_parity parity,
                                bq_prec prec, bq_recon recon, void* stream);
bq_status bq_schur_apply_multi(bq_lattice* lat, void* out, const void* in, void* tmp, int nrhs, double kappa, double csw,
                               bq_prec prec, bq_recon recon, void* stream);

/* Krylov method of the (inner) solver: BiCGStab on M^ (reading O4), or conjugate gradients on the normal equations
 * M^^dag M^ (uses the Ddag mode of the operator). */
typedef enum { BQ_BICGSTAB = 0, BQ_CGNR = 1 } bq_method;

typedef struct {
    int inner_prec;    /* bq_prec: BQ_FP64 = plain fp64 BiCGStab, no outer loop; BQ_FP32 / BQ_HALF = defect correction */
    int recon;         /* bq_recon used by the inner operator (the fp64 outer operator always uses 18 reals)          */
    double csw;        /* 0 = Wilson; otherwise the clover term is built for (csw, kappa)                              */
    double inner_tol;  /* relative residual reduction asked of one inner solve; <= 0 = default (1e-5 fp32, 2e-3 half)    */
    int max_inner;     /* cap on inner iterations per outer cycle; <= 0 = default (1000 fp32/fp64, 100 half)          */
    int max_outer;     /* cap on outer cycles; <= 0 = default (50)                                                    */
    int check_every;   /* inner iterations between host polls of the device-side convergence flag; <= 0 = default (8; half: 4) */
    int method;        /* bq_method: BQ_BICGSTAB (0, default) or BQ_CGNR = CG on the normal equations M^^dag M^ e = M^^dag r   */
    int lexical;       /* 0 (default): even-odd preconditioned Schur system; 1: BiCGStab on the full matrix D itself
                          (the paper's `lex` operator); bq_solve only, BQ_BICGSTAB only       */
    int x0_zero;       /* 1: the initial guess is zero and x is output only — its contents on entry are neither read nor
                          transferred (saves one host-to-device copy and one layout conversion per right-hand side)           */
    void* stream;      /* cudaStream_t whose earlier work (e.g. the kernels producing b) the solve waits for; NULL = none.
                          The solve runs on a stream of the handle and synchronises before returning                       */
} bq_solve_opts;

typedef struct {
    int status;               /* bq_status of the solve                                                         */
    int outer_cycles;         /* defect-correction cycles (0 for a pure fp64 solve)                             */
    int inner_iters;          /* total BiCGStab iterations  (= the paper's nconv; reading S9)    */
    int restarts;             /* BiCGStab restarts after a breakdown or a stalled inner solve                    */
    double true_rel_residual; /* |b - D x| / |b| recomputed in fp64 with the fp64 operator (= the paper's diff) */
    double seconds;           /* device time of the whole call (CUDA events), copies of b and x included       */
    double phase_seconds[5];  /* the same, by phase: [0] transfer + layout conversion of b (and x0), [1] source
                                 preparation b^_e (+ |b|), [2] the outer/inner iteration, [3] odd-site reconstruction +
                                 true residual, [4] layout conversion + transfer of x                            */
} bq_solve_info;

/* invert: solve D x = b on the whole lattice, D = Eq. 1 with the clover term for opts->csw != 0.
 * b, x: canonical fp64 layout, 24*V doubles each, HOST or DEVICE pointers (detected independently).  x is in/out:
 * initial guess on entry (zero it if none, or set opts->x0_zero), solution on return.
 * Method (readings O3, O4, S10): even-odd Schur system M^ x_e = b^_e solved by BiCGStab; for inner_prec != FP64 by
 * defect correction — fp64 true residual, low-precision inner BiCGStab on the normalised residual, fp64 update —
 * then x_o = A_oo^-1 (b_o + kappa H_oe x_e).  Stops when |b^_e - M^ x_e| <= tol*|b| (fp64), then reports the true
 * full-lattice residual.  opts == NULL: fp32 inner, 18-real, Wilson.  info may be NULL.  Synchronises.
 * Errors: BQ_ENOGAUGE, BQ_EINVAL (tol <= 0, NULLs), BQ_ENOTCONVERGED, BQ_EBREAKDOWN, BQ_ESINGULAR_CLOVER, BQ_ECUDA. */
bq_status bq_solve(bq_lattice* lat, const double* b, double* x, double kappa, double tol, const bq_solve_opts* opts,
                   bq_solve_info* info);

/* The same solve for nrhs right-hand sides at once (Fig. 1 of the paper loops over the 12 spin-colour
 * sources of a propagator on one configuration).  b, x: nrhs canonical fp64 fields one after the other
 * (24*V doubles each), HOST or DEVICE.  All right-hand sides advance together: every hop of the batched BiCGStab is ONE
 * multi-rhs kernel launch (links read once for the batch), every BLAS-1 step one batched launch; each right-hand side
 * keeps its own device-resident scalars, stops on its own criterion (its iterate is frozen from then on) and gets its
 * own entry of info[nrhs] (seconds = device time of the whole call).  The mathematics per right-hand side is that of
 * bq_solve.  Returns BQ_OK only if every right-hand side converged; otherwise the status of the failure, with
 * info[k].true_rel_residual telling which ones did. */
bq_status bq_solve_multi(bq_lattice* lat, const double* b, double* x, int nrhs, double kappa, double tol,
                         const bq_solve_opts* opts, bq_solve_info* info /*[nrhs]*/);

/* The program of the paper's Fig. 1: "for each spin id and colour ic: set a point source, invert" — the quark
 * propagator from one site — as ONE batched solve (bq_solve_multi with nrhs = 12).  src_site = {x, y, z, t} (0-based).
 * The 12 sources delta_{x,src} e_id (x) e_ic are made on the device; S (HOST or DEVICE, 12 * 24*V doubles, output only)
 * receives the 12 solutions in the canonical layout, solution k = 3*id + ic first index.  info: 12 entries or NULL. */
bq_status bq_propagator(bq_lattice* lat, const int* src_site /*[4]*/, double* S, double kappa, double tol,
                        const bq_solve_opts* opts, bq_solve_info* info /*[12]*/);

/* ---------------------------------------------------------------------------------------------
 * Domain decomposition — OPT-IN; the calls above never use it.  The paper's code is "parallelized with
 * MPI": a 4-D process grid, one halo exchange per matrix application overlapped with the bulk
 * (PAPER.md:95), weak scaling as its experiment.  Here: Wilson operator (csw = 0), fp64 / fp32 storage.
 *
 * bq_lattice_create_sub: the sub-lattice of one rank.  lx..lt = LOCAL extents (even), grid[4] = ranks per direction,
 * coords[4] = this rank's position (rank number = coords[0] + grid[0]*(coords[1] + ...)); bc_phase = the GLOBAL boundary
 * phases.  bq_gauge_load takes the rank's LOCAL block of the link field (no ghost links are needed).  On such a handle
 * bq_wilson_apply computes the INTERIOR part of the hop (hops that leave the rank in a partitioned direction contribute
 * nothing); the rest arrives through the faces.  Every other operator call (bq_dirac_apply, bq_schur_apply, the *_mode and
 * *_multi forms) and the solvers return BQ_EINVAL on a handle with a partitioned direction instead of an interior-only result:
 *   bq_dd_pack    send[2*mu + side], partitioned directions only: 12 reals per boundary site of the input parity, in the
 *                 storage type (bq_dd_face_bytes): side 0 = slice x_mu = 0, spin-projected with (1 - g_mu), for the rank
 *                 BELOW; side 1 = slice x_mu = l_mu - 1, projected with (1 + g_mu) and multiplied by U_mu^dag, for the rank ABOVE.
 *   bq_dd_unpack  recv[2*mu + side]: side 1 = what the rank above packed as its side 0 (added to our slice x_mu = l_mu - 1
 *                 after multiplication by our U_mu), side 0 = what the rank below packed as its side 1 (added to our slice
 *                 x_mu = 0).  out += scale * (...), scale = the factor the interior call used (-kappa for bq_wilson_apply);
 *                 the global boundary phase is applied here on the ranks at the edge of the grid.
 * A process per GPU moves send -> recv with peer copies or NCCL send/recv between pack and unpack while the interior
 * call runs (paper_2111_04457_b200/dd.py: DistributedHop, and DistributedSolver = the BiCGStab of bq_dd_solve with one
 * all-reduce of the packed partial sums per reduction point; both executed by two processes sharing one GPU in
 * tests/test_gpu_dd_multiprocess.py).  UNMEASURED on multi-GPU hardware: no such node was available to this build.
 *
 * bq_dd_wilson_apply / bq_dd_solve: the same with VIRTUAL RANKS — all nranks = prod(grid) handles in this process on one
 * device (ranks[r] at rank number r), faces moved by device copies: what the tests compare with the oracle on the global
 * lattice.  out / in / b / x: one pointer per rank (internal-layout fields; b, x: the rank's local canonical block, HOST or
 * DEVICE).  bq_dd_solve: fp64 even-odd BiCGStab to |b^_e - M^ x_e| <= tol |b|, every inner product a sum over ranks;
 * info->inner_iters, ->true_rel_residual (of the Schur system) and ->status are filled. */
bq_status bq_lattice_create_sub(int lx, int ly, int lz, int lt, const double* bc_phase, const int* grid /*[4]*/,
                                const int* coords /*[4]*/, bq_lattice** out);
bq_status bq_dd_face_bytes(const bq_lattice* lat, int mu, bq_prec prec, size_t* bytes);
bq_status bq_dd_pack(bq_lattice* lat, void* const* send /*[8]*/, const void* in, bq_parity out_parity, bq_prec prec, bq_recon recon,
                     void* stream);
bq_status bq_dd_unpack(bq_lattice* lat, void* out, void* const* recv /*[8]*/, double scale, bq_parity out_parity, bq_prec prec,
                       bq_recon recon, void* stream);
bq_status bq_dd_wilson_apply(bq_lattice* const* ranks, int nranks, void* const* out, const void* const* in, double kappa,
                             bq_parity parity, bq_prec prec, bq_recon recon, void* stream);
bq_status bq_dd_solve(bq_lattice* const* ranks, int nranks, const double* const* b, double* const* x, double kappa, double tol,
                      int max_iter, bq_solve_info* info);

/* ---------------------------------------------------------------------------------------------
 * A reduction for callers that cannot allocate device memory.
 *
 * Every other call of this library that sums over a field (the solver's |r|^2 and inner products) keeps its
 * per-block partial sums in a workspace the handle obtains with cudaMalloc on first use.  That is a problem for a host
 * program which has given the whole GPU to an allocator of its own (a deep-learning framework's caching allocator, a
 * serving process with a fixed arena: a foreign cudaMalloc fails or eats into the arena), for code that runs while
 * another thread captures a stream in the global capture mode (cudaMalloc is forbidden there and breaks that capture),
 * and for monitoring loops that must not stall the device on an allocation.  This one entry point serves them:
 *
 *   *result = |a|^2 = sum over the nsites sites of a, and the 24 reals of each, of v^2
 *
 * (the squared norm the solver's stopping test of invert(), is built on).  It creates no handle, calls no
 * cudaMalloc / cudaFree / allocating library routine, and uses a fixed scratch array compiled into libbq.so:
 * BQ_NOALLOC_SCRATCH_BYTES of device memory that EVERY GPU on which the library is loaded holds until the process
 * exits, whether or not this call is ever made.
 *
 *   a       DEVICE pointer, 16-byte aligned: an internal-layout field of precision prec as bq_field_import makes it —
 *           one parity (nsites = V/2) or [even | odd] (nsites = V); the caller owns it, it is only read.
 *   nsites  sites in a; a multiple of 8, at most BQ_NOALLOC_MAX_SITES (one scratch slot per 1024 sites) — a larger field
 *           is refused with BQ_EINVAL and a message that says so; sum it in pieces.  nsites = 0 gives 0.
 *   result  DEVICE pointer to one double, 8-byte aligned, the caller's; written by the kernel (no host synchronisation:
 *           read it after the stream has reached this point).
 *   stream  cudaStream_t of the CURRENT device (NULL = legacy default stream): one small memset node + one kernel.
 *   err     optional HOST buffer of errlen bytes that receives the reason when the call does not return BQ_OK.
 *
 * Arithmetic: as bq_blas_norm2 / the solver — fp64 throughout for BQ_FP64; for BQ_FP32 and BQ_HALF (mantissa x site
 * norm) squares are summed in fp32 per thread and in fp64 across threads.  The order of the additions is fixed, so the
 * result is bitwise reproducible, but it is not the order of the handle-based path: the two agree to rounding
 * (1e-13 relative in fp64, 1e-6 in fp32 / half), not bit for bit.
 *
 * First call on a device: looks up that device's copy of the scratch array (cudaGetSymbolAddress, with the device
 * current; this may also make the CUDA runtime load the library's kernels).  Make that first call at start-up — in
 * particular before any stream capture begins — so that later calls are a memset and a launch and nothing else.
 * Sharing: all calls on one device use the same scratch array, which keeps what the previous call left in it.  The
 * arrival counter is cleared on `stream` before every launch; the partial sums are overwritten before they are read.
 * Consequently two calls that may overlap on the GPU (different streams without an ordering between them, or two host
 * threads) race on the array and give garbage: order them on one stream or with events.
 * Errors: BQ_EINVAL (NULL / misaligned pointer, bad prec, nsites not a multiple of 8 or beyond the maximum), BQ_ECUDA.
 * --------------------------------------------------------------------------------------------- */
#define BQ_NOALLOC_MAX_SITES 16777216             /* 16384 scratch slots x 1024 sites (48^3 x 96 is 10.6 M sites) */
#define BQ_NOALLOC_SCRATCH_BYTES (131072 + 256)   /* 16384 partial sums of 8 bytes + a 256-byte slot for the arrival counter */
bq_status bq_field_norm2_noalloc(const void* a, long long nsites, bq_prec prec, double* result, void* stream, char* err,
                                 size_t errlen);

#ifdef __cplusplus
}
#endif
#endif /* BQ_H */
