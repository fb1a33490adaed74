/* bq_test.h — test and benchmark hooks of libbq.so.  NOT part of the product boundary (that is include/bq.h, the
 * calls SURVEY.md §8(b) lists): these entry points expose internal kernels of the hot path one by one so that the tests
 * can check them against the oracle (fused BLAS-1; fused inner products of the hop epilogue) and so that
 * bench.py (the contract line and its --kernels table) can time them with CUDA events on the library's own stream and count launches.
 * Same conventions as bq.h: extern "C", plain pointers, bq_status returns, internal-layout DEVICE fields.
 */
#ifndef BQ_TEST_H
#define BQ_TEST_H

#include "bq.h"

#ifdef __cplusplus
extern "C" {
#endif

/* The same operator with the BiCGStab inner products fused into the epilogue of its second hop kernel (SURVEY A6
 * (iii), (v): no separate reduction pass over the result), exposed for tests:
 *   w != NULL: dots[0..1] = <w, out>;      w == NULL: dots[0..1] = <out, in>, dots[2] = <out, out>
 * (<a,b> = sum conj(a_i) b_i).  The sums are taken over the values of out BEFORE they are rounded to the storage
 * precision (BQ_HALF: before the per-site renormalisation), per thread in the compute type, in fp64 across threads,
 * in a fixed order.  w: internal-layout even-site field of precision prec.  dots: HOST doubles.  Synchronises. */
bq_status bq_schur_apply_dots(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw,
                              bq_prec prec, bq_recon recon, const void* w, double* dots /*[3]*/);

/* Launch accounting for benchmarks: out[0] = kernels launched through this handle since creation,
 * out[1..3] = hop applications (per right-hand side) with fp64 / fp32 / half storage (each is 1320 flop x Vh sites),
 * out[4] = launches of the link-stationary multi-rhs hop kernels (hop_ls.cuh, hop_lsp.cuh) among them,
 * out[5..7] = of out[1..3], the applications that were no-ops: enqueued with a batch of solver iterations after their
 *            right-hand side had converged, they return at entry (the solver's device-side `done` flag); useful = out[1..3] - out[5..7].
 *            The count is INFERRED ON THE HOST, 4 x (iterations enqueued - iterations the device reports done), and so
 *            assumes an iteration that was not accepted ran no hop.  That is exact for convergence (the flag is set by the
 *            last kernel of an iteration) but not for a breakdown, whose flag is set in the middle of an iteration after its
 *            first two hops have run: there out[5..7] is too high by up to 2 per broken-down right-hand side and cycle, and
 *            "useful" correspondingly too low — a bias against the library's own flop rate, never in its favour,
 * out[8] = of out[4], the launches of the direction-split kernel (hop_lsp.cuh) made outside CUDA-graph replays. */
bq_status bq_get_counters(const bq_lattice* lat, unsigned long long* out /*[9]*/);

/* Fused BLAS-1 on one-parity internal-layout fields, exposed for tests and benchmarks.
 * All complex scalars are (re, im) pairs of doubles on the HOST; results are written to HOST doubles after a
 * stream synchronise.  <a,b> = sum conj(a_i) b_i.  Reductions are accumulated in fp64 for BQ_FP64 and in fp32
 * per thread, fp64 across threads, for BQ_FP32 / BQ_HALF; the summation order is fixed (bitwise reproducible). */
bq_status bq_blas_norm2(bq_lattice* lat, const void* a, bq_prec prec, double* result);
bq_status bq_blas_cdot(bq_lattice* lat, const void* a, const void* b, bq_prec prec, double* result /*[2]*/);
/* y <- y + alpha x */
bq_status bq_blas_caxpy(bq_lattice* lat, const double* alpha /*[2]*/, const void* x, void* y, bq_prec prec);
/* BiCGStab update (iv): x += alpha p + omega s;  r = s - omega t;  returns |r|^2 and <rhat, r>. */
bq_status bq_blas_bicg_update(bq_lattice* lat, const double* alpha, const double* omega, const void* p, const void* s,
                              const void* t, const void* rhat, void* x, void* r, bq_prec prec,
                              double* r_norm2, double* rhat_r /*[2]*/);

/* Benchmark hook: device time (CUDA events on the library's stream, after one warm-up launch per set) of ONE
 * internal kernel of the hot path, averaged over `reps` back-to-back launches that rotate over `nsets` (1..16) sets
 * of scratch vectors allocated inside the call, so that a launch does not find its operands in L2.
 * bytes_per_launch = the kernel's ALGORITHMIC bytes (every operand read once, every result written
 * once).  BQ_K_HOP* launch on even output sites; the clover variants need csw != 0.  Synchronises. */
typedef enum {
    BQ_K_HOP = 0,            /* out = -kappa H in                                   (A3, epilogue 0)                 */
    BQ_K_HOP_XPAY = 1,       /* out = z + kappa H in                                (A3, epilogue 1; Wilson M^ step 2) */
    BQ_K_HOP_CLOVINV = 2,    /* out = -kappa A^-1 H in                              (A3+A5, clover M^ step 1)        */
    BQ_K_HOP_CLOV_XPAY = 3,  /* out = A z + kappa H in                              (A3+A5, clover M^ step 2)        */
    BQ_K_SCHUR = 4,          /* out = M^ in (two hop launches)                      (A7)                             */
    BQ_K_NORM2 = 5,          /* |a|^2                                               (A6)                             */
    BQ_K_P_UPDATE = 6,       /* p = r + beta (p - omega v)                          (A6 i)                           */
    BQ_K_ALPHA = 7,          /* <rhat, v> -> alpha                                  (A6 v)                           */
    BQ_K_S_UPDATE = 8,       /* s = r - alpha v                                     (A6 ii)                          */
    BQ_K_OMEGA = 9,          /* <t,s>, <t,t> -> omega                               (A6 iii)                         */
    BQ_K_FINAL = 10,         /* x += alpha p + omega s; r = s - omega t; |r|^2; <rhat,r>   (A6 iv)                   */
    BQ_K_BICG_ITER = 11,     /* one whole inner BiCGStab iteration as bq_solve runs it: 4 hops (two of them with
                                fused inner products) + 3 BLAS-1 kernels                    (A8)                     */
    BQ_K_HOP_XPAY_ALPHA = 12,   /* out = [A] z + kappa H in and <w, out> -> alpha           (A3 [+A5] + A6 v)        */
    BQ_K_HOP_XPAY_OMEGA = 13,   /* out = [A] z + kappa H in and <out,z>, <out,out> -> omega  (A3 [+A5] + A6 iii)     */
    BQ_K_BICG_ITER_UNFUSED = 14 /* the same iteration with the two inner products as separate kernels (4 + 5)        */
} bq_kernel_id;
bq_status bq_bench_kernel(bq_lattice* lat, int which, bq_prec prec, bq_recon recon, double csw, double kappa, int reps,
                          int nsets, double* us_per_launch, double* bytes_per_launch);

/* The same for the multi-rhs kernels (BQ_K_HOP, BQ_K_HOP_XPAY, BQ_K_HOP_CLOVINV, BQ_K_HOP_CLOV_XPAY, BQ_K_SCHUR,
 * BQ_K_BICG_ITER = one batched inner iteration of bq_solve_multi):
 * one launch processes nrhs right-hand sides; bytes_per_launch counts links and clover blocks once and the spinors
 * once per right-hand side. */
bq_status bq_bench_kernel_multi(bq_lattice* lat, int which, bq_prec prec, bq_recon recon, double csw, double kappa,
                                int nrhs, int reps, int nsets, double* us_per_launch, double* bytes_per_launch);

#ifdef __cplusplus
}
#endif
#endif /* BQ_TEST_H */
