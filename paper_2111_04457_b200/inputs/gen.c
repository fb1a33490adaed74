/* Seeded synthetic input generator (gauge links, spinor sources, SU(3) site fields).
 *
 * This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench.  It holds
 * none of the method's arithmetic (no Dirac operator, no gamma matrices, no solver): it only
 * turns (seed, stream, index) into numbers, following the input recipe of BASELINE.json
 * configs ("Links U = exp(i*eps*H), H random traceless Hermitian 3x3 with Gaussian entries
 * (seeded), reunitarised.  Source psi: complex Gaussian 12 components/site") as fixed in
 * SURVEY.md §8(d) "Generator" and reading S13.  The exact recipe is restated in DESIGN.md §4.
 *
 * Counter based: every number is a pure function of (seed, stream, counter), so the result is
 * independent of thread count and generation order.
 *
 *   key        = mix64(seed ^ (stream * 0xD1B54A32D192ED03))
 *   draw(c)    = mix64(key + c * 0x9E3779B97F4A7C15)                (mix64 = splitmix64 finaliser)
 *   uniform(u) = ((u >> 11) + 0.5) * 2^-53                          in (0,1)
 *   pair j     : u1 = uniform(draw(2j)), u2 = uniform(draw(2j+1)),
 *                r = sqrt(-2 ln u1), n0 = r cos(2 pi u2), n1 = r sin(2 pi u2)   (Box-Muller)
 *
 * Canonical layouts: site s = x + Lx*(y + Ly*(z + Lz*t));
 *   gauge  U[s][mu][row][col][re,im]  (72 doubles per site), spinor psi[s][spin][colour][re,im].
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

static inline uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static inline uint64_t make_key(uint64_t seed, uint64_t stream) {
    return mix64(seed ^ (stream * 0xD1B54A32D192ED03ULL));
}
static inline double uniform01(uint64_t key, uint64_t c) {
    uint64_t u = mix64(key + c * 0x9E3779B97F4A7C15ULL);
    return ((double)(u >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}
static inline void normal_pair(uint64_t key, uint64_t j, double* n0, double* n1) {
    double u1 = uniform01(key, 2 * j), u2 = uniform01(key, 2 * j + 1);
    double r = sqrt(-2.0 * log(u1));
    double a = 6.283185307179586476925286766559 * u2;
    *n0 = r * cos(a);
    *n1 = r * sin(a);
}

/* ---- tiny 3x3 complex helpers on (re,im)-interleaved double[18], row-major ---- */
static void m3_mul(const double* a, const double* b, double* c) {
    double t[18];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            double re = 0, im = 0;
            for (int k = 0; k < 3; k++) {
                double ar = a[2 * (3 * i + k)], ai = a[2 * (3 * i + k) + 1];
                double br = b[2 * (3 * k + j)], bi = b[2 * (3 * k + j) + 1];
                re += ar * br - ai * bi;
                im += ar * bi + ai * br;
            }
            t[2 * (3 * i + j)] = re;
            t[2 * (3 * i + j) + 1] = im;
        }
    memcpy(c, t, sizeof t);
}

/* U = exp(i*eps*H) for Hermitian H: scale by 2^-k, Taylor to order 20, square k times. */
static void m3_exp_iH(const double* H, double eps, double* U) {
    double X[18]; /* X = i*eps*H / 2^k */
    double nrm = 0;
    for (int e = 0; e < 18; e++) nrm += H[e] * H[e];
    nrm = sqrt(nrm) * fabs(eps);
    int k = 0;
    while (nrm > 0.125 && k < 40) { nrm *= 0.5; k++; }
    double sc = eps / (double)(1ULL << k);
    for (int e = 0; e < 9; e++) { /* i*(a+ib) = -b + ia */
        X[2 * e] = -sc * H[2 * e + 1];
        X[2 * e + 1] = sc * H[2 * e];
    }
    double term[18], sum[18];
    memset(term, 0, sizeof term);
    term[0] = term[8] = term[16] = 1.0;
    memcpy(sum, term, sizeof sum);
    for (int n = 1; n <= 20; n++) {
        m3_mul(term, X, term);
        for (int e = 0; e < 18; e++) { term[e] /= (double)n; sum[e] += term[e]; }
    }
    for (int q = 0; q < k; q++) m3_mul(sum, sum, sum);
    memcpy(U, sum, sizeof sum);
}

/* Reunitarise (reading S13): Gram-Schmidt rows 0,1; row 2 = conj(row0 x row1). */
static void m3_reunit(double* U) {
    double* r0 = U; double* r1 = U + 6; double* r2 = U + 12;
    double n = 0;
    for (int e = 0; e < 6; e++) n += r0[e] * r0[e];
    n = 1.0 / sqrt(n);
    for (int e = 0; e < 6; e++) r0[e] *= n;
    /* <r0,r1> = sum conj(r0_j) r1_j */
    double pr = 0, pi = 0;
    for (int j = 0; j < 3; j++) {
        pr += r0[2 * j] * r1[2 * j] + r0[2 * j + 1] * r1[2 * j + 1];
        pi += r0[2 * j] * r1[2 * j + 1] - r0[2 * j + 1] * r1[2 * j];
    }
    for (int j = 0; j < 3; j++) {
        r1[2 * j] -= pr * r0[2 * j] - pi * r0[2 * j + 1];
        r1[2 * j + 1] -= pr * r0[2 * j + 1] + pi * r0[2 * j];
    }
    n = 0;
    for (int e = 0; e < 6; e++) n += r1[e] * r1[e];
    n = 1.0 / sqrt(n);
    for (int e = 0; e < 6; e++) r1[e] *= n;
    for (int j = 0; j < 3; j++) {
        int a = (j + 1) % 3, b = (j + 2) % 3;
        /* (r0 x r1)_j = r0_a r1_b - r0_b r1_a, then conjugate */
        double re = (r0[2 * a] * r1[2 * b] - r0[2 * a + 1] * r1[2 * b + 1]) -
                    (r0[2 * b] * r1[2 * a] - r0[2 * b + 1] * r1[2 * a + 1]);
        double im = (r0[2 * a] * r1[2 * b + 1] + r0[2 * a + 1] * r1[2 * b]) -
                    (r0[2 * b] * r1[2 * a + 1] + r0[2 * b + 1] * r1[2 * a]);
        r2[2 * j] = re;
        r2[2 * j + 1] = -im;
    }
}

/* One SU(3) matrix from normal pairs 9*idx .. 9*idx+8 of the keyed stream. */
static void su3_from_stream(uint64_t key, uint64_t idx, double eps, double* U) {
    double G[18], H[18];
    for (int e = 0; e < 9; e++) normal_pair(key, 9 * idx + (uint64_t)e, &G[2 * e], &G[2 * e + 1]);
    /* H = (G + G^dagger)/2 - tr/3 */
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            H[2 * (3 * i + j)] = 0.5 * (G[2 * (3 * i + j)] + G[2 * (3 * j + i)]);
            H[2 * (3 * i + j) + 1] = 0.5 * (G[2 * (3 * i + j) + 1] - G[2 * (3 * j + i) + 1]);
        }
    double tr = (H[0] + H[8] + H[16]) / 3.0;
    H[0] -= tr; H[8] -= tr; H[16] -= tr;
    m3_exp_iH(H, eps, U);
    m3_reunit(U);
}

/* nmat SU(3) matrices exp(i*eps*H_k), k = 0..nmat-1, into out[nmat][3][3][2].
 * Gauge field: nmat = 4*V, k = 4*s + mu, stream 1.  Gauge transform g(x): nmat = V, stream 4. */
void bqgen_su3(int64_t nmat, uint64_t seed, uint64_t stream, double eps, double* out) {
    uint64_t key = make_key(seed, stream);
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < nmat; k++) su3_from_stream(key, (uint64_t)k, eps, out + 18 * k);
}

/* ncomplex complex Gaussians n0 + i*n1 (one normal pair each) into out[ncomplex][2].
 * Spinor source: ncomplex = 12*V, stream 2 (source) or 3 (test vectors). */
void bqgen_gauss(int64_t ncomplex, uint64_t seed, uint64_t stream, double* out) {
    uint64_t key = make_key(seed, stream);
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < ncomplex; k++) normal_pair(key, (uint64_t)k, &out[2 * k], &out[2 * k + 1]);
}
