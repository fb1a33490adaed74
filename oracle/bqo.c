/* oracle/bqo.c — TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the hot path computes: the Wilson /
 * Wilson-clover fermion matrix D[U] of the paper's Eq. 1 (§3) and a textbook
 * BiCGStab on it.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file's library.  It shares no code, headers, tables or
 * helpers with the CUDA path (paper_2111_04457_b200/csrc): the gamma matrices below are typed
 * in as 4x4 matrices, the kernels hard-wire spin projections of their own.
 *
 * Everything is written site by site in the canonical lexicographic layout, in the order and
 * notation of Eq. 1; no checkerboarding, blocking, fusion or reordering.
 *
 * Canonical layouts; all arrays are C-contiguous doubles, complex = (re,im):
 *   site    s = x + Lx*(y + Ly*(z + Lz*t)),  L[4] = {Lx,Ly,Lz,Lt},  mu = 0..3 = x,y,z,t
 *   gauge   U[s][mu][row][col]          (9 complex per link; U_mu(x) of Eq. 1, row = output colour)
 *   spinor  psi[s][spin][colour]        (12 complex per site, "3 colour x 4 spinor")
 *   site-diagonal term  A[s][12][12]    (row-major, index = 3*spin + colour; A = 1 + F(x) of Eq. 1)
 *   bc[8] = 4 x (re,im): boundary phase phi_mu, psi(x + L_mu mu^) = phi_mu psi(x) (reading S3)
 *
 * Pins (tests/test_oracle_*.py): Clifford algebra, free-field plane-wave
 * eigenvalues in closed form, gamma5-hermiticity, gauge covariance, brute-force dense matrix on
 * 4^4 (assembled in numpy from Kronecker products: disjoint code path), abelian constant-flux
 * field strength, sign of the clover term, point-source pattern, even-odd Schur identities.
 * D^dagger (bqo_dirac_apply_dag, the definition of the adjoint as a scatter) and the CGNR of bqo.py are pinned by
 * tests/test_oracle_dagger_pins.py: conjugate transpose of the dense matrix, D^dag = g5 D g5, <x,Dy> = <D^dag x,y>,
 * free-field eigenvalue conj(lambda), point-source stencil, numpy.linalg.solve.
 * Unpinned readings: S5 (trace part of F_mu_nu is NOT subtracted; `traceless` flag, default 0)
 * and S9 (meaning of nconv/diff) — "parity unpinned" for those two choices, see DESIGN.md §3.
 * (The arithmetic of the optional traceless branch is pinned against the pinned default by
 * tests/test_oracle_clover_pins.py::test_traceless_option_removes_exactly_the_trace; which of the two the paper
 * means stays the unpinned reading S5.)
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

/* ------------------------------------------------------------------------------------------
 * Gamma matrices — Euclidean Dirac representation (reading S1, SURVEY.md Appendix A.1;
 * BASELINE.json config 1 "Dirac gamma basis").  gamma_k = [[0, -i sigma_k],[+i sigma_k, 0]],
 * gamma_4 = diag(1,1,-1,-1).  Index 0..3 = x,y,z,t (paper's mu = 1..4).
 * ------------------------------------------------------------------------------------------ */
#define II _Complex_I
static const cplx GAMMA[4][4][4] = {
    /* gamma_x */ {{0, 0, 0, -II}, {0, 0, -II, 0}, {0, II, 0, 0}, {II, 0, 0, 0}},
    /* gamma_y */ {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    /* gamma_z */ {{0, 0, -II, 0}, {0, 0, 0, II}, {II, 0, 0, 0}, {0, -II, 0, 0}},
    /* gamma_t */ {{1, 0, 0, 0}, {0, 1, 0, 0}, {0, 0, -1, 0}, {0, 0, 0, -1}},
};

/* gamma_mu for mu = 0..3; mu = 4 gives gamma_5 = gamma_x gamma_y gamma_z gamma_t. out[4][4]. */
void bqo_gamma(int mu, double* out) {
    cplx g[4][4];
    if (mu < 4) {
        memcpy(g, GAMMA[mu], sizeof g);
    } else {
        cplx a[4][4], b[4][4];
        memcpy(a, GAMMA[0], sizeof a);
        for (int m = 1; m < 4; m++) {
            for (int i = 0; i < 4; i++)
                for (int j = 0; j < 4; j++) {
                    b[i][j] = 0;
                    for (int k = 0; k < 4; k++) b[i][j] += a[i][k] * GAMMA[m][k][j];
                }
            memcpy(a, b, sizeof a);
        }
        memcpy(g, a, sizeof g);
    }
    memcpy(out, g, sizeof g);
}

/* sigma_mu_nu = (i/2) [gamma_mu, gamma_nu]   (reading O2) */
static void sigma_munu(int mu, int nu, cplx s[4][4]) {
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            cplx c = 0;
            for (int k = 0; k < 4; k++) c += GAMMA[mu][i][k] * GAMMA[nu][k][j] - GAMMA[nu][i][k] * GAMMA[mu][k][j];
            s[i][j] = 0.5 * II * c;
        }
}

/* ------------------------------------------------------------------------------------------ */
static inline void coords(const int* L, long s, int x[4]) {
    x[0] = (int)(s % L[0]); s /= L[0];
    x[1] = (int)(s % L[1]); s /= L[1];
    x[2] = (int)(s % L[2]); s /= L[2];
    x[3] = (int)s;
}
static inline long site_of(const int* L, const int x[4]) {
    return x[0] + (long)L[0] * (x[1] + (long)L[1] * (x[2] + (long)L[2] * x[3]));
}
/* site x + d*mu^ with periodic wrap of the coordinate (d = +1 or -1, or any integer) */
static inline long shifted(const int* L, const int x[4], int mu, int d) {
    int y[4] = {x[0], x[1], x[2], x[3]};
    y[mu] = ((y[mu] + d) % L[mu] + L[mu]) % L[mu];
    return site_of(L, y);
}
static inline long volume(const int* L) { return (long)L[0] * L[1] * L[2] * L[3]; }

/* (D psi)(x) for ONE site x, literally Eq. 1 with reading O1:
 *   (D psi)(x) = A(x) psi(x) - kappa sum_mu [ (1 - gamma_mu) U_mu(x)          phi+_mu(x) psi(x+mu^)
 *                                           + (1 + gamma_mu) U_mu(x-mu^)^dag  phi-_mu(x) psi(x-mu^) ]
 *   phi+ = phi_mu if x_mu = L_mu-1 else 1;  phi- = conj(phi_mu) if x_mu = 0 else 1.
 * A == NULL means A = 1 (Wilson, F = 0). */
static void dirac_site(const int* L, const cplx* bc, const cplx* U, double kappa, const cplx* A,
                       const cplx* psi, long s, cplx* out /*12*/) {
    int x[4];
    coords(L, s, x);
    /* site-diagonal term */
    if (A) {
        const cplx* As = A + 144 * s;
        for (int i = 0; i < 12; i++) {
            cplx c = 0;
            for (int j = 0; j < 12; j++) c += As[12 * i + j] * psi[12 * s + j];
            out[i] = c;
        }
    } else {
        for (int i = 0; i < 12; i++) out[i] = psi[12 * s + i];
    }
    for (int mu = 0; mu < 4; mu++) {
        /* forward: (1 - gamma_mu) U_mu(x) psi(x + mu^) */
        {
            long sf = shifted(L, x, mu, +1);
            cplx phase = (x[mu] == L[mu] - 1) ? bc[mu] : 1.0;
            const cplx* Um = U + 9 * (4 * s + mu);
            cplx w[4][3]; /* w = U psi(x+mu), colour multiply for each spin */
            for (int sp = 0; sp < 4; sp++)
                for (int a = 0; a < 3; a++) {
                    cplx c = 0;
                    for (int b = 0; b < 3; b++) c += Um[3 * a + b] * psi[12 * sf + 3 * sp + b];
                    w[sp][a] = phase * c;
                }
            for (int sp = 0; sp < 4; sp++)
                for (int a = 0; a < 3; a++) {
                    cplx c = 0;
                    for (int sq = 0; sq < 4; sq++) c += ((sp == sq ? 1.0 : 0.0) - GAMMA[mu][sp][sq]) * w[sq][a];
                    out[3 * sp + a] -= kappa * c;
                }
        }
        /* backward: (1 + gamma_mu) U_mu(x - mu^)^dagger psi(x - mu^) */
        {
            long sb = shifted(L, x, mu, -1);
            cplx phase = (x[mu] == 0) ? conj(bc[mu]) : 1.0;
            const cplx* Um = U + 9 * (4 * sb + mu);
            cplx w[4][3];
            for (int sp = 0; sp < 4; sp++)
                for (int a = 0; a < 3; a++) {
                    cplx c = 0;
                    for (int b = 0; b < 3; b++) c += conj(Um[3 * b + a]) * psi[12 * sb + 3 * sp + b];
                    w[sp][a] = phase * c;
                }
            for (int sp = 0; sp < 4; sp++)
                for (int a = 0; a < 3; a++) {
                    cplx c = 0;
                    for (int sq = 0; sq < 4; sq++) c += ((sp == sq ? 1.0 : 0.0) + GAMMA[mu][sp][sq]) * w[sq][a];
                    out[3 * sp + a] -= kappa * c;
                }
        }
    }
}

/* out = D in on the whole lattice. A may be NULL (Wilson). in and out must not alias. */
int bqo_dirac_apply(const int* L, const double* bc, const double* U, double kappa, const double* A,
                    const double* in, double* out) {
    long V = volume(L);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++)
        dirac_site(L, (const cplx*)bc, (const cplx*)U, kappa, (const cplx*)A, (const cplx*)in, s, (cplx*)out + 12 * s);
    return 0;
}

/* (D in)(x) at the listed sites only: out[k][12] for site sites[k] (full-size sampled parity checks). */
int bqo_dirac_apply_sites(const int* L, const double* bc, const double* U, double kappa, const double* A,
                          const double* in, long nsites, const long* sites, double* out) {
#pragma omp parallel for schedule(static)
    for (long k = 0; k < nsites; k++)
        dirac_site(L, (const cplx*)bc, (const cplx*)U, kappa, (const cplx*)A, (const cplx*)in, sites[k], (cplx*)out + 12 * k);
    return 0;
}

/* out = D^dagger in on the whole lattice, by the DEFINITION of the adjoint, (D^dag)_{y,x} = (D_{x,y})^dag
 * (the paper's set_mode("Ddag")): every 12x12 block D_{x,y} of Eq. 1 is
 * taken exactly as dirac_site uses it and its conjugate transpose is scattered,  out(y) += (D_{x,y})^dag in(x).
 *   D_{x,x}    = A(x)
 *   D_{x,x+mu} = -kappa phi+_mu(x) (1 - gamma_mu) (x) U_mu(x)
 *   D_{x,x-mu} = -kappa phi-_mu(x) (1 + gamma_mu) (x) U_mu(x-mu)^dag
 * Block element: D[(sp,a),(sq,b)] = c * P[sp][sq] * W[a][b]  =>  (D^dag in)[(sq,b)] += conj(c P[sp][sq] W[a][b]) in[(sp,a)].
 * Serial scatter (no derivation of a gather form, so that nothing but the definition is trusted).
 * in and out must not alias. */
int bqo_dirac_apply_dag(const int* L, const double* bc_, const double* U_, double kappa, const double* A_,
                        const double* in_, double* out_) {
    long V = volume(L);
    const cplx *bc = (const cplx*)bc_, *U = (const cplx*)U_, *A = (const cplx*)A_, *in = (const cplx*)in_;
    cplx* out = (cplx*)out_;
    for (long i = 0; i < 12 * V; i++) out[i] = 0;
    for (long s = 0; s < V; s++) {
        int x[4];
        coords(L, s, x);
        const cplx* v = in + 12 * s;
        /* diagonal block A(x) (identity for Wilson) */
        for (int j = 0; j < 12; j++) {
            if (A) {
                cplx c = 0;
                for (int i = 0; i < 12; i++) c += conj(A[144 * s + 12 * i + j]) * v[i];
                out[12 * s + j] += c;
            } else {
                out[12 * s + j] += v[j];
            }
        }
        for (int mu = 0; mu < 4; mu++) {
            for (int dir = 0; dir < 2; dir++) {   /* 0: block D_{x,x+mu}, 1: block D_{x,x-mu} */
                long y = shifted(L, x, mu, dir == 0 ? +1 : -1);
                cplx c = -kappa * (dir == 0 ? ((x[mu] == L[mu] - 1) ? bc[mu] : 1.0) : ((x[mu] == 0) ? conj(bc[mu]) : 1.0));
                const cplx* Um = U + 9 * (4 * (dir == 0 ? s : y) + mu);
                for (int sp = 0; sp < 4; sp++)
                    for (int sq = 0; sq < 4; sq++) {
                        cplx P = (sp == sq ? 1.0 : 0.0) + (dir == 0 ? -1.0 : 1.0) * GAMMA[mu][sp][sq];
                        if (P == 0) continue;
                        for (int a = 0; a < 3; a++)
                            for (int b = 0; b < 3; b++) {
                                cplx W = dir == 0 ? Um[3 * a + b] : conj(Um[3 * b + a]);
                                out[12 * y + 3 * sq + b] += conj(c * P * W) * v[3 * sp + a];
                            }
                    }
            }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Clover term (reading O2 / S4-S6; formula BASELINE.json config 4).
 * ------------------------------------------------------------------------------------------ */
static void m3_mul(const cplx* a, const cplx* b, cplx* c) { /* c = a b ; c must not alias */
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx t = 0;
            for (int k = 0; k < 3; k++) t += a[3 * i + k] * b[3 * k + j];
            c[3 * i + j] = t;
        }
}
static void m3_dag(const cplx* a, cplx* c) {
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) c[3 * i + j] = conj(a[3 * j + i]);
}
/* product of four matrices, with a per-factor dagger flag */
static void m3_prod4(const cplx* a, int da, const cplx* b, int db, const cplx* c, int dc, const cplx* d, int dd, cplx* out) {
    cplx A[9], B[9], C[9], D[9], t1[9], t2[9];
    if (da) m3_dag(a, A); else memcpy(A, a, sizeof A);
    if (db) m3_dag(b, B); else memcpy(B, b, sizeof B);
    if (dc) m3_dag(c, C); else memcpy(C, c, sizeof C);
    if (dd) m3_dag(d, D); else memcpy(D, d, sizeof D);
    m3_mul(A, B, t1);
    m3_mul(t1, C, t2);
    m3_mul(t2, D, out);
}

/* F_mu_nu(x) = (Q_mu_nu - Q_mu_nu^dagger)/(8 i), Q = sum of the four plaquette leaves that start and
 * end at x, counter-clockwise in the mu-nu plane (Appendix A.3).  No boundary phases (closed loops).
 *   Q = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
 *     + U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
 *     + U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
 *     + U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag                                         */
static void field_strength_site(const int* L, const cplx* U, long s, int mu, int nu, int traceless, cplx* F /*9*/) {
    int x[4];
    coords(L, s, x);
#define LINK(site, dir) (U + 9 * (4 * (site) + (dir)))
    int xm[4], xn[4];
    long s_pm = shifted(L, x, mu, +1), s_pn = shifted(L, x, nu, +1);
    long s_mm = shifted(L, x, mu, -1), s_mn = shifted(L, x, nu, -1);
    coords(L, s_mm, xm);
    coords(L, s_mn, xn);
    long s_mm_pn = shifted(L, xm, nu, +1); /* x - mu + nu */
    long s_mm_mn = shifted(L, xm, nu, -1); /* x - mu - nu */
    long s_pm_mn = shifted(L, xn, mu, +1); /* x + mu - nu */
    cplx leaf[9], Q[9];
    memset(Q, 0, sizeof Q);
    m3_prod4(LINK(s, mu), 0, LINK(s_pm, nu), 0, LINK(s_pn, mu), 1, LINK(s, nu), 1, leaf);
    for (int e = 0; e < 9; e++) Q[e] += leaf[e];
    m3_prod4(LINK(s, nu), 0, LINK(s_mm_pn, mu), 1, LINK(s_mm, nu), 1, LINK(s_mm, mu), 0, leaf);
    for (int e = 0; e < 9; e++) Q[e] += leaf[e];
    m3_prod4(LINK(s_mm, mu), 1, LINK(s_mm_mn, nu), 1, LINK(s_mm_mn, mu), 0, LINK(s_mn, nu), 0, leaf);
    for (int e = 0; e < 9; e++) Q[e] += leaf[e];
    m3_prod4(LINK(s_mn, nu), 1, LINK(s_mn, mu), 0, LINK(s_pm_mn, nu), 0, LINK(s, mu), 1, leaf);
    for (int e = 0; e < 9; e++) Q[e] += leaf[e];
#undef LINK
    cplx Qd[9];
    m3_dag(Q, Qd);
    for (int e = 0; e < 9; e++) F[e] = (Q[e] - Qd[e]) / (8.0 * II);
    if (traceless) { /* reading S5: off by default */
        cplx tr = (F[0] + F[4] + F[8]) / 3.0;
        F[0] -= tr; F[4] -= tr; F[8] -= tr;
    }
}

/* F[s][3][3] for one plane (mu,nu) on the whole lattice. */
int bqo_field_strength(const int* L, const double* U, int mu, int nu, int traceless, double* F) {
    long V = volume(L);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) field_strength_site(L, (const cplx*)U, s, mu, nu, traceless, (cplx*)F + 9 * s);
    return 0;
}

/* A(x) = 1 - csw*kappa * sum_{mu<nu} sigma_mu_nu (x) F_mu_nu(x), dense 12x12 per site (reading O2):
 *   A[(sp,a),(sq,b)] = delta - csw*kappa * sum_{mu<nu} sigma_mu_nu[sp][sq] * F_mu_nu[a][b]          */
int bqo_clover_build(const int* L, const double* U, double csw, double kappa, int traceless, double* A_) {
    long V = volume(L);
    cplx* A = (cplx*)A_;
    cplx sig[6][4][4];
    int pl[6][2], np = 0;
    for (int mu = 0; mu < 4; mu++)
        for (int nu = mu + 1; nu < 4; nu++) {
            pl[np][0] = mu; pl[np][1] = nu;
            sigma_munu(mu, nu, sig[np]);
            np++;
        }
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) {
        cplx* As = A + 144 * s;
        for (int i = 0; i < 144; i++) As[i] = 0;
        for (int i = 0; i < 12; i++) As[13 * i] = 1.0;
        for (int p = 0; p < 6; p++) {
            cplx F[9];
            field_strength_site(L, (const cplx*)U, s, pl[p][0], pl[p][1], traceless, F);
            for (int sp = 0; sp < 4; sp++)
                for (int sq = 0; sq < 4; sq++)
                    for (int a = 0; a < 3; a++)
                        for (int b = 0; b < 3; b++)
                            As[12 * (3 * sp + a) + (3 * sq + b)] -= csw * kappa * sig[p][sp][sq] * F[3 * a + b];
        }
    }
    return 0;
}

/* Invert a dense 12x12 complex matrix per site: Gauss-Jordan with partial pivoting (general LU-style;
 * deliberately NOT the 2x(6x6) Cholesky route the GPU takes).  Returns the number of singular sites. */
int bqo_site_matrix_invert(long V, const double* A_, double* Ainv_) {
    const cplx* A = (const cplx*)A_;
    cplx* Ainv = (cplx*)Ainv_;
    int nsing = 0;
#pragma omp parallel for schedule(static) reduction(+ : nsing)
    for (long s = 0; s < V; s++) {
        cplx M[12][24];
        for (int i = 0; i < 12; i++)
            for (int j = 0; j < 12; j++) {
                M[i][j] = A[144 * s + 12 * i + j];
                M[i][12 + j] = (i == j) ? 1.0 : 0.0;
            }
        int bad = 0;
        for (int c = 0; c < 12; c++) {
            int piv = c;
            double best = cabs(M[c][c]);
            for (int r = c + 1; r < 12; r++)
                if (cabs(M[r][c]) > best) { best = cabs(M[r][c]); piv = r; }
            if (best == 0.0) { bad = 1; break; }
            if (piv != c)
                for (int j = 0; j < 24; j++) { cplx t = M[c][j]; M[c][j] = M[piv][j]; M[piv][j] = t; }
            cplx inv = 1.0 / M[c][c];
            for (int j = 0; j < 24; j++) M[c][j] *= inv;
            for (int r = 0; r < 12; r++)
                if (r != c) {
                    cplx f = M[r][c];
                    if (f != 0)
                        for (int j = 0; j < 24; j++) M[r][j] -= f * M[c][j];
                }
        }
        nsing += bad;
        for (int i = 0; i < 12; i++)
            for (int j = 0; j < 12; j++) Ainv[144 * s + 12 * i + j] = bad ? NAN : M[i][12 + j];
    }
    return nsing;
}

/* out(x) = A(x) in(x), dense 12x12 per site. */
int bqo_site_matrix_apply(long V, const double* A_, const double* in_, double* out_) {
    const cplx *A = (const cplx*)A_, *in = (const cplx*)in_;
    cplx* out = (cplx*)out_;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++)
        for (int i = 0; i < 12; i++) {
            cplx c = 0;
            for (int j = 0; j < 12; j++) c += A[144 * s + 12 * i + j] * in[12 * s + j];
            out[12 * s + i] = c;
        }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * BiCGStab on the FULL (not even-odd preconditioned) D — reading O4, textbook van der Vorst form:
 *   <a,b> = sum conj(a_i) b_i.  x <- x0; r <- b - A x; rhat <- r; rho = alpha = omega = 1; v = p = 0.
 *   repeat: rho' = <rhat,r>; beta = (rho'/rho)(alpha/omega); rho = rho'; p = r + beta (p - omega v);
 *           v = A p; alpha = rho/<rhat,v>; s = r - alpha v; t = A s; omega = <t,s>/<t,t>;
 *           x += alpha p + omega s; r = s - omega t;
 *   stop when |r|/|b| <= tol, then recompute the true residual; if it exceeds tol, restart from x.
 * Outputs: iters = total iterations, relres = final TRUE relative residual |b - D x|/|b|.
 * Returns 0 converged, 1 max_iter reached, 2 breakdown (rho or <t,t> or <rhat,v> exactly zero).
 * ------------------------------------------------------------------------------------------ */
static cplx vdot(long n, const cplx* a, const cplx* b) {
    double re = 0, im = 0;
#pragma omp parallel for schedule(static) reduction(+ : re, im)
    for (long i = 0; i < n; i++) {
        cplx c = conj(a[i]) * b[i];
        re += creal(c);
        im += cimag(c);
    }
    return re + II * im;
}
static double vnorm2(long n, const cplx* a) { return creal(vdot(n, a, a)); }

int bqo_bicgstab(const int* L, const double* bc, const double* U, double kappa, const double* A,
                 const double* b_, double* x_, double tol, int max_iter, int* iters, double* relres, int* restarts) {
    long V = volume(L), n = 12 * V;
    const cplx* b = (const cplx*)b_;
    cplx* x = (cplx*)x_;
    cplx* r = malloc(n * sizeof(cplx));
    cplx* rhat = malloc(n * sizeof(cplx));
    cplx* p = malloc(n * sizeof(cplx));
    cplx* v = malloc(n * sizeof(cplx));
    cplx* sv = malloc(n * sizeof(cplx));
    cplx* t = malloc(n * sizeof(cplx));
    if (!r || !rhat || !p || !v || !sv || !t) return -1;
    double bnorm = sqrt(vnorm2(n, b));
    int it = 0, status = 1, nrestart = 0;
    double rel = 0;
    if (bnorm == 0.0) {
        for (long i = 0; i < n; i++) x[i] = 0;
        *iters = 0; *relres = 0; *restarts = 0;
        free(r); free(rhat); free(p); free(v); free(sv); free(t);
        return 0;
    }
    for (;;) {
        /* (re)start: true residual */
        bqo_dirac_apply(L, bc, U, kappa, A, (const double*)x, (double*)t);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) { r[i] = b[i] - t[i]; rhat[i] = r[i]; p[i] = 0; v[i] = 0; }
        rel = sqrt(vnorm2(n, r)) / bnorm;
        if (rel <= tol) { status = 0; break; }
        if (it >= max_iter) { status = 1; break; }
        if (nrestart > 50) { status = 1; break; }
        cplx rho = 1, alpha = 1, omega = 1;
        int inner_done = 0;
        while (it < max_iter) {
            cplx rho1 = vdot(n, rhat, r);
            if (rho1 == 0) { status = 2; inner_done = 2; break; }
            cplx beta = (rho1 / rho) * (alpha / omega);
            rho = rho1;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) p[i] = r[i] + beta * (p[i] - omega * v[i]);
            bqo_dirac_apply(L, bc, U, kappa, A, (const double*)p, (double*)v);
            cplx rv = vdot(n, rhat, v);
            if (rv == 0) { status = 2; inner_done = 2; break; }
            alpha = rho / rv;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) sv[i] = r[i] - alpha * v[i];
            bqo_dirac_apply(L, bc, U, kappa, A, (const double*)sv, (double*)t);
            cplx ts = vdot(n, t, sv);
            double tt = vnorm2(n, t);
            if (tt == 0) { status = 2; inner_done = 2; break; }
            omega = ts / tt;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) {
                x[i] += alpha * p[i] + omega * sv[i];
                r[i] = sv[i] - omega * t[i];
            }
            it++;
            if (sqrt(vnorm2(n, r)) / bnorm <= tol) { inner_done = 1; break; }
        }
        if (inner_done == 2) break;
        nrestart++; /* loop back: recompute the true residual, stop or restart from the current x */
        if (inner_done == 0) { /* max_iter: report the true residual and leave */
            bqo_dirac_apply(L, bc, U, kappa, A, (const double*)x, (double*)t);
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) r[i] = b[i] - t[i];
            rel = sqrt(vnorm2(n, r)) / bnorm;
            status = (rel <= tol) ? 0 : 1;
            break;
        }
    }
    *iters = it;
    *relres = rel;
    *restarts = nrestart > 0 ? nrestart - 1 : 0;
    free(r); free(rhat); free(p); free(v); free(sv); free(t);
    return status;
}

int bqo_num_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
