// clover.cu — clover term of Eq. 1: build and apply (A5).
//
// "F(x) is a 12x12 Hermitian matrix made of the link variables"; the formula is BASELINE.json
// config 4 / SURVEY O2:  A(x) = 1 - csw kappa sum_{mu<nu} sigma_mu_nu (x) F_mu_nu(x), F_mu_nu = (Q - Q^dag)/(8i),
// Q_mu_nu = the four plaquette leaves that start and end at x (Appendix A.3).  The GPU never forms the 12x12
// matrix: in the Dirac basis, after the spin rotation R of Appendix A.4, A = R diag(B+, B-) R with
//   B+- = 1 + csw kappa sum_k s_k (x) (Bf_k +- Ef_k),  Bf = (F_yz, F_zx, F_xy),  Ef = (F_xt, F_yt, F_zt),
// two Hermitian 6x6 blocks (72 reals per site), inverted by a Cholesky factorisation in fp64.
#include "clover.cuh"

struct c64 { double r, i; };
__device__ __forceinline__ c64 cmul(c64 a, c64 b) { return {a.r * b.r - a.i * b.i, a.r * b.i + a.i * b.r}; }
__device__ __forceinline__ c64 cconj(c64 a) { return {a.r, -a.i}; }
struct M3 { c64 e[9]; };

__device__ void m3_load(const double* U, int s, int mu, bool dag, M3& m) {
    const double* p = U + ((size_t)s * 4 + mu) * 18;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            if (!dag) m.e[3 * i + j] = {p[2 * (3 * i + j)], p[2 * (3 * i + j) + 1]};
            else m.e[3 * i + j] = {p[2 * (3 * j + i)], -p[2 * (3 * j + i) + 1]};
        }
}
__device__ void m3_mul(const M3& a, const M3& b, M3& c) {
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            c64 t = {0, 0};
            for (int k = 0; k < 3; k++) {
                c64 m = cmul(a.e[3 * i + k], b.e[3 * k + j]);
                t.r += m.r;
                t.i += m.i;
            }
            c.e[3 * i + j] = t;
        }
}

struct Site4 { int x[4]; };
__device__ __forceinline__ int site_index(const Geom& g, const Site4& c) {
    return c.x[0] + g.L[0] * (c.x[1] + g.L[1] * (c.x[2] + g.L[2] * c.x[3]));
}
__device__ __forceinline__ Site4 shift(const Geom& g, Site4 c, int mu, int d) {
    int v = c.x[mu] + d;
    if (v < 0) v += g.L[mu];
    if (v >= g.L[mu]) v -= g.L[mu];
    c.x[mu] = v;
    return c;
}

// one leaf: product of four links, each (site, direction, dagger)
__device__ void leaf(const double* U, int s0, int d0, bool g0, int s1, int d1, bool g1, int s2, int d2, bool g2, int s3,
                     int d3, bool g3, M3& acc) {
    M3 a, b, t;
    m3_load(U, s0, d0, g0, a);
    m3_load(U, s1, d1, g1, b);
    m3_mul(a, b, t);
    m3_load(U, s2, d2, g2, b);
    m3_mul(t, b, a);
    m3_load(U, s3, d3, g3, b);
    m3_mul(a, b, t);
    for (int e = 0; e < 9; e++) {
        acc.e[e].r += t.e[e].r;
        acc.e[e].i += t.e[e].i;
    }
}

// F_mu_nu(x) = (Q - Q^dag)/(8i): Hermitian 3x3.  Leaves, counter-clockwise in the mu-nu plane (Appendix A.3):
//   U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
//   U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
//   U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
//   U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
__device__ void field_strength(const Geom& g, const double* U, const Site4& x, int mu, int nu, M3& F) {
    const int s = site_index(g, x);
    const int s_pm = site_index(g, shift(g, x, mu, +1)), s_pn = site_index(g, shift(g, x, nu, +1));
    const Site4 xmm = shift(g, x, mu, -1), xmn = shift(g, x, nu, -1);
    const int s_mm = site_index(g, xmm), s_mn = site_index(g, xmn);
    const int s_mm_pn = site_index(g, shift(g, xmm, nu, +1));
    const int s_mm_mn = site_index(g, shift(g, xmm, nu, -1));
    const int s_pm_mn = site_index(g, shift(g, xmn, mu, +1));
    M3 Q;
    for (int e = 0; e < 9; e++) Q.e[e] = {0, 0};
    leaf(U, s, mu, false, s_pm, nu, false, s_pn, mu, true, s, nu, true, Q);
    leaf(U, s, nu, false, s_mm_pn, mu, true, s_mm, nu, true, s_mm, mu, false, Q);
    leaf(U, s_mm, mu, true, s_mm_mn, nu, true, s_mm_mn, mu, false, s_mn, nu, false, Q);
    leaf(U, s_mn, nu, true, s_mn, mu, false, s_pm_mn, nu, false, s, mu, true, Q);
    // (Q - Q^dag)/(8i):  (a + ib)/(8i) = (b - ia)/8
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            const c64 q = Q.e[3 * i + j], qd = cconj(Q.e[3 * j + i]);
            const double dr = q.r - qd.r, di = q.i - qd.i;
            F.e[3 * i + j] = {di / 8.0, -dr / 8.0};
        }
}

// 36-real packed form of a Hermitian 6x6 (see clover.cuh) <- full matrix
__device__ void pack_herm6(const c64 (*B)[6], double* out) {
    for (int i = 0; i < 6; i++) out[i] = B[i][i].r;
    for (int i = 1; i < 6; i++)
        for (int j = 0; j < i; j++) {
            const int k = i * (i - 1) / 2 + j;
            out[6 + 2 * k] = B[i][j].r;
            out[6 + 2 * k + 1] = B[i][j].i;
        }
}

// inverse of a Hermitian positive-definite 6x6 via Cholesky A = L L^dag, A^-1 = L^-dag L^-1.  false if not PD.
__device__ bool invert_herm6(const c64 (*A)[6], c64 (*Ainv)[6]) {
    c64 L[6][6], Li[6][6];
    for (int i = 0; i < 6; i++)
        for (int j = 0; j < 6; j++) L[i][j] = Li[i][j] = {0, 0};
    for (int j = 0; j < 6; j++) {
        double d = A[j][j].r;
        for (int k = 0; k < j; k++) d -= L[j][k].r * L[j][k].r + L[j][k].i * L[j][k].i;
        if (!(d > 0.0) || !isfinite(d)) return false;
        const double ljj = sqrt(d);
        L[j][j] = {ljj, 0};
        for (int i = j + 1; i < 6; i++) {
            c64 v = A[i][j];
            for (int k = 0; k < j; k++) {
                c64 m = cmul(L[i][k], cconj(L[j][k]));
                v.r -= m.r;
                v.i -= m.i;
            }
            L[i][j] = {v.r / ljj, v.i / ljj};
        }
    }
    // Li = L^-1 (lower triangular) by forward substitution, column by column
    for (int c = 0; c < 6; c++) {
        for (int i = c; i < 6; i++) {
            c64 v = {(i == c) ? 1.0 : 0.0, 0.0};
            for (int k = c; k < i; k++) {
                c64 m = cmul(L[i][k], Li[k][c]);
                v.r -= m.r;
                v.i -= m.i;
            }
            Li[i][c] = {v.r / L[i][i].r, v.i / L[i][i].r};
        }
    }
    for (int i = 0; i < 6; i++)
        for (int j = 0; j < 6; j++) {
            c64 v = {0, 0};
            for (int k = (i > j ? i : j); k < 6; k++) {
                c64 m = cmul(cconj(Li[k][i]), Li[k][j]);
                v.r += m.r;
                v.i += m.i;
            }
            Ainv[i][j] = v;
        }
    return true;
}

// 72 reals of site h into the fp64 clover store: real r -> 16-byte word r/2, slot r%2
__device__ __forceinline__ void store_clover64(double* base, int Vh, int h, const double* c) {
    char* b = reinterpret_cast<char*>(base);
    for (int k = 0; k < 36; k++) *reinterpret_cast<double2*>(b + CloverAddr<BQ_FP64>::word(Vh, h, k)) = make_double2(c[2 * k], c[2 * k + 1]);
}

__global__ void clover_build_kernel(Geom g, const double* __restrict__ U, double ck, double* __restrict__ A_out,
                                    double* __restrict__ Ainv_out, int* __restrict__ singular) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;   // (p, h)
    if (idx >= g.V) return;
    const int p = idx / g.Vh, h = idx % g.Vh;
    Site4 x;
    {
        const int xh = h % g.Lxh;
        int q = h / g.Lxh;
        x.x[1] = q % g.L[1]; q /= g.L[1];
        x.x[2] = q % g.L[2];
        x.x[3] = q / g.L[2];
        x.x[0] = 2 * xh + ((x.x[1] + x.x[2] + x.x[3] + p) & 1);
    }
    // W+-_k = Bf_k +- Ef_k, Bf = (F_yz, F_zx = -F_xz, F_xy), Ef = (F_xt, F_yt, F_zt)
    M3 Bf[3], Ef[3];
    field_strength(g, U, x, 1, 2, Bf[0]);
    field_strength(g, U, x, 2, 0, Bf[1]);
    field_strength(g, U, x, 0, 1, Bf[2]);
    field_strength(g, U, x, 0, 3, Ef[0]);
    field_strength(g, U, x, 1, 3, Ef[1]);
    field_strength(g, U, x, 2, 3, Ef[2]);
    double packed[72], packed_inv[72];
    bool ok = true;
    for (int blk = 0; blk < 2; blk++) {
        const double sg = blk == 0 ? 1.0 : -1.0;
        c64 B[6][6], Bi[6][6];
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
                c64 w[3];
                for (int k = 0; k < 3; k++)
                    w[k] = {Bf[k].e[3 * a + b].r + sg * Ef[k].e[3 * a + b].r, Bf[k].e[3 * a + b].i + sg * Ef[k].e[3 * a + b].i};
                const double d = (a == b) ? 1.0 : 0.0;
                // sum_k s_k (x) W_k: (0,0) = W_z, (1,1) = -W_z, (0,1) = W_x - i W_y, (1,0) = W_x + i W_y
                B[a][b] = {d + ck * w[2].r, ck * w[2].i};
                B[3 + a][3 + b] = {d - ck * w[2].r, -ck * w[2].i};
                B[a][3 + b] = {ck * (w[0].r + w[1].i), ck * (w[0].i - w[1].r)};
                B[3 + a][b] = {ck * (w[0].r - w[1].i), ck * (w[0].i + w[1].r)};
            }
        pack_herm6(B, packed + 36 * blk);
        if (invert_herm6(B, Bi)) pack_herm6(Bi, packed_inv + 36 * blk);
        else {
            ok = false;
            for (int i = 0; i < 36; i++) packed_inv[36 * blk + i] = nan("");
        }
    }
    if (!ok) atomicOr(singular, 1);
    const size_t pb = (size_t)p * CLOVER_REALS * g.Vh;
    store_clover64(A_out + pb, g.Vh, h, packed);
    store_clover64(Ainv_out + pb, g.Vh, h, packed_inv);
}

// fp64 clover store -> fp32 / half store (same word rule: real r -> word r/W, slot r%W)
template <int PREC> __global__ void clover_convert_kernel(int Vh, const double* __restrict__ src, void* __restrict__ dst_) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;   // (p, h)
    if (idx >= 2 * Vh) return;
    const int p = idx / Vh, h = idx % Vh;
    const char* s = reinterpret_cast<const char*>(src + (size_t)p * CLOVER_REALS * Vh);
    float f[72];
    for (int k = 0; k < 36; k++) {
        const double2 d = *reinterpret_cast<const double2*>(s + CloverAddr<BQ_FP64>::word(Vh, h, k));
        f[2 * k] = (float)d.x;
        f[2 * k + 1] = (float)d.y;
    }
    char* dst = static_cast<char*>(dst_) + (size_t)p * CLOVER_REALS * prec_real_bytes(PREC) * Vh;
    if (PREC == BQ_FP32) {
        for (int k = 0; k < 18; k++)
            *reinterpret_cast<float4*>(dst + CloverAddr<BQ_FP32>::word(Vh, h, k)) = make_float4(f[4 * k], f[4 * k + 1], f[4 * k + 2], f[4 * k + 3]);
    } else {
        for (int k = 0; k < 9; k++) *reinterpret_cast<uint4*>(dst + CloverAddr<BQ_HALF>::word(Vh, h, k)) = pack8(f + 8 * k);
    }
}

bq_status bq_clover_build(bq_lattice* lat, double csw, double kappa) {
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "clover build: no gauge field loaded");
    if (lat->sub) return bq_set_error(lat, BQ_EINVAL, "clover term on a sub-lattice: not built (the field strength needs the neighbours' links)");
    if (lat->have_clover && lat->clover_csw == csw && lat->clover_kappa == kappa) return BQ_OK;
    for (int p = 0; p < 3; p++)
        for (int i = 0; i < 2; i++) {
            if (lat->clover[p][i]) cudaFree(lat->clover[p][i]);
            lat->clover[p][i] = nullptr;
        }
    lat->have_clover = false;
    lat->epoch++;
    const Geom& g = lat->g;
    const size_t nb = (size_t)2 * CLOVER_REALS * g.Vh * sizeof(double);
    BQ_CUDA(lat, cudaMalloc(&lat->clover[BQ_FP64][0], nb));
    BQ_CUDA(lat, cudaMalloc(&lat->clover[BQ_FP64][1], nb));
    BQ_CUDA(lat, cudaMemset(lat->d_flag, 0, sizeof(int)));
    clover_build_kernel<<<(g.V + 63) / 64, 64>>>(g, lat->U_canon, csw * kappa, static_cast<double*>(lat->clover[BQ_FP64][0]),
                                                static_cast<double*>(lat->clover[BQ_FP64][1]), lat->d_flag);
    BQ_CHECK_LAUNCH(lat);
    int flag = 0;
    BQ_CUDA(lat, cudaMemcpy(&flag, lat->d_flag, sizeof(int), cudaMemcpyDeviceToHost));
    if (flag) return bq_set_error(lat, BQ_ESINGULAR_CLOVER, "clover block not positive definite (csw=%g kappa=%g)", csw, kappa);
    lat->have_clover = true;
    lat->clover_csw = csw;
    lat->clover_kappa = kappa;
    return BQ_OK;
}

bq_status bq_get_clover(bq_lattice* lat, int prec, int inverse, const void** out) {
    if (!lat->have_clover) return bq_set_error(lat, BQ_ENOCLOVER, "clover term not built");
    if (prec < 0 || prec > 2 || inverse < 0 || inverse > 1) return bq_set_error(lat, BQ_EINVAL, "bad prec/inverse");
    if (!lat->clover[prec][inverse]) {
        const Geom& g = lat->g;
        void* dst = nullptr;
        BQ_CUDA(lat, cudaMalloc(&dst, (size_t)2 * CLOVER_REALS * g.Vh * prec_real_bytes(prec)));
        const double* src = static_cast<const double*>(lat->clover[BQ_FP64][inverse]);
        const int grid = (2 * g.Vh + 127) / 128;
        if (prec == BQ_FP32) clover_convert_kernel<BQ_FP32><<<grid, 128>>>(g.Vh, src, dst);
        else clover_convert_kernel<BQ_HALF><<<grid, 128>>>(g.Vh, src, dst);
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        if (e != cudaSuccess) {
            cudaFree(dst);
            return bq_set_error(lat, BQ_ECUDA, "clover conversion failed: %s", cudaGetErrorString(e));
        }
        lat->clover[prec][inverse] = dst;
    }
    *out = lat->clover[prec][inverse];
    return BQ_OK;
}

template <int PREC>
__global__ void __launch_bounds__(128) clover_mul_kernel(int Vh, void* out, const void* in, const void* __restrict__ cl) {   // out may be in (in-place apply)
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= Vh) return;
    typename Prec<PREC>::comp v[24];
    load_spinor<PREC, true>(in, Vh, h, v);
    clover_site_mul<PREC>(cl, Vh, h, v);
    store_spinor<PREC, true>(out, Vh, h, v);
}

bq_status bq_clover_mul(bq_lattice* lat, void* out, const void* in, const void* cl, int prec, cudaStream_t stream) {
    const int Vh = lat->g.Vh, grid = (Vh + 127) / 128;
    if (prec == BQ_FP64) clover_mul_kernel<BQ_FP64><<<grid, 128, 0, stream>>>(Vh, out, in, cl);
    else if (prec == BQ_FP32) clover_mul_kernel<BQ_FP32><<<grid, 128, 0, stream>>>(Vh, out, in, cl);
    else clover_mul_kernel<BQ_HALF><<<grid, 128, 0, stream>>>(Vh, out, in, cl);
    BQ_CHECK_LAUNCH(lat);
    return BQ_OK;
}

extern "C" bq_status bq_clover_apply(bq_lattice* lat, double csw, double kappa, void* out, const void* in, bq_parity parity,
                                     int inverse, bq_prec prec, void* stream) {
    if (!lat) return BQ_EINVAL;
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "bq_clover_apply: no gauge field loaded");
    if ((out == nullptr) != (in == nullptr)) return bq_set_error(lat, BQ_EINVAL, "bq_clover_apply: only one of out/in is NULL");
    if (prec != BQ_FP64 && prec != BQ_FP32 && prec != BQ_HALF) return bq_set_error(lat, BQ_EINVAL, "bq_clover_apply: bad precision");
    if (parity != BQ_EVEN && parity != BQ_ODD && parity != BQ_FULL) return bq_set_error(lat, BQ_EINVAL, "bq_clover_apply: bad parity");
    BQ_TRY(bq_clover_build(lat, csw, kappa));
    if (!out) return BQ_OK;
    const void* cl = nullptr;
    BQ_TRY(bq_get_clover(lat, prec, inverse ? 1 : 0, &cl));
    const size_t fb = field_bytes_one_parity(lat->g, prec);
    const size_t cb = (size_t)lat->g.Vh * CLOVER_REALS * prec_real_bytes(prec);
    for (int p = 0; p < 2; p++) {
        if (parity != BQ_FULL && p != (int)parity) continue;
        const size_t off = (parity == BQ_FULL) ? p * fb : 0;
        BQ_TRY(bq_clover_mul(lat, static_cast<char*>(out) + off, static_cast<const char*>(in) + off,
                             static_cast<const char*>(cl) + p * cb, prec, static_cast<cudaStream_t>(stream)));
    }
    return BQ_OK;
}
