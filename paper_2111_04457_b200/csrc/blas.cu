// blas.cu — fused BLAS-1 kernels of the BiCGStab iteration and of the defect-correction outer loop
// (SURVEY.md §8(a) A6, A8, A9).  See blas.cuh for the work-item and reduction design.
#include "blas.cuh"
#include "blas_api.h"

#define BLAS_KERNEL __global__ void __cluster_dims__(BLAS_CLUSTER, 1, 1) __launch_bounds__(BLAS_BLOCK)

// Loop shape shared by all kernels below: a grid-stride loop in which every thread handles UNR items per trip
// (items i0 + u*BLAS_BLOCK), with all loads of a trip issued before any arithmetic, so that each thread keeps
// UNR x (operands) 16-byte requests in flight — BLAS-1 is pure streaming and lives on memory-level parallelism.
// Measured on B200 (32^3x64, one run, +-1%): reductions want 4 items in flight per operand, the read-modify-write
// updates 2, the 5-operand final update 1; 4 CTAs per SM beat 8 everywhere (profiles/r1_blas_launch_shape.txt).
#define BLAS_TRIPS(I, n) for (int i0 = blockIdx.x * (BLAS_BLOCK * UNR) + threadIdx.x; i0 < (n); i0 += gridDim.x * (BLAS_BLOCK * UNR))
#define BLAS_UNROLL(I) _Pragma("unroll") for (int u = 0; u < UNR; u++)
#ifndef BLAS_UNR_REDUCE
#define BLAS_UNR_REDUCE 4
#endif
#ifndef BLAS_UNR_UPDATE
#define BLAS_UNR_UPDATE 2
#endif
#ifndef BLAS_UNR_FINAL
#define BLAS_UNR_FINAL 1
#endif
#define UNR_REDUCE(I) (I::FLAT ? BLAS_UNR_REDUCE : 1)
#define UNR_UPDATE(I) (I::FLAT ? BLAS_UNR_UPDATE : 1)
#define BLAS_IDX (i0 + u * BLAS_BLOCK)

// ---------------------------------------------------------------------------------------------------
// generic reductions
// ---------------------------------------------------------------------------------------------------
template <int PREC> BLAS_KERNEL k_norm2(int Vh, const void* __restrict__ a, RedBuf rb, SolverScalars* sc, int stride) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = UNR_REDUCE(I);
    const int o = blockIdx.y * stride; sc += blockIdx.y; rb = rhs_redbuf(rb);
    C acc = 0;
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        C v[UNR][2 * I::NC];
        BLAS_UNROLL(I) I::load_or_zero(a, Vh, BLAS_IDX, n, v[u], o);
        BLAS_UNROLL(I)
#pragma unroll
        for (int k = 0; k < 2 * I::NC; k++) acc = mad(v[u][k], v[u][k], acc);
    }
    double red[1] = {(double)acc};
    grid_reduce<1>(red, rb, [sc](const double* r) { sc->red[0] = r[0]; });
}

template <int PREC> BLAS_KERNEL k_cdot(int Vh, const void* __restrict__ a, const void* __restrict__ b, RedBuf rb, SolverScalars* sc, int mode,
                                       int stride) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = UNR_REDUCE(I);
    const int o = blockIdx.y * stride; sc += blockIdx.y; rb = rhs_redbuf(rb);
    C re = 0, im = 0;
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        C x[UNR][2 * I::NC], y[UNR][2 * I::NC];
        BLAS_UNROLL(I) {
            I::load_or_zero(a, Vh, BLAS_IDX, n, x[u], o);
            I::load_or_zero(b, Vh, BLAS_IDX, n, y[u], o);
        }
        BLAS_UNROLL(I)
#pragma unroll
        for (int k = 0; k < I::NC; k++) {   // conj(x) y
            re = mad(x[u][2 * k + 1], y[u][2 * k + 1], mad(x[u][2 * k], y[u][2 * k], re));
            im = mad(-x[u][2 * k + 1], y[u][2 * k], mad(x[u][2 * k], y[u][2 * k + 1], im));
        }
    }
    double red[2] = {(double)re, (double)im};
    grid_reduce<2>(red, rb, [sc, mode](const double* r) {
        if (mode == 0) {
            sc->red[0] = r[0];
            sc->red[1] = r[1];
        } else {
            fin_alpha(sc, r);   // (v) alpha = rho / <rhat, v>
        }
    });
}

template <int PREC> BLAS_KERNEL k_caxpy(int Vh, double ar_, double ai_, const void* __restrict__ x, void* __restrict__ y) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = UNR_UPDATE(I);
    const C ar = (C)ar_, ai = (C)ai_;
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        C xv[UNR][2 * I::NC], yv[UNR][2 * I::NC];
        BLAS_UNROLL(I) {
            I::load_or_zero(x, Vh, BLAS_IDX, n, xv[u]);
            I::load_or_zero(y, Vh, BLAS_IDX, n, yv[u]);
        }
        BLAS_UNROLL(I) {
#pragma unroll
            for (int k = 0; k < I::NC; k++) cfma(yv[u] + 2 * k, ar, ai, xv[u] + 2 * k);
            if (BLAS_IDX < n) I::store(y, Vh, BLAS_IDX, yv[u]);
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// BiCGStab steps
// ---------------------------------------------------------------------------------------------------
// r2 = |r|^2; with rhat = r: rho = r2, beta = (rho/1)(1/1) = rho (p = v = 0 makes beta irrelevant), alpha = omega = 1
// stop2s != nullptr: one stopping threshold per right-hand side (device array), else `stop2` for all
template <int PREC> BLAS_KERNEL k_init(int Vh, const void* __restrict__ r, RedBuf rb, SolverScalars* sc, double stop2,
                                       const double* __restrict__ stop2s, int stride) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = UNR_REDUCE(I);
    const int o = blockIdx.y * stride; sc += blockIdx.y; rb = rhs_redbuf(rb);
    if (stop2s) stop2 = stop2s[blockIdx.y];
    C acc = 0;
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        C v[UNR][2 * I::NC];
        BLAS_UNROLL(I) I::load_or_zero(r, Vh, BLAS_IDX, n, v[u], o);
        BLAS_UNROLL(I)
#pragma unroll
        for (int k = 0; k < 2 * I::NC; k++) acc = mad(v[u][k], v[u][k], acc);
    }
    double red[1] = {(double)acc};
    grid_reduce<1>(red, rb, [sc, stop2](const double* r_) {
        sc->r2 = r_[0];
        sc->stop2 = stop2;
        sc->rho[0] = r_[0]; sc->rho[1] = 0;
        sc->beta[0] = 0; sc->beta[1] = 0;
        sc->alpha[0] = 1; sc->alpha[1] = 0;
        sc->omega[0] = 1; sc->omega[1] = 0;
        sc->iters = 0;
        sc->cg = 0;
        sc->done = (r_[0] > stop2) ? 0 : 1;      // also done when r2 is NaN or the threshold is infinite (a finished right-hand side)
    });
}

// ---------------------------------------------------------------------------------------------------
// CG on the normal equations M^dag M e = M^dag r, Hestenes-Stiefel form:
//   r_N = M^dag r ; p = r_N ; rho = |r_N|^2
//   q = M p ; alpha = rho / |q|^2 (hop epilogue, fin_omega) ; t = M^dag q
//   x += alpha p ; r_N -= alpha t ; rho' = |r_N|^2 ; beta = rho'/rho ; rho = rho'      (k_cg_update)
//   p = r_N + beta p                                                                    (k_cg_p)
// stop when |r_N|^2 <= rel2 * |r_N(0)|^2 (rel2 per right-hand side from stop2s, or `rel2`).
// ---------------------------------------------------------------------------------------------------
template <int PREC> BLAS_KERNEL k_cg_init(int Vh, const void* __restrict__ rn, void* __restrict__ p, RedBuf rb, SolverScalars* sc,
                                          double rel2, const double* __restrict__ rel2s, int stride) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = UNR_UPDATE(I);
    const int o = blockIdx.y * stride; sc += blockIdx.y; rb = rhs_redbuf(rb);
    if (rel2s) rel2 = rel2s[blockIdx.y];
    C acc = 0;
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        C v[UNR][2 * I::NC];
        BLAS_UNROLL(I) I::load_or_zero(rn, Vh, BLAS_IDX, n, v[u], o);
        BLAS_UNROLL(I) {
#pragma unroll
            for (int k = 0; k < 2 * I::NC; k++) acc = mad(v[u][k], v[u][k], acc);
            if (BLAS_IDX < n) I::store(p, Vh, BLAS_IDX + o, v[u]);
        }
    }
    double red[1] = {(double)acc};
    grid_reduce<1>(red, rb, [sc, rel2](const double* r_) {
        sc->r2 = r_[0];
        sc->stop2 = rel2 * r_[0];
        sc->rho[0] = r_[0]; sc->rho[1] = 0;
        sc->beta[0] = 0; sc->beta[1] = 0;
        sc->alpha[0] = 0; sc->alpha[1] = 0;
        sc->omega[0] = 1; sc->omega[1] = 0;
        sc->iters = 0;
        sc->cg = 1;
        sc->done = (r_[0] == 0.0 || !(rel2 < 1.0)) ? 1 : 0;   // rel2 >= 1 (or inf): nothing asked of this right-hand side
    });
}

// x += alpha p ; r_N -= alpha t ; |r_N|^2 -> beta, rho.  x: fp32 accumulator when the storage is half.
template <int PREC> BLAS_KERNEL k_cg_update(int Vh, const void* __restrict__ p, const void* __restrict__ t, void* __restrict__ x,
                                            void* __restrict__ rn, RedBuf rb, SolverScalars* sc, int stride, int xstride) {
    using I = Item<PREC>;
    using C = typename I::C;
    const int o = blockIdx.y * stride, xo = blockIdx.y * xstride;
    sc += blockIdx.y; rb = rhs_redbuf(rb);
    if (sc->done) return;
    const C a = (C)sc->alpha[0];
    C r2 = 0;
    const int n = I::count(Vh);
    if constexpr (PREC == BQ_HALF) {
        for (int i = blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n; i += gridDim.x * BLAS_BLOCK) {
            C xv[24], w[24], rv[24];
            typename I::Raw rp, rr, rt;              // all requests of the site in flight before the first conversion
            I::load_raw(p, Vh, i + o, rp);
            I::load_raw(rn, Vh, i + o, rr);
            I::load_raw(t, Vh, i + o, rt);
            load_spinor<BQ_FP32>(x, Vh, i + xo, xv);
            I::unpack(rp, w);
#pragma unroll
            for (int k = 0; k < 24; k++) xv[k] = mad(a, w[k], xv[k]);
            store_spinor<BQ_FP32>(x, Vh, i + xo, xv);
            I::unpack(rr, rv);
            I::unpack(rt, w);
#pragma unroll
            for (int k = 0; k < 24; k++) rv[k] = mad(-a, w[k], rv[k]);
            I::store(rn, Vh, i + o, rv);
            I::requantize(rv);       // the reduction sees r_N as stored
#pragma unroll
            for (int k = 0; k < 24; k++) r2 = mad(rv[k], rv[k], r2);
        }
    } else {
        constexpr int UNR = 1;
        BLAS_TRIPS(I, n) {
            C xv[UNR][2 * I::NC], pv[UNR][2 * I::NC], rv[UNR][2 * I::NC], tv[UNR][2 * I::NC];
            BLAS_UNROLL(I) {
                I::load_or_zero(x, Vh, BLAS_IDX, n, xv[u], xo);
                I::load_or_zero(p, Vh, BLAS_IDX, n, pv[u], o);
                I::load_or_zero(rn, Vh, BLAS_IDX, n, rv[u], o);
                I::load_or_zero(t, Vh, BLAS_IDX, n, tv[u], o);
            }
            BLAS_UNROLL(I) {
#pragma unroll
                for (int k = 0; k < 2 * I::NC; k++) {
                    xv[u][k] = mad(a, pv[u][k], xv[u][k]);
                    rv[u][k] = mad(-a, tv[u][k], rv[u][k]);
                    r2 = mad(rv[u][k], rv[u][k], r2);
                }
                if (BLAS_IDX < n) {
                    I::store(x, Vh, BLAS_IDX + xo, xv[u]);
                    I::store(rn, Vh, BLAS_IDX + o, rv[u]);
                }
            }
        }
    }
    double red[1] = {(double)r2};
    grid_reduce<1>(red, rb, [sc](const double* q) {
        sc->r2 = q[0];
        sc->iters += 1;
        if (q[0] <= sc->stop2) sc->done = 1;
        else if (sc->rho[0] == 0.0) sc->done = 2;
        else { sc->beta[0] = q[0] / sc->rho[0]; sc->beta[1] = 0; }
        sc->rho[0] = q[0];
    });
}

// p = r_N + beta p
template <int PREC> BLAS_KERNEL k_cg_p(int Vh, const void* __restrict__ rn, void* __restrict__ p, const SolverScalars* __restrict__ sc,
                                       int stride) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = UNR_UPDATE(I);
    const int o = blockIdx.y * stride; sc += blockIdx.y;
    if (sc->done) return;
    const C b = (C)sc->beta[0];
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        C rv[UNR][2 * I::NC], pv[UNR][2 * I::NC];
        BLAS_UNROLL(I) {
            I::load_or_zero(rn, Vh, BLAS_IDX, n, rv[u], o);
            I::load_or_zero(p, Vh, BLAS_IDX, n, pv[u], o);
        }
        BLAS_UNROLL(I) {
#pragma unroll
            for (int k = 0; k < 2 * I::NC; k++) rv[u][k] = mad(b, pv[u][k], rv[u][k]);
            if (BLAS_IDX < n) I::store(p, Vh, BLAS_IDX + o, rv[u]);
        }
    }
}

// (i) p = r + beta (p - omega v)
template <int PREC> BLAS_KERNEL k_p_update(int Vh, const void* __restrict__ r, void* __restrict__ p, const void* __restrict__ v,
                                           const SolverScalars* __restrict__ sc, int stride) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = UNR_UPDATE(I);
    const int o = blockIdx.y * stride; sc += blockIdx.y;
    if (sc->done) return;
    const C br = (C)sc->beta[0], bi = (C)sc->beta[1], wr = (C)sc->omega[0], wi = (C)sc->omega[1];
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        C rv[UNR][2 * I::NC], pv[UNR][2 * I::NC], vv[UNR][2 * I::NC];
        BLAS_UNROLL(I) {
            I::load_or_zero(r, Vh, BLAS_IDX, n, rv[u], o);
            I::load_or_zero(p, Vh, BLAS_IDX, n, pv[u], o);
            I::load_or_zero(v, Vh, BLAS_IDX, n, vv[u], o);
        }
        BLAS_UNROLL(I) {
#pragma unroll
            for (int k = 0; k < I::NC; k++) {
                cfma(pv[u] + 2 * k, -wr, -wi, vv[u] + 2 * k);    // p - omega v
                cfma(rv[u] + 2 * k, br, bi, pv[u] + 2 * k);      // r + beta (.)
            }
            if (BLAS_IDX < n) I::store(p, Vh, BLAS_IDX + o, rv[u]);
        }
    }
}

// (ii) s = r - alpha v
template <int PREC> BLAS_KERNEL k_s_update(int Vh, const void* __restrict__ r, const void* __restrict__ v, void* __restrict__ s,
                                           const SolverScalars* __restrict__ sc, int stride) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = UNR_UPDATE(I);
    const int o = blockIdx.y * stride; sc += blockIdx.y;
    if (sc->done) return;
    const C ar = (C)sc->alpha[0], ai = (C)sc->alpha[1];
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        C rv[UNR][2 * I::NC], vv[UNR][2 * I::NC];
        BLAS_UNROLL(I) {
            I::load_or_zero(r, Vh, BLAS_IDX, n, rv[u], o);
            I::load_or_zero(v, Vh, BLAS_IDX, n, vv[u], o);
        }
        BLAS_UNROLL(I) {
#pragma unroll
            for (int k = 0; k < I::NC; k++) cfma(rv[u] + 2 * k, -ar, -ai, vv[u] + 2 * k);
            if (BLAS_IDX < n) I::store(s, Vh, BLAS_IDX + o, rv[u]);
        }
    }
}

// (iii) <t,s>, <t,t> in one pass; omega = <t,s>/<t,t>
template <int PREC> BLAS_KERNEL k_omega(int Vh, const void* __restrict__ t, const void* __restrict__ s, RedBuf rb, SolverScalars* sc,
                                        int stride) {
    using I = Item<PREC>;
    using C = typename I::C;
    constexpr int UNR = UNR_REDUCE(I);
    const int o = blockIdx.y * stride; sc += blockIdx.y; rb = rhs_redbuf(rb);
    C re = 0, im = 0, tt = 0;
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        C x[UNR][2 * I::NC], y[UNR][2 * I::NC];
        BLAS_UNROLL(I) {
            I::load_or_zero(t, Vh, BLAS_IDX, n, x[u], o);
            I::load_or_zero(s, Vh, BLAS_IDX, n, y[u], o);
        }
        BLAS_UNROLL(I)
#pragma unroll
        for (int k = 0; k < I::NC; k++) {
            re = mad(x[u][2 * k + 1], y[u][2 * k + 1], mad(x[u][2 * k], y[u][2 * k], re));
            im = mad(-x[u][2 * k + 1], y[u][2 * k], mad(x[u][2 * k], y[u][2 * k + 1], im));
            tt = mad(x[u][2 * k + 1], x[u][2 * k + 1], mad(x[u][2 * k], x[u][2 * k], tt));
        }
    }
    double red[3] = {(double)re, (double)im, (double)tt};
    grid_reduce<3>(red, rb, [sc](const double* r) { fin_omega(sc, r); });
}

// (iv) x += alpha p + omega s ; r = s - omega t ; |r|^2 ; <rhat, r>   — one pass over 5 inputs, 2 outputs.
// The finaliser prepares the next iteration: rho' = <rhat,r>, beta = (rho'/rho)(alpha/omega), rho = rho'.
template <int PREC> BLAS_KERNEL k_final(int Vh, const void* __restrict__ p, const void* __restrict__ s, const void* __restrict__ t,
                                        const void* __restrict__ rhat, void* __restrict__ x, void* __restrict__ r, RedBuf rb,
                                        SolverScalars* sc, int stride, int xstride) {
    using I = Item<PREC>;
    using C = typename I::C;
    const int o = blockIdx.y * stride, xo = blockIdx.y * xstride;
    sc += blockIdx.y; rb = rhs_redbuf(rb);
    if (sc->done) return;   // converged or broken down in an earlier iteration of this batch: x stays frozen
    const C ar = (C)sc->alpha[0], ai = (C)sc->alpha[1], wr = (C)sc->omega[0], wi = (C)sc->omega[1];
    C r2 = 0, re = 0, im = 0;
    const int n = I::count(Vh);
    if constexpr (PREC == BQ_HALF) {
        for (int i = blockIdx.x * BLAS_BLOCK + threadIdx.x; i < n; i += gridDim.x * BLAS_BLOCK) {
            C xv[24], sv[24], w[24];
            typename I::Raw rp, rs, rt, rh;          // all 22 requests of the site in flight before the first conversion
            I::load_raw(p, Vh, i + o, rp);
            I::load_raw(s, Vh, i + o, rs);
            I::load_raw(t, Vh, i + o, rt);
            I::load_raw(rhat, Vh, i + o, rh);
            load_spinor<BQ_FP32>(x, Vh, i + xo, xv);   // fp32 solution accumulator
            I::unpack(rp, w);
#pragma unroll
            for (int k = 0; k < 12; k++) cfma(xv + 2 * k, ar, ai, w + 2 * k);
            I::unpack(rs, sv);
#pragma unroll
            for (int k = 0; k < 12; k++) cfma(xv + 2 * k, wr, wi, sv + 2 * k);
            store_spinor<BQ_FP32>(x, Vh, i + xo, xv);
            I::unpack(rt, w);
#pragma unroll
            for (int k = 0; k < 12; k++) cfma(sv + 2 * k, -wr, -wi, w + 2 * k);   // r = s - omega t
            I::store(r, Vh, i + o, sv);
            I::requantize(sv);       // reductions see r as stored (rounded to half storage)
            I::unpack(rh, w);
#pragma unroll
            for (int k = 0; k < 12; k++) {
                r2 = mad(sv[2 * k + 1], sv[2 * k + 1], mad(sv[2 * k], sv[2 * k], r2));
                re = mad(w[2 * k + 1], sv[2 * k + 1], mad(w[2 * k], sv[2 * k], re));
                im = mad(-w[2 * k + 1], sv[2 * k], mad(w[2 * k], sv[2 * k + 1], im));
            }
        }
    } else {
        constexpr int U2 = BLAS_UNR_FINAL;    // 5 operands = 5 requests in flight per thread (more was slower)
        for (int i0 = blockIdx.x * (BLAS_BLOCK * U2) + threadIdx.x; i0 < n; i0 += gridDim.x * (BLAS_BLOCK * U2)) {
            C xv[U2][2 * I::NC], pv[U2][2 * I::NC], sv[U2][2 * I::NC], tv[U2][2 * I::NC], hv[U2][2 * I::NC];
#pragma unroll
            for (int u = 0; u < U2; u++) {
                I::load_or_zero(x, Vh, BLAS_IDX, n, xv[u], xo);
                I::load_or_zero(p, Vh, BLAS_IDX, n, pv[u], o);
                I::load_or_zero(s, Vh, BLAS_IDX, n, sv[u], o);
                I::load_or_zero(t, Vh, BLAS_IDX, n, tv[u], o);
                I::load_or_zero(rhat, Vh, BLAS_IDX, n, hv[u], o);
            }
#pragma unroll
            for (int u = 0; u < U2; u++) {
#pragma unroll
                for (int k = 0; k < I::NC; k++) {
                    cfma(xv[u] + 2 * k, ar, ai, pv[u] + 2 * k);
                    cfma(xv[u] + 2 * k, wr, wi, sv[u] + 2 * k);
                    cfma(sv[u] + 2 * k, -wr, -wi, tv[u] + 2 * k);   // r = s - omega t
                    r2 = mad(sv[u][2 * k + 1], sv[u][2 * k + 1], mad(sv[u][2 * k], sv[u][2 * k], r2));
                    re = mad(hv[u][2 * k + 1], sv[u][2 * k + 1], mad(hv[u][2 * k], sv[u][2 * k], re));
                    im = mad(-hv[u][2 * k + 1], sv[u][2 * k], mad(hv[u][2 * k], sv[u][2 * k + 1], im));
                }
                if (BLAS_IDX < n) {
                    I::store(x, Vh, BLAS_IDX + xo, xv[u]);
                    I::store(r, Vh, BLAS_IDX + o, sv[u]);
                }
            }
        }
    }
    double red[3] = {(double)r2, (double)re, (double)im};
    grid_reduce<3>(red, rb, [sc](const double* q) {
        sc->r2 = q[0];
        sc->iters += 1;
        const double rho_new[2] = {q[1], q[2]};
        if (q[0] <= sc->stop2) {
            sc->done = 1;
        } else if ((rho_new[0] == 0.0 && rho_new[1] == 0.0) || (sc->omega[0] == 0.0 && sc->omega[1] == 0.0)) {
            sc->done = 2;
        } else {
            double a[2], b[2];
            cdiv(rho_new, sc->rho, a);
            cdiv(sc->alpha, sc->omega, b);
            cmuld(a, b, sc->beta);
        }
        sc->rho[0] = rho_new[0];
        sc->rho[1] = rho_new[1];
    });
}

// ---------------------------------------------------------------------------------------------------
// outer loop (fp64)
// ---------------------------------------------------------------------------------------------------
BLAS_KERNEL k_outer_residual(int Vh, const void* __restrict__ b, const void* __restrict__ t, void* __restrict__ r, RedBuf rb,
                             SolverScalars* sc, int bstride, int stride) {
    using I = Item<BQ_FP64>;
    constexpr int UNR = UNR_UPDATE(I);
    const int bo = blockIdx.y * bstride, o = blockIdx.y * stride; sc += blockIdx.y; rb = rhs_redbuf(rb);
    double acc = 0;
    const int n = I::count(Vh);
    BLAS_TRIPS(I, n) {
        double bv[UNR][2], tv[UNR][2];
        BLAS_UNROLL(I) {
            I::load_or_zero(b, Vh, BLAS_IDX, n, bv[u], bo);
            I::load_or_zero(t, Vh, BLAS_IDX, n, tv[u], o);
        }
        BLAS_UNROLL(I) {
            bv[u][0] -= tv[u][0];
            bv[u][1] -= tv[u][1];
            if (BLAS_IDX < n) I::store(r, Vh, BLAS_IDX + o, bv[u]);
            acc += bv[u][0] * bv[u][0] + bv[u][1] * bv[u][1];
        }
    }
    double red[1] = {acc};
    grid_reduce<1>(red, rb, [sc](const double* q) {
        sc->r2 = q[0];
        sc->red[0] = q[0];
        sc->rnorm = sqrt(q[0]);
        sc->scale = q[0] > 0.0 ? 1.0 / sqrt(q[0]) : 0.0;
    });
}

template <int PREC_LO> __global__ void __launch_bounds__(128) k_to_low(int Vh, const void* __restrict__ r64, void* __restrict__ lo,
                                                                      const SolverScalars* __restrict__ sc, int stride64, int stride_lo) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= Vh) return;
    sc += blockIdx.y;
    const double sca = sc->scale;
    double v[24];
    load_spinor<BQ_FP64, true>(r64, Vh, h + blockIdx.y * stride64, v);     // strides in sites
    typename Prec<PREC_LO>::comp w[24];
#pragma unroll
    for (int i = 0; i < 24; i++) w[i] = (typename Prec<PREC_LO>::comp)(v[i] * sca);
    store_spinor<PREC_LO>(lo, Vh, h + blockIdx.y * stride_lo, w);
}

template <int EPREC> __global__ void __launch_bounds__(128) k_accumulate(int Vh, const void* __restrict__ e, void* __restrict__ x64,
                                                                        const SolverScalars* __restrict__ sc, int estride, int xstride) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= Vh) return;
    sc += blockIdx.y;
    const int he = h + blockIdx.y * estride, hx = h + blockIdx.y * xstride;     // strides in sites
    const double rn = sc->rnorm;
    typename Prec<EPREC>::comp ev[24];
    load_spinor<EPREC, true>(e, Vh, he, ev);
    double xv[24];
    load_spinor<BQ_FP64, true>(x64, Vh, hx, xv);
#pragma unroll
    for (int i = 0; i < 24; i++) xv[i] += rn * (double)ev[i];
    store_spinor<BQ_FP64>(x64, Vh, hx, xv);
}

// ---------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------
bq_status blas_ctx_create(bq_lattice* lat, BlasCtx* c) {
    int dev = 0, sms = 0;
    BQ_CUDA(lat, cudaGetDevice(&dev));
    BQ_CUDA(lat, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    c->Vh = lat->g.Vh;
    // persistent-style grid: BLAS_CTAS_PER_SM CTAs of 256 threads per SM (a multiple of the SM count and of the
    // cluster size), trimmed for small lattices so that no cluster is empty-handed more than necessary
    int grid = sms * BLAS_CTAS_PER_SM;
    const int need = (12 * lat->g.Vh + BLAS_BLOCK - 1) / BLAS_BLOCK;
    if (grid > need) grid = need;
    grid = ((grid + BLAS_CLUSTER - 1) / BLAS_CLUSTER) * BLAS_CLUSTER;
    c->grid = grid;
    // a stream of its own (blocking: ordered with the legacy default stream exactly like the legacy stream itself), because
    // the legacy stream cannot be captured into a CUDA graph (solve.cu replays batches of iterations as graphs)
    c->stream = nullptr;
    BQ_CUDA(lat, cudaStreamCreateWithFlags(&c->stream, cudaStreamDefault));
    c->nrhs = 1; c->stride = 0; c->xstride = 0; c->stride64 = 0;
    c->cap = 0; c->partials = nullptr; c->ticket = nullptr; c->sc = nullptr; c->stop2s = nullptr;
    return blas_ctx_reserve(lat, c, 1);
}

// scratch and solver states for up to nrhs right-hand sides
bq_status blas_ctx_reserve(bq_lattice* lat, BlasCtx* c, int nrhs) {
    if (nrhs <= c->cap) return BQ_OK;
    blas_ctx_destroy(c);
    c->pstride = 4 * (c->grid / BLAS_CLUSTER);
    // all or nothing: on any failure the context is left empty (cap = 0, no pointer set), never half allocated
    cudaError_t e = cudaMalloc(&c->partials, sizeof(double) * c->pstride * nrhs);
    if (e == cudaSuccess) e = cudaMalloc(&c->ticket, sizeof(unsigned int) * nrhs);
    if (e == cudaSuccess) e = cudaMemset(c->ticket, 0, sizeof(unsigned int) * nrhs);
    if (e == cudaSuccess) e = cudaMalloc(&c->sc, sizeof(SolverScalars) * nrhs);
    if (e == cudaSuccess) e = cudaMemset(c->sc, 0, sizeof(SolverScalars) * nrhs);
    if (e == cudaSuccess) e = cudaMalloc(&c->stop2s, sizeof(double) * nrhs);
    if (e != cudaSuccess) {
        blas_ctx_destroy(c);
        return bq_set_error(lat, e == cudaErrorMemoryAllocation ? BQ_ENOMEM : BQ_ECUDA, "solver scratch for %d right-hand sides: %s", nrhs,
                            cudaGetErrorString(e));
    }
    c->cap = nrhs;
    return BQ_OK;
}

void blas_ctx_destroy(BlasCtx* c) {
    if (c->partials) cudaFree(c->partials);
    if (c->ticket) cudaFree(c->ticket);
    if (c->sc) cudaFree(c->sc);
    if (c->stop2s) cudaFree(c->stop2s);
    c->partials = nullptr; c->ticket = nullptr; c->sc = nullptr; c->stop2s = nullptr; c->cap = 0;
}

// c.nrhs right-hand sides per launch (gridDim.y).  The context holds the distances between the fields of one operand in
// BYTES; the kernels want them in items (blas.cuh): 16-byte chunks for fp64 / fp32 vectors, sites for half storage.
static int items_of(int prec, size_t bytes) { return (int)(bytes / (prec == BQ_HALF ? spinor_site_bytes(BQ_HALF) : 16)); }
// the solution accumulator of k_final / k_cg_update: an fp32 field read site-wise when the storage is half
static int x_items_of(int prec, size_t bytes) { return (int)(bytes / (prec == BQ_HALF ? spinor_site_bytes(BQ_FP32) : 16)); }
static int sites_of(int prec, size_t bytes) { return (int)(bytes / spinor_site_bytes(prec)); }
#define DISPATCH_PREC(prec, KERNEL, ...)                                                          \
    do {                                                                                          \
        const dim3 g_(c.grid, c.nrhs);                                                            \
        if ((prec) == BQ_FP64) KERNEL<BQ_FP64><<<g_, BLAS_BLOCK, 0, c.stream>>>(__VA_ARGS__);     \
        else if ((prec) == BQ_FP32) KERNEL<BQ_FP32><<<g_, BLAS_BLOCK, 0, c.stream>>>(__VA_ARGS__); \
        else KERNEL<BQ_HALF><<<g_, BLAS_BLOCK, 0, c.stream>>>(__VA_ARGS__);                       \
        BQ_CHECK_LAUNCH(lat);                                                                     \
        return BQ_OK;                                                                             \
    } while (0)

bq_status blas_norm2(bq_lattice* lat, const BlasCtx& c, int prec, const void* a) {
    RedBuf rb{c.partials, c.ticket, c.pstride};
    DISPATCH_PREC(prec, k_norm2, c.Vh, a, rb, c.sc, items_of(prec, c.stride));
}
bq_status blas_cdot(bq_lattice* lat, const BlasCtx& c, int prec, const void* a, const void* b) {
    RedBuf rb{c.partials, c.ticket, c.pstride};
    DISPATCH_PREC(prec, k_cdot, c.Vh, a, b, rb, c.sc, 0, items_of(prec, c.stride));
}
bq_status blas_caxpy(bq_lattice* lat, const BlasCtx& c, int prec, double ar, double ai, const void* x, void* y) {
    const BlasCtx one = blas_single(c);
    {
        const BlasCtx& c = one;
        DISPATCH_PREC(prec, k_caxpy, c.Vh, ar, ai, x, y);
    }
    return BQ_OK;
}
bq_status bicg_init(bq_lattice* lat, const BlasCtx& c, int prec, const void* r, double stop2, bool per_rhs_stop2) {
    RedBuf rb{c.partials, c.ticket, c.pstride};
    DISPATCH_PREC(prec, k_init, c.Vh, r, rb, c.sc, stop2, per_rhs_stop2 ? c.stop2s : nullptr, items_of(prec, c.stride));
}
bq_status cg_init(bq_lattice* lat, const BlasCtx& c, int prec, const void* rn, void* p, double rel2, bool per_rhs_rel2) {
    RedBuf rb{c.partials, c.ticket, c.pstride};
    DISPATCH_PREC(prec, k_cg_init, c.Vh, rn, p, rb, c.sc, rel2, per_rhs_rel2 ? c.stop2s : nullptr, items_of(prec, c.stride));
}
bq_status cg_update(bq_lattice* lat, const BlasCtx& c, int prec, const void* p, const void* t, void* x, void* rn) {
    RedBuf rb{c.partials, c.ticket, c.pstride};
    DISPATCH_PREC(prec, k_cg_update, c.Vh, p, t, x, rn, rb, c.sc, items_of(prec, c.stride), x_items_of(prec, c.xstride));
}
bq_status cg_p_update(bq_lattice* lat, const BlasCtx& c, int prec, const void* rn, void* p) {
    DISPATCH_PREC(prec, k_cg_p, c.Vh, rn, p, c.sc, items_of(prec, c.stride));
}
bq_status bicg_p_update(bq_lattice* lat, const BlasCtx& c, int prec, const void* r, void* p, const void* v) {
    DISPATCH_PREC(prec, k_p_update, c.Vh, r, p, v, c.sc, items_of(prec, c.stride));
}
bq_status bicg_alpha(bq_lattice* lat, const BlasCtx& c, int prec, const void* rhat, const void* v) {
    RedBuf rb{c.partials, c.ticket, c.pstride};
    DISPATCH_PREC(prec, k_cdot, c.Vh, rhat, v, rb, c.sc, 1, items_of(prec, c.stride));
}
bq_status bicg_s_update(bq_lattice* lat, const BlasCtx& c, int prec, const void* r, const void* v, void* s) {
    DISPATCH_PREC(prec, k_s_update, c.Vh, r, v, s, c.sc, items_of(prec, c.stride));
}
bq_status bicg_omega(bq_lattice* lat, const BlasCtx& c, int prec, const void* t, const void* s) {
    RedBuf rb{c.partials, c.ticket, c.pstride};
    DISPATCH_PREC(prec, k_omega, c.Vh, t, s, rb, c.sc, items_of(prec, c.stride));
}
bq_status bicg_final(bq_lattice* lat, const BlasCtx& c, int prec, const void* p, const void* s, const void* t, const void* rhat,
                     void* x, void* r) {
    RedBuf rb{c.partials, c.ticket, c.pstride};
    DISPATCH_PREC(prec, k_final, c.Vh, p, s, t, rhat, x, r, rb, c.sc, items_of(prec, c.stride), x_items_of(prec, c.xstride));
}

bq_status outer_residual(bq_lattice* lat, const BlasCtx& c, const void* b, size_t bstride, const void* t, void* r) {
    RedBuf rb{c.partials, c.ticket, c.pstride};
    k_outer_residual<<<dim3(c.grid, c.nrhs), BLAS_BLOCK, 0, c.stream>>>(c.Vh, b, t, r, rb, c.sc, items_of(BQ_FP64, bstride), items_of(BQ_FP64, c.stride64));
    BQ_CHECK_LAUNCH(lat);
    return BQ_OK;
}
bq_status outer_to_low(bq_lattice* lat, const BlasCtx& c, int prec_lo, const void* r64, void* lo) {
    const dim3 grid((c.Vh + 127) / 128, c.nrhs);
    if (prec_lo == BQ_FP64) k_to_low<BQ_FP64><<<grid, 128, 0, c.stream>>>(c.Vh, r64, lo, c.sc, sites_of(BQ_FP64, c.stride64), sites_of(prec_lo, c.stride));
    else if (prec_lo == BQ_FP32) k_to_low<BQ_FP32><<<grid, 128, 0, c.stream>>>(c.Vh, r64, lo, c.sc, sites_of(BQ_FP64, c.stride64), sites_of(prec_lo, c.stride));
    else k_to_low<BQ_HALF><<<grid, 128, 0, c.stream>>>(c.Vh, r64, lo, c.sc, sites_of(BQ_FP64, c.stride64), sites_of(prec_lo, c.stride));
    BQ_CHECK_LAUNCH(lat);
    return BQ_OK;
}
bq_status outer_accumulate(bq_lattice* lat, const BlasCtx& c, int e_prec, const void* e, void* x64, size_t x64stride) {
    const dim3 grid((c.Vh + 127) / 128, c.nrhs);
    if (e_prec == BQ_FP64) k_accumulate<BQ_FP64><<<grid, 128, 0, c.stream>>>(c.Vh, e, x64, c.sc, sites_of(e_prec, c.xstride), sites_of(BQ_FP64, x64stride));
    else if (e_prec == BQ_FP32) k_accumulate<BQ_FP32><<<grid, 128, 0, c.stream>>>(c.Vh, e, x64, c.sc, sites_of(e_prec, c.xstride), sites_of(BQ_FP64, x64stride));
    else return bq_set_error(lat, BQ_EINVAL, "outer_accumulate: accumulator cannot be half");
    BQ_CHECK_LAUNCH(lat);
    return BQ_OK;
}
