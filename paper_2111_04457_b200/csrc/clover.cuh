// clover.cuh — site-diagonal clover multiply in the chirality-block form.
// With R = (1/sqrt2) [[1,1],[1,-1]] (x) 1_2 acting on spin, R A R = diag(B+, B-), two Hermitian 6x6 blocks
// (index 3*spin' + colour).  A psi = R diag(B+,B-) R psi: chi+- = u +- l, y+- = B+- chi+-, result
// u' = (y+ + y-)/2, l' = (y+ - y-)/2  (the two 1/sqrt2 folded into one 1/2).  2 x 252 = 504 flop per site.
// Block storage, 36 reals: [0..5] real diagonal, then the strictly lower triangle row by row,
// element (i, j<i) at complex slot k = i(i-1)/2 + j -> reals [6 + 2k, 6 + 2k + 1].
#pragma once

#include "layout.cuh"

template <typename C> __device__ __forceinline__ void herm6_mul(const C* b, const C* x, C* y) {
#pragma unroll
    for (int i = 0; i < 6; i++) {
        y[2 * i] = b[i] * x[2 * i];
        y[2 * i + 1] = b[i] * x[2 * i + 1];
    }
#pragma unroll
    for (int i = 1; i < 6; i++)
#pragma unroll
        for (int j = 0; j < i; j++) {
            const int k = i * (i - 1) / 2 + j;
            const C lr = b[6 + 2 * k], li = b[6 + 2 * k + 1];
            // y_i += L_ij x_j ;  y_j += conj(L_ij) x_i
            y[2 * i] = mad(-li, x[2 * j + 1], mad(lr, x[2 * j], y[2 * i]));
            y[2 * i + 1] = mad(li, x[2 * j], mad(lr, x[2 * j + 1], y[2 * i + 1]));
            y[2 * j] = mad(li, x[2 * i + 1], mad(lr, x[2 * i], y[2 * j]));
            y[2 * j + 1] = mad(-li, x[2 * i], mad(lr, x[2 * i + 1], y[2 * j + 1]));
        }
}

// 36 reals of chirality block BLK (0: B+, 1: B-) of site h.  Clover store: 72 reals per site as 16-byte words (layout.cuh).
template <int PREC, int BLK, bool STREAM = true>
__device__ __forceinline__ void load_clover_block(const void* base, int Vh, int h, typename Prec<PREC>::comp* c) {
    using A = CloverAddr<PREC>;
    const char* b = static_cast<const char*>(base);
    if constexpr (PREC == BQ_FP64) {
#pragma unroll
        for (int k = 0; k < 18; k++) {
            double2 d = ld16<STREAM, double2>(b + A::word(Vh, h, 18 * BLK + k));
            c[2 * k] = d.x;
            c[2 * k + 1] = d.y;
        }
    } else if constexpr (PREC == BQ_FP32) {
#pragma unroll
        for (int k = 0; k < 9; k++) {
            float4 d = ld16<STREAM, float4>(b + A::word(Vh, h, 9 * BLK + k));
            c[4 * k] = d.x; c[4 * k + 1] = d.y; c[4 * k + 2] = d.z; c[4 * k + 3] = d.w;
        }
    } else {
        // 72 halfs = 9 planes of 8; block 0 = planes 0..3 + low half of plane 4, block 1 = high half of 4 + planes 5..8
        uint4 q[4];
#pragma unroll
        for (int k = 0; k < 4; k++) q[k] = ld16<STREAM, uint4>(b + A::word(Vh, h, (BLK ? 5 : 0) + k));
        uint2 d = ld16<STREAM, uint2>(b + A::word(Vh, h, 4) + (BLK ? 8 : 0));
        if (BLK == 0) {
#pragma unroll
            for (int k = 0; k < 4; k++) unpack8(q[k], c + 8 * k);
            unpack4(d, c + 32);
        } else {
            unpack4(d, c);
#pragma unroll
            for (int k = 0; k < 4; k++) unpack8(q[k], c + 4 + 8 * k);
        }
    }
}

// v <- C(x) v for the spinor v (24 reals) of site h, C = the two stored blocks (A or A^-1).
template <int PREC, bool STREAM = true>
__device__ __forceinline__ void clover_site_mul(const void* cl, int Vh, int h, typename Prec<PREC>::comp* v) {
    using C = typename Prec<PREC>::comp;
    C chi[12], yp[12], ym[12];
    {
        C blk[36];
        load_clover_block<PREC, 0, STREAM>(cl, Vh, h, blk);
#pragma unroll
        for (int i = 0; i < 12; i++) chi[i] = v[i] + v[12 + i];
        herm6_mul(blk, chi, yp);
    }
    {
        C blk[36];
        load_clover_block<PREC, 1, STREAM>(cl, Vh, h, blk);
#pragma unroll
        for (int i = 0; i < 12; i++) chi[i] = v[i] - v[12 + i];
        herm6_mul(blk, chi, ym);
    }
#pragma unroll
    for (int i = 0; i < 12; i++) {
        v[i] = C(0.5) * (yp[i] + ym[i]);
        v[12 + i] = C(0.5) * (yp[i] - ym[i]);
    }
}
