// layout.cuh — device-side access to the even-odd SoA stores (include/bq.h "Internal field layout").
//
// A site's S bytes are cut into 16-byte words: word k holds reals [k*W, (k+1)*W) of the site (W = 16/sizeof(real));
// leftover reals (18 = 4*4+2 floats, 18 = 2*8+2 halfs, 12 = 8+4 halfs) form a narrower trailing word, and half
// spinors carry a trailing fp32 word with the per-site norm (reading S11).  Sites are grouped in TILES of 8
// consecutive half indices (Vh is always a multiple of 8); inside a tile word k of the 8 sites is one contiguous
// 128-byte "plane" (a full cache line), the planes follow one another, and the tiles follow one another:
//     address(h, k) = base + (h >> 3) * 8*S + k*128 + (h & 7)*16
// A warp's 32 consecutive sites therefore read four whole 128-byte lines per load instruction (the B200 analogue of
// the paper's "coalesced" GPU layout, and of its site-vectorised SoA layouts), every
// word of a site sits at a compile-time offset from the first (one address computation per gather instead of one
// per plane), and the 4 tiles a warp gathers are one contiguous run of 32*S bytes in DRAM.
// BQ_TILED = 0 selects the plane-major form (plane k of all Vh sites contiguous), kept for A/B measurements.
#pragma once

#include "bq_internal.h"

#ifndef BQ_TILED
#define BQ_TILED 1
#endif

// Byte offsets inside a store of S bytes per site.
template <int S> struct Addr {
    static constexpr int N16 = S / 16, R = S % 16;   // full 16-byte words, width of the trailing word (0, 4 or 8)
    __device__ __forceinline__ static size_t word(int Vh, int h, int k) {
#if BQ_TILED
        return (size_t)(h >> 3) * (8 * S) + (size_t)(k * 128 + (h & 7) * 16);
#else
        return ((size_t)k * Vh + h) * 16;
#endif
    }
    __device__ __forceinline__ static size_t tail(int Vh, int h) {
#if BQ_TILED
        return (size_t)(h >> 3) * (8 * S) + (size_t)(N16 * 128 + (h & 7) * R);
#else
        return (size_t)N16 * Vh * 16 + (size_t)h * R;
#endif
    }
};
template <int PREC> struct SpinorAddr : Addr<PREC == BQ_FP64 ? 192 : (PREC == BQ_FP32 ? 96 : 52)> {};
template <int PREC, int RECON> struct LinkAddr
    : Addr<(RECON == BQ_RECON12 ? 12 : 18) * (PREC == BQ_FP64 ? 8 : (PREC == BQ_FP32 ? 4 : 2))> {};
template <int PREC> struct CloverAddr : Addr<72 * (PREC == BQ_FP64 ? 8 : (PREC == BQ_FP32 ? 4 : 2))> {};

template <int PREC> struct Prec;
template <> struct Prec<BQ_FP64> { using real = double; using comp = double; };
template <> struct Prec<BQ_FP32> { using real = float; using comp = float; };
template <> struct Prec<BQ_HALF> { using real = __half; using comp = float; };

// a*b + c in one rounding, spelled out so that complex products compile to FMA chains (1 FMUL + n FFMA).
__device__ __forceinline__ float mad(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double mad(double a, double b, double c) { return __fma_rn(a, b, c); }

// ---- raw loads with a cache policy: default = plain ld.global (L1-cached, normal L2 policy: spinors, of which
// every site is read by 8 neighbours and must survive in L2); STREAM = ld.global.cs, evict-first streaming
// (links, clover blocks, BLAS operands: read exactly once).  Both are coherent loads, so a kernel may read and
// then overwrite the same element (in-place updates) without touching the non-coherent path. ----
template <bool STREAM, typename V> __device__ __forceinline__ V ld16(const void* p) {
    if (STREAM) return __ldcs(reinterpret_cast<const V*>(p));
    return *reinterpret_cast<const V*>(p);
}

__device__ __forceinline__ void unpack8(const uint4& q, float* f) {
    const __half2* h = reinterpret_cast<const __half2*>(&q);
#pragma unroll
    for (int i = 0; i < 4; i++) {
        float2 t = __half22float2(h[i]);
        f[2 * i] = t.x;
        f[2 * i + 1] = t.y;
    }
}
__device__ __forceinline__ void unpack4(const uint2& q, float* f) {
    const __half2* h = reinterpret_cast<const __half2*>(&q);
#pragma unroll
    for (int i = 0; i < 2; i++) {
        float2 t = __half22float2(h[i]);
        f[2 * i] = t.x;
        f[2 * i + 1] = t.y;
    }
}
__device__ __forceinline__ uint4 pack8(const float* f) {
    uint4 q;
    __half2* h = reinterpret_cast<__half2*>(&q);
#pragma unroll
    for (int i = 0; i < 4; i++) h[i] = __floats2half2_rn(f[2 * i], f[2 * i + 1]);
    return q;
}

// ---------------------------------------------------------------------------------------------------
// Spinor: 24 reals, index 2*(3*spin + colour) + (0 = re, 1 = im)
// ---------------------------------------------------------------------------------------------------
// Raw form: for BQ_HALF the 24 fp16 mantissas come back un-scaled and the site norm in `n` (the hop kernel folds n
// into the per-direction weight of its accumulation FMAs, saving 24 multiplies per gather); n = 1 otherwise.
template <int PREC, bool STREAM = false>
__device__ __forceinline__ void load_spinor_raw(const void* base, int Vh, int h, typename Prec<PREC>::comp* v,
                                                typename Prec<PREC>::comp& n) {
    using A = SpinorAddr<PREC>;
    const char* b = static_cast<const char*>(base);
    n = 1;
    if constexpr (PREC == BQ_FP64) {
#pragma unroll
        for (int k = 0; k < 12; k++) {
            double2 d = ld16<STREAM, double2>(b + A::word(Vh, h, k));
            v[2 * k] = d.x;
            v[2 * k + 1] = d.y;
        }
    } else if constexpr (PREC == BQ_FP32) {
#pragma unroll
        for (int k = 0; k < 6; k++) {
            float4 d = ld16<STREAM, float4>(b + A::word(Vh, h, k));
            v[4 * k] = d.x; v[4 * k + 1] = d.y; v[4 * k + 2] = d.z; v[4 * k + 3] = d.w;
        }
    } else {
        uint4 q[3];
#pragma unroll
        for (int k = 0; k < 3; k++) q[k] = ld16<STREAM, uint4>(b + A::word(Vh, h, k));
        n = ld16<STREAM, float>(b + A::tail(Vh, h));
#pragma unroll
        for (int k = 0; k < 3; k++) unpack8(q[k], v + 8 * k);
    }
}

template <int PREC, bool STREAM = false>
__device__ __forceinline__ void load_spinor(const void* base, int Vh, int h, typename Prec<PREC>::comp* v) {
    typename Prec<PREC>::comp n;
    load_spinor_raw<PREC, STREAM>(base, Vh, h, v, n);
    if constexpr (PREC == BQ_HALF) {
        // __fmul_rn: a product of its own, never contracted into an FMA with whatever the caller adds to it — so that every
        // kernel that loads this site sees the same 24 values bit for bit, whatever ptxas fuses around the load
#pragma unroll
        for (int i = 0; i < 24; i++) v[i] = __fmul_rn(v[i], n);
    }
}

// Upper (W = 0: spins 0,1) or lower (W = 1: spins 2,3) half of a spinor, 12 reals — all the t-direction
// projectors (1 -+ gamma_4) need.
template <int PREC, int W>
__device__ __forceinline__ void load_spinor_half_raw(const void* base, int Vh, int h, typename Prec<PREC>::comp* v,
                                                     typename Prec<PREC>::comp& n) {
    using A = SpinorAddr<PREC>;
    const char* b = static_cast<const char*>(base);
    n = 1;
    if constexpr (PREC == BQ_FP64) {
#pragma unroll
        for (int k = 0; k < 6; k++) {
            double2 d = ld16<false, double2>(b + A::word(Vh, h, 6 * W + k));
            v[2 * k] = d.x;
            v[2 * k + 1] = d.y;
        }
    } else if constexpr (PREC == BQ_FP32) {
#pragma unroll
        for (int k = 0; k < 3; k++) {
            float4 d = ld16<false, float4>(b + A::word(Vh, h, 3 * W + k));
            v[4 * k] = d.x; v[4 * k + 1] = d.y; v[4 * k + 2] = d.z; v[4 * k + 3] = d.w;
        }
    } else {
        // reals 0..11 = plane 0 + low 8 bytes of plane 1; reals 12..23 = high 8 bytes of plane 1 + plane 2
        uint4 q = ld16<false, uint4>(b + A::word(Vh, h, W ? 2 : 0));
        uint2 d = ld16<false, uint2>(b + A::word(Vh, h, 1) + (W ? 8 : 0));
        n = ld16<false, float>(b + A::tail(Vh, h));
        if (W == 0) { unpack8(q, v); unpack4(d, v + 8); }
        else { unpack4(d, v); unpack8(q, v + 4); }
    }
}

template <int PREC, bool STREAM = false>
__device__ __forceinline__ void store_spinor(void* base, int Vh, int h, const typename Prec<PREC>::comp* v) {
    using A = SpinorAddr<PREC>;
    char* b = static_cast<char*>(base);
    if constexpr (PREC == BQ_FP64) {
#pragma unroll
        for (int k = 0; k < 12; k++) {
            double2 d = make_double2(v[2 * k], v[2 * k + 1]);
            double2* p = reinterpret_cast<double2*>(b + A::word(Vh, h, k));
            if (STREAM) __stcs(p, d); else *p = d;
        }
    } else if constexpr (PREC == BQ_FP32) {
#pragma unroll
        for (int k = 0; k < 6; k++) {
            float4 d = make_float4(v[4 * k], v[4 * k + 1], v[4 * k + 2], v[4 * k + 3]);
            float4* p = reinterpret_cast<float4*>(b + A::word(Vh, h, k));
            if (STREAM) __stcs(p, d); else *p = d;
        }
    } else {
        // reading S11: n = max_i |v_i| (fp32); mantissas fp16(v_i / n); zero site -> n = 0, mantissas 0
        float n = 0.f;
#pragma unroll
        for (int i = 0; i < 24; i++) n = fmaxf(n, fabsf(v[i]));
        float inv = n > 0.f ? 1.0f / n : 0.f;
        float m[24];
#pragma unroll
        for (int i = 0; i < 24; i++) m[i] = v[i] * inv;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            uint4* p = reinterpret_cast<uint4*>(b + A::word(Vh, h, k));
            uint4 q = pack8(m + 8 * k);
            if (STREAM) __stcs(p, q); else *p = q;
        }
        float* pn = reinterpret_cast<float*>(b + A::tail(Vh, h));
        if (STREAM) __stcs(pn, n); else *pn = n;
    }
}

// ---------------------------------------------------------------------------------------------------
// Link: u[2*(3*row + col) + reim], 18 reals; RECON12 stores rows 0,1 and rebuilds row 2 = conj(row0 x row1).
// `base` points at the (parity, mu) block of the gauge store.
// ---------------------------------------------------------------------------------------------------
__host__ __device__ constexpr size_t link_block_bytes(int prec, int recon, int Vh) {
    return (size_t)link_reals(recon) * prec_real_bytes(prec) * (size_t)Vh;
}

template <typename C> __device__ __forceinline__ void reconstruct_row2(C* u) {
    // row2_j = conj(row0_a row1_b - row0_b row1_a), (a, b) = (j+1, j+2) mod 3; FMA chains: 8 instructions per entry
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const int a = (j + 1) % 3, b = (j + 2) % 3;
        const C ar = u[2 * a], ai = u[2 * a + 1], br = u[2 * b], bi = u[2 * b + 1];                    // row 0
        const C cr = u[6 + 2 * a], ci = u[6 + 2 * a + 1], dr = u[6 + 2 * b], di = u[6 + 2 * b + 1];    // row 1
        C re = ar * dr;
        re = mad(-ai, di, re);
        re = mad(-br, cr, re);
        re = mad(bi, ci, re);
        C im = br * ci;            // -Im(row0_a row1_b - row0_b row1_a)
        im = mad(bi, cr, im);
        im = mad(-ar, di, im);
        im = mad(-ai, dr, im);
        u[12 + 2 * j] = re;
        u[12 + 2 * j + 1] = im;
    }
}

template <int PREC, int RECON, bool STREAM = true>
__device__ __forceinline__ void load_link(const void* base, int Vh, int idx, typename Prec<PREC>::comp* u) {
    using A = LinkAddr<PREC, RECON>;
    const char* b = static_cast<const char*>(base);
    constexpr int NR = (RECON == BQ_RECON12) ? 12 : 18;
    if constexpr (PREC == BQ_FP64) {
#pragma unroll
        for (int k = 0; k < NR / 2; k++) {
            double2 d = ld16<STREAM, double2>(b + A::word(Vh, idx, k));
            u[2 * k] = d.x;
            u[2 * k + 1] = d.y;
        }
    } else if constexpr (PREC == BQ_FP32) {
#pragma unroll
        for (int k = 0; k < NR / 4; k++) {
            float4 d = ld16<STREAM, float4>(b + A::word(Vh, idx, k));
            u[4 * k] = d.x; u[4 * k + 1] = d.y; u[4 * k + 2] = d.z; u[4 * k + 3] = d.w;
        }
        if constexpr (NR == 18) {
            float2 d = ld16<STREAM, float2>(b + A::tail(Vh, idx));
            u[16] = d.x; u[17] = d.y;
        }
    } else {
        if constexpr (NR == 18) {
            uint4 q0 = ld16<STREAM, uint4>(b + A::word(Vh, idx, 0));
            uint4 q1 = ld16<STREAM, uint4>(b + A::word(Vh, idx, 1));
            unsigned int r = ld16<STREAM, unsigned int>(b + A::tail(Vh, idx));
            unpack8(q0, u); unpack8(q1, u + 8);
            float2 t = __half22float2(*reinterpret_cast<const __half2*>(&r));
            u[16] = t.x; u[17] = t.y;
        } else {
            uint4 q0 = ld16<STREAM, uint4>(b + A::word(Vh, idx, 0));
            uint2 d = ld16<STREAM, uint2>(b + A::tail(Vh, idx));
            unpack8(q0, u); unpack4(d, u + 8);
        }
    }
    if constexpr (NR == 12) reconstruct_row2(u);
}

// Write link idx of a (parity, mu) block from 18 fp64 reals (rows 0,1 only for RECON12), rounding to nearest even;
// links have entries in [-1, 1], so fp16 needs no norm.
template <int PREC, int RECON>
__device__ __forceinline__ void store_link(void* base, int Vh, int idx, const double* u) {
    using A = LinkAddr<PREC, RECON>;
    char* b = static_cast<char*>(base);
    constexpr int NR = (RECON == BQ_RECON12) ? 12 : 18;
    if constexpr (PREC == BQ_FP64) {
#pragma unroll
        for (int k = 0; k < NR / 2; k++) *reinterpret_cast<double2*>(b + A::word(Vh, idx, k)) = make_double2(u[2 * k], u[2 * k + 1]);
    } else if constexpr (PREC == BQ_FP32) {
#pragma unroll
        for (int k = 0; k < NR / 4; k++)
            *reinterpret_cast<float4*>(b + A::word(Vh, idx, k)) =
                make_float4((float)u[4 * k], (float)u[4 * k + 1], (float)u[4 * k + 2], (float)u[4 * k + 3]);
        if constexpr (NR == 18) *reinterpret_cast<float2*>(b + A::tail(Vh, idx)) = make_float2((float)u[16], (float)u[17]);
    } else {
        float f[18];
#pragma unroll
        for (int i = 0; i < 18; i++) f[i] = (float)u[i];
        *reinterpret_cast<uint4*>(b + A::word(Vh, idx, 0)) = pack8(f);
        if constexpr (NR == 18) {
            *reinterpret_cast<uint4*>(b + A::word(Vh, idx, 1)) = pack8(f + 8);
            *reinterpret_cast<__half2*>(b + A::tail(Vh, idx)) = __floats2half2_rn(f[16], f[17]);
        } else {
            uint2 d;
            __half2* hh = reinterpret_cast<__half2*>(&d);
            hh[0] = __floats2half2_rn(f[8], f[9]);
            hh[1] = __floats2half2_rn(f[10], f[11]);
            *reinterpret_cast<uint2*>(b + A::tail(Vh, idx)) = d;
        }
    }
}
