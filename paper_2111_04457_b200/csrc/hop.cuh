// hop.cuh — per-site arithmetic of the hopping term of Eq. 1:
//   (H in)(x) = sum_mu [ (1 - g_mu) U_mu(x) in(x+mu) + (1 + g_mu) U_mu(x-mu)^dag in(x-mu) ]
// with the spin projection fused into the gather (Euclidean Dirac basis A.1).
// Writing psi = (u; l), u = spins 0,1 and l = spins 2,3 (each 2 spins x 3 colours):
//   (1 - g_k) psi = (h; -i s_k h),  h = u + i s_k l          k = x,y,z   (s_k = Pauli matrices)
//   (1 + g_k) psi = (h; +i s_k h),  h = u - i s_k l
//   (1 - g_t) psi = (0; 2 l),       (1 + g_t) psi = (2 u; 0)
// so only the 2-spin h is multiplied by the link: 8 x (12 + 132) + 168 = 1320 flop per site.
// Index convention of every register array: [2*(3*spin + colour) + reim].
#pragma once

#include "layout.cuh"

// i*s_k applied to a two-spin object (a0, a1) (3 colours each), added with a scalar weight w into (r0, r1):
//   i s_x (a0,a1) = ( i a1,  i a0);   i s_y (a0,a1) = ( a1, -a0);   i s_z (a0,a1) = ( i a0, -i a1)
// r += w * (i s_k a).   a, r: 12 reals [2*(3*s + c) + reim].  Each line is one FMA (the sign rides on the operand).
template <int K, typename C> __device__ __forceinline__ void add_isigma(C* r, const C* a, const C w) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const C a0r = a[2 * c], a0i = a[2 * c + 1], a1r = a[6 + 2 * c], a1i = a[6 + 2 * c + 1];
        if (K == 0) {         // ( i a1, i a0 ):  i*(x+iy) = -y + ix
            r[2 * c] += w * (-a1i);      r[2 * c + 1] += w * a1r;
            r[6 + 2 * c] += w * (-a0i);  r[6 + 2 * c + 1] += w * a0r;
        } else if (K == 1) {  // ( a1, -a0 )
            r[2 * c] += w * a1r;         r[2 * c + 1] += w * a1i;
            r[6 + 2 * c] += w * (-a0r);  r[6 + 2 * c + 1] += w * (-a0i);
        } else {              // ( i a0, -i a1 )
            r[2 * c] += w * (-a0i);      r[2 * c + 1] += w * a0r;
            r[6 + 2 * c] += w * a1i;     r[6 + 2 * c + 1] += w * (-a1r);
        }
    }
}

// chi = U h  (FWD) or U^dagger h (backward) for both spins of the half spinor.  66 flop per spin.
// Written as explicit FMA chains (1 FMUL + 5 FFMA per real output): `re += ur*hr - ui*hi` costs three
// instructions per term (FMUL, FFMA, FADD) because C forbids the reassociation.
template <bool DAG, typename C> __device__ __forceinline__ void su3_mul(const C* u, const C* h, C* chi) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            C re, im;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const C ur = DAG ? u[2 * (3 * b + a)] : u[2 * (3 * a + b)];
                const C ui = DAG ? -u[2 * (3 * b + a) + 1] : u[2 * (3 * a + b) + 1];
                const C hr = h[6 * s + 2 * b], hi = h[6 * s + 2 * b + 1];
                if (b == 0) {
                    re = ur * hr;
                    im = ur * hi;
                } else {
                    re = mad(ur, hr, re);
                    im = mad(ur, hi, im);
                }
                re = mad(-ui, hi, re);
                im = mad(ui, hr, im);
            }
            chi[6 * s + 2 * a] = re;
            chi[6 * s + 2 * a + 1] = im;
        }
}

template <typename C> __device__ __forceinline__ void phase_mul(C* chi, C pr, C pi) {
#pragma unroll
    for (int k = 0; k < 6; k++) {
        const C r = chi[2 * k], i = chi[2 * k + 1];
        chi[2 * k] = mad(-pi, i, pr * r);
        chi[2 * k + 1] = mad(pi, r, pr * i);
    }
}

// half storage: defined below (split load / compute, mixed-precision arithmetic)
struct HalfRaw;
template <int RECON, int MU, bool FWD, bool LSTREAM, bool DAG>
__device__ __forceinline__ void hop_load_half(HalfRaw& r, const void* in, int Vh, int nh, const void* ublock, int uidx);
template <int RECON, int MU, bool FWD, bool CPLX, bool DAG>
__device__ __forceinline__ void hop_compute_half(float* acc, const HalfRaw& r, float pr, float pi);
template <int PREC, int RECON, int MU, bool FWD, bool CPLX, bool LSTREAM, bool DAG>
__device__ __forceinline__ void hop_dir_half(float* acc, const void* in, int Vh, int nh, const void* ublock, int uidx, float pr, float pi);

// One of the 8 hops.  MU = 0..3, FWD = true: (1 - g_mu) U_mu(x) in(x+mu); false: (1 + g_mu) U_mu(x-mu)^dag in(x-mu).
//   in     : input spinor field (parity 1-p), nh = half index of the neighbour
//   ublock : (parity, MU) block of the gauge store; uidx = h (forward: the link lives on x) or nh (backward: on x-mu)
//   (pr, pi): weight of this hop = epilogue scale x boundary factor — phi_mu (forward) / conj(phi_mu) (backward) if
//   the hop wraps, else 1.
//   CPLX = false: every phase is real (+-1): pi is ignored and pr rides on the accumulation FMAs (no branch, no
//   extra instruction).  CPLX = true: general phases, one branch-free complex multiply of the half spinor.
//   Half storage: the neighbour's site norm is folded into the same weight (chi is linear in the spinor), so the
//   mantissas are never rescaled on their own.
//   LSTREAM: links read with the streaming (evict-first) policy — right when each link is used once (one right-hand
//   side); the multi-rhs kernel reads them with the default policy so that the other right-hand sides hit in L1/L2.
//   DAG: the hop of D^dagger = g5 D g5 (PAPER.md:44 set_mode).  In this basis g5 = -[[0,1],[1,0]]
//   exchanges the upper and lower spin pairs (the two signs cancel), so the dagger hop is the same arithmetic on the
//   gathered spinor with its halves exchanged (here) and on the accumulator with its halves exchanged (hop_site):
//   register renaming only, no extra instruction.  Links and boundary phases are those of D (the adjoint of the
//   forward hop from x+mu is the backward hop seen from there, with the conjugate phase — which is what D's backward
//   hop carries already).
template <int PREC, int RECON, int MU, bool FWD, bool CPLX, bool LSTREAM = true, bool DAG = false>
__device__ __forceinline__ void hop_dir(typename Prec<PREC>::comp* acc, const void* in, int Vh, int nh, const void* ublock,
                                        int uidx, typename Prec<PREC>::comp pr, typename Prec<PREC>::comp pi) {
    using C = typename Prec<PREC>::comp;
    if constexpr (PREC == BQ_HALF) {     // one implementation of the half-storage arithmetic for all kernels
        hop_dir_half<PREC, RECON, MU, FWD, CPLX, LSTREAM, DAG>(acc, in, Vh, nh, ublock, uidx, pr, pi);
        return;
    }
    C h[12], u[18], chi[12], n;
    if (MU < 3) {
        C psi[24];
        load_spinor_raw<PREC>(in, Vh, nh, psi, n);
        const C* up = DAG ? psi + 12 : psi;
        const C* lo = DAG ? psi : psi + 12;
#pragma unroll
        for (int i = 0; i < 12; i++) h[i] = up[i];            // u
        add_isigma<MU>(h, lo, C(FWD ? 1 : -1));               // h = u +- i s_k l
    } else {
        // (1 - g_t) psi = (0; 2l): forward needs l only; (1 + g_t) psi = (2u; 0): backward needs u only
        load_spinor_half_raw<PREC, (FWD != DAG) ? 1 : 0>(in, Vh, nh, h, n);
    }
    load_link<PREC, RECON, LSTREAM>(ublock, Vh, uidx, u);
    su3_mul<!FWD>(u, h, chi);
    C w = pr;
    if (CPLX) {
        phase_mul(chi, pr, pi);
        w = C(1);
    }
    if (PREC == BQ_HALF) w *= n;
    if (MU < 3) {
#pragma unroll
        for (int i = 0; i < 12; i++) acc[i] = mad(w, chi[i], acc[i]);   // upper two spins: h
        add_isigma<MU>(acc + 12, chi, FWD ? -w : w);                    // lower two spins: -+ i s_k h
    } else {
        const C w2 = 2 * w;
#pragma unroll
        for (int i = 0; i < 12; i++) acc[(FWD ? 12 : 0) + i] = mad(w2, chi[i], acc[(FWD ? 12 : 0) + i]);
    }
}

// ---------------------------------------------------------------------------------------------------
// Half storage: the same hop split into its LOAD (raw 16-byte words of the neighbour spinor and of the link, kept
// packed: 13 + 9 registers) and its COMPUTE (unpack, project, multiply, accumulate), so that hop_site can issue the
// loads of direction d+1 before it computes direction d.  A half-storage direction is only 88 bytes per thread; at the
// 16 warps per SM the register budget allows, the compiler's own batching (loads of ~3 directions, then their
// arithmetic) leaves part of every batch's memory latency exposed — ncu: long-scoreboard stalls dominate, issue slots
// 60 % busy on a kernel that needs them ~85 % busy to reach the HBM roofline.  ptxas still schedules the loads its own
// way, so the source-level pipeline only nudges it: measured 84.0 -> 82.0 us (18-real), 82.0 -> 76.6 us (12-real),
// 92.1 -> 84.0 us (xpay epilogue) on 32^3x64.
// ---------------------------------------------------------------------------------------------------
// sm_100 mixed-precision scalar arithmetic (PTX fma/add .f32.f16, SASS FHFMA / FHADD): d(fp32) = a(fp16) * b(fp16) + c(fp32)
// and d = a(fp16) + c(fp32) in ONE instruction, the fp16 operands taken straight from either half of a packed 32-bit
// register (operand selectors .H0/.H1, negation folded).  The product of two fp16 numbers is exact in fp32, so
// fhfma(a, b, c) is bit for bit fma(float(a), float(b), c): the arithmetic stays fp32 (reading S11) and the
// fp16 -> fp32 conversion instructions of these operands (one HADD2.F32 per real) disappear.
#ifndef HOP_HALF_MIXED
#define HOP_HALF_MIXED 1   // A/B switch
#endif
// low (H = 0: re) or high (H = 1: im) half of a packed complex number, as a 16-bit register
template <int H> __device__ __forceinline__ unsigned short half_of(unsigned int w) {
    unsigned short lo, hi;
    asm("mov.b32 {%0, %1}, %2;" : "=h"(lo), "=h"(hi) : "r"(w));
    return H ? hi : lo;
}
__device__ __forceinline__ float fhfma(unsigned short a, unsigned short b, float c) {          // a*b + c
    float d;
    asm("fma.rn.f32.f16 %0, %1, %2, %3;" : "=f"(d) : "h"(a), "h"(b), "f"(c));
    return d;
}
__device__ __forceinline__ float fhfma_neg(unsigned short a, unsigned short b, float c) {      // -a*b + c
    float d;
    asm("{ .reg .b16 t; neg.f16 t, %1; fma.rn.f32.f16 %0, t, %2, %3; }" : "=f"(d) : "h"(a), "h"(b), "f"(c));
    return d;
}
__device__ __forceinline__ float fhmul(unsigned short a, unsigned short b) {                   // a*b (exact product, as fmul)
    float d;
    asm("fma.rn.f32.f16 %0, %1, %2, 0f80000000;" : "=f"(d) : "h"(a), "h"(b));                  // + (-0): keeps the sign of a zero product
    return d;
}
__device__ __forceinline__ float fhadd(unsigned short a, float c) {                            // c + a
    float d;
    asm("add.rn.f32.f16 %0, %1, %2;" : "=f"(d) : "h"(a), "f"(c));
    return d;
}
__device__ __forceinline__ float fhsub(unsigned short a, float c) {                            // c - a
    float d;
    asm("{ .reg .b16 t; neg.f16 t, %1; add.rn.f32.f16 %0, t, %2; }" : "=f"(d) : "h"(a), "f"(c));
    return d;
}

// r += sgn * (i s_k a) with a given as 6 packed fp16 complex numbers (a[3*spin + colour]) and sgn = +-1: the projection
// h = u +- i s_k l of hop_dir with the conversion of l folded into the add (same table as add_isigma).
template <int K, bool PLUS> __device__ __forceinline__ void add_isigma_h16(float* r, const unsigned int* a) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const unsigned short a0r = half_of<0>(a[c]), a0i = half_of<1>(a[c]), a1r = half_of<0>(a[3 + c]), a1i = half_of<1>(a[3 + c]);
        // P(x): r += sgn * x ;  M(x): r += sgn * (-x)
#define BQ_P(dst, x) dst = PLUS ? fhadd(x, dst) : fhsub(x, dst)
#define BQ_M(dst, x) dst = PLUS ? fhsub(x, dst) : fhadd(x, dst)
        if (K == 0) {         // ( i a1, i a0 )
            BQ_M(r[2 * c], a1i);      BQ_P(r[2 * c + 1], a1r);
            BQ_M(r[6 + 2 * c], a0i);  BQ_P(r[6 + 2 * c + 1], a0r);
        } else if (K == 1) {  // ( a1, -a0 )
            BQ_P(r[2 * c], a1r);      BQ_P(r[2 * c + 1], a1i);
            BQ_M(r[6 + 2 * c], a0r);  BQ_M(r[6 + 2 * c + 1], a0i);
        } else {              // ( i a0, -i a1 )
            BQ_M(r[2 * c], a0i);      BQ_P(r[2 * c + 1], a0r);
            BQ_P(r[6 + 2 * c], a1i);  BQ_M(r[6 + 2 * c + 1], a1r);
        }
#undef BQ_P
#undef BQ_M
    }
}

// chi = U h (DAG: U^dagger h) with BOTH operands packed fp16: link entries u[3*row + col], half spinor h[3*spin + colour].
// Same FMA chains, in the same order, as su3_mul.
template <bool DAG> __device__ __forceinline__ void su3_mul_h16(const unsigned int* u, const unsigned int* h, float* chi) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            float re, im;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const unsigned int uw = DAG ? u[3 * b + a] : u[3 * a + b];
                const unsigned short ur = half_of<0>(uw), ui = half_of<1>(uw);
                const unsigned short hr = half_of<0>(h[3 * s + b]), hi = half_of<1>(h[3 * s + b]);
                if (b == 0) {
                    re = fhmul(ur, hr);
                    im = fhmul(ur, hi);
                } else {
                    re = fhfma(ur, hr, re);
                    im = fhfma(ur, hi, im);
                }
                // su3_mul: re = mad(-ui', hi, re); im = mad(ui', hr, im) with ui' = DAG ? -ui : ui
                if (DAG) {
                    re = fhfma(ui, hi, re);
                    im = fhfma_neg(ui, hr, im);
                } else {
                    re = fhfma_neg(ui, hi, re);
                    im = fhfma(ui, hr, im);
                }
            }
            chi[6 * s + 2 * a] = re;
            chi[6 * s + 2 * a + 1] = im;
        }
}

struct HalfRaw {
    uint4 s0, s1, s2;      // spinor mantissas (t direction: s0 = the full word, s1.x/.y = the half word)
    float n;               // site norm
    uint4 l0, l1;          // link words (12-real: l1.x/.y = the trailing 8 bytes)
    unsigned int lt;       // 18-real: trailing half2
};

template <int RECON, int MU, bool FWD, bool LSTREAM, bool DAG>
__device__ __forceinline__ void hop_load_half(HalfRaw& r, const void* in, int Vh, int nh, const void* ublock, int uidx) {
    using A = SpinorAddr<BQ_HALF>;
    using LA = LinkAddr<BQ_HALF, RECON>;
    const char* b = static_cast<const char*>(in);
    if (MU < 3) {
        r.s0 = ld16<false, uint4>(b + A::word(Vh, nh, 0));
        r.s1 = ld16<false, uint4>(b + A::word(Vh, nh, 1));
        r.s2 = ld16<false, uint4>(b + A::word(Vh, nh, 2));
    } else {
        constexpr int W = (FWD != DAG) ? 1 : 0;   // (1 - g_t) needs the lower spin pair, (1 + g_t) the upper one
        r.s0 = ld16<false, uint4>(b + A::word(Vh, nh, W ? 2 : 0));
        const uint2 d = ld16<false, uint2>(b + A::word(Vh, nh, 1) + (W ? 8 : 0));
        r.s1.x = d.x; r.s1.y = d.y;
    }
    r.n = ld16<false, float>(b + A::tail(Vh, nh));
    const char* ub = static_cast<const char*>(ublock);
    r.l0 = ld16<LSTREAM, uint4>(ub + LA::word(Vh, uidx, 0));
    if (RECON == BQ_RECON18) {
        r.l1 = ld16<LSTREAM, uint4>(ub + LA::word(Vh, uidx, 1));
        r.lt = ld16<LSTREAM, unsigned int>(ub + LA::tail(Vh, uidx));
    } else {
        const uint2 d = ld16<LSTREAM, uint2>(ub + LA::tail(Vh, uidx));
        r.l1.x = d.x; r.l1.y = d.y;
    }
}

template <int RECON, int MU, bool FWD, bool CPLX, bool DAG>
__device__ __forceinline__ void hop_compute_half(float* acc, const HalfRaw& r, float pr, float pi) {
    float h[12], u[18], chi[12];
    if (HOP_HALF_MIXED && MU == 3 && RECON == BQ_RECON18) {
        // t direction: the half spinor IS the stored fp16 data and so is the link: no conversion at all
        constexpr int W = (FWD != DAG) ? 1 : 0;
        const unsigned int hw[6] = {W ? r.s1.x : r.s0.x, W ? r.s1.y : r.s0.y, W ? r.s0.x : r.s0.z, W ? r.s0.y : r.s0.w,
                                    W ? r.s0.z : r.s1.x, W ? r.s0.w : r.s1.y};
        const unsigned int uw[9] = {r.l0.x, r.l0.y, r.l0.z, r.l0.w, r.l1.x, r.l1.y, r.l1.z, r.l1.w, r.lt};
        su3_mul_h16<!FWD>(uw, hw, chi);
    } else {
        if (MU < 3) {
            if (HOP_HALF_MIXED) {
                // h = u +- i s_k l: convert u, fold the conversion of l into the adds
                const unsigned int pw[12] = {r.s0.x, r.s0.y, r.s0.z, r.s0.w, r.s1.x, r.s1.y, r.s1.z, r.s1.w, r.s2.x, r.s2.y, r.s2.z, r.s2.w};
                const unsigned int* upw = DAG ? pw + 6 : pw;
                const unsigned int* low = DAG ? pw : pw + 6;
#pragma unroll
                for (int c = 0; c < 6; c++) {
                    const float2 t = __half22float2(*reinterpret_cast<const __half2*>(&upw[c]));
                    h[2 * c] = t.x; h[2 * c + 1] = t.y;
                }
                add_isigma_h16<MU, FWD>(h, low);
            } else {
                float psi[24];
                unpack8(r.s0, psi); unpack8(r.s1, psi + 8); unpack8(r.s2, psi + 16);
                const float* up = DAG ? psi + 12 : psi;
                const float* lo = DAG ? psi : psi + 12;
#pragma unroll
                for (int i = 0; i < 12; i++) h[i] = up[i];
                add_isigma<MU>(h, lo, float(FWD ? 1 : -1));
            }
        } else {
            constexpr int W = (FWD != DAG) ? 1 : 0;
            const uint2 d = make_uint2(r.s1.x, r.s1.y);
            if (W == 0) { unpack8(r.s0, h); unpack4(d, h + 8); }
            else { unpack4(d, h); unpack8(r.s0, h + 4); }
        }
        unpack8(r.l0, u);
        if (RECON == BQ_RECON18) {
            unpack8(r.l1, u + 8);
            const float2 t = __half22float2(*reinterpret_cast<const __half2*>(&r.lt));
            u[16] = t.x; u[17] = t.y;
        } else {
            unpack4(make_uint2(r.l1.x, r.l1.y), u + 8);
            reconstruct_row2(u);
        }
        su3_mul<!FWD>(u, h, chi);
    }
    float w = pr;
    if (CPLX) {
        phase_mul(chi, pr, pi);
        w = 1.0f;
    }
    w *= r.n;
    if (MU < 3) {
#pragma unroll
        for (int i = 0; i < 12; i++) acc[i] = mad(w, chi[i], acc[i]);
        add_isigma<MU>(acc + 12, chi, FWD ? -w : w);
    } else {
        const float w2 = 2 * w;
#pragma unroll
        for (int i = 0; i < 12; i++) acc[(FWD ? 12 : 0) + i] = mad(w2, chi[i], acc[(FWD ? 12 : 0) + i]);
    }
}

template <int PREC, int RECON, int MU, bool FWD, bool CPLX, bool LSTREAM, bool DAG>
__device__ __forceinline__ void hop_dir_half(float* acc, const void* in, int Vh, int nh, const void* ublock, int uidx, float pr, float pi) {
    HalfRaw r;
    hop_load_half<RECON, MU, FWD, LSTREAM, DAG>(r, in, Vh, nh, ublock, uidx);
    hop_compute_half<RECON, MU, FWD, CPLX, DAG>(acc, r, pr, pi);
}
