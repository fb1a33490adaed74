// hop_ls.cuh — "link-stationary" multi-right-hand-side hop (the paper's workload is the 12
// spin-colour sources of a propagator on ONE gauge field; north_star: "shared-memory or TMA staging").
//
// The per-(site, rhs) kernel of hop_kernels.cuh (hop_kernel_mrhs) reads the links from HBM once per launch, but every
// (site, rhs) still gathers its 8 neighbour spinors and its 8 links through L1: 590-680 B per (site, rhs) cross the
// L2 -> SM crossbar where 144 B (fp32/18, 12 rhs) are compulsory, and the kernel sits on the L2 output bandwidth
// (profiles/r1_hop_mrhs12.md).  On-chip capacity is what limits the reuse: a spatial block large enough to share its
// gathers needs ~65 KB of input spinors per right-hand side, and all right-hand sides want the same links.  This kernel
// splits the two reuses between the two big on-chip stores of an SM:
//   * LINKS live in REGISTERS.  A CTA owns a 4-D block of 8 x BY x BZ x BT output sites (one layout tile of 8 half
//     indices in x), one thread per site; the thread loads its 8 links once (144 registers in fp32) and keeps them for
//     ALL right-hand sides: link traffic per (site, rhs) = 8 links / nrhs, no link load or reconstruction in the loop.
//   * SPINORS stream through SHARED MEMORY.  The right-hand sides are processed one after the other; for each one the
//     block's input tiles and their y/z/t halo tiles are brought in by TMA tensor copies (cp.async.bulk.tensor.5d: the
//     tiled layout makes a field a dense 5-D tensor (tile element, x-tile, y, z, t)), signalled through an mbarrier,
//     into a ring of 2-3 stages, so that the copies of right-hand side k+1, k+2 overlap the arithmetic of k.  The t
//     halos carry only the spin half the projector (1 -+ g_t) keeps (the tiled layout stores the two spin pairs in
//     separate planes).  The one x-neighbour per row that lies outside the tile comes in through cp.async (LDGSTS,
//     16 bytes per thread) completing on the same mbarrier.  All 8 gathers of a site are shared-memory reads:
//     (BY, BZ, BT) = (4, 4, 2): 88 tile loads per 32 output tiles = 264 B per (site, rhs) in fp32.
//   * The xpay operand z and the left operand w of a fused inner product come the same way (one stage each).
// Per (site, rhs) the arithmetic is hop.cuh's, direction by direction in the same order, so results are bit for bit
// those of hop_kernel / hop_kernel_mrhs.  fp32 and half storage; all four epilogues (Wilson and clover) with the fused reductions:
// for the clover ones the block's clover tiles sit in shared memory for all right-hand sides (one more TMA copy per block).
// Needs Lx % 16 == 0 (tiles are pieces of x-rows) and extents divisible by the block; anything else takes hop_kernel_mrhs.  fp64 (288
// link registers do not exist) takes the direction-split form of this kernel, hop_lsp.cuh, from 8 right-hand sides on.  Blocks are
// launched in 4 x 4 x 4 bricks (ls_block_coords) so that the CTAs in flight share their halos in L2.
#pragma once

#include <cuda.h>

#include <cstdio>
#include <cstdlib>

#include <type_traits>

#ifndef LS_BY
#define LS_BY 4
#endif
#ifndef LS_BZ
#define LS_BZ 4
#endif
#ifndef LS_BT
#define LS_BT 1
#endif

#ifndef LS_LINK_NOALLOC
#define LS_LINK_NOALLOC 1     // fp32 links of the prologue: ld.global.nc.L1::no_allocate (A/B switch; x12 hop 637.4 -> 630.4 us, x2 193.7 -> 188.5 us)
#endif
constexpr int LS_NT = LS_BY * LS_BZ * LS_BT;      // tiles (rows of 8 sites) per block
constexpr int LS_THREADS = 8 * LS_NT;             // one thread per output site
constexpr int LS_MAX_RHS = 32;                    // right-hand sides per launch (active list = one ballot)
// 255 registers per thread either way: one CTA of 256 threads per SM, or two of 128 — two CTAs overlap one's prologue (its
// 8 x 18 link loads per thread, 147 KB per 256 sites, nothing to compute yet) with the other's arithmetic
constexpr int LS_MINB = LS_THREADS <= 128 ? 2 : 1;
static_assert(LS_NT % 8 == 0 && LS_THREADS % 32 == 0 && LS_THREADS <= 1024, "block shape");
static_assert((LS_BY * LS_BZ) % 4 == 0 && (LS_BZ * LS_BT) % 4 == 0 && (LS_BY * LS_BT) % 4 == 0,
              "every halo region must be a multiple of 4 tiles (128-byte alignment of the TMA destinations in half storage)");

#ifndef LS_WIDEX
#define LS_WIDEX 0            // conflict-free placement of the x-halo sites in shared memory: A/B switch, OFF — measured slower on B200
#endif                        // (fp32 x12 hop 660 vs 631 us, x4 308 vs 279, x2 215 vs 189; profiles/r3_ls_widex_ab.txt)
// shared-memory geometry of one stage (one right-hand side): byte offsets of the regions.
// WIDEX: the x-halo site of a row sits in 16-byte slot 0 (rows that read it as their forward neighbour) or slot 7 (backward) of a
// 128-byte line of its own per (row pair, word).  The 7 other threads of the row read slots 1..7 (resp. 0..6) of the centre tile
// with the same LDS.128, so the halo slot is the one bank group they leave free; in the compact form (8 rows share a pseudo tile,
// slot = row & 7) 7 of 8 rows replay every x-direction load once (profiles/r2_hop_ls.md: 17 % of the shared wavefronts).
// Removing those replays this way did NOT pay: the stage grows by 4.5 KB and the 96 cp.async of the x halo scatter over 48 lines
// instead of 12; the kernel got 5-14 % slower, so the compact form stays the default.
template <int PREC, bool WIDEX = false> struct LsGeom {
    static constexpr int S = PREC == BQ_FP64 ? 192 : (PREC == BQ_FP32 ? 96 : 52);   // bytes per site
    static constexpr int TS = 8 * S;                                               // bytes per tile
    static constexpr bool SPLIT_T = PREC != BQ_HALF;      // spin pairs in separate planes: t halos are half tiles
    static constexpr int HT = SPLIT_T ? TS / 2 : TS;      // bytes per t-halo tile
    static constexpr int NW = S / 16;                     // 16-byte words per site
    static constexpr int C = 0;
    static constexpr int YM = C + LS_NT * TS, YP = YM + LS_BZ * LS_BT * TS;
    static constexpr int ZM = YP + LS_BZ * LS_BT * TS, ZP = ZM + LS_BY * LS_BT * TS;
    static constexpr int TM = ZP + LS_BY * LS_BT * TS, TP = TM + LS_BY * LS_BZ * HT;
    static constexpr int X = TP + LS_BY * LS_BZ * HT;     // x halo sites, 8 to a pseudo tile
    static constexpr int XBYTES = WIDEX ? (LS_NT / 2) * NW * 128 : (LS_NT / 8) * TS;
    static constexpr int STAGE = (X + XBYTES + 127) / 128 * 128;
    static constexpr int TX = X;                          // bytes a stage receives through TMA (everything but the x halo)
    static constexpr int OPER = LS_NT * TS;               // one interior-only operand buffer (z or w)
    static constexpr int CLS = 72 * (PREC == BQ_FP64 ? 8 : (PREC == BQ_FP32 ? 4 : 2));   // clover blocks: bytes per site = 3 spinor-fp-tiles' worth per 8 sites
    static constexpr int CLOV = LS_NT * 8 * CLS;          // the block's clover tiles (site-diagonal epilogues EPI 2, 3)
    static constexpr int NXC = (PREC == BQ_HALF ? 4 : NW) * LS_NT;   // cp.async copies of the x halo per stage
    static_assert(STAGE % 128 == 0 && OPER % 128 == 0, "alignment");
    static_assert(PREC == BQ_FP64 || NXC <= LS_THREADS, "one x-halo copy per thread");
};

struct LsMaps {
    alignas(64) CUtensorMap in_c, in_y, in_z, in_t;   // input field: interior box, y-halo box, z-halo box, t-halo box
    alignas(64) CUtensorMap z_c, w_c;                 // interior boxes of the xpay operand and of the inner-product operand
    alignas(64) CUtensorMap cl_c;                     // interior box of the clover store (EPI 2, 3)
};

template <typename C> struct LsParams {
    HopArgs<C> a;
    LsMaps m;
    int nxt, nyb, nzb;           // x tiles per row; blocks in y, z
    int gy, gz, gt;              // launch order of the blocks: bricks of nxt x gy x gz x gt blocks (ls_block_coords)
    int tk_in, tk_z, tk_w;       // t'-extent between consecutive right-hand sides of in / z / w (their byte strides in t slices)
    const SolverScalars* done;   // solver: per-rhs states whose `done` flag switches a right-hand side off (nullptr: all run)
};

// ---- PTX wrappers: mbarrier, TMA, cp.async ----
__device__ __forceinline__ unsigned int ls_smem_u32(const void* p) { return (unsigned int)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void ls_mbar_init(unsigned int bar, unsigned int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void ls_mbar_expect_tx(unsigned int bar, unsigned int bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void ls_mbar_arrive(unsigned int bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void ls_mbar_wait(unsigned int bar, unsigned int parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LS_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LS_DONE;\n"
        "bra LS_WAIT;\n"
        "LS_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void ls_tma5(unsigned int dst, const CUtensorMap* map, unsigned int bar, int c0, int c1, int c2, int c3, int c4) {
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
                 ::"r"(dst), "l"(reinterpret_cast<unsigned long long>(map)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
                 : "memory");
}
template <int BYTES> __device__ __forceinline__ void ls_cp_async(unsigned int dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst), "l"(src), "n"(BYTES) : "memory");
}
// arrive on `bar` once all cp.async of this thread issued so far have landed (the arrival is part of the barrier's count)
__device__ __forceinline__ void ls_cp_async_arrive(unsigned int bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}

// Launch order of the blocks.  The CTAs in flight at one time (one or two per SM) work on consecutive block indices, and what
// one block reads as halo is the interior of its neighbours: whatever two neighbours do not read within the same wave must
// survive in L2 from one wave to the next, against a working set of ~200 MB per wave (12 right-hand sides x 148-296 blocks).
// With the blocks in lexicographic order (x, y, z, t) a wave is a slab of 1-2 t slices and every t halo — the largest,
// since the blocks are one site thick in t — is re-read from HBM (fp64, 12 rhs: 5.7 GB of DRAM reads where 3.6 GB are
// compulsory).  So the index runs over compact bricks of nxt x gy x gz x gt blocks (4 x 4 x 4 where the extents divide:
// 128 blocks ~ one wave), bricks following one another in t first.
__host__ __device__ inline int ls_brick_dim(int n) { return n % 4 == 0 ? 4 : (n % 2 == 0 ? 2 : 1); }
inline void ls_brick(int nyb, int nzb, int ntb, int& gy, int& gz, int& gt) {
    gy = ls_brick_dim(nyb); gz = ls_brick_dim(nzb); gt = ls_brick_dim(ntb);
    static int cap[3] = {0, 0, 0};     // A/B switch: BQ_LS_BRICK="y,z,t" caps the brick (1,1,1 = lexicographic order)
    if (!cap[0]) {
        cap[0] = cap[1] = cap[2] = 4;
        if (const char* e = getenv("BQ_LS_BRICK")) sscanf(e, "%d,%d,%d", &cap[0], &cap[1], &cap[2]);
        for (int i = 0; i < 3; i++) if (cap[i] < 1) cap[i] = 1;
    }
    while (gy > cap[0]) gy /= 2;
    while (gz > cap[1]) gz /= 2;
    while (gt > cap[2]) gt /= 2;
}
__device__ __forceinline__ void ls_block_coords(int b, int nxt, int nyb, int nzb, int gy, int gz, int gt, int& xt, int& yb, int& zb, int& tb) {
    xt = b % nxt; b /= nxt;
    const int iy = b % gy; b /= gy;
    const int iz = b % gz; b /= gz;
    const int it = b % gt; b /= gt;
    // bricks: t fastest, then y, then z
    const int by = nyb / gy;
    // number of bricks in t is implied by the grid size: b = bt + nbt * (byi + by * bzi) with nbt = gridDim.x / (nxt * nyb * nzb * gt)
    const int nbt = (int)(gridDim.x / (unsigned)(nxt * nyb * nzb * gt));
    const int bt = b % nbt; b /= nbt;
    const int byi = b % by;
    const int bzi = b / by;
    yb = byi * gy + iy; zb = bzi * gz + iz; tb = bt * gt + it;
}

// ---- one of the 8 hops with the neighbour spinor in shared memory and the link in registers (arithmetic = hop_dir) ----
template <int PREC, int RECON> struct LsLink { typename Prec<PREC>::comp u[18]; };
template <int RECON> struct LsLink<BQ_HALF, RECON> { uint4 l0, l1; unsigned int lt; };   // packed, as HalfRaw holds them

template <int PREC, int RECON>
__device__ __forceinline__ void ls_load_link(LsLink<PREC, RECON>& L, const void* ublock, int Vh, int idx) {
    if constexpr (PREC == BQ_HALF) {
        using LA = LinkAddr<BQ_HALF, RECON>;
        const char* ub = static_cast<const char*>(ublock);
        L.l0 = ld16<true, uint4>(ub + LA::word(Vh, idx, 0));
        if (RECON == BQ_RECON18) {
            L.l1 = ld16<true, uint4>(ub + LA::word(Vh, idx, 1));
            L.lt = ld16<true, unsigned int>(ub + LA::tail(Vh, idx));
        } else {
            const uint2 d = ld16<true, uint2>(ub + LA::tail(Vh, idx));
            L.l1 = make_uint4(d.x, d.y, 0u, 0u);
            L.lt = 0u;
        }
    } else if constexpr (PREC == BQ_FP32 && LS_LINK_NOALLOC) {
        // read-only streaming loads that do not allocate in L1 (ld.global.nc.L1::no_allocate): same values as load_link
        using A = LinkAddr<PREC, RECON>;
        const char* bp = static_cast<const char*>(ublock);
        constexpr int NR = (RECON == BQ_RECON12) ? 12 : 18;
#pragma unroll
        for (int k = 0; k < NR / 4; k++) {
            float4 d;
            asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(d.x), "=f"(d.y), "=f"(d.z), "=f"(d.w) : "l"(bp + A::word(Vh, idx, k)));
            L.u[4 * k] = d.x; L.u[4 * k + 1] = d.y; L.u[4 * k + 2] = d.z; L.u[4 * k + 3] = d.w;
        }
        if constexpr (NR == 18) {
            float2 d;
            asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(d.x), "=f"(d.y) : "l"(bp + A::tail(Vh, idx)));
            L.u[16] = d.x; L.u[17] = d.y;
        }
        if constexpr (NR == 12) reconstruct_row2(L.u);
    } else {
        load_link<PREC, RECON, true>(ublock, Vh, idx, L.u);    // 12-real: row 2 rebuilt here, once for all right-hand sides
    }
}

// sp: address of word 0 of the neighbour site in its (possibly half) tile; np (half storage): address of its norm
template <int PREC, int RECON, int MU, bool FWD, bool CPLX, bool DAG>
__device__ __forceinline__ void ls_dir(typename Prec<PREC>::comp* acc, const char* sp, const char* np, const LsLink<PREC, RECON>& L,
                                       typename Prec<PREC>::comp pr, typename Prec<PREC>::comp pi) {
    using C = typename Prec<PREC>::comp;
    if constexpr (PREC == BQ_HALF) {
        HalfRaw r;
        if (MU < 3) {
            r.s0 = *reinterpret_cast<const uint4*>(sp);
            r.s1 = *reinterpret_cast<const uint4*>(sp + 128);
            r.s2 = *reinterpret_cast<const uint4*>(sp + 256);
        } else {
            constexpr int W = (FWD != DAG) ? 1 : 0;
            r.s0 = *reinterpret_cast<const uint4*>(sp + (W ? 256 : 0));
            const uint2 d = *reinterpret_cast<const uint2*>(sp + 128 + (W ? 8 : 0));
            r.s1.x = d.x; r.s1.y = d.y;
        }
        r.n = *reinterpret_cast<const float*>(np);
        r.l0 = L.l0; r.l1 = L.l1; r.lt = L.lt;
        hop_compute_half<RECON, MU, FWD, CPLX, DAG>(acc, r, pr, pi);
    } else {
        using V = typename std::conditional<PREC == BQ_FP64, double2, float4>::type;
        constexpr int W = 16 / sizeof(C), NWS = 24 / W;      // reals per word, words per site
        C h[12], chi[12];
        if (MU < 3) {
            C psi[24];
#pragma unroll
            for (int k = 0; k < NWS; k++) {
                const V d = *reinterpret_cast<const V*>(sp + k * 128);
                if constexpr (PREC == BQ_FP64) { psi[2 * k] = d.x; psi[2 * k + 1] = d.y; }
                else { psi[4 * k] = d.x; psi[4 * k + 1] = d.y; psi[4 * k + 2] = d.z; psi[4 * k + 3] = d.w; }
            }
            const C* up = DAG ? psi + 12 : psi;
            const C* lo = DAG ? psi : psi + 12;
#pragma unroll
            for (int i = 0; i < 12; i++) h[i] = up[i];
            add_isigma<MU>(h, lo, C(FWD ? 1 : -1));
        } else {
            // sp points at the spin half the projector keeps (forward: lower pair, backward: upper pair; exchanged for DAG)
#pragma unroll
            for (int k = 0; k < NWS / 2; k++) {
                const V d = *reinterpret_cast<const V*>(sp + k * 128);
                if constexpr (PREC == BQ_FP64) { h[2 * k] = d.x; h[2 * k + 1] = d.y; }
                else { h[4 * k] = d.x; h[4 * k + 1] = d.y; h[4 * k + 2] = d.z; h[4 * k + 3] = d.w; }
            }
        }
        su3_mul<!FWD>(L.u, h, chi);
        C w = pr;
        if (CPLX) {
            phase_mul(chi, pr, pi);
            w = C(1);
        }
        if (MU < 3) {
#pragma unroll
            for (int i = 0; i < 12; i++) acc[i] = mad(w, chi[i], acc[i]);
            add_isigma<MU>(acc + 12, chi, FWD ? -w : w);
        } else {
            const C w2 = 2 * w;
#pragma unroll
            for (int i = 0; i < 12; i++) acc[(FWD ? 12 : 0) + i] = mad(w2, chi[i], acc[(FWD ? 12 : 0) + i]);
        }
    }
}

// a whole site from an interior-only operand buffer in shared memory (same values as load_spinor from global memory)
template <int PREC> __device__ __forceinline__ void ls_load_site(const char* tile, int pos, typename Prec<PREC>::comp* v) {
    if constexpr (PREC == BQ_HALF) {
#pragma unroll
        for (int k = 0; k < 3; k++) unpack8(*reinterpret_cast<const uint4*>(tile + k * 128 + pos * 16), v + 8 * k);
        const float n = *reinterpret_cast<const float*>(tile + 384 + pos * 4);
#pragma unroll
        for (int i = 0; i < 24; i++) v[i] = __fmul_rn(v[i], n);      // as load_spinor: never contracted
    } else if constexpr (PREC == BQ_FP32) {
#pragma unroll
        for (int k = 0; k < 6; k++) {
            const float4 d = *reinterpret_cast<const float4*>(tile + k * 128 + pos * 16);
            v[4 * k] = d.x; v[4 * k + 1] = d.y; v[4 * k + 2] = d.z; v[4 * k + 3] = d.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < 12; k++) {
            const double2 d = *reinterpret_cast<const double2*>(tile + k * 128 + pos * 16);
            v[2 * k] = d.x; v[2 * k + 1] = d.y;
        }
    }
}

// wide x-halo placement: fp32, Wilson epilogues (with the clover tiles resident the 9 KB it costs would end two CTAs per SM)
template <int PREC, int EPI> __host__ __device__ constexpr bool ls_widex() { return LS_WIDEX && PREC == BQ_FP32 && EPI < 2 && LS_NT % 2 == 0 && LS_BY % 2 == 0; }
template <int EPI, int RED> __host__ __device__ constexpr int ls_stages() { return (EPI == 0 && LS_MINB == 1) ? 3 : 2; }
template <int PREC, int EPI, int RED> __host__ __device__ constexpr size_t ls_smem_bytes() {
    return (size_t)ls_stages<EPI, RED>() * LsGeom<PREC, ls_widex<PREC, EPI>()>::STAGE + (EPI == 1 ? LsGeom<PREC>::OPER : 0) + (EPI == 1 && RED == 1 ? LsGeom<PREC>::OPER : 0) +
           (EPI >= 2 ? LsGeom<PREC>::CLOV : 0) + 256 /* mbarriers, active list */ + (RED ? 2 * 3 * (LS_THREADS / 32) * sizeof(double) : 0);
}

template <int PREC, int RECON, int EPI, bool CPLX, int RED, bool DAG>
__global__ void __launch_bounds__(LS_THREADS, LS_MINB) hop_ls_kernel(const __grid_constant__ LsParams<typename Prec<PREC>::comp> P) {
    using C = typename Prec<PREC>::comp;
    constexpr bool WX = ls_widex<PREC, EPI>();
    using G = LsGeom<PREC, WX>;
    constexpr int NS = ls_stages<EPI, RED>();
    constexpr int NRED = RED == 1 ? 2 : 3;
    extern __shared__ __align__(128) unsigned char ls_smem[];
    unsigned char* const stage0 = ls_smem;
    unsigned char* const zbuf = ls_smem + NS * G::STAGE;
    unsigned char* const wbuf = zbuf + (EPI == 1 ? G::OPER : 0);
    unsigned char* const cbuf = wbuf + (EPI == 1 && RED == 1 ? G::OPER : 0);         // clover tiles of the block (EPI 2, 3)
    unsigned char* const ctl = cbuf + (EPI >= 2 ? G::CLOV : 0);
    unsigned long long* const bars = reinterpret_cast<unsigned long long*>(ctl);     // full[NS], fullz, clover
    int* const act = reinterpret_cast<int*>(ctl + 64);                              // [0] = count, [1] = mask, [2..] = list of active rhs
    double* const s_red = reinterpret_cast<double*>(ctl + 256);                     // [2][NRED][warps]
    const HopArgs<C>& a = P.a;

    const int tid = threadIdx.x, s8 = tid & 7, tl = tid >> 3;
    const int ty = tl % LS_BY, tz = (tl / LS_BY) % LS_BZ, tt = tl / (LS_BY * LS_BZ);
    int xt, yb, zb, tb;
    ls_block_coords(blockIdx.x, P.nxt, P.nyb, P.nzb, P.gy, P.gz, P.gt, xt, yb, zb, tb);
    const int y0 = yb * LS_BY, z0 = zb * LS_BZ, t0 = tb * LS_BT;
    const int xh = 8 * xt + s8, y = y0 + ty, z = z0 + tz, t = t0 + tt;
    const int Vh = a.Vh;
    const int sy = a.Lxh, sz = a.Lxh * a.Ly, st = sz * a.Lz;
    const int h = xh + sy * y + sz * z + st * t;
    const int r = (y + z + t + a.p) & 1;

    // ---- barriers and the list of active right-hand sides ----
    if (tid < 32) {
        unsigned int mask;
        if (P.done) {
            const bool on = tid < a.nrhs && P.done[tid].done == 0;
            mask = __ballot_sync(0xffffffffu, on);
        } else {
            mask = a.nrhs >= 32 ? 0xffffffffu : ((1u << a.nrhs) - 1u);
        }
        if (mask & (1u << tid)) act[2 + __popc(mask & ((1u << tid) - 1u))] = tid;    // act[2 + i] = i-th active right-hand side
        if (tid == 0) {
            act[0] = __popc(mask);
            act[1] = (int)mask;
            for (int s = 0; s < NS; s++) ls_mbar_init(ls_smem_u32(bars + s), 1 + LS_THREADS);
            ls_mbar_init(ls_smem_u32(bars + NS), 1);
            ls_mbar_init(ls_smem_u32(bars + NS + 1), 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    __syncthreads();
    const int nact = act[0];
    if (nact == 0) return;
    auto rhs_of = [&](int i) { return act[2 + i]; };

    // ---- this thread's x-halo copy (cp.async): row jr of the block, 16-byte word jk (half storage: jk == 3 is the norm) ----
    const bool xcopy = tid < G::NXC;
    unsigned int xsrc = 0, xdst = 0;
    {
        const int jr = tid % LS_NT, jk = tid / LS_NT;
        const int jy = y0 + jr % LS_BY, jz = z0 + (jr / LS_BY) % LS_BZ, jt = t0 + jr / (LS_BY * LS_BZ);
        const int jrr = (jy + jz + jt + a.p) & 1;              // 1: the row needs site 0 of the next x tile, 0: site 7 of the previous one
        const int nxtile = jrr ? (xt + 1 == P.nxt ? 0 : xt + 1) : (xt == 0 ? P.nxt - 1 : xt - 1);
        const int site = jrr ? 0 : 7;
        const unsigned int tile = (unsigned int)(nxtile + P.nxt * (jy + a.Ly * (jz + a.Lz * jt)));
        const unsigned int dtile = G::X + (jr >> 3) * G::TS;
        if (PREC == BQ_HALF && jk == 3) {
            xsrc = tile * G::TS + 384 + site * 4;
            xdst = dtile + 384 + (jr & 7) * 4;
        } else {
            xsrc = tile * G::TS + jk * 128 + site * 16;
            xdst = WX ? G::X + ((jr >> 1) * G::NW + jk) * 128 + (jrr ? 0 : 7 * 16) : dtile + jk * 128 + (jr & 7) * 16;
        }
    }
    const size_t slice_bytes = (size_t)P.nxt * a.Ly * a.Lz * G::TS;

    // ---- fills ----
    const int ym = y0 == 0 ? a.Ly - 1 : y0 - 1, yp = y0 + LS_BY == a.Ly ? 0 : y0 + LS_BY;
    const int zm = z0 == 0 ? a.Lz - 1 : z0 - 1, zp = z0 + LS_BZ == a.Lz ? 0 : z0 + LS_BZ;
    const int tm = t0 == 0 ? a.Lt - 1 : t0 - 1, tp = t0 + LS_BT == a.Lt ? 0 : t0 + LS_BT;
    constexpr int EH = G::SPLIT_T ? (G::TS / 2) / (int)sizeof(typename Prec<PREC>::real) : 0;   // element offset of the lower spin pair
    auto fill = [&](int i) {       // input tiles of the i-th active right-hand side -> stage i % NS   (all threads)
        const int k = rhs_of(i), s = i % NS;
        const unsigned int sb = ls_smem_u32(stage0 + s * G::STAGE), bar = ls_smem_u32(bars + s);
        // the 7 tensor copies are issued by lane 0 of 4 different warps (a transfer may complete before the expect_tx of
        // thread 0 is counted: the phase cannot end before all 1 + LS_THREADS arrivals are in)
        if ((tid & 31) == 0) {
            const int tk = k * P.tk_in, wq = (tid >> 5) & 3;
            if (wq == 0) {
                if (tid == 0) {
                    ls_mbar_expect_tx(bar, G::TX);
                    ls_tma5(sb + G::C, &P.m.in_c, bar, 0, xt, y0, z0, t0 + tk);
                }
            } else if (tid < 128) {
                if (wq == 1) {
                    ls_tma5(sb + G::YM, &P.m.in_y, bar, 0, xt, ym, z0, t0 + tk);
                    ls_tma5(sb + G::YP, &P.m.in_y, bar, 0, xt, yp, z0, t0 + tk);
                } else if (wq == 2) {
                    ls_tma5(sb + G::ZM, &P.m.in_z, bar, 0, xt, y0, zm, t0 + tk);
                    ls_tma5(sb + G::ZP, &P.m.in_z, bar, 0, xt, y0, zp, t0 + tk);
                } else {
                    // backward t hop: (1 + g_t) keeps the upper spin pair, forward: (1 - g_t) the lower one (exchanged for DAG)
                    ls_tma5(sb + G::TM, &P.m.in_t, bar, DAG ? EH : 0, xt, y0, z0, tm + tk);
                    ls_tma5(sb + G::TP, &P.m.in_t, bar, DAG ? 0 : EH, xt, y0, z0, tp + tk);
                }
            }
        }
        if (xcopy) {
            const char* src = static_cast<const char*>(a.in) + (size_t)k * a.s_in + xsrc;
            if (PREC == BQ_HALF && tid >= 3 * LS_NT) ls_cp_async<4>(sb + xdst, src);
            else ls_cp_async<16>(sb + xdst, src);
            ls_cp_async_arrive(bar);
        } else {
            ls_mbar_arrive(bar);
        }
    };
    auto fill_oper = [&](int i) {  // z and w of the i-th active right-hand side   (thread 0)
        if (EPI != 1) return;
        const int k = rhs_of(i);
        const unsigned int bar = ls_smem_u32(bars + NS);
        ls_mbar_expect_tx(bar, G::OPER * (RED == 1 ? 2 : 1));
        ls_tma5(ls_smem_u32(zbuf), &P.m.z_c, bar, 0, xt, y0, z0, t0 + k * P.tk_z);
        if (RED == 1) ls_tma5(ls_smem_u32(wbuf), &P.m.w_c, bar, 0, xt, y0, z0, t0 + k * P.tk_w);
    };
    for (int i = 0; i < NS && i < nact; i++) fill(i);
    if (tid == 0) fill_oper(0);
    if (EPI >= 2 && tid == 32) {     // the clover blocks of the block's sites: once, for all right-hand sides (a clover tile = 3 x 192 reals)
        const unsigned int bar = ls_smem_u32(bars + NS + 1);
        ls_mbar_expect_tx(bar, G::CLOV);
        ls_tma5(ls_smem_u32(cbuf), &P.m.cl_c, bar, 0, 3 * xt, y0, z0, t0);
    }

    // ---- neighbour addresses inside a stage (bytes from its base) ----
    const bool wxf = r && (xh == a.Lxh - 1), wxb = !r && (xh == 0);
    const bool wyf = (y == a.Ly - 1), wyb = (y == 0), wzf = (z == a.Lz - 1), wzb = (z == 0), wtf = (t == a.Lt - 1), wtb = (t == 0);
    int off[8];
    {
        const int ctile = G::C + tl * G::TS;
        const int xslot = WX ? G::X + (tl >> 1) * G::NW * 128 + (r ? 0 : 7 * 16) : G::X + (tl >> 3) * G::TS + (tl & 7) * 16;
        const int pf = r ? s8 + 1 : s8, pb = r ? s8 : s8 - 1;
        off[0] = pf < 8 ? ctile + pf * 16 : xslot;
        off[1] = pb >= 0 ? ctile + pb * 16 : xslot;
        off[2] = (ty + 1 < LS_BY ? ctile + G::TS : G::YP + (tz + LS_BZ * tt) * G::TS) + s8 * 16;
        off[3] = (ty > 0 ? ctile - G::TS : G::YM + (tz + LS_BZ * tt) * G::TS) + s8 * 16;
        off[4] = (tz + 1 < LS_BZ ? ctile + LS_BY * G::TS : G::ZP + (ty + LS_BY * tt) * G::TS) + s8 * 16;
        off[5] = (tz > 0 ? ctile - LS_BY * G::TS : G::ZM + (ty + LS_BY * tt) * G::TS) + s8 * 16;
        // t: in an interior tile the kept spin pair starts at plane NW/2 (lower) or 0 (upper); a halo tile holds only that pair
        constexpr int WF = G::SPLIT_T ? ((DAG ? 0 : 1) * G::TS / 2) : 0, WB = G::SPLIT_T ? ((DAG ? 1 : 0) * G::TS / 2) : 0;
        off[6] = (tt + 1 < LS_BT ? ctile + LS_BY * LS_BZ * G::TS + WF : G::TP + (ty + LS_BY * tz) * G::HT) + s8 * 16;
        off[7] = (tt > 0 ? ctile - LS_BY * LS_BZ * G::TS + WB : G::TM + (ty + LS_BY * tz) * G::HT) + s8 * 16;
    }
    // half storage: address of the neighbour's norm = its tile + 384 + position * 4
    int offn[PREC == BQ_HALF ? 8 : 1];
    if constexpr (PREC == BQ_HALF) {
        const int ctile = G::C + tl * G::TS, xtile = G::X + (tl >> 3) * G::TS;
        const int pf = r ? s8 + 1 : s8, pb = r ? s8 : s8 - 1;
        offn[0] = pf < 8 ? ctile + 384 + pf * 4 : xtile + 384 + (tl & 7) * 4;
        offn[1] = pb >= 0 ? ctile + 384 + pb * 4 : xtile + 384 + (tl & 7) * 4;
#pragma unroll
        for (int d = 2; d < 8; d++) offn[d] = off[d] - s8 * 16 + 384 + s8 * 4;
    } else {
        offn[0] = 0;
    }

    // ---- links: loaded once, kept for all right-hand sides ----
    LsLink<PREC, RECON> Lk[8];
    {
        const char* gf = static_cast<const char*>(a.gf);
        const char* gb = static_cast<const char*>(a.gb);
        const int nxb = r ? h : (wxb ? h + (a.Lxh - 1) : h - 1);
        const int nyb = wyb ? h + (a.Ly - 1) * sy : h - sy;
        const int nzb = wzb ? h + (a.Lz - 1) * sz : h - sz;
        const int ntb = wtb ? h + (a.Lt - 1) * st : h - st;
        ls_load_link<PREC, RECON>(Lk[0], gf, Vh, h);
        ls_load_link<PREC, RECON>(Lk[1], gb, Vh, nxb);
        ls_load_link<PREC, RECON>(Lk[2], gf + a.ublk, Vh, h);
        ls_load_link<PREC, RECON>(Lk[3], gb + a.ublk, Vh, nyb);
        ls_load_link<PREC, RECON>(Lk[4], gf + 2 * a.ublk, Vh, h);
        ls_load_link<PREC, RECON>(Lk[5], gb + 2 * a.ublk, Vh, nzb);
        ls_load_link<PREC, RECON>(Lk[6], gf + 3 * a.ublk, Vh, h);
        ls_load_link<PREC, RECON>(Lk[7], gb + 3 * a.ublk, Vh, ntb);
    }
    const C one = a.scale, zero = 0;
    const C w0r = wxf ? a.phr[0] : one, w0i = wxf ? a.phi[0] : zero, w1r = wxb ? a.phr[0] : one, w1i = wxb ? -a.phi[0] : zero;
    const C w2r = wyf ? a.phr[1] : one, w2i = wyf ? a.phi[1] : zero, w3r = wyb ? a.phr[1] : one, w3i = wyb ? -a.phi[1] : zero;
    const C w4r = wzf ? a.phr[2] : one, w4i = wzf ? a.phi[2] : zero, w5r = wzb ? a.phr[2] : one, w5i = wzb ? -a.phi[2] : zero;
    const C w6r = wtf ? a.phr[3] : one, w6i = wtf ? a.phi[3] : zero, w7r = wtb ? a.phr[3] : one, w7i = wtb ? -a.phi[3] : zero;

    // ---- the right-hand sides, one after the other ----
    for (int i = 0; i < nact; i++) {
        const int k = rhs_of(i), s = i % NS;
        const char* sb = reinterpret_cast<const char*>(stage0 + s * G::STAGE);
        if (EPI == 3 && s8 == 0) {   // the tile's 768 / 416 bytes of z (and w): asked into L2 now, read in the epilogue
            const char* zt = static_cast<const char*>(a.z) + (size_t)k * a.s_z + (size_t)(h >> 3) * G::TS;
#pragma unroll
            for (int q = 0; q < (G::TS + 127) / 128; q++) asm volatile("prefetch.global.L2 [%0];" ::"l"(zt + q * 128));
            if (RED == 1) {
                const char* wt = static_cast<const char*>(a.w) + (size_t)k * a.s_w + (size_t)(h >> 3) * G::TS;
#pragma unroll
                for (int q = 0; q < (G::TS + 127) / 128; q++) asm volatile("prefetch.global.L2 [%0];" ::"l"(wt + q * 128));
            }
        }
        ls_mbar_wait(ls_smem_u32(bars + s), (unsigned int)(i / NS) & 1u);
        C acc[24];
#pragma unroll
        for (int q = 0; q < 24; q++) acc[q] = 0;
        constexpr bool HN = PREC == BQ_HALF;
        ls_dir<PREC, RECON, 0, true, CPLX, DAG>(acc, sb + off[0], sb + offn[HN ? 0 : 0], Lk[0], w0r, w0i);
        ls_dir<PREC, RECON, 0, false, CPLX, DAG>(acc, sb + off[1], sb + offn[HN ? 1 : 0], Lk[1], w1r, w1i);
        ls_dir<PREC, RECON, 1, true, CPLX, DAG>(acc, sb + off[2], sb + offn[HN ? 2 : 0], Lk[2], w2r, w2i);
        ls_dir<PREC, RECON, 1, false, CPLX, DAG>(acc, sb + off[3], sb + offn[HN ? 3 : 0], Lk[3], w3r, w3i);
        ls_dir<PREC, RECON, 2, true, CPLX, DAG>(acc, sb + off[4], sb + offn[HN ? 4 : 0], Lk[4], w4r, w4i);
        ls_dir<PREC, RECON, 2, false, CPLX, DAG>(acc, sb + off[5], sb + offn[HN ? 5 : 0], Lk[5], w5r, w5i);
        ls_dir<PREC, RECON, 3, true, CPLX, DAG>(acc, sb + off[6], sb + offn[HN ? 6 : 0], Lk[6], w6r, w6i);
        ls_dir<PREC, RECON, 3, false, CPLX, DAG>(acc, sb + off[7], sb + offn[HN ? 7 : 0], Lk[7], w7r, w7i);
        if (DAG) {
#pragma unroll
            for (int q = 0; q < 12; q++) {
                const C tmp = acc[q];
                acc[q] = acc[12 + q];
                acc[12 + q] = tmp;
            }
        }
        C red[3] = {0, 0, 0};
        if (EPI == 2) {      // out = scale * Cl(H in): the scale already inside acc commutes with the site-diagonal multiply
            ls_mbar_wait(ls_smem_u32(bars + NS + 1), 0u);
            clover_site_mul<PREC, false>(cbuf, Vh, tl * 8 + s8, acc);
        }
        if (EPI == 1 || EPI == 3) {
            C zz[24];
            if (EPI == 1) {
                ls_mbar_wait(ls_smem_u32(bars + NS), (unsigned int)i & 1u);
                ls_load_site<PREC>(reinterpret_cast<const char*>(zbuf) + tl * G::TS, s8, zz);
#pragma unroll
                for (int q = 0; q < 24; q++) acc[q] += zz[q];
            } else {         // out = Cl(z) + scale * H in; z (and w below) straight from global memory: requested into L2 before the hops
                load_spinor<PREC, true>(static_cast<const char*>(a.z) + (size_t)k * a.s_z, Vh, h, zz);
                C az[24];
#pragma unroll
                for (int q = 0; q < 24; q++) az[q] = zz[q];
                ls_mbar_wait(ls_smem_u32(bars + NS + 1), 0u);
                clover_site_mul<PREC, false>(cbuf, Vh, tl * 8 + s8, az);
#pragma unroll
                for (int q = 0; q < 24; q++) acc[q] += az[q];
            }
            if (RED == 2) {
#pragma unroll
                for (int q = 0; q < 12; q++) {
                    red[0] = mad(acc[2 * q + 1], zz[2 * q + 1], mad(acc[2 * q], zz[2 * q], red[0]));
                    red[1] = mad(-acc[2 * q + 1], zz[2 * q], mad(acc[2 * q], zz[2 * q + 1], red[1]));
                    red[2] = mad(acc[2 * q + 1], acc[2 * q + 1], mad(acc[2 * q], acc[2 * q], red[2]));
                }
            }
            if (RED == 1) {
                C wv[24];
                if (EPI == 1) ls_load_site<PREC>(reinterpret_cast<const char*>(wbuf) + tl * G::TS, s8, wv);
                else load_spinor<PREC, true>(static_cast<const char*>(a.w) + (size_t)k * a.s_w, Vh, h, wv);
#pragma unroll
                for (int q = 0; q < 12; q++) {
                    red[0] = mad(wv[2 * q + 1], acc[2 * q + 1], mad(wv[2 * q], acc[2 * q], red[0]));
                    red[1] = mad(-wv[2 * q + 1], acc[2 * q], mad(wv[2 * q], acc[2 * q + 1], red[1]));
                }
            }
        }
        store_spinor<PREC, true>(static_cast<char*>(a.out) + (size_t)k * a.s_out, Vh, h, acc);
        if (RED) {
            double* sw = s_red + (i & 1) * NRED * (LS_THREADS / 32);
            const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
            for (int q = 0; q < NRED; q++) {
                const double x = warp_sum((double)red[q]);
                if (lane == 0) sw[q * (LS_THREADS / 32) + warp] = x;
            }
        }
        __syncthreads();     // every thread is done with stage s and with the operand buffers
        if (RED && tid < NRED) {
            const double* sw = s_red + (i & 1) * NRED * (LS_THREADS / 32) + tid * (LS_THREADS / 32);
            double v = 0;
#pragma unroll
            for (int q = 0; q < LS_THREADS / 32; q++) v += sw[q];
            a.partials[((size_t)k * gridDim.x + blockIdx.x) * NRED + tid] = v;
        }
        if (i + NS < nact) fill(i + NS);
        if (tid == 0 && i + 1 < nact) fill_oper(i + 1);
    }
}

// ---------------------------------------------------------------------------------------------------
// host side: tensor maps and launch
// ---------------------------------------------------------------------------------------------------
typedef CUresult (*ls_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                 const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
ls_encode_fn ls_get_encoder();     // hop.cu: cuTensorMapEncodeTiled through cudaGetDriverEntryPoint (no link-time dependency on libcuda)

// field of `nf` right-hand sides, consecutive ones `tk` t-slices apart, as a 5-D tensor (tile element, x tile, y, z, t');
// box = (e_box, 1, by, bz, bt) tiles
template <int PREC>
static bool ls_make_map(CUtensorMap* m, const void* base, const Geom& g, int nf, int tk, int e_box, int by, int bz, int bt) {
    using G = LsGeom<PREC>;
    ls_encode_fn enc = ls_get_encoder();
    if (!enc) return false;
    const int nxt = g.Lxh / 8;
    const cuuint64_t es = prec_real_bytes(PREC);
    const cuuint64_t dims[5] = {(cuuint64_t)(G::TS / es), (cuuint64_t)nxt, (cuuint64_t)g.L[1], (cuuint64_t)g.L[2],
                                (cuuint64_t)((nf - 1) * (cuuint64_t)tk + g.L[3])};
    const cuuint64_t strides[4] = {(cuuint64_t)G::TS, (cuuint64_t)G::TS * nxt, (cuuint64_t)G::TS * nxt * g.L[1],
                                   (cuuint64_t)G::TS * nxt * g.L[1] * g.L[2]};
    const cuuint32_t box[5] = {(cuuint32_t)e_box, 1u, (cuuint32_t)by, (cuuint32_t)bz, (cuuint32_t)bt};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUtensorMapDataType dt = PREC == BQ_FP64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64
                                                   : (PREC == BQ_FP32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_UINT16);
    return enc(m, dt, 5, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
               CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Can this launch take the link-stationary kernel?  (geometry, operand strides, epilogue)
template <int PREC> static bool ls_eligible(const bq_lattice* lat, const HopMulti* m, const void* in, const void* z, const void* w, int cl_mode) {
    if constexpr (PREC == BQ_FP64) return false;
    if (!m || !lat->mrhs_ls || cl_mode < 0 || cl_mode > 2) return false;
    const Geom& g = lat->g;
    if (m->nrhs < 2 || m->nrhs > LS_MAX_RHS) return false;
    if (g.Lxh % 8 || g.L[1] % LS_BY || g.L[2] % LS_BZ || g.L[3] % LS_BT) return false;
    const size_t slice = (size_t)(g.Lxh / 8) * g.L[1] * g.L[2] * LsGeom<PREC>::TS;
    // z and w come through TMA for the Wilson xpay epilogue (their strides must be whole t slices), by plain loads for the clover ones
    if (m->s_in % slice || (cl_mode == 0 && ((z && m->s_z % slice) || (w && m->s_w % slice)))) return false;
    if (((uintptr_t)in & 15) || ((uintptr_t)z & 15) || ((uintptr_t)w & 15)) return false;
    return ls_get_encoder() != nullptr;
}

template <int PREC, int RECON, int EPI, bool CPLX, int RED, bool DAG>
static bq_status ls_launch_one(bq_lattice* lat, const LsParams<typename Prec<PREC>::comp>& P, int grid, cudaStream_t stream) {
    constexpr size_t smem = ls_smem_bytes<PREC, EPI, RED>();
    // the shared-memory limit is a property of the (kernel, device) pair: remember it per device ordinal, not per process
    static bool attr_set[64] = {};
    int dev = 0;
    BQ_CUDA(lat, cudaGetDevice(&dev));
    const bool known = dev >= 0 && dev < 64;
    auto kern = hop_ls_kernel<PREC, RECON, EPI, CPLX, RED, DAG>;
    if (!known || !attr_set[dev]) {
        BQ_CUDA(lat, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (known) attr_set[dev] = true;
    }
    kern<<<grid, LS_THREADS, smem, stream>>>(P);
    return BQ_OK;
}

// a: the HopArgs launch_hop has filled (operands, links, geometry, weights, partials); nslots_out: partial sums per rhs
template <int PREC, int RECON>
static bq_status ls_launch(bq_lattice* lat, const HopArgs<typename Prec<PREC>::comp>& a, bool cplx, int rmode, bool dag, const HopMulti* m,
                           const SolverScalars* done, cudaStream_t stream, int cl_mode) {
    using C = typename Prec<PREC>::comp;
    using G = LsGeom<PREC>;
    const Geom& g = lat->g;
    LsParams<C> P;
    P.a = a;
    P.nxt = g.Lxh / 8; P.nyb = g.L[1] / LS_BY; P.nzb = g.L[2] / LS_BZ;
    const size_t slice = (size_t)P.nxt * g.L[1] * g.L[2] * G::TS;
    P.tk_in = (int)(m->s_in / slice); P.tk_z = a.z ? (int)(m->s_z / slice) : 0; P.tk_w = a.w ? (int)(m->s_w / slice) : 0;
    P.done = done;
    ls_brick(P.nyb, P.nzb, g.L[3] / LS_BT, P.gy, P.gz, P.gt);
    const int E = G::TS / (int)prec_real_bytes(PREC);
    bool ok = ls_make_map<PREC>(&P.m.in_c, a.in, g, m->nrhs, P.tk_in, E, LS_BY, LS_BZ, LS_BT) &&
              ls_make_map<PREC>(&P.m.in_y, a.in, g, m->nrhs, P.tk_in, E, 1, LS_BZ, LS_BT) &&
              ls_make_map<PREC>(&P.m.in_z, a.in, g, m->nrhs, P.tk_in, E, LS_BY, 1, LS_BT) &&
              ls_make_map<PREC>(&P.m.in_t, a.in, g, m->nrhs, P.tk_in, G::SPLIT_T ? E / 2 : E, LS_BY, LS_BZ, 1);
    const bool tma_zw = cl_mode == 0;
    ok = ok && ls_make_map<PREC>(&P.m.z_c, tma_zw && a.z ? a.z : a.in, g, m->nrhs, tma_zw && a.z ? P.tk_z : P.tk_in, E, LS_BY, LS_BZ, LS_BT);
    ok = ok && ls_make_map<PREC>(&P.m.w_c, tma_zw && a.w ? a.w : a.in, g, m->nrhs, tma_zw && a.w ? P.tk_w : P.tk_in, E, LS_BY, LS_BZ, LS_BT);
    if (cl_mode) {
        // the clover store of one parity as a 5-D tensor of 192-real pieces: a tile of 8 sites x 72 reals is 3 of them
        ls_encode_fn enc = ls_get_encoder();
        const cuuint64_t es = prec_real_bytes(PREC), piece = 192 * es;
        const cuuint64_t dims[5] = {192, (cuuint64_t)3 * P.nxt, (cuuint64_t)g.L[1], (cuuint64_t)g.L[2], (cuuint64_t)g.L[3]};
        const cuuint64_t strides[4] = {piece, piece * 3 * P.nxt, piece * 3 * P.nxt * g.L[1], piece * 3 * P.nxt * g.L[1] * g.L[2]};
        const cuuint32_t box[5] = {192, 3, LS_BY, LS_BZ, LS_BT}, estr[5] = {1, 1, 1, 1, 1};
        ok = ok && enc && enc(&P.m.cl_c, PREC == BQ_FP32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_UINT16, 5, const_cast<void*>(a.cl), dims,
                              strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
    } else {
        P.m.cl_c = P.m.in_c;
    }
    if (!ok) return bq_set_error(lat, BQ_ECUDA, "bq_hop: cuTensorMapEncodeTiled failed");
    const int grid = P.nxt * P.nyb * P.nzb * (g.L[3] / LS_BT);
    const int epi = cl_mode == 0 ? (a.z ? 1 : 0) : (cl_mode == 1 ? 2 : 3);
#define LS_GO(E_, R_)                                                                                                   \
    do {                                                                                                                \
        if (dag) return cplx ? ls_launch_one<PREC, RECON, E_, true, 0, true>(lat, P, grid, stream)                      \
                             : ls_launch_one<PREC, RECON, E_, false, 0, true>(lat, P, grid, stream);                    \
        return cplx ? ls_launch_one<PREC, RECON, E_, true, R_, false>(lat, P, grid, stream)                             \
                    : ls_launch_one<PREC, RECON, E_, false, R_, false>(lat, P, grid, stream);                           \
    } while (0)
    if (epi == 0) LS_GO(0, 0);
    if (epi == 2) LS_GO(2, 0);
    if (epi == 1) {
        if (rmode == 0) LS_GO(1, 0);
        if (rmode == 1) LS_GO(1, 1);
        LS_GO(1, 2);
    }
    if (rmode == 0) LS_GO(3, 0);
    if (rmode == 1) LS_GO(3, 1);
    LS_GO(3, 2);
#undef LS_GO
}
