// hop_lsp.cuh — link-stationary multi-right-hand-side hop, DIRECTION-SPLIT and PIPELINED (the
// paper's workload is the 12 spin-colour sources of a propagator on ONE gauge field).
//
// hop_ls.cuh keeps the 8 links of a site in the registers of ONE thread (144 registers in fp32): 8 warps per SM, the
// issue slots 59 % busy (profiles/r2_hop_ls.md), and no room at all for fp64 links (288 registers).  Here TWO threads
// serve a site, four directions each, and the accumulator travels between them through shared memory — in the order
// of the single-rhs kernel, so the result stays bit for bit that of hop_kernel:
//   * role A (threads 0..127 of a CTA, one per site of the 8 x 4 x 4 x 1 block) holds the x and y links and adds the hops
//     +x, -x, +y, -y of right-hand side i into a zero accumulator (step i of the CTA's loop), then writes the 24 sums
//     into the hand-off buffer;
//   * role B (threads 128..255) holds the z and t links, picks the sums of right-hand side i - 1 up in step i, adds
//     +z, -z, +t, -t, runs the epilogue (xpay operand and the fused inner products; z and w come by plain streaming
//     loads, requested into L2 at the top of the step) and stores.
// A software pipeline one step deep: while A works on right-hand side i, B finishes i - 1.  72 link registers per
// thread instead of 144 -> 128 registers, two 256-thread CTAs per SM = 16 warps (fp64: 255 registers, one CTA).
// Half storage: the spatial links sit unpacked (fp32) in registers — their 18 conversions per direction are paid once
// per block instead of once per right-hand side; the t links stay packed for the fp16 x fp16 FHFMA path of hop.cuh.
//
// Spinors stream through shared memory by TMA as in hop_ls.cuh, but in three rings so that what only one role needs is
// held only as long as that role needs it (two whole 3-deep stages per CTA would not fit twice on an SM):
//   C  ring, 3 slots: the block's own 16 tiles (x/y neighbours for A in step i, z/t neighbours for B in step i + 1);
//   AH ring, 2 slots: y halos + the x-halo sites (cp.async), used by A in step i;
//   BH ring, 2 slots: z halos + t halos (half tiles: only the spin pair the projector keeps), used by B in step i + 1.
// Slot j % n of a ring is refilled right behind the CTA barrier that ends the last step using it, one whole step before
// its next use.  fp32: 3 x 12288 + 2 x 7680 + 2 x 18432 + 12288 (hand-off) = 101.4 KB per CTA.
// Wilson epilogues (EPI 0, 1); the clover epilogues stay with hop_ls.cuh.  Same geometry conditions as hop_ls.cuh.
#pragma once

static_assert(BQ_TILED, "the link-stationary kernels address tiles");

constexpr int LP_SITES = 8 * LS_NT;          // output sites per CTA
constexpr int LP_THREADS = 2 * LP_SITES;     // role A | role B

template <int PREC> struct LpGeom {
    using G = LsGeom<PREC>;
    using C = typename Prec<PREC>::comp;
    static constexpr int TS = G::TS, HT = G::HT;
    static constexpr int CS = LS_NT * TS;                                          // one C slot
    static constexpr int A_YM = 0, A_YP = A_YM + LS_BZ * LS_BT * TS, A_X = A_YP + LS_BZ * LS_BT * TS;
    static constexpr int AHS = (A_X + (LS_NT / 8) * TS + 127) / 128 * 128;        // one AH slot
    static constexpr int A_TX = CS + 2 * LS_BZ * LS_BT * TS;                       // bytes a fill of (C, AH) receives through TMA
    static constexpr int B_ZM = 0, B_ZP = B_ZM + LS_BY * LS_BT * TS, B_TM = B_ZP + LS_BY * LS_BT * TS, B_TP = B_TM + LS_BY * LS_BZ * HT;
    static constexpr int BHS = B_TP + LS_BY * LS_BZ * HT;                          // one BH slot (all of it through TMA)
    static constexpr int NC = 3, NA = 2, NB = 2;
    static constexpr int HW = 24 * (int)sizeof(C) / 16;                            // 16-byte words of an accumulator
    static constexpr int HAND = LP_SITES * 24 * (int)sizeof(C);
    static constexpr int TAB = LP_THREADS * 24;   // per-thread constants (neighbour slots, output offset, wrap bits, x-halo copy): see the kernel
    static constexpr int R_C = 0, R_A = R_C + NC * CS, R_B = R_A + NA * AHS, R_H = R_B + NB * BHS, R_T = R_H + HAND, R_CTL = R_T + TAB;
    static constexpr int TOTAL = R_CTL + 512;     // control: mbarriers (64 B), active list (192 B), reduction scratch (256 B)
    static_assert(CS % 128 == 0 && AHS % 128 == 0 && BHS % 128 == 0 && A_YP % 128 == 0 && B_ZP % 128 == 0 && B_TM % 128 == 0 && B_TP % 128 == 0,
                  "TMA destinations are 128-byte aligned");
    static_assert(G::NXC <= LP_THREADS, "one x-halo copy per thread");
    static_assert(TOTAL <= 232448, "shared memory of one CTA");
};

template <typename C> struct LpParams {
    HopArgs<C> a;
    alignas(64) CUtensorMap in_c, in_y, in_z, in_t;   // input field: interior box, y-halo box, z-halo box, t-halo box
    int nxt, nyb, nzb;           // x tiles per row; blocks in y, z
    int gy, gz, gt;              // launch order of the blocks: bricks of nxt x gy x gz x gt blocks (ls_block_coords)
    int tk_in;                   // t'-extent between consecutive right-hand sides of `in`
    const SolverScalars* done;   // solver: per-rhs states whose `done` flag switches a right-hand side off (nullptr: all run)
};

// threadIdx.x read afresh (S2R): inside the loop over the right-hand sides nothing derived from the thread index is kept in a
// register — ptxas spills such loop invariants first, and a spill costs an L2 round trip per step here
__device__ __forceinline__ unsigned int lp_tid() {
    unsigned int t;
    asm volatile("mov.u32 %0, %%tid.x;" : "=r"(t));
    return t;
}
__device__ __forceinline__ void lp_bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void lp_bar_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }

// One hop with the neighbour spinor in shared memory and the link in registers; arithmetic = hop_dir (hop.cuh) step by step.
// u: the link as 18 reals of the compute type (row 2 already rebuilt for 12-real storage); tw: half storage, 18-real, t direction:
// the link packed as stored (fp16 x fp16 products, su3_mul_h16).
template <int PREC, int RECON, int MU, bool FWD, bool CPLX, bool DAG>
__device__ __forceinline__ void lp_dir(typename Prec<PREC>::comp* acc, const char* sp, const char* np, const typename Prec<PREC>::comp* u,
                                       const unsigned int* tw, typename Prec<PREC>::comp pr, typename Prec<PREC>::comp pi) {
    using C = typename Prec<PREC>::comp;
    C h[12], chi[12];
    C w = pr;
    if constexpr (PREC == BQ_HALF) {
        const float n = *reinterpret_cast<const float*>(np);
        if (MU < 3) {
            const uint4 s0 = *reinterpret_cast<const uint4*>(sp);
            const uint4 s1 = *reinterpret_cast<const uint4*>(sp + 128);
            const uint4 s2 = *reinterpret_cast<const uint4*>(sp + 256);
            const unsigned int pw[12] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w, s2.x, s2.y, s2.z, s2.w};
            const unsigned int* upw = DAG ? pw + 6 : pw;
            const unsigned int* low = DAG ? pw : pw + 6;
#pragma unroll
            for (int c = 0; c < 6; c++) {
                const float2 t = __half22float2(*reinterpret_cast<const __half2*>(&upw[c]));
                h[2 * c] = t.x; h[2 * c + 1] = t.y;
            }
            add_isigma_h16<MU, FWD>(h, low);
            su3_mul<!FWD>(u, h, chi);
        } else {
            constexpr int W = (FWD != DAG) ? 1 : 0;
            const uint4 s0 = *reinterpret_cast<const uint4*>(sp + (W ? 256 : 0));
            const uint2 d = *reinterpret_cast<const uint2*>(sp + 128 + (W ? 8 : 0));
            if constexpr (RECON == BQ_RECON18) {
                const unsigned int hw[6] = {W ? d.x : s0.x, W ? d.y : s0.y, W ? s0.x : s0.z, W ? s0.y : s0.w, W ? s0.z : d.x, W ? s0.w : d.y};
                su3_mul_h16<!FWD>(tw, hw, chi);
            } else {
                if (W == 0) { unpack8(s0, h); unpack4(d, h + 8); }
                else { unpack4(d, h); unpack8(s0, h + 4); }
                su3_mul<!FWD>(u, h, chi);
            }
        }
        if (CPLX) {
            phase_mul(chi, pr, pi);
            w = 1.0f;
        }
        w *= n;
    } else {
        using V = typename std::conditional<PREC == BQ_FP64, double2, float4>::type;
        constexpr int W = 16 / sizeof(C), NWS = 24 / W;      // reals per word, words per site
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
        su3_mul<!FWD>(u, h, chi);
        if (CPLX) {
            phase_mul(chi, pr, pi);
            w = C(1);
        }
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

template <int PREC, int RECON, int EPI, bool CPLX, int RED, bool DAG>
__global__ void __launch_bounds__(LP_THREADS, PREC == BQ_FP64 ? 1 : 2) hop_lsp_kernel(const __grid_constant__ LpParams<typename Prec<PREC>::comp> P) {
    using C = typename Prec<PREC>::comp;
    using G = LsGeom<PREC>;
    using Q = LpGeom<PREC>;
    using V = typename std::conditional<PREC == BQ_FP64, double2, float4>::type;
    static_assert(EPI == 0 || EPI == 1, "Wilson epilogues only");
    constexpr int NRED = RED == 1 ? 2 : 3;
    constexpr bool TPACK = PREC == BQ_HALF && RECON == BQ_RECON18;      // t links stay packed
    extern __shared__ __align__(128) unsigned char lp_smem[];
    unsigned char* const ctl = lp_smem + Q::R_CTL;
    unsigned long long* const bars = reinterpret_cast<unsigned long long*>(ctl);     // barA[3], barB[2]
    int* const act = reinterpret_cast<int*>(ctl + 64);                              // [0] = count, [1] = mask, [2..] = active rhs
    double* const s_red = reinterpret_cast<double*>(ctl + 256);                     // [2][NRED][4 B-warps]
    const HopArgs<C>& a = P.a;

    const int tid = threadIdx.x;
    const bool roleB = tid >= LP_SITES;
    const int ts = roleB ? tid - LP_SITES : tid, s8 = ts & 7, tl = ts >> 3;
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
        if (mask & (1u << tid)) act[2 + __popc(mask & ((1u << tid) - 1u))] = tid;
        if (tid == 0) {
            act[0] = __popc(mask);
            act[1] = (int)mask;
            for (int s = 0; s < Q::NC; s++) ls_mbar_init(ls_smem_u32(bars + s), 1 + LP_THREADS);
            for (int s = 0; s < Q::NB; s++) ls_mbar_init(ls_smem_u32(bars + Q::NC + s), 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    __syncthreads();
    const int nact = act[0];
    if (nact == 0) return;
    auto rhs_of = [&](int i) { return act[2 + i]; };

    // Per-thread constants live in SHARED memory, not in registers (16 + 8 bytes per thread, read back once per step): with 72
    // link registers and 24 accumulators the 128-register budget has no room for loop invariants, and a spilled one costs an
    // L2 round trip per step here (the L1 is carved down to a few KB by the 2 x 106 KB of shared memory).
    //   tab4[tid] = { f0 | f1 << 16, f2 | f3 << 16, output site offset / 16, wrap bits };  f_d = slot of the neighbour in direction d of
    //   this role: (tile base / 16) | position in the tile << 12 | (1 << 15 if the tile is in the C ring, else in the role's halo ring)
    //   tab2[tid] = { x-halo copy: source offset in the field, destination offset in the AH slot }
    uint4* const tab4 = reinterpret_cast<uint4*>(lp_smem + Q::R_T);
    uint2* const tab2 = reinterpret_cast<uint2*>(lp_smem + Q::R_T + LP_THREADS * 16);
    {
        const int jr = tid % LS_NT, jk = tid / LS_NT;
        const int jy = y0 + jr % LS_BY, jz = z0 + (jr / LS_BY) % LS_BZ, jt = t0 + jr / (LS_BY * LS_BZ);
        const int jrr = (jy + jz + jt + a.p) & 1;              // 1: the row needs site 0 of the next x tile, 0: site 7 of the previous one
        const int nxtile = jrr ? (xt + 1 == P.nxt ? 0 : xt + 1) : (xt == 0 ? P.nxt - 1 : xt - 1);
        const int site = jrr ? 0 : 7;
        const unsigned int tile = (unsigned int)(nxtile + P.nxt * (jy + a.Ly * (jz + a.Lz * jt)));
        const unsigned int dtile = Q::A_X + (jr >> 3) * G::TS;
        unsigned int xsrc, xdst;
        if (PREC == BQ_HALF && jk == 3) {
            xsrc = tile * G::TS + 384 + site * 4;
            xdst = dtile + 384 + (jr & 7) * 4;
        } else {
            xsrc = tile * G::TS + jk * 128 + site * 16;
            xdst = dtile + jk * 128 + (jr & 7) * 16;
        }
        tab2[tid] = make_uint2(xsrc, xdst);
    }

    // ---- fills ----
    const int ym = y0 == 0 ? a.Ly - 1 : y0 - 1, yp = y0 + LS_BY == a.Ly ? 0 : y0 + LS_BY;
    const int zm = z0 == 0 ? a.Lz - 1 : z0 - 1, zp = z0 + LS_BZ == a.Lz ? 0 : z0 + LS_BZ;
    const int tm = t0 == 0 ? a.Lt - 1 : t0 - 1, tp = t0 + LS_BT == a.Lt ? 0 : t0 + LS_BT;
    constexpr int EH = G::SPLIT_T ? (G::TS / 2) / (int)sizeof(typename Prec<PREC>::real) : 0;   // element offset of the lower spin pair
    const unsigned int smem0 = ls_smem_u32(lp_smem);
    auto fillA = [&](int j) {      // C and AH of the j-th active right-hand side   (all threads: each arrives once on barA[j % 3])
        const int k = rhs_of(j);
        const unsigned int cb = smem0 + Q::R_C + (j % Q::NC) * Q::CS, ab = smem0 + Q::R_A + (j % Q::NA) * Q::AHS;
        const unsigned int bar = ls_smem_u32(bars + j % Q::NC);
        const int tk = k * P.tk_in;
        const unsigned int tid = lp_tid();
        if (tid == 0) {
            ls_mbar_expect_tx(bar, Q::A_TX);
            ls_tma5(cb, &P.in_c, bar, 0, xt, y0, z0, t0 + tk);
        } else if (tid == 32) {      // (a transfer may complete before the expect_tx of thread 0 is counted: the phase cannot end before all arrivals)
            ls_tma5(ab + Q::A_YM, &P.in_y, bar, 0, xt, ym, z0, t0 + tk);
            ls_tma5(ab + Q::A_YP, &P.in_y, bar, 0, xt, yp, z0, t0 + tk);
        }
        if (tid < G::NXC) {
            const uint2 xc = tab2[tid];
            const char* src = static_cast<const char*>(a.in) + (size_t)k * a.s_in + xc.x;
            if (PREC == BQ_HALF && tid >= 3 * LS_NT) ls_cp_async<4>(ab + xc.y, src);
            else ls_cp_async<16>(ab + xc.y, src);
            ls_cp_async_arrive(bar);
        } else {
            ls_mbar_arrive(bar);
        }
    };
    auto fillB = [&](int j) {      // BH of the j-th active right-hand side   (one thread)
        if (lp_tid() != LP_SITES) return;
        const int k = rhs_of(j), tk = k * P.tk_in;
        const unsigned int bb = smem0 + Q::R_B + (j % Q::NB) * Q::BHS, bar = ls_smem_u32(bars + Q::NC + j % Q::NB);
        ls_mbar_expect_tx(bar, Q::BHS);
        ls_tma5(bb + Q::B_ZM, &P.in_z, bar, 0, xt, y0, zm, t0 + tk);
        ls_tma5(bb + Q::B_ZP, &P.in_z, bar, 0, xt, y0, zp, t0 + tk);
        // backward t hop: (1 + g_t) keeps the upper spin pair, forward: (1 - g_t) the lower one (exchanged for DAG)
        ls_tma5(bb + Q::B_TM, &P.in_t, bar, DAG ? EH : 0, xt, y0, z0, tm + tk);
        ls_tma5(bb + Q::B_TP, &P.in_t, bar, DAG ? 0 : EH, xt, y0, z0, tp + tk);
    };
    fillA(0);
    if (nact > 1) fillA(1);
    fillB(0);
    if (nact > 1) fillB(1);

    // ---- neighbour slots, output offset and wrap bits of this thread -> tab4 (see above) ----
    const bool wxf = r && (xh == a.Lxh - 1), wxb = !r && (xh == 0);
    const bool wyf = (y == a.Ly - 1), wyb = (y == 0), wzf = (z == a.Lz - 1), wzb = (z == 0), wtf = (t == a.Lt - 1), wtb = (t == 0);
    {
        auto slot = [](int tile_base, int pos, bool in_c) { return (unsigned int)(tile_base >> 4) | ((unsigned int)pos << 12) | (in_c ? 0x8000u : 0u); };
        const int ctile = tl * G::TS;
        unsigned int f[4], wbits;
        if (!roleB) {
            const int xtile = Q::A_X + (tl >> 3) * G::TS;
            const int pf = r ? s8 + 1 : s8, pb = r ? s8 : s8 - 1;
            f[0] = pf < 8 ? slot(ctile, pf, true) : slot(xtile, tl & 7, false);
            f[1] = pb >= 0 ? slot(ctile, pb, true) : slot(xtile, tl & 7, false);
            f[2] = ty + 1 < LS_BY ? slot(ctile + G::TS, s8, true) : slot(Q::A_YP + (tz + LS_BZ * tt) * G::TS, s8, false);
            f[3] = ty > 0 ? slot(ctile - G::TS, s8, true) : slot(Q::A_YM + (tz + LS_BZ * tt) * G::TS, s8, false);
            wbits = (wxf ? 1u : 0u) | (wxb ? 2u : 0u) | (wyf ? 4u : 0u) | (wyb ? 8u : 0u);
        } else {
            f[0] = tz + 1 < LS_BZ ? slot(ctile + LS_BY * G::TS, s8, true) : slot(Q::B_ZP + (ty + LS_BY * tt) * G::TS, s8, false);
            f[1] = tz > 0 ? slot(ctile - LS_BY * G::TS, s8, true) : slot(Q::B_ZM + (ty + LS_BY * tt) * G::TS, s8, false);
            // t: in an interior tile the kept spin pair starts at plane NW/2 (lower) or 0 (upper); a halo tile holds only that pair
            constexpr int WF = G::SPLIT_T ? ((DAG ? 0 : 1) * G::TS / 2) : 0, WB = G::SPLIT_T ? ((DAG ? 1 : 0) * G::TS / 2) : 0;
            f[2] = tt + 1 < LS_BT ? slot(ctile + LS_BY * LS_BZ * G::TS + WF, s8, true) : slot(Q::B_TP + (ty + LS_BY * tz) * G::HT, s8, false);
            f[3] = tt > 0 ? slot(ctile - LS_BY * LS_BZ * G::TS + WB, s8, true) : slot(Q::B_TM + (ty + LS_BY * tz) * G::HT, s8, false);
            wbits = (wzf ? 1u : 0u) | (wzb ? 2u : 0u) | (wtf ? 4u : 0u) | (wtb ? 8u : 0u);
        }
        const unsigned int osite = (unsigned int)(((size_t)(h >> 3) * G::TS) >> 4);      // the site's tile, in 16-byte units
        tab4[tid] = make_uint4(f[0] | (f[1] << 16), f[2] | (f[3] << 16), osite, wbits);
    }

    // ---- links: this role's four, loaded once, kept for all right-hand sides ----
    C u[4][18];
    unsigned int tw[TPACK ? 2 : 1][9];
    {
        const char* gf = static_cast<const char*>(a.gf);
        const char* gb = static_cast<const char*>(a.gb);
        if (!roleB) {
            const int nxb = r ? h : (wxb ? h + (a.Lxh - 1) : h - 1);
            const int nyb = wyb ? h + (a.Ly - 1) * sy : h - sy;
            load_link<PREC, RECON, true>(gf, Vh, h, u[0]);
            load_link<PREC, RECON, true>(gb, Vh, nxb, u[1]);
            load_link<PREC, RECON, true>(gf + a.ublk, Vh, h, u[2]);
            load_link<PREC, RECON, true>(gb + a.ublk, Vh, nyb, u[3]);
        } else {
            const int nzb = wzb ? h + (a.Lz - 1) * sz : h - sz;
            const int ntb = wtb ? h + (a.Lt - 1) * st : h - st;
            load_link<PREC, RECON, true>(gf + 2 * a.ublk, Vh, h, u[0]);
            load_link<PREC, RECON, true>(gb + 2 * a.ublk, Vh, nzb, u[1]);
            if constexpr (TPACK) {
                using LA = LinkAddr<BQ_HALF, RECON>;
#pragma unroll
                for (int q = 0; q < 2; q++) {
                    const char* ub = (q ? gb : gf) + 3 * a.ublk;
                    const int idx = q ? ntb : h;
                    const uint4 l0 = ld16<true, uint4>(ub + LA::word(Vh, idx, 0)), l1 = ld16<true, uint4>(ub + LA::word(Vh, idx, 1));
                    tw[q][0] = l0.x; tw[q][1] = l0.y; tw[q][2] = l0.z; tw[q][3] = l0.w;
                    tw[q][4] = l1.x; tw[q][5] = l1.y; tw[q][6] = l1.z; tw[q][7] = l1.w;
                    tw[q][8] = ld16<true, unsigned int>(ub + LA::tail(Vh, idx));
                }
            } else {
                load_link<PREC, RECON, true>(gf + 3 * a.ublk, Vh, h, u[2]);
                load_link<PREC, RECON, true>(gb + 3 * a.ublk, Vh, ntb, u[3]);
            }
        }
    }

    // neighbour address of direction d from its packed slot f: site word 0 (sp) and, half storage, the site norm (np)
    auto nb_addr = [&](unsigned int f, const char* cb, const char* hb, const char*& sp, const char*& np) {
        const char* tile = ((f & 0x8000u) ? cb : hb) + ((f & 0xfffu) << 4);
        const unsigned int pos = (f >> 12) & 7u;
        sp = tile + pos * 16;
        np = PREC == BQ_HALF ? tile + 384 + pos * 4 : tile;
    };
    // weight of direction d of this role (mu = its axis): scale x boundary phase if the hop wraps, else scale
    auto weight = [&](unsigned int wbits, int d, int mu, C& pr, C& pi) {
        const bool wrap = (wbits >> d) & 1u;
        pr = wrap ? a.phr[mu] : a.scale;
        pi = wrap ? ((d & 1) ? -a.phi[mu] : a.phi[mu]) : C(0);
    };

    // ---- the pipeline: step i = A on right-hand side i, B on right-hand side i - 1 ----
    for (int i = 0; i <= nact; i++) {
        if (!roleB) {       // (a bool that ptxas keeps in a predicate register: no S2R on the critical path of the step)
            if (i < nact) {
                const char* cb = reinterpret_cast<const char*>(lp_smem) + Q::R_C + (i % Q::NC) * Q::CS;
                const char* hb = reinterpret_cast<const char*>(lp_smem) + Q::R_A + (i % Q::NA) * Q::AHS;
                ls_mbar_wait(ls_smem_u32(bars + i % Q::NC), (unsigned int)(i / Q::NC) & 1u);
                const uint4 tb4 = tab4[lp_tid()];
                C acc[24];
#pragma unroll
                for (int q = 0; q < 24; q++) acc[q] = 0;
                const char *sp, *np;
                C pr, pi;
                nb_addr(tb4.x & 0xffffu, cb, hb, sp, np); weight(tb4.w, 0, 0, pr, pi);
                lp_dir<PREC, RECON, 0, true, CPLX, DAG>(acc, sp, np, u[0], nullptr, pr, pi);
                nb_addr(tb4.x >> 16, cb, hb, sp, np); weight(tb4.w, 1, 0, pr, pi);
                lp_dir<PREC, RECON, 0, false, CPLX, DAG>(acc, sp, np, u[1], nullptr, pr, pi);
                nb_addr(tb4.y & 0xffffu, cb, hb, sp, np); weight(tb4.w, 2, 1, pr, pi);
                lp_dir<PREC, RECON, 1, true, CPLX, DAG>(acc, sp, np, u[2], nullptr, pr, pi);
                nb_addr(tb4.y >> 16, cb, hb, sp, np); weight(tb4.w, 3, 1, pr, pi);
                lp_dir<PREC, RECON, 1, false, CPLX, DAG>(acc, sp, np, u[3], nullptr, pr, pi);
                if (i >= 1) lp_bar_sync(1, LP_THREADS);      // B has picked up the sums of right-hand side i - 1
                unsigned char* const hand = lp_smem + Q::R_H + lp_tid() * 16;      // word q of this site's accumulator: hand + q * (LP_SITES * 16)
#pragma unroll
                for (int q = 0; q < Q::HW; q++) {
                    if constexpr (PREC == BQ_FP64) *reinterpret_cast<double2*>(hand + q * (LP_SITES * 16)) = make_double2(acc[2 * q], acc[2 * q + 1]);
                    else *reinterpret_cast<float4*>(hand + q * (LP_SITES * 16)) = make_float4(acc[4 * q], acc[4 * q + 1], acc[4 * q + 2], acc[4 * q + 3]);
                }
            }
        } else if (i >= 1) {
            const int j = i - 1, k = rhs_of(j);
            const uint4 tb4 = tab4[lp_tid()];
            const size_t otile = (size_t)tb4.z << 4;          // byte offset of this thread's tile in a field; its site is number tid & 7 there
            if (EPI == 1 && (lp_tid() & 7) == 0) {   // the tile's bytes of z (and w): asked into L2 now, read in the epilogue
                const char* zt = static_cast<const char*>(a.z) + (size_t)k * a.s_z + otile;
#pragma unroll
                for (int q = 0; q < (G::TS + 127) / 128; q++) asm volatile("prefetch.global.L2 [%0];" ::"l"(zt + q * 128));
                if (RED == 1) {
                    const char* wt = static_cast<const char*>(a.w) + (size_t)k * a.s_w + otile;
#pragma unroll
                    for (int q = 0; q < (G::TS + 127) / 128; q++) asm volatile("prefetch.global.L2 [%0];" ::"l"(wt + q * 128));
                }
            }
            C acc[24];
            {
                const unsigned char* const hand = lp_smem + Q::R_H + (lp_tid() - LP_SITES) * 16;
#pragma unroll
                for (int q = 0; q < Q::HW; q++) {
                    const V d = *reinterpret_cast<const V*>(hand + q * (LP_SITES * 16));
                    if constexpr (PREC == BQ_FP64) { acc[2 * q] = d.x; acc[2 * q + 1] = d.y; }
                    else { acc[4 * q] = d.x; acc[4 * q + 1] = d.y; acc[4 * q + 2] = d.z; acc[4 * q + 3] = d.w; }
                }
            }
            if (i < nact) lp_bar_arrive(1, LP_THREADS);
            const char* cb = reinterpret_cast<const char*>(lp_smem) + Q::R_C + (j % Q::NC) * Q::CS;
            const char* hb = reinterpret_cast<const char*>(lp_smem) + Q::R_B + (j % Q::NB) * Q::BHS;
            ls_mbar_wait(ls_smem_u32(bars + j % Q::NC), (unsigned int)(j / Q::NC) & 1u);
            ls_mbar_wait(ls_smem_u32(bars + Q::NC + j % Q::NB), (unsigned int)(j / Q::NB) & 1u);
            const char *sp, *np;
            C pr, pi;
            nb_addr(tb4.x & 0xffffu, cb, hb, sp, np); weight(tb4.w, 0, 2, pr, pi);
            lp_dir<PREC, RECON, 2, true, CPLX, DAG>(acc, sp, np, u[0], nullptr, pr, pi);
            nb_addr(tb4.x >> 16, cb, hb, sp, np); weight(tb4.w, 1, 2, pr, pi);
            lp_dir<PREC, RECON, 2, false, CPLX, DAG>(acc, sp, np, u[1], nullptr, pr, pi);
            nb_addr(tb4.y & 0xffffu, cb, hb, sp, np); weight(tb4.w, 2, 3, pr, pi);
            lp_dir<PREC, RECON, 3, true, CPLX, DAG>(acc, sp, np, u[2], tw[0], pr, pi);
            nb_addr(tb4.y >> 16, cb, hb, sp, np); weight(tb4.w, 3, 3, pr, pi);
            lp_dir<PREC, RECON, 3, false, CPLX, DAG>(acc, sp, np, u[3], tw[TPACK ? 1 : 0], pr, pi);
            if (DAG) {
#pragma unroll
                for (int q = 0; q < 12; q++) {
                    const C tmp = acc[q];
                    acc[q] = acc[12 + q];
                    acc[12 + q] = tmp;
                }
            }
            C red[3] = {0, 0, 0};
            if (EPI == 1) {
                C zz[24];
                load_spinor<PREC, true>(static_cast<const char*>(a.z) + (size_t)k * a.s_z + otile, Vh, (int)(lp_tid() & 7), zz);   // h < 8: site of this tile
#pragma unroll
                for (int q = 0; q < 24; q++) acc[q] += zz[q];
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
                    load_spinor<PREC, true>(static_cast<const char*>(a.w) + (size_t)k * a.s_w + otile, Vh, (int)(lp_tid() & 7), wv);
#pragma unroll
                    for (int q = 0; q < 12; q++) {
                        red[0] = mad(wv[2 * q + 1], acc[2 * q + 1], mad(wv[2 * q], acc[2 * q], red[0]));
                        red[1] = mad(-wv[2 * q + 1], acc[2 * q], mad(wv[2 * q], acc[2 * q + 1], red[1]));
                    }
                }
            }
            store_spinor<PREC, true>(static_cast<char*>(a.out) + (size_t)k * a.s_out + otile, Vh, (int)(lp_tid() & 7), acc);
            if (RED) {
                double* sw = s_red + (j & 1) * NRED * (LP_SITES / 32);
                const int lane = lp_tid() & 31, warp = (lp_tid() - LP_SITES) >> 5;
#pragma unroll
                for (int q = 0; q < NRED; q++) {
                    const double x = warp_sum((double)red[q]);
                    if (lane == 0) sw[q * (LP_SITES / 32) + warp] = x;
                }
            }
        }
        __syncthreads();     // A is done with C(i), AH(i) and has handed right-hand side i over; B is done with C(i-1), BH(i-1)
        if (RED && i >= 1 && roleB && lp_tid() < LP_SITES + NRED) {
            const int j = i - 1, q0 = lp_tid() - LP_SITES;
            const double* sw = s_red + (j & 1) * NRED * (LP_SITES / 32) + q0 * (LP_SITES / 32);
            double v = 0;
#pragma unroll
            for (int q = 0; q < LP_SITES / 32; q++) v += sw[q];
            a.partials[((size_t)rhs_of(j) * gridDim.x + blockIdx.x) * NRED + q0] = v;
        }
        if (i + 2 < nact) fillA(i + 2);                  // C slot (i+2) % 3 = that of i - 1, AH slot that of i
        if (i >= 1 && i + 1 < nact) fillB(i + 1);        // BH slot that of i - 1
    }
}

// ---------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------
// Can this launch take the direction-split kernel?  (geometry, operand alignment, Wilson epilogue)
template <int PREC> static bool lp_eligible(const bq_lattice* lat, const HopMulti* m, const void* in, const void* z, const void* w, int cl_mode) {
    if (!m || lat->mrhs_ls < 2 || cl_mode != 0) return false;
    // Measured on 32^3 x 64 (profiles/r2_kbench.txt): in fp64, where hop_ls.cuh cannot hold the links at all, this kernel beats the
    // per-(site, rhs) kernel from 8 right-hand sides on (12: 1725 vs 1962 us; 4: 878 vs 673 us — the pipeline is nrhs + 1 steps long
    // and a CTA's link loads are not overlapped); in fp32 and half storage hop_ls.cuh is the faster one (12: 637 vs 840 us, 570 vs
    // 690 us: same arithmetic, but ~30 % more instructions per (site, rhs) — hand-off, slot decoding, two loops — and a CTA
    // barrier per step).  BQ_MRHS_LS=3 forces this kernel wherever it applies.
    if (lat->mrhs_ls == 2 && !(PREC == BQ_FP64 && m->nrhs >= 8)) return false;
    const Geom& g = lat->g;
    if (m->nrhs < 2 || m->nrhs > LS_MAX_RHS) return false;
    if (g.Lxh % 8 || g.L[1] % LS_BY || g.L[2] % LS_BZ || g.L[3] % LS_BT) return false;
    const size_t slice = (size_t)(g.Lxh / 8) * g.L[1] * g.L[2] * LsGeom<PREC>::TS;
    if (m->s_in % slice) return false;
    if (((uintptr_t)in & 15) || ((uintptr_t)z & 15) || ((uintptr_t)w & 15)) return false;
    return ls_get_encoder() != nullptr;
}

template <int PREC, int RECON, int EPI, bool CPLX, int RED, bool DAG>
static bq_status lp_launch_one(bq_lattice* lat, const LpParams<typename Prec<PREC>::comp>& P, int grid, cudaStream_t stream) {
    constexpr size_t smem = LpGeom<PREC>::TOTAL;
    // the shared-memory limit is a property of the (kernel, device) pair: remember it per device ordinal, not per process
    static bool attr_set[64] = {};
    int dev = 0;
    BQ_CUDA(lat, cudaGetDevice(&dev));
    const bool known = dev >= 0 && dev < 64;
    auto kern = hop_lsp_kernel<PREC, RECON, EPI, CPLX, RED, DAG>;
    if (!known || !attr_set[dev]) {
        BQ_CUDA(lat, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (known) attr_set[dev] = true;
    }
    kern<<<grid, LP_THREADS, smem, stream>>>(P);
    return BQ_OK;
}

template <int PREC, int RECON>
static bq_status lp_launch(bq_lattice* lat, const HopArgs<typename Prec<PREC>::comp>& a, bool cplx, int rmode, bool dag, const HopMulti* m,
                           const SolverScalars* done, cudaStream_t stream) {
    using C = typename Prec<PREC>::comp;
    using G = LsGeom<PREC>;
    const Geom& g = lat->g;
    LpParams<C> P;
    P.a = a;
    P.nxt = g.Lxh / 8; P.nyb = g.L[1] / LS_BY; P.nzb = g.L[2] / LS_BZ;
    const size_t slice = (size_t)P.nxt * g.L[1] * g.L[2] * G::TS;
    P.tk_in = (int)(m->s_in / slice);
    P.done = done;
    ls_brick(P.nyb, P.nzb, g.L[3] / LS_BT, P.gy, P.gz, P.gt);
    const int E = G::TS / (int)prec_real_bytes(PREC);
    const bool ok = ls_make_map<PREC>(&P.in_c, a.in, g, m->nrhs, P.tk_in, E, LS_BY, LS_BZ, LS_BT) &&
                    ls_make_map<PREC>(&P.in_y, a.in, g, m->nrhs, P.tk_in, E, 1, LS_BZ, LS_BT) &&
                    ls_make_map<PREC>(&P.in_z, a.in, g, m->nrhs, P.tk_in, E, LS_BY, 1, LS_BT) &&
                    ls_make_map<PREC>(&P.in_t, a.in, g, m->nrhs, P.tk_in, G::SPLIT_T ? E / 2 : E, LS_BY, LS_BZ, 1);
    if (!ok) return bq_set_error(lat, BQ_ECUDA, "bq_hop: cuTensorMapEncodeTiled failed");
    const int grid = P.nxt * P.nyb * P.nzb * (g.L[3] / LS_BT);
#define LP_GO(E_, R_)                                                                                                   \
    do {                                                                                                                \
        if (dag) return cplx ? lp_launch_one<PREC, RECON, E_, true, 0, true>(lat, P, grid, stream)                      \
                             : lp_launch_one<PREC, RECON, E_, false, 0, true>(lat, P, grid, stream);                    \
        return cplx ? lp_launch_one<PREC, RECON, E_, true, R_, false>(lat, P, grid, stream)                             \
                    : lp_launch_one<PREC, RECON, E_, false, R_, false>(lat, P, grid, stream);                           \
    } while (0)
    if (!a.z) LP_GO(0, 0);
    if (rmode == 0) LP_GO(1, 0);
    if (rmode == 1) LP_GO(1, 1);
    LP_GO(1, 2);
#undef LP_GO
}
