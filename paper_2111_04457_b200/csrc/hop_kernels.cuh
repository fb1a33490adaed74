// hop_kernels.cuh — the even-odd hopping kernels H_{p,1-p} and their launcher.  Included by hop.cu
// (declarations of the launcher's instantiations) and by the six hop_inst_*.cu translation units, each of which
// instantiates the launcher — and with it every kernel variant — for ONE (precision, link form), so that they compile
// in parallel.  One thread per output site; 32 consecutive half-indices per warp so every spinor-word, link-word and
// output access is a 512-byte coalesced request.  Neighbours in y,z,t are whole shifted rows (still coalesced); the x
// neighbour is the same half-index or +-1 (Appendix A.5), which the L1 serves.  Links are read exactly once
// (streaming / evict-first loads) so that L2 keeps the input spinor, each site of which is gathered by its 8
// neighbours; outputs are streamed.
#pragma once

#include "blas.cuh"
#include "clover.cuh"
#include "hop.cuh"

// Launch shape: HOP_BLOCK threads per CTA, HOP_MINB_* resident CTAs per SM asked of ptxas (register cap).
#ifndef HOP_BLOCK
#define HOP_BLOCK 128
#endif
#ifndef HOP_MINB_LO
#define HOP_MINB_LO 4   // fp32 storage
#endif
#ifndef HOP_MINB_HALF
#define HOP_MINB_HALF 4 // half storage
#endif
#ifndef HOP_MINB_64
#define HOP_MINB_64 2   // fp64
#endif
#ifndef HOP_HALF_PIPELINE
#define HOP_HALF_PIPELINE 1   // half storage: explicit load/compute software pipeline over the directions (A/B switch)
#endif

template <typename C> struct HopArgs {
    void* out;
    const void* in;
    const void* z;        // xpay operand (parity p) or nullptr
    const void* gf;       // gauge blocks of parity p   (forward links U_mu(x)),    4 blocks of `ublk` bytes
    const void* gb;       // gauge blocks of parity 1-p (backward links U_mu(x-mu))
    const void* cl;       // clover blocks of parity p (epilogue) or nullptr
    size_t ublk;          // bytes of one (parity, mu) gauge block
    int Lxh, Ly, Lz, Lt, Vh, p;
    C scale;              // epilogue scale: weight of a hop that does not wrap
    C phr[4], phi[4];     // scale x boundary phase phi_mu: weight of a hop that wraps in direction mu
    // fused reduction epilogue (RED != 0)
    const void* w;        // RED 1: left operand of <w, out>
    double* partials;     // [rhs][grid][NRED]: one partial sum per CTA (and right-hand side)
    // multi-rhs form (hop_kernel_mrhs): nrhs fields per operand, `s_*` bytes apart; T tiles of 8 sites per CTA
    int nrhs, T;
    size_t s_in, s_out, s_z, s_w;
    // patch mapping of the multi-rhs kernel (patch != 0): a CTA = 4 right-hand sides x a 2 x 2 patch of tiles in (y, z)
    int patch, nxt, ngroups;
    // solver: device-resident state(s) of the right-hand side(s); a set `done` flag (converged / broken down) turns the
    // launch (single field) or that right-hand side (multi-rhs) into a no-op, as in the BLAS-1 kernels, so that the rest of
    // a batch of iterations costs nothing once the solve is over (nullptr: always run)
    const SolverScalars* done;
};

// Grid-wide sum for the hop kernel's reduction epilogues (no clusters here: the hop grid is one CTA per 128 sites).
// Per CTA: warp shuffles -> shared memory -> one partial per CTA, stored and forgotten (no ticket, no fence: a CTA
// that waited ~2 us for an atomic's return at the end of its ~10 us life cost the memory-bound hop 15-20 %).
// A one-CTA kernel launched right behind the hop (k_hop_red_final) adds the partials — each thread a fixed strided
// subset in index order, then a fixed-order tree — and runs the finaliser.  The order of every addition is fixed,
// so the result is bitwise reproducible.
template <int NRED> __device__ __forceinline__ void hop_block_partial(const double* v, double* partials) {
    __shared__ double s_w[NRED][HOP_BLOCK / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NRED; k++) {
        const double x = warp_sum(v[k]);
        if (lane == 0) s_w[k][warp] = x;
    }
    __syncthreads();
    if (threadIdx.x < NRED) {
        double a = 0;
#pragma unroll
        for (int i = 0; i < HOP_BLOCK / 32; i++) a += s_w[threadIdx.x][i];
        partials[(size_t)blockIdx.x * NRED + threadIdx.x] = a;
    }
}

constexpr int HOP_RED_FINAL_BLOCK = 1024;
// MODE 1: NRED = 2, fin_alpha;  MODE 2: NRED = 3, fin_omega
// One CTA per right-hand side (blockIdx.x): partials [rhs][n][NRED], scalars sc[rhs].
template <int MODE> __global__ void __launch_bounds__(HOP_RED_FINAL_BLOCK) k_hop_red_final(const double* __restrict__ partials, int n,
                                                                                        SolverScalars* sc) {
    constexpr int NRED = MODE == 1 ? 2 : 3;
    partials += (size_t)blockIdx.x * n * NRED;
    sc += blockIdx.x;
    if (sc->done) return;      // the hop that feeds this reduction did not run (HopArgs::done)
    __shared__ double s_w[NRED][HOP_RED_FINAL_BLOCK / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double acc[NRED];
#pragma unroll
    for (int k = 0; k < NRED; k++) acc[k] = 0;
#pragma unroll 4
    for (int c = threadIdx.x; c < n; c += HOP_RED_FINAL_BLOCK)
#pragma unroll
        for (int k = 0; k < NRED; k++) acc[k] += partials[(size_t)c * NRED + k];
#pragma unroll
    for (int k = 0; k < NRED; k++) {
        const double x = warp_sum(acc[k]);
        if (lane == 0) s_w[k][warp] = x;
    }
    __syncthreads();
    if (warp == 0) {
        double red[NRED];
#pragma unroll
        for (int k = 0; k < NRED; k++) red[k] = warp_sum(s_w[k][lane]);
        if (lane == 0) {
            if (MODE == 1) fin_alpha(sc, red);
            else fin_omega(sc, red);
        }
    }
}

// EPI: 0: out = scale*acc;  1: out = z + scale*acc;  2: out = scale * Cl(acc);  3: out = Cl(z) + scale*acc
// (acc = H in; `scale` is carried by the per-direction weights, so acc arrives at the epilogue already scaled)
// CPLX: false = all boundary phases real (+-1), true = general complex phases (see hop_dir)
// RED: fused inner products of the BiCGStab iteration on the value just computed (before it is rounded to the
// storage precision), so that the solver needs no separate reduction pass over it:
//   0: none;  1: <w, out> -> alpha = rho / <w, out>;  2 (EPI 1, 3 only): <out, z>, <out, out> -> omega
// in / out / zp / wp: the operand fields of this thread's right-hand side; LSTREAM: see hop_dir.
template <int PREC, int RECON, int EPI, bool CPLX, int RED, bool LSTREAM = true, bool DAG = false>
__device__ __forceinline__ void hop_site(const HopArgs<typename Prec<PREC>::comp>& a, const int h, const void* in, void* out,
                                         const void* zp, const void* wp, typename Prec<PREC>::comp* red) {
    using C = typename Prec<PREC>::comp;
    const int Vh = a.Vh;
    const int xh = h % a.Lxh;
    int q = h / a.Lxh;
    const int y = q % a.Ly;
    q /= a.Ly;
    const int z = q % a.Lz;
    const int t = q / a.Lz;
    const int r = (y + z + t + a.p) & 1;   // x = 2*xh + r
    const int sy = a.Lxh, sz = a.Lxh * a.Ly, st = sz * a.Lz;
    const char* gf = static_cast<const char*>(a.gf);
    const char* gb = static_cast<const char*>(a.gb);
    const C one = a.scale, zero = 0;   // weight of an interior hop (the epilogue scale rides on the accumulation)

    C acc[24];
#pragma unroll
    for (int i = 0; i < 24; i++) acc[i] = 0;

    if constexpr (PREC == BQ_HALF && HOP_HALF_PIPELINE && LSTREAM) {
        // software pipeline over the 8 directions (hop.cuh, HalfRaw): the packed words of direction d+1 are requested
        // before direction d is computed.  Single-rhs kernels only (LSTREAM): measured -2 % (18-real) to -9 % (12-real, xpay)
        // there, +6 % in the multi-rhs kernel, which keeps the plain form (same arithmetic, bitwise equal results)
        const bool wxf = r && (xh == a.Lxh - 1), wxb = !r && (xh == 0);
        const bool wyf = (y == a.Ly - 1), wyb = (y == 0), wzf = (z == a.Lz - 1), wzb = (z == 0), wtf = (t == a.Lt - 1), wtb = (t == 0);
        const int nxf = r ? (wxf ? h - (a.Lxh - 1) : h + 1) : h;
        const int nxb = r ? h : (wxb ? h + (a.Lxh - 1) : h - 1);
        const int nyf = wyf ? h - (a.Ly - 1) * sy : h + sy, nyb = wyb ? h + (a.Ly - 1) * sy : h - sy;
        const int nzf = wzf ? h - (a.Lz - 1) * sz : h + sz, nzb = wzb ? h + (a.Lz - 1) * sz : h - sz;
        const int ntf = wtf ? h - (a.Lt - 1) * st : h + st, ntb = wtb ? h + (a.Lt - 1) * st : h - st;
        HalfRaw ra, rb;
        hop_load_half<RECON, 0, true, LSTREAM, DAG>(ra, in, Vh, nxf, gf, h);
        hop_load_half<RECON, 0, false, LSTREAM, DAG>(rb, in, Vh, nxb, gb, nxb);
        hop_compute_half<RECON, 0, true, CPLX, DAG>(acc, ra, wxf ? a.phr[0] : one, wxf ? a.phi[0] : zero);
        hop_load_half<RECON, 1, true, LSTREAM, DAG>(ra, in, Vh, nyf, gf + a.ublk, h);
        hop_compute_half<RECON, 0, false, CPLX, DAG>(acc, rb, wxb ? a.phr[0] : one, wxb ? -a.phi[0] : zero);
        hop_load_half<RECON, 1, false, LSTREAM, DAG>(rb, in, Vh, nyb, gb + a.ublk, nyb);
        hop_compute_half<RECON, 1, true, CPLX, DAG>(acc, ra, wyf ? a.phr[1] : one, wyf ? a.phi[1] : zero);
        hop_load_half<RECON, 2, true, LSTREAM, DAG>(ra, in, Vh, nzf, gf + 2 * a.ublk, h);
        hop_compute_half<RECON, 1, false, CPLX, DAG>(acc, rb, wyb ? a.phr[1] : one, wyb ? -a.phi[1] : zero);
        hop_load_half<RECON, 2, false, LSTREAM, DAG>(rb, in, Vh, nzb, gb + 2 * a.ublk, nzb);
        hop_compute_half<RECON, 2, true, CPLX, DAG>(acc, ra, wzf ? a.phr[2] : one, wzf ? a.phi[2] : zero);
        hop_load_half<RECON, 3, true, LSTREAM, DAG>(ra, in, Vh, ntf, gf + 3 * a.ublk, h);
        hop_compute_half<RECON, 2, false, CPLX, DAG>(acc, rb, wzb ? a.phr[2] : one, wzb ? -a.phi[2] : zero);
        hop_load_half<RECON, 3, false, LSTREAM, DAG>(rb, in, Vh, ntb, gb + 3 * a.ublk, ntb);
        hop_compute_half<RECON, 3, true, CPLX, DAG>(acc, ra, wtf ? a.phr[3] : one, wtf ? a.phi[3] : zero);
        hop_compute_half<RECON, 3, false, CPLX, DAG>(acc, rb, wtb ? a.phr[3] : one, wtb ? -a.phi[3] : zero);
    } else {
    // ---- x ----
    {
        const bool wf = r && (xh == a.Lxh - 1);
        const int nf = r ? (wf ? h - (a.Lxh - 1) : h + 1) : h;
        hop_dir<PREC, RECON, 0, true, CPLX, LSTREAM, DAG>(acc, in, Vh, nf, gf, h, wf ? a.phr[0] : one, wf ? a.phi[0] : zero);
        const bool wb = !r && (xh == 0);
        const int nb = r ? h : (wb ? h + (a.Lxh - 1) : h - 1);
        hop_dir<PREC, RECON, 0, false, CPLX, LSTREAM, DAG>(acc, in, Vh, nb, gb, nb, wb ? a.phr[0] : one, wb ? -a.phi[0] : zero);
    }
    // ---- y ----
    {
        const bool wf = (y == a.Ly - 1);
        const int nf = wf ? h - (a.Ly - 1) * sy : h + sy;
        hop_dir<PREC, RECON, 1, true, CPLX, LSTREAM, DAG>(acc, in, Vh, nf, gf + a.ublk, h, wf ? a.phr[1] : one, wf ? a.phi[1] : zero);
        const bool wb = (y == 0);
        const int nb = wb ? h + (a.Ly - 1) * sy : h - sy;
        hop_dir<PREC, RECON, 1, false, CPLX, LSTREAM, DAG>(acc, in, Vh, nb, gb + a.ublk, nb, wb ? a.phr[1] : one, wb ? -a.phi[1] : zero);
    }
    // ---- z ----
    {
        const bool wf = (z == a.Lz - 1);
        const int nf = wf ? h - (a.Lz - 1) * sz : h + sz;
        hop_dir<PREC, RECON, 2, true, CPLX, LSTREAM, DAG>(acc, in, Vh, nf, gf + 2 * a.ublk, h, wf ? a.phr[2] : one, wf ? a.phi[2] : zero);
        const bool wb = (z == 0);
        const int nb = wb ? h + (a.Lz - 1) * sz : h - sz;
        hop_dir<PREC, RECON, 2, false, CPLX, LSTREAM, DAG>(acc, in, Vh, nb, gb + 2 * a.ublk, nb, wb ? a.phr[2] : one, wb ? -a.phi[2] : zero);
    }
    // ---- t ----
    {
        const bool wf = (t == a.Lt - 1);
        const int nf = wf ? h - (a.Lt - 1) * st : h + st;
        hop_dir<PREC, RECON, 3, true, CPLX, LSTREAM, DAG>(acc, in, Vh, nf, gf + 3 * a.ublk, h, wf ? a.phr[3] : one, wf ? a.phi[3] : zero);
        const bool wb = (t == 0);
        const int nb = wb ? h + (a.Lt - 1) * st : h - st;
        hop_dir<PREC, RECON, 3, false, CPLX, LSTREAM, DAG>(acc, in, Vh, nb, gb + 3 * a.ublk, nb, wb ? a.phr[3] : one, wb ? -a.phi[3] : zero);
    }

    }

    if (DAG) {   // H^dag = S H S, S = exchange of the upper and lower spin pairs (hop_dir): the outer S
#pragma unroll
        for (int i = 0; i < 12; i++) {
            const C tmp = acc[i];
            acc[i] = acc[12 + i];
            acc[12 + i] = tmp;
        }
    }
    // ---- epilogue ----
    if (EPI == 2) clover_site_mul<PREC, LSTREAM>(a.cl, Vh, h, acc);   // linear: the scale already inside acc commutes with it
    if (EPI == 1 || EPI == 3) {
        C zz[24];
        load_spinor<PREC, true>(zp, Vh, h, zz);
        if (EPI == 3) {
            C az[24];
#pragma unroll
            for (int i = 0; i < 24; i++) az[i] = zz[i];
            clover_site_mul<PREC, LSTREAM>(a.cl, Vh, h, az);
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] += az[i];
        } else {
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] += zz[i];
        }
        if (RED == 2) {   // <out, z> = sum conj(out) z ;  <out, out>
#pragma unroll
            for (int k = 0; k < 12; k++) {
                red[0] = mad(acc[2 * k + 1], zz[2 * k + 1], mad(acc[2 * k], zz[2 * k], red[0]));
                red[1] = mad(-acc[2 * k + 1], zz[2 * k], mad(acc[2 * k], zz[2 * k + 1], red[1]));
                red[2] = mad(acc[2 * k + 1], acc[2 * k + 1], mad(acc[2 * k], acc[2 * k], red[2]));
            }
        }
    }
    if (RED == 1) {       // <w, out> = sum conj(w) out
        C wv[24];
        load_spinor<PREC, true>(wp, Vh, h, wv);
#pragma unroll
        for (int k = 0; k < 12; k++) {
            red[0] = mad(wv[2 * k + 1], acc[2 * k + 1], mad(wv[2 * k], acc[2 * k], red[0]));
            red[1] = mad(-wv[2 * k + 1], acc[2 * k], mad(wv[2 * k], acc[2 * k + 1], red[1]));
        }
    }
    store_spinor<PREC, true>(out, Vh, h, acc);
}

// SMALL: the same kernel compiled without a register cap, for lattices that do not fill the chip (16^4: 256 CTAs, 7 warps per SM):
// there the hop is a chain of L2 round trips, not a bandwidth matter, and with 255 registers ptxas keeps the loads of more
// directions in flight at once.  fp32 storage, real boundary phases, no dagger.  Measured (profiles/r2_small_lattice_ab.txt, A/B in one
// call, BQ_HOP_SMALL=0 vs on): 16^4: hop 7.0 -> 4.7 us (18-real), 6.2 -> 5.6 us (12-real), Schur operator 13.2 -> 9.2 us, BiCGStab
// iteration 55.2 -> 51.0 us; 16^3 x 32 (512 CTAs: two waves at the 2 CTAs per SM the uncapped build allows): 8.6 -> 9.0 us, worse — hence the
// bound Vh <= 2 x SMs x 128.  Half storage gained on the bare hop (5.4 -> 4.7 us) but lost on the whole iteration (45.1 -> 47.3 us) and keeps
// the capped build.
template <int PREC, int RECON, int EPI, bool CPLX, int RED, bool DAG = false, bool SMALL = false>
__global__ void __launch_bounds__(HOP_BLOCK, SMALL ? 1 : (PREC == BQ_FP64 ? HOP_MINB_64 : (PREC == BQ_FP32 ? HOP_MINB_LO : HOP_MINB_HALF)))
hop_kernel(const HopArgs<typename Prec<PREC>::comp> a) {
    using C = typename Prec<PREC>::comp;
    // Programmatic dependent launch (small lattices, where a hop lasts a few microseconds and the launch latency between two
    // kernels of a stream is a third of it): the NEXT kernel of the stream may be launched and scheduled now; this one waits
    // here until the kernel before it has completed and its writes are visible.  Both are no-ops in an ordinary launch.
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (a.done && a.done->done) return;     // uniform over the grid
    const int h = blockIdx.x * HOP_BLOCK + threadIdx.x;
    if (RED == 0) {
        if (h >= a.Vh) return;
        hop_site<PREC, RECON, EPI, CPLX, 0, true, DAG>(a, h, a.in, a.out, a.z, a.w, nullptr);
    } else {
        C red[3] = {0, 0, 0};
        if (h < a.Vh) hop_site<PREC, RECON, EPI, CPLX, RED, true, DAG>(a, h, a.in, a.out, a.z, a.w, red);
        const double v[3] = {(double)red[0], (double)red[1], (double)red[2]};
        hop_block_partial<RED == 1 ? 2 : 3>(v, a.partials);
    }
}

// ---------------------------------------------------------------------------------------------------
// Multi-right-hand-side hop (the paper's workload is the 12 spin-colour sources of a
// propagator on ONE gauge field).  One thread per (site, rhs); the 8 sites of a tile are the
// fastest index, then the rhs, then the tile:  thread q*8 + s8 of a CTA handles site 8*(T*blockIdx.x + q / nrhs) + s8
// of right-hand side q % nrhs.  A warp is therefore 8 sites x 4 right-hand sides: every spinor load instruction reads
// four whole 128-byte planes (one per rhs field), and every link load instruction reads ONE 128-byte plane that its
// four 8-lane groups share (identical addresses merge in the load unit).  All nrhs right-hand sides of a tile live in
// the same CTA, so a link plane is fetched from L2/DRAM once per CTA and found in L1 by the other warps: compulsory
// DRAM traffic per (site, rhs) drops from 8 links + 2 spinors to 8/nrhs links + 2 spinors (fp32/18: 768 -> 240 B at
// nrhs = 12).  Links are read with the default cache policy here (not evict-first).
// ---------------------------------------------------------------------------------------------------
constexpr int HOP_MRHS_MAX = 16;      // right-hand sides per launch (8 * nrhs * T <= 128 threads)

// partial sums of one CTA: v[k] of the threads with the same right-hand side (q % R == rl) are added and stored at
// partials[(rhs0 + rl) * nslots + slot]
template <int NRED>
__device__ __forceinline__ void hop_block_partial_mrhs(const double* v, double* partials, int R, int T, int rhs0, int nrhs, int slot,
                                                       int nslots) {
    __shared__ double s_g[NRED][HOP_BLOCK / 8];
#pragma unroll
    for (int k = 0; k < NRED; k++) {
        double x = v[k];
        x += __shfl_xor_sync(0xffffffffu, x, 4);
        x += __shfl_xor_sync(0xffffffffu, x, 2);
        x += __shfl_xor_sync(0xffffffffu, x, 1);
        if ((threadIdx.x & 7) == 0) s_g[k][threadIdx.x >> 3] = x;
    }
    __syncthreads();
    if (threadIdx.x < R * NRED) {
        const int rl = threadIdx.x / NRED, k = threadIdx.x % NRED;
        if (rhs0 + rl < nrhs) {
            double a = 0;
            for (int t = 0; t < T; t++) a += s_g[k][t * R + rl];
            partials[((size_t)(rhs0 + rl) * nslots + slot) * NRED + k] = a;
        }
    }
}

// Thread -> (site, rhs).  Plain mapping: T consecutive tiles x all nrhs right-hand sides per CTA.  Patch mapping
// (a.patch; needs tiles that are pieces of x-rows, Lxh % 8 == 0): by default 4 right-hand sides x the 2 x 2 tiles (y, y+1) x (z, z+1)
// per CTA, the CTAs of the other rhs groups of the same patch next in blockIdx (they run at the same time, so the links
// still come from HBM once and from L2 for the other groups).  Every input spinor is gathered by its 8 neighbours and L1
// only catches what a CTA's own warps share; the patch keeps half of the y and z gathers inside the SM.  Measured
// (ncu, fp32/18, 12 rhs, 32^3x64): L2 -> L1 traffic 8.5 -> 7.4 GB per launch, L1 hit rate 18 -> 27.5 %; time -3 % in
// fp32 (78.3 vs 81.0 us per rhs), -18 % in fp64 (164.6 vs 199.7), +-1 % in half.  BQ_MRHS_PATCH=0 selects the plain mapping.
#ifndef HOP_MINB_MRHS_LO
#define HOP_MINB_MRHS_LO HOP_MINB_LO       // resident CTAs per SM asked for the multi-rhs kernel, fp32 storage
#endif
#ifndef HOP_MINB_MRHS_HALF
#define HOP_MINB_MRHS_HALF HOP_MINB_HALF
#endif
#ifndef HOP_MINB_MRHS_64
#define HOP_MINB_MRHS_64 HOP_MINB_64
#endif
template <int PREC, int RECON, int EPI, bool CPLX, int RED, bool DAG = false>
__global__ void __launch_bounds__(HOP_BLOCK, PREC == BQ_FP64 ? HOP_MINB_MRHS_64 : (PREC == BQ_FP32 ? HOP_MINB_MRHS_LO : HOP_MINB_MRHS_HALF))
hop_kernel_mrhs(const HopArgs<typename Prec<PREC>::comp> a) {
    using C = typename Prec<PREC>::comp;
    const int q = threadIdx.x >> 3, s8 = threadIdx.x & 7;
    int rhs, h, R, T, rhs0, slot, nslots;
    bool live;
    if (a.patch) {
        // a.patch packs the CTA shape: log2 of (rhs per CTA, tiles in y, in z, in t), 4 bits each; their product is 16
        const int lR = a.patch & 15, ly = (a.patch >> 4) & 15, lz = (a.patch >> 8) & 15, lt = (a.patch >> 12) & 15;
        R = 1 << lR; T = 16 >> lR;
        const int rl = q & (R - 1), tl = q >> lR;
        const int dy = tl & ((1 << ly) - 1), dz = (tl >> ly) & ((1 << lz) - 1), dt = tl >> (ly + lz);
        const int g = blockIdx.x % a.ngroups;
        int pb = blockIdx.x / a.ngroups;
        slot = pb; nslots = gridDim.x / a.ngroups;
        const int xt = pb % a.nxt; pb /= a.nxt;
        const int yp = pb % (a.Ly >> ly); pb /= (a.Ly >> ly);
        const int zp = pb % (a.Lz >> lz);
        const int tp = pb / (a.Lz >> lz);
        const int tile = xt + a.nxt * (((yp << ly) + dy) + a.Ly * (((zp << lz) + dz) + a.Lz * ((tp << lt) + dt)));
        h = tile * 8 + s8;
        rhs0 = g * R; rhs = rhs0 + rl;
        live = rhs < a.nrhs;
    } else {
        R = a.nrhs; T = a.T; rhs0 = 0; slot = blockIdx.x; nslots = gridDim.x;
        rhs = q % a.nrhs;
        const int tl = q / a.nrhs;
        h = (blockIdx.x * a.T + tl) * 8 + s8;
        live = tl < a.T && h < a.Vh;     // the CTA is padded to whole warps
    }
    if (a.done && live && a.done[rhs].done) live = false;     // this right-hand side has stopped: its output is left alone
    const char* in = static_cast<const char*>(a.in) + (size_t)rhs * a.s_in;
    char* out = static_cast<char*>(a.out) + (size_t)rhs * a.s_out;
    const char* zp_ = a.z ? static_cast<const char*>(a.z) + (size_t)rhs * a.s_z : nullptr;
    const char* wp = a.w ? static_cast<const char*>(a.w) + (size_t)rhs * a.s_w : nullptr;
    if (RED == 0) {
        if (live) hop_site<PREC, RECON, EPI, CPLX, 0, false, DAG>(a, h, in, out, zp_, wp, nullptr);
    } else {
        C red[3] = {0, 0, 0};
        if (live) hop_site<PREC, RECON, EPI, CPLX, RED, false, DAG>(a, h, in, out, zp_, wp, red);
        const double v[3] = {(double)red[0], (double)red[1], (double)red[2]};
        hop_block_partial_mrhs<RED == 1 ? 2 : 3>(v, a.partials, R, T, rhs0, a.nrhs, slot, nslots);
    }
}

#include "hop_ls.cuh"
#include "hop_lsp.cuh"

// <<<grid, block, 0, stream>>> with the programmatic-stream-serialization attribute when `pdl` (see hop_kernel)
template <class K, class A> static cudaError_t hop_launch_pdl(K kern, int grid, int block, cudaStream_t stream, const A& a, bool pdl) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = 0; cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, a);
}

template <int PREC, int RECON>
bq_status launch_hop(bq_lattice* lat, void* out, const void* in, const void* z, double scale, int p, const void* gauge,
                            const void* cl, int cl_mode, const HopRed* red, cudaStream_t stream, const HopMulti* m, bool dag) {
    using C = typename Prec<PREC>::comp;
    const Geom& g = lat->g;
    HopArgs<C> a;
    a.out = out; a.in = in; a.z = z; a.cl = cl;
    a.ublk = link_block_bytes(PREC, RECON, g.Vh);
    a.gf = static_cast<const char*>(gauge) + (size_t)p * 4 * a.ublk;
    a.gb = static_cast<const char*>(gauge) + (size_t)(1 - p) * 4 * a.ublk;
    a.Lxh = g.Lxh; a.Ly = g.L[1]; a.Lz = g.L[2]; a.Lt = g.L[3]; a.Vh = g.Vh; a.p = p;
    a.scale = (C)scale;
    bool cplx = false;
    for (int mu = 0; mu < 4; mu++) {
        // sub-lattice of a process grid (dd.cu): a hop that wraps in a partitioned direction leaves the rank — weight 0 here,
        // its contribution arrives with the neighbour's face (bq_dd_unpack)
        const bool off_rank = lat->sub && lat->grid[mu] > 1;
        a.phr[mu] = off_rank ? (C)0 : (C)(scale * lat->bc[2 * mu]);
        a.phi[mu] = off_rank ? (C)0 : (C)(scale * lat->bc[2 * mu + 1]);
        if (!off_rank && lat->bc[2 * mu + 1] != 0.0) cplx = true;
    }
    // launch shape: one thread per site (128 per CTA), or — multi-rhs — T tiles x nrhs x 8 sites per CTA, padded to warps
    const bool multi = m != nullptr;
    const int nrhs = multi ? m->nrhs : 1;
    a.nrhs = nrhs;
    a.T = multi ? (HOP_BLOCK / 8 / nrhs > 0 ? HOP_BLOCK / 8 / nrhs : 1) : 0;
    a.s_in = multi ? m->s_in : 0; a.s_out = multi ? m->s_out : 0; a.s_z = multi ? m->s_z : 0; a.s_w = multi ? m->s_w : 0;
    int block = multi ? ((8 * nrhs * a.T + 31) / 32) * 32 : HOP_BLOCK;
    int grid = multi ? (g.Vh / 8 + a.T - 1) / a.T : (g.Vh + HOP_BLOCK - 1) / HOP_BLOCK;
    int nslots = grid;                    // partial sums per right-hand side of the fused reductions
    a.patch = 0; a.nxt = 0; a.ngroups = 1;
    if (multi && nrhs >= 3 && g.Lxh % 8 == 0 && lat->mrhs_patch) {
        // CTA shape (log2): rhs per CTA, tiles in y, z, t.  Default 4 rhs x 2 x 2 x 1; lat->mrhs_patch > 1 carries another
        // packed shape (env BQ_MRHS_PATCH=0xtzyR, tuning switch).  Falls back to the plain mapping if the extents do not divide.
        const int shape = lat->mrhs_patch > 1 ? lat->mrhs_patch : 0x0112;
        const int lR = shape & 15, ly = (shape >> 4) & 15, lz = (shape >> 8) & 15, lt = (shape >> 12) & 15;
        if (lR + ly + lz + lt == 4 && g.L[1] % (1 << ly) == 0 && g.L[2] % (1 << lz) == 0 && g.L[3] % (1 << lt) == 0) {
            a.patch = shape; a.nxt = g.Lxh / 8; a.ngroups = (nrhs + (1 << lR) - 1) >> lR;
            nslots = g.Vh / 8 / (16 >> lR);            // patches
            grid = nslots * a.ngroups;
            block = HOP_BLOCK;
        }
    }
    const int rmode = red ? red->mode : 0;
    const bool pdl = !multi && lat->hop_pdl && g.Vh <= lat->hop_pdl;     // programmatic dependent launch on small lattices
    const bool small = !multi && PREC == BQ_FP32 && g.Vh <= lat->hop_small;
    a.done = lat->hop_done;
    // link-stationary kernel (hop_ls.cuh) where the geometry, the operand strides and the epilogue allow
    // direction-split pipelined form of it (hop_lsp.cuh; Wilson epilogues, all precisions) first, then the one-thread-per-site form
    const bool use_lp = multi && !(dag && rmode) && lp_eligible<PREC>(lat, m, in, z, rmode == 1 ? red->w : nullptr, cl_mode);
    const bool use_ls = !use_lp && multi && !(dag && rmode) && ls_eligible<PREC>(lat, m, in, z, rmode == 1 ? red->w : nullptr, cl_mode);
    if (use_ls || use_lp) nslots = (g.Lxh / 8) * (g.L[1] / LS_BY) * (g.L[2] / LS_BZ) * (g.L[3] / LS_BT);
    a.w = nullptr; a.partials = nullptr;
    if (rmode) {
        if ((rmode != 1 && rmode != 2) || !red->sc || (rmode == 1 && !red->w) || !z)
            return bq_set_error(lat, BQ_EINVAL, "bq_hop: bad fused reduction (mode %d)", rmode);
        const size_t need = (size_t)3 * nslots * nrhs;
        if (lat->hop_partials_cap < need) {
            if (lat->hop_partials) BQ_CUDA(lat, cudaFree(lat->hop_partials));
            lat->hop_partials = nullptr; lat->hop_partials_cap = 0;
            lat->epoch++;     // cached solver graphs hold the old address
            BQ_CUDA(lat, cudaMalloc(&lat->hop_partials, sizeof(double) * need));
            lat->hop_partials_cap = need;
        }
        a.w = red->w; a.partials = lat->hop_partials;
    }
    int epi;
    if (cl_mode == 0) epi = z ? 1 : 0;
    else if (cl_mode == 1 && !z) epi = 2;
    else if (cl_mode == 2 && z) epi = 3;
    else return bq_set_error(lat, BQ_EINVAL, "bq_hop: unsupported epilogue (cl_mode=%d, z=%p)", cl_mode, z);
    // the dagger hop exists without fused reductions (the CG of the normal equations reduces on the plain hop)
    if (dag && rmode) return bq_set_error(lat, BQ_EINVAL, "bq_hop: the dagger hop has no fused reduction");
    if (use_ls || use_lp) {
        bool launched = false;
        if (use_lp) {
            BQ_TRY((lp_launch<PREC, RECON>(lat, a, cplx, rmode, dag, m, lat->hop_done, stream)));
            lat->n_lsp++;
            launched = true;
        } else if constexpr (PREC != BQ_FP64) {
            BQ_TRY((ls_launch<PREC, RECON>(lat, a, cplx, rmode, dag, m, lat->hop_done, stream, cl_mode)));
            launched = true;
        }
        if (launched) {
            BQ_CHECK_LAUNCH(lat);
            lat->n_hop[PREC] += nrhs;
            lat->n_ls++;
            if (rmode) {
                if (rmode == 1) k_hop_red_final<1><<<nrhs, HOP_RED_FINAL_BLOCK, 0, stream>>>(lat->hop_partials, nslots, red->sc);
                else k_hop_red_final<2><<<nrhs, HOP_RED_FINAL_BLOCK, 0, stream>>>(lat->hop_partials, nslots, red->sc);
                BQ_CHECK_LAUNCH(lat);
            }
            return BQ_OK;
        }
    }
#define BQ_HOP_LAUNCH_DAG(E)                                                                        \
    do {                                                                                            \
        if (multi) {                                                                                \
            if (cplx) hop_kernel_mrhs<PREC, RECON, E, true, 0, true><<<grid, block, 0, stream>>>(a);  \
            else hop_kernel_mrhs<PREC, RECON, E, false, 0, true><<<grid, block, 0, stream>>>(a);      \
        } else {                                                                                    \
            if (cplx) lerr = hop_launch_pdl(hop_kernel<PREC, RECON, E, true, 0, true>, grid, HOP_BLOCK, stream, a, pdl);   \
            else lerr = hop_launch_pdl(hop_kernel<PREC, RECON, E, false, 0, true>, grid, HOP_BLOCK, stream, a, pdl);       \
        }                                                                                           \
    } while (0)
#define BQ_HOP_LAUNCH(E, R)                                                                         \
    do {                                                                                            \
        if (multi) {                                                                                \
            if (cplx) hop_kernel_mrhs<PREC, RECON, E, true, R><<<grid, block, 0, stream>>>(a);       \
            else hop_kernel_mrhs<PREC, RECON, E, false, R><<<grid, block, 0, stream>>>(a);           \
        } else {                                                                                    \
            if (cplx) lerr = hop_launch_pdl(hop_kernel<PREC, RECON, E, true, R>, grid, HOP_BLOCK, stream, a, pdl);        \
            else if (small) lerr = hop_launch_pdl(hop_kernel<PREC, RECON, E, false, R, false, PREC == BQ_FP32>, grid, HOP_BLOCK, stream, a, pdl); \
            else lerr = hop_launch_pdl(hop_kernel<PREC, RECON, E, false, R>, grid, HOP_BLOCK, stream, a, pdl);            \
        }                                                                                           \
    } while (0)
    cudaError_t lerr = cudaSuccess;   // status of cudaLaunchKernelEx (the <<<>>> launches report through cudaGetLastError below)
    // fused reductions exist for the xpay epilogues only (the second hop of M^, which produces v and t)
    if (dag) {
        switch (epi) {
            case 0: BQ_HOP_LAUNCH_DAG(0); break;
            case 1: BQ_HOP_LAUNCH_DAG(1); break;
            case 2: BQ_HOP_LAUNCH_DAG(2); break;
            default: BQ_HOP_LAUNCH_DAG(3); break;
        }
    } else
    switch (epi * 3 + rmode) {
        case 0: BQ_HOP_LAUNCH(0, 0); break;
        case 3: BQ_HOP_LAUNCH(1, 0); break;
        case 4: BQ_HOP_LAUNCH(1, 1); break;
        case 5: BQ_HOP_LAUNCH(1, 2); break;
        case 6: BQ_HOP_LAUNCH(2, 0); break;
        case 9: BQ_HOP_LAUNCH(3, 0); break;
        case 10: BQ_HOP_LAUNCH(3, 1); break;
        case 11: BQ_HOP_LAUNCH(3, 2); break;
        default: return bq_set_error(lat, BQ_EINVAL, "bq_hop: epilogue %d has no fused reduction %d", epi, rmode);
    }
#undef BQ_HOP_LAUNCH
#undef BQ_HOP_LAUNCH_DAG
    BQ_CUDA(lat, lerr);
    BQ_CHECK_LAUNCH(lat);
    lat->n_hop[PREC] += nrhs;     // counted per right-hand side: each is 1320 flop x Vh sites
    if (rmode) {
        if (rmode == 1) k_hop_red_final<1><<<nrhs, HOP_RED_FINAL_BLOCK, 0, stream>>>(lat->hop_partials, nslots, red->sc);
        else k_hop_red_final<2><<<nrhs, HOP_RED_FINAL_BLOCK, 0, stream>>>(lat->hop_partials, nslots, red->sc);
        BQ_CHECK_LAUNCH(lat);
    }
    return BQ_OK;
}

