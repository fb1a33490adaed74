// dd.cu — opt-in domain decomposition of the Wilson hop and of its even-odd BiCGStab.
//
// The paper runs everywhere as a 4-D domain decomposition: "parallelized with MPI", one nearest-neighbour
// halo exchange per matrix application, overlapped with the bulk ("the smaller local volume is too small to hide the
// neighboring communication"), weak scaling as its experiment (Figs. 3-4).  BASELINE.json's
// north_star keeps the DEFAULT path on one GPU, so nothing here is used unless a handle is made with
// bq_lattice_create_sub.  What is built:
//   * a sub-lattice handle: local extents l_mu, a process grid g_mu and this rank's coordinates.  Fields, the gauge store and
//     every kernel work on the local volume; l_mu is even, so local and global parity agree.
//   * the hop on a sub-lattice in three parts (the split that lets transport overlap the bulk):
//       pack      per partitioned direction and side: the input spinor on the boundary slice is spin-projected to a
//                 half spinor, 12 reals per site (PAPER.md:95's message; the projection halves it).  The slice x_mu = 0
//                 goes DOWN as h = P^-_mu psi; the slice x_mu = l_mu - 1 goes UP already multiplied by the link it sits
//                 on, chi = U_mu(y)^dag P^+_mu psi(y), so no ghost links are ever needed.
//       interior  the ordinary hop kernels on the local volume; a hop that would leave the rank gets weight 0 (the
//                 per-direction weight that carries the boundary phase on one GPU), so the bulk needs no second kernel.
//       unpack    per received face: forward hops multiply the received h by the local link U_mu(x), backward hops take
//                 chi as it is; expanded to 4 spins, weighted (epilogue scale x boundary phase if the rank sits at the
//                 global boundary) and added to the output slice.  Faces run one after the other (edge sites belong to two).
//   * transport: here, "virtual ranks" — all ranks of the grid live in ONE process on ONE device and the faces move by
//     device-to-device copies (bq_dd_hop).  That is what the one-GPU test box can run and what the tests compare with the
//     plain CPU operator on the global lattice.  A process per GPU calls bq_dd_pack / bq_wilson_apply / bq_dd_unpack itself and
//     moves the face buffers with cudaMemcpyPeerAsync or NCCL send/recv (paper_2111_04457_b200/dd.py, torch.distributed);
//     that path is UNMEASURED on hardware: no multi-GPU node was available to this build.
//   * bq_dd_solve: fp64 even-odd BiCGStab over the virtual ranks; every inner product is a per-rank device reduction
//     followed by a sum over ranks on the host (the all-reduce of the real thing: 5 scalars per iteration).
// Wilson operator (csw = 0), fp64 and fp32 storage, D (not D^dagger).  Clover on sub-lattices would need ghost links for
// the field strength and is not built.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include "blas.cuh"
#include "blas_api.h"
#include "hop.cuh"

struct DdBufs {
    void* send[4][2];   // [mu][side]: side 0 = slice x_mu = 0 (goes down), 1 = slice x_mu = l_mu - 1 (goes up)
    void* recv[4][2];   // [mu][side]: side 0 = for our slice x_mu = 0 (comes from below), 1 = for our slice x_mu = l_mu - 1
    size_t cap[4];
    cudaStream_t side;  // pack + transport run here while the interior hop runs on the caller's stream
    cudaEvent_t ev_in, ev_faces;
};

void bq_dd_free(bq_lattice* lat) {
    DdBufs* d = static_cast<DdBufs*>(lat->dd);
    if (!d) return;
    for (int mu = 0; mu < 4; mu++)
        for (int s = 0; s < 2; s++) {
            if (d->send[mu][s]) cudaFree(d->send[mu][s]);
            if (d->recv[mu][s]) cudaFree(d->recv[mu][s]);
        }
    if (d->side) cudaStreamDestroy(d->side);
    if (d->ev_in) cudaEventDestroy(d->ev_in);
    if (d->ev_faces) cudaEventDestroy(d->ev_faces);
    free(d);
    lat->dd = nullptr;
}

extern "C" bq_status bq_lattice_create_sub(int lx, int ly, int lz, int lt, const double* bc_phase, const int* grid, const int* coords,
                                           bq_lattice** out) {
    if (!out || !grid || !coords) return BQ_EINVAL;
    for (int mu = 0; mu < 4; mu++)
        if (grid[mu] < 1 || coords[mu] < 0 || coords[mu] >= grid[mu]) return BQ_EINVAL;
    BQ_TRY(bq_lattice_create(lx, ly, lz, lt, bc_phase, out));
    bq_lattice* lat = *out;
    lat->sub = 1;
    for (int mu = 0; mu < 4; mu++) { lat->grid[mu] = grid[mu]; lat->coords[mu] = coords[mu]; }
    DdBufs* d = static_cast<DdBufs*>(calloc(1, sizeof(DdBufs)));
    if (!d) { bq_lattice_destroy(lat); *out = nullptr; return BQ_ENOMEM; }
    lat->dd = d;
    if (cudaStreamCreateWithFlags(&d->side, cudaStreamNonBlocking) != cudaSuccess || cudaEventCreateWithFlags(&d->ev_in, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&d->ev_faces, cudaEventDisableTiming) != cudaSuccess) {
        bq_lattice_destroy(lat);
        *out = nullptr;
        return BQ_ECUDA;
    }
    return BQ_OK;
}

static int face_sites(const Geom& g, int mu) { return g.V / g.L[mu] / 2; }   // boundary sites of ONE parity in the slice x_mu = const

extern "C" bq_status bq_dd_face_bytes(const bq_lattice* lat, int mu, bq_prec prec, size_t* bytes) {
    if (!lat || !bytes || mu < 0 || mu > 3 || (prec != BQ_FP64 && prec != BQ_FP32)) return BQ_EINVAL;
    *bytes = (size_t)face_sites(lat->g, mu) * 12 * prec_real_bytes(prec);
    return BQ_OK;
}

static bq_status dd_reserve(bq_lattice* lat, int prec) {
    DdBufs* d = static_cast<DdBufs*>(lat->dd);
    for (int mu = 0; mu < 4; mu++) {
        if (lat->grid[mu] == 1) continue;
        const size_t need = (size_t)face_sites(lat->g, mu) * 12 * sizeof(double);   // sized for fp64, reused for fp32
        (void)prec;
        if (d->cap[mu] >= need) continue;
        for (int s = 0; s < 2; s++) {
            if (d->send[mu][s]) cudaFree(d->send[mu][s]);
            if (d->recv[mu][s]) cudaFree(d->recv[mu][s]);
            d->send[mu][s] = d->recv[mu][s] = nullptr;
        }
        d->cap[mu] = 0;
        for (int s = 0; s < 2; s++) {
            BQ_CUDA(lat, cudaMalloc(&d->send[mu][s], need));
            BQ_CUDA(lat, cudaMalloc(&d->recv[mu][s], need));
        }
        d->cap[mu] = need;
    }
    return BQ_OK;
}

// face site f of parity `par` in the slice x_mu = xmu  ->  half index.  The three other coordinates are counted with the
// lowest direction fastest; of two sites that differ by one in that direction exactly one has the parity, so f = T >> 1
// (T = lexicographic index in the slice) and sender and receiver agree on f without exchanging anything.
template <int MU> __device__ __forceinline__ int face_half_index(const Geom& g, int f, int xmu, int par) {
    constexpr int D0 = MU == 0 ? 1 : 0, D1 = MU <= 1 ? 2 : 1, D2 = MU <= 2 ? 3 : 2;
    const int e0 = g.L[D0], e1 = g.L[D1];
    int x[4];
    x[MU] = xmu;
    const int c0h = f % (e0 / 2);
    const int q = f / (e0 / 2);
    x[D1] = q % e1;
    x[D2] = q / e1;
    x[D0] = 2 * c0h;
    x[D0] += (par - (x[0] + x[1] + x[2] + x[3])) & 1;
    return (x[0] >> 1) + g.Lxh * (x[1] + g.L[1] * (x[2] + g.L[2] * x[3]));
}

// pack: SIDE 0: h = P^-_mu psi on the slice x_mu = 0 (the receiver's FORWARD hop (1 - g_mu) U_mu(x) psi(x + mu));
//       SIDE 1: chi = U_mu(y)^dag P^+_mu psi(y) on the slice x_mu = l_mu - 1 (the receiver's BACKWARD hop).
// Projections as in hop.cuh: P^-+ psi = u +- i s_k l (k = x,y,z); t: (1 - g_t) keeps l, (1 + g_t) keeps u (the factor 2 is
// applied on arrival, as in hop_dir).
template <int PREC, int RECON, int MU, int SIDE>
__global__ void __launch_bounds__(128) k_dd_pack(const Geom g, int par_in, const void* __restrict__ in, const void* __restrict__ ublock,
                                                  typename Prec<PREC>::comp* __restrict__ buf, int nface) {
    using C = typename Prec<PREC>::comp;
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= nface) return;
    const int h = face_half_index<MU>(g, f, SIDE ? g.L[MU] - 1 : 0, par_in);
    C psi[24], hh[12];
    load_spinor<PREC>(in, g.Vh, h, psi);
    if (MU < 3) {
#pragma unroll
        for (int i = 0; i < 12; i++) hh[i] = psi[i];
        add_isigma<MU>(hh, psi + 12, C(SIDE ? -1 : 1));
    } else {
#pragma unroll
        for (int i = 0; i < 12; i++) hh[i] = SIDE ? psi[i] : psi[12 + i];
    }
    C* o = buf + (size_t)f * 12;
    if (SIDE) {
        C u[18], chi[12];
        load_link<PREC, RECON, true>(ublock, g.Vh, h, u);
        su3_mul<true>(u, hh, chi);
#pragma unroll
        for (int i = 0; i < 12; i++) o[i] = chi[i];
    } else {
#pragma unroll
        for (int i = 0; i < 12; i++) o[i] = hh[i];
    }
}

// unpack: SIDE 1: our slice x_mu = l_mu - 1, forward hop with the received h: chi = U_mu(x) h; SIDE 0: our slice x_mu = 0,
// backward hop, chi = the received vector.  out(x) += w * expand(chi), w = (wr, wi) = epilogue scale x boundary phase.
template <int PREC, int RECON, int MU, int SIDE>
__global__ void __launch_bounds__(128) k_dd_unpack(const Geom g, int par_out, void* __restrict__ out, const void* __restrict__ ublock,
                                                    const typename Prec<PREC>::comp* __restrict__ buf, int nface,
                                                    typename Prec<PREC>::comp wr, typename Prec<PREC>::comp wi) {
    using C = typename Prec<PREC>::comp;
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= nface) return;
    const int h = face_half_index<MU>(g, f, SIDE ? g.L[MU] - 1 : 0, par_out);
    C acc[24], hh[12], chi[12];
    load_spinor<PREC>(out, g.Vh, h, acc);
    const C* in = buf + (size_t)f * 12;
#pragma unroll
    for (int i = 0; i < 12; i++) hh[i] = in[i];
    if (SIDE) {
        C u[18];
        load_link<PREC, RECON, true>(ublock, g.Vh, h, u);
        su3_mul<false>(u, hh, chi);
    } else {
#pragma unroll
        for (int i = 0; i < 12; i++) chi[i] = hh[i];
    }
    phase_mul(chi, wr, wi);
    if (MU < 3) {
#pragma unroll
        for (int i = 0; i < 12; i++) acc[i] += chi[i];
        add_isigma<MU>(acc + 12, chi, C(SIDE ? -1 : 1));
    } else {
#pragma unroll
        for (int i = 0; i < 12; i++) acc[(SIDE ? 12 : 0) + i] += 2 * chi[i];
    }
    store_spinor<PREC>(out, g.Vh, h, acc);
}

template <int PREC, int RECON>
static bq_status dd_pack_t(bq_lattice* lat, void* const* send, const void* in, int par_in, const void* gauge, cudaStream_t s) {
    using C = typename Prec<PREC>::comp;
    const Geom& g = lat->g;
    const size_t ublk = link_block_bytes(PREC, RECON, g.Vh);
    for (int mu = 0; mu < 4; mu++) {
        if (lat->grid[mu] == 1) continue;
        const int nf = face_sites(g, mu), grid = (nf + 127) / 128;
        const void* ub = static_cast<const char*>(gauge) + ((size_t)par_in * 4 + mu) * ublk;   // links on the sending sites
        C* s0 = static_cast<C*>(send[2 * mu]);
        C* s1 = static_cast<C*>(send[2 * mu + 1]);
        switch (mu) {
            case 0: k_dd_pack<PREC, RECON, 0, 0><<<grid, 128, 0, s>>>(g, par_in, in, ub, s0, nf); k_dd_pack<PREC, RECON, 0, 1><<<grid, 128, 0, s>>>(g, par_in, in, ub, s1, nf); break;
            case 1: k_dd_pack<PREC, RECON, 1, 0><<<grid, 128, 0, s>>>(g, par_in, in, ub, s0, nf); k_dd_pack<PREC, RECON, 1, 1><<<grid, 128, 0, s>>>(g, par_in, in, ub, s1, nf); break;
            case 2: k_dd_pack<PREC, RECON, 2, 0><<<grid, 128, 0, s>>>(g, par_in, in, ub, s0, nf); k_dd_pack<PREC, RECON, 2, 1><<<grid, 128, 0, s>>>(g, par_in, in, ub, s1, nf); break;
            default: k_dd_pack<PREC, RECON, 3, 0><<<grid, 128, 0, s>>>(g, par_in, in, ub, s0, nf); k_dd_pack<PREC, RECON, 3, 1><<<grid, 128, 0, s>>>(g, par_in, in, ub, s1, nf); break;
        }
        BQ_CHECK_LAUNCH(lat);
        lat->n_launch++;
    }
    return BQ_OK;
}

template <int PREC, int RECON>
static bq_status dd_unpack_t(bq_lattice* lat, void* out, void* const* recv, double scale, int par_out, const void* gauge, cudaStream_t s) {
    using C = typename Prec<PREC>::comp;
    const Geom& g = lat->g;
    const size_t ublk = link_block_bytes(PREC, RECON, g.Vh);
    for (int mu = 0; mu < 4; mu++) {
        if (lat->grid[mu] == 1) continue;
        const int nf = face_sites(g, mu), grid = (nf + 127) / 128;
        const void* ub = static_cast<const char*>(gauge) + ((size_t)par_out * 4 + mu) * ublk;  // links on the receiving sites
        // the boundary phase multiplies the hop that crosses the GLOBAL boundary: forward on the last rank, backward (conjugate) on the first
        const bool top = lat->coords[mu] == lat->grid[mu] - 1, bottom = lat->coords[mu] == 0;
        const double fr = top ? lat->bc[2 * mu] : 1.0, fi = top ? lat->bc[2 * mu + 1] : 0.0;
        const double br = bottom ? lat->bc[2 * mu] : 1.0, bi = bottom ? -lat->bc[2 * mu + 1] : 0.0;
        const C* r0 = static_cast<const C*>(recv[2 * mu]);
        const C* r1 = static_cast<const C*>(recv[2 * mu + 1]);
#define DD_UNPACK(M)                                                                                                               \
    k_dd_unpack<PREC, RECON, M, 1><<<grid, 128, 0, s>>>(g, par_out, out, ub, r1, nf, (C)(scale * fr), (C)(scale * fi));            \
    k_dd_unpack<PREC, RECON, M, 0><<<grid, 128, 0, s>>>(g, par_out, out, ub, r0, nf, (C)(scale * br), (C)(scale * bi));
        switch (mu) {
            case 0: DD_UNPACK(0) break;
            case 1: DD_UNPACK(1) break;
            case 2: DD_UNPACK(2) break;
            default: DD_UNPACK(3) break;
        }
#undef DD_UNPACK
        BQ_CHECK_LAUNCH(lat);
        lat->n_launch++;
    }
    return BQ_OK;
}

static bq_status dd_check(bq_lattice* lat, int prec, int recon, const char* fn) {
    if (!lat) return BQ_EINVAL;
    if (!lat->sub) return bq_set_error(lat, BQ_EINVAL, "%s: not a sub-lattice handle (bq_lattice_create_sub)", fn);
    if (prec != BQ_FP64 && prec != BQ_FP32) return bq_set_error(lat, BQ_EINVAL, "%s: sub-lattices support fp64 and fp32 storage", fn);
    if (recon != BQ_RECON18 && recon != BQ_RECON12) return bq_set_error(lat, BQ_EINVAL, "%s: bad recon", fn);
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "%s: no gauge field loaded", fn);
    return BQ_OK;
}

extern "C" bq_status bq_dd_pack(bq_lattice* lat, void* const* send, const void* in, bq_parity out_parity, bq_prec prec, bq_recon recon,
                                void* stream) {
    BQ_TRY(dd_check(lat, prec, recon, "bq_dd_pack"));
    if (!send || !in || (out_parity != BQ_EVEN && out_parity != BQ_ODD)) return bq_set_error(lat, BQ_EINVAL, "bq_dd_pack: bad arguments");
    const void* gauge = nullptr;
    BQ_TRY(bq_get_gauge(lat, prec, recon, &gauge));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int par_in = 1 - (int)out_parity;
    if (prec == BQ_FP64) return recon ? dd_pack_t<BQ_FP64, BQ_RECON12>(lat, send, in, par_in, gauge, s) : dd_pack_t<BQ_FP64, BQ_RECON18>(lat, send, in, par_in, gauge, s);
    return recon ? dd_pack_t<BQ_FP32, BQ_RECON12>(lat, send, in, par_in, gauge, s) : dd_pack_t<BQ_FP32, BQ_RECON18>(lat, send, in, par_in, gauge, s);
}

extern "C" bq_status bq_dd_unpack(bq_lattice* lat, void* out, void* const* recv, double scale, bq_parity out_parity, bq_prec prec,
                                  bq_recon recon, void* stream) {
    BQ_TRY(dd_check(lat, prec, recon, "bq_dd_unpack"));
    if (!recv || !out || (out_parity != BQ_EVEN && out_parity != BQ_ODD)) return bq_set_error(lat, BQ_EINVAL, "bq_dd_unpack: bad arguments");
    const void* gauge = nullptr;
    BQ_TRY(bq_get_gauge(lat, prec, recon, &gauge));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (prec == BQ_FP64) return recon ? dd_unpack_t<BQ_FP64, BQ_RECON12>(lat, out, recv, scale, (int)out_parity, gauge, s)
                                      : dd_unpack_t<BQ_FP64, BQ_RECON18>(lat, out, recv, scale, (int)out_parity, gauge, s);
    return recon ? dd_unpack_t<BQ_FP32, BQ_RECON12>(lat, out, recv, scale, (int)out_parity, gauge, s)
                 : dd_unpack_t<BQ_FP32, BQ_RECON18>(lat, out, recv, scale, (int)out_parity, gauge, s);
}

// ---------------------------------------------------------------------------------------------------
// virtual ranks: the whole process grid in one process on one device
// ---------------------------------------------------------------------------------------------------
static int rank_of(const int* grid, const int* c) { return c[0] + grid[0] * (c[1] + grid[1] * (c[2] + grid[2] * c[3])); }

static bq_status dd_check_ranks(bq_lattice* const* ranks, int nranks, const char* fn) {
    if (!ranks || nranks < 1 || !ranks[0]) return BQ_EINVAL;
    bq_lattice* l0 = ranks[0];
    if (!l0->sub) return bq_set_error(l0, BQ_EINVAL, "%s: not sub-lattice handles", fn);
    if (l0->grid[0] * l0->grid[1] * l0->grid[2] * l0->grid[3] != nranks) return bq_set_error(l0, BQ_EINVAL, "%s: %d handles for a %dx%dx%dx%d grid", fn, nranks, l0->grid[0], l0->grid[1], l0->grid[2], l0->grid[3]);
    for (int r = 0; r < nranks; r++) {
        bq_lattice* l = ranks[r];
        if (!l || !l->sub) return bq_set_error(l0, BQ_EINVAL, "%s: handle %d is not a sub-lattice", fn, r);
        for (int mu = 0; mu < 4; mu++)
            if (l->grid[mu] != l0->grid[mu] || l->g.L[mu] != l0->g.L[mu]) return bq_set_error(l0, BQ_EINVAL, "%s: handle %d has another grid or other extents", fn, r);
        if (rank_of(l->grid, l->coords) != r) return bq_set_error(l0, BQ_EINVAL, "%s: handle %d does not sit at rank %d of the grid (x fastest)", fn, r, r);
    }
    return BQ_OK;
}

// out_r = [z_r +] scale * H_{p,1-p} in on every rank r: pack and face copies on the ranks' side streams, interior hops on
// `stream`, then the unpack of every rank behind both.
static bq_status dd_hop(bq_lattice* const* ranks, int n, void* const* out, const void* const* in, const void* const* z, double scale, int p,
                        int prec, int recon, cudaStream_t stream) {
    const int* grid = ranks[0]->grid;
    for (int r = 0; r < n; r++) {
        bq_lattice* l = ranks[r];
        DdBufs* d = static_cast<DdBufs*>(l->dd);
        BQ_TRY(dd_reserve(l, prec));
        BQ_CUDA(l, cudaEventRecord(d->ev_in, stream));            // `in` was produced on `stream`
        BQ_CUDA(l, cudaStreamWaitEvent(d->side, d->ev_in, 0));
        BQ_TRY(bq_dd_pack(l, &d->send[0][0], in[r], (bq_parity)p, (bq_prec)prec, (bq_recon)recon, d->side));
    }
    // transport.  A face packed on the slice x_mu = 0 (side 0) is the forward neighbour of the rank BELOW's last slice: it lands
    // in that rank's recv[mu][1]; a face packed on the last slice (side 1) lands in the rank ABOVE's recv[mu][0].
    for (int r = 0; r < n; r++) {
        bq_lattice* l = ranks[r];
        DdBufs* d = static_cast<DdBufs*>(l->dd);
        for (int mu = 0; mu < 4; mu++) {
            if (grid[mu] == 1) continue;
            const size_t nb = (size_t)face_sites(l->g, mu) * 12 * prec_real_bytes(prec);
            int c[4] = {l->coords[0], l->coords[1], l->coords[2], l->coords[3]};
            c[mu] = (l->coords[mu] + grid[mu] - 1) % grid[mu];
            DdBufs* below = static_cast<DdBufs*>(ranks[rank_of(grid, c)]->dd);
            c[mu] = (l->coords[mu] + 1) % grid[mu];
            DdBufs* above = static_cast<DdBufs*>(ranks[rank_of(grid, c)]->dd);
            // the receiving rank's unpack waits for ev_faces of EVERY rank, so the copies may run on the sender's side stream
            BQ_CUDA(l, cudaMemcpyAsync(below->recv[mu][1], d->send[mu][0], nb, cudaMemcpyDeviceToDevice, d->side));
            BQ_CUDA(l, cudaMemcpyAsync(above->recv[mu][0], d->send[mu][1], nb, cudaMemcpyDeviceToDevice, d->side));
        }
        BQ_CUDA(l, cudaEventRecord(d->ev_faces, d->side));
    }
    for (int r = 0; r < n; r++)      // bulk: overlaps the packing and the copies above
        BQ_TRY(bq_hop(ranks[r], out[r], in[r], z ? z[r] : nullptr, scale, p, prec, recon, nullptr, 0, stream));
    for (int r = 0; r < n; r++) BQ_CUDA(ranks[r], cudaStreamWaitEvent(stream, static_cast<DdBufs*>(ranks[r]->dd)->ev_faces, 0));
    for (int r = 0; r < n; r++) {
        DdBufs* d = static_cast<DdBufs*>(ranks[r]->dd);
        BQ_TRY(bq_dd_unpack(ranks[r], out[r], &d->recv[0][0], scale, (bq_parity)p, (bq_prec)prec, (bq_recon)recon, stream));
    }
    return BQ_OK;
}

extern "C" bq_status bq_dd_wilson_apply(bq_lattice* const* ranks, int nranks, void* const* out, const void* const* in, double kappa,
                                        bq_parity parity, bq_prec prec, bq_recon recon, void* stream) {
    BQ_TRY(dd_check_ranks(ranks, nranks, "bq_dd_wilson_apply"));
    if (!out || !in) return bq_set_error(ranks[0], BQ_EINVAL, "bq_dd_wilson_apply: NULL argument");
    for (int r = 0; r < nranks; r++) BQ_TRY(dd_check(ranks[r], prec, recon, "bq_dd_wilson_apply"));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (parity == BQ_EVEN || parity == BQ_ODD) return dd_hop(ranks, nranks, out, in, nullptr, -kappa, (int)parity, prec, recon, s);
    if (parity != BQ_FULL) return bq_set_error(ranks[0], BQ_EINVAL, "bq_dd_wilson_apply: bad parity");
    // [even | odd] buffers: out_p = in_p - kappa H_{p,1-p} in_{1-p}
    const size_t fb = field_bytes_one_parity(ranks[0]->g, prec);
    void** o = static_cast<void**>(malloc(sizeof(void*) * 4 * nranks));
    if (!o) return BQ_ENOMEM;
    const void** i1 = const_cast<const void**>(o + nranks);
    void** o1 = o + 2 * nranks;
    const void** i0 = const_cast<const void**>(o + 3 * nranks);
    for (int r = 0; r < nranks; r++) {
        o[r] = out[r]; i1[r] = static_cast<const char*>(in[r]) + fb;
        o1[r] = static_cast<char*>(out[r]) + fb; i0[r] = in[r];
    }
    bq_status st = dd_hop(ranks, nranks, o, i1, i0, -kappa, 0, prec, recon, s);
    if (st == BQ_OK) st = dd_hop(ranks, nranks, o1, i0, i1, -kappa, 1, prec, recon, s);
    free(o);
    return st;
}

// ---------------------------------------------------------------------------------------------------
// bq_dd_solve: fp64 even-odd BiCGStab over the virtual ranks (textbook van der Vorst recurrences, reading O4, as in
// solve.cu; scalars on the host because every inner product ends in a sum over ranks)
// ---------------------------------------------------------------------------------------------------
bq_status bq_solver_blas(bq_lattice* lat, BlasCtx** ctx, SolverScalars** host_mirror);   // solve.cu

namespace {
struct DdVecs {
    int n;
    size_t fb;
    void** v;     // n pointers
};
struct Cx { double re, im; };
Cx cdiv_h(Cx a, Cx b) { const double d = b.re * b.re + b.im * b.im; return Cx{(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d}; }
Cx cmul_h(Cx a, Cx b) { return Cx{a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
}  // namespace

extern "C" bq_status bq_dd_solve(bq_lattice* const* ranks, int nranks, const double* const* b, double* const* x, double kappa, double tol,
                                 int max_iter, bq_solve_info* info) {
    BQ_TRY(dd_check_ranks(ranks, nranks, "bq_dd_solve"));
    bq_lattice* l0 = ranks[0];
    if (info) { memset(info, 0, sizeof *info); info->status = BQ_EINVAL; info->true_rel_residual = NAN; }
    if (!b || !x || !(tol > 0)) return bq_set_error(l0, BQ_EINVAL, "bq_dd_solve: bad arguments");
    for (int r = 0; r < nranks; r++) BQ_TRY(dd_check(ranks[r], BQ_FP64, BQ_RECON18, "bq_dd_solve"));
    if (max_iter <= 0) max_iter = 1000;
    const int n = nranks;
    const size_t fb = field_bytes_one_parity(l0->g, BQ_FP64), nb = (size_t)l0->g.V * 24 * sizeof(double);
    // per rank: b (full), x (full), bhat, r, rhat, p, v, s, t, tmp, q (one parity each), canonical staging
    enum { B = 0, X, BHAT, R, RHAT, P, V, S, T, TMP, Q, NVEC };
    const size_t off[NVEC + 1] = {0, 2 * fb, 4 * fb, 5 * fb, 6 * fb, 7 * fb, 8 * fb, 9 * fb, 10 * fb, 11 * fb, 12 * fb, 13 * fb};
    char** pool = static_cast<char**>(calloc(n, sizeof(char*)));
    BlasCtx** bc = static_cast<BlasCtx**>(calloc(n, sizeof(BlasCtx*)));
    SolverScalars** hs = static_cast<SolverScalars**>(calloc(n, sizeof(SolverScalars*)));
    void** ptr = static_cast<void**>(calloc((size_t)n * 8, sizeof(void*)));
    bq_status st = (pool && bc && hs && ptr) ? BQ_OK : BQ_ENOMEM;
    cudaStream_t s = nullptr;
    for (int r = 0; r < n && st == BQ_OK; r++) {
        st = bq_solver_blas(ranks[r], &bc[r], &hs[r]);
        if (st == BQ_OK && cudaMalloc(&pool[r], off[NVEC] + nb) != cudaSuccess) st = bq_set_error(l0, BQ_ENOMEM, "bq_dd_solve: device allocation failed");
    }
    if (st == BQ_OK) s = bc[0]->stream;     // everything runs on rank 0's solver stream
    auto vec = [&](int r, int which) { return static_cast<void*>(pool[r] + off[which]); };
    auto odd = [&](int r, int which) { return static_cast<void*>(pool[r] + off[which] + fb); };
    void** A = ptr;            // scratch pointer lists for dd_hop
    void** Bp = ptr + n;
    void** Cp = ptr + 2 * n;
    // sums over the lattice = per-rank device reduction, then a sum over ranks on the host (the all-reduce)
    auto cdot = [&](int a, int c2, Cx* out) -> bq_status {
        for (int r = 0; r < n; r++) {
            BlasCtx c = *bc[r]; c.stream = s;
            BQ_TRY(blas_cdot(ranks[r], c, BQ_FP64, vec(r, a), vec(r, c2)));
            if (cudaMemcpyAsync(hs[r], c.sc, sizeof(SolverScalars), cudaMemcpyDeviceToHost, s) != cudaSuccess) return BQ_ECUDA;
        }
        if (cudaStreamSynchronize(s) != cudaSuccess) return bq_set_error(l0, BQ_ECUDA, "bq_dd_solve: reduction failed");
        out->re = out->im = 0;
        for (int r = 0; r < n; r++) { out->re += hs[r]->red[0]; out->im += hs[r]->red[1]; }
        return BQ_OK;
    };
    auto axpy = [&](Cx a, int xv, int yv) -> bq_status {       // y += a x
        for (int r = 0; r < n; r++) {
            BlasCtx c = *bc[r]; c.stream = s;
            BQ_TRY(blas_caxpy(ranks[r], c, BQ_FP64, a.re, a.im, vec(r, xv), vec(r, yv)));
        }
        return BQ_OK;
    };
    auto copy = [&](int dst, int src) -> bq_status {
        for (int r = 0; r < n; r++)
            if (cudaMemcpyAsync(vec(r, dst), vec(r, src), fb, cudaMemcpyDeviceToDevice, s) != cudaSuccess) return BQ_ECUDA;
        return BQ_OK;
    };
    auto hop = [&](void** o, void** i, void** zz, double scale, int p) -> bq_status {
        return dd_hop(ranks, n, o, const_cast<const void* const*>(i), const_cast<const void* const*>(zz), scale, p, BQ_FP64, BQ_RECON18, s);
    };
    // out = M^ in = in - kappa^2 H_eo H_oe in (even-site vectors; TMP is the odd intermediate)
    auto schur = [&](int o, int i) -> bq_status {
        for (int r = 0; r < n; r++) { A[r] = vec(r, TMP); Bp[r] = vec(r, i); Cp[r] = vec(r, o); }
        BQ_TRY(hop(A, Bp, nullptr, -kappa, 1));
        return hop(Cp, A, Bp, kappa, 0);
    };
    int iters = 0;
    double bnorm = 0, rel = NAN;
    bq_status result = BQ_OK;
#define DD_TRY(e) do { if (st == BQ_OK) st = (e); } while (0)
    if (st == BQ_OK) {
        // import b and x0 (local canonical fields, host or device)
        for (int r = 0; r < n && st == BQ_OK; r++) {
            double* stage = reinterpret_cast<double*>(pool[r] + off[NVEC]);
            if (cudaMemcpyAsync(stage, b[r], nb, cudaMemcpyDefault, s) != cudaSuccess) st = BQ_ECUDA;
            DD_TRY(bq_field_import(ranks[r], vec(r, B), stage, BQ_FULL, BQ_FP64, s));
            if (st == BQ_OK && cudaMemcpyAsync(stage, x[r], nb, cudaMemcpyDefault, s) != cudaSuccess) st = BQ_ECUDA;
            DD_TRY(bq_field_import(ranks[r], vec(r, X), stage, BQ_FULL, BQ_FP64, s));
        }
        // |b|^2 on the full lattice: even and odd halves are consecutive one-parity fields
        Cx d{0, 0}, e{0, 0};
        DD_TRY(cdot(B, B, &d));
        if (st == BQ_OK) {
            for (int r = 0; r < n; r++) { BlasCtx c = *bc[r]; c.stream = s; DD_TRY(blas_norm2(ranks[r], c, BQ_FP64, odd(r, B))); if (cudaMemcpyAsync(hs[r], c.sc, sizeof(SolverScalars), cudaMemcpyDeviceToHost, s) != cudaSuccess) st = BQ_ECUDA; }
            if (st == BQ_OK && cudaStreamSynchronize(s) != cudaSuccess) st = BQ_ECUDA;
            for (int r = 0; r < n; r++) e.re += hs[r]->red[0];
        }
        bnorm = sqrt(d.re + e.re);
        if (st == BQ_OK && !isfinite(bnorm)) st = bq_set_error(l0, BQ_EINVAL, "bq_dd_solve: the right-hand side contains NaN or Inf");
        if (st == BQ_OK && bnorm > 0) {
            // b^_e = b_e + kappa H_eo b_o
            for (int r = 0; r < n; r++) { A[r] = vec(r, BHAT); Bp[r] = odd(r, B); Cp[r] = vec(r, B); }
            DD_TRY(hop(A, Bp, Cp, kappa, 0));
            const double target2 = tol * tol * bnorm * bnorm;
            Cx rho{1, 0}, alpha{1, 0}, omega{1, 0};
            bool restart = true;
            while (st == BQ_OK) {
                if (restart) {
                    // r = b^_e - M^ x_e ; rhat = r ; p = v = 0
                    for (int r = 0; r < n; r++) { A[r] = vec(r, TMP); Bp[r] = vec(r, X); Cp[r] = vec(r, T); }
                    DD_TRY(hop(A, Bp, nullptr, -kappa, 1));
                    DD_TRY(hop(Cp, A, Bp, kappa, 0));
                    DD_TRY(copy(R, BHAT));
                    DD_TRY(axpy(Cx{-1, 0}, T, R));
                    DD_TRY(copy(RHAT, R));
                    for (int r = 0; r < n && st == BQ_OK; r++)
                        if (cudaMemsetAsync(vec(r, P), 0, fb, s) != cudaSuccess || cudaMemsetAsync(vec(r, V), 0, fb, s) != cudaSuccess) st = BQ_ECUDA;
                    rho = alpha = omega = Cx{1, 0};
                    Cx rr;
                    DD_TRY(cdot(R, R, &rr));
                    if (st != BQ_OK) break;
                    rel = sqrt(rr.re) / bnorm;
                    if (rr.re <= target2) break;            // true residual reached the target
                    if (iters >= max_iter) { result = bq_set_error(l0, BQ_ENOTCONVERGED, "bq_dd_solve: max_iter reached, |r|/|b| = %.3e", rel); break; }
                    restart = false;
                }
                Cx rho1, rv, ts, tt, rr;
                DD_TRY(cdot(RHAT, R, &rho1));
                if (st != BQ_OK) break;
                if (rho1.re == 0 && rho1.im == 0) { result = bq_set_error(l0, BQ_EBREAKDOWN, "bq_dd_solve: rho = 0"); break; }
                const Cx beta = cmul_h(cdiv_h(rho1, rho), cdiv_h(alpha, omega));
                rho = rho1;
                // p = r + beta (p - omega v): p -= omega v ; q = r + beta p ; p <- q
                DD_TRY(axpy(Cx{-omega.re, -omega.im}, V, P));
                DD_TRY(copy(Q, R));
                DD_TRY(axpy(beta, P, Q));
                DD_TRY(copy(P, Q));
                DD_TRY(schur(V, P));
                DD_TRY(cdot(RHAT, V, &rv));
                if (st != BQ_OK) break;
                if (rv.re == 0 && rv.im == 0) { result = bq_set_error(l0, BQ_EBREAKDOWN, "bq_dd_solve: <rhat, v> = 0"); break; }
                alpha = cdiv_h(rho, rv);
                DD_TRY(copy(S, R));
                DD_TRY(axpy(Cx{-alpha.re, -alpha.im}, V, S));
                DD_TRY(schur(T, S));
                DD_TRY(cdot(T, S, &ts));
                DD_TRY(cdot(T, T, &tt));
                if (st != BQ_OK) break;
                if (tt.re == 0) { result = bq_set_error(l0, BQ_EBREAKDOWN, "bq_dd_solve: <t, t> = 0"); break; }
                omega = Cx{ts.re / tt.re, ts.im / tt.re};
                DD_TRY(axpy(alpha, P, X));
                DD_TRY(axpy(omega, S, X));
                DD_TRY(copy(R, S));
                DD_TRY(axpy(Cx{-omega.re, -omega.im}, T, R));
                DD_TRY(cdot(R, R, &rr));
                iters++;
                if (st != BQ_OK) break;
                rel = sqrt(rr.re) / bnorm;
                if (rr.re <= target2 || iters >= max_iter) restart = true;   // confirm with the true residual (or give up there)
            }
            // x_o = b_o + kappa H_oe x_e
            for (int r = 0; r < n; r++) { A[r] = odd(r, X); Bp[r] = vec(r, X); Cp[r] = odd(r, B); }
            DD_TRY(hop(A, Bp, Cp, kappa, 1));
        } else if (st == BQ_OK) {
            for (int r = 0; r < n; r++) cudaMemsetAsync(vec(r, X), 0, 2 * fb, s);
            rel = 0;
        }
        for (int r = 0; r < n && st == BQ_OK; r++) {
            double* stage = reinterpret_cast<double*>(pool[r] + off[NVEC]);
            DD_TRY(bq_field_export(ranks[r], stage, vec(r, X), BQ_FULL, BQ_FP64, s));
            if (st == BQ_OK && cudaMemcpyAsync(x[r], stage, nb, cudaMemcpyDefault, s) != cudaSuccess) st = BQ_ECUDA;
        }
        if (st == BQ_OK && cudaStreamSynchronize(s) != cudaSuccess) st = bq_set_error(l0, BQ_ECUDA, "bq_dd_solve: %s", cudaGetErrorString(cudaGetLastError()));
    }
#undef DD_TRY
    for (int r = 0; r < n; r++)
        if (pool && pool[r]) cudaFree(pool[r]);
    free(pool); free(bc); free(hs); free(ptr);
    if (st != BQ_OK) return st;
    if (info) { info->status = result; info->inner_iters = iters; info->true_rel_residual = rel; }
    return result;
}
