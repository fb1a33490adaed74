// hop.cu — bq_wilson_apply / bq_dirac_apply / bq_schur_apply and their multi-rhs and dagger forms, built on the hop
// launcher of hop_kernels.cuh (whose kernels are instantiated in hop_inst_*.cu, one translation unit per
// (precision, link form)).
#include "hop_kernels.cuh"

#define BQ_HOP_EXTERN(P, R)                                                                                                    \
    extern template bq_status launch_hop<P, R>(bq_lattice*, void*, const void*, const void*, double, int, const void*, const void*, \
                                               int, const HopRed*, cudaStream_t, const HopMulti*, bool);
BQ_HOP_EXTERN(BQ_FP64, BQ_RECON18)
BQ_HOP_EXTERN(BQ_FP64, BQ_RECON12)
BQ_HOP_EXTERN(BQ_FP32, BQ_RECON18)
BQ_HOP_EXTERN(BQ_FP32, BQ_RECON12)
BQ_HOP_EXTERN(BQ_HALF, BQ_RECON18)
BQ_HOP_EXTERN(BQ_HALF, BQ_RECON12)
#undef BQ_HOP_EXTERN

// cuTensorMapEncodeTiled, looked up in the driver at run time (the library does not link against libcuda)
ls_encode_fn ls_get_encoder() {
    static ls_encode_fn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<ls_encode_fn>(p);
        else
            cudaGetLastError();
    }
    return fn;
}

extern "C" bq_status bq_get_counters(const bq_lattice* lat, unsigned long long* out) {
    if (!lat || !out) return BQ_EINVAL;
    out[0] = lat->n_launch;
    for (int p = 0; p < 3; p++) out[1 + p] = lat->n_hop[p];
    out[4] = lat->n_ls;
    out[8] = lat->n_lsp;
    for (int p = 0; p < 3; p++) out[5 + p] = lat->n_hop_idle[p];
    return BQ_OK;
}

bq_status bq_hop(bq_lattice* lat, void* out, const void* in, const void* z, double scale, int p, int prec, int recon,
                 const void* cl, int cl_mode, cudaStream_t stream, const HopRed* red, const HopMulti* m, bool dag) {
    const void* gauge = nullptr;
    BQ_TRY(bq_get_gauge(lat, prec, recon, &gauge));
    if (m && m->nrhs < 1) return bq_set_error(lat, BQ_EINVAL, "bq_hop: nrhs must be >= 1");
    if (m && m->nrhs > HOP_MRHS_MAX) {
        // more right-hand sides than one CTA shape holds: equal chunks of <= HOP_MRHS_MAX, one launch each
        const int nchunk = (m->nrhs + HOP_MRHS_MAX - 1) / HOP_MRHS_MAX, per = (m->nrhs + nchunk - 1) / nchunk;
        for (int r0 = 0; r0 < m->nrhs; r0 += per) {
            HopMulti c = *m;
            c.nrhs = (m->nrhs - r0) < per ? (m->nrhs - r0) : per;
            HopRed rc;
            if (red) { rc = *red; rc.sc = red->sc + r0; if (rc.w) rc.w = static_cast<const char*>(red->w) + (size_t)r0 * m->s_w; }
            BQ_TRY(bq_hop(lat, static_cast<char*>(out) + (size_t)r0 * m->s_out, static_cast<const char*>(in) + (size_t)r0 * m->s_in,
                          z ? static_cast<const char*>(z) + (size_t)r0 * m->s_z : nullptr, scale, p, prec, recon, cl, cl_mode, stream,
                          red ? &rc : nullptr, &c, dag));
        }
        return BQ_OK;
    }
#define BQ_HOP_CASE(P, R) \
    if (prec == P && recon == R) return launch_hop<P, R>(lat, out, in, z, scale, p, gauge, cl, cl_mode, red, stream, m, dag);
    BQ_HOP_CASE(BQ_FP64, BQ_RECON18)
    BQ_HOP_CASE(BQ_FP64, BQ_RECON12)
    BQ_HOP_CASE(BQ_FP32, BQ_RECON18)
    BQ_HOP_CASE(BQ_FP32, BQ_RECON12)
    BQ_HOP_CASE(BQ_HALF, BQ_RECON18)
    BQ_HOP_CASE(BQ_HALF, BQ_RECON12)
#undef BQ_HOP_CASE
    return bq_set_error(lat, BQ_EINVAL, "bq_hop: bad prec/recon (%d, %d)", prec, recon);
}

static bool valid_prec(int p) { return p == BQ_FP64 || p == BQ_FP32 || p == BQ_HALF; }
static bool valid_recon(int r) { return r == BQ_RECON18 || r == BQ_RECON12; }

// On a sub-lattice handle with a partitioned direction the hop kernels compute the INTERIOR part only (off-rank hops get
// weight zero; the rest arrives through bq_dd_unpack).  bq_wilson_apply documents that; every other operator call would
// return a silently incomplete result, so it refuses such a handle.
static bool partitioned(const bq_lattice* lat) {
    return lat->sub && (lat->grid[0] > 1 || lat->grid[1] > 1 || lat->grid[2] > 1 || lat->grid[3] > 1);
}
#define BQ_REJECT_PARTITIONED(lat, fn)                                                                                              \
    do {                                                                                                                            \
        if (partitioned(lat))                                                                                                       \
            return bq_set_error(lat, BQ_EINVAL, fn ": a sub-lattice handle computes interior hops only; use bq_wilson_apply + bq_dd_pack / bq_dd_unpack, or bq_dd_wilson_apply"); \
    } while (0)

static bq_status dirac_apply_impl(bq_lattice* lat, void* out, const void* in, double kappa, double csw, bq_prec prec, bq_recon recon,
                                  void* stream);

extern "C" bq_status bq_wilson_apply(bq_lattice* lat, void* out, const void* in, double kappa, bq_parity parity, bq_prec prec,
                                     bq_recon recon, void* stream) {
    if (!lat) return BQ_EINVAL;
    if (!out || !in || out == in) return bq_set_error(lat, BQ_EINVAL, "bq_wilson_apply: out/in NULL or aliased");
    if (!valid_prec(prec) || !valid_recon(recon)) return bq_set_error(lat, BQ_EINVAL, "bq_wilson_apply: bad prec/recon");
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "bq_wilson_apply: no gauge field loaded");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (parity == BQ_EVEN || parity == BQ_ODD)
        return bq_hop(lat, out, in, nullptr, -kappa, (int)parity, prec, recon, nullptr, 0, s);
    if (parity != BQ_FULL) return bq_set_error(lat, BQ_EINVAL, "bq_wilson_apply: bad parity %d", (int)parity);
    return dirac_apply_impl(lat, out, in, kappa, 0.0, prec, recon, stream);   // on a sub-lattice: the interior part of D, as documented
}

extern "C" bq_status bq_dirac_apply(bq_lattice* lat, void* out, const void* in, double kappa, double csw, bq_prec prec,
                                    bq_recon recon, void* stream) {
    if (!lat) return BQ_EINVAL;
    BQ_REJECT_PARTITIONED(lat, "bq_dirac_apply");
    return dirac_apply_impl(lat, out, in, kappa, csw, prec, recon, stream);
}

static bq_status dirac_apply_impl(bq_lattice* lat, void* out, const void* in, double kappa, double csw, bq_prec prec, bq_recon recon,
                                  void* stream) {
    if (!lat) return BQ_EINVAL;
    if (!out || !in || out == in) return bq_set_error(lat, BQ_EINVAL, "bq_dirac_apply: out/in NULL or aliased");
    if (!valid_prec(prec) || !valid_recon(recon)) return bq_set_error(lat, BQ_EINVAL, "bq_dirac_apply: bad prec/recon");
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "bq_dirac_apply: no gauge field loaded");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t fb = field_bytes_one_parity(lat->g, prec);
    char* o = static_cast<char*>(out);
    const char* i = static_cast<const char*>(in);
    // out_p = A_pp in_p - kappa H_{p,1-p} in_{1-p}
    if (csw == 0.0) {
        BQ_TRY(bq_hop(lat, o, i + fb, i, -kappa, 0, prec, recon, nullptr, 0, s));
        return bq_hop(lat, o + fb, i, i + fb, -kappa, 1, prec, recon, nullptr, 0, s);
    }
    BQ_TRY(bq_clover_build(lat, csw, kappa));
    const void* cl = nullptr;
    BQ_TRY(bq_get_clover(lat, prec, 0, &cl));
    const size_t cb = (size_t)lat->g.Vh * CLOVER_REALS * prec_real_bytes(prec);
    BQ_TRY(bq_hop(lat, o, i + fb, i, -kappa, 0, prec, recon, cl, 2, s));
    return bq_hop(lat, o + fb, i, i + fb, -kappa, 1, prec, recon, static_cast<const char*>(cl) + cb, 2, s);
}

extern "C" bq_status bq_schur_apply(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw,
                                    bq_prec prec, bq_recon recon, void* stream) {
    if (!lat) return BQ_EINVAL;
    BQ_REJECT_PARTITIONED(lat, "bq_schur_apply");
    return bq_schur_red(lat, out, in, tmp, kappa, csw, prec, recon, static_cast<cudaStream_t>(stream), nullptr, 0);
}

bq_status bq_schur_red(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw, int prec, int recon,
                       cudaStream_t s, const HopRed* red, int nrhs, bool dag) {
    if (!lat) return BQ_EINVAL;
    if (!out || !in || !tmp || out == in || tmp == in || tmp == out)
        return bq_set_error(lat, BQ_EINVAL, "bq_schur_apply: NULL or aliased buffers");
    if (!valid_prec(prec) || !valid_recon(recon)) return bq_set_error(lat, BQ_EINVAL, "bq_schur_apply: bad prec/recon");
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "bq_schur_apply: no gauge field loaded");
    const size_t fb = field_bytes_one_parity(lat->g, prec);
    const HopMulti mm{nrhs, fb, fb, fb, fb};
    const HopMulti* m = nrhs >= 1 ? &mm : nullptr;
    if (csw == 0.0) {
        // tmp_o = -kappa H_oe in_e ;  out_e = in_e + kappa H_eo tmp_o = in_e - kappa^2 H_eo H_oe in_e
        // (dag: H^dag in place of H — M^^dag = 1 - kappa^2 H^dag_eo H^dag_oe)
        BQ_TRY(bq_hop(lat, tmp, in, nullptr, -kappa, 1, prec, recon, nullptr, 0, s, nullptr, m, dag));
        return bq_hop(lat, out, tmp, in, kappa, 0, prec, recon, nullptr, 0, s, red, m, dag);
    }
    BQ_TRY(bq_clover_build(lat, csw, kappa));
    const void *cl = nullptr, *cli = nullptr;
    BQ_TRY(bq_get_clover(lat, prec, 0, &cl));
    BQ_TRY(bq_get_clover(lat, prec, 1, &cli));
    const size_t cb = (size_t)lat->g.Vh * CLOVER_REALS * prec_real_bytes(prec);
    // tmp_o = -kappa A_oo^-1 H_oe in_e ;  out_e = A_ee in_e + kappa H_eo tmp_o
    // (A is Hermitian, so the dagger only turns H into H^dag)
    BQ_TRY(bq_hop(lat, tmp, in, nullptr, -kappa, 1, prec, recon, static_cast<const char*>(cli) + cb, 1, s, nullptr, m, dag));
    return bq_hop(lat, out, tmp, in, kappa, 0, prec, recon, cl, 2, s, red, m, dag);
}

// ---------------------------------------------------------------------------------------------------
// operator modes of the paper's interface, set_mode("D" | "Ddag" | "DdagD")
// ---------------------------------------------------------------------------------------------------
bq_status bq_dirac_full(bq_lattice* lat, void* out, const void* in, double kappa, double csw, int prec, int recon,
                        cudaStream_t s, bool dag) {
    const size_t fb = field_bytes_one_parity(lat->g, prec);
    char* o = static_cast<char*>(out);
    const char* i = static_cast<const char*>(in);
    // out_p = A_pp in_p - kappa H_{p,1-p} in_{1-p}   (dag: H^dag; A^dag = A)
    if (csw == 0.0) {
        BQ_TRY(bq_hop(lat, o, i + fb, i, -kappa, 0, prec, recon, nullptr, 0, s, nullptr, nullptr, dag));
        return bq_hop(lat, o + fb, i, i + fb, -kappa, 1, prec, recon, nullptr, 0, s, nullptr, nullptr, dag);
    }
    BQ_TRY(bq_clover_build(lat, csw, kappa));
    const void* cl = nullptr;
    BQ_TRY(bq_get_clover(lat, prec, 0, &cl));
    const size_t cb = (size_t)lat->g.Vh * CLOVER_REALS * prec_real_bytes(prec);
    BQ_TRY(bq_hop(lat, o, i + fb, i, -kappa, 0, prec, recon, cl, 2, s, nullptr, nullptr, dag));
    return bq_hop(lat, o + fb, i, i + fb, -kappa, 1, prec, recon, static_cast<const char*>(cl) + cb, 2, s, nullptr, nullptr, dag);
}

extern "C" bq_status bq_dirac_apply_mode(bq_lattice* lat, void* out, const void* in, void* tmp, double kappa, double csw,
                                         bq_mode mode, bq_prec prec, bq_recon recon, void* stream) {
    if (!lat) return BQ_EINVAL;
    BQ_REJECT_PARTITIONED(lat, "bq_dirac_apply_mode");
    if (!out || !in || out == in) return bq_set_error(lat, BQ_EINVAL, "bq_dirac_apply_mode: out/in NULL or aliased");
    if (!valid_prec(prec) || !valid_recon(recon)) return bq_set_error(lat, BQ_EINVAL, "bq_dirac_apply_mode: bad prec/recon");
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "bq_dirac_apply_mode: no gauge field loaded");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    switch (mode) {
        case BQ_MODE_D: return bq_dirac_full(lat, out, in, kappa, csw, prec, recon, s, false);
        case BQ_MODE_DDAG: return bq_dirac_full(lat, out, in, kappa, csw, prec, recon, s, true);
        case BQ_MODE_DDAGD:
            if (!tmp || tmp == in || tmp == out) return bq_set_error(lat, BQ_EINVAL, "bq_dirac_apply_mode: DdagD needs a distinct tmp field");
            BQ_TRY(bq_dirac_full(lat, tmp, in, kappa, csw, prec, recon, s, false));
            return bq_dirac_full(lat, out, tmp, kappa, csw, prec, recon, s, true);
    }
    return bq_set_error(lat, BQ_EINVAL, "bq_dirac_apply_mode: bad mode %d", (int)mode);
}

extern "C" bq_status bq_schur_apply_mode(bq_lattice* lat, void* out, const void* in, void* tmp, void* tmp2, double kappa, double csw,
                                         bq_mode mode, bq_prec prec, bq_recon recon, void* stream) {
    if (!lat) return BQ_EINVAL;
    BQ_REJECT_PARTITIONED(lat, "bq_schur_apply_mode");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    switch (mode) {
        case BQ_MODE_D: return bq_schur_red(lat, out, in, tmp, kappa, csw, prec, recon, s, nullptr, 0, false);
        case BQ_MODE_DDAG: return bq_schur_red(lat, out, in, tmp, kappa, csw, prec, recon, s, nullptr, 0, true);
        case BQ_MODE_DDAGD:
            if (!tmp2 || tmp2 == in || tmp2 == out || tmp2 == tmp)
                return bq_set_error(lat, BQ_EINVAL, "bq_schur_apply_mode: DdagD needs a second distinct scratch field");
            BQ_TRY(bq_schur_red(lat, tmp2, in, tmp, kappa, csw, prec, recon, s, nullptr, 0, false));
            return bq_schur_red(lat, out, tmp2, tmp, kappa, csw, prec, recon, s, nullptr, 0, true);
    }
    return bq_set_error(lat, BQ_EINVAL, "bq_schur_apply_mode: bad mode %d", (int)mode);
}

// ---------------------------------------------------------------------------------------------------
// multi-rhs entry points
// ---------------------------------------------------------------------------------------------------
extern "C" bq_status bq_wilson_apply_multi(bq_lattice* lat, void* out, const void* in, int nrhs, double kappa, bq_parity parity,
                                           bq_prec prec, bq_recon recon, void* stream) {
    if (!lat) return BQ_EINVAL;
    BQ_REJECT_PARTITIONED(lat, "bq_wilson_apply_multi");
    if (!out || !in || out == in) return bq_set_error(lat, BQ_EINVAL, "bq_wilson_apply_multi: out/in NULL or aliased");
    if (nrhs < 1) return bq_set_error(lat, BQ_EINVAL, "bq_wilson_apply_multi: nrhs must be >= 1");
    if (!valid_prec(prec) || !valid_recon(recon)) return bq_set_error(lat, BQ_EINVAL, "bq_wilson_apply_multi: bad prec/recon");
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "bq_wilson_apply_multi: no gauge field loaded");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t fb = field_bytes_one_parity(lat->g, prec);
    if (parity == BQ_EVEN || parity == BQ_ODD) {
        const HopMulti m{nrhs, fb, fb, fb, fb};
        return bq_hop(lat, out, in, nullptr, -kappa, (int)parity, prec, recon, nullptr, 0, s, nullptr, &m);
    }
    if (parity != BQ_FULL) return bq_set_error(lat, BQ_EINVAL, "bq_wilson_apply_multi: bad parity %d", (int)parity);
    // [rhs][even | odd] buffers: out_p = in_p - kappa H_{p,1-p} in_{1-p}
    const HopMulti m{nrhs, 2 * fb, 2 * fb, 2 * fb, 2 * fb};
    char* o = static_cast<char*>(out);
    const char* i = static_cast<const char*>(in);
    BQ_TRY(bq_hop(lat, o, i + fb, i, -kappa, 0, prec, recon, nullptr, 0, s, nullptr, &m));
    return bq_hop(lat, o + fb, i, i + fb, -kappa, 1, prec, recon, nullptr, 0, s, nullptr, &m);
}

extern "C" bq_status bq_schur_apply_multi(bq_lattice* lat, void* out, const void* in, void* tmp, int nrhs, double kappa, double csw,
                                          bq_prec prec, bq_recon recon, void* stream) {
    if (!lat) return BQ_EINVAL;
    BQ_REJECT_PARTITIONED(lat, "bq_schur_apply_multi");
    if (nrhs < 1) return bq_set_error(lat, BQ_EINVAL, "bq_schur_apply_multi: nrhs must be >= 1");
    return bq_schur_red(lat, out, in, tmp, kappa, csw, prec, recon, static_cast<cudaStream_t>(stream), nullptr, nrhs);
}
