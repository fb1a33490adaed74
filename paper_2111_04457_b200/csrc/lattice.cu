// lattice.cu — handle, geometry, gauge store and field import/export (A1).
#include <math.h>
#include <stdarg.h>
#include <stdlib.h>
#include <string.h>

#include "layout.cuh"

// ---------------------------------------------------------------------------------------------------
// errors
// ---------------------------------------------------------------------------------------------------
bq_status bq_set_error(bq_lattice* lat, bq_status s, const char* fmt, ...) {
    if (lat) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(lat->err, sizeof lat->err, fmt, ap);
        va_end(ap);
    }
    return s;
}

extern "C" const char* bq_status_string(bq_status s) {
    switch (s) {
        case BQ_OK: return "ok";
        case BQ_EINVAL: return "invalid argument";
        case BQ_EODD_EXTENT: return "lattice extent odd or < 2";
        case BQ_ENOGAUGE: return "no gauge field loaded";
        case BQ_ENOCLOVER: return "no clover term";
        case BQ_ESINGULAR_CLOVER: return "clover block not positive definite";
        case BQ_ECUDA: return "CUDA error";
        case BQ_ENOMEM: return "out of device memory";
        case BQ_ENOTCONVERGED: return "solver did not converge";
        case BQ_EBREAKDOWN: return "BiCGStab breakdown";
    }
    return "unknown status";
}

extern "C" const char* bq_last_error(const bq_lattice* lat) { return lat ? lat->err : "null handle"; }

// ---------------------------------------------------------------------------------------------------
// create / destroy
// ---------------------------------------------------------------------------------------------------
extern "C" bq_status bq_lattice_create(int Lx, int Ly, int Lz, int Lt, const double* bc_phase, bq_lattice** out) {
    if (!out) return BQ_EINVAL;
    *out = nullptr;
    const int L[4] = {Lx, Ly, Lz, Lt};
    for (int mu = 0; mu < 4; mu++)
        if (L[mu] < 2 || (L[mu] & 1)) return BQ_EODD_EXTENT;
    const double vol = (double)Lx * Ly * Lz * Lt;
    if (vol >= 2147483648.0) return BQ_EINVAL;
    double bc[8] = {1, 0, 1, 0, 1, 0, -1, 0};
    if (bc_phase) {
        for (int mu = 0; mu < 4; mu++) {
            const double re = bc_phase[2 * mu], im = bc_phase[2 * mu + 1];
            if (!(fabs(re * re + im * im - 1.0) < 1e-12)) return BQ_EINVAL;
            bc[2 * mu] = re;
            bc[2 * mu + 1] = im;
        }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return BQ_ECUDA;  // no CPU fallback
    bq_lattice* lat = static_cast<bq_lattice*>(calloc(1, sizeof(bq_lattice)));
    if (!lat) return BQ_ENOMEM;
    for (int mu = 0; mu < 4; mu++) lat->g.L[mu] = L[mu];
    lat->g.Lxh = Lx / 2;
    lat->g.V = (int)vol;
    lat->g.Vh = lat->g.V / 2;
    memcpy(lat->bc, bc, sizeof bc);
    for (int mu = 0; mu < 4; mu++) lat->bc_nontrivial[mu] = !(bc[2 * mu] == 1.0 && bc[2 * mu + 1] == 0.0);
    if (cudaMalloc(&lat->d_flag, 4 * sizeof(int)) != cudaSuccess) {
        free(lat);
        return BQ_ECUDA;
    }
    {
        const char* e = getenv("BQ_MRHS_PATCH");      // A/B switch of the multi-rhs hop's thread mapping (hop_kernels.cuh)
        lat->mrhs_patch = e ? (int)strtol(e, nullptr, 0) : 1;
        const char* pdl = getenv("BQ_PDL");           // A/B switch: programmatic dependent launch of the single-rhs hop (hop_kernels.cuh)
        lat->hop_pdl = pdl ? atoi(pdl) : 262144;
        const char* ls = getenv("BQ_MRHS_LS");        // A/B switch: link-stationary multi-rhs hop (hop_ls.cuh)
        lat->mrhs_ls = ls ? atoi(ls) : 2;
        const char* sm = getenv("BQ_HOP_SMALL");      // A/B switch: uncapped-register hop kernel on small lattices (hop_kernels.cuh)
        int nsm = 148, cur = 0;                       // default: lattices whose CTAs (128 sites each) are all resident at once at 2 CTAs per SM
        if (cudaGetDevice(&cur) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, cur) != cudaSuccess) {
            cudaGetLastError();
            nsm = 148;
        }
        lat->hop_small = sm ? atoi(sm) : 2 * nsm * 128;
        const char* gph = getenv("BQ_GRAPH");         // A/B switch: CUDA-graph replay of the solver's iteration batches (solve.cu)
        lat->use_graphs = gph ? atoi(gph) : 1;
    }
    lat->err[0] = 0;
    *out = lat;
    return BQ_OK;
}

static void free_gauge(bq_lattice* lat) {
    lat->epoch++;
    for (int p = 0; p < 3; p++)
        for (int r = 0; r < 2; r++) {
            if (lat->gauge[p][r]) cudaFree(lat->gauge[p][r]);
            lat->gauge[p][r] = nullptr;
        }
    if (lat->U_canon) cudaFree(lat->U_canon);
    lat->U_canon = nullptr;
    lat->have_gauge = false;
}
static void free_clover(bq_lattice* lat) {
    lat->epoch++;
    for (int p = 0; p < 3; p++)
        for (int i = 0; i < 2; i++) {
            if (lat->clover[p][i]) cudaFree(lat->clover[p][i]);
            lat->clover[p][i] = nullptr;
        }
    lat->have_clover = false;
}

extern "C" bq_status bq_lattice_destroy(bq_lattice* lat) {
    if (!lat) return BQ_EINVAL;
    cudaDeviceSynchronize();
    free_gauge(lat);
    free_clover(lat);
    bq_solver_free(lat);
    bq_dd_free(lat);
    if (lat->d_flag) cudaFree(lat->d_flag);
    if (lat->hop_partials) cudaFree(lat->hop_partials);
    free(lat);
    return BQ_OK;
}

extern "C" bq_status bq_field_bytes(const bq_lattice* lat, bq_prec prec, bq_parity parity, size_t* bytes) {
    if (!lat || !bytes) return BQ_EINVAL;
    if (prec != BQ_FP64 && prec != BQ_FP32 && prec != BQ_HALF) return BQ_EINVAL;
    if (parity != BQ_EVEN && parity != BQ_ODD && parity != BQ_FULL) return BQ_EINVAL;
    *bytes = field_bytes_one_parity(lat->g, prec) * (parity == BQ_FULL ? 2 : 1);
    return BQ_OK;
}

// ---------------------------------------------------------------------------------------------------
// index helpers: half index h of parity p  ->  canonical site index s
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ int canonical_site(const Geom& g, int p, int h) {
    const int xh = h % g.Lxh;
    int q = h / g.Lxh;
    const int y = q % g.L[1];
    q /= g.L[1];
    const int z = q % g.L[2];
    const int t = q / g.L[2];
    const int x = 2 * xh + ((y + z + t + p) & 1);
    return x + g.L[0] * (y + g.L[1] * (z + g.L[2] * t));
}

// ---------------------------------------------------------------------------------------------------
// gauge store
// ---------------------------------------------------------------------------------------------------
// canonical U[s][mu][3][3][2] (fp64)  ->  fp64 18-real even-odd store [p][mu][link store over Vh]
__global__ void gauge_relayout_kernel(Geom g, const double* __restrict__ U, void* __restrict__ out) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;   // (p, mu, h) flattened, h fastest
    if (idx >= 8 * g.Vh) return;
    const int h = idx % g.Vh, pm = idx / g.Vh, mu = pm & 3, p = pm >> 2;
    const int s = canonical_site(g, p, h);
    const double2* src = reinterpret_cast<const double2*>(U + ((size_t)s * 4 + mu) * 18);
    double u[18];
#pragma unroll
    for (int k = 0; k < 9; k++) {
        const double2 d = src[k];
        u[2 * k] = d.x;
        u[2 * k + 1] = d.y;
    }
    store_link<BQ_FP64, BQ_RECON18>(static_cast<char*>(out) + (size_t)pm * link_block_bytes(BQ_FP64, BQ_RECON18, g.Vh), g.Vh, h, u);
}

// fp64 18-real store -> store of (PREC, RECON): plain rounding (links have entries in [-1,1]: fp16 needs no norm)
template <int PREC, int RECON>
__global__ void gauge_convert_kernel(int Vh, const void* __restrict__ src, void* __restrict__ dst) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 8 * Vh) return;
    const int h = idx % Vh, pm = idx / Vh;
    double u[18];
    load_link<BQ_FP64, BQ_RECON18>(static_cast<const char*>(src) + (size_t)pm * link_block_bytes(BQ_FP64, BQ_RECON18, Vh), Vh, h, u);
    store_link<PREC, RECON>(static_cast<char*>(dst) + (size_t)pm * link_block_bytes(PREC, RECON, Vh), Vh, h, u);
}

extern "C" bq_status bq_gauge_load(bq_lattice* lat, const double* U) {
    if (!lat) return BQ_EINVAL;
    if (!U) return bq_set_error(lat, BQ_EINVAL, "bq_gauge_load: U is NULL");
    free_gauge(lat);
    free_clover(lat);
    const Geom& g = lat->g;
    const size_t nbytes = (size_t)g.V * 72 * sizeof(double);
    BQ_CUDA(lat, cudaMalloc(&lat->U_canon, nbytes));
    BQ_CUDA(lat, cudaMemcpy(lat->U_canon, U, nbytes, cudaMemcpyDefault));   // host or device source
    BQ_CUDA(lat, cudaMalloc(&lat->gauge[BQ_FP64][BQ_RECON18], 8 * link_block_bytes(BQ_FP64, BQ_RECON18, g.Vh)));
    const int n = 8 * g.Vh;
    gauge_relayout_kernel<<<(n + 255) / 256, 256>>>(g, lat->U_canon, lat->gauge[BQ_FP64][BQ_RECON18]);
    BQ_CHECK_LAUNCH(lat);
    BQ_CUDA(lat, cudaDeviceSynchronize());
    lat->have_gauge = true;
    return BQ_OK;
}

bq_status bq_get_gauge(bq_lattice* lat, int prec, int recon, const void** out) {
    if (!lat->have_gauge) return bq_set_error(lat, BQ_ENOGAUGE, "no gauge field loaded");
    if (prec < 0 || prec > 2 || recon < 0 || recon > 1) return bq_set_error(lat, BQ_EINVAL, "bad prec/recon");
    if (!lat->gauge[prec][recon]) {
        const Geom& g = lat->g;
        void* dst = nullptr;
        BQ_CUDA(lat, cudaMalloc(&dst, 8 * link_block_bytes(prec, recon, g.Vh)));
        const void* src = lat->gauge[BQ_FP64][BQ_RECON18];
        const int n = 8 * g.Vh, grid = (n + 255) / 256;
        if (prec == BQ_FP64) gauge_convert_kernel<BQ_FP64, BQ_RECON12><<<grid, 256>>>(g.Vh, src, dst);
        else if (prec == BQ_FP32 && recon == BQ_RECON18) gauge_convert_kernel<BQ_FP32, BQ_RECON18><<<grid, 256>>>(g.Vh, src, dst);
        else if (prec == BQ_FP32) gauge_convert_kernel<BQ_FP32, BQ_RECON12><<<grid, 256>>>(g.Vh, src, dst);
        else if (recon == BQ_RECON18) gauge_convert_kernel<BQ_HALF, BQ_RECON18><<<grid, 256>>>(g.Vh, src, dst);
        else gauge_convert_kernel<BQ_HALF, BQ_RECON12><<<grid, 256>>>(g.Vh, src, dst);
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        if (e != cudaSuccess) {
            cudaFree(dst);
            return bq_set_error(lat, BQ_ECUDA, "gauge conversion failed: %s", cudaGetErrorString(e));
        }
        lat->gauge[prec][recon] = dst;
    }
    *out = lat->gauge[prec][recon];
    return BQ_OK;
}

// ---------------------------------------------------------------------------------------------------
// spinor import / export
// ---------------------------------------------------------------------------------------------------
template <int PREC>
__global__ void import_kernel(Geom g, int p, const double* __restrict__ canon, void* __restrict__ internal) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= g.Vh) return;
    const int s = canonical_site(g, p, h);
    const double2* src = reinterpret_cast<const double2*>(canon + (size_t)s * 24);
    double v[24];
#pragma unroll
    for (int k = 0; k < 12; k++) {
        const double2 d = src[k];
        v[2 * k] = d.x;
        v[2 * k + 1] = d.y;
    }
    if constexpr (PREC == BQ_FP64) {
        store_spinor<BQ_FP64>(internal, g.Vh, h, v);
    } else if constexpr (PREC == BQ_FP32) {
        float f[24];
#pragma unroll
        for (int i = 0; i < 24; i++) f[i] = (float)v[i];   // round to nearest even
        store_spinor<BQ_FP32>(internal, g.Vh, h, f);
    } else {
        // n = fp32(max|v_i|), mantissas fp16(v_i / n) with the quotient formed in fp64
        double m = 0;
#pragma unroll
        for (int i = 0; i < 24; i++) m = fmax(m, fabs(v[i]));
        const float n = (float)m;
        const double inv = n > 0.f ? 1.0 / (double)n : 0.0;
        float f[24];
#pragma unroll
        for (int i = 0; i < 24; i++) f[i] = (float)(v[i] * inv);
        using A = SpinorAddr<BQ_HALF>;
        char* b = static_cast<char*>(internal);
#pragma unroll
        for (int k = 0; k < 3; k++) *reinterpret_cast<uint4*>(b + A::word(g.Vh, h, k)) = pack8(f + 8 * k);
        *reinterpret_cast<float*>(b + A::tail(g.Vh, h)) = n;
    }
}

template <int PREC>
__global__ void export_kernel(Geom g, int p, double* __restrict__ canon, const void* __restrict__ internal) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= g.Vh) return;
    const int s = canonical_site(g, p, h);
    typename Prec<PREC>::comp v[24];
    load_spinor<PREC>(internal, g.Vh, h, v);
    double2* dst = reinterpret_cast<double2*>(canon + (size_t)s * 24);
#pragma unroll
    for (int k = 0; k < 12; k++) dst[k] = make_double2((double)v[2 * k], (double)v[2 * k + 1]);
}

template <bool IMPORT>
static bq_status import_export(bq_lattice* lat, void* internal, double* canon, bq_parity parity, bq_prec prec, void* stream) {
    if (!lat) return BQ_EINVAL;
    if (!internal || !canon) return bq_set_error(lat, BQ_EINVAL, "field import/export: NULL buffer");
    if (prec != BQ_FP64 && prec != BQ_FP32 && prec != BQ_HALF) return bq_set_error(lat, BQ_EINVAL, "bad precision");
    if (parity != BQ_EVEN && parity != BQ_ODD && parity != BQ_FULL) return bq_set_error(lat, BQ_EINVAL, "bad parity");
    const Geom& g = lat->g;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int grid = (g.Vh + 127) / 128;
    const size_t fb = field_bytes_one_parity(g, prec);
    for (int p = 0; p < 2; p++) {
        if (parity != BQ_FULL && p != (int)parity) continue;
        char* buf = static_cast<char*>(internal) + (parity == BQ_FULL ? p * fb : 0);
        if (IMPORT) {
            if (prec == BQ_FP64) import_kernel<BQ_FP64><<<grid, 128, 0, s>>>(g, p, canon, buf);
            else if (prec == BQ_FP32) import_kernel<BQ_FP32><<<grid, 128, 0, s>>>(g, p, canon, buf);
            else import_kernel<BQ_HALF><<<grid, 128, 0, s>>>(g, p, canon, buf);
        } else {
            if (prec == BQ_FP64) export_kernel<BQ_FP64><<<grid, 128, 0, s>>>(g, p, canon, buf);
            else if (prec == BQ_FP32) export_kernel<BQ_FP32><<<grid, 128, 0, s>>>(g, p, canon, buf);
            else export_kernel<BQ_HALF><<<grid, 128, 0, s>>>(g, p, canon, buf);
        }
        BQ_CHECK_LAUNCH(lat);
    }
    return BQ_OK;
}

extern "C" bq_status bq_field_import(bq_lattice* lat, void* internal, const double* canonical, bq_parity parity, bq_prec prec,
                                     void* stream) {
    return import_export<true>(lat, internal, const_cast<double*>(canonical), parity, prec, stream);
}
extern "C" bq_status bq_field_export(bq_lattice* lat, double* canonical, const void* internal, bq_parity parity, bq_prec prec,
                                     void* stream) {
    return import_export<false>(lat, const_cast<void*>(internal), canonical, parity, prec, stream);
}
