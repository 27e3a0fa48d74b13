// incident.cu — ps_make_incident: incident waves in real space (PAPER.md:378-380 plane wave, "aperture=0";
// PAPER.md:404-419 focused probe, 30 mrad example; readings A12, A18 of DESIGN.md §3).
//   plane:  psi0 = 1
//   tilt:   psi0 = exp(2 pi i (m_t x/Lx + n_t y/Ly)) on a reciprocal-grid point
//   probe:  Psi0(k) = [lambda |k| <= alpha] A(k) exp(-2 pi i k.r0),  psi0 = ifft2(Psi0) scaled to sum|psi0|^2 = nx ny
// The probe's k-space fill is generated inside the column pass (no k-space array is stored).
#include <math.h>
#include <type_traits>

#include "common.cuh"
#include "fft_core.cuh"

namespace psb {

__global__ void k_fill_plane_tilt(float2* __restrict__ psi, const int nx, const int ny, const int n,
                                  const int32_t* __restrict__ tilts /* [n][2] or null */) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)n * nx * ny;
    if (i >= total) return;
    if (!tilts) { psi[i] = make_float2(1.f, 0.f); return; }
    const int ix = (int)(i % nx), iy = (int)((i / nx) % ny), p = (int)(i / ((long long)nx * ny));
    const int mt = tilts[2 * p], nt = tilts[2 * p + 1];
    const int a = (int)(((long long)mt * ix) % nx + nx) % nx, b = (int)(((long long)nt * iy) % ny + ny) % ny;
    float s, c;
    sincospif(2.0f * ((float)a / (float)nx + (float)b / (float)ny), &s, &c);
    psi[i] = make_float2(c, s);
}

template <int NY> struct PColCfg {
    static constexpr int T = Plan<NY>::T;
    static constexpr int C = (NY <= 1024) ? 8 : 4;
    static constexpr int THREADS = C * T;
    static constexpr size_t SMEM = (size_t)NY * C * sizeof(float2);
};

// column pass of the probe: generate Psi0(kx, :) and inverse-transform along y -> mixed layout
template <int NY>
__global__ void __launch_bounds__(PColCfg<NY>::THREADS)
k_probe_col(float2* __restrict__ psi, const int nx, const int32_t* __restrict__ tiles, const int n_tiles,
            const int32_t* __restrict__ pmax /* [nx] per-column limit of |n| inside probe aperture and band limit */,
            const uint32_t* __restrict__ U0 /* [n][2] fixed-point probe positions */, const float scale,
            const float2* __restrict__ abtab /* [NY][nx] exp(-i chi) or NULL */, const int n_items) {
    using Cfg = PColCfg<NY>;
    constexpr int T = Cfg::T, C = Cfg::C, SUB = kColTile / C;
    extern __shared__ float2 smem[];
    const int c = threadIdx.x % C, t = threadIdx.x / C;
    ColSlots<C> slots(smem + c, t);
    Twiddles<NY> tw;
    tw.init(t);
    const int per_wave = n_tiles * SUB;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int p = item / per_wave, rem = item % per_wave;
        const int kx = tiles[rem / SUB] * kColTile + (rem % SUB) * C + c;
        const int m = kx < nx / 2 ? kx : kx - nx;
        const int nm = pmax[kx];
        const uint32_t ux = U0[2 * p], uy = U0[2 * p + 1];
        float2 v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int iy = t + e * T;
            const int n = iy < NY / 2 ? iy : iy - NY;
            float2 z = make_float2(0.f, 0.f);
            if (abs(n) <= nm) {
                const uint32_t ph = (uint32_t)m * ux + (uint32_t)n * uy;
                float s, cc;
                sincospif((float)(ph >> 8) * (2.0f / 16777216.0f), &s, &cc);
                z = make_float2(cc * scale, -s * scale);
                if (abtab) z = cmul(z, __ldg(abtab + (size_t)iy * nx + kx));
            }
            v[e] = z;
        }
        fft_inverse<NY, ColSlots<C>, BlockSync>(v, t, tw, slots);
        float2* dst = psi + (size_t)p * NY * nx + kx;
#pragma unroll
        for (int e = 0; e < 16; ++e) dst[(size_t)(t + e * T) * nx] = v[e];
    }
}

template <int NX> struct PRowCfg {
    static constexpr int T = Plan<NX>::T;
    static constexpr int THREADS = 256;
    static constexpr int RPB = THREADS / T;
    static constexpr size_t SMEM = (size_t)RPB * RowLine<NX>::LEN * sizeof(float2);
    using Sync = typename std::conditional<(T <= 32), WarpSync, BlockSync>::type;
};

// in-place inverse row transform of the mixed array (only active column tiles hold data)
template <int NX>
__global__ void __launch_bounds__(PRowCfg<NX>::THREADS)
k_row_ifft(float2* __restrict__ psi, const uint8_t* __restrict__ tile_active, const long long n_rows,
           const int n_items) {
    using Cfg = PRowCfg<NX>;
    constexpr int T = Cfg::T;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, r = threadIdx.x / T;
    RowSlots slots{smem + (size_t)r * RowLine<NX>::LEN};
    Twiddles<NX> tw;
    tw.init(t);
    unsigned amask = 0;
#pragma unroll
    for (int e = 0; e < 16; ++e) amask |= (tile_active[(t + e * T) / kColTile] ? 1u : 0u) << e;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const long long rho = (long long)item * Cfg::RPB + r;
        const bool valid = rho < n_rows;
        float2* row = psi + (size_t)(valid ? rho : 0) * NX;
        float2 v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e)
            v[e] = (valid && ((amask >> e) & 1u)) ? row[t + e * T] : make_float2(0.f, 0.f);
        fft_inverse<NX, RowSlots, typename Cfg::Sync>(v, t, tw, slots);
        if (valid) {
#pragma unroll
            for (int e = 0; e < 16; ++e) row[t + e * T] = v[e];
        }
    }
}

template <int NY>
static cudaError_t launch_probe_col(ps_ctx* c, float2* psi, const int32_t* pmax, const uint32_t* U0, float scale,
                                    const float2* abtab, int n) {
    using Cfg = PColCfg<NY>;
    auto kern = k_probe_col<NY>;
    int cap = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &cap);
    if (ce != cudaSuccess) return ce;
    const int n_items = n * c->n_tiles_active * (kColTile / Cfg::C);
    kern<<<n_items < cap ? n_items : cap, Cfg::THREADS, Cfg::SMEM, c->stream>>>(psi, c->nx, c->d_tiles, c->n_tiles_active,
                                                                               pmax, U0, scale, abtab, n_items);
    return cudaGetLastError();
}

template <int NX>
static cudaError_t launch_row_ifft(ps_ctx* c, float2* psi, int n) {
    using Cfg = PRowCfg<NX>;
    auto kern = k_row_ifft<NX>;
    int cap = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &cap);
    if (ce != cudaSuccess) return ce;
    const long long n_rows = (long long)n * c->ny;
    const int n_items = (int)((n_rows + Cfg::RPB - 1) / Cfg::RPB);
    kern<<<n_items < cap ? n_items : cap, Cfg::THREADS, Cfg::SMEM, c->stream>>>(psi, c->d_tile_active, n_rows, n_items);
    return cudaGetLastError();
}

#define PSB_DISPATCH_N(n, CALL)                                                    \
    switch (n) {                                                                   \
        case 32: { constexpr int N_ = 32; CALL; } break;                           \
        case 64: { constexpr int N_ = 64; CALL; } break;                           \
        case 128: { constexpr int N_ = 128; CALL; } break;                         \
        case 256: { constexpr int N_ = 256; CALL; } break;                         \
        case 512: { constexpr int N_ = 512; CALL; } break;                         \
        case 1024: { constexpr int N_ = 1024; CALL; } break;                       \
        case 2048: { constexpr int N_ = 2048; CALL; } break;                       \
        default: break;                                                            \
    }

static uint32_t host_fixed(double pos, double L) {
    const double q = pos / L;
    const double u = q - floor(q);
    double U = floor(u * 4294967296.0);
    if (U > 4294967295.0) U = 4294967295.0;
    return (uint32_t)U;
}

}  // namespace psb

using namespace psb;

// ---------------------------------------------------------------- aberrations (A24)
namespace psb {

// exp(-i chi(k)) on the full grid, float64 on the host, complex64 on the device; cached per (geometry, kV, coefficients)
ps_status ensure_abtab(ps_ctx* c, double kV) {
    if (c->ab_kV == kV && c->abtab.p) return PS_OK;
    const int nx = c->nx, ny = c->ny;
    const double lam = kHC_keVA / sqrt(kV * (2.0 * kM0C2_keV + kV));
    const double* a = c->ab;
    std::vector<float2> h((size_t)nx * ny);
    for (int iy = 0; iy < ny; ++iy) {
        const double ky = signed_index(iy, ny) / c->cell[1];
        for (int ix = 0; ix < nx; ++ix) {
            const double kx = signed_index(ix, nx) / c->cell[0];
            const double th = lam * sqrt(kx * kx + ky * ky), phi = atan2(ky, kx);
            const double th2 = th * th;
            const double chi = (2.0 * M_PI / lam) * (0.5 * a[0] * th2 + 0.5 * a[1] * th2 * cos(2.0 * (phi - a[2])) +
                                                    a[3] * th2 * th / 3.0 * cos(phi - a[4]) +
                                                    a[5] * th2 * th / 3.0 * cos(3.0 * (phi - a[6])) + 0.25 * a[7] * th2 * th2);
            h[(size_t)iy * nx + ix] = make_float2((float)cos(chi), (float)(-sin(chi)));
        }
    }
    ps_status st = ensure_buf(c, c->abtab, h.size() * sizeof(float2));
    if (st != PS_OK) return st;
    if ((st = upload_async(c, c->abtab.p, h.data(), h.size() * sizeof(float2))) != PS_OK) return st;   // set-up path
    c->ab_kV = kV;
    return PS_OK;
}

__global__ void k_apply_table(float2* __restrict__ w, const float2* __restrict__ tab, const size_t npix, const size_t total) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x)
        w[i] = cmul(w[i], __ldg(tab + i % npix));
}

}  // namespace psb

extern "C" ps_status ps_set_aberrations(ps_ctx* c, const double* coef) {
    if (!c) return PS_EINVAL;
    c->have_ab = coef != nullptr;
    for (int i = 0; i < 8; ++i) {
        const double v = coef ? coef[i] : 0.0;
        if (!(v == v) || fabs(v) > 1e300) return fail(c, PS_EINVAL, "ps_set_aberrations: coefficient is not finite");
        c->ab[i] = v;
    }
    c->ab_kV = -1.0;
    return PS_OK;
}

extern "C" ps_status ps_apply_aberrations(ps_ctx* c, double kV, void* d_waves_k, long long n_waves) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_apply_aberrations: ps_set_geometry has not been called");
    if (!c->have_ab) return fail(c, PS_ESTATE, "ps_apply_aberrations: ps_set_aberrations has not been called");
    if (!d_waves_k || n_waves < 1 || !(kV > 0.0)) return fail(c, PS_EINVAL, "ps_apply_aberrations: null pointer or non-positive size / voltage");
    ps_status st = enter(c, "ps_apply_aberrations");
    if (st != PS_OK) return st;
    if ((st = ensure_abtab(c, kV)) != PS_OK) return st;
    const size_t npix = (size_t)c->nx * c->ny, total = npix * (size_t)n_waves;
    const size_t nb = (total + 255) / 256;
    ProfScope ps_(c, K_INCIDENT);
    k_apply_table<<<(unsigned)(nb < 148 * 32 ? nb : 148 * 32), 256, 0, c->stream>>>((float2*)d_waves_k, (const float2*)c->abtab.p, npix, total);
    PSB_LAUNCH_CHECK(c, "k_apply_table");
    return PS_OK;
}

extern "C" ps_status ps_make_incident(ps_ctx* c, double kV, double semi_angle_mrad, int n, const double* xy_or_tilt,
                                      int is_tilt, void* d_psi0) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_make_incident: ps_set_geometry has not been called");
    if (!d_psi0 || n < 1 || !(kV > 0.0) || semi_angle_mrad < 0.0)
        return fail(c, PS_EINVAL, "ps_make_incident: null pointer, non-positive count/voltage or negative angle");
    const int nx = c->nx, ny = c->ny;
    ps_status st0 = enter(c, "ps_make_incident");
    if (st0 != PS_OK) return st0;
    ProfScope ps_(c, K_INCIDENT);
    float2* psi = (float2*)d_psi0;
    const long long total = (long long)n * nx * ny;
    const bool probe = !is_tilt && semi_angle_mrad > 0.0;
    if ((is_tilt || probe) && !xy_or_tilt) return fail(c, PS_EINVAL, "ps_make_incident: xy_or_tilt is NULL");

    if (!probe) {
        int32_t* d_t = nullptr;
        if (is_tilt) {
            std::vector<int32_t> h(2 * (size_t)n);
            for (int i = 0; i < 2 * n; ++i) {
                const double v = xy_or_tilt[i];
                if (v != floor(v) || fabs(v) > 1e6) return fail(c, PS_EINVAL, "ps_make_incident: tilt indices must be integers");
                h[i] = (int32_t)v;
            }
            ps_status st = ensure_buf(c, c->inc_buf, h.size() * 4);
            if (st != PS_OK) return st;
            d_t = (int32_t*)c->inc_buf.p;
            if ((st = upload_async(c, d_t, h.data(), h.size() * 4)) != PS_OK) return st;   // staged: no host wait
            c->inc_pmax_host.clear();
        }
        k_fill_plane_tilt<<<(unsigned)((total + 255) / 256), 256, 0, c->stream>>>(psi, nx, ny, n, d_t);
        PSB_LAUNCH_CHECK(c, "k_fill_plane_tilt");
        return PS_OK;
    }

    // focused probe: per-column limits of the probe aperture (float64, same predicate as the definition)
    const double lam = kHC_keVA / sqrt(kV * (2.0 * kM0C2_keV + kV));
    const double alpha = semi_angle_mrad * 1.0e-3;
    std::vector<int32_t> pmax(nx, -1);
    long long n_ap = 0;
    for (int ix = 0; ix < nx; ++ix) {
        const double kx = signed_index(ix, nx) / c->cell[0];
        int best = -1;
        for (int nn = 0; nn <= c->h_nmax[ix]; ++nn) {
            const double ky = nn / c->cell[1];
            const double k2 = kx * kx + ky * ky;
            if (lam * sqrt(k2) <= alpha) best = nn; else break;
        }
        pmax[ix] = best;
        if (best >= 0) n_ap += 2 * best + 1;
    }
    if (n_ap == 0) return fail(c, PS_EINVAL, "ps_make_incident: probe aperture holds no grid point");
    std::vector<uint32_t> U0(2 * (size_t)n);
    for (int i = 0; i < n; ++i) {
        U0[2 * i] = host_fixed(xy_or_tilt[2 * i], c->cell[0]);
        U0[2 * i + 1] = host_fixed(xy_or_tilt[2 * i + 1], c->cell[1]);
    }
    const size_t pmax_bytes = ((size_t)nx * 4 + 255) & ~(size_t)255;
    const bool grown = c->inc_buf.bytes < pmax_bytes + U0.size() * 4;
    ps_status st = ensure_buf(c, c->inc_buf, pmax_bytes + U0.size() * 4);
    if (st != PS_OK) return st;
    int32_t* d_pmax = (int32_t*)c->inc_buf.p;
    uint32_t* d_U0 = (uint32_t*)((char*)c->inc_buf.p + pmax_bytes);
    // staged through the ctx's pinned ring: the host vectors may die at return and nothing waits for the stream
    if (grown || pmax != c->inc_pmax_host) {
        if ((st = upload_async(c, d_pmax, pmax.data(), (size_t)nx * 4)) != PS_OK) return st;
        c->inc_pmax_host = pmax;
    }
    if ((st = upload_async(c, d_U0, U0.data(), U0.size() * 4)) != PS_OK) return st;
    const float scale = (float)(1.0 / sqrt((double)n_ap));
    cudaError_t e = cudaErrorInvalidValue;
    const float2* abtab = nullptr;
    if (c->have_ab) {
        if ((st = ensure_abtab(c, kV)) != PS_OK) return st;
        abtab = (const float2*)c->abtab.p;
    }
    PSB_DISPATCH_N(ny, (e = launch_probe_col<N_>(c, psi, d_pmax, d_U0, scale, abtab, n)));
    if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_probe_col: ") + cudaGetErrorString(e));
    c->launches++;
    e = cudaErrorInvalidValue;
    PSB_DISPATCH_N(nx, (e = launch_row_ifft<N_>(c, psi, n)));
    if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_row_ifft: ") + cudaGetErrorString(e));
    c->launches++;
    return PS_OK;
}
