// multislice.cu — the slice loop of PAPER.md:79 (§2.2):
//     psi <- psi * exp(i sigma V_s);   psi <- ifft2( P(k) A(k) fft2(psi) ),   s = 0..S-1
//     exit(k) = fft2(psi)/sqrt(nx ny)                        (exit waves kept in k-space)
// as two fused passes per slice over the wave stored in the "mixed" layout M[y][kx]:
//
//   row pass  (k_row_transmit):   M[y][:] <- FFT_x[ exp(i sigma V_s[y][:]) * IFFT_x[ M[y][:] ] ]
//   col pass  (k_col_propagate):  M[:][kx] <- IFFT_y[ Px(kx) Py(:) A(kx,:) FFT_y[ M[:][kx] ] ]
//
// Each pass reads and writes every wave element once (8 B + 8 B per pixel; the row pass also
// reads 4 B of V).  Columns kx outside the band limit are identically zero after A(k), so neither
// pass touches column tiles that lie wholly outside the aperture (pruned traffic).
// The first row pass reads the incident wave psi0 (real space) instead of M; the last column
// pass skips the inverse transform and writes the k-space exit wave for all columns.
// The propagation is done in place inside the caller's exit-wave array.
#include "common.cuh"
#include "fft_core.cuh"
#include <type_traits>

namespace psb {

// ------------------------------------------------------------------------------------ row pass
template <int NX> struct RowCfg {
    static constexpr int T = Plan<NX>::T;
    static constexpr int THREADS = (T > 256) ? T : 256;
    static constexpr int RPB = THREADS / T;                               // rows per block
    static constexpr int MIN_BLOCKS = (THREADS <= 256) ? 2 : 1;           // cap registers at 128
    static constexpr size_t SMEM = (size_t)RPB * RowLine<NX>::LEN * sizeof(float2);
    using Sync = typename std::conditional<(T <= 32), WarpSync, BlockSync>::type;
};

struct ChunkMap {           // chunk of waves: probes [p0,p0+np) x frames [f0,f0+nf); local l = lf*np + lp
    int p0, np, f0, nf, F;  // F = total frames (exit layout [P][F][ny][nx])
};

template <int NX, bool FIRST>
__global__ void __launch_bounds__(RowCfg<NX>::THREADS, RowCfg<NX>::MIN_BLOCKS)
k_row_transmit(float2* __restrict__ W, const float2* __restrict__ psi0, const float* __restrict__ V,
               const uint8_t* __restrict__ tile_active, const ChunkMap cm, const int ny, const int n_slices,
               const int slice, const float sigma, const int n_items) {
    using Cfg = RowCfg<NX>;
    constexpr int T = Cfg::T;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, r = threadIdx.x / T;
    RowSlots slots{smem + (size_t)r * RowLine<NX>::LEN};
    Twiddles<NX> tw;
    tw.init(t);
    unsigned amask = 0;                                  // bit e: column t+e*T lies in an active tile
#pragma unroll
    for (int e = 0; e < 16; ++e) amask |= (tile_active[(t + e * T) / kColTile] ? 1u : 0u) << e;
    const long long n_rows = (long long)cm.np * cm.nf * ny;

    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const long long rho = (long long)item * Cfg::RPB + r;
        const bool valid = rho < n_rows;
        int y = 0, p = 0, f = 0;
        if (valid) {
            const int l = (int)(rho / ny);
            y = (int)(rho % ny);
            p = cm.p0 + l % cm.np;
            f = cm.f0 + l / cm.np;
        }
        float2* wrow = W + (((size_t)p * cm.F + f) * ny + y) * NX;
        float2 v[16];
        float sv[16];                                    // sigma * V of this row, fetched with the wave
        {
            const float* vrow = V + (((size_t)f * n_slices + slice) * ny + y) * NX;
#pragma unroll
            for (int e = 0; e < 16; ++e) sv[e] = valid ? __ldg(vrow + t + e * T) : 0.f;
        }
        if (FIRST) {
            const float2* src = psi0 + ((size_t)p * ny + y) * NX;
#pragma unroll
            for (int e = 0; e < 16; ++e) v[e] = valid ? __ldg(src + t + e * T) : make_float2(0.f, 0.f);
        } else {
#pragma unroll
            for (int e = 0; e < 16; ++e)
                v[e] = (valid && ((amask >> e) & 1u)) ? wrow[t + e * T] : make_float2(0.f, 0.f);
            fft_inverse<NX, RowSlots, typename Cfg::Sync>(v, t, tw, slots);
        }
#pragma unroll
        for (int e = 0; e < 16; ++e) v[e] = cmul(v[e], cis_fast(sigma * sv[e]));
        fft_forward<NX, RowSlots, typename Cfg::Sync>(v, t, tw, slots);
        if (valid) {
#pragma unroll
            for (int e = 0; e < 16; ++e)
                if ((amask >> e) & 1u) wrow[t + e * T] = v[e];
        }
    }
}

// ------------------------------------------------------------------------------------ column pass
template <int NY> struct ColCfg {
    static constexpr int T = Plan<NY>::T;
    static constexpr int C = (NY <= 512) ? 16 : 8;                        // columns per block
    static constexpr int THREADS = C * T;
    static constexpr size_t SMEM = ((size_t)NY * C + NY) * sizeof(float2);
};

template <int NY, bool LAST>
__global__ void __launch_bounds__(ColCfg<NY>::THREADS)
k_col_propagate(float2* __restrict__ W, const int nx, const int32_t* __restrict__ tiles, const int n_tiles,
                const uint8_t* __restrict__ tile_active, const int32_t* __restrict__ nmax,
                const float2* __restrict__ px, const float2* __restrict__ py, const ChunkMap cm,
                const int n_items) {
    using Cfg = ColCfg<NY>;
    constexpr int T = Cfg::T, C = Cfg::C, SUB = kColTile / C;
    extern __shared__ float2 smem[];
    float2* py_s = smem + (size_t)NY * C;
    const int c = threadIdx.x % C, t = threadIdx.x / C;
    ColSlots<C> slots{smem + c};
    for (int i = threadIdx.x; i < NY; i += Cfg::THREADS) py_s[i] = py[i];
    Twiddles<NY> tw;
    tw.init(t);
    __syncthreads();
    const int per_wave = n_tiles * SUB;

    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int l = item / per_wave, rem = item % per_wave;
        const int tile = LAST ? rem / SUB : tiles[rem / SUB];
        const int kx = tile * kColTile + (rem % SUB) * C + c;
        const int p = cm.p0 + l % cm.np, f = cm.f0 + l / cm.np;
        float2* wcol = W + ((size_t)p * cm.F + f) * NY * nx + kx;
        float2 v[16];
        if (LAST && !tile_active[tile]) {                 // block-uniform: column tile outside the band limit
#pragma unroll
            for (int e = 0; e < 16; ++e) wcol[(size_t)(t + e * T) * nx] = make_float2(0.f, 0.f);
            continue;
        }
#pragma unroll
        for (int e = 0; e < 16; ++e) v[e] = wcol[(size_t)(t + e * T) * nx];
        fft_forward<NY, ColSlots<C>, BlockSync>(v, t, tw, slots);
        const int nm = nmax[kx];
        const float2 pxv = px[kx];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int iy = t + e * T;
            const int n = iy < NY / 2 ? iy : NY - iy;     // |signed index|
            v[e] = (n <= nm) ? cmul(v[e], cmul(pxv, py_s[iy])) : make_float2(0.f, 0.f);
        }
        if (!LAST) fft_inverse<NY, ColSlots<C>, BlockSync>(v, t, tw, slots);
#pragma unroll
        for (int e = 0; e < 16; ++e) wcol[(size_t)(t + e * T) * nx] = v[e];
    }
}

// ------------------------------------------------------------------------------------ launch helpers
template <class K>
static int persistent_grid(K kernel, int threads, size_t smem, int n_items) {
    int per_sm = 1;
    int dev = 0, n_sm = kNumSM;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem) != cudaSuccess || per_sm < 1)
        per_sm = 1;
    const long long cap = (long long)n_sm * per_sm;
    return (int)(n_items < cap ? n_items : cap);
}

template <int NX, bool FIRST>
static cudaError_t launch_row(ps_ctx* c, float2* W, const float2* psi0, const float* V, const ChunkMap& cm,
                              int slice, float sigma) {
    using Cfg = RowCfg<NX>;
    auto kern = k_row_transmit<NX, FIRST>;
    static bool attr_done = false;
    static int per_sm_grid = 0;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
        per_sm_grid = persistent_grid(kern, Cfg::THREADS, Cfg::SMEM, 1 << 30);
        attr_done = true;
    }
    const long long n_rows = (long long)cm.np * cm.nf * c->ny;
    const int n_items = (int)((n_rows + Cfg::RPB - 1) / Cfg::RPB);
    const int grid = n_items < per_sm_grid ? n_items : per_sm_grid;
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(W, psi0, V, c->d_tile_active, cm, c->ny, c->n_slices, slice,
                                                      sigma, n_items);
    return cudaGetLastError();
}

template <int NY, bool LAST>
static cudaError_t launch_col(ps_ctx* c, float2* W, const ChunkMap& cm) {
    using Cfg = ColCfg<NY>;
    auto kern = k_col_propagate<NY, LAST>;
    static bool attr_done = false;
    static int per_sm_grid = 0;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
        per_sm_grid = persistent_grid(kern, Cfg::THREADS, Cfg::SMEM, 1 << 30);
        attr_done = true;
    }
    const int n_tiles = LAST ? c->nx / kColTile : c->n_tiles_active;
    const int n_items = cm.np * cm.nf * n_tiles * (kColTile / Cfg::C);
    const int grid = n_items < per_sm_grid ? n_items : per_sm_grid;
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(W, c->nx, c->d_tiles, n_tiles, c->d_tile_active, c->d_nmax,
                                                      LAST ? c->kv.d_px_last : c->kv.d_px_mid, c->kv.d_py, cm, n_items);
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

}  // namespace psb

using namespace psb;

extern "C" ps_status ps_multislice(ps_ctx* c, double kV, const void* d_psi0, int n_probes, const float* d_V,
                                   int n_frames, void* d_exit, int exit_layout) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_multislice: ps_set_geometry has not been called");
    if (!d_psi0 || !d_V || !d_exit || n_probes < 1 || n_frames < 1 || !(kV > 0.0))
        return fail(c, PS_EINVAL, "ps_multislice: null pointer or non-positive size / voltage");
    if (exit_layout != PS_LAYOUT_DENSE) return fail(c, PS_EUNSUPPORTED, "ps_multislice: unknown exit layout");
    ps_status st = ensure_kv(c, kV);
    if (st != PS_OK) return st;

    const size_t wave_bytes = (size_t)c->nx * c->ny * sizeof(float2);
    int chunk = c->wave_chunk;
    if (chunk <= 0) {
        chunk = (int)((size_t)40 * 1024 * 1024 / wave_bytes);
        if (chunk < 1) chunk = 1;
    }
    const int np = n_probes < chunk ? n_probes : chunk;
    int nf = chunk / np;
    if (nf < 1) nf = 1;
    if (nf < n_frames) {                                     // equal-sized frame chunks (no short tail chunk)
        const int n_chunks = (n_frames + nf - 1) / nf;
        nf = (n_frames + n_chunks - 1) / n_chunks;
    }
    float2* W = (float2*)d_exit;
    const float2* psi0 = (const float2*)d_psi0;
    const float sigma = (float)c->kv.sigma;
    const int S = c->n_slices;

    for (int p0 = 0; p0 < n_probes; p0 += np) {
        for (int f0 = 0; f0 < n_frames; f0 += nf) {
            ChunkMap cm;
            cm.p0 = p0; cm.np = (n_probes - p0 < np) ? n_probes - p0 : np;
            cm.f0 = f0; cm.nf = (n_frames - f0 < nf) ? n_frames - f0 : nf;
            cm.F = n_frames;
            for (int s = 0; s < S; ++s) {
                cudaError_t e = cudaErrorInvalidValue;
                {
                ProfScope ps_(c, K_ROW_TRANSMIT);
                if (s == 0) { PSB_DISPATCH_N(c->nx, (e = launch_row<N_, true>(c, W, psi0, d_V, cm, s, sigma))); }
                else        { PSB_DISPATCH_N(c->nx, (e = launch_row<N_, false>(c, W, psi0, d_V, cm, s, sigma))); }
                }
                if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_row_transmit: ") + cudaGetErrorString(e));
                c->launches++;
                e = cudaErrorInvalidValue;
                {
                ProfScope ps_(c, K_COL_PROPAGATE);
                if (s == S - 1) { PSB_DISPATCH_N(c->ny, (e = launch_col<N_, true>(c, W, cm))); }
                else            { PSB_DISPATCH_N(c->ny, (e = launch_col<N_, false>(c, W, cm))); }
                }
                if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_col_propagate: ") + cudaGetErrorString(e));
                c->launches++;
            }
        }
    }
    return PS_OK;
}
