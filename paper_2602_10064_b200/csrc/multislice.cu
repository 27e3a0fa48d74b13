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
#include "tma.cuh"
#include <type_traits>

namespace psb {

// ------------------------------------------------------------------------------------ row pass
template <int NX> struct RowCfg {
    static constexpr int T = Plan<NX>::T;
    static constexpr int THREADS = (T > 256) ? T : 256;
    static constexpr int RPB = THREADS / T;                               // rows per block
    static constexpr int MIN_BLOCKS = (THREADS <= 256) ? 2 : 1;           // cap registers at 128
    static constexpr size_t SMEM = (size_t)RPB * RowLine<NX>::LEN * sizeof(float2);
    // rows are independent: only the T threads of a row synchronise (a warp, or a named barrier per row)
    using Sync = typename std::conditional<(T <= 32), WarpSync,
                                           typename std::conditional<(RPB > 1), GroupSync<T>, BlockSync>::type>::type;
};

struct ChunkMap {           // chunk of waves: probes [p0,p0+np) x frames [f0,f0+nf); local l = lf*np + lp
    int p0, np, f0, nf, F;  // F = total frames (exit layout [P][F][ny][nx])
};

template <int NX, bool FIRST>
__global__ void __launch_bounds__(RowCfg<NX>::THREADS, RowCfg<NX>::MIN_BLOCKS)
k_row_transmit(float2* __restrict__ W, const float2* __restrict__ psi0, const float* __restrict__ V,
               const uint8_t* __restrict__ tile_active, const ChunkMap cm, const int ny, const int n_slices,
               const int slice, const float sigma, const int n_items, const int col_lo, const int col_hi,
               const int vacuum_shortcut) {
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
    // 32-bit index arithmetic (ps_multislice checks n_probes * n_frames * ny < 2^31; ny is a power of two):
    // 64-bit divisions here cost about a tenth of the kernel's instructions
    const unsigned n_rows = (unsigned)cm.np * (unsigned)cm.nf * (unsigned)ny;
    const int ny_shift = __ffs(ny) - 1;
    const unsigned np_u = (unsigned)cm.np;

    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const unsigned rho = (unsigned)item * Cfg::RPB + r;
        const bool valid = rho < n_rows;
        int y = 0, p = 0, f = 0;
        if (valid) {
            const unsigned l = rho >> ny_shift;
            y = (int)(rho & (unsigned)(ny - 1));
            const unsigned lf = (np_u == 1u) ? l : l / np_u;
            p = cm.p0 + (int)(l - lf * np_u);
            f = cm.f0 + (int)lf;
        }
        if (NX >= 512 && t == 0) {                           // this block's next row: HBM -> L2 while this one is transformed
                                                             // (measured: +3 % at 512^2, +4 % at 2048^2, -4 % at 256^2)
            const unsigned rn = rho + gridDim.x * Cfg::RPB;
            if (rn < n_rows) {
                const unsigned ln = rn >> ny_shift;
                const int yn = (int)(rn & (unsigned)(ny - 1));
                const unsigned lfn = (np_u == 1u) ? ln : ln / np_u;
                const int pn = cm.p0 + (int)(ln - lfn * np_u), fn = cm.f0 + (int)lfn;
                tma::bulk_prefetch_l2(V + (((size_t)fn * n_slices + slice) * ny + yn) * NX, NX * sizeof(float));
                if (!FIRST) {
                    const float2* wn = W + (((size_t)pn * cm.F + fn) * ny + yn) * NX;
                    if (col_lo > 0) tma::bulk_prefetch_l2(wn, col_lo * sizeof(float2));
                    if (col_hi < NX) tma::bulk_prefetch_l2(wn + col_hi, (NX - col_hi) * sizeof(float2));
                }
            }
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
            if (vacuum_shortcut) {
                // V == 0 on the whole row (vacuum): exp(i sigma V) = 1 and FFT_x[IFFT_x[M]] = NX * M exactly, so the
                // row is only rescaled (NX is a power of two: no rounding).  Decided per warp (T <= 32: the rows this
                // warp carries) or per block, from the potential itself: any input with vacuum rows benefits.
                bool z = true;
#pragma unroll
                for (int e = 0; e < 16; ++e) z = z && (sv[e] == 0.f);
                const bool all_z = (T <= 32) ? (bool)__all_sync(0xffffffffu, z) : (bool)__syncthreads_and(z);
                if (all_z) {
                    if (valid) {
#pragma unroll
                        for (int e = 0; e < 16; ++e)
                            if ((amask >> e) & 1u) wrow[t + e * T] = make_float2(v[e].x * (float)NX, v[e].y * (float)NX);
                    }
                    continue;
                }
            }
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
// A block owns C adjacent k-columns x all NY rows of one wave per item.  The tile travels
// global -> shared -> global through the TMA engine (2-D tensor map over the wave array viewed as
// float32 [P*F*ny][2 nx]); the ring of NS shared-memory stages is, in turn, TMA destination, FFT
// exchange buffer and TMA store source, so the load of item i+1 and the store of item i-1 overlap the
// transforms of item i and no register is spent on staging.
template <int NY> struct ColCfg {
    static constexpr int T = Plan<NY>::T;
    static constexpr int C = (NY <= 1024) ? 8 : 4;   // columns per block
    static constexpr int THREADS = C * T;
    static constexpr int NS = 3;                                          // pipeline stages
    static constexpr int BOX_R = (NY < 256) ? NY : 256;                   // TMA box rows (<= 256)
    static constexpr int NBOX = NY / BOX_R;
    static constexpr int MIN_BLOCKS = (THREADS <= 256) ? 2 : 1;           // cap registers at 128
    static constexpr uint32_t STAGE_BYTES = (uint32_t)NY * C * sizeof(float2);
    static constexpr size_t SMEM = (size_t)NS * STAGE_BYTES + (size_t)NY * sizeof(float2) + NS * sizeof(uint64_t) + 128;
};

template <int NY, bool LAST>
__global__ void __launch_bounds__(ColCfg<NY>::THREADS, ColCfg<NY>::MIN_BLOCKS)
k_col_propagate(const __grid_constant__ CUtensorMap wmap, const int tiles_lo, const int tile_gap, const int n_tiles,
                const int32_t* __restrict__ nmax, const float2* __restrict__ px, const float2* __restrict__ py,
                const ChunkMap cm, const int n_items) {
    using Cfg = ColCfg<NY>;
    constexpr int T = Cfg::T, C = Cfg::C, SUB = kColTile / C, NS = Cfg::NS, PF = NS - 2;   // prefetch distance
    extern __shared__ __align__(1024) float2 smem_col[];      // no static shared memory: the window starts aligned
    float2* stage0 = smem_col;
    float2* py_s = smem_col + (size_t)NS * NY * C;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_col + (size_t)NS * NY * C + NY);
    const int c = threadIdx.x % C, t = threadIdx.x / C;
    const int per_wave = n_tiles * SUB;

    auto issue_load = [&](const int item, const int s) {      // one thread: arm the barrier, launch the boxes
        const int l = item / per_wave, rem = item % per_wave;
        const int tj = rem / SUB;                             // active tiles: [0, tiles_lo) and [tiles_lo + gap, ..)
        const int kx0 = (tj < tiles_lo ? tj : tj + tile_gap) * kColTile + (rem % SUB) * C;
        const int p = cm.p0 + l % cm.np, f = cm.f0 + l / cm.np;
        const int row0 = (p * cm.F + f) * NY;
        tma::mbar_arrive_expect_tx(&full[s], Cfg::STAGE_BYTES);
#pragma unroll
        for (int b = 0; b < Cfg::NBOX; ++b)
            tma::tensor_load_2d(stage0 + (size_t)s * NY * C + (size_t)b * Cfg::BOX_R * C, &wmap, 2 * kx0,
                                row0 + b * Cfg::BOX_R, &full[s]);
    };

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) tma::mbar_init(&full[s], 1);
        tma::fence_mbar_init();
    }
    for (int i = threadIdx.x; i < NY; i += Cfg::THREADS) py_s[i] = py[i];
    Twiddles<NY> tw;
    tw.init(t);
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < PF; ++k)
            if (blockIdx.x + k * gridDim.x < n_items) issue_load(blockIdx.x + k * gridDim.x, k);
    }

    int it = 0;
    int rem = blockIdx.x % per_wave;                         // item % per_wave, kept incrementally (no division per item)
    const int rem_step = gridDim.x % per_wave;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++it) {
        const int s = it % NS;
        if (threadIdx.x == 0) {
            const int nxt = item + PF * gridDim.x;
            if (nxt < n_items) {
                tma::bulk_wait_read<1>();                     // stage (it+PF)%NS was stored NS-PF = 2 items ago: drained
                issue_load(nxt, (it + PF) % NS);
            }
        }
        const int tj = rem / SUB;
        const int kx0 = (tj < tiles_lo ? tj : tj + tile_gap) * kColTile + (rem % SUB) * C;
        const int kx = kx0 + c;
        const int nm = nmax[kx];
        const float2 pxv = px[kx];
        float2* st = stage0 + (size_t)s * NY * C;
        ColSlots<C> slots(st + c, t);
        tma::mbar_wait(&full[s], (it / NS) & 1);
        float2 v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) v[e] = slots.at(t + e * T);
        fft_forward<NY, ColSlots<C>, BlockSync>(v, t, tw, slots);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int iy = t + e * T;
            const int n = iy < NY / 2 ? iy : NY - iy;         // |signed index|
            v[e] = (n <= nm) ? cmul(v[e], cmul(pxv, py_s[iy])) : make_float2(0.f, 0.f);
        }
        if (!LAST) fft_inverse<NY, ColSlots<C>, BlockSync>(v, t, tw, slots);
        __syncthreads();                                      // exchange reads of this stage are done
#pragma unroll
        for (int e = 0; e < 16; ++e) slots.at(t + e * T) = v[e];
        tma::fence_proxy_async();
        __syncthreads();
        if (threadIdx.x == 0) {
            const int l = item / per_wave;
            const int p = cm.p0 + l % cm.np, f = cm.f0 + l / cm.np;
            const int row0 = (p * cm.F + f) * NY;
#pragma unroll
            for (int b = 0; b < Cfg::NBOX; ++b)
                tma::tensor_store_2d(&wmap, 2 * kx0, row0 + b * Cfg::BOX_R, st + (size_t)b * Cfg::BOX_R * C);
            tma::bulk_commit();
        }
        rem += rem_step;
        if (rem >= per_wave) rem -= per_wave;
    }
    if (threadIdx.x == 0) tma::bulk_wait_all<0>();
}

// last slice: column tiles outside the band limit of the k-space exit wave are exact zeros
__global__ void k_zero_cols(float2* __restrict__ W, const int nx, const int ny, const int col_lo, const int col_hi,
                            const ChunkMap cm) {
    const int width = col_hi - col_lo;
    const long long total = (long long)cm.np * cm.nf * ny * width;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(i % width);
        const long long row = i / width;
        const int y = (int)(row % ny), l = (int)(row / ny);
        const int p = cm.p0 + l % cm.np, f = cm.f0 + l / cm.np;
        W[(((size_t)p * cm.F + f) * ny + y) * nx + col_lo + x] = make_float2(0.f, 0.f);
    }
}

// ------------------------------------------------------------------------------------ launch helpers
template <int NX, bool FIRST>
static cudaError_t launch_row(ps_ctx* c, float2* W, const float2* psi0, const float* V, const ChunkMap& cm,
                              int slice, float sigma, int col_lo, int col_hi) {
    using Cfg = RowCfg<NX>;
    auto kern = k_row_transmit<NX, FIRST>;
    int per_sm_grid = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &per_sm_grid);
    if (ce != cudaSuccess) return ce;
    const long long n_rows = (long long)cm.np * cm.nf * c->ny;
    const int n_items = (int)((n_rows + Cfg::RPB - 1) / Cfg::RPB);
    const int grid = n_items < per_sm_grid ? n_items : per_sm_grid;
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(W, psi0, V, c->d_tile_active, cm, c->ny, c->n_slices, slice,
                                                      sigma, n_items, col_lo, col_hi, c->vacuum_shortcut);
    return cudaGetLastError();
}

template <int NY, bool LAST>
static cudaError_t launch_col(ps_ctx* c, const CUtensorMap& wmap, const ChunkMap& cm, int zero_lo, int zero_hi) {
    using Cfg = ColCfg<NY>;
    auto kern = k_col_propagate<NY, LAST>;
    int per_sm_grid = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &per_sm_grid);
    if (ce != cudaSuccess) return ce;
    const int n_tiles = c->n_tiles_active;
    const int n_items = cm.np * cm.nf * n_tiles * (kColTile / Cfg::C);
    const int grid = n_items < per_sm_grid ? n_items : per_sm_grid;
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(wmap, zero_lo / kColTile, (zero_hi - zero_lo) / kColTile, n_tiles, c->d_nmax,
                                                      LAST ? c->kv.d_px_last : c->kv.d_px_mid, c->kv.d_py, cm, n_items);
    return cudaGetLastError();
}

template <int NY>
static bool make_wave_map(CUtensorMap* map, void* W, int nx, long long rows) {
    using Cfg = ColCfg<NY>;
    return tma::make_map_2d_f32(map, W, 2ull * nx, (uint64_t)rows, 2 * Cfg::C, Cfg::BOX_R);
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

static constexpr long long kResidentMaxWaves = 2 * kNumSM;   // auto rule of the chip-resident path

extern "C" ps_status ps_multislice(ps_ctx* c, double kV, const void* d_psi0, int n_probes, const float* d_V,
                                   int n_frames, void* d_exit, int exit_layout) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_multislice: ps_set_geometry has not been called");
    if (!d_psi0 || !d_V || !d_exit || n_probes < 1 || n_frames < 1 || !(kV > 0.0))
        return fail(c, PS_EINVAL, "ps_multislice: null pointer or non-positive size / voltage");
    if (exit_layout != PS_LAYOUT_DENSE) return fail(c, PS_EUNSUPPORTED, "ps_multislice: unknown exit layout");
    ps_status st = enter(c, "ps_multislice");
    if (st != PS_OK) return st;
    if ((st = ensure_kv(c, kV)) != PS_OK) return st;

    // Waves per launch.  Measured on B200 (c2, 256^2, 512 waves; profiles/r1_chunk_sweep.md): streaming the whole
    // batch from HBM in one launch per pass beats L2-resident chunks of 40-80 MB, whose launches are too short
    // to amortise launch latency, twiddle set-up and the last partial wave of blocks.  Default: no chunking.
    long long chunk = c->wave_chunk;
    if (chunk <= 0) chunk = (long long)n_probes * n_frames;
    const int np = (int)(n_probes < chunk ? n_probes : chunk);
    int nf = (int)(chunk / np);
    if (nf < 1) nf = 1;
    if (nf < n_frames) {                                     // equal-sized frame chunks (no short tail chunk)
        const int n_chunks = (n_frames + nf - 1) / nf;
        nf = (n_frames + n_chunks - 1) / n_chunks;
    }
    float2* W = (float2*)d_exit;
    const float2* psi0 = (const float2*)d_psi0;
    const float sigma = (float)c->kv.sigma;
    const int S = c->n_slices;

    // TMA view of the wave array: float32 [P*F*ny][2 nx]; box = C columns x up to 256 rows
    const long long wave_rows = (long long)n_probes * n_frames * c->ny;
    if (wave_rows > 0x7fffffffLL) return fail(c, PS_EUNSUPPORTED, "ps_multislice: n_probes*n_frames*ny exceeds 2^31");
    CUtensorMap wmap;
    bool map_ok = false;
    PSB_DISPATCH_N(c->ny, (map_ok = make_wave_map<N_>(&wmap, d_exit, c->nx, wave_rows)));
    if (!map_ok) return fail(c, PS_ECUDA, "ps_multislice: cuTensorMapEncodeTiled failed (exit-wave array must be 16-byte aligned)");
    // contiguous range of columns outside the band limit (zero in the k-space exit wave)
    int zero_lo = 0, zero_hi = 0;
    {
        const int nt = c->nx / kColTile;
        std::vector<char> act(nt, 0);
        for (int tI : c->h_tiles) act[tI] = 1;
        int a = 0;
        while (a < nt && act[a]) ++a;
        int b = nt;
        while (b > a && act[b - 1]) --b;
        zero_lo = a * kColTile; zero_hi = b * kColTile;
    }

    // Small square grids, small batches: the whole slice loop in one launch with the wave resident in shared memory
    // (resident.cu).  Batches that fill the GPU stay on the streaming passes (measured cross-over: profiles/r2_resident.md).
    if (resident_supported(c) && !c->vacuum_shortcut && c->wave_chunk == 0 &&
        (c->tune_resident == 1 || (c->tune_resident == 0 && (long long)n_probes * n_frames <= kResidentMaxWaves))) {
        cudaError_t e = launch_slice_resident(c, W, psi0, d_V, n_probes, n_frames, sigma, zero_lo, zero_hi);
        if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_slice_resident: ") + cudaGetErrorString(e));
        c->launches++;
        return PS_OK;
    }

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
                if (s == 0) { PSB_DISPATCH_N(c->nx, (e = launch_row<N_, true>(c, W, psi0, d_V, cm, s, sigma, zero_lo, zero_hi))); }
                else        { PSB_DISPATCH_N(c->nx, (e = launch_row<N_, false>(c, W, psi0, d_V, cm, s, sigma, zero_lo, zero_hi))); }
                }
                if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_row_transmit: ") + cudaGetErrorString(e));
                c->launches++;
                e = cudaErrorInvalidValue;
                {
                ProfScope ps_(c, K_COL_PROPAGATE);
                if (s == S - 1) {
                    if (zero_hi > zero_lo) {
                        const long long tot = (long long)cm.np * cm.nf * c->ny * (zero_hi - zero_lo);
                        const int zb = (int)((tot + 255) / 256 < 148 * 16 ? (tot + 255) / 256 : 148 * 16);
                        k_zero_cols<<<zb, 256, 0, c->stream>>>(W, c->nx, c->ny, zero_lo, zero_hi, cm);
                        c->launches++;
                    }
                    PSB_DISPATCH_N(c->ny, (e = launch_col<N_, true>(c, wmap, cm, zero_lo, zero_hi)));
                } else {
                    PSB_DISPATCH_N(c->ny, (e = launch_col<N_, false>(c, wmap, cm, zero_lo, zero_hi)));
                }
                }
                if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_col_propagate: ") + cudaGetErrorString(e));
                c->launches++;
            }
        }
    }
    return PS_OK;
}
