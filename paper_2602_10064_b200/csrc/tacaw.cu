// tacaw.cu — the TACAW transform (§2.1; Suppl. Eq. 5-6 at PAPER.md:295-301):
//     Psi~(k, w_n) = sum_j ( Psi(k, t_j) - <Psi(k, t)>_t ) exp(-2 pi i n j / F),   I(k, w_n) = |Psi~|^2
// Path A (ps_tacaw): one batched length-F FFT along the time axis per (probe, k) with the |.|^2 epilogue,
//   reading the exit-wave stack [P][F][ny][nx] once; a block owns C adjacent k-pixels x all F frames, so
//   every global access is a C*8-byte contiguous segment.  Pixels outside the band limit are exactly zero
//   in every frame (ps_multislice wrote them as zeros) and are not read: their I is written as 0.
//   The mean is removed by (i) subtracting the first frame's value before the transform, which strips
//   the large elastic (Bragg) part so that fp32 rounding of it cannot leak into other bins, and
//   (ii) zeroing bin 0 afterwards — identical to subtracting <Psi>_t for exact FFT bins (A14).
// Path B (ps_tacaw_begin/add/finish): streaming per-bin DFT accumulation for stacks that do not fit HBM.
#include "common.cuh"
#include "fft_core.cuh"
#include "tma.cuh"

namespace psb {

// TILED: the exit waves come in PS_LAYOUT_TILED_APERTURE, [P][ny][tile][F][8 kx]: a pixel group must lie inside one
// 8-column tile (C <= 8), and its F frames are one contiguous run of F * 64 bytes.
template <int NF, bool TILED = false> struct TacawCfg {
    static constexpr int T = Plan<NF>::T;
    // pixels per group: narrower groups would allow two resident blocks at 512 / 1024 frames but read 32-byte pieces:
    // measured 0.39 -> 0.16 of the HBM roofline at 1024 frames (profiles/r2_tacaw.md)
    static constexpr int C0 = (NF <= 512) ? 16 : ((NF == 1024) ? 8 : 4);
    static constexpr int C = (TILED && C0 > kColTile) ? kColTile : C0;
    static constexpr int THREADS = C * T;
    static constexpr size_t SMEM = (size_t)NF * C * sizeof(float2);
};

template <int NF, bool TILED>
__global__ void __launch_bounds__(TacawCfg<NF, TILED>::THREADS)
k_tacaw_fft(const float2* __restrict__ exitw, float* __restrict__ I, const int32_t* __restrict__ slot_of_bin,
            const int n_out, const int nx, const int ny, const int32_t* __restrict__ nmax, const int n_items,
            const int prefetch, const int32_t* __restrict__ tile_slot, const int n_tiles) {
    using Cfg = TacawCfg<NF, TILED>;
    constexpr int T = Cfg::T, C = Cfg::C;
    extern __shared__ float2 smem[];
    const int c = threadIdx.x % C, t = threadIdx.x / C;
    ColSlots<C> slots(smem + c, t);
    Twiddles<NF> tw;
    tw.init(t);
    const size_t npix = (size_t)nx * ny;
    const int groups_per_row = nx / C, groups_per_probe = groups_per_row * ny;
    int slot[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) slot[e] = slot_of_bin[t + e * T];

    // nx, ny and C are powers of two: shifts instead of four integer divisions per item and thread
    const int gpr_shift = __ffs(groups_per_row) - 1, gpp_shift = __ffs(groups_per_probe) - 1;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int p = item >> gpp_shift, g = item & (groups_per_probe - 1);
        const int iy = g >> gpr_shift, ix0 = (g & (groups_per_row - 1)) * C;
        const int ay = iy < ny / 2 ? iy : ny - iy;
        const size_t pix = (size_t)iy * nx + ix0 + c;
        {
            // this block's NEXT item: pull its F segments of C*8 bytes from HBM into L2 while the current item is
            // transformed, so that the register-staged loads below find them there.  One prefetch per lane and segment.
            // Measured (profiles/r2_tacaw.md): +5...+28 % for stacks of up to 512 frames on grids up to 512^2, a loss
            // beyond (an item then touches more 2 MB pages than the TLB holds, and the prefetch doubles the misses):
            // the host switches it per shape.
            const int nxt = item + gridDim.x;
            if (!TILED && prefetch && nxt < n_items) {
                const int pn = nxt >> gpp_shift, gn = nxt & (groups_per_probe - 1);
                const int iyn = gn >> gpr_shift, ixn = (gn & (groups_per_row - 1)) * C;
                const int ayn = iyn < ny / 2 ? iyn : ny - iyn;
                if (ayn <= max(nmax[ixn], nmax[ixn + C - 1])) {              // nmax is monotone in |m|: the group's best column is an end
                    const float2* nsrc = exitw + (size_t)pn * NF * npix + (size_t)iyn * nx + ixn;
                    for (int j = threadIdx.x; j < NF; j += Cfg::THREADS) tma::prefetch_l2(nsrc + (size_t)j * npix);
                }
            }
        }
        float* out = I + (size_t)p * n_out * npix + pix;
        const bool mine = ay <= nmax[ix0 + c];
        if (!__syncthreads_or(mine)) {                       // whole group outside the band limit
#pragma unroll
            for (int e = 0; e < 16; ++e)
                if (slot[e] >= 0) out[(size_t)slot[e] * npix] = 0.f;
            continue;
        }
        // frame j of this thread's pixel: dense [P][F][ny][nx], or tiled [P][ny][tile][F][8]
        const float2* src = TILED ? exitw + ((((size_t)p * ny + iy) * n_tiles + tile_slot[ix0 / kColTile]) * NF) * kColTile +
                                        (ix0 % kColTile) + c
                                  : exitw + (size_t)p * NF * npix + pix;
        const size_t fstride = TILED ? (size_t)kColTile : npix;
        const float2 ref = __ldg(src);                       // frame 0 (A14: mean removal, see header)
        float2 v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float2 x = src[(size_t)(t + e * T) * fstride];
            v[e] = make_float2(x.x - ref.x, x.y - ref.y);
        }
        fft_forward<NF, ColSlots<C>, BlockSync>(v, t, tw, slots);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            if (slot[e] >= 0) {
                const bool dc = (t + e * T) == 0 || !mine;   // out-of-band pixels of a group that straddles the edge
                out[(size_t)slot[e] * npix] = dc ? 0.f : fmaf(v[e].x, v[e].x, v[e].y * v[e].y);
            }
        }
    }
}

// ------------------------------------------------------------------------------------ path A, TMA-staged
// Same transform, fed by the copy engine: the exit-wave stack is viewed as a 2-D float32 tensor
// [P*F rows][2*nx*ny floats]; one item = C adjacent in-band pixels x all F frames = NBOX boxes of (2C floats x
// <=256 rows) landing in one shared-memory stage, which then serves as the FFT exchange buffer.  A ring of NS stages
// keeps the loads of the next items in flight while the current one is transformed, so one 512-thread block per SM
// streams from HBM without exposing the load latency.  Only groups with at least one in-band pixel are visited (list
// built once per geometry); the other pixels of I are zero-filled by k_tacaw_zero.
template <int NF, bool TILED = false> struct TacawTmaCfg {
    static constexpr int T = Plan<NF>::T;
    static constexpr int C0 = (NF <= 512) ? 16 : ((NF == 1024) ? 8 : 4);
    static constexpr int C = (TILED && C0 > kColTile) ? kColTile : C0;
    static constexpr int THREADS = C * T;
    static constexpr int NS = 3;
    static constexpr int BOX_R = (NF < 256) ? NF : 256;
    static constexpr int NBOX = NF / BOX_R;
    static constexpr uint32_t STAGE_BYTES = (uint32_t)NF * C * sizeof(float2);
    static constexpr size_t SMEM = (size_t)NS * STAGE_BYTES + NS * sizeof(uint64_t) + 128;
    static constexpr int MIN_BLOCKS = (THREADS <= 256) ? 2 : 1;
};

// TILED: emap views the tiled array as float32 [P*ny*n_tiles*F rows][16]; the F frames of a (row, tile) are consecutive
// rows, so an item is NBOX boxes of up to 256 consecutive 64-byte rows: contiguous runs for the copy engine.
template <int NF, bool TILED>
__global__ void __launch_bounds__(TacawTmaCfg<NF, TILED>::THREADS, TacawTmaCfg<NF, TILED>::MIN_BLOCKS)
k_tacaw_tma(const __grid_constant__ CUtensorMap emap, float* __restrict__ I, const int32_t* __restrict__ slot_of_bin,
            const int n_out, const int nx, const int ny, const int32_t* __restrict__ nmax,
            const int32_t* __restrict__ groups, const int n_groups, const int n_items,
            const int32_t* __restrict__ tile_slot, const int n_tiles) {
    using Cfg = TacawTmaCfg<NF, TILED>;
    constexpr int T = Cfg::T, C = Cfg::C, NS = Cfg::NS, PF = NS - 1;
    extern __shared__ __align__(1024) float2 smem_t[];
    float2* stage0 = smem_t;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_t + (size_t)NS * NF * C);
    const int c = threadIdx.x % C, t = threadIdx.x / C;
    const size_t npix = (size_t)nx * ny;

    auto issue_load = [&](const int item, const int s) {
        const int p = item / n_groups;
        int c0 = 2 * groups[item % n_groups], c1 = p * NF;
        if (TILED) {
            const int pix0 = groups[item % n_groups];
            const int gx = pix0 & (nx - 1), gy = pix0 / nx;
            c0 = 2 * (gx % kColTile);
            c1 = ((p * ny + gy) * n_tiles + tile_slot[gx / kColTile]) * NF;
        }
        tma::mbar_arrive_expect_tx(&full[s], Cfg::STAGE_BYTES);
#pragma unroll
        for (int b = 0; b < Cfg::NBOX; ++b)
            tma::tensor_load_2d(stage0 + (size_t)s * NF * C + (size_t)b * Cfg::BOX_R * C, &emap, c0,
                                c1 + b * Cfg::BOX_R, &full[s]);
    };

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) tma::mbar_init(&full[s], 1);
        tma::fence_mbar_init();
    }
    Twiddles<NF> tw;
    tw.init(t);
    int slot[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) slot[e] = slot_of_bin[t + e * T];
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < PF; ++k)
            if (blockIdx.x + k * gridDim.x < n_items) issue_load(blockIdx.x + k * gridDim.x, k);
    }

    int it = 0;
    const int nx_shift = __ffs(nx) - 1;
    int g_rem = blockIdx.x % n_groups, p_cur = blockIdx.x / n_groups;
    const int g_step = gridDim.x % n_groups, p_step = gridDim.x / n_groups;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++it) {
        const int s = it % NS;
        // every thread is past the exchange of item it-1, whose stage (it+PF)%NS is the next load's target
        tma::fence_proxy_async();
        __syncthreads();
        if (threadIdx.x == 0) {
            const int nxt = item + PF * gridDim.x;
            if (nxt < n_items) issue_load(nxt, (it + PF) % NS);
        }
        const int pix0 = groups[g_rem];                      // g_rem = item % n_groups, p_cur = item / n_groups (incremental)
        const int p = p_cur;
        const int ix = (pix0 & (nx - 1)) + c, iy = pix0 >> nx_shift;
        const int ay = iy < ny / 2 ? iy : ny - iy;
        const bool mine = ay <= nmax[ix];                    // the group has in-band pixels; this one may not be
        float* out = I + (size_t)p * n_out * npix + pix0 + c;
        ColSlots<C> slots(stage0 + (size_t)s * NF * C + c, t);
        tma::mbar_wait(&full[s], (it / NS) & 1);
        const float2 ref = slots.at(0);                      // frame 0 (A14: mean removal, see header)
        float2 v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float2 x = slots.at(t + e * T);
            v[e] = make_float2(x.x - ref.x, x.y - ref.y);
        }
        fft_forward<NF, ColSlots<C>, BlockSync>(v, t, tw, slots);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            if (slot[e] >= 0) {
                const bool zero = (t + e * T) == 0 || !mine;
                out[(size_t)slot[e] * npix] = zero ? 0.f : fmaf(v[e].x, v[e].x, v[e].y * v[e].y);
            }
        }
        g_rem += g_step; p_cur += p_step;
        if (g_rem >= n_groups) { g_rem -= n_groups; ++p_cur; }
    }
}

// I = 0 on the pixel groups that lie wholly outside the band limit (the exit wave is exactly zero there);
// groups are C >= 4 pixels wide and C-aligned, so every store is one aligned float4
__global__ void k_tacaw_zero(float* __restrict__ I, const int32_t* __restrict__ groups, const int n_groups, const int C4,
                             const size_t npix, const long long total /* P * n_out * n_groups * C4 */) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int c = (int)(i % C4);
        const long long r = i / C4;
        const int g = (int)(r % n_groups);
        const long long pb = r / n_groups;                  // p * n_out + slot
        *reinterpret_cast<float4*>(I + (size_t)pb * npix + groups[g] + 4 * c) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// ------------------------------------------------------------------------------------ path B: streaming DFT
// acc[p][b][k] += sum_{j in chunk} (Psi[p][j][k] - ref[p][k]) exp(-2 pi i n_b (frame0 + j) / F)
//
// One block owns a tile of SB_PIX adjacent pixels x up to SB_FR frames of the chunk, staged ONCE in shared memory by the
// copy engine (one 2-D TMA box, 64 KB), strips the reference wave from it (the elastic part, ~100x the signal: without
// it the fp32 partial sums of the Bragg term over thousands of frames would swamp weak bins; a constant
// shift of every frame changes no bin n != 0 of the complete sum, and bin 0 is written as exact zero), and then sweeps ALL
// bins over the tile: thread = (pixel, bin half), SB_BINS complex accumulators in registers per sweep, the twiddles of
// the sweep (SB_FR x 2 SB_BINS, read from a per-chunk table built by k_tacaw_twiddles in float64) broadcast from shared
// memory.  Every exit value is read from HBM once per chunk; the accumulators are read and written once per tile.
// Bound: FP32 FMA issue (4 n_bins FMA per sample against 8 bytes), not HBM.
constexpr int SB_PIX = 128, SB_BINS = 16, SB_FR = 64, SB_THREADS = 2 * SB_PIX;
constexpr size_t SB_SMEM = (size_t)SB_FR * SB_PIX * sizeof(float2) + (size_t)SB_FR * 2 * SB_BINS * sizeof(float2) + 64;

// tw[j][b] = exp(-2 pi i n_b (frame0 + j) / F), j < n_frames_chunk: float64 sincospi on an exactly reduced phase
__global__ void k_tacaw_twiddles(float2* __restrict__ tw, const int32_t* __restrict__ bins, const int n_bins,
                                 const int n_frames_total, const int frame0, const int n_frames_chunk) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_frames_chunk * n_bins) return;
    const int j = i / n_bins, b = i % n_bins;
    const long long ph = ((long long)bins[b] * (long long)(frame0 + j)) % n_frames_total;     // bins already in [0, F)
    double sn, cs;
    sincospi(2.0 * (double)ph / (double)n_frames_total, &sn, &cs);
    tw[i] = make_float2((float)cs, (float)(-sn));
}

__global__ void __launch_bounds__(SB_THREADS, 2)
k_tacaw_accum(const __grid_constant__ CUtensorMap cmap, float2* __restrict__ acc, const float2* __restrict__ ref,
              const float2* __restrict__ twtab, const int n_bins, const int n_frames_chunk, const size_t npix,
              const int nx, const int ny, const int32_t* __restrict__ nmax) {
    extern __shared__ __align__(1024) float2 smem_b[];
    float2* tile = smem_b;                                             // [SB_FR][SB_PIX]
    float2* wsm = smem_b + (size_t)SB_FR * SB_PIX;                     // [SB_FR][2 SB_BINS]
    uint64_t* full = reinterpret_cast<uint64_t*>(wsm + (size_t)SB_FR * 2 * SB_BINS);
    const int px = threadIdx.x % SB_PIX, half = threadIdx.x / SB_PIX;
    const size_t pix0 = (size_t)blockIdx.x * SB_PIX, pix = pix0 + px;
    const int p = blockIdx.y;
    const int iy = (int)(pix / nx), ix = (int)(pix % nx);
    const int ay = iy < ny / 2 ? iy : ny - iy;
    const bool mine = ay <= nmax[ix];
    if (!__syncthreads_or(mine)) return;                                // tile wholly outside the band: acc stays zero
    if (threadIdx.x == 0) { tma::mbar_init(full, 1); tma::fence_mbar_init(); }
    __syncthreads();
    const float2 rf = mine ? __ldg(ref + (size_t)p * npix + pix) : make_float2(0.f, 0.f);
    int it = 0;
    for (int j0 = 0; j0 < n_frames_chunk; j0 += SB_FR, ++it) {
        const int cnt = min(SB_FR, n_frames_chunk - j0);
        if (threadIdx.x == 0) {                                         // rows past the chunk / the probe are never used
            tma::fence_proxy_async();                                   // earlier generic-proxy accesses of the tile
            tma::mbar_arrive_expect_tx(full, (uint32_t)(SB_FR * SB_PIX * sizeof(float2)));
            tma::tensor_load_2d(tile, &cmap, (int)(2 * pix0), p * n_frames_chunk + j0, full);
        }
        tma::mbar_wait(full, it & 1);
        for (int jj = half; jj < cnt; jj += 2) {                        // strip the reference from this thread's pixel
            float2 x = tile[jj * SB_PIX + px];
            x.x -= rf.x; x.y -= rf.y;
            tile[jj * SB_PIX + px] = x;
        }
        for (int b0 = 0; b0 < n_bins; b0 += 2 * SB_BINS) {
            __syncthreads();                                            // tile ready / previous sweep done with wsm
            for (int i = threadIdx.x; i < cnt * 2 * SB_BINS; i += SB_THREADS) {
                const int jj = i / (2 * SB_BINS), b = b0 + i % (2 * SB_BINS);
                wsm[i] = (b < n_bins) ? __ldg(twtab + (size_t)(j0 + jj) * n_bins + b) : make_float2(0.f, 0.f);
            }
            __syncthreads();
            float2 a[SB_BINS];
#pragma unroll
            for (int b = 0; b < SB_BINS; ++b) a[b] = make_float2(0.f, 0.f);
            const float4* wrow = reinterpret_cast<const float4*>(wsm + half * SB_BINS);
#pragma unroll 2
            for (int jj = 0; jj < cnt; ++jj) {
                const float2 x = tile[jj * SB_PIX + px];
#pragma unroll
                for (int q = 0; q < SB_BINS / 2; ++q) {
                    const float4 ww = wrow[jj * SB_BINS + q];           // two twiddles, same address in the whole warp
                    a[2 * q].x = fmaf(x.x, ww.x, a[2 * q].x); a[2 * q].x = fmaf(-x.y, ww.y, a[2 * q].x);
                    a[2 * q].y = fmaf(x.x, ww.y, a[2 * q].y); a[2 * q].y = fmaf(x.y, ww.x, a[2 * q].y);
                    a[2 * q + 1].x = fmaf(x.x, ww.z, a[2 * q + 1].x); a[2 * q + 1].x = fmaf(-x.y, ww.w, a[2 * q + 1].x);
                    a[2 * q + 1].y = fmaf(x.x, ww.w, a[2 * q + 1].y); a[2 * q + 1].y = fmaf(x.y, ww.z, a[2 * q + 1].y);
                }
            }
            if (mine) {
#pragma unroll
                for (int b = 0; b < SB_BINS; ++b) {
                    const int bb = b0 + half * SB_BINS + b;
                    if (bb < n_bins) {
                        float2* d = acc + ((size_t)p * n_bins + bb) * npix + pix;
                        const float2 o = *d;
                        *d = make_float2(o.x + a[b].x, o.y + a[b].y);
                    }
                }
            }
        }
        __syncthreads();                                                // everyone is done with the tile before the next load
    }
}

// I = |acc|^2; bin 0 is sum_j (Psi_j - <Psi>) = 0 exactly (A14)
__global__ void k_tacaw_finish(const float2* __restrict__ acc, float* __restrict__ I, const int32_t* __restrict__ bins,
                               const int n_bins, const size_t npix, const long long total) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int b = (int)((i / npix) % n_bins);
    const float2 a = acc[i];
    I[i] = (bins[b] == 0) ? 0.f : fmaf(a.x, a.x, a.y * a.y);
}

template <int NF, bool TILED>
static cudaError_t launch_tacaw(ps_ctx* c, const float2* exitw, float* I, const int32_t* slot, int n_out, int P) {
    using Cfg = TacawCfg<NF, TILED>;
    auto kern = k_tacaw_fft<NF, TILED>;
    int cap = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &cap);
    if (ce != cudaSuccess) return ce;
    const long long n_items = (long long)P * c->ny * (c->nx / Cfg::C);
    if (n_items > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int prefetch = (NF <= 512 && (long long)c->nx * c->ny <= 512LL * 512LL) ? 1 : 0;
    kern<<<(int)(n_items < cap ? n_items : cap), Cfg::THREADS, Cfg::SMEM, c->stream>>>(exitw, I, slot, n_out, c->nx, c->ny,
                                                                                      c->d_nmax, (int)n_items, prefetch,
                                                                                      c->d_tile_slot, c->n_tiles_active);
    return cudaGetLastError();
}

// pixel groups of width C (first pixel of each): [active..., inactive...], cached per geometry
static ps_status ensure_tacaw_groups(ps_ctx* c, int C) {
    if (c->tacaw_groups_C == C) return PS_OK;
    std::vector<int32_t> act, inact;
    for (int iy = 0; iy < c->ny; ++iy) {
        const int ay = iy < c->ny / 2 ? iy : c->ny - iy;
        for (int ix0 = 0; ix0 < c->nx; ix0 += C) {
            bool any = false;
            for (int j = 0; j < C; ++j) any = any || (ay <= c->h_nmax[ix0 + j]);
            (any ? act : inact).push_back(iy * c->nx + ix0);
        }
    }
    c->tacaw_n_active = (int)act.size(); c->tacaw_n_inactive = (int)inact.size();
    act.insert(act.end(), inact.begin(), inact.end());
    ps_status st = ensure_buf(c, c->tacaw_groups, act.size() * sizeof(int32_t));
    if (st != PS_OK) return st;
    if ((st = upload_async(c, c->tacaw_groups.p, act.data(), act.size() * sizeof(int32_t))) != PS_OK) return st;   // once per geometry
    c->tacaw_groups_C = C;
    return PS_OK;
}

template <int NF, bool TILED>
static ps_status launch_tacaw_tma(ps_ctx* c, const float2* exitw, float* I, const int32_t* slot, int n_out, int P) {
    using Cfg = TacawTmaCfg<NF, TILED>;
    auto kern = k_tacaw_tma<NF, TILED>;
    int cap = 0;
    PSB_CUDA(c, kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &cap));
    ps_status st = ensure_tacaw_groups(c, Cfg::C);
    if (st != PS_OK) return st;
    const size_t npix = (size_t)c->nx * c->ny;
    const long long tiled_rows = (long long)P * c->ny * c->n_tiles_active * NF;
    if ((long long)P * NF > 0x7fffffffLL || 2 * npix > 0xffffffffULL || (TILED && tiled_rows > 0x7fffffffLL))
        return fail(c, PS_EUNSUPPORTED, "ps_tacaw: exit-wave stack has more than 2^31 rows");
    CUtensorMap emap;
    const bool map_ok = TILED ? tma::make_map_2d_f32(&emap, (void*)exitw, 2ull * kColTile, (uint64_t)tiled_rows, 2 * Cfg::C, Cfg::BOX_R)
                              : tma::make_map_2d_f32(&emap, (void*)exitw, 2ull * npix, (uint64_t)P * NF, 2 * Cfg::C, Cfg::BOX_R);
    if (!map_ok)
        return fail(c, PS_ECUDA, "ps_tacaw: cuTensorMapEncodeTiled failed (exit-wave array must be 16-byte aligned)");
    const int32_t* groups = (const int32_t*)c->tacaw_groups.p;
    const long long n_items = (long long)P * c->tacaw_n_active;
    if (n_items > 0x7fffffffLL) return fail(c, PS_EUNSUPPORTED, "ps_tacaw: too many pixel groups");
    if (c->tacaw_n_inactive > 0) {
        const long long total = (long long)P * n_out * c->tacaw_n_inactive * (Cfg::C / 4);
        const long long nb = (total + 255) / 256;
        k_tacaw_zero<<<(unsigned)(nb < 148 * 64 ? nb : 148 * 64), 256, 0, c->stream>>>(
            I, groups + c->tacaw_n_active, c->tacaw_n_inactive, Cfg::C / 4, npix, total);
        PSB_LAUNCH_CHECK(c, "k_tacaw_zero");
    }
    if (n_items > 0) {
        kern<<<(int)(n_items < cap ? n_items : cap), Cfg::THREADS, Cfg::SMEM, c->stream>>>(
            emap, I, slot, n_out, c->nx, c->ny, c->d_nmax, groups, c->tacaw_n_active, (int)n_items, c->d_tile_slot,
            c->n_tiles_active);
        PSB_LAUNCH_CHECK(c, "k_tacaw_tma");
    }
    return PS_OK;
}

// ref[p][q] = chunk[p][frame 0][q]: the default reference wave of a stream (first frame of every probe)
__global__ void k_tacaw_first_frame(const float4* __restrict__ chunk, float4* __restrict__ ref, const size_t q_per_probe,
                                    const size_t probe_stride, const size_t total) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t p = i / q_per_probe, q = i - p * q_per_probe;
        ref[i] = chunk[p * probe_stride + q];
    }
}

}  // namespace psb

using namespace psb;

extern "C" ps_status ps_tacaw(ps_ctx* c, const void* d_exit, int exit_layout, int n_probes, int n_frames, double dt_fs,
                              int n_bins, const int32_t* bins, float* d_I) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_tacaw: ps_set_geometry has not been called");
    if (!d_exit || !d_I || n_probes < 1 || n_frames < 1 || n_bins < 1 || !(dt_fs > 0.0))
        return fail(c, PS_EINVAL, "ps_tacaw: null pointer or non-positive size / dt");
    if (exit_layout != PS_LAYOUT_DENSE && exit_layout != PS_LAYOUT_TILED_APERTURE)
        return fail(c, PS_EUNSUPPORTED, "ps_tacaw: unknown exit layout");
    const bool tiled = exit_layout == PS_LAYOUT_TILED_APERTURE;
    if (!is_pow2(n_frames) || n_frames < 32 || n_frames > 4096)
        return fail(c, PS_EUNSUPPORTED, "ps_tacaw: n_frames must be a power of two in [32, 4096] (use ps_tacaw_begin/add/finish otherwise)");
    if (!bins && n_bins != n_frames) return fail(c, PS_EINVAL, "ps_tacaw: bins == NULL requires n_bins == n_frames");
    ps_status st_in = enter(c, "ps_tacaw");
    if (st_in != PS_OK) return st_in;
    std::vector<int32_t> slot(n_frames, -1);
    for (int b = 0; b < n_bins; ++b) {
        long long n = bins ? bins[b] : b;
        n %= n_frames; if (n < 0) n += n_frames;
        if (slot[n] >= 0) return fail(c, PS_EINVAL, "ps_tacaw: duplicate bin in list");
        slot[n] = b;
    }
    // the bin -> output-slot table lives in its own buffer and is uploaded only when it changes: repeated calls with
    // the same bin list (every step of a run) enqueue work without a host-side wait
    if (slot != c->tacaw_slot_host || !c->tacaw_slot.p) {
        ps_status st = ensure_buf(c, c->tacaw_slot, (size_t)n_frames * 4);
        if (st != PS_OK) return st;
        if ((st = upload_async(c, c->tacaw_slot.p, slot.data(), (size_t)n_frames * 4)) != PS_OK) return st;   // staged: no host wait
        c->tacaw_slot_host = slot;
    }
    int32_t* d_slot = (int32_t*)c->tacaw_slot.p;
    ProfScope ps_(c, K_TACAW_FFT);
    const float2* ex = (const float2*)d_exit;
    // Kernel choice measured on B200 (profiles/r1_tacaw_kernels.md): the TMA-staged ring wins where one block per
    // SM is all that fits anyway (2048 frames) and where few bins are written (reads dominate, 512-1024 frames);
    // the register-staged kernel with several resident blocks wins for short stacks and when every bin is written.
    // tiled layout: the ring kernel at every length it covers (register-staged on the tiled layout measured 0.44 against
    // 0.65 at 1024 frames); dense layout: measured choice per shape (profiles/r1_tacaw_kernels.md)
    const bool use_ring = tiled ? (n_frames <= 2048)
                                : (n_frames == 2048 || ((n_frames == 512 || n_frames == 1024) && 4 * n_bins <= n_frames));
#define PSB_TACAW_CASE(NFV)                                                                                         \
    case NFV:                                                                                                       \
        if (use_ring) return tiled ? launch_tacaw_tma<NFV, true>(c, ex, d_I, d_slot, n_bins, n_probes)             \
                                   : launch_tacaw_tma<NFV, false>(c, ex, d_I, d_slot, n_bins, n_probes);           \
        e = tiled ? launch_tacaw<NFV, true>(c, ex, d_I, d_slot, n_bins, n_probes)                                   \
                  : launch_tacaw<NFV, false>(c, ex, d_I, d_slot, n_bins, n_probes);                                 \
        break;
    cudaError_t e = cudaErrorInvalidValue;
    switch (n_frames) {
        PSB_TACAW_CASE(32) PSB_TACAW_CASE(64) PSB_TACAW_CASE(128) PSB_TACAW_CASE(256) PSB_TACAW_CASE(512)
        PSB_TACAW_CASE(1024)
        case 2048:
            if (use_ring) return tiled ? launch_tacaw_tma<2048, true>(c, ex, d_I, d_slot, n_bins, n_probes)
                                       : launch_tacaw_tma<2048, false>(c, ex, d_I, d_slot, n_bins, n_probes);
            break;
        case 4096:
            e = tiled ? launch_tacaw<4096, true>(c, ex, d_I, d_slot, n_bins, n_probes)
                      : launch_tacaw<4096, false>(c, ex, d_I, d_slot, n_bins, n_probes);
            break;
        default: break;
    }
#undef PSB_TACAW_CASE
    if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_tacaw_fft: ") + cudaGetErrorString(e));
    c->launches++;
    return PS_OK;
}

extern "C" ps_status ps_tacaw_begin(ps_ctx* c, int n_probes, int n_frames_total, double dt_fs, int n_bins,
                                    const int32_t* bins, void* d_acc) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_tacaw_begin: ps_set_geometry has not been called");
    if (!d_acc || !bins || n_probes < 1 || n_frames_total < 1 || n_bins < 1 || !(dt_fs > 0.0))
        return fail(c, PS_EINVAL, "ps_tacaw_begin: null pointer or non-positive size / dt");
    TacawStream& ts = c->ts;
    ts.bins.resize(n_bins);
    for (int b = 0; b < n_bins; ++b) {
        long long n = bins[b] % n_frames_total; if (n < 0) n += n_frames_total;
        ts.bins[b] = (int32_t)n;
    }
    ps_status st = enter(c, "ps_tacaw_begin");
    if (st != PS_OK) return st;
    const size_t npix = (size_t)c->nx * c->ny;
    if ((st = ensure_buf(c, ts.d_bins, (size_t)n_bins * 4)) != PS_OK) return st;           // grows only; no free/alloc per call
    if ((st = ensure_buf(c, ts.d_ref, (size_t)n_probes * npix * sizeof(float2))) != PS_OK) return st;
    if ((st = upload_async(c, ts.d_bins.p, ts.bins.data(), (size_t)n_bins * 4)) != PS_OK) return st;
    const size_t bytes = (size_t)n_probes * n_bins * npix * sizeof(float2);
    PSB_CUDA(c, cudaMemsetAsync(d_acc, 0, bytes, c->stream));
    ts.active = true; ts.n_probes = n_probes; ts.n_frames_total = n_frames_total; ts.n_bins = n_bins;
    ts.frames_seen = 0; ts.next_frame = -1; ts.have_ref = false; ts.d_acc = d_acc;
    return PS_OK;
}

extern "C" ps_status ps_tacaw_set_reference(ps_ctx* c, const void* d_ref) {
    if (!c) return PS_EINVAL;
    TacawStream& ts = c->ts;
    if (!ts.active) return fail(c, PS_ESTATE, "ps_tacaw_set_reference: ps_tacaw_begin has not been called");
    if (ts.frames_seen > 0) return fail(c, PS_ESTATE, "ps_tacaw_set_reference: frames have already been added");
    ps_status st = enter(c, "ps_tacaw_set_reference");
    if (st != PS_OK) return st;
    const size_t bytes = (size_t)ts.n_probes * c->nx * c->ny * sizeof(float2);
    if (d_ref) PSB_CUDA(c, cudaMemcpyAsync(ts.d_ref.p, d_ref, bytes, cudaMemcpyDeviceToDevice, c->stream));
    else PSB_CUDA(c, cudaMemsetAsync(ts.d_ref.p, 0, bytes, c->stream));
    ts.have_ref = true;
    return PS_OK;
}

extern "C" ps_status ps_tacaw_add(ps_ctx* c, const void* d_exit_chunk, int frame0, int n_frames_chunk) {
    if (!c) return PS_EINVAL;
    TacawStream& ts = c->ts;
    if (!ts.active) return fail(c, PS_ESTATE, "ps_tacaw_add: ps_tacaw_begin has not been called");
    ps_status st = enter(c, "ps_tacaw_add");
    if (st != PS_OK) return st;
    if (!d_exit_chunk || frame0 < 0 || n_frames_chunk < 1 || frame0 + n_frames_chunk > ts.n_frames_total)
        return fail(c, PS_EINVAL, "ps_tacaw_add: null pointer or frame range outside [0, n_frames_total)");
    // chunks arrive in ascending, contiguous frame order (a shard may start anywhere): a frame can be neither counted
    // twice nor skipped
    if (ts.next_frame >= 0 && frame0 != ts.next_frame)
        return fail(c, PS_ESTATE, "ps_tacaw_add: chunk starts at frame " + std::to_string(frame0) + ", expected frame " +
                                      std::to_string(ts.next_frame) + " (chunks must be contiguous and ascending)");
    const size_t npix = (size_t)c->nx * c->ny;
    if ((long long)ts.n_probes * n_frames_chunk > 0x7fffffffLL || 2 * npix > 0xffffffffULL)
        return fail(c, PS_EUNSUPPORTED, "ps_tacaw_add: chunk has more than 2^31 rows");
    if (!ts.have_ref) {                                                 // reference = the first frame this stream sees
        // a strided gather of our own: cudaMemcpy2D refuses source pitches above 2^31-1 bytes, i.e. any chunk of 2 GiB
        // or more per probe (1024^2 x 256 frames, 512^2 x 1024 frames)
        const size_t q_per_probe = npix / 2;                            // float4 = two complex64
        const size_t total = q_per_probe * ts.n_probes;
        const size_t nb = (total + 255) / 256;
        k_tacaw_first_frame<<<(unsigned)(nb < (size_t)kNumSM * 16 ? nb : (size_t)kNumSM * 16), 256, 0, c->stream>>>(
            reinterpret_cast<const float4*>(d_exit_chunk), reinterpret_cast<float4*>(ts.d_ref.p), q_per_probe,
            q_per_probe * (size_t)n_frames_chunk, total);
        PSB_LAUNCH_CHECK(c, "k_tacaw_first_frame");
        ts.have_ref = true;
    }
    if ((st = ensure_buf(c, ts.d_tw, (size_t)n_frames_chunk * ts.n_bins * sizeof(float2))) != PS_OK) return st;
    CUtensorMap cmap;
    if (!tma::make_map_2d_f32(&cmap, (void*)d_exit_chunk, 2ull * npix, (uint64_t)ts.n_probes * n_frames_chunk, 2 * SB_PIX, SB_FR))
        return fail(c, PS_ECUDA, "ps_tacaw_add: cuTensorMapEncodeTiled failed (chunk must be 16-byte aligned)");
    int cap_unused = 0;
    PSB_CUDA(c, kernel_cap(c, k_tacaw_accum, SB_THREADS, SB_SMEM, &cap_unused));
    ProfScope ps_(c, K_TACAW_ACCUM);
    const int n_tw = n_frames_chunk * ts.n_bins;
    k_tacaw_twiddles<<<(n_tw + 255) / 256, 256, 0, c->stream>>>((float2*)ts.d_tw.p, (const int32_t*)ts.d_bins.p, ts.n_bins,
                                                               ts.n_frames_total, frame0, n_frames_chunk);
    PSB_LAUNCH_CHECK(c, "k_tacaw_twiddles");
    dim3 grid((unsigned)(npix / SB_PIX), ts.n_probes);
    k_tacaw_accum<<<grid, SB_THREADS, SB_SMEM, c->stream>>>(cmap, (float2*)ts.d_acc, (const float2*)ts.d_ref.p,
                                                           (const float2*)ts.d_tw.p, ts.n_bins, n_frames_chunk, npix, c->nx,
                                                           c->ny, c->d_nmax);
    PSB_LAUNCH_CHECK(c, "k_tacaw_accum");
    ts.frames_seen += n_frames_chunk;
    ts.next_frame = frame0 + n_frames_chunk;
    return PS_OK;
}

static ps_status tacaw_finish_impl(ps_ctx* c, const void* d_acc, size_t n_k, float* d_I) {
    TacawStream& ts = c->ts;
    const long long total = (long long)ts.n_probes * ts.n_bins * (long long)n_k;
    ProfScope ps_(c, K_TACAW_FINISH);
    k_tacaw_finish<<<(unsigned)((total + 255) / 256), 256, 0, c->stream>>>((const float2*)d_acc, d_I, (const int32_t*)ts.d_bins.p,
                                                                           ts.n_bins, n_k, total);
    PSB_LAUNCH_CHECK(c, "k_tacaw_finish");
    return PS_OK;
}

extern "C" ps_status ps_tacaw_finish(ps_ctx* c, float* d_I) {
    if (!c) return PS_EINVAL;
    TacawStream& ts = c->ts;
    if (!ts.active) return fail(c, PS_ESTATE, "ps_tacaw_finish: ps_tacaw_begin has not been called");
    ps_status st = enter(c, "ps_tacaw_finish");
    if (st != PS_OK) return st;
    if (!d_I) return fail(c, PS_EINVAL, "ps_tacaw_finish: d_I is NULL");
    if (ts.frames_seen != ts.n_frames_total)
        return fail(c, PS_ESTATE, "ps_tacaw_finish: " + std::to_string(ts.frames_seen) + " of " +
                                      std::to_string(ts.n_frames_total) + " frames were added");
    st = tacaw_finish_impl(c, ts.d_acc, (size_t)c->nx * c->ny, d_I);
    if (st == PS_OK) ts.active = false;
    return st;
}

extern "C" ps_status ps_tacaw_finish_shard(ps_ctx* c, const void* d_acc_shard, size_t n_k, float* d_I_shard) {
    if (!c) return PS_EINVAL;
    TacawStream& ts = c->ts;
    if (!ts.active) return fail(c, PS_ESTATE, "ps_tacaw_finish_shard: ps_tacaw_begin has not been called");
    ps_status st = enter(c, "ps_tacaw_finish_shard");
    if (st != PS_OK) return st;
    if (!d_acc_shard || !d_I_shard || n_k == 0) return fail(c, PS_EINVAL, "ps_tacaw_finish_shard: null pointer or empty shard");
    st = tacaw_finish_impl(c, d_acc_shard, n_k, d_I_shard);
    if (st == PS_OK) ts.active = false;
    return st;
}
