// resident.cu — chip-resident slice loop for small square grids (nx = ny <= 128; SURVEY.md 8(d) "128^2 in one SM's SMEM
// ... move only V", the slice loop):
//     psi <- psi exp(i sigma V_s);   psi <- ifft2( P A fft2(psi) ),   s = 0..S-1;     exit = fft2(psi)/sqrt(nx ny)
// One CTA keeps one wave in shared memory (128 x 136 complex64 = 136 KB at 128^2, rows padded 1 per 16 so that both the
// row and the column transforms are bank-conflict free) through ALL slices: per slice it reads only V_s (4 B per pixel)
// from HBM/L2, and the whole loop is ONE launch instead of 2 S.  The arithmetic is that of the two streaming passes
// (multislice.cu): row phase  M[y][:] <- FFT_x[ t(y,:) IFFT_x[ M[y][:] ] ],  column phase  M[:][kx] <- IFFT_y[ P A FFT_y[..] ],
// the wave living in the mixed layout M[y][kx] between them; the last column phase skips the inverse transform and
// writes the unitary k-space exit wave to HBM.  Used for batches too small to fill the GPU with streaming launches
// (config 1: 64 waves x 12 slices = 24 launches of ~5 us each); large batches stay on the streaming kernels, which
// prune the out-of-band columns of the column pass more finely (profiles/r2_resident.md).
#include "common.cuh"
#include "fft_core.cuh"
#include <type_traits>

namespace psb {

template <int N> struct ResCfg {
    static constexpr int T = Plan<N>::T;                                  // threads per transform
    static constexpr int THREADS = (N * T < 512) ? N * T : 512;           // 128 -> 512, 64 -> 256, 32 -> 64
    static constexpr int LEN = RowLine<N>::LEN;                           // padded row pitch (float2)
    static constexpr int ROWS_PER_ROUND = THREADS / T;
    static constexpr int CG_THREADS = 32 * T;                             // one column group: 32 columns x T threads
    static constexpr int N_CG = THREADS / CG_THREADS;                     // column groups in flight
    static constexpr size_t SMEM = ((size_t)N * LEN + N + TwiddlesShared<N>::TABLE) * sizeof(float2);
    using RowSync = typename std::conditional<(T <= 32), WarpSync, GroupSync<T>>::type;
    using ColSync = typename std::conditional<(N_CG > 1), GroupSync<CG_THREADS>, BlockSync>::type;
};

// a column of the padded wave array: element `row` of column kx at wave[row * LEN + kx + (kx >> 4)]
template <int LEN> struct PitchSlots {
    float2* base;                                                         // wave + padded(kx)
    __device__ __forceinline__ float2& at(const int idx) const { return base[idx * LEN]; }
    __device__ __forceinline__ float2& x1w(const int t, const int r) const { return at(16 * t + r); }
    template <int T> __device__ __forceinline__ float2& x1r(const int t, const int e) const { return at(t + e * T); }
    template <int N> __device__ __forceinline__ float2& x2w(const int t, const int b, const int r) const {
        const int j = t + b * Plan<N>::T;
        return at((j >> 4) * (16 * Plan<N>::R2) + (j & 15) + 16 * r);
    }
    template <int T> __device__ __forceinline__ float2& x2r(const int t, const int e) const { return at(t + e * T); }
};

struct ResWaves {            // waves of this launch: probes [p0, p0+np) x frames [f0, f0+nf); F = frames of the exit layout
    int p0, np, f0, nf, F;
};

template <int N>
__global__ void __launch_bounds__(ResCfg<N>::THREADS, 1)
k_slice_resident(float2* __restrict__ W, const float2* __restrict__ psi0, const float* __restrict__ V,
                 const int32_t* __restrict__ nmax, const float2* __restrict__ px_mid, const float2* __restrict__ px_last,
                 const float2* __restrict__ py, const ResWaves rw, const int n_slices, const float sigma,
                 const int col_lo, const int col_hi) {
    using Cfg = ResCfg<N>;
    using TW = TwiddlesShared<N>;
    constexpr int T = Cfg::T, LEN = Cfg::LEN;
    extern __shared__ __align__(16) float2 smem_r[];
    float2* wave = smem_r;                                                // [N][LEN]
    float2* py_s = smem_r + (size_t)N * LEN;                              // [N]
    float2* tab = py_s + N;                                               // stage-2 twiddle table
    for (int i = threadIdx.x; i < N; i += Cfg::THREADS) py_s[i] = py[i];
    TW::fill(tab, threadIdx.x, Cfg::THREADS);
    __syncthreads();

    // row-phase role: row r_row of a round, position t_row in its transform
    const int t_row = threadIdx.x % T, r_row = threadIdx.x / T;
    TW tw_row;
    tw_row.init(t_row, tab);
    unsigned amask = 0;                                                   // bit e: column t_row + e T is inside the band limit tiles
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const int col = t_row + e * T;
        amask |= ((col < col_lo || col >= col_hi) ? 1u : 0u) << e;
    }
    // column-phase role: column group g, position t_col, column lane c
    const int g = threadIdx.x / Cfg::CG_THREADS, t_col = (threadIdx.x / 32) % T, c = threadIdx.x % 32;
    TW tw_col;
    tw_col.init(t_col, tab);
    const int n_active = col_lo + (N - col_hi);
    const int n_cgroups = (n_active + 31) / 32;
    const int gap = col_hi - col_lo;

    const int n_waves = rw.np * rw.nf;
    for (int l = blockIdx.x; l < n_waves; l += gridDim.x) {
        const int p = rw.p0 + l % rw.np, f = rw.f0 + l / rw.np;
        float2* wout = W + ((size_t)p * rw.F + f) * N * N;
        for (int s = 0; s < n_slices; ++s) {
            // ------------------------------------------------------------ row phase
            const float* Vs = V + ((size_t)f * n_slices + s) * N * N;
            for (int y0 = 0; y0 < N; y0 += Cfg::ROWS_PER_ROUND) {
                const int y = y0 + r_row;
                RowSlots slots{wave + (size_t)y * LEN};
                float2 v[16];
                float sv[16];
#pragma unroll
                for (int e = 0; e < 16; ++e) sv[e] = __ldg(Vs + (size_t)y * N + t_row + e * T);
                if (s == 0) {
                    const float2* src = psi0 + ((size_t)p * N + y) * N;
#pragma unroll
                    for (int e = 0; e < 16; ++e) v[e] = __ldg(src + t_row + e * T);
                } else {
#pragma unroll
                    for (int e = 0; e < 16; ++e) v[e] = slots.at(t_row + e * T);
                    fft_inverse<N, RowSlots, typename Cfg::RowSync, TW>(v, t_row, tw_row, slots);
                }
#pragma unroll
                for (int e = 0; e < 16; ++e) v[e] = cmul(v[e], cis_fast(sigma * sv[e]));
                fft_forward<N, RowSlots, typename Cfg::RowSync, TW>(v, t_row, tw_row, slots);
                Cfg::RowSync::sync();                                     // exchange reads of this line are done
                // columns outside the band-limit tiles are never transformed by the column phase: they must hold zeros
#pragma unroll
                for (int e = 0; e < 16; ++e) slots.at(t_row + e * T) = ((amask >> e) & 1u) ? v[e] : make_float2(0.f, 0.f);
            }
            __syncthreads();
            // ------------------------------------------------------------ column phase
            const bool last = (s == n_slices - 1);
            const float2* pxt = last ? px_last : px_mid;
            if (last) {                                                   // out-of-band columns of the exit wave: exact zeros
                for (int i = threadIdx.x; i < N * gap; i += Cfg::THREADS) {
                    const int row = i / gap, col = col_lo + i % gap;
                    wout[(size_t)row * N + col] = make_float2(0.f, 0.f);
                }
            }
            for (int cg = g; cg < n_cgroups; cg += Cfg::N_CG) {
                const int ci = cg * 32 + c;                               // index into the list of active columns; the tail of the
                const int kx = ci < col_lo ? ci : (ci < n_active ? ci + gap : col_lo + (ci - n_active));   // last group takes
                const int nm = nmax[kx];                                  // out-of-band columns (zeros in, zeros out)
                const float2 pxv = pxt[kx];
                PitchSlots<LEN> slots{wave + kx + (kx >> 4)};
                float2 v[16];
#pragma unroll
                for (int e = 0; e < 16; ++e) v[e] = slots.at(t_col + e * T);
                fft_forward<N, PitchSlots<LEN>, typename Cfg::ColSync, TW>(v, t_col, tw_col, slots);
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const int iy = t_col + e * T;
                    const int n = iy < N / 2 ? iy : N - iy;
                    v[e] = (n <= nm) ? cmul(v[e], cmul(pxv, py_s[iy])) : make_float2(0.f, 0.f);
                }
                if (!last) {
                    fft_inverse<N, PitchSlots<LEN>, typename Cfg::ColSync, TW>(v, t_col, tw_col, slots);
                    Cfg::ColSync::sync();                                 // exchange reads of these columns are done
#pragma unroll
                    for (int e = 0; e < 16; ++e) slots.at(t_col + e * T) = v[e];
                } else {
#pragma unroll
                    for (int e = 0; e < 16; ++e) wout[(size_t)(t_col + e * T) * N + kx] = v[e];
                }
            }
            __syncthreads();
        }
    }
}

template <int N>
static cudaError_t launch_resident(ps_ctx* c, float2* W, const float2* psi0, const float* V, const ResWaves& rw, float sigma,
                                   int col_lo, int col_hi) {
    using Cfg = ResCfg<N>;
    auto kern = k_slice_resident<N>;
    int cap = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &cap);
    if (ce != cudaSuccess) return ce;
    const int n_waves = rw.np * rw.nf;
    kern<<<n_waves < cap ? n_waves : cap, Cfg::THREADS, Cfg::SMEM, c->stream>>>(
        W, psi0, V, c->d_nmax, c->kv.d_px_mid, c->kv.d_px_last, c->kv.d_py, rw, c->n_slices, sigma, col_lo, col_hi);
    return cudaGetLastError();
}

// true when the chip-resident kernel handles this geometry (square grid of at most 128^2)
bool resident_supported(const ps_ctx* c) { return c->nx == c->ny && c->nx <= 128; }

// the whole slice loop of waves probes [0, n_probes) x frames [0, n_frames) in one launch (ctx tables already built)
cudaError_t launch_slice_resident(ps_ctx* c, float2* W, const float2* psi0, const float* V, int n_probes, int n_frames,
                                  float sigma, int col_lo, int col_hi) {
    ResWaves rw{0, n_probes, 0, n_frames, n_frames};
    ProfScope ps_(c, K_SLICE_RESIDENT);
    switch (c->nx) {
        case 32: return launch_resident<32>(c, W, psi0, V, rw, sigma, col_lo, col_hi);
        case 64: return launch_resident<64>(c, W, psi0, V, rw, sigma, col_lo, col_hi);
        case 128: return launch_resident<128>(c, W, psi0, V, rw, sigma, col_lo, col_hi);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace psb
