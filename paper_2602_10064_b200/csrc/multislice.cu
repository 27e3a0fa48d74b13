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
    // two blocks of eight warps per SM at up to 128 registers; measured at 512^2 (config 3): four blocks of 128
    // threads the same (69.7 vs 69.2 ms per 80 slices), five blocks at 96 registers slower (75.9), six at 80 slower (82.3)
    static constexpr int MIN_BLOCKS = (THREADS <= 256) ? 2 : 1;
    static constexpr size_t SMEM = (size_t)RPB * RowLine<NX>::LEN * sizeof(float2);
    // rows are independent: only the T threads of a row synchronise (a warp, or a named barrier per row)
    using Sync = typename std::conditional<(T <= 32), WarpSync,
                                           typename std::conditional<(RPB > 1), GroupSync<T>, BlockSync>::type>::type;
};

struct ChunkMap {           // chunk of waves: probes [p0,p0+np) x frames [f0,f0+nf); local l = lf*np + lp
    int p0, np, f0, nf, F;  // F = total frames of the call (tiled exit layout, V and psi0 use p0 + lp, f0 + lf)
    // the array the wave is propagated in, [.][wF][ny][nx]: wave (lp, lf) lives at ((wp0 + lp) * wF + wf0 + lf).
    // Dense layout: the caller's exit array itself (wp0 = p0, wf0 = f0, wF = F); tiled layout: a chunk-local work
    // array in scratch (wp0 = wf0 = 0, wF = nf).
    int wp0, wf0, wF;
};

// Row coordinates of a persistent thread group: rho = (lf * np + lp) * ny + y, advanced by a constant stride per item.
// The stride is decomposed once (one integer division per kernel, none per item), so that an item costs a handful of
// integer instructions instead of the two 32-bit divisions and the 64-bit address chains it cost in round 1
// (ncu: 400 of the 1650 warp instructions of a 512-point row were index arithmetic).
struct RowCursor {
    unsigned y, lp, lf;
    __device__ __forceinline__ void init(const unsigned rho, const int ny_shift, const unsigned np) {
        y = rho & ((1u << ny_shift) - 1u);
        const unsigned l = rho >> ny_shift;
        lf = l / np;
        lp = l - lf * np;
    }
    __device__ __forceinline__ void advance(const unsigned dy, const unsigned dlp, const unsigned dlf, const int ny_shift,
                                            const unsigned np) {
        y += dy;
        lp += dlp + (y >> ny_shift);
        y &= (1u << ny_shift) - 1u;
        lf += dlf;
        if (lp >= np) { lp -= np; ++lf; }
        if (lp >= np) { lp -= np; ++lf; }                     // dlp + carry can reach np
    }
};

// PAT510: the active columns are [0, col_lo) and [col_hi, NX) with 5T < col_lo <= 6T and 10T <= col_hi < 11T (every
// grid whose band limit is set by the x direction: all five BASELINE configs).  Then the elements e = t + e T of a thread
// are active for e < 5 and e > 10, inactive for 6 <= e <= 9 (compile-time zeros in, dead values out: the compiler prunes
// the first and last butterflies accordingly), and only e = 5 and e = 10 carry a per-thread predicate.  The generic
// variant tests one bit of a mask per element.
template <int NX, bool FIRST, bool VAC /* vacuum shortcut (ps_set_vacuum_shortcut) */, bool PAT510>
__global__ void __launch_bounds__(RowCfg<NX>::THREADS, RowCfg<NX>::MIN_BLOCKS)
k_row_transmit(float2* __restrict__ W, const float2* __restrict__ psi0, const float* __restrict__ V, const ChunkMap cm,
               const int ny_shift, const int n_slices, const int slice, const float sigma, const int n_items,
               const int col_lo, const int col_hi) {
    using Cfg = RowCfg<NX>;
    constexpr int T = Cfg::T;
    using Slots = typename std::conditional<(T % 16 == 0), RowSlotsF<NX>, RowSlots>::type;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, r = threadIdx.x / T;
    Twiddles<NX> tw;
    tw.init(t);
    // bit e: column t + e T lies in an active tile.  Active tiles are [0, col_lo) and [col_hi, NX) (FFT order).
    unsigned amask = 0;
#pragma unroll
    for (int e = 0; e < 16; ++e) amask |= ((t + e * T < col_lo || t + e * T >= col_hi) ? 1u : 0u) << e;
    const bool a_lo = t + 5 * T < col_lo, a_hi = t + 10 * T >= col_hi;          // PAT510: the two boundary elements
    // 32-bit row indices (ps_multislice checks n_probes * n_frames * ny < 2^31 and n_frames * n_slices * ny < 2^31)
    const unsigned np = (unsigned)cm.np;
    const unsigned n_rows = np * (unsigned)cm.nf << ny_shift;
    const unsigned stride = gridDim.x * Cfg::RPB;
    const unsigned dy = stride & ((1u << ny_shift) - 1u), dl = stride >> ny_shift;
    const unsigned dlf = dl / np, dlp = dl - dlf * np;
    unsigned rho = blockIdx.x * Cfg::RPB + r;
    RowCursor cur;
    cur.init(rho, ny_shift, np);
    // L2 prefetch of this group's NEXT row while the current one is transformed (measured: +3 % at 512^2, +4 % at
    // 2048^2, -4 % at 256^2): one 128-byte line per thread, the T threads of a row cover the NX * 8 bytes of the wave
    // row (lines wholly inside the inactive column range are skipped) and the first T/2 the NX * 4 bytes of V
    const bool pf_wave = (16 * t < col_lo) || (16 * t + 16 > col_hi);
    // rows per block divide ny for NX >= 128 (RPB <= 32 <= ny): every item is a full set of rows
    constexpr bool ALWAYS_VALID = Cfg::RPB <= kMinGrid;

    for (int item = blockIdx.x; item < n_items; item += gridDim.x, rho += stride) {
        const bool valid = ALWAYS_VALID || rho < n_rows;
        const unsigned cur_lp = cur.lp, cur_lf = cur.lf;
        const unsigned p = cm.p0 + cur_lp, f = cm.f0 + cur_lf, y = cur.y;
        const unsigned wrow_i = ((((unsigned)cm.wp0 + cur_lp) * (unsigned)cm.wF + (unsigned)cm.wf0 + cur_lf) << ny_shift) + y;
        const unsigned vrow_i = ((f * (unsigned)n_slices + (unsigned)slice) << ny_shift) + y;
        cur.advance(dy, dlp, dlf, ny_shift, np);
        if (NX >= 512 && rho + stride < n_rows) {
            const unsigned fn = cm.f0 + cur.lf;
            const unsigned wn_i = ((((unsigned)cm.wp0 + cur.lp) * (unsigned)cm.wF + (unsigned)cm.wf0 + cur.lf) << ny_shift) + cur.y;
            const unsigned vn_i = ((fn * (unsigned)n_slices + (unsigned)slice) << ny_shift) + cur.y;
            if (2 * t < T) tma::prefetch_l2(V + (size_t)vn_i * NX + 32 * t);
            if (!FIRST && pf_wave) tma::prefetch_l2(W + (size_t)wn_i * NX + 16 * t);
        }
        float2* wrow = W + (size_t)wrow_i * NX + t;
        const float* vrow = V + (size_t)vrow_i * NX + t;
        const Slots slots = [&]() {
            if constexpr (T % 16 == 0) return RowSlotsF<NX>(smem + (size_t)r * RowLine<NX>::LEN, t);
            else return RowSlots{smem + (size_t)r * RowLine<NX>::LEN};
        }();
        unsigned am = valid ? amask : 0u;
        asm volatile("" : "+r"(am));                     // keep the mask in ONE register: bit tests, not 16 hoisted flags
        auto active = [&](const int e) -> bool {
            if constexpr (PAT510) return e < 5 || e > 10 || (e == 5 && a_lo) || (e == 10 && a_hi);
            else return (am & (1u << e)) != 0u;
        };
        float2 v[16];
        float sv[16];                                    // V of this row
        // Where V is fetched: with the wave (NX <= 256: everything fits in registers) or after the inverse transform
        // (NX >= 512: sixteen more live registers across the inverse transform would be spilled to local memory; the
        // row was pulled into L2 by the previous item's prefetch, so the load is an L2 hit the other warps cover)
        constexpr bool V_LATE = !FIRST && !VAC && NX >= 512;
        if (!V_LATE) {
#pragma unroll
            for (int e = 0; e < 16; ++e) sv[e] = valid ? __ldg(vrow + e * T) : 0.f;
        }
        if (FIRST) {
            const float2* src = psi0 + (((size_t)p << ny_shift) + y) * NX + t;
#pragma unroll
            for (int e = 0; e < 16; ++e) v[e] = valid ? __ldg(src + e * T) : make_float2(0.f, 0.f);
        } else {
#pragma unroll
            for (int e = 0; e < 16; ++e) v[e] = active(e) ? wrow[e * T] : make_float2(0.f, 0.f);
            if (VAC) {
                // V == 0 on the whole row (vacuum): exp(i sigma V) = 1 and FFT_x[IFFT_x[M]] = NX * M exactly, so the
                // row is only rescaled (NX is a power of two: no rounding).  Decided per warp (T <= 32: the rows this
                // warp carries) or per block, from the potential itself: any input with vacuum rows benefits.
                bool z = true;
#pragma unroll
                for (int e = 0; e < 16; ++e) z = z && (sv[e] == 0.f);
                const bool all_z = (T <= 32) ? (bool)__all_sync(0xffffffffu, z) : (bool)__syncthreads_and(z);
                if (all_z) {
#pragma unroll
                    for (int e = 0; e < 16; ++e)
                        if (active(e)) wrow[e * T] = make_float2(v[e].x * (float)NX, v[e].y * (float)NX);
                    continue;
                }
            }
            fft_inverse<NX, Slots, typename Cfg::Sync>(v, t, tw, slots);
            if (V_LATE) {
#pragma unroll
                for (int e = 0; e < 16; ++e) sv[e] = __ldg(vrow + e * T);
            }
        }
#pragma unroll
        for (int e = 0; e < 16; ++e) v[e] = cmul(v[e], cis_fast(sigma * sv[e]));
        fft_forward<NX, Slots, typename Cfg::Sync>(v, t, tw, slots);
        asm volatile("" : "+r"(am));                     // test the bits again rather than keep 16 flags alive (spills)
#pragma unroll
        for (int e = 0; e < 16; ++e)
            if (active(e)) wrow[e * T] = v[e];
    }
}

// ------------------------------------------------------------------------------------ row pass, potential from Zm
// ps_multislice_fused (second half; "An inverse FFT then yields the real-space
// projected potential"): the row pass takes row y of the y-transformed slice PAIR (s/2) from the mixed array Zm,
// runs the x-inverse transform itself — real part = slice 2 pr, imaginary part = slice 2 pr + 1, exactly what k_v_row
// would have written to V — parks the row of V it needs in shared memory and carries on as k_row_transmit does.  V is
// never written to or read from HBM.  Costs a third transform per row and slice; meant for single-probe runs.
template <int NX> struct RowZmCfg {
    static constexpr int T = Plan<NX>::T;
    static constexpr int THREADS = RowCfg<NX>::THREADS;
    static constexpr int RPB = RowCfg<NX>::RPB;
    static constexpr int MIN_BLOCKS = RowCfg<NX>::MIN_BLOCKS;
    static constexpr size_t SMEM = (size_t)RPB * (RowLine<NX>::LEN * sizeof(float2) + NX * sizeof(float));
    using Sync = typename RowCfg<NX>::Sync;
};

template <int NX, bool FIRST>
__global__ void __launch_bounds__(RowZmCfg<NX>::THREADS, RowZmCfg<NX>::MIN_BLOCKS)
k_row_transmit_zm(float2* __restrict__ W, const float2* __restrict__ psi0, const float2* __restrict__ Zm,
                  const int32_t* __restrict__ offsets, const int zm_f0, const int n_pairs, const int n_elem,
                  const ChunkMap cm, const int ny_shift, const int n_slices, const int slice, const float sigma,
                  const int n_items, const int col_lo, const int col_hi) {
    using Cfg = RowZmCfg<NX>;
    constexpr int T = Cfg::T;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, r = threadIdx.x / T;
    RowSlots slots{smem + (size_t)r * RowLine<NX>::LEN};
    float* svline = reinterpret_cast<float*>(smem + (size_t)Cfg::RPB * RowLine<NX>::LEN) + (size_t)r * NX;
    Twiddles<NX> tw;
    tw.init(t);
    unsigned amask = 0;
#pragma unroll
    for (int e = 0; e < 16; ++e) amask |= ((t + e * T < col_lo || t + e * T >= col_hi) ? 1u : 0u) << e;
    const unsigned np = (unsigned)cm.np;
    const unsigned n_rows = np * (unsigned)cm.nf << ny_shift;
    const unsigned stride = gridDim.x * Cfg::RPB;
    const unsigned dy = stride & ((1u << ny_shift) - 1u), dl = stride >> ny_shift;
    const unsigned dlf = dl / np, dlp = dl - dlf * np;
    unsigned rho = blockIdx.x * Cfg::RPB + r;
    RowCursor cur;
    cur.init(rho, ny_shift, np);
    const int pr = slice >> 1, part = slice & 1, n_bins = n_slices * n_elem;
    const int sa = 2 * pr, sb = 2 * pr + 1;

    for (int item = blockIdx.x; item < n_items; item += gridDim.x, rho += stride) {
        const bool valid = rho < n_rows;
        const unsigned cur_lp = cur.lp, cur_lf = cur.lf;
        const unsigned p = cm.p0 + cur_lp, f = cm.f0 + cur_lf, y = cur.y;
        const unsigned wrow_i = ((((unsigned)cm.wp0 + cur_lp) * (unsigned)cm.wF + (unsigned)cm.wf0 + cur_lf) << ny_shift) + y;
        cur.advance(dy, dlp, dlf, ny_shift, np);
        float2* wrow = W + (size_t)wrow_i * NX + t;
        unsigned am = valid ? amask : 0u;
        asm volatile("" : "+r"(am));
        // ---- V of this row: x-inverse transform of the pair's mixed row (skipped when both slices are vacuum)
        const int fl = (int)f - zm_f0;                                       // frame inside the Zm chunk
        bool any = false;
        if (valid) {
            const int32_t* off = offsets + (size_t)fl * (n_bins + 1);
            const bool has_a = off[(sa + 1) * n_elem] > off[sa * n_elem];
            const bool has_b = (sb < n_slices) && off[(sb + 1) * n_elem] > off[sb * n_elem];
            any = has_a || has_b;
        }
        float2 v[16];
        {
            const float2* zrow = Zm + ((((size_t)fl * n_pairs + pr) << ny_shift) + y) * NX + t;
#pragma unroll
            for (int e = 0; e < 16; ++e) v[e] = (any && (am & (1u << e))) ? zrow[e * T] : make_float2(0.f, 0.f);
        }
        fft_inverse<NX, RowSlots, typename Cfg::Sync>(v, t, tw, slots);
#pragma unroll
        for (int e = 0; e < 16; ++e) svline[t + e * T] = any ? (part ? v[e].y : v[e].x) : 0.f;
        // ---- the wave row (each thread re-reads the elements of V it wrote itself: no barrier needed)
        asm volatile("" : "+r"(am));
        if (FIRST) {
            const float2* src = psi0 + (((size_t)p << ny_shift) + y) * NX + t;
#pragma unroll
            for (int e = 0; e < 16; ++e) v[e] = valid ? __ldg(src + e * T) : make_float2(0.f, 0.f);
        } else {
#pragma unroll
            for (int e = 0; e < 16; ++e) v[e] = (am & (1u << e)) ? wrow[e * T] : make_float2(0.f, 0.f);
            fft_inverse<NX, RowSlots, typename Cfg::Sync>(v, t, tw, slots);
        }
#pragma unroll
        for (int e = 0; e < 16; ++e) v[e] = cmul(v[e], cis_fast(sigma * svline[t + e * T]));
        fft_forward<NX, RowSlots, typename Cfg::Sync>(v, t, tw, slots);
        asm volatile("" : "+r"(am));
#pragma unroll
        for (int e = 0; e < 16; ++e)
            if (am & (1u << e)) wrow[e * T] = v[e];
    }
}

// ------------------------------------------------------------------------------------ row pass, 32 values per thread
// NX = 512 and 1024 with the 32-value transform plan: T = NX/32 threads per row (half a warp / one warp: no block
// barrier at all), one shared-memory exchange per transform.  Used for the slices after the first when the active
// columns [0, col_lo) and [col_hi, NX) satisfy 10T <= col_lo <= 12T and 20T <= col_hi <= 22T (band limit set by the
// x direction): elements e <= 9 and e >= 22 are then always active, 12 <= e <= 19 never (compile-time zeros in, dead
// values out), and e = 10, 11, 20, 21 carry a per-thread predicate.
template <int NX> struct RowCfg32 {
    static constexpr int T = Plan32<NX>::T;
    static constexpr int THREADS = 128;
    static constexpr int RPB = THREADS / T;
    static constexpr int MIN_BLOCKS = 3;                                  // 168 registers; 2 and 4 blocks measured slower
    static constexpr size_t SMEM = (size_t)RPB * RowLine32<NX>::LEN * sizeof(float2);
};

template <int NX>
__global__ void __launch_bounds__(RowCfg32<NX>::THREADS, RowCfg32<NX>::MIN_BLOCKS)
k_row_transmit32(float2* __restrict__ W, const float* __restrict__ V, const ChunkMap cm, const int ny_shift,
                 const int n_slices, const int slice, const float sigma, const int n_items, const int col_lo,
                 const int col_hi) {
    using Cfg = RowCfg32<NX>;
    constexpr int T = Cfg::T;
    using Slots = RowSlots32<NX>;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, r = threadIdx.x / T;
    Twiddles32<NX> tw;
    tw.init(t);
    const Slots slots(smem + (size_t)r * RowLine32<NX>::LEN, t);
    const bool a10 = t + 10 * T < col_lo, a11 = t + 11 * T < col_lo, a20 = t + 20 * T >= col_hi, a21 = t + 21 * T >= col_hi;
    auto active = [&](const int e) -> bool {
        return e <= 9 || e >= 22 || (e == 10 && a10) || (e == 11 && a11) || (e == 20 && a20) || (e == 21 && a21);
    };
    const unsigned np = (unsigned)cm.np;
    const unsigned n_rows = np * (unsigned)cm.nf << ny_shift;
    const unsigned stride = gridDim.x * Cfg::RPB;
    const unsigned dy = stride & ((1u << ny_shift) - 1u), dl = stride >> ny_shift;
    const unsigned dlf = dl / np, dlp = dl - dlf * np;
    unsigned rho = blockIdx.x * Cfg::RPB + r;
    RowCursor cur;
    cur.init(rho, ny_shift, np);
    // next-row L2 prefetch: the wave row is 2T lines of 128 bytes (two per thread), the V row T lines
    const bool pf0 = (16 * t < col_lo) || (16 * t + 16 > col_hi);
    const bool pf1 = (16 * (t + T) < col_lo) || (16 * (t + T) + 16 > col_hi);

    for (int item = blockIdx.x; item < n_items; item += gridDim.x, rho += stride) {
        const unsigned cur_lp = cur.lp, cur_lf = cur.lf;
        const unsigned f = cm.f0 + cur_lf, y = cur.y;
        const unsigned wrow_i = ((((unsigned)cm.wp0 + cur_lp) * (unsigned)cm.wF + (unsigned)cm.wf0 + cur_lf) << ny_shift) + y;
        const unsigned vrow_i = ((f * (unsigned)n_slices + (unsigned)slice) << ny_shift) + y;
        cur.advance(dy, dlp, dlf, ny_shift, np);
        if (rho + stride < n_rows) {
            const unsigned fn = cm.f0 + cur.lf;
            const unsigned wn_i = ((((unsigned)cm.wp0 + cur.lp) * (unsigned)cm.wF + (unsigned)cm.wf0 + cur.lf) << ny_shift) + cur.y;
            const unsigned vn_i = ((fn * (unsigned)n_slices + (unsigned)slice) << ny_shift) + cur.y;
            tma::prefetch_l2(V + (size_t)vn_i * NX + 32 * t);
            if (pf0) tma::prefetch_l2(W + (size_t)wn_i * NX + 16 * t);
            if (pf1) tma::prefetch_l2(W + (size_t)wn_i * NX + 16 * (t + T));
        }
        float2* wrow = W + (size_t)wrow_i * NX + t;
        const float* vrow = V + (size_t)vrow_i * NX + t;
        float2 v[32];
#pragma unroll
        for (int e = 0; e < 32; ++e) v[e] = active(e) ? wrow[e * T] : make_float2(0.f, 0.f);
        fft32_inverse<NX, Slots, WarpSync>(v, tw, slots);
        {
            float sv[32];                                  // V of this row: an L2 hit (prefetched with the previous item)
#pragma unroll
            for (int e = 0; e < 32; ++e) sv[e] = __ldg(vrow + e * T);
#pragma unroll
            for (int e = 0; e < 32; ++e) v[e] = cmul(v[e], cis_fast(sigma * sv[e]));
        }
        fft32_forward<NX, Slots, WarpSync>(v, tw, slots);
#pragma unroll
        for (int e = 0; e < 32; ++e)
            if (active(e)) wrow[e * T] = v[e];
    }
}

// ------------------------------------------------------------------------------------ column pass
// A block owns C adjacent k-columns x all NY rows of one wave per item.  The tile travels
// global -> shared -> global through the TMA engine (2-D tensor map over the wave array viewed as
// float32 [P*F*ny][2 nx]); the ring of NS shared-memory stages is, in turn, TMA destination, FFT
// exchange buffer and TMA store source, so the load of item i+1 and the store of item i-1 overlap the
// transforms of item i and no register is spent on staging.
//
// E = values per thread of the transform plan (fft_core.cuh).  E = 16: NY/16 threads per column, two shared-memory
// exchanges per transform at NY >= 512.  E = 32 (NY = 512, 1024): NY/32 threads per column, ONE exchange; blocks are
// half as large (128 threads, 168 registers), three of them per SM with a 2-stage ring.  The pass is bound by the LSU
// data pipe, which every element crosses 10 (E = 16) or 6 (E = 32) times per transform pair (profiles/r2_slice_step.md).
template <int NY, int E> struct ColCfg {
    static_assert(E == 16 || (E == 32 && (NY == 512 || NY == 1024)), "32 values per thread: NY = 512 or 1024");
    static constexpr int T = NY / E;
    static constexpr int C = (E == 32) ? ((NY <= 512) ? 8 : 4) : ((NY <= 1024) ? 8 : 4);   // columns per block
    static constexpr int THREADS = C * T;
    static constexpr int NS = (E == 32) ? 2 : 3;                          // pipeline stages
    static constexpr int BOX_R = (NY < 256) ? NY : 256;                   // TMA box rows (<= 256)
    static constexpr int NBOX = NY / BOX_R;
    // E = 32: three blocks at 168 registers (two blocks x three stages at 218 registers measured 8 % slower);
    // E = 16: cap registers at 128
    static constexpr int MIN_BLOCKS = (E == 32) ? 3 : (THREADS <= 256) ? 2 : 1;
    static constexpr uint32_t STAGE_BYTES = (uint32_t)NY * C * sizeof(float2);
    static constexpr size_t SMEM = (size_t)NS * STAGE_BYTES + (size_t)NY * sizeof(float2) + NS * sizeof(uint64_t) + 128;
};

// the transform plan of a column pass: slots, twiddles, forward / inverse
template <int NY, int E, int C> struct ColFft;
template <int NY, int C> struct ColFft<NY, 16, C> {
    using Slots = ColSlots<C>;
    using TW = Twiddles<NY>;
    static __device__ __forceinline__ void forward(float2 (&v)[16], const int t, const TW& tw, const Slots& sm) {
        fft_forward<NY, Slots, BlockSync>(v, t, tw, sm);
    }
    static __device__ __forceinline__ void inverse(float2 (&v)[16], const int t, const TW& tw, const Slots& sm) {
        fft_inverse<NY, Slots, BlockSync>(v, t, tw, sm);
    }
};
template <int NY, int C> struct ColFft<NY, 32, C> {
    using Slots = ColSlots32<C, NY / 32>;
    using TW = Twiddles32<NY>;
    static __device__ __forceinline__ void forward(float2 (&v)[32], const int, const TW& tw, const Slots& sm) {
        fft32_forward<NY, Slots, BlockSync>(v, tw, sm);
    }
    static __device__ __forceinline__ void inverse(float2 (&v)[32], const int, const TW& tw, const Slots& sm) {
        fft32_inverse<NY, Slots, BlockSync>(v, tw, sm);
    }
};

// TILED (last pass only): the k-space exit wave goes to the time-tiled layout [P][ny][active tile][F][8 kx] through a
// second, 5-D tensor map instead of back into the array it was propagated in.
template <int NY, int E, bool LAST, bool TILED>
__global__ void __launch_bounds__(ColCfg<NY, E>::THREADS, ColCfg<NY, E>::MIN_BLOCKS)
k_col_propagate(const __grid_constant__ CUtensorMap wmap, const __grid_constant__ CUtensorMap tmap, const int tiles_lo,
                const int tile_gap, const int n_tiles, const int32_t* __restrict__ nmax, const float2* __restrict__ px,
                const float2* __restrict__ py, const ChunkMap cm, const int n_items) {
    using Cfg = ColCfg<NY, E>;
    constexpr int T = Cfg::T, C = Cfg::C, SUB = kColTile / C, NS = Cfg::NS;
    using Fft = ColFft<NY, E, C>;
    using Slots = typename Fft::Slots;
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
        const int row0 = ((cm.wp0 + l % cm.np) * cm.wF + cm.wf0 + l / cm.np) * NY;
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
    typename Fft::TW tw;
    tw.init(t);
    __syncthreads();
    if (threadIdx.x == 0 && blockIdx.x < n_items) issue_load(blockIdx.x, 0);   // the load runs one item ahead

    int it = 0;
    int rem = blockIdx.x % per_wave;                         // item % per_wave, kept incrementally (no division per item)
    const int rem_step = gridDim.x % per_wave;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++it) {
        const int s = it % NS;
        if (threadIdx.x == 0) {
            const int nxt = item + gridDim.x;
            if (nxt < n_items) {
                tma::bulk_wait_read<NS - 2>();                // the store that last used stage (it + 1) % NS has drained
                issue_load(nxt, (it + 1) % NS);
            }
        }
        const int tj = rem / SUB;
        const int kx0 = (tj < tiles_lo ? tj : tj + tile_gap) * kColTile + (rem % SUB) * C;
        const int kx = kx0 + c;
        const int nm = nmax[kx];
        const float2 pxv = px[kx];
        float2* st = stage0 + (size_t)s * NY * C;
        const Slots slots(st + c, t);
        tma::mbar_wait(&full[s], (it / NS) & 1);
        float2 v[E];
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = slots.at(t + e * T);
        auto propagate = [&]() {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int iy = t + e * T;
                const int n = iy < NY / 2 ? iy : NY - iy;     // |signed index|
                v[e] = (n <= nm) ? cmul(v[e], cmul(pxv, py_s[iy])) : make_float2(0.f, 0.f);
            }
        };
        // E = 32, NY = 1024: both transforms run the SAME forward code in a two-trip loop, so that the loop body of the
        // kernel fits the instruction cache (two unrolled copies of the 32-value transform do not; ncu: 10 % of the stall
        // samples were "no instruction"; measured +5 % at 1024, -8 % at 512, hence per size).  The inverse is the forward
        // transform read backwards: sum_k X[k] e^{+2 pi i n k / N} is element (-n) mod N of the forward transform of X,
        // so after the second trip canonical position j holds row (-j) mod NY, and the tile is written back with
        // reversed row addressing.
        constexpr bool LOOPED = (E == 32) && (NY == 1024) && !LAST;
        if constexpr (LOOPED) {
#pragma unroll 1
            for (int pass = 0; pass < 2; ++pass) {
                Fft::forward(v, t, tw, slots);
                if (pass == 0) propagate();
            }
        } else {
            Fft::forward(v, t, tw, slots);
            propagate();
            if (!LAST) Fft::inverse(v, t, tw, slots);
        }
        __syncthreads();                                      // exchange reads of this stage are done
        if constexpr (!LOOPED) {
#pragma unroll
            for (int e = 0; e < E; ++e) slots.at(t + e * T) = v[e];
        } else {
            // row (NY - t - e T) mod NY = (T - t) + (E - 1 - e) T, except (t, e) = (0, 0), which is row 0
            float2* const pr = st + c + (size_t)(T - t) * C;
            float2* const p0 = (t == 0) ? st + c : pr + (E - 1) * T * C;
            *p0 = v[0];
#pragma unroll
            for (int e = 1; e < E; ++e) pr[(E - 1 - e) * T * C] = v[e];
        }
        tma::fence_proxy_async();
        __syncthreads();
        if (threadIdx.x == 0) {
            const int l = item / per_wave;
            if (TILED) {
                const int p = cm.p0 + l % cm.np, f = cm.f0 + l / cm.np;
#pragma unroll
                for (int b = 0; b < Cfg::NBOX; ++b)
                    tma::tensor_store_5d(&tmap, 2 * (rem % SUB) * C, f, rem / SUB, b * Cfg::BOX_R, p,
                                         st + (size_t)b * Cfg::BOX_R * C);
            } else {
                const int row0 = ((cm.wp0 + l % cm.np) * cm.wF + cm.wf0 + l / cm.np) * NY;
#pragma unroll
                for (int b = 0; b < Cfg::NBOX; ++b)
                    tma::tensor_store_2d(&wmap, 2 * kx0, row0 + b * Cfg::BOX_R, st + (size_t)b * Cfg::BOX_R * C);
            }
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
        const int p = cm.wp0 + l % cm.np, f = cm.wf0 + l / cm.np;
        W[(((size_t)p * cm.wF + f) * ny + y) * nx + col_lo + x] = make_float2(0.f, 0.f);
    }
}

// ------------------------------------------------------------------------------------ launch helpers
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

template <int NX, bool FIRST>
static cudaError_t launch_row(ps_ctx* c, float2* W, const float2* psi0, const float* V, const ChunkMap& cm,
                              int slice, float sigma, int col_lo, int col_hi) {
    using Cfg = RowCfg<NX>;
    constexpr int T = Cfg::T;
    const bool pat510 = !FIRST && !c->vacuum_shortcut && NX >= 256 && col_lo > 5 * T && col_lo <= 6 * T && col_hi >= 10 * T &&
                        col_hi < 11 * T;
    auto kern = (c->vacuum_shortcut && !FIRST) ? k_row_transmit<NX, FIRST, true, false>
                : pat510                       ? k_row_transmit<NX, FIRST, false, (!FIRST && NX >= 256)>
                                               : k_row_transmit<NX, FIRST, false, false>;
    int per_sm_grid = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &per_sm_grid);
    if (ce != cudaSuccess) return ce;
    const long long n_rows = (long long)cm.np * cm.nf * c->ny;
    const int n_items = (int)((n_rows + Cfg::RPB - 1) / Cfg::RPB);
    const int grid = n_items < per_sm_grid ? n_items : per_sm_grid;
    int ny_shift = 0;
    while ((1 << ny_shift) < c->ny) ++ny_shift;
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(W, psi0, V, cm, ny_shift, c->n_slices, slice, sigma, n_items, col_lo,
                                                      col_hi);
    return cudaGetLastError();
}

template <int NX, bool FIRST>
static cudaError_t launch_row_zm(ps_ctx* c, float2* W, const float2* psi0, const VSrc& src, const ChunkMap& cm, int slice,
                                 float sigma, int col_lo, int col_hi) {
    using Cfg = RowZmCfg<NX>;
    auto kern = k_row_transmit_zm<NX, FIRST>;
    int per_sm_grid = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &per_sm_grid);
    if (ce != cudaSuccess) return ce;
    const long long n_rows = (long long)cm.np * cm.nf * c->ny;
    const int n_items = (int)((n_rows + Cfg::RPB - 1) / Cfg::RPB);
    const int grid = n_items < per_sm_grid ? n_items : per_sm_grid;
    int ny_shift = 0;
    while ((1 << ny_shift) < c->ny) ++ny_shift;
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(W, psi0, src.Zm, src.off, src.zm_f0, (c->n_slices + 1) / 2, c->n_elem, cm,
                                                      ny_shift, c->n_slices, slice, sigma, n_items, col_lo, col_hi);
    return cudaGetLastError();
}

template <int NX>
static cudaError_t launch_row32(ps_ctx* c, float2* W, const float* V, const ChunkMap& cm, int slice, float sigma, int col_lo,
                                int col_hi) {
    using Cfg = RowCfg32<NX>;
    auto kern = k_row_transmit32<NX>;
    int per_sm_grid = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &per_sm_grid);
    if (ce != cudaSuccess) return ce;
    const long long n_rows = (long long)cm.np * cm.nf * c->ny;
    const int n_items = (int)(n_rows / Cfg::RPB);                       // RPB <= 8 divides ny
    const int grid = n_items < per_sm_grid ? n_items : per_sm_grid;
    int ny_shift = 0;
    while ((1 << ny_shift) < c->ny) ++ny_shift;
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(W, V, cm, ny_shift, c->n_slices, slice, sigma, n_items, col_lo, col_hi);
    return cudaGetLastError();
}

// the row pass of slices s > 0 with the 32-value plan (ps_set_tuning "row32": 1 on where available; 0 auto = off:
// measured 10 % slower than the 16-value pass at 512^2 and 1024^2, its 12 warps per SM do not cover the load latency)
static bool use_row32(const ps_ctx* c, int col_lo, int col_hi) {
    if (!(c->nx == 512 || c->nx == 1024) || c->tune_row32 < 1 || c->vacuum_shortcut) return false;
    const int T = c->nx / 32;
    return col_lo >= 10 * T && col_lo <= 12 * T && col_hi >= 20 * T && col_hi <= 22 * T;
}

template <int NY, int E, bool LAST, bool TILED = false>
static cudaError_t launch_col(ps_ctx* c, const CUtensorMap& wmap, const CUtensorMap& tmap, const ChunkMap& cm, int zero_lo,
                              int zero_hi) {
    using Cfg = ColCfg<NY, E>;
    auto kern = k_col_propagate<NY, E, LAST, TILED>;
    int per_sm_grid = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &per_sm_grid);
    if (ce != cudaSuccess) return ce;
    const int n_tiles = c->n_tiles_active;
    const int n_items = cm.np * cm.nf * n_tiles * (kColTile / Cfg::C);
    const int grid = n_items < per_sm_grid ? n_items : per_sm_grid;
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(wmap, tmap, zero_lo / kColTile, (zero_hi - zero_lo) / kColTile, n_tiles, c->d_nmax,
                                                      LAST ? c->kv.d_px_last : c->kv.d_px_mid, c->kv.d_py, cm, n_items);
    return cudaGetLastError();
}

// column pass of size ny: 32 values per thread where available and wanted, 16 otherwise
template <bool LAST, bool TILED>
static cudaError_t launch_col_any(ps_ctx* c, bool col32, const CUtensorMap& wmap, const CUtensorMap& tmap, const ChunkMap& cm,
                                  int zero_lo, int zero_hi) {
    cudaError_t e = cudaErrorInvalidValue;
    if (col32 && c->ny == 512) return launch_col<512, 32, LAST, TILED>(c, wmap, tmap, cm, zero_lo, zero_hi);
    if (col32 && c->ny == 1024) return launch_col<1024, 32, LAST, TILED>(c, wmap, tmap, cm, zero_lo, zero_hi);
    PSB_DISPATCH_N(c->ny, (e = launch_col<N_, 16, LAST, TILED>(c, wmap, tmap, cm, zero_lo, zero_hi)));
    return e;
}

// the column pass of this grid uses the 32-value plan (ps_set_tuning "col32": 0 auto, 1 on where available, -1 off)
static bool use_col32(const ps_ctx* c) { return (c->ny == 512 || c->ny == 1024) && c->tune_col32 >= 0; }

template <int NY>
static bool make_wave_map(CUtensorMap* map, void* W, int nx, long long rows, bool col32) {
    if constexpr (NY == 512 || NY == 1024) {
        if (col32) return tma::make_map_2d_f32(map, W, 2ull * nx, (uint64_t)rows, 2 * ColCfg<NY, 32>::C, ColCfg<NY, 32>::BOX_R);
    }
    using Cfg = ColCfg<NY, 16>;
    return tma::make_map_2d_f32(map, W, 2ull * nx, (uint64_t)rows, 2 * Cfg::C, Cfg::BOX_R);
}


static constexpr long long kResidentMaxWaves = 2 * kNumSM;   // auto rule of the chip-resident path

// scratch for the chunk-local work array of the tiled exit layout: the installed workspace, else the library-owned
// buffer under the same budget rule as ps_build_slices (an eighth of the free device memory, 768 MB ... 16 GB, decided
// once per context); returns the number of waves it holds
static ps_status tiled_work_buffer(ps_ctx* c, long long n_waves_wanted, float2** W, long long* n_waves) {
    const size_t per_wave = (size_t)c->nx * c->ny * sizeof(float2);
    if (c->user_ws) {
        *n_waves = (long long)(c->user_ws_bytes / per_wave);
        if (*n_waves < 1) return fail(c, PS_EWORKSPACE, "ps_multislice: workspace smaller than one wave (tiled exit layout)");
        *W = (float2*)c->user_ws;
    } else {
        if (c->scratch_budget == 0) {
            size_t free_b = 0, total_b = 0;
            c->scratch_budget = (size_t)768 << 20;
            if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
                size_t want = (free_b + c->scratch.bytes) / 8;
                if (want > ((size_t)16 << 30)) want = (size_t)16 << 30;
                if (want > c->scratch_budget) c->scratch_budget = want;
            }
        }
        size_t avail = c->scratch_budget > c->scratch.bytes ? c->scratch_budget : c->scratch.bytes;
        long long nw = (long long)(avail / per_wave);
        if (nw < 1) nw = 1;
        if (nw > n_waves_wanted) nw = n_waves_wanted;
        ps_status st = ensure_buf(c, c->scratch, (size_t)nw * per_wave);
        if (st != PS_OK) return st;
        *n_waves = nw;
        *W = (float2*)c->scratch.p;
    }
    if (*n_waves > n_waves_wanted) *n_waves = n_waves_wanted;
    return PS_OK;
}

// tiled exit layout -> dense [P][F][ny][nx] (zeros outside the stored tiles): for consumers that take the dense
// layout only, and for parity tests.  One thread per complex value of the dense array.
__global__ void k_exit_to_dense(const float2* __restrict__ Tl, float2* __restrict__ D, const int32_t* __restrict__ tile_slot,
                                const int nx, const int ny, const int n_tiles, const int F, const long long total) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(i % nx);
        long long r = i / nx;
        const int y = (int)(r % ny); r /= ny;
        const int f = (int)(r % F);
        const long long p = r / F;
        const int tj = tile_slot[x / kColTile];
        D[i] = tj < 0 ? make_float2(0.f, 0.f)
                      : Tl[((((size_t)p * ny + y) * n_tiles + tj) * F + f) * kColTile + (x % kColTile)];
    }
}

}  // namespace psb
using namespace psb;

extern "C" size_t ps_exit_bytes(const ps_ctx* c, int n_probes, int n_frames, int exit_layout) {
    if (!c || !c->have_geom || n_probes < 1 || n_frames < 1) return 0;
    if (exit_layout == PS_LAYOUT_DENSE) return (size_t)n_probes * n_frames * c->nx * c->ny * sizeof(float2);
    if (exit_layout == PS_LAYOUT_TILED_APERTURE)
        return (size_t)n_probes * c->ny * c->n_tiles_active * n_frames * kColTile * sizeof(float2);
    return 0;
}

extern "C" ps_status ps_exit_to_dense(ps_ctx* c, const void* d_tiled, int n_probes, int n_frames, void* d_dense) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_exit_to_dense: ps_set_geometry has not been called");
    if (!d_tiled || !d_dense || n_probes < 1 || n_frames < 1) return fail(c, PS_EINVAL, "ps_exit_to_dense: null pointer or non-positive size");
    ps_status st = enter(c, "ps_exit_to_dense");
    if (st != PS_OK) return st;
    const long long total = (long long)n_probes * n_frames * c->nx * c->ny;
    const long long nb = (total + 255) / 256;
    k_exit_to_dense<<<(unsigned)(nb < 148 * 64 ? nb : 148 * 64), 256, 0, c->stream>>>(
        (const float2*)d_tiled, (float2*)d_dense, c->d_tile_slot, c->nx, c->ny, c->n_tiles_active, n_frames, total);
    PSB_LAUNCH_CHECK(c, "k_exit_to_dense");
    return PS_OK;
}

extern "C" ps_status ps_multislice(ps_ctx* c, double kV, const void* d_psi0, int n_probes, const float* d_V,
                                   int n_frames, void* d_exit, int exit_layout) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_multislice: ps_set_geometry has not been called");
    if (!d_psi0 || !d_V || !d_exit || n_probes < 1 || n_frames < 1 || !(kV > 0.0))
        return fail(c, PS_EINVAL, "ps_multislice: null pointer or non-positive size / voltage");
    if (exit_layout != PS_LAYOUT_DENSE && exit_layout != PS_LAYOUT_TILED_APERTURE)
        return fail(c, PS_EUNSUPPORTED, "ps_multislice: unknown exit layout");
    ps_status st = enter(c, "ps_multislice");
    if (st != PS_OK) return st;
    VSrc src;
    src.V = d_V;
    return multislice_range(c, kV, d_psi0, n_probes, src, n_frames, 0, n_frames, d_exit, exit_layout);
}

// The slice loop of frames [fr0, fr0 + fr_n) of an exit array laid out for n_frames frames.  ps_multislice runs the whole
// range with the potential taken from V; ps_multislice_fused calls it once per frame chunk with the chunk's mixed array.
ps_status psb::multislice_range(ps_ctx* c, double kV, const void* d_psi0, int n_probes, const VSrc& src, int n_frames,
                                int fr0, int fr_n, void* d_exit, int exit_layout) {
    const bool tiled = exit_layout == PS_LAYOUT_TILED_APERTURE;
    const float* d_V = src.V;
    ps_status st;
    if ((st = ensure_kv(c, kV)) != PS_OK) return st;

    const long long wave_rows = (long long)n_probes * n_frames * c->ny;
    if (wave_rows > 0x7fffffffLL) return fail(c, PS_EUNSUPPORTED, "ps_multislice: n_probes*n_frames*ny exceeds 2^31");
    if ((long long)n_frames * c->n_slices * c->ny > 0x7fffffffLL)
        return fail(c, PS_EUNSUPPORTED, "ps_multislice: n_frames*n_slices*ny exceeds 2^31 (propagate the frames in chunks)");

    // Waves per launch.  Measured on B200 (c2, 256^2, 512 waves; profiles/r1_chunk_sweep.md): streaming the whole
    // batch from HBM in one launch per pass beats L2-resident chunks of 40-80 MB, whose launches are too short
    // to amortise launch latency, twiddle set-up and the last partial wave of blocks.  Default: no chunking in the
    // dense layout (the wave is propagated inside the caller's array); the tiled layout propagates chunk by chunk in a
    // work array that lives in scratch, as many waves at a time as it holds.
    float2* W = (float2*)d_exit;
    long long chunk = c->wave_chunk;
    if (chunk <= 0) chunk = (long long)n_probes * fr_n;
    if (tiled) {
        long long held = 0;
        if ((st = tiled_work_buffer(c, chunk, &W, &held)) != PS_OK) return st;
        if (held < chunk) chunk = held;
    }
    const int np = (int)(n_probes < chunk ? n_probes : chunk);
    int nf = (int)(chunk / np);
    if (nf < 1) nf = 1;
    if (nf > fr_n) nf = fr_n;
    if (nf < fr_n) {                                         // equal-sized frame chunks (no short tail chunk)
        const int n_chunks = (fr_n + nf - 1) / nf;
        nf = (fr_n + n_chunks - 1) / n_chunks;
    }
    const float2* psi0 = (const float2*)d_psi0;
    const float sigma = (float)c->kv.sigma;
    const int S = c->n_slices;

    // TMA view of the array the wave is propagated in: float32 [waves*ny][2 nx]; box = C columns x up to 256 rows
    CUtensorMap wmap, tmap;
    memset(&tmap, 0, sizeof(tmap));
    bool map_ok = false;
    const bool col32 = use_col32(c);
    const long long w_rows = tiled ? (long long)np * nf * c->ny : wave_rows;
    PSB_DISPATCH_N(c->ny, (map_ok = make_wave_map<N_>(&wmap, W, c->nx, w_rows, col32)));
    if (!map_ok) return fail(c, PS_ECUDA, "ps_multislice: cuTensorMapEncodeTiled failed (exit-wave array must be 16-byte aligned)");
    if (tiled) {
        // [P][ny][active tile][F][8 kx] as float32, innermost first: (16, F, n_tiles, ny, P); box = one column (sub)tile x
        // up to 256 rows of one frame
        // columns per block of the column pass that will run (ColCfg<NY, E>::C)
        const int Cc = (col32 && c->ny == 512) ? ColCfg<512, 32>::C : (col32 && c->ny == 1024) ? ColCfg<1024, 32>::C
                       : (c->ny == 2048) ? ColCfg<2048, 16>::C : ColCfg<1024, 16>::C;
        const uint64_t dims[5] = {2ull * kColTile, (uint64_t)n_frames, (uint64_t)c->n_tiles_active, (uint64_t)c->ny, (uint64_t)n_probes};
        const uint64_t row_b = 2ull * kColTile * sizeof(float);
        const uint64_t strides[4] = {row_b, row_b * n_frames, row_b * n_frames * c->n_tiles_active,
                                     row_b * n_frames * c->n_tiles_active * c->ny};
        const uint32_t box[5] = {2u * Cc, 1u, 1u, (uint32_t)(c->ny < 256 ? c->ny : 256), 1u};
        if (!tma::make_map_5d_f32(&tmap, d_exit, dims, strides, box))
            return fail(c, PS_ECUDA, "ps_multislice: cuTensorMapEncodeTiled failed for the tiled exit layout (array must be 16-byte aligned)");
    }
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
    if (!tiled && d_V && fr0 == 0 && fr_n == n_frames && resident_supported(c) && !c->vacuum_shortcut && c->wave_chunk == 0 &&
        (c->tune_resident == 1 || (c->tune_resident == 0 && (long long)n_probes * n_frames <= kResidentMaxWaves))) {
        cudaError_t e = launch_slice_resident(c, W, psi0, d_V, n_probes, n_frames, sigma, zero_lo, zero_hi);
        if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_slice_resident: ") + cudaGetErrorString(e));
        c->launches++;
        return PS_OK;
    }

    const bool row32 = d_V && use_row32(c, zero_lo, zero_hi);
    for (int p0 = 0; p0 < n_probes; p0 += np) {
        for (int f0 = fr0; f0 < fr0 + fr_n; f0 += nf) {
            ChunkMap cm;
            cm.p0 = p0; cm.np = (n_probes - p0 < np) ? n_probes - p0 : np;
            cm.f0 = f0; cm.nf = (fr0 + fr_n - f0 < nf) ? fr0 + fr_n - f0 : nf;
            cm.F = n_frames;
            if (tiled) { cm.wp0 = 0; cm.wf0 = 0; cm.wF = cm.nf; }
            else       { cm.wp0 = cm.p0; cm.wf0 = cm.f0; cm.wF = n_frames; }
            for (int s = 0; s < S; ++s) {
                cudaError_t e = cudaErrorInvalidValue;
                {
                ProfScope ps_(c, K_ROW_TRANSMIT);
                if (!d_V) {                                          // potential from the mixed array (ps_multislice_fused)
                    if (s == 0) { PSB_DISPATCH_N(c->nx, (e = launch_row_zm<N_, true>(c, W, psi0, src, cm, s, sigma, zero_lo, zero_hi))); }
                    else        { PSB_DISPATCH_N(c->nx, (e = launch_row_zm<N_, false>(c, W, psi0, src, cm, s, sigma, zero_lo, zero_hi))); }
                }
                else if (s == 0) { PSB_DISPATCH_N(c->nx, (e = launch_row<N_, true>(c, W, psi0, d_V, cm, s, sigma, zero_lo, zero_hi))); }
                else if (row32 && c->nx == 512) e = launch_row32<512>(c, W, d_V, cm, s, sigma, zero_lo, zero_hi);
                else if (row32 && c->nx == 1024) e = launch_row32<1024>(c, W, d_V, cm, s, sigma, zero_lo, zero_hi);
                else        { PSB_DISPATCH_N(c->nx, (e = launch_row<N_, false>(c, W, psi0, d_V, cm, s, sigma, zero_lo, zero_hi))); }
                }
                if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_row_transmit: ") + cudaGetErrorString(e));
                c->launches++;
                e = cudaErrorInvalidValue;
                {
                ProfScope ps_(c, K_COL_PROPAGATE);
                if (s == S - 1 && tiled) {
                    e = launch_col_any<true, true>(c, col32, wmap, tmap, cm, zero_lo, zero_hi);
                } else if (s == S - 1) {
                    if (zero_hi > zero_lo) {
                        const long long tot = (long long)cm.np * cm.nf * c->ny * (zero_hi - zero_lo);
                        const int zb = (int)((tot + 255) / 256 < 148 * 16 ? (tot + 255) / 256 : 148 * 16);
                        k_zero_cols<<<zb, 256, 0, c->stream>>>(W, c->nx, c->ny, zero_lo, zero_hi, cm);
                        c->launches++;
                    }
                    e = launch_col_any<true, false>(c, col32, wmap, tmap, cm, zero_lo, zero_hi);
                } else {
                    e = launch_col_any<false, false>(c, col32, wmap, tmap, cm, zero_lo, zero_hi);
                }
                }
                if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_col_propagate: ") + cudaGetErrorString(e));
                c->launches++;
            }
        }
    }
    return PS_OK;
}
