// potential.cu — ps_build_slices: projected potential of every slice of every frame (§2.2):
//     V_s(k) = sum_{j in slice s} f_Zj(|k|) exp(-2 pi i k.r_j),   V_s(r) = inverse FFT of V_s(k)
// with f(q) = sum a_i/(q^2+b_i) + sum c_i exp(-d_i q^2) tabulated per element on the band-limited
// half plane (A2, A5, A10).  Pipeline per chunk of frames:
//   k_bin      float32 positions -> 2^-32 fixed-point fractions, slice index, (slice, element) key   (a0)
//   k_sort     stable counting sort of each frame's atoms by key (one warp per frame, deterministic)
//   k_vk       structure factor x form factor on the in-aperture half plane, direct separable sum    (a2)
//   k_v_col    Hermitian completion + two slices packed as re/im + inverse column FFT                (a3)
//   k_v_row    inverse row FFT, unpack -> V[f][s][ny][nx] float32 (V*Angstrom)
// Phases are formed as (m * U) mod 2^32 in integer arithmetic, so their error does not grow with |m|.
#include <functional>
#include <type_traits>

#include "common.cuh"
#include "fft_core.cuh"

namespace psb {

// ------------------------------------------------------------------------------------ a0: ingest
__global__ void k_check_Z(const int32_t* __restrict__ Z, const int n_atoms, const int32_t* __restrict__ elem_of_Z,
                          int* __restrict__ flag) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_atoms) return;
    const int z = Z[j];
    if (z < 1 || z > 127 || elem_of_Z[z] < 0) atomicExch(flag, z == 0 ? -1 : z);
}

__device__ __forceinline__ uint32_t to_fixed(const float pos, const double L) {
    const double q = __ddiv_rn((double)pos, L);
    const double u = __dsub_rn(q, floor(q));
    double U = floor(__dmul_rn(u, 4294967296.0));
    if (U > 4294967295.0) U = 4294967295.0;
    return (uint32_t)U;
}

__global__ void k_bin(const float* __restrict__ pos, const int32_t* __restrict__ Z,
                      const int32_t* __restrict__ elem_of_Z, const long long n_total, const int n_atoms,
                      const double Lx, const double Ly, const double Lz, const int n_slices, const int n_elem,
                      uint32_t* __restrict__ Ux, uint32_t* __restrict__ Uy, int32_t* __restrict__ key,
                      int32_t* __restrict__ slice_idx, int* __restrict__ async_err, int* __restrict__ bad_dev) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_total) return;
    const int j = (int)(i % n_atoms);
    const float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
    Ux[i] = to_fixed(x, Lx);
    Uy[i] = to_fixed(y, Ly);
    const uint32_t Uz = to_fixed(z, Lz);
    const int s = (int)(((unsigned long long)Uz * (unsigned long long)n_slices) >> 32);
    const int zz = Z[j];
    const int e = (zz >= 1 && zz <= 127) ? elem_of_Z[zz] : -1;
    key[i] = (e >= 0) ? s * n_elem + e : -1;
    if (e < 0) {
        *(volatile int*)bad_dev = 1;                                       // device word: k_poison of this chunk reads it
        *(volatile int*)async_err = (zz == 0) ? -1 : zz; __threadfence_system();   // mapped host word (ps_ctx)
    }
    if (slice_idx) slice_idx[i] = s;
}

// NaN-fills `dst` when the device error word is set (unknown atomic number in this or an earlier, still unreported
// ps_build_slices); returns at once otherwise.
__global__ void k_poison(float4* __restrict__ dst, const size_t n4, const int* __restrict__ bad_dev) {
    if (*(volatile const int*)bad_dev == 0) return;
    const float q = __int_as_float(0x7fc00000);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x)
        dst[i] = make_float4(q, q, q, q);
}

// One block per frame, W warps: warp w owns the contiguous atom segment [w*seg, (w+1)*seg).  Per-warp histograms,
// a (bin-major, warp-minor) exclusive scan, then every warp places its own segment in order: a stable counting
// sort, so the order of atoms inside a (slice, element) bin — and with it every float sum downstream — is fixed.
__global__ void __launch_bounds__(1024)
k_sort(const uint32_t* __restrict__ Ux, const uint32_t* __restrict__ Uy, const int32_t* __restrict__ key,
       const int n_atoms, const int n_bins, uint32_t* __restrict__ sUx, uint32_t* __restrict__ sUy,
       int32_t* __restrict__ offsets) {
    extern __shared__ int sm_sort[];                      // [W][n_bins] cursors, then [n_bins + 1] bin starts
    const int f = blockIdx.x, lane = threadIdx.x & 31, w = threadIdx.x >> 5, W = blockDim.x >> 5;
    int* cursor = sm_sort + (size_t)w * n_bins;
    int* start = sm_sort + (size_t)W * n_bins;
    const size_t base = (size_t)f * n_atoms;
    const int seg = (n_atoms + W - 1) / W;
    const int j_lo = min(w * seg, n_atoms), j_hi = min(j_lo + seg, n_atoms);
    for (int i = threadIdx.x; i < W * n_bins; i += blockDim.x) sm_sort[i] = 0;
    __syncthreads();
    for (int j = j_lo + lane; j < j_hi; j += 32) {
        const int k = key[base + j];
        if (k >= 0) atomicAdd(&cursor[k], 1);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < n_bins; b += blockDim.x) {      // per bin: prefix over warps, total
        int run = 0;
        for (int ww = 0; ww < W; ++ww) {
            const int t = sm_sort[(size_t)ww * n_bins + b];
            sm_sort[(size_t)ww * n_bins + b] = run;
            run += t;
        }
        start[b] = run;
    }
    __syncthreads();
    if (w == 0) {                                         // exclusive scan of the bin totals, 32 bins at a time
        int carry = 0;
        for (int b0 = 0; b0 <= n_bins; b0 += 32) {
            const int b = b0 + lane;
            const int cnt = (b < n_bins) ? start[b] : 0;
            int incl = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += o;
            }
            if (b <= n_bins) {
                start[b] = carry + incl - cnt;
                offsets[(size_t)f * (n_bins + 1) + b] = carry + incl - cnt;
            }
            carry += __shfl_sync(0xffffffffu, incl, 31);
        }
    }
    __syncthreads();
    for (int b = lane; b < n_bins; b += 32) cursor[b] += start[b];
    __syncwarp();
    for (int j0 = j_lo; j0 < j_hi; j0 += 32) {
        const int j = j0 + lane;
        const int k = (j < j_hi) ? key[base + j] : -1;
        const unsigned grp = __match_any_sync(0xffffffffu, k);
        const int rank = __popc(grp & ((1u << lane) - 1u));
        int dst = -1;
        if (k >= 0) dst = cursor[k] + rank;
        __syncwarp();
        if (k >= 0 && rank == __popc(grp) - 1) cursor[k] += __popc(grp);
        __syncwarp();
        if (dst >= 0) {
            sUx[base + dst] = Ux[base + j];
            sUy[base + dst] = Uy[base + j];
        }
    }
}

// ------------------------------------------------------------------------------------ a2: V(k) assembly
// Separable direct sum on the quarter plane m >= 0, n >= 0.  With theta_x = 2 pi m u_x, theta_y = 2 pi n u_y,
//     exp(-2 pi i k.r) = (cx cy - sx sy) - i (sx cy + cx sy)            at (+m, n)
//                      = (cx cy + sx sy) - i (cx sy - sx cy)            at (-m, n)
// so the four real sums  cc = sum cx cy, ss = sum sx sy, cs = sum cx sy, sc = sum sx cy  over the atoms of one
// (slice, element) give both columns +m and -m of the Hermitian half plane: 4 FMA per atom per pair of outputs.
constexpr int VK_TM = 64, VK_TN = 32, VK_CH = 32, VK_THREADS = 128;

__device__ __forceinline__ float2 phase_cs(const int m, const uint32_t U) {
    // (cos, sin) of 2 pi m u, u = U/2^32: the fraction (m*U mod 2^32) is formed exactly in integers, read as a
    // signed turn in [-1/2, 1/2) and handed to the SFU sine / cosine (abs. error 2^-21.4 on [-pi, pi]).
    const int32_t ph = (int32_t)((uint32_t)m * U);
    const float r = (float)ph * 1.4629180792671596e-9f;             // 2 pi / 2^32
    return make_float2(__cosf(r), __sinf(r));
}

__global__ void __launch_bounds__(VK_THREADS, 4)
k_vk(const uint32_t* __restrict__ sUx, const uint32_t* __restrict__ sUy, const int32_t* __restrict__ offsets,
     const float* __restrict__ ftab, const int32_t* __restrict__ nmax, float2* __restrict__ Vk, const int n_atoms,
     const int n_slices, const int n_elem, const int mcut, const int ncut, const int tiles_m) {
    __shared__ __align__(16) float2 ex[VK_CH][VK_TM];                      // (cos, sin) of 2 pi m u_x
    __shared__ __align__(16) float2 ey[VK_CH][VK_TN];                      // (cos, sin) of 2 pi n u_y
    const int f = blockIdx.z, s = blockIdx.y;
    const int tmx = blockIdx.x % tiles_m, tny = blockIdx.x / tiles_m;
    const int m0 = tmx * VK_TM, n0 = tny * VK_TN;
    const int mw = 2 * mcut + 1, nh = ncut + 1;
    const int n_bins = n_slices * n_elem;
    const int32_t* off = offsets + (size_t)f * (n_bins + 1) + (size_t)s * n_elem;
    if (off[n_elem] == off[0]) return;                                     // empty slice: Vk left unwritten
    // warp w owns the 32 x 16 sub-tile (m: 32 * (w & 1), n: 16 * (w >> 1)); lane -> 4 x 4 register tile
    const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
    const int tx = (lane & 7) + 8 * (wrp & 1), ty = (lane >> 3) + 4 * (wrp >> 1);
    const size_t abase = (size_t)f * n_atoms;
    float2* out = Vk + ((size_t)f * n_slices + s) * nh * mw;

    // is any point of this tile inside the aperture?  (nmax is even in m: column m >= 0 is FFT index m)
    int inside = 0;
    if (threadIdx.x < VK_TM) {
        const int m = m0 + threadIdx.x;
        if (m <= mcut) inside = nmax[m] >= n0;
    }
    if (!__syncthreads_or(inside)) return;                                 // never read by k_v_col
    // warp-uniform: does this warp's 32 x 16 sub-tile touch the aperture?  (A(k) = 0 there otherwise)
    bool warp_in = false;
    {
        const int m = m0 + 32 * (wrp & 1) + lane, nlo = n0 + 16 * (wrp >> 1);
        warp_in = __any_sync(0xffffffffu, (m <= mcut) && (nmax[m] >= nlo));
    }
    bool first = true;
    for (int e = 0; e < n_elem; ++e) {
        const int jb = off[e], je = off[e + 1];
        if (jb == je) continue;
        float cc[4][4], ss[4][4], cs[4][4], sc[4][4];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) cc[a][b] = ss[a][b] = cs[a][b] = sc[a][b] = 0.f;
        for (int j0 = jb; j0 < je; j0 += VK_CH) {
            const int cnt = min(VK_CH, je - j0);
            __syncthreads();
            for (int i = threadIdx.x; i < cnt * VK_TM; i += VK_THREADS) {
                const int jj = i / VK_TM, a = i % VK_TM;
                ex[jj][a] = phase_cs(m0 + a, sUx[abase + j0 + jj]);
            }
            for (int i = threadIdx.x; i < cnt * VK_TN; i += VK_THREADS) {
                const int jj = i / VK_TN, b = i % VK_TN;
                ey[jj][b] = phase_cs(n0 + b, sUy[abase + j0 + jj]);
            }
            __syncthreads();
            if (warp_in)
#pragma unroll 2
            for (int jj = 0; jj < cnt; ++jj) {
                const float4 x01 = *reinterpret_cast<const float4*>(&ex[jj][tx * 4]);
                const float4 x23 = *reinterpret_cast<const float4*>(&ex[jj][tx * 4 + 2]);
                const float4 y01 = *reinterpret_cast<const float4*>(&ey[jj][ty * 4]);
                const float4 y23 = *reinterpret_cast<const float4*>(&ey[jj][ty * 4 + 2]);
                const float cx[4] = {x01.x, x01.z, x23.x, x23.z}, sx[4] = {x01.y, x01.w, x23.y, x23.w};
                const float cy[4] = {y01.x, y01.z, y23.x, y23.z}, sy[4] = {y01.y, y01.w, y23.y, y23.w};
#pragma unroll
                for (int a = 0; a < 4; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        cc[a][b] = fmaf(cx[a], cy[b], cc[a][b]);
                        ss[a][b] = fmaf(sx[a], sy[b], ss[a][b]);
                        cs[a][b] = fmaf(cx[a], sy[b], cs[a][b]);
                        sc[a][b] = fmaf(sx[a], cy[b], sc[a][b]);
                    }
            }
        }
        if (warp_in) {
            const float* ft = ftab + (size_t)e * nh * mw;
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const int m = m0 + tx * 4 + a, n = n0 + ty * 4 + b;
                    if (m <= mcut && n <= ncut) {
                        float2* op = out + (size_t)n * mw + (mcut + m);
                        float2* om = out + (size_t)n * mw + (mcut - m);
                        const float fv = __ldg(ft + (size_t)n * mw + (mcut + m));     // f(|k|) A(k): even in m
                        float2 vp = make_float2(fv * (cc[a][b] - ss[a][b]), -fv * (cs[a][b] + sc[a][b]));
                        float2 vm = make_float2(fv * (cc[a][b] + ss[a][b]), fv * (sc[a][b] - cs[a][b]));
                        if (!first) {                                      // later elements add to the first one's
                            const float2 p0 = *op, m0v = *om;
                            vp.x += p0.x; vp.y += p0.y; vm.x += m0v.x; vm.y += m0v.y;
                        }
                        *op = vp;
                        if (m > 0) *om = vm;
                    }
                }
        }
        first = false;
    }
}

// ------------------------------------------------------------------------------------ a3: inverse FFT of slice pairs
template <int NY> struct VColCfg {
    static constexpr int T = Plan<NY>::T;
    static constexpr int C = (NY <= 1024) ? 8 : 4;
    static constexpr int THREADS = C * T;
    // up to 1024: 1024 threads per SM at 64 registers — the gather is latency-bound, and twice the warps of the
    // 128-register build cover more of it (measured per 64 frames: 512^2 2.07 -> 1.96 ms, 1024^2 12.1 -> 9.8 ms; at
    // 2048^2 the 64-register build spills 144 bytes and loses, 19.3 -> 21.6 ms, so it keeps 512 threads per SM)
    static constexpr int PER_SM = (NY <= 1024) ? 1024 : 512;
    static constexpr int MIN_BLOCKS = (THREADS >= PER_SM) ? 1 : (PER_SM / THREADS > 4 ? 4 : PER_SM / THREADS);
    static constexpr size_t SMEM = (size_t)NY * C * sizeof(float2);
};

// reads the half-plane box of Va (slice 2*pr) and Vb (slice 2*pr+1), forms z = Va + i Vb on the full
// plane by Hermitian symmetry, inverse-transforms along y, writes the mixed array Zm[f][pr][y][kx].
template <int NY>
__global__ void __launch_bounds__(VColCfg<NY>::THREADS, VColCfg<NY>::MIN_BLOCKS)
k_v_col(const float2* __restrict__ Vk, const int32_t* __restrict__ offsets, float2* __restrict__ Zm, const int nx,
        const int32_t* __restrict__ tiles, const int n_tiles, const int32_t* __restrict__ nmax, const int n_slices,
        const int n_elem, const int mcut, const int ncut, const int n_pairs, const int n_items) {
    using Cfg = VColCfg<NY>;
    constexpr int T = Cfg::T, C = Cfg::C, SUB = kColTile / C;
    extern __shared__ float2 smem[];
    const int c = threadIdx.x % C, t = threadIdx.x / C;
    ColSlots<C> slots(smem + c, t);
    Twiddles<NY> tw;
    tw.init(t);
    const int per_pair = n_tiles * SUB;
    const int mw = 2 * mcut + 1, nh = ncut + 1, n_bins = n_slices * n_elem;
    // item-invariant part of the gather: row iy = t + e T  ->  |n| and the row offset |n| * mw in the half-plane box;
    // rows with n < 0 (bit e of negmask) are read through V(-k) = conj V(k)
    int absn[16];
    unsigned negmask = 0;
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const int iy = t + e * T;
        const int n = iy < NY / 2 ? iy : iy - NY;
        absn[e] = abs(n);
        negmask |= (n < 0 ? 1u : 0u) << e;
    }

    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int fp = item / per_pair, rem = item % per_pair;
        const int f = fp / n_pairs, pr = fp % n_pairs;
        const int sa = 2 * pr, sb = 2 * pr + 1;
        const int32_t* off = offsets + (size_t)f * (n_bins + 1);
        const bool has_a = off[(sa + 1) * n_elem] > off[sa * n_elem];
        const bool has_b = (sb < n_slices) && off[(sb + 1) * n_elem] > off[sb * n_elem];
        if (!has_a && !has_b) continue;                                    // block-uniform
        const int kx = tiles[rem / SUB] * kColTile + (rem % SUB) * C + c;
        const int m = kx < nx / 2 ? kx : kx - nx;
        const int nm = nmax[kx];
        // vacuum slices read slice sa's box with weight 0 (no branch in the loop)
        const float2* Va = Vk + ((size_t)f * n_slices + (has_a ? sa : sb)) * nh * mw;
        const float2* Vb = Vk + ((size_t)f * n_slices + (has_b ? sb : sa)) * nh * mw;
        const float wa = has_a ? 1.f : 0.f, wb = has_b ? 1.f : 0.f;
        const int col_dir = mcut + m, col_mir = mcut - m;
        const unsigned mirmask = negmask | ((m < 0 && t == 0) ? 1u : 0u);  // n == 0 (t == 0, e == 0) with m < 0: mirrored too
        float2 v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            float2 z = make_float2(0.f, 0.f);
            if (absn[e] <= nm) {
                const bool mir = (mirmask >> e) & 1u;
                const int idx = absn[e] * mw + (mir ? col_mir : col_dir);
                float2 a = __ldg(Va + idx), b = __ldg(Vb + idx);
                a.x *= wa; a.y *= wa; b.x *= wb; b.y *= wb;
                const float sg = mir ? -1.f : 1.f;                         // conj of both for mirrored rows
                z = make_float2(fmaf(-sg, b.y, a.x), fmaf(sg, a.y, b.x));
            }
            v[e] = z;
        }
        fft_inverse<NY, ColSlots<C>, BlockSync>(v, t, tw, slots);
        float2* dst = Zm + ((size_t)fp * NY) * nx + kx;
#pragma unroll
        for (int e = 0; e < 16; ++e) dst[(size_t)(t + e * T) * nx] = v[e];
    }
}

template <int NX> struct VRowCfg {
    static constexpr int T = Plan<NX>::T;
    static constexpr int THREADS = 256;
    static constexpr int RPB = THREADS / T;
    static constexpr size_t SMEM = (size_t)RPB * RowLine<NX>::LEN * sizeof(float2);
    using Sync = typename std::conditional<(T <= 32), WarpSync,
                                           typename std::conditional<(RPB > 1), GroupSync<T>, BlockSync>::type>::type;
};

template <int NX>
__global__ void __launch_bounds__(VRowCfg<NX>::THREADS)
k_v_row(const float2* __restrict__ Zm, const int32_t* __restrict__ offsets, float* __restrict__ V,
        const uint8_t* __restrict__ tile_active, const int ny, const int n_slices, const int n_elem,
        const int n_pairs, const long long n_rows, const int n_items) {
    using Cfg = VRowCfg<NX>;
    constexpr int T = Cfg::T;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, r = threadIdx.x / T;
    RowSlots slots{smem + (size_t)r * RowLine<NX>::LEN};
    Twiddles<NX> tw;
    tw.init(t);
    unsigned amask = 0;
#pragma unroll
    for (int e = 0; e < 16; ++e) amask |= (tile_active[(t + e * T) / kColTile] ? 1u : 0u) << e;
    const int n_bins = n_slices * n_elem;
    const int ny_shift = __ffs(ny) - 1;                       // ny is a power of two

    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const unsigned rho = (unsigned)item * Cfg::RPB + r;       // < 2^31: the mixed array lives in scratch
        const bool valid = (long long)rho < n_rows;
        int y = 0, fp = 0;
        if (valid) { fp = (int)(rho >> ny_shift); y = (int)(rho & (unsigned)(ny - 1)); }
        const int f = fp / n_pairs, pr = fp % n_pairs;
        const int sa = 2 * pr, sb = 2 * pr + 1;
        const int32_t* off = offsets + (size_t)f * (n_bins + 1);
        const bool has_a = valid && off[(sa + 1) * n_elem] > off[sa * n_elem];
        const bool has_b = valid && (sb < n_slices) && off[(sb + 1) * n_elem] > off[sb * n_elem];
        const bool any = has_a || has_b;
        const float2* src = Zm + ((size_t)fp * ny + y) * NX;
        float2 v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e)
            v[e] = (any && ((amask >> e) & 1u)) ? src[t + e * T] : make_float2(0.f, 0.f);
        // both slices of every row of this block empty (vacuum): V = 0, no transform.  When the block's RPB rows lie
        // inside one slice-pair image (RPB <= ny; both are powers of two, so they are then contiguous in V) they are
        // cleared with 16-byte stores; on smaller grids a block spans several slice pairs and every row group clears
        // its own row through the normal (f, sa, sb, y) addressing.
        if (!__syncthreads_or(any)) {
            if (Cfg::RPB <= ny) {
                const unsigned rho0 = (unsigned)item * Cfg::RPB;
                if ((long long)rho0 < n_rows) {
                    const int fp0 = (int)(rho0 >> ny_shift), y0 = (int)(rho0 & (unsigned)(ny - 1));
                    const int f0 = fp0 / n_pairs, s0 = 2 * (fp0 % n_pairs);
                    float4* za = reinterpret_cast<float4*>(V + (((size_t)f0 * n_slices + s0) * ny + y0) * NX);
                    float4* zb = reinterpret_cast<float4*>(V + (((size_t)f0 * n_slices + s0 + 1) * ny + y0) * NX);
                    for (int k = threadIdx.x; k < Cfg::RPB * NX / 4; k += Cfg::THREADS) {
                        za[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (s0 + 1 < n_slices) zb[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                }
            } else if (valid) {
                float* va = V + (((size_t)f * n_slices + sa) * ny + y) * NX;
#pragma unroll
                for (int e = 0; e < 16; ++e) va[t + e * T] = 0.f;
                if (sb < n_slices) {
                    float* vb = V + (((size_t)f * n_slices + sb) * ny + y) * NX;
#pragma unroll
                    for (int e = 0; e < 16; ++e) vb[t + e * T] = 0.f;
                }
            }
            continue;
        }
        fft_inverse<NX, RowSlots, typename Cfg::Sync>(v, t, tw, slots);
        if (valid) {
            float* va = V + (((size_t)f * n_slices + sa) * ny + y) * NX;
#pragma unroll
            for (int e = 0; e < 16; ++e) va[t + e * T] = v[e].x;
            if (sb < n_slices) {
                float* vb = V + (((size_t)f * n_slices + sb) * ny + y) * NX;
#pragma unroll
                for (int e = 0; e < 16; ++e) vb[t + e * T] = v[e].y;
            }
        }
    }
}

// ------------------------------------------------------------------------------------ host side
struct ScratchLayout {
    size_t ux, uy, key, sux, suy, off, vk, zm, total;
};
static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static ScratchLayout scratch_layout(const ps_ctx* c, int nfc, int n_atoms) {
    ScratchLayout L;
    const size_t na = (size_t)nfc * n_atoms;
    const int n_pairs = (c->n_slices + 1) / 2;
    size_t o = 0;
    L.ux = o; o += align256(na * 4);
    L.uy = o; o += align256(na * 4);
    L.key = o; o += align256(na * 4);
    L.sux = o; o += align256(na * 4);
    L.suy = o; o += align256(na * 4);
    L.off = o; o += align256((size_t)nfc * ((size_t)c->n_slices * c->n_elem + 1) * 4);
    L.vk = o; o += align256((size_t)nfc * c->n_slices * (c->ncut + 1) * (2 * c->mcut + 1) * sizeof(float2));
    L.zm = o; o += align256((size_t)nfc * n_pairs * c->nx * c->ny * sizeof(float2));
    L.total = o + 256;
    return L;
}

template <int NY>
static cudaError_t launch_v_col(ps_ctx* c, const float2* Vk, const int32_t* off, float2* Zm, int nfc) {
    using Cfg = VColCfg<NY>;
    auto kern = k_v_col<NY>;
    int cap = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &cap);
    if (ce != cudaSuccess) return ce;
    const int n_pairs = (c->n_slices + 1) / 2;
    const long long n_items = (long long)nfc * n_pairs * c->n_tiles_active * (kColTile / Cfg::C);
    const int grid = (int)(n_items < cap ? n_items : cap);
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(Vk, off, Zm, c->nx, c->d_tiles, c->n_tiles_active, c->d_nmax,
                                                      c->n_slices, c->n_elem, c->mcut, c->ncut, n_pairs, (int)n_items);
    return cudaGetLastError();
}

template <int NX>
static cudaError_t launch_v_row(ps_ctx* c, const float2* Zm, const int32_t* off, float* V, int nfc) {
    using Cfg = VRowCfg<NX>;
    auto kern = k_v_row<NX>;
    int cap = 0;
    cudaError_t ce = kernel_cap(c, kern, Cfg::THREADS, Cfg::SMEM, &cap);
    if (ce != cudaSuccess) return ce;
    const int n_pairs = (c->n_slices + 1) / 2;
    const long long n_rows = (long long)nfc * n_pairs * c->ny;
    const long long n_items = (n_rows + Cfg::RPB - 1) / Cfg::RPB;
    const int grid = (int)(n_items < cap ? n_items : cap);
    kern<<<grid, Cfg::THREADS, Cfg::SMEM, c->stream>>>(Zm, off, V, c->d_tile_active, c->ny, c->n_slices, c->n_elem,
                                                      n_pairs, n_rows, (int)n_items);
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

extern "C" size_t ps_workspace_bytes(const ps_ctx* c, int n_frames_chunk, int n_atoms) {
    if (!c || !c->have_geom || !c->have_ff || n_frames_chunk < 1 || n_atoms < 1) return 0;
    return scratch_layout(c, n_frames_chunk, n_atoms).total;
}

// Frame chunk by frame chunk: ingest, sort, V(k), y-inverse transform into the mixed array Zm.  Then either the
// x-inverse transform into the caller's V (ps_build_slices) or `consume(f0, nf, Zm, offsets)` (ps_multislice_fused: the
// slice loop of these frames takes the potential from Zm directly).
typedef std::function<ps_status(int f0, int nf, const float2* Zm, const int32_t* off)> ZmConsumer;

static ps_status build_chunks(ps_ctx* c, const float* d_pos, const int32_t* d_Z, int n_frames, int n_atoms, float* d_V,
                              int32_t* d_slice_idx, const ZmConsumer* consume) {
    ps_status st;
    if ((st = ensure_ftab(c)) != PS_OK) return st;
    const long long n_bins = (long long)c->n_slices * c->n_elem;
    if ((2 * n_bins + 2) * 4 > 200 * 1024)
        return fail(c, PS_EUNSUPPORTED, "ps_build_slices: n_slices * n_elements too large for the sort kernel");

    // Z validation.  The first time a (d_Z, n_atoms) pair is seen, one 4-byte read-back rejects unknown atomic numbers
    // before any work is queued (a blocking call, like every first call with new parameters).  Later calls with the
    // same pair queue their work without waiting; k_bin re-checks every atom of every call on the device and raises the
    // ctx's mapped error word, which the next ps_* call reports (enter()).
    if (c->z_checked != (const void*)d_Z || c->z_checked_n != n_atoms) {
        if ((st = ensure_buf(c, c->misc, 4096)) != PS_OK) return st;
        int* d_flag = (int*)c->misc.p;
        PSB_CUDA(c, cudaMemsetAsync(d_flag, 0, sizeof(int), c->stream));
        k_check_Z<<<(n_atoms + 255) / 256, 256, 0, c->stream>>>(d_Z, n_atoms, c->d_elem_of_Z, d_flag);
        PSB_LAUNCH_CHECK(c, "k_check_Z");
        int h_flag = 0;
        PSB_CUDA(c, cudaMemcpyAsync(&h_flag, d_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        PSB_CUDA(c, cudaStreamSynchronize(c->stream));
        if (h_flag != 0)
            return fail(c, PS_EUNSUPPORTED, "ps_build_slices: atomic number " + std::to_string(h_flag == -1 ? 0 : h_flag) +
                                                " has no form-factor coefficients");
        c->z_checked = (const void*)d_Z; c->z_checked_n = n_atoms;
    }

    // scratch: installed workspace or library-owned buffer; frames are processed in chunks that fit
    const size_t per_frame = scratch_layout(c, 1, n_atoms).total;
    // library-owned scratch: an eighth of the free device memory, between 768 MB and 16 GB (at 1024^2 x 120 slices
    // one frame needs 0.6 GB: with less, frames go one per launch and the sort / V(k) launches cannot fill the GPU)
    size_t avail = c->user_ws_bytes;
    if (!c->user_ws) {
        size_t free_b = 0, total_b = 0;
        avail = (size_t)768 << 20;
        const int f_all = n_frames < 65535 ? n_frames : 65535;
        if (c->scratch.bytes >= scratch_layout(c, f_all, n_atoms).total) {
            avail = c->scratch.bytes;                                      // everything fits what is already held
        } else {
            if (c->scratch_budget == 0) {                                  // one driver query per context
                c->scratch_budget = avail;
                if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
                    size_t want = (free_b + c->scratch.bytes) / 8;
                    if (want > ((size_t)16 << 30)) want = (size_t)16 << 30;
                    if (want > c->scratch_budget) c->scratch_budget = want;
                }
            }
            avail = c->scratch_budget;
        }
        if (c->scratch.bytes > avail) avail = c->scratch.bytes;           // never less than what is already held
    }
    int nfc = (int)(avail / per_frame);
    if (nfc < 1) {
        if (c->user_ws) return fail(c, PS_EWORKSPACE, "ps_build_slices: workspace smaller than one frame needs (" +
                                                          std::to_string(per_frame) + " bytes)");
        nfc = 1;
    }
    if (nfc > n_frames) nfc = n_frames;
    if (nfc > 65535) nfc = 65535;                                          // grid.z limit of k_vk
    nfc = (n_frames + (n_frames + nfc - 1) / nfc - 1) / ((n_frames + nfc - 1) / nfc);   // equal chunks, no short tail
    ScratchLayout L = scratch_layout(c, nfc, n_atoms);
    while (c->user_ws && L.total > c->user_ws_bytes && nfc > 1) L = scratch_layout(c, --nfc, n_atoms);
    char* ws = (char*)c->user_ws;
    if (!ws) {
        if ((st = ensure_buf(c, c->scratch, L.total)) != PS_OK) return st;
        ws = (char*)c->scratch.p;
    } else if (L.total > c->user_ws_bytes) {
        return fail(c, PS_EWORKSPACE, "ps_build_slices: workspace too small");
    }
    uint32_t *Ux = (uint32_t*)(ws + L.ux), *Uy = (uint32_t*)(ws + L.uy);
    uint32_t *sUx = (uint32_t*)(ws + L.sux), *sUy = (uint32_t*)(ws + L.suy);
    int32_t *key = (int32_t*)(ws + L.key), *off = (int32_t*)(ws + L.off);
    float2 *Vk = (float2*)(ws + L.vk), *Zm = (float2*)(ws + L.zm);

    const int tiles_m = (c->mcut + 1 + VK_TM - 1) / VK_TM, tiles_n = (c->ncut + 1 + VK_TN - 1) / VK_TN;
    const size_t img = (size_t)c->nx * c->ny;
    {
        int cap_unused = 0;                                                // sets the 200 KB attribute once per ctx
        PSB_CUDA(c, kernel_cap(c, k_sort, 1024, (size_t)200 * 1024, &cap_unused));
    }

    for (int f0 = 0; f0 < n_frames; f0 += nfc) {
        const int nf = (n_frames - f0 < nfc) ? n_frames - f0 : nfc;
        const long long n_total = (long long)nf * n_atoms;
        { ProfScope ps_(c, K_BIN);
        k_bin<<<(unsigned)((n_total + 255) / 256), 256, 0, c->stream>>>(
            d_pos + (size_t)f0 * n_atoms * 3, d_Z, c->d_elem_of_Z, n_total, n_atoms, c->cell[0], c->cell[1], c->cell[2],
            c->n_slices, c->n_elem, Ux, Uy, key, d_slice_idx ? d_slice_idx + (size_t)f0 * n_atoms : nullptr,
            c->d_async_err, c->d_bad_z);
        }
        PSB_LAUNCH_CHECK(c, "k_bin");
        { ProfScope ps_(c, K_SORT);
        {
            // as many warps as the 200 KB of cursors allow, at most 32, at least one per 64 atoms
            int W = (int)((size_t)200 * 1024 / sizeof(int) / (size_t)(n_bins + 1)) - 1;
            if (W > 32) W = 32;
            if (W > (n_atoms + 63) / 64) W = (n_atoms + 63) / 64;
            if (W < 1) W = 1;
            const size_t smem = ((size_t)W * n_bins + n_bins + 1) * sizeof(int);
            k_sort<<<nf, 32 * W, smem, c->stream>>>(Ux, Uy, key, n_atoms, (int)n_bins, sUx, sUy, off);
        }
        }
        PSB_LAUNCH_CHECK(c, "k_sort");
        // tensor-core sums pay off once a (slice, element) group fills a few K = 16 stages
        const bool use_tc = c->vk_mode == 2 ||
                            (c->vk_mode == 0 && (long long)n_atoms >= 48LL * c->n_slices * c->n_elem);
        if (use_tc) {
            cudaError_t e;
            { ProfScope ps_(c, K_VK); e = launch_vk_tc(c, sUx, sUy, off, Vk, n_atoms, nf); }
            if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_vk_tc: ") + cudaGetErrorString(e));
            c->launches++;
        } else {
            { ProfScope ps_(c, K_VK);
            k_vk<<<dim3(tiles_m * tiles_n, c->n_slices, nf), VK_THREADS, 0, c->stream>>>(
                sUx, sUy, off, c->d_ftab, c->d_nmax, Vk, n_atoms, c->n_slices, c->n_elem, c->mcut, c->ncut, tiles_m);
            }
            PSB_LAUNCH_CHECK(c, "k_vk");
        }
        cudaError_t e = cudaErrorInvalidValue;
        { ProfScope ps_(c, K_V_COL);
        PSB_DISPATCH_N(c->ny, (e = launch_v_col<N_>(c, Vk, off, Zm, nf))); }
        if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_v_col: ") + cudaGetErrorString(e));
        c->launches++;
        if (d_V) {
            e = cudaErrorInvalidValue;
            { ProfScope ps_(c, K_V_ROW);
            PSB_DISPATCH_N(c->nx, (e = launch_v_row<N_>(c, Zm, off, d_V + (size_t)f0 * c->n_slices * img, nf))); }
            if (e != cudaSuccess) return fail(c, PS_ECUDA, std::string("k_v_row: ") + cudaGetErrorString(e));
            c->launches++;
        }
        // An atom k_bin could not place (no coefficients for its Z) was dropped from the sums: what this chunk produced
        // must not be consumed as if it were a potential.  NaN-fill it (no-op launch unless k_bin raised the word).
        {
            float* dst = d_V ? d_V + (size_t)f0 * c->n_slices * img : (float*)Zm;
            const size_t n4 = d_V ? (size_t)nf * c->n_slices * img / 4 : (L.total - L.zm) / 16;
            k_poison<<<kNumSM * 4, 256, 0, c->stream>>>(reinterpret_cast<float4*>(dst), n4, c->d_bad_z);
            PSB_LAUNCH_CHECK(c, "k_poison");
        }
        if (consume && (st = (*consume)(f0, nf, Zm, off)) != PS_OK) return st;
    }
    return PS_OK;
}

extern "C" ps_status ps_build_slices(ps_ctx* c, const float* d_pos, const int32_t* d_Z, int n_frames, int n_atoms,
                                     float* d_V, int32_t* d_slice_idx) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom || !c->have_ff)
        return fail(c, PS_ESTATE, "ps_build_slices: ps_set_geometry and ps_set_form_factors must be called first");
    if (!d_pos || !d_Z || !d_V || n_frames < 1 || n_atoms < 1)
        return fail(c, PS_EINVAL, "ps_build_slices: null pointer or non-positive size");
    ps_status st = enter(c, "ps_build_slices");
    if (st != PS_OK) return st;
    return build_chunks(c, d_pos, d_Z, n_frames, n_atoms, d_V, d_slice_idx, nullptr);
}

extern "C" ps_status ps_multislice_fused(ps_ctx* c, double kV, const void* d_psi0, int n_probes, const float* d_pos,
                                         const int32_t* d_Z, int n_frames, int n_atoms, void* d_exit, int exit_layout) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom || !c->have_ff)
        return fail(c, PS_ESTATE, "ps_multislice_fused: ps_set_geometry and ps_set_form_factors must be called first");
    if (!d_psi0 || !d_pos || !d_Z || !d_exit || n_probes < 1 || n_frames < 1 || n_atoms < 1 || !(kV > 0.0))
        return fail(c, PS_EINVAL, "ps_multislice_fused: null pointer or non-positive size / voltage");
    if (exit_layout != PS_LAYOUT_DENSE)
        return fail(c, PS_EUNSUPPORTED, "ps_multislice_fused: the wave is propagated in place inside d_exit: dense layout only");
    ps_status st = enter(c, "ps_multislice_fused");
    if (st != PS_OK) return st;
    const ZmConsumer slice_loop = [&](int f0, int nf, const float2* Zm, const int32_t* off) -> ps_status {
        VSrc src;
        src.Zm = Zm; src.off = off; src.zm_f0 = f0;
        return multislice_range(c, kV, d_psi0, n_probes, src, n_frames, f0, nf, d_exit, exit_layout);
    };
    return build_chunks(c, d_pos, d_Z, n_frames, n_atoms, nullptr, nullptr, &slice_loop);
}
