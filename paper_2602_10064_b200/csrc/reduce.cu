// reduce.cu — reductions over I[P][n_bins][ny][nx] (PAPER.md:89 TACAWData methods; PAPER.md:394 dispersion,
// 397 spectral_diffraction, 422 spectrum_image, 107 frequency bands; readings A15-A17 of DESIGN.md §3).
// All sums run in a fixed order (no floating-point atomics): results are bit-reproducible.
// Index work (detector membership, nearest path pixel, radial q bin) is done in float64 with explicitly
// rounded operations (no FMA contraction) so that it is bit-exact against the float64 definition.
#include <math.h>

#include "common.cuh"

namespace psb {

__device__ __forceinline__ double k_abs(const int ix, const int iy, const int nx, const int ny, const double Lx,
                                        const double Ly) {
    const int m = ix < (nx + 1) / 2 ? ix : ix - nx, n = iy < (ny + 1) / 2 ? iy : iy - ny;
    const double kx = __ddiv_rn((double)m, Lx), ky = __ddiv_rn((double)n, Ly);
    return __dsqrt_rn(__dadd_rn(__dmul_rn(kx, kx), __dmul_rn(ky, ky)));
}

__device__ __forceinline__ float block_sum(float v, float* sh) {   // fixed-order tree; result valid in thread 0
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_down_sync(0xffffffffu, v, d);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) sh[w] = v;
    __syncthreads();
    if (w == 0) {
        v = (lane < (blockDim.x + 31) / 32) ? sh[lane] : 0.f;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v += __shfl_down_sync(0xffffffffu, v, d);
    }
    __syncthreads();
    return v;
}

// ---------------------------------------------------------------- spectral diffraction pattern
__global__ void k_sdp(const float* __restrict__ I, float* __restrict__ out, const int P, const int n_bins,
                      const int lo, const int hi, const size_t npix) {
    const size_t pix = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (pix >= npix) return;
    float s = 0.f;
    for (int p = 0; p < P; ++p)
        for (int b = lo; b <= hi; ++b) s += I[((size_t)p * n_bins + b) * npix + pix];
    out[pix] = s;
}

// ---------------------------------------------------------------- spectrum image
__global__ void k_detector_mask(uint8_t* __restrict__ mask, const int nx, const int ny, const double Lx, const double Ly,
                                const double k_in, const double k_out, const int has_out) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)nx * ny) return;
    const double k = k_abs((int)(i % nx), (int)(i / nx), nx, ny, Lx, Ly);
    mask[i] = (k >= k_in && (!has_out || k < k_out)) ? 1 : 0;
}

__global__ void __launch_bounds__(1024)
k_spectrum_image(const float* __restrict__ I, const uint8_t* __restrict__ mask, float* __restrict__ out,
                 const size_t npix) {
    __shared__ float sh[32];
    const float4* src = reinterpret_cast<const float4*>(I + (size_t)blockIdx.x * npix);   // blockIdx.x = p * n_bins + b
    const uchar4* m4 = reinterpret_cast<const uchar4*>(mask);
    float s = 0.f;
    for (size_t i = threadIdx.x; i < npix / 4; i += blockDim.x) {      // npix is a multiple of 1024
        const float4 x = src[i];
        const uchar4 m = m4[i];
        float q = m.x ? x.x : 0.f;                                     // fixed order inside the quad
        q += m.y ? x.y : 0.f;
        q += m.z ? x.z : 0.f;
        q += m.w ? x.w : 0.f;
        s += q;
    }
    s = block_sum(s, sh);
    if (threadIdx.x == 0) out[blockIdx.x] = s;
}

// ---------------------------------------------------------------- HAADF (annular detector on the exit waves)
// tmp[p * F + f] = sum_{k in detector} |Psi_pf(k)|^2, fixed order; k_haadf_mean then averages over frames
__global__ void __launch_bounds__(1024)
k_haadf_frame(const float2* __restrict__ exitw, const uint8_t* __restrict__ mask, float* __restrict__ tmp, const size_t npix) {
    __shared__ float sh[32];
    const float4* src = reinterpret_cast<const float4*>(exitw + (size_t)blockIdx.x * npix);   // two pixels per float4
    const uchar2* m2 = reinterpret_cast<const uchar2*>(mask);
    float s = 0.f;
    for (size_t i = threadIdx.x; i < npix / 2; i += blockDim.x) {
        const float4 x = src[i];
        const uchar2 m = m2[i];
        float q = m.x ? fmaf(x.x, x.x, x.y * x.y) : 0.f;
        q += m.y ? fmaf(x.z, x.z, x.w * x.w) : 0.f;
        s += q;
    }
    s = block_sum(s, sh);
    if (threadIdx.x == 0) tmp[blockIdx.x] = s;
}
// Tiled exit layout [P][ny][tile][F][8]: a block owns one (probe, row) and sums |Psi|^2 over the row's in-band tiles for
// every frame (threads = frames: consecutive 64-byte chunks), part[(p * ny + iy) * F + f]; k_haadf_rows then adds the
// rows in fixed order into the same tmp[p * F + f] the dense path produces.
__global__ void __launch_bounds__(256)
k_haadf_tiled(const float2* __restrict__ Tl, const uint8_t* __restrict__ mask, const int32_t* __restrict__ tiles,
              float* __restrict__ part, const int nx, const int ny, const int n_tiles, const int F) {
    const int iy = blockIdx.x, p = blockIdx.y;
    const float2* row = Tl + ((size_t)p * ny + iy) * n_tiles * F * kColTile;
    for (int f = threadIdx.x; f < F; f += blockDim.x) {
        float s = 0.f;
        for (int tj = 0; tj < n_tiles; ++tj) {
            const float4* src = reinterpret_cast<const float4*>(row + ((size_t)tj * F + f) * kColTile);
            const uint8_t* m = mask + (size_t)iy * nx + tiles[tj] * kColTile;
#pragma unroll
            for (int q = 0; q < kColTile / 2; ++q) {
                const float4 x = src[q];
                float v = m[2 * q] ? fmaf(x.x, x.x, x.y * x.y) : 0.f;
                v += m[2 * q + 1] ? fmaf(x.z, x.z, x.w * x.w) : 0.f;
                s += v;
            }
        }
        part[((size_t)p * ny + iy) * F + f] = s;
    }
}
__global__ void k_haadf_rows(const float* __restrict__ part, float* __restrict__ tmp, const int ny, const int F, const long long total) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;       // p * F + f
    if (i >= total) return;
    const long long p = i / F; const int f = (int)(i % F);
    float s = 0.f;
    for (int iy = 0; iy < ny; ++iy) s += part[((size_t)p * ny + iy) * F + f];
    tmp[i] = s;
}
__global__ void k_haadf_mean(const float* __restrict__ tmp, float* __restrict__ out, const int P, const int F, const float scale) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    float s = 0.f;
    for (int f = 0; f < F; ++f) s += tmp[(size_t)p * F + f];
    out[p] = s * scale;
}

// acc <- w_acc * acc + w_new * I  (trajectory / segment averaging of |Psi(k,w)|^2)
__global__ void k_accumulate(float* __restrict__ acc, const float* __restrict__ I, const size_t n4, const float w_acc,
                             const float w_new) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        float4 a = reinterpret_cast<float4*>(acc)[i];
        const float4 x = reinterpret_cast<const float4*>(I)[i];
        a.x = fmaf(w_acc, a.x, w_new * x.x); a.y = fmaf(w_acc, a.y, w_new * x.y);
        a.z = fmaf(w_acc, a.z, w_new * x.z); a.w = fmaf(w_acc, a.w, w_new * x.w);
        reinterpret_cast<float4*>(acc)[i] = a;
    }
}

// ---------------------------------------------------------------- dispersion
__global__ void k_path_pixels(const double* __restrict__ kx, const double* __restrict__ ky, int32_t* __restrict__ pix,
                              const int n_path, const int nx, const int ny, const double Lx, const double Ly) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_path) return;
    const long long ax = (long long)floor(__dadd_rn(__dmul_rn(kx[i], Lx), 0.5));
    const long long ay = (long long)floor(__dadd_rn(__dmul_rn(ky[i], Ly), 0.5));
    const int ix = (int)(((ax % nx) + nx) % nx), iy = (int)(((ay % ny) + ny) % ny);
    pix[i] = iy * nx + ix;
}

__global__ void k_dispersion(const float* __restrict__ I, const int32_t* __restrict__ pix, float* __restrict__ out,
                             const int P, const int n_bins, const int n_path, const size_t npix) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_bins * n_path) return;
    const int b = i / n_path, j = i % n_path;
    float s = 0.f;
    for (int p = 0; p < P; ++p) s += I[((size_t)p * n_bins + b) * npix + pix[j]];
    out[i] = s;
}

// ---------------------------------------------------------------- radial q bins
__global__ void k_qidx(int32_t* __restrict__ qidx, const int nx, const int ny, const double Lx, const double Ly,
                       const double dq, const int n_q) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)nx * ny) return;
    const double k = k_abs((int)(i % nx), (int)(i / nx), nx, ny, Lx, Ly);
    const double b = floor(__ddiv_rn(k, dq));
    qidx[i] = (b >= (double)n_q) ? -1 : (int32_t)b;
}

// one warp: histogram + exclusive scan + stable placement of pixel indices by q bin (deterministic order)
__global__ void __launch_bounds__(32)
k_order_by_bin(const int32_t* __restrict__ qidx, const int npix, const int n_q, int32_t* __restrict__ cursor /*[n_q+1]*/,
               int32_t* __restrict__ offsets /*[n_q+1]*/, int32_t* __restrict__ order /*[npix]*/) {
    const int lane = threadIdx.x;
    for (int b = lane; b <= n_q; b += 32) cursor[b] = 0;
    __syncwarp();
    for (int j = lane; j < npix; j += 32) {
        const int k = qidx[j];
        if (k >= 0) atomicAdd(&cursor[k], 1);
    }
    __syncwarp();
    int carry = 0;
    for (int b0 = 0; b0 <= n_q; b0 += 32) {
        const int b = b0 + lane;
        const int cnt = (b < n_q) ? cursor[b] : 0;
        int incl = cnt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += o;
        }
        const int excl = carry + incl - cnt;
        __syncwarp();
        if (b <= n_q) { cursor[b] = excl; offsets[b] = excl; }
        carry += __shfl_sync(0xffffffffu, incl, 31);
    }
    __syncwarp();
    for (int j0 = 0; j0 < npix; j0 += 32) {
        const int j = j0 + lane;
        const int k = (j < npix) ? qidx[j] : -1;
        const unsigned grp = __match_any_sync(0xffffffffu, k);
        const int rank = __popc(grp & ((1u << lane) - 1u));
        int dst = -1;
        if (k >= 0) dst = cursor[k] + rank;
        __syncwarp();
        if (k >= 0 && rank == __popc(grp) - 1) cursor[k] += __popc(grp);
        __syncwarp();
        if (dst >= 0) order[dst] = j;
    }
}

// one warp per (bin b, q): ordered segment sum
__global__ void __launch_bounds__(128)
k_qbin_sum(const float* __restrict__ I, const int32_t* __restrict__ offsets, const int32_t* __restrict__ order,
           float* __restrict__ out, const int P, const int n_bins, const int n_q, const size_t npix) {
    const int wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (wid >= n_bins * n_q) return;
    const int b = wid / n_q, q = wid % n_q;
    const int j0 = offsets[q], j1 = offsets[q + 1];
    float s = 0.f;
    for (int j = j0 + lane; j < j1; j += 32) {
        const int pix = order[j];
        for (int p = 0; p < P; ++p) s += I[((size_t)p * n_bins + b) * npix + pix];
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_down_sync(0xffffffffu, s, d);
    if (lane == 0) out[wid] = s;
}

}  // namespace psb

using namespace psb;

static ps_status check_I(ps_ctx* c, const char* who, const float* d_I, int P, int n_bins, const void* d_out) {
    ps_status st = enter(c, who);
    if (st != PS_OK) return st;
    if (!c->have_geom) return fail(c, PS_ESTATE, std::string(who) + ": ps_set_geometry has not been called");
    if (!d_I || !d_out || P < 1 || n_bins < 1) return fail(c, PS_EINVAL, std::string(who) + ": null pointer or non-positive size");
    return PS_OK;
}

extern "C" ps_status ps_sdp(ps_ctx* c, const float* d_I, int P, int n_bins, int bin_lo, int bin_hi, float* d_out) {
    if (!c) return PS_EINVAL;
    ps_status st = check_I(c, "ps_sdp", d_I, P, n_bins, d_out);
    if (st != PS_OK) return st;
    ProfScope ps_(c, K_REDUCE);
    if (bin_lo < 0 || bin_hi >= n_bins || bin_lo > bin_hi) return fail(c, PS_EINVAL, "ps_sdp: bin range outside [0, n_bins)");
    const size_t npix = (size_t)c->nx * c->ny;
    k_sdp<<<(unsigned)((npix + 255) / 256), 256, 0, c->stream>>>(d_I, d_out, P, n_bins, bin_lo, bin_hi, npix);
    PSB_LAUNCH_CHECK(c, "k_sdp");
    return PS_OK;
}

extern "C" ps_status ps_spectrum_image(ps_ctx* c, const float* d_I, int P, int n_bins, double k_in, double k_out,
                                       float* d_out) {
    if (!c) return PS_EINVAL;
    ps_status st = check_I(c, "ps_spectrum_image", d_I, P, n_bins, d_out);
    if (st != PS_OK) return st;
    ProfScope ps_(c, K_REDUCE);
    if (k_in < 0.0) return fail(c, PS_EINVAL, "ps_spectrum_image: k_in must be >= 0");
    const size_t npix = (size_t)c->nx * c->ny;
    if ((st = ensure_buf(c, c->misc, 4096 + npix)) != PS_OK) return st;
    uint8_t* d_mask = (uint8_t*)c->misc.p + 4096;
    k_detector_mask<<<(unsigned)((npix + 255) / 256), 256, 0, c->stream>>>(d_mask, c->nx, c->ny, c->cell[0], c->cell[1], k_in,
                                                                           k_out, k_out > 0.0 ? 1 : 0);
    PSB_LAUNCH_CHECK(c, "k_detector_mask");
    k_spectrum_image<<<P * n_bins, 1024, 0, c->stream>>>(d_I, d_mask, d_out, npix);
    PSB_LAUNCH_CHECK(c, "k_spectrum_image");
    return PS_OK;
}

extern "C" ps_status ps_haadf(ps_ctx* c, const void* d_exit, int exit_layout, int n_probes, int n_frames, double k_in,
                              double k_out, float* d_out) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_haadf: ps_set_geometry has not been called");
    if (!d_exit || !d_out || n_probes < 1 || n_frames < 1) return fail(c, PS_EINVAL, "ps_haadf: null pointer or non-positive size");
    if (exit_layout != PS_LAYOUT_DENSE && exit_layout != PS_LAYOUT_TILED_APERTURE)
        return fail(c, PS_EUNSUPPORTED, "ps_haadf: unknown exit layout");
    const bool tiled = exit_layout == PS_LAYOUT_TILED_APERTURE;
    if (k_in < 0.0) return fail(c, PS_EINVAL, "ps_haadf: k_in must be >= 0");
    ps_status st_in = enter(c, "ps_haadf");
    if (st_in != PS_OK) return st_in;
    const size_t npix = (size_t)c->nx * c->ny;
    const size_t tmp_off = (4096 + npix + 255) & ~(size_t)255;
    const size_t tmp_bytes = ((size_t)n_probes * n_frames * sizeof(float) + 255) & ~(size_t)255;
    const size_t part_bytes = tiled ? (size_t)n_probes * c->ny * n_frames * sizeof(float) : 0;   // per-row partial sums
    ps_status st = ensure_buf(c, c->misc, tmp_off + tmp_bytes + part_bytes);
    if (st != PS_OK) return st;
    uint8_t* d_mask = (uint8_t*)c->misc.p + 4096;
    float* d_tmp = (float*)((char*)c->misc.p + tmp_off);
    ProfScope ps_(c, K_REDUCE);
    k_detector_mask<<<(unsigned)((npix + 255) / 256), 256, 0, c->stream>>>(d_mask, c->nx, c->ny, c->cell[0], c->cell[1], k_in,
                                                                           k_out, k_out > 0.0 ? 1 : 0);
    PSB_LAUNCH_CHECK(c, "k_detector_mask");
    if (tiled) {
        if (n_probes > 65535) return fail(c, PS_EUNSUPPORTED, "ps_haadf: more than 65535 probes in the tiled layout");
        float* d_part = (float*)((char*)c->misc.p + tmp_off + tmp_bytes);
        k_haadf_tiled<<<dim3(c->ny, n_probes), 256, 0, c->stream>>>((const float2*)d_exit, d_mask, c->d_tiles, d_part, c->nx,
                                                                    c->ny, c->n_tiles_active, n_frames);
        PSB_LAUNCH_CHECK(c, "k_haadf_tiled");
        const long long total = (long long)n_probes * n_frames;
        k_haadf_rows<<<(unsigned)((total + 255) / 256), 256, 0, c->stream>>>(d_part, d_tmp, c->ny, n_frames, total);
        PSB_LAUNCH_CHECK(c, "k_haadf_rows");
    } else {
        k_haadf_frame<<<n_probes * n_frames, 1024, 0, c->stream>>>((const float2*)d_exit, d_mask, d_tmp, npix);
        PSB_LAUNCH_CHECK(c, "k_haadf_frame");
    }
    k_haadf_mean<<<(n_probes + 127) / 128, 128, 0, c->stream>>>(d_tmp, d_out, n_probes, n_frames,
                                                                 (float)(1.0 / ((double)n_frames * (double)npix)));
    PSB_LAUNCH_CHECK(c, "k_haadf_mean");
    return PS_OK;
}

extern "C" ps_status ps_accumulate_intensity(ps_ctx* c, float* d_acc, const float* d_I, size_t n_values, double w_acc,
                                             double w_new) {
    if (!c) return PS_EINVAL;
    if (!d_acc || !d_I || n_values == 0) return fail(c, PS_EINVAL, "ps_accumulate_intensity: null pointer or zero size");
    if (n_values % 4 != 0 || (((uintptr_t)d_acc | (uintptr_t)d_I) & 15u))
        return fail(c, PS_EINVAL, "ps_accumulate_intensity: arrays must be 16-byte aligned with a multiple of 4 values");
    ps_status st_in = enter(c, "ps_accumulate_intensity");
    if (st_in != PS_OK) return st_in;
    const size_t n4 = n_values / 4;
    const size_t nb = (n4 + 255) / 256;
    ProfScope ps_(c, K_REDUCE);
    k_accumulate<<<(unsigned)(nb < 148 * 16 ? nb : 148 * 16), 256, 0, c->stream>>>(d_acc, d_I, n4, (float)w_acc, (float)w_new);
    PSB_LAUNCH_CHECK(c, "k_accumulate");
    return PS_OK;
}

extern "C" ps_status ps_dispersion(ps_ctx* c, const float* d_I, int P, int n_bins, int n_path, const double* kx,
                                   const double* ky, int32_t* d_pix, float* d_out) {
    if (!c) return PS_EINVAL;
    ps_status st = check_I(c, "ps_dispersion", d_I, P, n_bins, d_out);
    if (st != PS_OK) return st;
    ProfScope ps_(c, K_REDUCE);
    if (!kx || !ky || !d_pix || n_path < 1) return fail(c, PS_EINVAL, "ps_dispersion: null pointer or empty path");
    if ((st = ensure_buf(c, c->path_buf, 2 * (size_t)n_path * sizeof(double))) != PS_OK) return st;
    double* d_k = (double*)c->path_buf.p;
    // the caller's host arrays are copied into the ctx's pinned ring and sent asynchronously: not retained, no wait
    if ((st = upload_async(c, d_k, kx, (size_t)n_path * 8)) != PS_OK) return st;
    if ((st = upload_async(c, d_k + n_path, ky, (size_t)n_path * 8)) != PS_OK) return st;
    k_path_pixels<<<(n_path + 127) / 128, 128, 0, c->stream>>>(d_k, d_k + n_path, d_pix, n_path, c->nx, c->ny, c->cell[0],
                                                               c->cell[1]);
    PSB_LAUNCH_CHECK(c, "k_path_pixels");
    const int total = n_bins * n_path;
    k_dispersion<<<(total + 127) / 128, 128, 0, c->stream>>>(d_I, d_pix, d_out, P, n_bins, n_path, (size_t)c->nx * c->ny);
    PSB_LAUNCH_CHECK(c, "k_dispersion");
    return PS_OK;
}

extern "C" ps_status ps_qbin(ps_ctx* c, const float* d_I, int P, int n_bins, double dq, int n_q, int32_t* d_qidx,
                             float* d_out) {
    if (!c) return PS_EINVAL;
    ps_status st = check_I(c, "ps_qbin", d_I, P, n_bins, d_out);
    if (st != PS_OK) return st;
    ProfScope ps_(c, K_REDUCE);
    if (!d_qidx || !(dq > 0.0) || n_q < 1) return fail(c, PS_EINVAL, "ps_qbin: null pointer, dq <= 0 or n_q < 1");
    const size_t npix = (size_t)c->nx * c->ny;
    // pixel order by q bin depends only on (geometry, dq, n_q): built once and kept in the ctx
    const size_t need = (2 * ((size_t)n_q + 1) + npix) * 4 + 512;
    const bool cached = c->qorder_valid && c->qorder_dq == dq && c->qorder_nq == n_q && c->qorder.bytes >= need;
    if (!cached && (st = ensure_buf(c, c->qorder, need)) != PS_OK) return st;
    int32_t* d_cursor = (int32_t*)c->qorder.p;
    int32_t* d_off = d_cursor + (n_q + 1);
    int32_t* d_order = d_off + (n_q + 1);
    k_qidx<<<(unsigned)((npix + 255) / 256), 256, 0, c->stream>>>(d_qidx, c->nx, c->ny, c->cell[0], c->cell[1], dq, n_q);
    PSB_LAUNCH_CHECK(c, "k_qidx");
    if (!cached) {
        k_order_by_bin<<<1, 32, 0, c->stream>>>(d_qidx, (int)npix, n_q, d_cursor, d_off, d_order);
        PSB_LAUNCH_CHECK(c, "k_order_by_bin");
        c->qorder_valid = true; c->qorder_dq = dq; c->qorder_nq = n_q;
    }
    const long long warps = (long long)n_bins * n_q;
    k_qbin_sum<<<(unsigned)((warps * 32 + 127) / 128), 128, 0, c->stream>>>(d_I, d_off, d_order, d_out, P, n_bins, n_q, npix);
    PSB_LAUNCH_CHECK(c, "k_qbin_sum");
    return PS_OK;
}
