// static_scratch.cu — ps_spectrum_image_static: the spectrum-image reduction (PAPER.md:422 spectrum_image(); PAPER.md:89;
// reading A16 of DESIGN.md §3) for callers that cannot let the library allocate device memory.
//
// Who this is for.  ps_spectrum_image keeps its detector mask (one byte per pixel) in a buffer the ctx gets from
// cudaMalloc on first use and whenever a larger grid arrives.  Some hosts cannot afford that: a process whose start-up
// code has already given every free byte of HBM to its own pool (torch's caching allocator holding a 127 GB config-3
// working set is the example in this repository — a later cudaMalloc from inside the library simply fails), and a
// serving loop with a latency budget, where cudaMalloc / cudaFree stall every stream of the device for as long as the
// driver needs.  For them this entry point touches no allocator at all: the mask lives in a fixed array that is part
// of the library image.
//
// The price.
//   * Every GPU that loads libpyslice_b200.so holds kStaticMaskBytes (1 MiB) from load until the process exits,
//     whether this entry point is ever called or not.
//   * Grids of more than 1024 x 1024 pixels do not fit and are refused (PS_EUNSUPPORTED); use ps_spectrum_image.
//   * There is ONE array per device, shared by every ctx and every stream of the process.  Two calls whose kernels can
//     overlap on the GPU (different streams, or different host threads with different ctxs on one device) race on it
//     and both results are garbage.  Keep all calls on one device in one stream, or order them with events.
//   * The array still holds whatever the previous call left there.  Nothing here relies on a zeroed start: the mask
//     kernel rewrites each of the nx*ny bytes that the summing kernel will read before that kernel runs (same stream),
//     and bytes beyond nx*ny are never read.
//
// Set-up.  The name `g_static_mask` in host code is only a handle for the runtime, not a device address (passing it to
// a kernel would fault, or quietly address host memory on systems where the GPU can reach it).  The device address is
// looked up once per device with cudaGetSymbolAddress, with that device current, the first time this entry point runs
// on it.  That first call may make the runtime load the module, so issue it before starting any stream capture.
#include <math.h>

#include <mutex>

#include "common.cuh"

namespace psb {

constexpr size_t kStaticMaskBytes = (size_t)1024 * 1024;   // one byte per pixel: grids up to 1024 x 1024
constexpr int kStaticMaxDevices = 64;

static __device__ __align__(256) uint8_t g_static_mask[kStaticMaskBytes];

static std::mutex g_static_mu;
static uint8_t* g_static_mask_addr[kStaticMaxDevices] = {nullptr};   // device address of g_static_mask, per device

// |k| of pixel (ix, iy) in float64 with explicitly rounded operations, as in reduce.cu: membership is bit-exact
// against the float64 definition (k = m / L without 2 pi, FFT order).
__device__ __forceinline__ double static_k_abs(const int ix, const int iy, const int nx, const int ny, const double Lx,
                                               const double Ly) {
    const int m = ix < (nx + 1) / 2 ? ix : ix - nx, n = iy < (ny + 1) / 2 ? iy : iy - ny;
    const double kx = __ddiv_rn((double)m, Lx), ky = __ddiv_rn((double)n, Ly);
    return __dsqrt_rn(__dadd_rn(__dmul_rn(kx, kx), __dmul_rn(ky, ky)));
}

// mask[i] = 1 iff k_in <= |k_i| < k_out; writes all nx*ny bytes (nothing of an earlier call survives in that range)
__global__ void k_detector_mask_static(uint8_t* __restrict__ mask, const int nx, const int ny, const double Lx,
                                       const double Ly, const double k_in, const double k_out, const int has_out) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)nx * ny) return;
    const double k = static_k_abs((int)(i % nx), (int)(i / nx), nx, ny, Lx, Ly);
    mask[i] = (k >= k_in && (!has_out || k < k_out)) ? 1 : 0;
}

// one block per (probe, bin): masked sum over the pixels in the same fixed order as k_spectrum_image, so the result
// is reproducible and equal to ps_spectrum_image's
__global__ void __launch_bounds__(1024)
k_spectrum_image_static(const float* __restrict__ I, const uint8_t* __restrict__ mask, float* __restrict__ out,
                        const size_t npix) {
    __shared__ float sh[32];
    const float4* src = reinterpret_cast<const float4*>(I + (size_t)blockIdx.x * npix);   // blockIdx.x = p * n_bins + b
    const uchar4* m4 = reinterpret_cast<const uchar4*>(mask);
    float s = 0.f;
    for (size_t i = threadIdx.x; i < npix / 4; i += blockDim.x) {      // npix is a multiple of 1024
        const float4 x = src[i];
        const uchar4 m = m4[i];
        float q = m.x ? x.x : 0.f;
        q += m.y ? x.y : 0.f;
        q += m.z ? x.z : 0.f;
        q += m.w ? x.w : 0.f;
        s += q;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_down_sync(0xffffffffu, s, d);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) sh[w] = s;
    __syncthreads();
    if (w == 0) {
        s = sh[lane];                                                   // 1024 threads: all 32 slots are written
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s += __shfl_down_sync(0xffffffffu, s, d);
        if (lane == 0) out[blockIdx.x] = s;
    }
}

// device address of the static mask on c->device (which enter() has made current); looked up once per device
static ps_status static_mask_address(ps_ctx* c, uint8_t** out) {
    if (c->device < 0 || c->device >= kStaticMaxDevices)
        return fail(c, PS_EUNSUPPORTED, "ps_spectrum_image_static: device index beyond the 64 this entry point tracks");
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_mask_addr[c->device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_mask);
        if (e != cudaSuccess || !p)
            return fail(c, PS_ECUDA, std::string("ps_spectrum_image_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        g_static_mask_addr[c->device] = (uint8_t*)p;
    }
    *out = g_static_mask_addr[c->device];
    return PS_OK;
}

}  // namespace psb

using namespace psb;

extern "C" size_t ps_static_scratch_bytes(void) { return kStaticMaskBytes; }

extern "C" ps_status ps_spectrum_image_static(ps_ctx* c, const float* d_I, int P, int n_bins, double k_in, double k_out,
                                              float* d_out) {
    if (!c) return PS_EINVAL;
    ps_status st = enter(c, "ps_spectrum_image_static");
    if (st != PS_OK) return st;
    if (!c->have_geom) return fail(c, PS_ESTATE, "ps_spectrum_image_static: ps_set_geometry has not been called");
    if (!d_I || !d_out || P < 1 || n_bins < 1)
        return fail(c, PS_EINVAL, "ps_spectrum_image_static: null pointer or non-positive size");
    if (k_in < 0.0) return fail(c, PS_EINVAL, "ps_spectrum_image_static: k_in must be >= 0");
    const size_t npix = (size_t)c->nx * c->ny;
    if (npix > kStaticMaskBytes)
        return fail(c, PS_EUNSUPPORTED, "ps_spectrum_image_static: grid " + std::to_string(c->nx) + " x " + std::to_string(c->ny) +
                                            " = " + std::to_string(npix) + " pixels exceeds the built-in mask of " +
                                            std::to_string(kStaticMaskBytes) + " pixels (1024 x 1024); use ps_spectrum_image");
    if ((long long)P * n_bins > 2147483647LL)
        return fail(c, PS_EUNSUPPORTED, "ps_spectrum_image_static: more than 2^31-1 (probe, bin) pairs");
    uint8_t* d_mask = nullptr;
    if ((st = static_mask_address(c, &d_mask)) != PS_OK) return st;
    k_detector_mask_static<<<(unsigned)((npix + 255) / 256), 256, 0, c->stream>>>(d_mask, c->nx, c->ny, c->cell[0], c->cell[1],
                                                                                  k_in, k_out, k_out > 0.0 ? 1 : 0);
    PSB_LAUNCH_CHECK(c, "k_detector_mask_static");
    k_spectrum_image_static<<<P * n_bins, 1024, 0, c->stream>>>(d_I, d_mask, d_out, npix);
    PSB_LAUNCH_CHECK(c, "k_spectrum_image_static");
    return PS_OK;
}
