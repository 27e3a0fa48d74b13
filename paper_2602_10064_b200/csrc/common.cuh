// common.cuh — context object and host helpers shared by the translation units of libpyslice_b200.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <deque>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/pyslice_b200.h"

namespace psb {

constexpr int kColTile = 8;         // columns per tile of the column passes / activity granularity (16 measured
                                    // 2 % slower at 256^2: 192 instead of 176 of 256 columns touched)
constexpr int kMaxGrid = 2048;
constexpr int kMinGrid = 32;
constexpr int kNumSM = 148;         // B200

struct DeviceBuf {                  // library-owned device allocation, grown on demand
    void* p = nullptr;
    size_t bytes = 0;
};

struct KvTables {                   // tables that depend on the accelerating voltage
    double kV = -1.0;
    double lambda = 0.0, sigma = 0.0;
    float2* d_px_mid = nullptr;     // [nx]  exp(-i pi lambda dz kx^2) / (nx ny)   (inverse-FFT norm folded in)
    float2* d_px_last = nullptr;    // [nx]  exp(-i pi lambda dz kx^2) / sqrt(nx ny)
    float2* d_py = nullptr;         // [ny]  exp(-i pi lambda dz ky^2)
};

enum KernelId {                      // per-kernel timing slots (ps_profile_*)
    K_BIN = 0, K_SORT, K_VK, K_V_COL, K_V_ROW, K_INCIDENT, K_ROW_TRANSMIT, K_COL_PROPAGATE, K_TACAW_FFT,
    K_TACAW_ACCUM, K_TACAW_FINISH, K_REDUCE, K_SLICE_RESIDENT, K_COUNT
};
static const char* const kKernelNames[K_COUNT] = {
    "k_bin", "k_sort", "k_vk", "k_v_col", "k_v_row", "k_incident", "k_row_transmit", "k_col_propagate",
    "k_tacaw_fft", "k_tacaw_accum", "k_tacaw_finish", "k_reduce", "k_slice_resident"};

struct ProfRec { cudaEvent_t a, b; int id; };

// Pinned host staging ring: small host tables (bin lists, tilt indices, path points) are copied into page-locked
// memory owned by the ctx and sent with cudaMemcpyAsync, so the caller's array need not outlive the call and the
// hot path never waits for the stream.  A segment is reused only after the event recorded behind its copy has fired
// (cudaEventSynchronize on wrap-around: reached only if the device is a whole ring of uploads behind).
struct PinnedRing {
    struct Seg { size_t off, end; cudaEvent_t ev; };
    char* base = nullptr;
    size_t cap = 0, head = 0;
    std::deque<Seg> live;
    std::vector<cudaEvent_t> pool;
};

struct TacawStream {                // state of ps_tacaw_begin/add/finish
    bool active = false;
    int n_probes = 0, n_frames_total = 0, n_bins = 0, frames_seen = 0;
    void* d_acc = nullptr;
    DeviceBuf d_bins;               // [n_bins] bins mod F (library-owned)
    DeviceBuf d_ref;                // complex64 [P][ny][nx] reference wave subtracted from every frame
    DeviceBuf d_tw;                 // complex64 [chunk frames][n_bins] twiddles of the current chunk
    bool have_ref = false;
    std::vector<int32_t> bins;
    int next_frame = 0;             // chunks must arrive in ascending, contiguous frame order
};

}  // namespace psb

struct ps_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    long long launches = 0;
    psb::PinnedRing ring;                   // staging of small host tables (no host wait on the hot path)
    std::unordered_map<const void*, int> kern_cap;   // per kernel: resident blocks on this device (attributes set once)
    int* h_async_err = nullptr;             // mapped pinned word written by kernels (bad atomic number, ...)
    int* d_async_err = nullptr;             // its device alias
    int* d_bad_z = nullptr;                 // device-memory twin of the word: set by k_bin, read by k_poison (in stream order)

    // geometry
    bool have_geom = false;
    double cell[3] = {0, 0, 0};
    int nx = 0, ny = 0, n_slices = 0;
    double dz_eff = 0.0, kc = 0.0;
    int n_k_aperture = 0;
    int mcut = 0, ncut = 0;                 // largest |m|, |n| inside the aperture
    std::vector<int32_t> h_nmax;            // [nx] per column m (FFT order): max |n| with A=1, -1 if none
    int32_t* d_nmax = nullptr;
    std::vector<int32_t> h_tiles;           // active column tiles (kColTile columns) in the aperture
    int32_t* d_tiles = nullptr;
    uint8_t* d_tile_active = nullptr;       // [nx/kColTile]
    std::vector<int32_t> h_tile_slot;       // [nx/kColTile] position of a tile among the active ones, -1 if inactive
    int32_t* d_tile_slot = nullptr;
    int n_tiles_active = 0;
    int wave_chunk = 0;
    int vacuum_shortcut = 0;                // ps_set_vacuum_shortcut: rows with V == 0 skip the transmit + FFT pair (exact)
    int vk_mode = 0;                        // ps_set_vk_mode: 0 auto, 1 FP32 SIMT sums, 2 tcgen05 3xTF32 sums
    int tune_resident = 0;                  // ps_set_tuning("resident"): chip-resident slice loop, 0 auto, 1 always, -1 never
    int tune_row32 = 0;                     // ps_set_tuning("row32"): 32-value row pass at nx = 512/1024, 0 auto (off), 1 on, -1 off
    int tune_col32 = 0;                     // ps_set_tuning("col32"): 32-value column pass at ny = 512/1024, 0 auto (on), -1 off

    // form factors
    bool have_ff = false;
    int n_elem = 0, n_lorentz = 0, n_gauss = 0;
    std::vector<int32_t> ffZ;
    std::vector<double> ffcoef;
    float* d_ftab = nullptr;                // [n_elem][ncut+1][2 mcut+1]  C/(LxLy) f_Z(|k|) A(k)
    int32_t* d_elem_of_Z = nullptr;         // [128] element row of atomic number Z, -1 if absent
    bool ftab_valid = false;

    psb::KvTables kv;

    // aberrations (ps_set_aberrations): C10, C12, phi12, C21, phi21, C23, phi23, C30 (Angstrom / rad)
    bool have_ab = false;
    double ab[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    psb::DeviceBuf abtab;                   // complex64 [ny][nx] exp(-i chi(k)) for ab_kV
    double ab_kV = -1.0;

    // scratch
    psb::DeviceBuf scratch;                 // library-owned
    size_t scratch_budget = 0;              // bytes the library may use for scratch (decided at the first need)
    void* user_ws = nullptr;
    size_t user_ws_bytes = 0;

    psb::TacawStream ts;
    psb::DeviceBuf tacaw_groups;            // ps_tacaw: pixel-group lists [active..., inactive...] (first pixel of each)
    int tacaw_groups_C = 0;                 // group width the lists were built for (0 = not built)
    int tacaw_n_active = 0, tacaw_n_inactive = 0;
    psb::DeviceBuf tacaw_slot;              // ps_tacaw: output slot of every FFT bin (-1 = not requested)
    std::vector<int32_t> tacaw_slot_host;   // its host copy (uploaded again only when the bin list changes)
    psb::DeviceBuf misc;                    // detector mask + per-frame partial sums (ps_spectrum_image, ps_haadf)
    psb::DeviceBuf path_buf;                // ps_dispersion: path points (float64 kx, ky)
    psb::DeviceBuf inc_buf;                 // ps_make_incident: tilt indices / probe-aperture limits + probe positions
    std::vector<int32_t> inc_pmax_host;     // last uploaded probe-aperture limits (uploaded again only when they change)
    const void* z_checked = nullptr;        // ps_build_slices: (d_Z, n_atoms) already validated synchronously
    int z_checked_n = 0;
    psb::DeviceBuf qorder;                  // ps_qbin: cursor, offsets and pixel order by q bin (cached)
    bool qorder_valid = false;
    double qorder_dq = 0.0;
    int qorder_nq = 0;

    // optional per-launch timing (CUDA events on the ctx stream)
    bool prof_on = false;
    std::vector<psb::ProfRec> prof_pending;
    std::vector<cudaEvent_t> prof_pool;
    double prof_ms[psb::K_COUNT] = {0};
    long long prof_n[psb::K_COUNT] = {0};
};

namespace psb {

inline ps_status fail(ps_ctx* c, ps_status s, const std::string& msg) {
    if (c) c->err = msg;
    return s;
}

#define PSB_CUDA(ctx, expr)                                                                         \
    do {                                                                                            \
        cudaError_t _e = (expr);                                                                    \
        if (_e != cudaSuccess)                                                                      \
            return psb::fail((ctx), PS_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(_e)); \
    } while (0)

#define PSB_LAUNCH_CHECK(ctx, name)                                                                 \
    do {                                                                                            \
        cudaError_t _e = cudaGetLastError();                                                        \
        if (_e != cudaSuccess)                                                                      \
            return psb::fail((ctx), PS_ECUDA, std::string("launch ") + name + ": " + cudaGetErrorString(_e)); \
        (ctx)->launches++;                                                                          \
    } while (0)

// records an event pair around the launches made while it is alive (only when profiling is enabled)
struct ProfScope {
    ps_ctx* c; int id; cudaEvent_t a = nullptr, b = nullptr;
    ProfScope(ps_ctx* ctx, int kid) : c(ctx), id(kid) {
        if (!c->prof_on) return;
        for (cudaEvent_t* e : {&a, &b}) {
            if (!c->prof_pool.empty()) { *e = c->prof_pool.back(); c->prof_pool.pop_back(); }
            else if (cudaEventCreate(e) != cudaSuccess) { *e = nullptr; }
        }
        if (a && b) cudaEventRecord(a, c->stream);
    }
    ~ProfScope() {
        if (!c->prof_on || !a || !b) return;
        cudaEventRecord(b, c->stream);
        c->prof_pending.push_back({a, b, id});
    }
};

inline bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
inline int signed_index(int i, int n) { return i < (n + 1) / 2 ? i : i - n; }

ps_status ensure_buf(ps_ctx* c, DeviceBuf& b, size_t bytes);
// asynchronous upload of a small host table through the ctx's pinned ring (api.cu); never blocks in steady state
ps_status upload_async(ps_ctx* c, void* d_dst, const void* h_src, size_t bytes);
// makes c->device current, and reports (once) an error a kernel of an earlier asynchronous call has flagged
ps_status enter(ps_ctx* c, const char* who);

// Resident-block cap of `kern` on the ctx's device; the first use sets the dynamic shared-memory attribute.  Cached in
// the ctx (not in a process-wide static): attributes and occupancy are per device, and ctxs of different devices or
// host threads share nothing.
template <class K>
inline cudaError_t kernel_cap(ps_ctx* c, K kern, int threads, size_t smem, int* cap) {
    const void* key = reinterpret_cast<const void*>(kern);
    auto it = c->kern_cap.find(key);
    if (it != c->kern_cap.end()) { *cap = it->second; return cudaSuccess; }
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    int per_sm = 1, n_sm = kNumSM;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, c->device);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
    *cap = n_sm * per_sm;
    c->kern_cap.emplace(key, *cap);
    return cudaSuccess;
}
// Where the slice loop takes the projected potential from: the V array of ps_build_slices, or (ps_multislice_fused) the
// mixed array Zm[(f - zm_f0) * n_pairs + pair][y][kx] of a frame chunk — the y-transformed pair of slices, complex, in-band
// column tiles only — whose x-inverse transform the row pass then runs itself; `off` = sorted-atom offsets of that chunk
// ([frames][n_slices * n_elem + 1]), which say which slices of a pair are empty.
struct VSrc {
    const float* V = nullptr;
    const float2* Zm = nullptr;
    const int32_t* off = nullptr;
    int zm_f0 = 0;
};
// the slice loop of frames [fr0, fr0 + fr_n) of an exit array of n_frames frames (multislice.cu)
ps_status multislice_range(ps_ctx* c, double kV, const void* d_psi0, int n_probes, const VSrc& src, int n_frames, int fr0,
                           int fr_n, void* d_exit, int exit_layout);
ps_status ensure_kv(ps_ctx* c, double kV);
ps_status ensure_ftab(ps_ctx* c);
ps_status ensure_abtab(ps_ctx* c, double kV);                           // incident.cu
bool resident_supported(const ps_ctx* c);                               // resident.cu
cudaError_t launch_slice_resident(ps_ctx* c, float2* W, const float2* psi0, const float* V, int n_probes, int n_frames,
                                  float sigma, int col_lo, int col_hi);
cudaError_t launch_vk_tc(ps_ctx* c, const uint32_t* sUx, const uint32_t* sUy, const int32_t* off, float2* Vk, int n_atoms,
                         int nf);                                          // vk_tc.cu

// physical constants (CODATA values; DESIGN.md §3 "Constants")
constexpr double kHC_keVA = 12.398419843;
constexpr double kM0C2_keV = 510.99895;
constexpr double kBohr_A = 0.529177211;
constexpr double kE2_VA = 14.3996455;

}  // namespace psb
