// common.cuh — context object and host helpers shared by the translation units of libpyslice_b200.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string>
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
    K_TACAW_ACCUM, K_TACAW_FINISH, K_REDUCE, K_COUNT
};
static const char* const kKernelNames[K_COUNT] = {
    "k_bin", "k_sort", "k_vk", "k_v_col", "k_v_row", "k_incident", "k_row_transmit", "k_col_propagate",
    "k_tacaw_fft", "k_tacaw_accum", "k_tacaw_finish", "k_reduce"};

struct ProfRec { cudaEvent_t a, b; int id; };

struct TacawStream {                // state of ps_tacaw_begin/add/finish
    bool active = false;
    int n_probes = 0, n_frames_total = 0, n_bins = 0, frames_seen = 0;
    void* d_acc = nullptr;
    int32_t* d_bins = nullptr;      // [n_bins] bins mod F (library-owned)
    std::vector<int32_t> bins;
};

}  // namespace psb

struct ps_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    long long launches = 0;

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
    int n_tiles_active = 0;
    int wave_chunk = 0;
    int vacuum_shortcut = 0;                // ps_set_vacuum_shortcut: rows with V == 0 skip the transmit + FFT pair (exact)
    int vk_mode = 0;                        // ps_set_vk_mode: 0 auto, 1 FP32 SIMT sums, 2 tcgen05 3xTF32 sums

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
    psb::DeviceBuf misc;                    // small per-call tables (bin slots, path pixels)
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
ps_status ensure_kv(ps_ctx* c, double kV);
ps_status ensure_ftab(ps_ctx* c);
ps_status ensure_abtab(ps_ctx* c, double kV);                           // incident.cu
cudaError_t launch_vk_tc(ps_ctx* c, const uint32_t* sUx, const uint32_t* sUy, const int32_t* off, float2* Vk, int n_atoms,
                         int nf);                                          // vk_tc.cu

// physical constants (CODATA values; DESIGN.md §3 "Constants")
constexpr double kHC_keVA = 12.398419843;
constexpr double kM0C2_keV = 510.99895;
constexpr double kBohr_A = 0.529177211;
constexpr double kE2_VA = 14.3996455;

}  // namespace psb
