// api.cu — context life cycle, geometry / aperture tables, voltage tables, form-factor tables.
// Host-side setup only (not on the timed path).  Formulas: DESIGN.md §3 (readings A2-A7, A10, A11).
#include <math.h>

#include "common.cuh"

namespace psb {

static thread_local std::string g_create_err;

ps_status ensure_buf(ps_ctx* c, DeviceBuf& b, size_t bytes) {
    if (b.bytes >= bytes) return PS_OK;
    if (b.p) {
        PSB_CUDA(c, cudaStreamSynchronize(c->stream));       // growth only: never on a warmed-up hot path
        cudaFree(b.p);
        b.p = nullptr; b.bytes = 0;
    }
    cudaError_t e = cudaMalloc(&b.p, bytes);
    if (e != cudaSuccess) {
        b.p = nullptr;
        return fail(c, PS_EWORKSPACE, std::string("scratch allocation of ") + std::to_string(bytes) +
                                          " bytes failed: " + cudaGetErrorString(e));
    }
    b.bytes = bytes;
    return PS_OK;
}

// ------------------------------------------------------------------------------------ pinned staging ring
static constexpr size_t kRingBytes = (size_t)4 << 20;     // 4 MB: the largest steady-state table is a bin list (16 KB)

static cudaEvent_t ring_event(PinnedRing& r) {
    cudaEvent_t e = nullptr;
    if (!r.pool.empty()) { e = r.pool.back(); r.pool.pop_back(); return e; }
    if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return nullptr;
    return e;
}

ps_status upload_async(ps_ctx* c, void* d_dst, const void* h_src, size_t bytes) {
    if (bytes == 0) return PS_OK;
    PinnedRing& r = c->ring;
    if (!r.base) {
        PSB_CUDA(c, cudaHostAlloc((void**)&r.base, kRingBytes, cudaHostAllocDefault));
        r.cap = kRingBytes;
    }
    const size_t need = (bytes + 255) & ~(size_t)255;
    if (need > r.cap / 2) {                                  // a table too large for the ring (set-up paths only): blocking copy
        PSB_CUDA(c, cudaMemcpyAsync(d_dst, h_src, bytes, cudaMemcpyHostToDevice, c->stream));
        PSB_CUDA(c, cudaStreamSynchronize(c->stream));
        return PS_OK;
    }
    while (!r.live.empty() && cudaEventQuery(r.live.front().ev) == cudaSuccess) {   // retire finished copies
        r.pool.push_back(r.live.front().ev);
        r.live.pop_front();
    }
    if (r.head + need > r.cap) r.head = 0;                   // wrap
    const size_t lo = r.head, hi = r.head + need;
    // Any in-flight copy whose source overlaps [lo, hi) must finish first.  After a wrap the oldest segment may sit in
    // the skipped tail while younger ones occupy the start of the ring, so every live segment is examined, not only the
    // front.  Copies complete in stream order: waiting for the youngest overlapping one retires all that precede it.
    int last = -1;
    for (int i = 0; i < (int)r.live.size(); ++i)
        if (r.live[i].off < hi && r.live[i].end > lo) last = i;
    if (last >= 0) {
        PSB_CUDA(c, cudaEventSynchronize(r.live[last].ev));
        for (int i = 0; i <= last; ++i) {
            r.pool.push_back(r.live.front().ev);
            r.live.pop_front();
        }
    }
    memcpy(r.base + lo, h_src, bytes);
    PSB_CUDA(c, cudaMemcpyAsync(d_dst, r.base + lo, bytes, cudaMemcpyHostToDevice, c->stream));
    cudaEvent_t ev = ring_event(r);
    if (!ev) return fail(c, PS_ECUDA, "upload_async: cudaEventCreate failed");
    PSB_CUDA(c, cudaEventRecord(ev, c->stream));
    r.live.push_back({lo, hi, ev});
    r.head = hi;
    return PS_OK;
}

ps_status enter(ps_ctx* c, const char* who) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device) PSB_CUDA(c, cudaSetDevice(c->device));
    if (c->h_async_err) {
        const int z = *(volatile int*)c->h_async_err;        // written by k_bin of an earlier asynchronous call
        if (z != 0) {
            *(volatile int*)c->h_async_err = 0;
            if (c->d_bad_z) cudaMemsetAsync(c->d_bad_z, 0, sizeof(int), c->stream);   // builds queued from here on are clean
            return fail(c, PS_EUNSUPPORTED, std::string(who) + ": an earlier ps_build_slices met atomic number " +
                                                std::to_string(z == -1 ? 0 : z) + " without form-factor coefficients "
                                                "(its potentials are invalid)");
        }
    }
    return PS_OK;
}

template <class T>
static ps_status upload(ps_ctx* c, T** d, const std::vector<T>& h) {
    if (*d) { cudaFree(*d); *d = nullptr; }
    if (h.empty()) return PS_OK;
    PSB_CUDA(c, cudaMalloc((void**)d, h.size() * sizeof(T)));
    PSB_CUDA(c, cudaMemcpy(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    return PS_OK;
}

// relativistic de Broglie wavelength and interaction parameter (A3, A4)
static double wavelength_A(double kV) { return kHC_keVA / sqrt(kV * (2.0 * kM0C2_keV + kV)); }
static double sigma_rad_per_VA(double kV) {
    return (2.0 * M_PI / (wavelength_A(kV) * kV * 1.0e3)) * (kM0C2_keV + kV) / (2.0 * kM0C2_keV + kV);
}

ps_status ensure_kv(ps_ctx* c, double kV) {
    if (c->kv.kV == kV && c->kv.d_py) return PS_OK;
    PSB_CUDA(c, cudaStreamSynchronize(c->stream));
    const double lam = wavelength_A(kV);
    const int nx = c->nx, ny = c->ny;
    std::vector<float2> pxm(nx), pxl(nx), py(ny);
    const double inv_n = 1.0 / ((double)nx * ny), inv_sq = 1.0 / sqrt((double)nx * ny);
    for (int i = 0; i < nx; ++i) {
        const double kx = signed_index(i, nx) / c->cell[0];
        const double ph = -M_PI * lam * c->dz_eff * kx * kx;
        pxm[i] = make_float2((float)(cos(ph) * inv_n), (float)(sin(ph) * inv_n));
        pxl[i] = make_float2((float)(cos(ph) * inv_sq), (float)(sin(ph) * inv_sq));
    }
    for (int i = 0; i < ny; ++i) {
        const double ky = signed_index(i, ny) / c->cell[1];
        const double ph = -M_PI * lam * c->dz_eff * ky * ky;
        py[i] = make_float2((float)cos(ph), (float)sin(ph));
    }
    ps_status s;
    if ((s = upload(c, &c->kv.d_px_mid, pxm)) != PS_OK) return s;
    if ((s = upload(c, &c->kv.d_px_last, pxl)) != PS_OK) return s;
    if ((s = upload(c, &c->kv.d_py, py)) != PS_OK) return s;
    c->kv.kV = kV; c->kv.lambda = lam; c->kv.sigma = sigma_rad_per_VA(kV);
    return PS_OK;
}

static double form_factor(double q2, const double* coef, int nl, int ng) {
    const double *a = coef, *b = coef + nl, *cc = coef + 2 * nl, *d = coef + 2 * nl + ng;
    double f = 0.0;
    for (int i = 0; i < nl; ++i) f += a[i] / (q2 + b[i]);
    for (int i = 0; i < ng; ++i) f += cc[i] * exp(-d[i] * q2);
    return f;
}

ps_status ensure_ftab(ps_ctx* c) {
    if (c->ftab_valid) return PS_OK;
    if (!c->have_geom || !c->have_ff) return fail(c, PS_ESTATE, "geometry and form factors must be set first");
    const int mw = 2 * c->mcut + 1, nh = c->ncut + 1, ncoef = 2 * c->n_lorentz + 2 * c->n_gauss;
    const double pref = 2.0 * M_PI * kBohr_A * kE2_VA / (c->cell[0] * c->cell[1]);   // C/(Lx Ly), A2
    std::vector<float> tab((size_t)c->n_elem * nh * mw, 0.f);
    for (int e = 0; e < c->n_elem; ++e)
        for (int n = 0; n < nh; ++n)
            for (int mi = 0; mi < mw; ++mi) {
                const int m = mi - c->mcut;
                const int ix = m < 0 ? m + c->nx : m;
                if (n > c->h_nmax[ix]) continue;                                       // A(k) = 0
                const double kx = m / c->cell[0], ky = n / c->cell[1];
                tab[((size_t)e * nh + n) * mw + mi] =
                    (float)(pref * form_factor(kx * kx + ky * ky, &c->ffcoef[(size_t)e * ncoef], c->n_lorentz, c->n_gauss));
            }
    std::vector<int32_t> eoz(128, -1);
    for (int e = 0; e < c->n_elem; ++e) eoz[c->ffZ[e]] = e;
    ps_status s;
    if ((s = upload(c, &c->d_ftab, tab)) != PS_OK) return s;
    if ((s = upload(c, &c->d_elem_of_Z, eoz)) != PS_OK) return s;
    c->ftab_valid = true;
    return PS_OK;
}

}  // namespace psb

using namespace psb;

extern "C" const char* ps_version(void) { return "pyslice_b200 0.1 (sm_100a)"; }

extern "C" ps_status ps_create(ps_ctx** out, int device, void* cuda_stream) {
    if (!out) { g_create_err = "ps_create: out is NULL"; return PS_EINVAL; }
    *out = nullptr;
    int n_dev = 0;
    cudaError_t e = cudaGetDeviceCount(&n_dev);
    if (e != cudaSuccess || n_dev < 1) {
        g_create_err = std::string("ps_create: no CUDA device (") + cudaGetErrorString(e) + ")";
        return PS_ECUDA;
    }
    if (device < 0 || device >= n_dev) { g_create_err = "ps_create: device index out of range"; return PS_EINVAL; }
    if ((e = cudaSetDevice(device)) != cudaSuccess) {
        g_create_err = std::string("ps_create: cudaSetDevice: ") + cudaGetErrorString(e);
        return PS_ECUDA;
    }
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) {
        g_create_err = std::string("ps_create: cudaGetDeviceProperties: ") + cudaGetErrorString(e);
        return PS_ECUDA;
    }
    if (prop.major != 10) {
        g_create_err = "ps_create: this library holds sm_100a code only; device is sm_" + std::to_string(prop.major) +
                       std::to_string(prop.minor);
        return PS_EUNSUPPORTED;
    }
    ps_ctx* c = new (std::nothrow) ps_ctx();
    if (!c) { g_create_err = "ps_create: out of host memory"; return PS_EINVAL; }
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    // error word kernels can raise without the host waiting for them: page-locked, mapped into the device
    if (cudaHostAlloc((void**)&c->h_async_err, sizeof(int), cudaHostAllocMapped) == cudaSuccess) {
        *c->h_async_err = 0;
        if (cudaHostGetDevicePointer((void**)&c->d_async_err, c->h_async_err, 0) != cudaSuccess) c->d_async_err = nullptr;
    }
    if (!c->d_async_err) {
        g_create_err = "ps_create: mapped pinned allocation failed";
        if (c->h_async_err) cudaFreeHost(c->h_async_err);
        delete c;
        return PS_ECUDA;
    }
    if (cudaMalloc((void**)&c->d_bad_z, 256) != cudaSuccess || cudaMemset(c->d_bad_z, 0, 256) != cudaSuccess) {
        g_create_err = "ps_create: device allocation of the error word failed";
        cudaFree(c->d_bad_z); cudaFreeHost(c->h_async_err);
        delete c;
        return PS_ECUDA;
    }
    *out = c;
    return PS_OK;
}

extern "C" void ps_destroy(ps_ctx* c) {
    if (!c) return;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    if (c->h_async_err && *(volatile int*)c->h_async_err != 0)         // nobody called ps_check_async: do not lose it silently
        fprintf(stderr, "pyslice_b200: ps_destroy: an earlier ps_build_slices met an atomic number without form-factor "
                        "coefficients (%d) and its potentials were NaN-filled; the error was never read (ps_check_async)\n",
                *(volatile int*)c->h_async_err == -1 ? 0 : *(volatile int*)c->h_async_err);
    cudaFree(c->d_bad_z);
    cudaFree(c->d_nmax); cudaFree(c->d_tiles); cudaFree(c->d_tile_active); cudaFree(c->d_tile_slot);
    cudaFree(c->d_ftab); cudaFree(c->d_elem_of_Z);
    cudaFree(c->kv.d_px_mid); cudaFree(c->kv.d_px_last); cudaFree(c->kv.d_py);
    cudaFree(c->scratch.p); cudaFree(c->misc.p); cudaFree(c->qorder.p); cudaFree(c->ts.d_bins.p); cudaFree(c->ts.d_ref.p); cudaFree(c->ts.d_tw.p);
    cudaFree(c->path_buf.p); cudaFree(c->inc_buf.p);
    for (auto& sg : c->ring.live) cudaEventDestroy(sg.ev);
    for (auto e : c->ring.pool) cudaEventDestroy(e);
    if (c->ring.base) cudaFreeHost(c->ring.base);
    if (c->h_async_err) cudaFreeHost(c->h_async_err);
    cudaFree(c->tacaw_groups.p); cudaFree(c->abtab.p); cudaFree(c->tacaw_slot.p);
    for (auto& r : c->prof_pending) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto e : c->prof_pool) cudaEventDestroy(e);
    delete c;
}

extern "C" const char* ps_last_error(const ps_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

extern "C" long long ps_launch_count(const ps_ctx* c) { return c ? c->launches : 0; }

extern "C" ps_status ps_set_form_factors(ps_ctx* c, int n_elem, const int32_t* Z, int n_lorentz, int n_gauss,
                                         const double* coef) {
    if (!c) return PS_EINVAL;
    if (!Z || !coef || n_elem < 1 || n_elem > 16 || n_lorentz < 0 || n_gauss < 0 || n_lorentz + n_gauss < 1 ||
        n_lorentz > 8 || n_gauss > 8)
        return fail(c, PS_EINVAL, "ps_set_form_factors: need 1..16 elements and 1..8 terms of each kind");
    for (int e = 0; e < n_elem; ++e)
        if (Z[e] < 1 || Z[e] > 127) return fail(c, PS_EINVAL, "ps_set_form_factors: Z out of range 1..127");
    const int ncoef = 2 * n_lorentz + 2 * n_gauss;
    c->n_elem = n_elem; c->n_lorentz = n_lorentz; c->n_gauss = n_gauss;
    c->ffZ.assign(Z, Z + n_elem);
    c->ffcoef.assign(coef, coef + (size_t)n_elem * ncoef);
    c->have_ff = true;
    c->ftab_valid = false;
    c->z_checked = nullptr;                                  // the set of known atomic numbers changed
    return PS_OK;
}

extern "C" ps_status ps_set_geometry(ps_ctx* c, const double cell[3], int nx, int ny, double slice_dz) {
    if (!c) return PS_EINVAL;
    if (!cell || !(cell[0] > 0) || !(cell[1] > 0) || !(cell[2] > 0) || !(slice_dz > 0))
        return fail(c, PS_EINVAL, "ps_set_geometry: cell and slice_dz must be positive");
    if (!is_pow2(nx) || !is_pow2(ny) || nx < kMinGrid || ny < kMinGrid || nx > kMaxGrid || ny > kMaxGrid)
        return fail(c, PS_EUNSUPPORTED, "ps_set_geometry: nx, ny must be powers of two in [32, 2048]");
    PSB_CUDA(c, cudaSetDevice(c->device));
    PSB_CUDA(c, cudaStreamSynchronize(c->stream));
    c->cell[0] = cell[0]; c->cell[1] = cell[1]; c->cell[2] = cell[2];
    c->nx = nx; c->ny = ny;
    long ns = lround(cell[2] / slice_dz);                           // A7
    if (ns < 1) ns = 1;
    if (ns > 65535) return fail(c, PS_EUNSUPPORTED, "ps_set_geometry: more than 65535 slices");
    c->n_slices = (int)ns;
    c->dz_eff = cell[2] / c->n_slices;
    const double nyq_x = nx / (2.0 * cell[0]), nyq_y = ny / (2.0 * cell[1]);
    c->kc = (2.0 / 3.0) * (nyq_x < nyq_y ? nyq_x : nyq_y);          // A10
    const double kc2 = c->kc * c->kc;
    c->h_nmax.assign(nx, -1);
    c->mcut = 0; c->ncut = 0; c->n_k_aperture = 0;
    for (int ix = 0; ix < nx; ++ix) {
        const int m = signed_index(ix, nx);
        const double kx = m / cell[0];
        int best = -1;
        for (int n = 0; n < ny / 2; ++n) {
            const double ky = n / cell[1];
            if (kx * kx + ky * ky <= kc2) best = n; else break;     // A11: inclusive, float64
        }
        c->h_nmax[ix] = best;
        if (best >= 0) {
            c->n_k_aperture += 2 * best + 1;
            if (abs(m) > c->mcut) c->mcut = abs(m);
            if (best > c->ncut) c->ncut = best;
        }
    }
    const int nt = nx / kColTile;
    std::vector<uint8_t> act(nt, 0);
    c->h_tiles.clear();
    for (int tI = 0; tI < nt; ++tI) {
        for (int j = 0; j < kColTile; ++j)
            if (c->h_nmax[tI * kColTile + j] >= 0) act[tI] = 1;
        if (act[tI]) c->h_tiles.push_back(tI);
    }
    c->n_tiles_active = (int)c->h_tiles.size();
    ps_status s;
    if ((s = upload(c, &c->d_nmax, c->h_nmax)) != PS_OK) return s;
    if ((s = upload(c, &c->d_tiles, c->h_tiles)) != PS_OK) return s;
    if ((s = upload(c, &c->d_tile_active, act)) != PS_OK) return s;
    c->h_tile_slot.assign(nt, -1);                               // tile -> position among the active tiles (tiled exit layout)
    for (int j = 0; j < c->n_tiles_active; ++j) c->h_tile_slot[c->h_tiles[j]] = j;
    if ((s = upload(c, &c->d_tile_slot, c->h_tile_slot)) != PS_OK) return s;
    c->kv.kV = -1.0;
    c->ftab_valid = false;
    c->qorder_valid = false;
    c->tacaw_groups_C = 0;
    c->ab_kV = -1.0;
    c->have_geom = true;
    return PS_OK;
}

extern "C" ps_status ps_get_geometry(const ps_ctx* c, int* n_slices, double* dz_eff, int* n_k_aperture) {
    if (!c) return PS_EINVAL;
    if (!c->have_geom) return PS_ESTATE;
    if (n_slices) *n_slices = c->n_slices;
    if (dz_eff) *dz_eff = c->dz_eff;
    if (n_k_aperture) *n_k_aperture = c->n_k_aperture;
    return PS_OK;
}

extern "C" ps_status ps_set_wave_chunk(ps_ctx* c, int n_waves) {
    if (!c) return PS_EINVAL;
    if (n_waves < 0) return fail(c, PS_EINVAL, "ps_set_wave_chunk: negative chunk");
    c->wave_chunk = n_waves;
    return PS_OK;
}

extern "C" ps_status ps_set_vacuum_shortcut(ps_ctx* c, int on) {
    if (!c) return PS_EINVAL;
    c->vacuum_shortcut = on ? 1 : 0;
    return PS_OK;
}

extern "C" ps_status ps_set_vk_mode(ps_ctx* c, int mode) {
    if (!c) return PS_EINVAL;
    if (mode < 0 || mode > 2) return fail(c, PS_EINVAL, "ps_set_vk_mode: mode must be 0 (auto), 1 (FP32 SIMT) or 2 (tcgen05 3xTF32)");
    c->vk_mode = mode;
    return PS_OK;
}

extern "C" ps_status ps_set_tuning(ps_ctx* c, const char* key, int value) {
    if (!c) return PS_EINVAL;
    if (!key) return fail(c, PS_EINVAL, "ps_set_tuning: key is NULL");
    const std::string k(key);
    if (k == "resident") {
        if (value < -1 || value > 1) return fail(c, PS_EINVAL, "ps_set_tuning: resident must be -1 (never), 0 (auto) or 1 (always)");
        c->tune_resident = value;
    } else if (k == "row32") {
        if (value < -1 || value > 1) return fail(c, PS_EINVAL, "ps_set_tuning: row32 must be -1 (off), 0 (auto) or 1 (on)");
        c->tune_row32 = value;
    } else if (k == "col32") {
        if (value < -1 || value > 1) return fail(c, PS_EINVAL, "ps_set_tuning: col32 must be -1 (off), 0 (auto) or 1 (on)");
        c->tune_col32 = value;
    } else {
        return fail(c, PS_EINVAL, "ps_set_tuning: unknown key '" + k + "'");
    }
    return PS_OK;
}

extern "C" ps_status ps_set_workspace(ps_ctx* c, void* d_ws, size_t bytes) {
    if (!c) return PS_EINVAL;
    if (d_ws && bytes == 0) return fail(c, PS_EINVAL, "ps_set_workspace: zero-sized workspace");
    if (((uintptr_t)d_ws & 255u) != 0) return fail(c, PS_EINVAL, "ps_set_workspace: pointer must be 256-byte aligned");
    c->user_ws = d_ws;
    c->user_ws_bytes = d_ws ? bytes : 0;
    return PS_OK;
}

extern "C" ps_status ps_check_async(ps_ctx* c) {
    if (!c) return PS_EINVAL;
    PSB_CUDA(c, cudaSetDevice(c->device));
    PSB_CUDA(c, cudaStreamSynchronize(c->stream));
    return enter(c, "ps_check_async");
}

extern "C" ps_status ps_profile_enable(ps_ctx* c, int on) {
    if (!c) return PS_EINVAL;
    c->prof_on = on != 0;
    return PS_OK;
}

extern "C" ps_status ps_profile_read(ps_ctx* c, int reset, int* n_kernels, const char** names, double* ms,
                                     long long* launches) {
    if (!c) return PS_EINVAL;
    if (!c->prof_pending.empty()) {
        PSB_CUDA(c, cudaStreamSynchronize(c->stream));
        for (auto& r : c->prof_pending) {
            float t = 0.f;
            if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess) { c->prof_ms[r.id] += t; c->prof_n[r.id]++; }
            c->prof_pool.push_back(r.a); c->prof_pool.push_back(r.b);
        }
        c->prof_pending.clear();
    }
    if (n_kernels) *n_kernels = K_COUNT;
    for (int i = 0; i < K_COUNT; ++i) {
        if (names) names[i] = kKernelNames[i];
        if (ms) ms[i] = c->prof_ms[i];
        if (launches) launches[i] = c->prof_n[i];
        if (reset) { c->prof_ms[i] = 0.0; c->prof_n[i] = 0; }
    }
    return enter(c, "ps_profile_read");                           // the outputs above are filled either way
}
