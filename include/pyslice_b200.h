/* pyslice_b200.h — C ABI of the B200-native TACAW hot path (arxiv 2602.10064, "PySlice").
 *
 * What the library computes (citations are lines of the paper text, PAPER.md, with the
 * section / equation they fall in; readings A1..A22 are listed in DESIGN.md §3):
 *
 *   PAPER.md:81  (§2.2 "Atomic Scattering Potentials")
 *        f(q) = sum_i a_i/(q^2+b_i) + sum_i c_i exp(-d_i q^2)
 *        V_s(k) = sum_{j in slice s} f_Zj(|k|) exp(-2 pi i k.r_j),  inverse FFT -> V_s(r)
 *   PAPER.md:79  (§2.2 "Multislice")
 *        t(r) = exp(i sigma V(r)),  P(k) = exp(-i pi lambda dz |k|^2),
 *        psi_exit = P_{N-1} t_N ... P_1 t_2 P_0 t_1 psi_probe
 *   PAPER.md:89  (§2.2 data containers)  exit waves indexed (probe, time, kx, ky): k-space
 *   PAPER.md:73  (§2.1 "TACAW")
 *        psi~(k,w) = F_t[ psi(k,t) - <psi(k,t)>_t ],   I(k,w) = |psi~(k,w)|^2
 *   PAPER.md:89, 394, 397, 422  dispersion(), spectral_diffraction(), spectrum_image()
 *   PAPER.md:289-301 (Suppl. Eq. 4-6)  dk = 1/L, df = 1/(N dt), f_max = 1/(2 dt)
 *
 * Conventions
 *   - Every pointer named d_* is DEVICE memory owned by the caller (e.g. a torch tensor);
 *     every other pointer is HOST memory, read during the call and never retained.
 *   - All hot-path calls enqueue their work on the stream given to ps_create() and return; the
 *     library never frees caller memory.  WHEN A CALL MAY BLOCK THE HOST (and only then):
 *       (a) set-up: ps_set_geometry, and the first hot-path call after a change of geometry,
 *           voltage, form factors or aberration coefficients (tables are rebuilt on the host);
 *       (b) growth: a call that needs more library-owned scratch than any earlier call
 *           (the buffer is re-allocated after a stream wait);
 *       (c) ps_build_slices the first time it sees a (d_Z, n_atoms) pair: one 4-byte read-back
 *           validates the atomic numbers before any work is queued;
 *       (d) ps_profile_read, ps_destroy.
 *     A repeated call with the same parameters and sizes ("warmed up") never waits for the
 *     device: small host tables (bin lists, tilt indices, probe positions, path points) are
 *     copied into a page-locked staging ring owned by the ctx and sent with cudaMemcpyAsync,
 *     so host arrays are never retained past the call.
 *   - Asynchronous errors: ps_build_slices re-checks every atomic number on the device in
 *     every call; an unknown Z met by a call that did not validate synchronously (case c: the
 *     same (d_Z, n_atoms) pair as a validated call, e.g. Z edited in place, or a new tensor the
 *     allocator placed at the old address) is raised through a page-locked word and reported as
 *     PS_EUNSUPPORTED by the next ps_* call on the ctx that observes it.  What that call produced
 *     is not left looking valid: its V (ps_build_slices) or its potential chunk and with it the
 *     exit waves (ps_multislice_fused) are filled with NaN on the device.  ps_check_async() waits
 *     for the stream and reports the word; call it after the last call of a run, before results
 *     are read.  ps_profile_read reports it too, and ps_destroy prints a warning to stderr if it
 *     was never read.
 *   - Scratch memory the library needs is allocated by the ctx itself (cudaMalloc, grown
 *     on demand, freed by ps_destroy) unless the caller installs a workspace with
 *     ps_set_workspace().
 *   - Every failure is a negative ps_status plus a message from ps_last_error(); nothing
 *     aborts or throws across this boundary.  There is no CPU fallback of any kind.
 *   - Grids: nx, ny powers of two in [32, 2048]; cells orthorhombic (Angstrom).
 *     k = m/L (no 2 pi), FFT index order 0..N/2-1,-N/2..-1, forward transform
 *     exp(-2 pi i ...), as numpy (A1).
 *   - Band limit (A10): A(k) = [kx^2+ky^2 <= kc^2], kc = (2/3) min(nx/(2Lx), ny/(2Ly)),
 *     applied in every propagator, to V(k) and to the probe.
 *   - Results are deterministic for fixed inputs (no floating-point atomics anywhere).
 *   - One ctx per host thread at a time; ctxs share no state (kernel attributes and
 *     occupancy figures are cached per ctx, i.e. per device), so one process may drive several
 *     devices or threads with one ctx each.  Every call makes the ctx's device current.
 */
#ifndef PYSLICE_B200_H
#define PYSLICE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define PS_API __attribute__((visibility("default")))
#else
#define PS_API
#endif

typedef struct ps_ctx ps_ctx;   /* opaque: owns its tables, plans and the scratch it allocated */

typedef enum {
    PS_OK = 0,
    PS_EINVAL = -1,        /* bad argument (null pointer, size <= 0, bin out of range, ...)   */
    PS_EUNSUPPORTED = -2,  /* non power-of-two grid, grid out of range, Z without coefficients,
                              n_frames not a power of two in ps_tacaw, ...                     */
    PS_EWORKSPACE = -3,    /* installed workspace too small / scratch allocation failed       */
    PS_ECUDA = -4,         /* a CUDA runtime call or kernel launch failed                      */
    PS_ESTATE = -5         /* call order violated (geometry / form factors not set, ...)       */
} ps_status;

/* exit-wave layouts (PAPER.md:89 WFData "indexed by probe position, time, and reciprocal space
 * coordinates").  Values are identical in both; ps_exit_bytes gives the size of an array, ps_exit_to_dense converts. */
#define PS_LAYOUT_DENSE 0           /* complex64 [P][F][ny][nx], k-space, FFT index order (A13); accepted everywhere */
#define PS_LAYOUT_TILED_APERTURE 1  /* complex64 [P][ny][n_tiles][F][8]: only the column tiles (8 adjacent kx, FFT order,
                                     * ascending) that hold at least one in-band point, and the F frames of a (row, tile)
                                     * contiguous: the time transform streams F*64-byte runs instead of gathering 64-byte
                                     * pieces 8*nx*ny bytes apart.  n_tiles/(nx/8) = 0.69 of the dense size at the 2/3
                                     * band limit.  Written by ps_multislice (the wave is then propagated chunk by chunk in
                                     * a work array in scratch / the installed workspace), read by ps_tacaw, ps_haadf and
                                     * ps_exit_to_dense; ps_tacaw_add (chunks of a stream) and ps_apply_aberrations take
                                     * dense arrays. */

/* ---------------------------------------------------------------- life cycle */

/* Create a context bound to CUDA device `device` and to `cuda_stream` (a cudaStream_t; NULL =
 * the legacy default stream).  Fails with PS_ECUDA when no usable device exists. */
PS_API ps_status ps_create(ps_ctx** out, int device, void* cuda_stream);
PS_API void ps_destroy(ps_ctx* ctx);
/* Message of the last failure on this ctx (valid until the next call on it); "" if none.
 * With ctx == NULL returns the message of the last failed ps_create of this thread. */
PS_API const char* ps_last_error(const ps_ctx* ctx);
/* Library version string, e.g. "pyslice_b200 0.1 (sm_100a)". */
PS_API const char* ps_version(void);

/* ---------------------------------------------------------------- host-side setup (not timed) */

/* Form-factor coefficients, general (n_lorentz, n_gauss) form (A5):
 *   f_Z(q) = sum_{i<n_lorentz} a_i/(q^2+b_i) + sum_{i<n_gauss} c_i exp(-d_i q^2),  q = |k| in 1/A.
 * coef is host [n_elem][2*n_lorentz+2*n_gauss], row layout a.., b.., c.., d..
 * (a: 1/A, b: 1/A^2, c: A, d: A^2).  Z lists the atomic number of each row.  Copied. */
PS_API ps_status ps_set_form_factors(ps_ctx* ctx, int n_elem, const int32_t* Z, int n_lorentz, int n_gauss,
                              const double* coef);

/* Cell (orthorhombic, Angstrom), grid and slicing (A7):
 * n_slices = max(1, round(Lz/slice_dz)), dz_eff = Lz/n_slices; slices are half-open
 * [s dz, (s+1) dz), z wrapped periodically, beam along +z (A8).  Builds the aperture tables. */
PS_API ps_status ps_set_geometry(ps_ctx* ctx, const double cell[3], int nx, int ny, double slice_dz);
/* n_k_aperture = number of grid points with A(k) = 1.  Any out pointer may be NULL. */
PS_API ps_status ps_get_geometry(const ps_ctx* ctx, int* n_slices, double* dz_eff, int* n_k_aperture);

/* Scratch needed by ps_build_slices / ps_multislice_fused on `n_frames_chunk` frames of `n_atoms` atoms at
 * a time (fixed-point coordinates and sort keys, 5 x 4 B per atom-frame, plus V(k) and the mixed
 * array of the inverse transform, which depend on the geometry alone).  The only other user of
 * scratch is ps_multislice with PS_LAYOUT_TILED_APERTURE, whose dense work array takes nx*ny*8
 * bytes per wave of a chunk (it uses whatever the workspace or the library-owned buffer holds).
 * NOTE: SURVEY.md 8(b) sketched the second argument as `n_probes_chunk`; the probe count does not
 * enter the scratch of the potential build (and ps_multislice with the dense layout propagates in
 * place inside d_exit and needs none), while the atom count does, so the argument is `n_atoms`.  Returns 0 before geometry and form
 * factors are set.  ps_set_workspace installs caller-owned device memory (d_ws == NULL removes
 * it and returns the ctx to self-allocation).  ps_build_slices processes frames in chunks that
 * fit whatever scratch is available. */
PS_API size_t    ps_workspace_bytes(const ps_ctx* ctx, int n_frames_chunk, int n_atoms);
PS_API ps_status ps_set_workspace(ps_ctx* ctx, void* d_ws, size_t bytes);

/* Tuning knob: number of waves whose slice loop runs back to back (a small chunk stays resident in
 * the 126 MB L2 between the two FFT passes of a slice; a large one amortises launch costs).
 * 0 = library default = the whole batch in one launch per pass (profiles/r1_chunk_sweep.md). */
PS_API ps_status ps_set_wave_chunk(ps_ctx* ctx, int n_waves);

/* Named tuning knobs (results are identical to rounding order):
 *   "resident"  chip-resident slice loop for square grids nx = ny <= 128 (one launch per ps_multislice, the wave kept
 *               in shared memory through all slices; resident.cu): 0 = auto (batches of at most 2 x 148 waves, which
 *               cannot fill the GPU with streaming launches), 1 = always, -1 = never
 *   "row32"     the row pass of ps_multislice at nx = 512 and 1024 (slices after the first) with 32 values per thread:
 *               0 = auto (off: measured slower than the 16-value pass), 1 = on, -1 = off
 *   "col32"     the column pass of ps_multislice at ny = 512 and 1024 with 32 values per thread (one shared-memory exchange
 *               per transform instead of two): 0 = auto (on), 1 = on, -1 = off (the 16-value pass used at every other size)
 * Unknown keys and values are PS_EINVAL. */
PS_API ps_status ps_set_tuning(ps_ctx* ctx, const char* key, int value);

/* Tuning knob (default off, so that every row of every slice goes through the full transforms): rows of a slice on which V is exactly zero (vacuum) have exp(i sigma V) = 1, and the
 * inverse + forward row transform around it is NX times the identity, so ps_multislice only rescales such rows (an
 * exact shortcut, decided from d_V itself row group by row group; measured +4 % on config 2, whose slices are 90 % vacuum). */
PS_API ps_status ps_set_vacuum_shortcut(ps_ctx* ctx, int on);

/* Tuning knob: how ps_build_slices forms the structure-factor sums of V(k).
 *   1 = FP32 FMA pipes (k_vk);  2 = tensor cores, tcgen05.mma kind::tf32 with the 3xTF32 operand split, FP32
 *   accumulation in TMEM (k_vk_tc);  0 = library default (2 when the mean (slice, element) group has >= 48 atoms). */
PS_API ps_status ps_set_vk_mode(ps_ctx* ctx, int mode);

/* Aberrations (A24).  coef = {C10, C12, phi12, C21, phi21, C23, phi23,
 * C30} in Angstrom / radians (host, 8 doubles; NULL switches aberrations off):
 *   chi(k) = (2 pi/lambda) [C10 th^2/2 + C12 th^2/2 cos 2(phi-phi12) + C21 th^3/3 cos(phi-phi21)
 *                           + C23 th^3/3 cos 3(phi-phi23) + C30 th^4/4],   th = lambda |k|, phi = atan2(ky, kx).
 * While set, ps_make_incident builds probes as A(k) exp(-i chi) exp(-2 pi i k.r_p).  ps_apply_aberrations multiplies
 * n_waves stored k-space waves complex64 [n_waves][ny][nx] (exit waves of ps_multislice) by exp(-i chi) in place. */
PS_API ps_status ps_set_aberrations(ps_ctx* ctx, const double* coef);
PS_API ps_status ps_apply_aberrations(ps_ctx* ctx, double kV, void* d_waves_k, long long n_waves);

/* ---------------------------------------------------------------- hot path */

/* a0+a2+a3: projected potentials of every slice of every frame.
 *   d_pos        float32 [n_frames][n_atoms][3] Cartesian positions, Angstrom
 *   d_Z          int32   [n_atoms] atomic numbers (every value must have coefficients)
 *   d_V          float32 [n_frames][n_slices][ny][nx], V*Angstrom               (written)
 *   d_slice_idx  int32   [n_frames][n_atoms] slice of every atom, or NULL       (written)
 * Fixed-point ingest: u = pos/L - floor(pos/L) (float64), U = floor(u 2^32) clamped,
 * slice = (U_z * n_slices) >> 32 — bit-exact against the oracle. */
PS_API ps_status ps_build_slices(ps_ctx* ctx, const float* d_pos, const int32_t* d_Z, int n_frames, int n_atoms,
                          float* d_V, int32_t* d_slice_idx);

/* a4: incident waves (PAPER.md:378-380 plane wave; 404-419 focused probe; A12, A18).
 *   semi_angle_mrad == 0 and is_tilt == 0 : plane wave psi0 = 1 (xy ignored, may be NULL)
 *   is_tilt != 0 : xy_or_tilt[i] = integer reciprocal-grid point (m_t, n_t):
 *                  psi0 = exp(2 pi i (m_t x/Lx + n_t y/Ly))
 *   else         : probe at xy_or_tilt[i] = (x0, y0) Angstrom:
 *                  Psi0(k) = [lambda|k| <= alpha] A(k) exp(-2 pi i k.r0), psi0 = ifft2(Psi0),
 *                  scaled so that sum_r |psi0|^2 = nx ny.
 *   d_psi0  complex64 [n][ny][nx], real space                                   (written) */
PS_API ps_status ps_make_incident(ps_ctx* ctx, double kV, double semi_angle_mrad, int n, const double* xy_or_tilt,
                           int is_tilt, void* d_psi0);

/* a5+a6: multislice for every (probe, frame) pair:
 *   for s = 0..S-1: psi <- psi exp(i sigma V_s); psi <- ifft2(P A fft2(psi));
 *   exit = fft2(psi)/sqrt(nx ny)   (k-space, unitary, A9, A13)
 *   d_psi0  complex64 [n_probes][ny][nx]
 *   d_V     float32   [n_frames][n_slices][ny][nx]
 *   d_exit  exit waves in `exit_layout` (ps_exit_bytes bytes)                   (written)
 * PS_LAYOUT_DENSE: the wave is propagated in place inside d_exit (no other wave storage).  PS_LAYOUT_TILED_APERTURE: it is
 * propagated in a dense work array of as many waves as the scratch holds (installed workspace, else a library-owned
 * buffer of an eighth of the free device memory, 768 MB ... 16 GB), chunk by chunk, and the last column pass of every
 * chunk writes the k-space exit waves straight into the tiled array. */
PS_API ps_status ps_multislice(ps_ctx* ctx, double kV, const void* d_psi0, int n_probes, const float* d_V,
                        int n_frames, void* d_exit, int exit_layout);

/* a0 ... a6 in one call, without the V array (second half; "An inverse FFT then yields
 * the real-space projected potential"): positions -> exit waves.  Frame chunk by frame chunk (as many frames
 * as the scratch holds) the library bins and sorts the atoms, forms V(k) and its y-inverse transform, and runs the slice
 * loop of those frames with a row pass that performs the x-inverse transform of the slice pair itself: the projected
 * potential exists only row by row in shared memory and never travels through HBM.  Same values as ps_build_slices
 * followed by ps_multislice to FP32 rounding (the same transforms in the same order).  It costs a third 1-D transform per
 * row and slice, so it pays only where V would be used once (a single probe per frame) and memory, not time, is short:
 * measured numbers in DESIGN.md section 10.  d_exit: PS_LAYOUT_DENSE only (the wave is propagated in place).
 *   d_pos float32 [n_frames][n_atoms][3], d_Z int32 [n_atoms], d_psi0 complex64 [n_probes][ny][nx],
 *   d_exit complex64 [n_probes][n_frames][ny][nx]                                (written) */
PS_API ps_status ps_multislice_fused(ps_ctx* ctx, double kV, const void* d_psi0, int n_probes, const float* d_pos,
                              const int32_t* d_Z, int n_frames, int n_atoms, void* d_exit, int exit_layout);

/* Bytes of an exit-wave array of n_probes x n_frames waves in `exit_layout` (0 for an unknown layout or before
 * ps_set_geometry).  ps_exit_to_dense expands a PS_LAYOUT_TILED_APERTURE array into the dense one (exact zeros in the
 * column tiles the tiled layout does not store); both arrays caller-owned device memory, asynchronous on the ctx stream. */
PS_API size_t    ps_exit_bytes(const ps_ctx* ctx, int n_probes, int n_frames, int exit_layout);
PS_API ps_status ps_exit_to_dense(ps_ctx* ctx, const void* d_tiled, int n_probes, int n_frames, void* d_dense);

/* a7: TACAW transform (A14): for every probe and k,
 *   Psi~_n = sum_j (Psi_j - <Psi>_t) exp(-2 pi i n j / F),  I = |Psi~_n|^2,  f_n = n/(F dt).
 *   bins: host list of n_bins signed FFT bins n (taken mod F), or NULL for all F bins in FFT
 *   order (then n_bins must equal n_frames).  n_frames must be a power of two in [32, 4096].
 *   d_I  float32 [n_probes][n_bins][ny][nx]                                      (written)
 * dt_fs only defines the frequency axis (f_n in THz = n/(F dt_fs 1e-3)); it does not enter I. */
PS_API ps_status ps_tacaw(ps_ctx* ctx, const void* d_exit, int exit_layout, int n_probes, int n_frames, double dt_fs,
                   int n_bins, const int32_t* bins, float* d_I);

/* Streaming variant for frames x grid > HBM (BASELINE config 4, Suppl. Eq. 5 at PAPER.md:295): per-bin DFT
 * accumulation over frame chunks,
 *     acc[p][b][k] += sum_{j in chunk} (Psi_j - ref) e^{-2 pi i n_b j / F},      finish: I = |acc_b|^2, bin 0 := 0.
 * `ref` is one wave per probe subtracted from every frame (it strips the elastic part so that fp32 partial sums stay
 * small; over the complete set of F frames a constant shift changes no bin n != 0, and bin 0 of the mean-subtracted
 * series is zero by definition (A14), so the result equals F_t[Psi - <Psi>_t] for integer bins).  By default ref = the
 * first frame the stream receives; ps_tacaw_set_reference installs another one (copied; NULL = zeros) — required when
 * several streams (GPUs) each sum a shard of the frames and their accumulators are added afterwards: all shards must
 * subtract the SAME wave.
 *   d_acc  complex64 [n_probes][n_bins][ny][nx], zeroed by begin; any n_frames_total >= 1.
 * Every exit value of a chunk is read from HBM once; the accumulators are read and written once per 64 frames. */
PS_API ps_status ps_tacaw_begin(ps_ctx* ctx, int n_probes, int n_frames_total, double dt_fs, int n_bins,
                         const int32_t* bins, void* d_acc);
/* Optional, after begin and before the first add: d_ref complex64 [n_probes][ny][nx] (device), or NULL for zeros. */
PS_API ps_status ps_tacaw_set_reference(ps_ctx* ctx, const void* d_ref);
/* d_exit_chunk complex64 [n_probes][n_frames_chunk][ny][nx] = frames frame0.. of every probe.  Chunks must arrive in
 * ascending, contiguous frame order (the first chunk may start at any frame: a shard); anything else is PS_ESTATE. */
PS_API ps_status ps_tacaw_add(ps_ctx* ctx, const void* d_exit_chunk, int frame0, int n_frames_chunk);
/* PS_ESTATE unless exactly n_frames_total frames were added. */
PS_API ps_status ps_tacaw_finish(ps_ctx* ctx, float* d_I /* float32 [n_probes][n_bins][ny][nx] */);
/* Sharded finish (frame shards + reduce-scatter): the caller has summed the accumulators of all shards
 * (each fed through begin / set_reference / add on its own ctx) and owns n_k of the k points of every (probe, bin):
 *   d_acc_shard complex64 [n_probes][n_bins][n_k]  ->  d_I_shard float32 [n_probes][n_bins][n_k].
 * No frame-count check (this ctx saw only its shard); ends the stream like ps_tacaw_finish. */
PS_API ps_status ps_tacaw_finish_shard(ps_ctx* ctx, const void* d_acc_shard, size_t n_k, float* d_I_shard);

/* a8: reductions over d_I = float32 [P][n_bins][ny][nx] (A15-A17).
 * ps_sdp: spectral diffraction pattern, sum over probes and bins bin_lo..bin_hi inclusive
 *         (positions in the bin list) -> d_out float32 [ny][nx]. */
PS_API ps_status ps_sdp(ps_ctx* ctx, const float* d_I, int P, int n_bins, int bin_lo, int bin_hi, float* d_out);
/* ps_spectrum_image: d_out[p][b] = sum over k with k_in <= |k| < k_out (1/A; k_out <= 0 means
 * no outer limit) of I[p][b][k] -> float32 [P][n_bins]. */
PS_API ps_status ps_spectrum_image(ps_ctx* ctx, const float* d_I, int P, int n_bins, double k_in, double k_out,
                            float* d_out);
/* ps_spectrum_image_static: same arguments, same result as ps_spectrum_image (A16), for callers that
 * cannot let the library allocate: a process that has handed all free HBM to its own pool at start-up (a cudaMalloc
 * made by the library then fails), or a latency-bound loop that cannot take the device-wide stall of cudaMalloc /
 * cudaFree.  ps_spectrum_image keeps its one-byte-per-pixel detector mask in a ctx buffer from cudaMalloc; this
 * variant keeps it in a fixed 1 MiB array inside the library image and calls no allocator, ever.
 *   - Cost: every GPU that loads the library holds those ps_static_scratch_bytes() bytes until the process exits.
 *   - Limit: nx * ny <= ps_static_scratch_bytes() (1024 x 1024 pixels); larger grids return PS_EUNSUPPORTED with a
 *     message and launch nothing.
 *   - One array per device, shared by all ctxs and streams: calls that can overlap on the GPU race on it (wrong
 *     results, no error).  Keep them in one stream or order them yourself.  The array keeps the previous call's
 *     bytes; each call rewrites every byte it later reads, so no clearing is needed or done.
 *   - The first call on a device looks up the array's device address (cudaGetSymbolAddress, once per device, with
 *     that device current) and may trigger module loading: make that first call before any stream capture begins.
 * d_I and d_out are caller-owned device memory as for ps_spectrum_image; asynchronous on the ctx stream. */
PS_API ps_status ps_spectrum_image_static(ps_ctx* ctx, const float* d_I, int P, int n_bins, double k_in, double k_out,
                                   float* d_out);
/* size in bytes (= pixels) of the built-in scratch array used by ps_spectrum_image_static */
PS_API size_t ps_static_scratch_bytes(void);
/* ps_haadf: annular detector on the k-space exit waves,
 *   d_out[p] = (1/F) sum_f sum_{k_in <= |k| < k_out} |Psi_pf(k)|^2 / (nx ny)      (k_out <= 0: no outer limit)
 * = fraction of the incident intensity on the detector, averaged over frames -> float32 [n_probes].
 * d_exit: exit waves as written by ps_multislice, in either layout. */
PS_API ps_status ps_haadf(ps_ctx* ctx, const void* d_exit, int exit_layout, int n_probes, int n_frames, double k_in,
                   double k_out, float* d_out);
/* ps_accumulate_intensity: d_acc <- w_acc * d_acc + w_new * d_I over
 * n_values float32 (16-byte aligned, n_values % 4 == 0): averaging |Psi(k,w)|^2 over independent trajectories or
 * trajectory segments; the running mean over n results uses w_acc = (n-1)/n, w_new = 1/n. */
PS_API ps_status ps_accumulate_intensity(ps_ctx* ctx, float* d_acc, const float* d_I, size_t n_values, double w_acc,
                                  double w_new);
/* ps_dispersion: nearest grid pixel of each path point, ix = floor(kx Lx + 0.5) mod nx (A17);
 * d_pix int32 [n_path] = iy*nx+ix (bit-exact), d_out[b][i] = sum_p I[p][b][pix_i]. */
PS_API ps_status ps_dispersion(ps_ctx* ctx, const float* d_I, int P, int n_bins, int n_path, const double* kx,
                        const double* ky, int32_t* d_pix, float* d_out);
/* ps_qbin: radial histogram, bin = floor(sqrt(kx^2+ky^2)/dq), dropped (-1) if >= n_q;
 * d_qidx int32 [ny][nx] (bit-exact), d_out[b][q] = sum_p sum_{k in q} I[p][b][k]. */
PS_API ps_status ps_qbin(ps_ctx* ctx, const float* d_I, int P, int n_bins, double dq, int n_q, int32_t* d_qidx,
                  float* d_out);

/* Waits for the ctx stream, then reports (once) an error that a kernel of an earlier asynchronous call raised
 * (today: an atomic number without coefficients met by ps_build_slices / ps_multislice_fused after their one-time
 * synchronous validation) as PS_EUNSUPPORTED with a message; PS_OK if there is none.  Blocks the host. */
PS_API ps_status ps_check_async(ps_ctx* ctx);

/* Optional per-kernel timing.  While enabled, every launch group of the hot path is bracketed by a CUDA
 * event pair on the ctx stream.  ps_profile_read synchronises the stream, folds the pending pairs into
 * per-kernel totals and returns them: names[i] (static strings), ms[i] (summed device time) and
 * launches[i] for i < *n_kernels (arrays of at least 16 entries; any may be NULL); reset != 0 clears
 * the totals afterwards.  Kernel slots: k_bin, k_sort, k_vk, k_v_col, k_v_row, k_incident,
 * k_row_transmit, k_col_propagate, k_tacaw_fft, k_tacaw_accum, k_tacaw_finish, k_reduce, k_slice_resident. */
PS_API ps_status ps_profile_enable(ps_ctx* ctx, int on);
PS_API ps_status ps_profile_read(ps_ctx* ctx, int reset, int* n_kernels, const char** names, double* ms,
                                 long long* launches);

/* Number of kernels this ctx has launched so far (bench.py's `gpu_launches`). */
PS_API long long ps_launch_count(const ps_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* PYSLICE_B200_H */
