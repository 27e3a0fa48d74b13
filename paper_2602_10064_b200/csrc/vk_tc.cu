// vk_tc.cu — k_vk_tc: the V(k) structure-factor sums as tcgen05 TF32 GEMMs (design: vk_tc.cuh).
#include "common.cuh"
#include "vk_tc.cuh"
#include <type_traits>

namespace psb {

using namespace tc;

__device__ __forceinline__ float2 phase_cs_tc(const int m, const uint32_t U) {
    // (cos, sin) of 2 pi m u, u = U/2^32; same construction as phase_cs in potential.cu
    const int32_t ph = (int32_t)((uint32_t)m * U);
    const float r = (float)ph * 1.4629180792671596e-9f;             // 2 pi / 2^32
    return make_float2(__cosf(r), __sinf(r));
}

// grid = (tiles_m * tiles_n, n_slices, frames); block = 544 threads; dynamic smem = tc::SMEM_BYTES
__global__ void __launch_bounds__(THREADS, 1)
k_vk_tc(const uint32_t* __restrict__ sUx, const uint32_t* __restrict__ sUy, const int32_t* __restrict__ offsets,
        const float* __restrict__ ftab, const int32_t* __restrict__ nmax, float2* __restrict__ Vk, const int n_atoms,
        const int n_slices, const int n_elem, const int mcut, const int ncut, const int tiles_m, const int Tn) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* stages = smem_raw;                                            // NS x STAGE_BYTES
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)NS * STAGE_BYTES);   // [NS] producers -> MMA
    uint64_t* empty = full + NS;                                           // [NS] MMA done with a stage
    uint64_t* acc_full = empty + NS;                                       // accumulators of an element complete
    uint64_t* acc_free = acc_full + 1;                                     // epilogue has read them
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_free + 1);

    const int f = blockIdx.z, s = blockIdx.y;
    const int tmx = blockIdx.x % tiles_m, tny = blockIdx.x / tiles_m;
    const int m0 = tmx * TM, n0 = tny * Tn;
    const int mw = 2 * mcut + 1, nh = ncut + 1;
    const int n_bins = n_slices * n_elem;
    const int32_t* off = offsets + (size_t)f * (n_bins + 1) + (size_t)s * n_elem;
    if (off[n_elem] == off[0]) return;                                     // empty slice: Vk left unwritten
    if (m0 > mcut || n0 > ncut || nmax[m0] < n0) return;                   // tile wholly outside the aperture
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const size_t abase = (size_t)f * n_atoms;

    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) { mbar_init(&full[i], PROD_WARPS); mbar_init(&empty[i], 1); }   // one arrival per warp
        mbar_init(acc_full, 1);
        mbar_init(acc_free, PROD_WARPS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == PROD_WARPS) tmem_alloc(tmem_slot);
    fence_before_sync();
    __syncthreads();
    fence_after_sync();
    const uint32_t tmem = *tmem_slot;

    if (warp == PROD_WARPS) {
        // ------------------------------------------------------------ MMA issuer (one lane)
        const uint32_t idesc = instr_desc(2 * Tn);
        int c = 0, el = 0;
        for (int e = 0; e < n_elem; ++e) {
            const int jb = off[e], je = off[e + 1];
            if (jb == je) continue;
            if (el > 0) { mbar_wait(acc_free, (el - 1) & 1); fence_after_sync(); }
            for (int j0 = jb; j0 < je; j0 += KB, ++c) {
                const int st = c % NS;
                mbar_wait(&full[st], (c / NS) & 1);
                fence_after_sync();
                if (lane == 0) {
                    const uint32_t sa = smem_u32(stages + (size_t)st * STAGE_BYTES);
                    const uint32_t a_cxh = sa, a_cxl = sa + A_BYTES, a_sxh = sa + 2 * A_BYTES, a_sxl = sa + 3 * A_BYTES;
                    const uint32_t b_h = sa + 4 * A_BYTES, b_l = b_h + B_BYTES;
#pragma unroll
                    for (int ks = 0; ks < KB / 8; ++ks) {
                        const uint32_t ko = ks * 2 * LBO;                  // two 16-byte K chunks per instruction
                        const uint32_t acc = (j0 > jb || ks > 0) ? 1u : 0u;
                        mma_tf32(tmem, smem_desc(a_cxh + ko), smem_desc(b_h + ko), idesc, acc);
                        mma_tf32(tmem, smem_desc(a_cxh + ko), smem_desc(b_l + ko), idesc, 1u);
                        mma_tf32(tmem, smem_desc(a_cxl + ko), smem_desc(b_h + ko), idesc, 1u);
                        mma_tf32(tmem + D2_COL, smem_desc(a_sxh + ko), smem_desc(b_h + ko), idesc, acc);
                        mma_tf32(tmem + D2_COL, smem_desc(a_sxh + ko), smem_desc(b_l + ko), idesc, 1u);
                        mma_tf32(tmem + D2_COL, smem_desc(a_sxl + ko), smem_desc(b_h + ko), idesc, 1u);
                    }
                    mma_commit(&empty[st]);                                // stage reusable when these MMAs are done
                    if (j0 + KB >= je) mma_commit(acc_full);               // ... and the element's sums complete
                }
                __syncwarp();
            }
            ++el;
        }
    } else {
        // ------------------------------------------------------------ producers (warps 0-15), then epilogue
        const int r = threadIdx.x & 127;                                   // operand row = TMEM lane = m - m0
        const int part = threadIdx.x >> 7;                                 // which atoms of a stage (KG_PER groups of 4)
        const int m = m0 + r;
        float2* out = Vk + ((size_t)f * n_slices + s) * nh * mw;
        const uint32_t row_off = (uint32_t)((r >> 3) * SBO + (r & 7) * 16);
        const uint32_t brow_c = row_off;                                   // B row r       : cos(2 pi (n0 + r) u_y)
        const uint32_t brow_s = (uint32_t)(((r + Tn) >> 3) * SBO + ((r + Tn) & 7) * 16);   // B row Tn + r: sin
        // U of the first chunk (lanes 0..15: Ux of atom lane; 16..31: Uy), then always one chunk ahead
        auto load_u = [&](const int j0, const int je) -> uint32_t {
            return (j0 + (lane & 15) < je) ? (lane < 16 ? sUx : sUy)[abase + j0 + (lane & 15)] : 0u;
        };
        int c = 0, el = 0;
        for (int e = 0; e < n_elem; ++e) {
            const int jb = off[e], je = off[e + 1];
            if (jb == je) continue;
            uint32_t u_next = load_u(jb, je);
            for (int j0 = jb; j0 < je; j0 += KB, ++c) {
                const int st = c % NS, cnt = min(KB, je - j0);
                const uint32_t u = u_next;
                u_next = load_u(j0 + KB, je);
                if (c >= NS) mbar_wait(&empty[st], ((c / NS) - 1) & 1);
                uint8_t* sb = stages + (size_t)st * STAGE_BYTES;
                // phase factors of this thread's row for its atoms -> hi / lo operand tiles (K-major core matrices)
                auto generate = [&](auto tail_tag) {
                    constexpr bool TAIL = decltype(tail_tag)::value;       // last chunk of an element: atoms >= cnt are zero
#pragma unroll
                    for (int kgi = 0; kgi < KG_PER; ++kgi) {
                        const int kg = part * KG_PER + kgi;
                        float ch[4], cl[4], sh[4], sl[4], bch[4], bcl[4], bsh[4], bsl[4];
#pragma unroll
                        for (int kk = 0; kk < 4; ++kk) {
                            const int k = kg * 4 + kk;
                            const uint32_t ux = __shfl_sync(0xffffffffu, u, k), uy = __shfl_sync(0xffffffffu, u, 16 + k);
                            float2 px = phase_cs_tc(m, ux), py = phase_cs_tc(n0 + r, uy);
                            if (TAIL && k >= cnt) { px = make_float2(0.f, 0.f); py = make_float2(0.f, 0.f); }
                            split_tf32(px.x, ch[kk], cl[kk]); split_tf32(px.y, sh[kk], sl[kk]);
                            split_tf32(py.x, bch[kk], bcl[kk]); split_tf32(py.y, bsh[kk], bsl[kk]);
                        }
                        const uint32_t ko = kg * 128;
                        *reinterpret_cast<float4*>(sb + 0 * A_BYTES + row_off + ko) = make_float4(ch[0], ch[1], ch[2], ch[3]);
                        *reinterpret_cast<float4*>(sb + 1 * A_BYTES + row_off + ko) = make_float4(cl[0], cl[1], cl[2], cl[3]);
                        *reinterpret_cast<float4*>(sb + 2 * A_BYTES + row_off + ko) = make_float4(sh[0], sh[1], sh[2], sh[3]);
                        *reinterpret_cast<float4*>(sb + 3 * A_BYTES + row_off + ko) = make_float4(sl[0], sl[1], sl[2], sl[3]);
                        if (r < Tn) {
                            uint8_t* bh = sb + 4 * A_BYTES; uint8_t* bl = bh + B_BYTES;
                            *reinterpret_cast<float4*>(bh + brow_c + ko) = make_float4(bch[0], bch[1], bch[2], bch[3]);
                            *reinterpret_cast<float4*>(bl + brow_c + ko) = make_float4(bcl[0], bcl[1], bcl[2], bcl[3]);
                            *reinterpret_cast<float4*>(bh + brow_s + ko) = make_float4(bsh[0], bsh[1], bsh[2], bsh[3]);
                            *reinterpret_cast<float4*>(bl + brow_s + ko) = make_float4(bsl[0], bsl[1], bsl[2], bsl[3]);
                        }
                    }
                };
                if (cnt == KB) generate(std::false_type{}); else generate(std::true_type{});
                fence_proxy_async_smem();                                  // generic-proxy stores -> tensor-core reads
                __syncwarp();
                if (lane == 0) mbar_arrive(&full[st]);                     // one arrival per warp (512 would serialise)
            }
            // ---- epilogue of this element: TMEM lane r = row m; columns n (cc), Tn + n (cs); D2: sc, ss
            mbar_wait(acc_full, el & 1);
            fence_after_sync();
            const uint32_t tl = tmem + ((uint32_t)((warp & 3) * 32) << 16);
            const int q_step = ((Tn + PARTS - 1) / PARTS + 7) & ~7;         // columns split between the row's threads
            const int q_lo = min(part * q_step, Tn), q_hi = min(q_lo + q_step, Tn);
            const float* ft = ftab + (size_t)e * nh * mw;
            const int nm = (m <= mcut) ? nmax[m] : -1;
            for (int q = q_lo; q < q_hi; q += 8) {
                float cc[8], cs[8], sc[8], ss[8];
                tmem_ld8(tl + q, cc);
                tmem_ld8(tl + Tn + q, cs);
                tmem_ld8(tl + D2_COL + q, sc);
                tmem_ld8(tl + D2_COL + Tn + q, ss);
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int n = n0 + q + i;
                    if (n <= ncut && n <= nm) {                            // inside the aperture (the rest is never read)
                        float2* op = out + (size_t)n * mw + (mcut + m);
                        float2* om = out + (size_t)n * mw + (mcut - m);
                        const float fv = __ldg(ft + (size_t)n * mw + (mcut + m));
                        float2 vp = make_float2(fv * (cc[i] - ss[i]), -fv * (cs[i] + sc[i]));
                        float2 vm = make_float2(fv * (cc[i] + ss[i]), fv * (sc[i] - cs[i]));
                        if (el > 0) {
                            const float2 p0 = *op, q0 = *om;
                            vp.x += p0.x; vp.y += p0.y; vm.x += q0.x; vm.y += q0.y;
                        }
                        *op = vp;
                        if (m > 0) *om = vm;
                    }
                }
            }
            fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive(acc_free);
            ++el;
        }
    }
    fence_before_sync();
    __syncthreads();
    if (warp == PROD_WARPS) tmem_dealloc(tmem);
}

// host launcher (called from ps_build_slices): tiles of 128 m-values x Tn n-values over the quarter plane
cudaError_t launch_vk_tc(ps_ctx* c, const uint32_t* sUx, const uint32_t* sUy, const int32_t* off, float2* Vk, int n_atoms,
                         int nf) {
    int cap_unused = 0;                                                    // sets the shared-memory attribute once per ctx
    cudaError_t ce = kernel_cap(c, k_vk_tc, THREADS, SMEM_BYTES, &cap_unused);
    if (ce != cudaSuccess) return ce;
    const int tiles_m = (c->mcut + 1 + TM - 1) / TM;
    const int tiles_n = (c->ncut + 1 + TN_MAX - 1) / TN_MAX;
    int Tn = ((c->ncut + 1 + tiles_n - 1) / tiles_n + 7) & ~7;            // equal-width n tiles, multiple of 8
    if (Tn < 8) Tn = 8;
    k_vk_tc<<<dim3(tiles_m * tiles_n, c->n_slices, nf), THREADS, SMEM_BYTES, c->stream>>>(
        sUx, sUy, off, c->d_ftab, c->d_nmax, Vk, n_atoms, c->n_slices, c->n_elem, c->mcut, c->ncut, tiles_m, Tn);
    return cudaGetLastError();
}

}  // namespace psb
