// vk_tc.cuh — V(k) assembly (the structure-factor sum) on the 5th-generation tensor cores.
//
// The separable sum  S(m, n) = sum_j exp(-2 pi i m u_xj) exp(-2 pi i n u_yj)  over the atoms of one (slice, element)
// is a dense contraction over atoms.  With cx, sx = cos, sin(2 pi m u_x) and cy, sy likewise in n, the four real
// sums  cc = cx.cy, cs = cx.sy, sc = sx.cy, ss = sx.sy  are two real GEMMs with the atoms as the K dimension:
//     D1[m][0:Tn | Tn:2Tn] = cx[m][j] * [cy | sy][n][j]^T          D2[m][...] = sx[m][j] * [cy | sy][n][j]^T
// issued as tcgen05.mma kind::tf32 (M = 128 m-values = the 128 TMEM lanes, N = 2 Tn <= 256, K = 8 atoms per
// instruction), accumulators D1, D2 in TMEM.  FP32 accuracy comes from the 3xTF32 split: every operand x is stored
// as hi = tf32(x) (rounded to nearest) and lo = x - hi and each product is issued as hi*hi + hi*lo + lo*hi (the dropped
// lo*lo term is 2^-22 relative).  Then, as in the SIMT kernel (potential.cu),
//     V(+m, n) = f (cc - ss, -(cs + sc)),     V(-m, n) = f (cc + ss, sc - cs).
//
// One CTA = one (frame, slice, 128 x Tn tile of the quarter plane).  Warps 0-15 turn atoms into operand tiles in
// shared memory (canonical K-major, no-swizzle UMMA layout: 8-row x 16-byte core matrices), ring of NS stages;
// warp 16 owns TMEM (512 columns) and issues the MMAs from one lane; tcgen05.commit on mbarriers frees stages and
// hands the accumulators to warps 0-15, which read them back with tcgen05.ld (warp w <-> TMEM lanes 32 (w % 4) ...) and
// write V(k).  No TMA: the operands do not exist in global memory, they are generated on the fly.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace psb {
namespace tc {

constexpr int TM = 128;                 // m values per tile = TMEM lanes = MMA M
constexpr int KB = 16;                  // atoms per shared-memory stage (two K = 8 instructions)
constexpr int NS = 3;                   // stages
constexpr int TN_MAX = 128;             // n values per tile at most (MMA N = 2 Tn <= 256)
constexpr int PROD_WARPS = 16;          // producer / epilogue warps: warps w, w + 4, ... share rows, split the atoms
constexpr int PARTS = PROD_WARPS / 4;   // producer threads per operand row
constexpr int KG_PER = (KB / 4) / PARTS; // 4-atom groups per producer thread and stage
constexpr int THREADS = 32 * (PROD_WARPS + 1);   // + 1 MMA warp
constexpr int A_BYTES = TM * KB * 4;                    // one A operand array of a stage (8 KB)
constexpr int B_BYTES = 2 * TN_MAX * KB * 4;            // one B operand array of a stage (16 KB)
constexpr int STAGE_BYTES = 4 * A_BYTES + 2 * B_BYTES;  // cx_hi cx_lo sx_hi sx_lo | b_hi b_lo  (64 KB)
constexpr int SBO = (KB / 4) * 128;                     // byte stride between 8-row groups
constexpr int LBO = 128;                                // byte stride between the two 16-byte K chunks of an instruction
constexpr int TMEM_COLS = 512;
constexpr int D2_COL = 256;                             // D1 at columns [0, 2Tn), D2 at [256, 256 + 2Tn)
constexpr size_t SMEM_BYTES = (size_t)NS * STAGE_BYTES + 256 + 1024;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- mbarrier
__device__ __forceinline__ void mbar_init(uint64_t* bar, const uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, const uint32_t parity) {
    const uint32_t a = smem_u32(bar);
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(a), "r"(parity) : "memory");
}

// ---- tcgen05
__device__ __forceinline__ void tmem_alloc(uint32_t* slot_in_smem) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot_in_smem)), "r"((uint32_t)TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(const uint32_t base) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"((uint32_t)TMEM_COLS) : "memory");
}
__device__ __forceinline__ void fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// arrives on the mbarrier when every MMA issued so far by this thread has completed
__device__ __forceinline__ void mma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, kind::tf32, M = 128, N from idesc, K = 8
__device__ __forceinline__ void mma_tf32(const uint32_t d_tmem, const uint64_t adesc, const uint64_t bdesc,
                                         const uint32_t idesc, const uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// shared-memory matrix descriptor: K-major, SWIZZLE_NONE, version 1 (sm_100)
__device__ __forceinline__ uint64_t smem_desc(const uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFF) >> 4) | ((uint64_t)(LBO >> 4) << 16) | ((uint64_t)(SBO >> 4) << 32) | (1ull << 46);
}
// instruction descriptor: D = F32, A = B = TF32, both K-major, M = 128, N = n
__host__ __device__ __forceinline__ uint32_t instr_desc(const int n) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);
}
// 8 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld8(const uint32_t taddr, float (&v)[8]) {
    uint32_t r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr));
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// x = hi + lo with hi representable in TF32 (10 mantissa bits, rounded to nearest by an integer add on the bit
// pattern: cvt.rna.tf32.f32 is emulated with ~8 integer instructions on sm_100a) and lo = x - hi exact in FP32;
// the tensor core reads the top 19 bits of lo, i.e. drops at most 2^-10 |lo| <= 2^-21 |x|.
__device__ __forceinline__ void split_tf32(const float x, float& hi, float& lo) {
    hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
    lo = x - hi;
}

}  // namespace tc
}  // namespace psb
