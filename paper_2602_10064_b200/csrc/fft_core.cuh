// fft_core.cuh — in-register / shared-memory radix FFT building blocks for sm_100a.
//
// One transform of length N (a power of two, 32 <= N <= 4096) is carried by T = N/16 threads,
// each holding 16 complex values in registers in the "canonical" layout
//      v[e] = x[t + e*T],   t = thread index inside the transform, e = 0..15.
// The transform is a mixed-radix Stockham autosort FFT with at most three stages
//      N = 16 * R2 * R3,   R2 = min(16, N/16),  R3 = N/(16*R2)
// (stage s reads x[j + r*N/R], multiplies by W_{Ns*R}^{(j mod Ns) r}, does an R-point DFT and
// writes y[(j/Ns)*Ns*R + (j mod Ns) + r*Ns]).  Both the input of the first stage and the output
// of the last stage are canonical, so a pointwise product between two transforms (transmission
// function, propagator) needs no data movement, and only the (#stages-1) exchanges between
// stages go through shared memory.  Stage twiddles depend only on t, so each thread computes
// them once (sincospif on exactly reduced integer phases) and keeps them in registers while it
// loops over rows / columns / batches.
//
// Only the forward transform exp(-2 pi i nk/N) is coded; the inverse (unnormalised) is obtained
// by swapping real and imaginary parts on the way in and out (free register renaming).
//
// Implements the transforms of PAPER.md:79 (fft2/ifft2 of the slice loop), PAPER.md:81 (inverse
// FFT of V(k)) and PAPER.md:73 (time-axis transform); numpy sign convention (A1).
#pragma once
#include <cuda_runtime.h>

namespace psb {

__device__ __forceinline__ float2 cmul(const float2 a, const float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cswap(const float2 a) { return make_float2(a.y, a.x); }

// exp(i x) for |x| up to a few thousand radians: two-constant Cody-Waite reduction to [-pi, pi]
// (exact for the quotients that occur), then the SFU sine / cosine (abs. error 2^-21.4 there).
// Error budget: DESIGN.md section 7.
__device__ __forceinline__ float2 cis_fast(const float x) {
    const float k = rintf(x * 0.15915494309189535f);
    float r = fmaf(-k, 6.28125f, x);                       // 2 pi = 6.28125 + 1.9353071795864769e-3
    r = fmaf(-k, 1.9353071795864769e-3f, r);
    return make_float2(__cosf(r), __sinf(r));
}

// ---------------------------------------------------------------- small DFTs (forward, natural order)
__device__ __forceinline__ void dft2(float2& a, float2& b) {
    const float2 t = a;
    a = make_float2(t.x + b.x, t.y + b.y);
    b = make_float2(t.x - b.x, t.y - b.y);
}
// X0=a+b+c+d, X1=a-ib-c+id, X2=a-b+c-d, X3=a+ib-c-id   (W4 = -i)
__device__ __forceinline__ void dft4(float2& a, float2& b, float2& c, float2& d) {
    const float2 s0 = make_float2(a.x + c.x, a.y + c.y);
    const float2 s1 = make_float2(a.x - c.x, a.y - c.y);
    const float2 s2 = make_float2(b.x + d.x, b.y + d.y);
    const float2 s3 = make_float2(b.x - d.x, b.y - d.y);
    a = make_float2(s0.x + s2.x, s0.y + s2.y);
    c = make_float2(s0.x - s2.x, s0.y - s2.y);
    b = make_float2(s1.x + s3.y, s1.y - s3.x);
    d = make_float2(s1.x - s3.y, s1.y + s3.x);
}

template <int R> struct Dft;
template <> struct Dft<2> {
    static __device__ __forceinline__ void run(float2 (&w)[2]) { dft2(w[0], w[1]); }
};
template <> struct Dft<4> {
    static __device__ __forceinline__ void run(float2 (&w)[4]) { dft4(w[0], w[1], w[2], w[3]); }
};
template <> struct Dft<8> {
    // n = 2 n1 + n2, k = k1 + 4 k2
    static __device__ __forceinline__ void run(float2 (&w)[8]) {
        constexpr float h = 0.70710678118654752440f;
        dft4(w[0], w[2], w[4], w[6]);
        dft4(w[1], w[3], w[5], w[7]);
        // y[1][k1] *= W8^k1
        w[3] = make_float2((w[3].x + w[3].y) * h, (w[3].y - w[3].x) * h);       // (1-i)/sqrt2
        w[5] = make_float2(w[5].y, -w[5].x);                                    // -i
        w[7] = make_float2((w[7].y - w[7].x) * h, -(w[7].x + w[7].y) * h);      // (-1-i)/sqrt2
        dft2(w[0], w[1]); dft2(w[2], w[3]); dft2(w[4], w[5]); dft2(w[6], w[7]);
        // now w = {X0,X4,X1,X5,X2,X6,X3,X7}
        const float2 x4 = w[1], x1 = w[2], x5 = w[3], x2 = w[4], x6 = w[5], x3 = w[6];
        w[1] = x1; w[2] = x2; w[3] = x3; w[4] = x4; w[5] = x5; w[6] = x6;
    }
};
template <> struct Dft<16> {
    // n = 4 n1 + n2, k = k1 + 4 k2
    static __device__ __forceinline__ void run(float2 (&w)[16]) {
        constexpr float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;
        constexpr float h = 0.70710678118654752440f;
        dft4(w[0], w[4], w[8], w[12]);      // y[0][k1] at w[4 k1 + 0]
        dft4(w[1], w[5], w[9], w[13]);
        dft4(w[2], w[6], w[10], w[14]);
        dft4(w[3], w[7], w[11], w[15]);
        // w[4 k1 + n2] *= W16^(n2 k1)
        w[5] = cmul(w[5], make_float2(c1, -s1));                                    // W^1
        w[6] = make_float2((w[6].x + w[6].y) * h, (w[6].y - w[6].x) * h);           // W^2
        w[7] = cmul(w[7], make_float2(s1, -c1));                                    // W^3
        w[9] = make_float2((w[9].x + w[9].y) * h, (w[9].y - w[9].x) * h);           // W^2
        w[10] = make_float2(w[10].y, -w[10].x);                                     // W^4 = -i
        w[11] = make_float2((w[11].y - w[11].x) * h, -(w[11].x + w[11].y) * h);     // W^6
        w[13] = cmul(w[13], make_float2(s1, -c1));                                  // W^3
        w[14] = make_float2((w[14].y - w[14].x) * h, -(w[14].x + w[14].y) * h);     // W^6
        w[15] = cmul(w[15], make_float2(-c1, s1));                                  // W^9
        dft4(w[0], w[1], w[2], w[3]);       // X[k1 + 4 k2] at w[4 k1 + k2]
        dft4(w[4], w[5], w[6], w[7]);
        dft4(w[8], w[9], w[10], w[11]);
        dft4(w[12], w[13], w[14], w[15]);
        // transpose 4x4 to natural order
        float2 t;
        t = w[1]; w[1] = w[4]; w[4] = t;
        t = w[2]; w[2] = w[8]; w[8] = t;
        t = w[3]; w[3] = w[12]; w[12] = t;
        t = w[6]; w[6] = w[9]; w[9] = t;
        t = w[7]; w[7] = w[13]; w[13] = t;
        t = w[11]; w[11] = w[14]; w[14] = t;
    }
};

template <> struct Dft<32> {
    // decimation in time over two 16-point transforms: X[k] = E[k] + W32^k O[k], X[k + 16] = E[k] - W32^k O[k]
    static __device__ __forceinline__ void run(float2 (&w)[32]) {
        float2 a[16], b[16];
#pragma unroll
        for (int s = 0; s < 16; ++s) { a[s] = w[2 * s]; b[s] = w[2 * s + 1]; }
        Dft<16>::run(a);
        Dft<16>::run(b);
        constexpr float h = 0.70710678118654752440f;
        constexpr float c[16] = {1.f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                                 0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                                 0.19509032201612826785f, 0.f, -0.19509032201612826785f, -0.38268343236508977173f,
                                 -0.55557023301960222474f, -0.70710678118654752440f, -0.83146961230254523708f,
                                 -0.92387953251128675613f, -0.98078528040323044913f};
        constexpr float sn[16] = {0.f, 0.19509032201612826785f, 0.38268343236508977173f, 0.55557023301960222474f,
                                  0.70710678118654752440f, 0.83146961230254523708f, 0.92387953251128675613f,
                                  0.98078528040323044913f, 1.f, 0.98078528040323044913f, 0.92387953251128675613f,
                                  0.83146961230254523708f, 0.70710678118654752440f, 0.55557023301960222474f,
                                  0.38268343236508977173f, 0.19509032201612826785f};
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            float2 o;
            if (k == 0) o = b[0];
            else if (k == 4) o = make_float2((b[4].x + b[4].y) * h, (b[4].y - b[4].x) * h);            // (1 - i)/sqrt2
            else if (k == 8) o = make_float2(b[8].y, -b[8].x);                                         // -i
            else if (k == 12) o = make_float2((b[12].y - b[12].x) * h, -(b[12].x + b[12].y) * h);      // (-1 - i)/sqrt2
            else o = cmul(b[k], make_float2(c[k], -sn[k]));                                             // W32^k
            w[k] = make_float2(a[k].x + o.x, a[k].y + o.y);
            w[k + 16] = make_float2(a[k].x - o.x, a[k].y - o.y);
        }
    }
};

// ---------------------------------------------------------------- plan
template <int N> struct Plan {
    static_assert(N >= 32 && N <= 4096 && (N & (N - 1)) == 0, "N must be a power of two in [32, 4096]");
    static constexpr int T = N / 16;                          // threads per transform
    static constexpr int R2 = (N / 16 >= 16) ? 16 : N / 16;   // second-stage radix
    static constexpr int R3 = N / (16 * R2);                  // third-stage radix (1 = none)
    static constexpr int B2 = 16 / R2;                        // butterflies per thread, stage 2
    static constexpr int B3 = (R3 > 1) ? 16 / R3 : 1;
    static constexpr int NTW2 = B2 * (R2 - 1);
};

// exp(-2 pi i num/den), num reduced mod den exactly in integers first
__device__ __forceinline__ float2 root_of_unity(int num, int den) {
    num &= (den - 1);                                          // den is a power of two
    float s, c;
    sincospif(2.0f * (float)num / (float)den, &s, &c);         // num/den exact in fp32 (den <= 4096)
    return make_float2(c, -s);
}

template <int N> struct Twiddles {
    using P = Plan<N>;
    float2 w2[P::NTW2];                 // stage 2: W_{16 R2}^{(j mod 16) r}, r = 1..R2-1, per butterfly
    float2 w3[P::B3];                   // stage 3: base W_N^{(j mod 16 R2)} per butterfly
    __device__ __forceinline__ void init(const int t) {
#pragma unroll
        for (int b = 0; b < P::B2; ++b) {
            const int q = (t + b * P::T) & 15;
#pragma unroll
            for (int r = 1; r < P::R2; ++r) w2[b * (P::R2 - 1) + r - 1] = root_of_unity(q * r, 16 * P::R2);
        }
        if (P::R3 > 1) {
#pragma unroll
            for (int b = 0; b < P::B3; ++b) {
                const int q = (t + b * P::T) & (16 * P::R2 - 1);
                w3[b] = root_of_unity(q, N);
            }
        } else {
            w3[0] = make_float2(1.f, 0.f);
        }
    }
    __device__ __forceinline__ float2 tw2(const int b, const int r) const { return w2[b * (P::R2 - 1) + r - 1]; }
    __device__ __forceinline__ float2 tw3(const int b) const { return w3[b]; }
};

// Register-light variant: the stage-2 twiddles W_{16 R2}^{q r} depend on the thread only through q = j mod 16, so a block
// keeps one table [16][R2 - 1] in shared memory (filled once per kernel) and every thread re-reads its R2 - 1 values per
// transform (one broadcast-friendly LDS.64 each) instead of holding 2 (R2 - 1) registers across the persistent loop.
template <int N> struct TwiddlesShared {
    using P = Plan<N>;
    static constexpr int TABLE = 16 * (P::R2 - 1);       // float2 entries
    // stage 3: W_N^{t + b T}; when T B3/2 = N/4 (N = 512) the upper half of the b range is the lower half times -i
    static constexpr bool HALF3 = (P::R3 > 1) && (P::T * P::B3 / 2 * 4 == N);
    static constexpr int NW3 = HALF3 ? P::B3 / 2 : P::B3;
    const float2* row[P::B2];                            // table row of (t + b T) mod 16
    float2 w3[NW3];
    // every thread of the block calls fill() (followed by a block barrier) before the first transform
    static __device__ __forceinline__ void fill(float2* tab, const int tid, const int nthreads) {
        for (int i = tid; i < TABLE; i += nthreads) {
            const int q = i / (P::R2 - 1), r = i % (P::R2 - 1) + 1;
            tab[i] = root_of_unity(q * r, 16 * P::R2);
        }
    }
    __device__ __forceinline__ void init(const int t, const float2* tab) {
#pragma unroll
        for (int b = 0; b < P::B2; ++b) row[b] = tab + ((t + b * P::T) & 15) * (P::R2 - 1);
        if (P::R3 > 1) {
#pragma unroll
            for (int b = 0; b < NW3; ++b) w3[b] = root_of_unity((t + b * P::T) & (16 * P::R2 - 1), N);
        } else {
            w3[0] = make_float2(1.f, 0.f);
        }
    }
    __device__ __forceinline__ float2 tw2(const int b, const int r) const { return row[b][r - 1]; }
    __device__ __forceinline__ float2 tw3(const int b) const {
        if constexpr (HALF3) {
            if (b >= NW3) return make_float2(w3[b - NW3].y, -w3[b - NW3].x);     // times W_4 = -i
        }
        return w3[b < NW3 ? b : 0];
    }
};

// ---------------------------------------------------------------- exchange policies
// A policy gives the shared-memory slot of logical element idx of *this thread's* transform and
// the barrier covering all threads of that transform.
// `at` is the layout the caller sees (first read, last write, second exchange); x1w / x1r address the FIRST exchange
// (element 16 t + r written, element t + e T read), whose layout may differ as long as write and read agree.
// x2w / x2r address the SECOND exchange (element j0 + 16 r written by butterfly b, element t + e T read).
struct RowSlots {            // one transform per contiguous padded line; pad 1 per 16 (conflict-free)
    float2* line;
    __device__ __forceinline__ float2& at(const int idx) const { return line[idx + (idx >> 4)]; }
    __device__ __forceinline__ float2& x1w(const int t, const int r) const { return at(16 * t + r); }
    template <int T> __device__ __forceinline__ float2& x1r(const int t, const int e) const { return at(t + e * T); }
    template <int N> __device__ __forceinline__ float2& x2w(const int t, const int b, const int r) const {
        const int j = t + b * Plan<N>::T;
        return at((j >> 4) * (16 * Plan<N>::R2) + (j & 15) + 16 * r);
    }
    template <int T> __device__ __forceinline__ float2& x2r(const int t, const int e) const { return at(t + e * T); }
};
// The same padded line with every access written as (per-thread base pointer) + (compile-time offset): for
// T = N/16 a multiple of 16 the pad term of t + e T and of the second-exchange index separates into a part that depends
// on the thread only and a part that depends on the unrolled loop index only.  (With at() the compiler rebuilt
// idx + (idx >> 4) per element and per item: ncu showed ~130 of the 1650 warp instructions of a 512-point row pass
// spent there.)  Three base registers per thread, zero address arithmetic per access.
template <int N> struct RowSlotsF {
    static constexpr int T = Plan<N>::T, R2 = Plan<N>::R2;
    static_assert(T % 16 == 0, "RowSlotsF needs N >= 256");
    float2 *w1, *rd, *w2;
    __device__ __forceinline__ RowSlotsF(float2* line, const int t)
        : w1(line + 17 * t), rd(line + t + (t >> 4)), w2(line + (t >> 4) * (17 * R2) + (t & 15)) {}
    __device__ __forceinline__ float2& x1w(const int, const int r) const { return w1[r]; }                  // 16 t + r, r < 16
    template <int T_> __device__ __forceinline__ float2& x1r(const int, const int e) const { return rd[e * T + e * T / 16]; }
    template <int N_> __device__ __forceinline__ float2& x2w(const int, const int b, const int r) const {
        return w2[b * (T / 16) * (17 * R2) + 17 * r];
    }
    template <int T_> __device__ __forceinline__ float2& x2r(const int, const int e) const { return rd[e * T + e * T / 16]; }
};
// C transforms interleaved (a warp = 32/C consecutive t x C columns), linear so that a TMA box [rows][C] can land in it.
// First exchange: the writes 16 t + r of the 32/C t-values of a warp would all fall on the same C*8-byte slice of the
// 128-byte bank window (a 16/C-way conflict for C < 16).  XOR-ing the row index with (row >> 4) & M, M = 16/C - 1,
// spreads them over the whole window (2 wavefronts per 256-byte warp access, the minimum).  The XOR term is a per-thread
// constant (t & M for the writes, (t >> 4) & M for the reads when T is a multiple of 16 (M + 1)), so it is folded into
// M + 2 base pointers computed once per item and every access keeps an immediate offset.
template <int C> struct ColSlots {
    static constexpr int M = (C < 16) ? 16 / C - 1 : 0;
    float2* base;                    // already offset by the column index c
    float2* wb[M + 1];
    float2* rb;
    __device__ __forceinline__ ColSlots(float2* b, const int t) : base(b) {
        const int sw = t & M;
#pragma unroll
        for (int k = 0; k <= M; ++k) wb[k] = b + (16 * t + ((k ^ sw) - k)) * C;
        rb = b + (t ^ ((t >> 4) & M)) * C;
    }
    __device__ __forceinline__ float2& at(const int idx) const { return base[idx * C]; }
    template <int N> __device__ __forceinline__ float2& x2w(const int t, const int b, const int r) const {
        const int j = t + b * Plan<N>::T;
        return at((j >> 4) * (16 * Plan<N>::R2) + (j & 15) + 16 * r);
    }
    template <int T> __device__ __forceinline__ float2& x2r(const int t, const int e) const { return at(t + e * T); }
    __device__ __forceinline__ float2& x1w(const int, const int r) const { return wb[r & M][r * C]; }
    template <int T> __device__ __forceinline__ float2& x1r(const int t, const int e) const {
        if constexpr (T % (16 * (M + 1)) == 0) {
            return rb[e * T * C];
        } else {
            const int idx = t + e * T;
            return base[(idx ^ ((idx >> 4) & M)) * C];
        }
    }
};
struct BlockSync { static __device__ __forceinline__ void sync() { __syncthreads(); } };
struct WarpSync  { static __device__ __forceinline__ void sync() { __syncwarp(); } };
// the T threads (whole warps) that carry one transform of a block holding several: named barrier 1 + threadIdx.x / T
template <int T> struct GroupSync {
    static_assert(T % 32 == 0, "a transform must be carried by whole warps");
    static __device__ __forceinline__ void sync() {
        asm volatile("bar.sync %0, %1;" ::"r"(1 + (int)threadIdx.x / T), "r"(T) : "memory");
    }
};

template <int N> struct RowLine { static constexpr int LEN = N + N / 16; };      // padded line length (float2)

// ---------------------------------------------------------------- the transform
template <int N, class Slots, class Sync, class TW = Twiddles<N>>
__device__ __forceinline__ void fft_forward(float2 (&v)[16], const int t, const TW& tw, const Slots& sm) {
    using P = Plan<N>;
    constexpr int T = P::T;
    // stage 1: radix 16, Ns = 1, no twiddle
    Dft<16>::run(v);
    Sync::sync();                                             // earlier readers of the buffer are done
#pragma unroll
    for (int r = 0; r < 16; ++r) sm.x1w(t, r) = v[r];
    Sync::sync();
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = sm.template x1r<T>(t, e);
    // stage 2: radix R2, Ns = 16
    constexpr int R2 = P::R2, B2 = P::B2;
#pragma unroll
    for (int b = 0; b < B2; ++b) {
        float2 w[R2];
#pragma unroll
        for (int r = 0; r < R2; ++r) w[r] = v[b + r * B2];
#pragma unroll
        for (int r = 1; r < R2; ++r) w[r] = cmul(w[r], tw.tw2(b, r));
        Dft<R2>::run(w);
#pragma unroll
        for (int r = 0; r < R2; ++r) v[b + r * B2] = w[r];
    }
    if constexpr (P::R3 > 1) {
        constexpr int R3 = P::R3, B3 = P::B3;
        Sync::sync();
#pragma unroll
        for (int b = 0; b < B2; ++b) {
#pragma unroll
            for (int r = 0; r < R2; ++r) sm.template x2w<N>(t, b, r) = v[b + r * B2];
        }
        Sync::sync();
#pragma unroll
        for (int e = 0; e < 16; ++e) v[e] = sm.template x2r<T>(t, e);
        // stage 3: radix R3, Ns = 16 R2, twiddle base^r
#pragma unroll
        for (int b = 0; b < B3; ++b) {
            float2 w[R3];
#pragma unroll
            for (int r = 0; r < R3; ++r) w[r] = v[b + r * B3];
            float2 p[R3];                                     // p[r] = base^r (balanced products)
            p[1] = tw.tw3(b);
#pragma unroll
            for (int r = 2; r < R3; ++r) p[r] = cmul(p[r / 2], p[r - r / 2]);
#pragma unroll
            for (int r = 1; r < R3; ++r) w[r] = cmul(w[r], p[r]);
            Dft<R3>::run(w);
#pragma unroll
            for (int r = 0; r < R3; ++r) v[b + r * B3] = w[r];
        }
    }
}

// unnormalised inverse: swap, forward, swap
template <int N, class Slots, class Sync, class TW = Twiddles<N>>
__device__ __forceinline__ void fft_inverse(float2 (&v)[16], const int t, const TW& tw, const Slots& sm) {
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = cswap(v[e]);
    fft_forward<N, Slots, Sync, TW>(v, t, tw, sm);
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = cswap(v[e]);
}

// ================================================================ 32 values per thread (N = 512, 1024)
// The same Stockham scheme with E = 32 values per thread: T = N/32 threads per transform, canonical layout
// v[e] = x[t + e T], first stage radix 32, second stage radix R2 = N/32 (16 or 32) and ONE shared-memory exchange
// instead of the two the 16-value plan needs at these lengths.  The column-type kernels move every element through
// shared memory 6 instead of 10 times per transform pair, which is what bounds them (ncu: LSU data pipe 64 % busy at
// 57 % issue utilisation with the 16-value plan).  Costs registers: 64 for the data and 2 (R2 - 1) B2 for the twiddles.
template <int N> struct Plan32 {
    static_assert(N == 512 || N == 1024, "the 32-value plan covers N = 512 and 1024");
    static constexpr int T = N / 32;
    static constexpr int R2 = N / 32;                         // 16 or 32
    static constexpr int B2 = 32 / R2;                        // butterflies per thread in stage 2
    static constexpr int NTW2 = B2 * (R2 - 1);
};

template <int N> struct Twiddles32 {
    using P = Plan32<N>;
    float2 w2[P::NTW2];                                      // W_N^{((t + b T) mod 32) r}, r = 1..R2-1
    __device__ __forceinline__ void init(const int t) {
#pragma unroll
        for (int b = 0; b < P::B2; ++b) {
            const int q = (t + b * P::T) & 31;
#pragma unroll
            for (int r = 1; r < P::R2; ++r) w2[b * (P::R2 - 1) + r - 1] = root_of_unity(q * r, N);
        }
    }
    __device__ __forceinline__ float2 tw2(const int b, const int r) const { return w2[b * (P::R2 - 1) + r - 1]; }
};

// C transforms interleaved as in ColSlots (a warp = 32/C consecutive t x C columns, linear [row][C] so that a TMA box
// lands in it).  The exchange writes rows 32 t + r and reads rows t + e T; XOR-ing the row with (row >> 5) & M,
// M = 16/C - 1, spreads the 32/C writes of a warp over the whole 128-byte bank window.  Both XOR terms are constants of
// the thread (t & M) or of the unrolled index ((e T / 32) & M), folded into M + 1 base pointers on each side.
template <int C, int T> struct ColSlots32 {
    static constexpr int M = (C < 16) ? 16 / C - 1 : 0;
    static_assert(T == 16 || T == 32, "ColSlots32: N = 512 or 1024");
    float2* base;
    float2* wb[M + 1];
    float2* rb[M + 1];
    __device__ __forceinline__ ColSlots32(float2* b, const int t) : base(b) {
        const int sw = t & M;
#pragma unroll
        for (int k = 0; k <= M; ++k) {
            wb[k] = b + (32 * t + ((k ^ sw) - k)) * C;
            rb[k] = b + (t ^ k) * C;
        }
    }
    __device__ __forceinline__ float2& at(const int idx) const { return base[idx * C]; }
    __device__ __forceinline__ float2& x1w(const int r) const { return wb[r & M][r * C]; }
    __device__ __forceinline__ float2& x1r(const int e) const { return rb[((e * T) >> 5) & M][e * T * C]; }
};

// One transform per contiguous line padded by one element per 32 (the 32 t + r writes of consecutive t land 33 elements
// apart: conflict-free); every access is a per-thread base pointer plus a compile-time offset.
template <int N> struct RowLine32 { static constexpr int LEN = N + N / 32; };
template <int N> struct RowSlots32 {
    static constexpr int T = Plan32<N>::T;
    float2 *w1, *rd;
    __device__ __forceinline__ RowSlots32(float2* line, const int t) : w1(line + 33 * t), rd(line + t) {}
    __device__ __forceinline__ float2& x1w(const int r) const { return w1[r]; }
    __device__ __forceinline__ float2& x1r(const int e) const { return rd[e * T + ((e * T) >> 5)]; }
};

template <int N, class Slots, class Sync>
__device__ __forceinline__ void fft32_forward(float2 (&v)[32], const Twiddles32<N>& tw, const Slots& sm) {
    using P = Plan32<N>;
    Dft<32>::run(v);                                          // stage 1: radix 32, Ns = 1
    Sync::sync();                                             // earlier readers of the buffer are done
#pragma unroll
    for (int r = 0; r < 32; ++r) sm.x1w(r) = v[r];
    Sync::sync();
#pragma unroll
    for (int e = 0; e < 32; ++e) v[e] = sm.x1r(e);
    constexpr int R2 = P::R2, B2 = P::B2;                     // stage 2: radix R2, Ns = 32 (last stage: output canonical)
#pragma unroll
    for (int b = 0; b < B2; ++b) {
        float2 w[R2];
#pragma unroll
        for (int r = 0; r < R2; ++r) w[r] = v[b + r * B2];
#pragma unroll
        for (int r = 1; r < R2; ++r) w[r] = cmul(w[r], tw.tw2(b, r));
        Dft<R2>::run(w);
#pragma unroll
        for (int r = 0; r < R2; ++r) v[b + r * B2] = w[r];
    }
}

template <int N, class Slots, class Sync>
__device__ __forceinline__ void fft32_inverse(float2 (&v)[32], const Twiddles32<N>& tw, const Slots& sm) {
#pragma unroll
    for (int e = 0; e < 32; ++e) v[e] = cswap(v[e]);
    fft32_forward<N, Slots, Sync>(v, tw, sm);
#pragma unroll
    for (int e = 0; e < 32; ++e) v[e] = cswap(v[e]);
}

}  // namespace psb
