// fft_aos.cuh -- register-resident Stockham FFT with ONE complex number per packed f32x2 register pair (re, im).
//
// The sm_100 packed instructions accept lane-swapped, per-lane-negated operands (SASS `.F32x2.LO_HI.NP`) and scalar
// broadcasts (`.F32`), so with the natural (re, im) layout
//   complex add / sub      = 1 FADD2
//   times +-i              = an operand swizzle of the consumer (no instruction; ~1 extra cycle in a consuming FADD2)
//   complex * complex      = FMUL2 + FFMA2:   x*w = x*(c, c) + (i*x)*(s, s)
// i.e. half the issue slots of scalar FADD/FMUL/FFMA at the same FP32 lane throughput (profiles/r1b_fp32_issue.md),
// with 2 registers per element: 16 elements per thread leave room for 1024 threads (four independent groups) per SM.
//
// Indexing: element slot m of thread t is i = t + m*TPU (TPU = N/16); a radix-R pass runs S = 16/R butterflies per
// thread on slots q + r*S; after the last pass the spectrum is back in the same slot map, so forward FFT -> chirp ->
// inverse FFT needs no exchange in between.
#pragma once
#include <cuda_runtime.h>

namespace dedisp_aos {

typedef float2 C;  // (re, im)

__device__ __forceinline__ C cadd(C a, C b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ C csub(C a, C b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ C mul_i(C a) { return make_float2(-a.y, a.x); }  // i*a: folds into the consumer's operand
// a * (c + i*s)
__device__ __forceinline__ C crot(C a, float c, float s)
{
    return __ffma2_rn(mul_i(a), make_float2(s, s), __fmul2_rn(a, make_float2(c, c)));
}
__device__ __forceinline__ C cmul(C a, C w) { return crot(a, w.x, w.y); }

// d * exp(SIGN * 2*pi*i * j/16), j in [0, 8); j and SIGN are compile-time constants after unrolling.
template <int SIGN>
__device__ __forceinline__ C mul_w16(C d, int j)
{
    constexpr float s = (float)SIGN;
    constexpr float C1 = 0.92387953251128674f;  // cos(pi/8)
    constexpr float S1 = 0.38268343236508977f;  // sin(pi/8)
    constexpr float H = 0.70710678118654752f;   // sqrt(1/2)
    const C sid = SIGN > 0 ? mul_i(d) : make_float2(d.y, -d.x);  // SIGN * i * d
    switch (j) {
        case 0: return d;
        case 1: return crot(d, C1, s * S1);
        case 2: return __fmul2_rn(__fadd2_rn(d, sid), make_float2(H, H));
        case 3: return crot(d, S1, s * C1);
        case 4: return sid;
        case 5: return crot(d, -S1, s * C1);
        case 6: return __fmul2_rn(__fadd2_rn(sid, make_float2(-d.x, -d.y)), make_float2(H, H));
        default: return crot(d, -C1, s * S1);
    }
}

__host__ __device__ constexpr int bitrev(int r, int R)
{
    int o = 0;
    for (int b = 1; b < R; b <<= 1) { o = (o << 1) | (r & 1); r >>= 1; }
    return o;
}

// In-register radix-R DFT (decimation in frequency) on slots q + r*S; X[r] ends up in slot q + bitrev(r)*S.
template <int R, int SIGN>
__device__ __forceinline__ void butterfly(C (&x)[16], int q)
{
    constexpr int S = 16 / R;
#pragma unroll
    for (int half = R / 2; half >= 1; half >>= 1) {
#pragma unroll
        for (int g = 0; g < R; g += 2 * half) {
#pragma unroll
            for (int k = 0; k < half; ++k) {
                const C u = x[q + (g + k) * S], w = x[q + (g + k + half) * S];
                x[q + (g + k) * S] = cadd(u, w);
                x[q + (g + k + half) * S] = mul_w16<SIGN>(csub(u, w), k * (8 / half));
            }
        }
    }
}

template <int R, int SIGN>
__device__ __forceinline__ void pass_butterflies(C (&x)[16])
{
#pragma unroll
    for (int q = 0; q < 16 / R; ++q) butterfly<R, SIGN>(x, q);
}

// Twiddles of one pass in two steps, so that the serial part (table load, squarings) runs in the window between the
// scatter and the gather of the preceding exchange, where the thread would otherwise wait at the barrier.
// prepare = w1 (for radix 16 also the powers 2, 3, 4, 8, 12); apply = the remaining products and x[q + r*S] *= w1^r.
// Every power is a product of depth <= log2 R.
template <int R> struct TwSet { C w1[16 / R]; };
template <> struct TwSet<16> { C w1, w2, w3, w4, w8, w12; };

template <int N, int R, int NS, int SIGN>
__device__ __forceinline__ TwSet<R> twiddle_prepare(int t, const float2* __restrict__ tw)
{
    constexpr int S = 16 / R;
    constexpr int TPU = N / 16;
    TwSet<R> s;
    if constexpr (R == 16) {
        s.w1 = __ldg(&tw[(t & (NS - 1)) * (N / (NS * R))]);
        if (SIGN > 0) s.w1.y = -s.w1.y;
        s.w2 = cmul(s.w1, s.w1);
        s.w3 = cmul(s.w2, s.w1);
        s.w4 = cmul(s.w2, s.w2);
        s.w8 = cmul(s.w4, s.w4);
        s.w12 = cmul(s.w8, s.w4);
    } else {
#pragma unroll
        for (int q = 0; q < S; ++q) {
            s.w1[q] = __ldg(&tw[((t + q * TPU) & (NS - 1)) * (N / (NS * R))]);
            if (SIGN > 0) s.w1[q].y = -s.w1[q].y;
        }
    }
    return s;
}

template <int R>
__device__ __forceinline__ void twiddle_apply(C (&x)[16], const TwSet<R>& tw)
{
    constexpr int S = 16 / R;
    if constexpr (R == 16) {
        x[1] = cmul(x[1], tw.w1);
        x[2] = cmul(x[2], tw.w2);
        x[3] = cmul(x[3], tw.w3);
        x[4] = cmul(x[4], tw.w4);
        x[5] = cmul(x[5], cmul(tw.w4, tw.w1));
        x[6] = cmul(x[6], cmul(tw.w4, tw.w2));
        x[7] = cmul(x[7], cmul(tw.w4, tw.w3));
        x[8] = cmul(x[8], tw.w8);
        x[9] = cmul(x[9], cmul(tw.w8, tw.w1));
        x[10] = cmul(x[10], cmul(tw.w8, tw.w2));
        x[11] = cmul(x[11], cmul(tw.w8, tw.w3));
        x[12] = cmul(x[12], tw.w12);
        x[13] = cmul(x[13], cmul(tw.w12, tw.w1));
        x[14] = cmul(x[14], cmul(tw.w12, tw.w2));
        x[15] = cmul(x[15], cmul(tw.w12, tw.w3));
    } else {
#pragma unroll
        for (int q = 0; q < S; ++q) {
#define XR(r) x[q + (r) * S]
            const C w1 = tw.w1[q];
            XR(1) = cmul(XR(1), w1);
            if constexpr (R >= 4) {
                const C w2 = cmul(w1, w1);
                const C w3 = cmul(w2, w1);
                XR(2) = cmul(XR(2), w2);
                XR(3) = cmul(XR(3), w3);
                if constexpr (R >= 8) {
                    const C w4 = cmul(w2, w2);
                    XR(4) = cmul(XR(4), w4);
                    XR(5) = cmul(XR(5), cmul(w4, w1));
                    XR(6) = cmul(XR(6), cmul(w4, w2));
                    XR(7) = cmul(XR(7), cmul(w4, w3));
                }
            }
#undef XR
        }
    }
}

// One 8-byte cell of padding per 16 keeps the strided STS.64 of an exchange (stride R*NS cells) and its contiguous
// LDS.64 free of bank conflicts (a 64-bit access is served 16 lanes at a time: 17*t mod 16 = t).
__device__ __forceinline__ int pad16(int i) { return i + (i >> 4); }
__host__ __device__ constexpr int padded_len(int n) { return n + (n >> 4); }

// Exchange through shared memory, in two halves so that the caller can place its barrier (and work that only needs the
// barrier, like a prefetch) between them: scatter the pass outputs to their Stockham positions; [barrier]; gather the
// next slot map; [barrier before the buffer is written again].
template <int N, int R, int NS>
__device__ __forceinline__ void exchange_scatter(const C (&x)[16], int t, C* __restrict__ sm)
{
    constexpr int S = 16 / R;
    constexpr int TPU = N / 16;
    static_assert(NS == 1 ? R == 16 : NS % 16 == 0, "pad16(j0 + r*NS) must split into pad16(j0) + constant");
    // j0 is a multiple of 16 when NS == 1 (and r < 16); r*NS is a multiple of 16 otherwise: either way the padded
    // position of output r is pad16(j0) plus a compile-time constant, so every store is base + immediate.
    constexpr int STEP = NS == 1 ? 1 : NS + NS / 16;
#pragma unroll
    for (int q = 0; q < S; ++q) {
        const int jv = t + q * TPU;
        const int k = jv & (NS - 1);
        C* base = sm + pad16((jv - k) * R + k);
#pragma unroll
        for (int r = 0; r < R; ++r) base[r * STEP] = x[q + bitrev(r, R) * S];
    }
}

template <int N>
__device__ __forceinline__ void exchange_gather(C (&x)[16], int t, const C* __restrict__ sm)
{
    constexpr int TPU = N / 16;  // a multiple of 16: pad16(t + m*TPU) = pad16(t) + m*(TPU + TPU/16)
    const C* base = sm + pad16(t);
#pragma unroll
    for (int m = 0; m < 16; ++m) x[m] = base[m * (TPU + TPU / 16)];
}

// Named barrier over the `count` threads that share one exchange buffer (ids 1..15; 0 is __syncthreads).
__device__ __forceinline__ void group_bar(int id, int count)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}

// Puts the outputs of a final radix-R pass (left bit-reversed by butterfly()) back into the canonical slot map.
template <int R>
__device__ __forceinline__ void natural_order(C (&x)[16])
{
    constexpr int S = 16 / R;
    C y[16];
#pragma unroll
    for (int q = 0; q < S; ++q)
#pragma unroll
        for (int r = 0; r < R; ++r) y[q + r * S] = x[q + bitrev(r, R) * S];
#pragma unroll
    for (int m = 0; m < 16; ++m) x[m] = y[m];
}

// Full N-point transform (N = R0*R1*R2*R3, R3 = 1 for three passes); unnormalised; kernel exp(SIGN*2*pi*i*k*n/N).
// tw[m] = exp(-2*pi*i*m/N).  `after_first` runs once between the first barrier and the first gather (the fused kernel
// issues its input prefetch there).
template <int N, int R0, int R1, int R2, int R3, int SIGN, class F>
__device__ __forceinline__ void fft_aos(C (&x)[16], int t, C* __restrict__ sm, const float2* __restrict__ tw, int bar_id,
                                        int bar_count, F after_first)
{
    static_assert(R0 * R1 * R2 * R3 == N, "radix plan");
    pass_butterflies<R0, SIGN>(x);
    exchange_scatter<N, R0, 1>(x, t, sm);
    const TwSet<R1> tw1 = twiddle_prepare<N, R1, R0, SIGN>(t, tw);
    group_bar(bar_id, bar_count);
    after_first();
    exchange_gather<N>(x, t, sm);
    group_bar(bar_id, bar_count);
    twiddle_apply<R1>(x, tw1);
    pass_butterflies<R1, SIGN>(x);
    exchange_scatter<N, R1, R0>(x, t, sm);
    const TwSet<R2> tw2 = twiddle_prepare<N, R2, R0 * R1, SIGN>(t, tw);
    group_bar(bar_id, bar_count);
    exchange_gather<N>(x, t, sm);
    group_bar(bar_id, bar_count);
    twiddle_apply<R2>(x, tw2);
    pass_butterflies<R2, SIGN>(x);
    if constexpr (R3 > 1) {
        exchange_scatter<N, R2, R0 * R1>(x, t, sm);
        const TwSet<R3> tw3 = twiddle_prepare<N, R3, R0 * R1 * R2, SIGN>(t, tw);
        group_bar(bar_id, bar_count);
        exchange_gather<N>(x, t, sm);
        group_bar(bar_id, bar_count);
        twiddle_apply<R3>(x, tw3);
        pass_butterflies<R3, SIGN>(x);
        natural_order<R3>(x);
    } else {
        natural_order<R2>(x);
    }
}

}  // namespace dedisp_aos
