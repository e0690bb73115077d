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

// ---------------------------------------------------------------------------------------------------------------
// Radix-R pass = decimation-in-TIME butterflies with the pass's input twiddles folded in.
//
// A pass transforms y[r] = w^r x[r], r < R (w = the Stockham twiddle of this thread and pass; w = 1 in the first pass):
// X[k] = sum_r y[r] W^{rk}, W = exp(SIGN 2 pi i / R).  With G_{M,o}[k] = (the M-point DFT of y[o + (R/M) j], j < M) / w^o
//      G_{2M,o}[k]     = G_{M,o}[k] + T G_{M,o+s'}[k]
//      G_{2M,o}[k + M] = G_{M,o}[k] - T G_{M,o+s'}[k],      T = w^{s'} W_{2M}^k,  s' = R/(2M),  o < s',  k < M
// and X = G_{R,0}: the powers w^r never multiply the data on their own, every butterfly is u = a + T b, v = a - T b
//      t = b * (c, c) + a;   u = (i b) * (s, s) + t;   v = a * 2 - u            (3 FFMA2, T = c + i s)
// instead of FMUL2 + FFMA2 + 2 FADD2, and a pass needs only log2(R) powers of w and R/2 - 1 products with constants:
// T for k >= M/2 is (SIGN i) T_{k - M/2}, an operand swizzle.  Measured per butterfly (bench.py --ubench fp32-issue):
// 8.3 against 9.9 SM sub-partition cycles.  In the first pass T is a compile-time constant; 1 and +-i cost two FADD2.
// ---------------------------------------------------------------------------------------------------------------

// index of T = w^{R/M2} W_{M2}^{kb}, kb < max(1, M2/4), in a pass's twiddle set: M2 = 2, 4, 8, 16 -> 0, 1, 2..3, 4..7
__host__ __device__ constexpr int tw_index(int M2, int kb) { return (M2 >= 4 ? M2 / 4 : 0) + kb; }
template <int R> struct TwSet { C t[16 / R][R / 2]; };  // [sub-butterfly q][tw_index]; R/2 = 1 + 1 + 2 + 4 ... entries
template <> struct TwSet<1> {};

// (cos, SIGN sin) of 2 pi kb / M2 for the constants a radix <= 16 pass needs (kb < M2/4, so M2 = 8: kb = 1; 16: 1..3)
template <int SIGN>
__device__ __forceinline__ C w_const(int M2, int kb)
{
    constexpr float s = (float)SIGN;
    constexpr float C1 = 0.92387953251128674f;  // cos(pi/8)
    constexpr float S1 = 0.38268343236508977f;  // sin(pi/8)
    constexpr float H = 0.70710678118654752f;   // sqrt(1/2)
    if (kb == 0) return make_float2(1.f, 0.f);
    if (M2 == 8) return make_float2(H, s * H);
    return kb == 1 ? make_float2(C1, s * S1) : kb == 2 ? make_float2(H, s * H) : make_float2(S1, s * C1);
}

// u = a + T b, v = a - T b with T = (c + i s) (SIGN i)^rot
template <int SIGN>
__device__ __forceinline__ void bfly_tw(C& a, C& b, C T, bool rot)
{
    const C sib = SIGN > 0 ? mul_i(b) : make_float2(b.y, -b.x);  // SIGN * i * b
    C u;
    if (!rot) {  // T b = c b + s (i b)
        u = __ffma2_rn(b, make_float2(T.x, T.x), a);
        u = __ffma2_rn(sib, make_float2((float)SIGN * T.y, (float)SIGN * T.y), u);
    } else {  // (SIGN i) T b = c (SIGN i b) - SIGN s b
        u = __ffma2_rn(sib, make_float2(T.x, T.x), a);
        u = __ffma2_rn(b, make_float2(-(float)SIGN * T.y, -(float)SIGN * T.y), u);
    }
    b = __ffma2_rn(a, make_float2(2.f, 2.f), make_float2(-u.x, -u.y));
    a = u;
}

// In-register radix-R DFT of slots q + r*S (natural order in, natural order out), input twiddles folded when TW.
template <int R, int SIGN, bool TW>
__device__ __forceinline__ void dft_dit(C (&x)[16], int q, const C (&tw)[R / 2])
{
    constexpr int S = 16 / R;
    C cur[R];
#pragma unroll
    for (int r = 0; r < R; ++r) cur[r] = x[q + r * S];
#pragma unroll
    for (int M2 = 2; M2 <= R; M2 <<= 1) {
        const int s2 = R / M2, M = M2 / 2, quarter = M2 >= 4 ? M2 / 4 : 1;
        C nxt[R];
#pragma unroll
        for (int o = 0; o < s2; ++o) {
#pragma unroll
            for (int k = 0; k < M; ++k) {
                C a = cur[o + 2 * s2 * k], b = cur[o + s2 + 2 * s2 * k];
                const int kb = k % quarter;
                const bool rot = k >= quarter;
                if (TW) {
                    bfly_tw<SIGN>(a, b, tw[tw_index(M2, kb)], rot);
                } else if (kb == 0) {  // T = 1 or SIGN i
                    const C tb = !rot ? b : (SIGN > 0 ? mul_i(b) : make_float2(b.y, -b.x));
                    const C u = cadd(a, tb);
                    b = csub(a, tb);
                    a = u;
                } else {
                    bfly_tw<SIGN>(a, b, w_const<SIGN>(M2, kb), rot);
                }
                nxt[o + s2 * k] = a;
                nxt[o + s2 * (k + M)] = b;
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) cur[r] = nxt[r];
    }
#pragma unroll
    for (int r = 0; r < R; ++r) x[q + r * S] = cur[r];
}

// The twiddle set of one pass from w = exp(SIGN 2 pi i (j mod NS) / (NS R)): powers by squaring, the rest by products
// with constants (FMUL2 + FFMA2 with immediates).  Runs in the window between the scatter and the gather of the
// preceding exchange, where the thread would otherwise wait at the barrier.
template <int N, int R, int NS, int SIGN>
__device__ __forceinline__ TwSet<R> twiddle_prepare(int t, const float2* __restrict__ tw)
{
    constexpr int S = 16 / R;
    constexpr int TPU = N / 16;
    TwSet<R> s;
#pragma unroll
    for (int q = 0; q < S; ++q) {
        C w = __ldg(&tw[((t + q * TPU) & (NS - 1)) * (N / (NS * R))]);
        if (SIGN > 0) w.y = -w.y;
        // w^{R/M2} for M2 = R, R/2, ..., 2
#pragma unroll
        for (int M2 = R; M2 >= 2; M2 >>= 1) {
            s.t[q][tw_index(M2, 0)] = w;
#pragma unroll
            for (int kb = 1; kb < M2 / 4; ++kb) {
                const C k = w_const<SIGN>(M2, kb);
                s.t[q][tw_index(M2, kb)] = (M2 == 8 || kb == 2)
                    ? __fmul2_rn(__fadd2_rn(w, SIGN > 0 ? mul_i(w) : make_float2(w.y, -w.x)), make_float2(k.x, k.x))
                    : crot(w, k.x, k.y);
            }
            if (M2 > 2) w = cmul(w, w);
        }
    }
    return s;
}

template <int R, int SIGN, bool TW>
__device__ __forceinline__ void pass_dit(C (&x)[16], const TwSet<TW ? R : 1>& tw)
{
#pragma unroll
    for (int q = 0; q < 16 / R; ++q) {
        if constexpr (TW) {
            dft_dit<R, SIGN, true>(x, q, tw.t[q]);
        } else {
            const C none[R / 2] = {};
            dft_dit<R, SIGN, false>(x, q, none);
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
        for (int r = 0; r < R; ++r) base[r * STEP] = x[q + r * S];
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

// Full N-point transform (N = R0*R1*R2*R3, R3 = 1 for three passes); unnormalised; kernel exp(SIGN*2*pi*i*k*n/N).
// tw[m] = exp(-2*pi*i*m/N).  `after_first` runs once between the first barrier and the first gather (the fused kernel
// issues its input prefetch there).
template <int N, int R0, int R1, int R2, int R3, int SIGN, class F>
__device__ __forceinline__ void fft_aos(C (&x)[16], int t, C* __restrict__ sm, const float2* __restrict__ tw, int bar_id,
                                        int bar_count, F after_first)
{
    static_assert(R0 * R1 * R2 * R3 == N, "radix plan");
    pass_dit<R0, SIGN, false>(x, TwSet<1>{});
    exchange_scatter<N, R0, 1>(x, t, sm);
    const TwSet<R1> tw1 = twiddle_prepare<N, R1, R0, SIGN>(t, tw);
    group_bar(bar_id, bar_count);
    after_first();
    exchange_gather<N>(x, t, sm);
    group_bar(bar_id, bar_count);
    pass_dit<R1, SIGN, true>(x, tw1);
    exchange_scatter<N, R1, R0>(x, t, sm);
    const TwSet<R2> tw2 = twiddle_prepare<N, R2, R0 * R1, SIGN>(t, tw);
    group_bar(bar_id, bar_count);
    exchange_gather<N>(x, t, sm);
    group_bar(bar_id, bar_count);
    pass_dit<R2, SIGN, true>(x, tw2);
    if constexpr (R3 > 1) {
        exchange_scatter<N, R2, R0 * R1>(x, t, sm);
        const TwSet<R3> tw3 = twiddle_prepare<N, R3, R0 * R1 * R2, SIGN>(t, tw);
        group_bar(bar_id, bar_count);
        exchange_gather<N>(x, t, sm);
        group_bar(bar_id, bar_count);
        pass_dit<R3, SIGN, true>(x, tw3);
    }
}

}  // namespace dedisp_aos
