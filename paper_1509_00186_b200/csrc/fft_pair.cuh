// fft_pair.cuh -- register-resident Stockham FFT on PACKED pairs, for the sm_100 f32x2 instructions (FADD2/FMUL2/FFMA2).
//
// A thread holds 16 complex "slots"; each slot carries TWO independent complex numbers in the two lanes of a packed
// float2: lane .x belongs to unit A, lane .y to unit B (two overlap-save blocks of the same channel).  Both units go
// through identical butterflies with identical twiddles, so every FP32 instruction of the transform is a packed one:
// half the issue slots of the scalar form for the same lane throughput (profiles/r1b_fp32_issue.md), and the index
// arithmetic, twiddle loads and twiddle powers (kept scalar, broadcast into the packed multiplies) are shared by the
// two units.
//
// Indexing is the one of fft_regs.cuh: slot m of thread t is element i = t + m*TPU (TPU = N/16); a radix-R pass runs
// S = 16/R butterflies per thread on slots q + r*S; after the last pass the spectrum is back in the same slot map.
#pragma once
#include <cuda_runtime.h>

namespace dedisp_pair {

typedef float2 V;  // two fp32 lanes: (unit A, unit B)
struct C2 { V re, im; };

__device__ __forceinline__ V vdup(float a) { return make_float2(a, a); }
__device__ __forceinline__ V vneg(V a) { return make_float2(-a.x, -a.y); }  // folds into operand modifiers
__device__ __forceinline__ V vadd(V a, V b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ V vsub(V a, V b) { return __fadd2_rn(a, vneg(b)); }
__device__ __forceinline__ V vmul(V a, V b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ V vfma(V a, V b, V c) { return __ffma2_rn(a, b, c); }

__device__ __forceinline__ C2 cadd(C2 a, C2 b) { return C2{vadd(a.re, b.re), vadd(a.im, b.im)}; }
__device__ __forceinline__ C2 csub(C2 a, C2 b) { return C2{vsub(a.re, b.re), vsub(a.im, b.im)}; }
__device__ __forceinline__ C2 cmul(C2 a, C2 w)
{
    return C2{vfma(vneg(a.im), w.im, vmul(a.re, w.re)), vfma(a.im, w.re, vmul(a.re, w.im))};
}
__device__ __forceinline__ C2 csqr(C2 w)
{
    const V t = vmul(w.re, w.im);
    return C2{vfma(vneg(w.im), w.im, vmul(w.re, w.re)), vadd(t, t)};
}

// d * exp(SIGN * 2*pi*i * j/16), j in [0, 8); j and SIGN are compile-time constants after unrolling.
template <int SIGN>
__device__ __forceinline__ C2 mul_w16(C2 d, int j)
{
    constexpr float s = (float)SIGN;
    constexpr float C1 = 0.92387953251128674f;  // cos(pi/8)
    constexpr float S1 = 0.38268343236508977f;  // sin(pi/8)
    constexpr float H = 0.70710678118654752f;   // sqrt(1/2)
    switch (j) {
        case 0: return d;
        case 1: return C2{vfma(d.im, vdup(-s * S1), vmul(d.re, vdup(C1))), vfma(d.re, vdup(s * S1), vmul(d.im, vdup(C1)))};
        case 2: return SIGN > 0 ? C2{vmul(vsub(d.re, d.im), vdup(H)), vmul(vadd(d.re, d.im), vdup(H))}
                                : C2{vmul(vadd(d.re, d.im), vdup(H)), vmul(vsub(d.im, d.re), vdup(H))};
        case 3: return C2{vfma(d.im, vdup(-s * C1), vmul(d.re, vdup(S1))), vfma(d.re, vdup(s * C1), vmul(d.im, vdup(S1)))};
        case 4: return SIGN > 0 ? C2{vneg(d.im), d.re} : C2{d.im, vneg(d.re)};
        case 5: return C2{vfma(d.im, vdup(-s * C1), vmul(d.re, vdup(-S1))), vfma(d.re, vdup(s * C1), vmul(d.im, vdup(-S1)))};
        case 6: return SIGN > 0 ? C2{vmul(vadd(d.re, d.im), vdup(-H)), vmul(vsub(d.re, d.im), vdup(H))}
                                : C2{vmul(vsub(d.im, d.re), vdup(H)), vmul(vadd(d.re, d.im), vdup(-H))};
        default: return C2{vfma(d.im, vdup(-s * S1), vmul(d.re, vdup(-C1))), vfma(d.re, vdup(s * S1), vmul(d.im, vdup(-C1)))};
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
__device__ __forceinline__ void butterfly(C2 (&x)[16], int q)
{
    constexpr int S = 16 / R;
#pragma unroll
    for (int half = R / 2; half >= 1; half >>= 1) {
#pragma unroll
        for (int g = 0; g < R; g += 2 * half) {
#pragma unroll
            for (int k = 0; k < half; ++k) {
                const C2 u = x[q + (g + k) * S], w = x[q + (g + k + half) * S];
                x[q + (g + k) * S] = cadd(u, w);
                x[q + (g + k + half) * S] = mul_w16<SIGN>(csub(u, w), k * (8 / half));
            }
        }
    }
}

// Twiddles are the same for both lanes, so they live as SCALAR complex numbers (half the registers, and their powers
// cost scalar FMUL/FFMA: half the FP32 pipe time of packed ones); the packed multiply takes them as broadcast operands.
__device__ __forceinline__ float2 smul(float2 a, float2 b)
{
    return make_float2(fmaf(-a.y, b.y, a.x * b.x), fmaf(a.y, b.x, a.x * b.y));
}
__device__ __forceinline__ float2 ssqr(float2 w) { return make_float2(fmaf(-w.y, w.y, w.x * w.x), 2.0f * w.x * w.y); }
__device__ __forceinline__ C2 cmul_s(C2 a, float2 w) { return cmul(a, C2{vdup(w.x), vdup(w.y)}); }

// Twiddles of one pass, in two steps so that the serial part (table load, squarings) runs in the window between the
// scatter and the gather of the preceding exchange, where the thread would otherwise wait at the barrier:
// prepare = w1 (and for radix 16 the powers 2, 3, 4, 8, 12);  apply = the remaining products and
// x[q + r*S] *= w1^r, r = 1..R-1.  Every power is a product of depth <= log2 R.
template <int R> struct TwSet { float2 w1[16 / R]; };
template <> struct TwSet<16> { float2 w1, w2, w3, w4, w8, w12; };

template <int N, int R, int NS, int SIGN>
__device__ __forceinline__ TwSet<R> twiddle_prepare(int t, const float2* __restrict__ tw)
{
    constexpr int S = 16 / R;
    constexpr int TPU = N / 16;
    TwSet<R> s;
    if constexpr (R == 16) {
        s.w1 = __ldg(&tw[(t & (NS - 1)) * (N / (NS * R))]);
        if (SIGN > 0) s.w1.y = -s.w1.y;
        s.w2 = ssqr(s.w1);
        s.w3 = smul(s.w2, s.w1);
        s.w4 = ssqr(s.w2);
        s.w8 = ssqr(s.w4);
        s.w12 = smul(s.w8, s.w4);
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
__device__ __forceinline__ void twiddle_apply(C2 (&x)[16], const TwSet<R>& tw)
{
    constexpr int S = 16 / R;
    if constexpr (R == 16) {
        x[1] = cmul_s(x[1], tw.w1);
        x[2] = cmul_s(x[2], tw.w2);
        x[3] = cmul_s(x[3], tw.w3);
        x[4] = cmul_s(x[4], tw.w4);
        x[5] = cmul_s(x[5], smul(tw.w4, tw.w1));
        x[6] = cmul_s(x[6], smul(tw.w4, tw.w2));
        x[7] = cmul_s(x[7], smul(tw.w4, tw.w3));
        x[8] = cmul_s(x[8], tw.w8);
        x[9] = cmul_s(x[9], smul(tw.w8, tw.w1));
        x[10] = cmul_s(x[10], smul(tw.w8, tw.w2));
        x[11] = cmul_s(x[11], smul(tw.w8, tw.w3));
        x[12] = cmul_s(x[12], tw.w12);
        x[13] = cmul_s(x[13], smul(tw.w12, tw.w1));
        x[14] = cmul_s(x[14], smul(tw.w12, tw.w2));
        x[15] = cmul_s(x[15], smul(tw.w12, tw.w3));
    } else {
#pragma unroll
        for (int q = 0; q < S; ++q) {
#define XR(r) x[q + (r) * S]
            const float2 w1 = tw.w1[q];
            XR(1) = cmul_s(XR(1), w1);
            if constexpr (R >= 4) {
                const float2 w2 = ssqr(w1);
                const float2 w3 = smul(w2, w1);
                XR(2) = cmul_s(XR(2), w2);
                XR(3) = cmul_s(XR(3), w3);
                if constexpr (R >= 8) {
                    const float2 w4 = ssqr(w2);
                    XR(4) = cmul_s(XR(4), w4);
                    XR(5) = cmul_s(XR(5), smul(w4, w1));
                    XR(6) = cmul_s(XR(6), smul(w4, w2));
                    XR(7) = cmul_s(XR(7), smul(w4, w3));
                }
            }
#undef XR
        }
    }
}

// One 16-byte cell of padding per 16 keeps the strided STS.128 of an exchange (stride R*NS cells) and its contiguous
// LDS.128 free of bank conflicts (a 128-bit access is served 8 lanes at a time).
__device__ __forceinline__ int pad16(int i) { return i + (i >> 4); }
__host__ __device__ constexpr int padded_len(int n) { return n + (n >> 4); }

// The butterflies of one pass (after twiddle_apply when NS > 1).
template <int R, int SIGN>
__device__ __forceinline__ void pass_butterflies(C2 (&x)[16])
{
#pragma unroll
    for (int q = 0; q < 16 / R; ++q) butterfly<R, SIGN>(x, q);
}

// Exchange through shared memory in (reA, reB, imA, imB) cells, in two halves so that the caller can place its barrier
// (and work that only needs the barrier, like a prefetch) between them: scatter the pass outputs to their Stockham
// positions; [barrier]; gather the next slot map; [barrier before the buffer is written again].
template <int N, int R, int NS>
__device__ __forceinline__ void exchange_scatter(const C2 (&x)[16], int t, float4* __restrict__ sm)
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
        const unsigned base = (unsigned)__cvta_generic_to_shared(sm + pad16((jv - k) * R + k));
#pragma unroll
        for (int r = 0; r < R; ++r) {
            // two 8-byte stores written in asm: the (re, im) register pairs of a slot are rarely adjacent, and nvcc
            // would pay four register moves to build a 16-byte store (ptxas still pairs them when they are adjacent,
            // and folds the constant address increments into the immediate offset)
            const C2 v = x[q + bitrev(r, R) * S];
            asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(base + 16 * r * STEP), "f"(v.re.x), "f"(v.re.y)
                         : "memory");
            asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(base + 16 * r * STEP + 8), "f"(v.im.x), "f"(v.im.y)
                         : "memory");
        }
    }
}

template <int N>
__device__ __forceinline__ void exchange_gather(C2 (&x)[16], int t, const float4* __restrict__ sm)
{
    constexpr int TPU = N / 16;  // a multiple of 16: pad16(t + m*TPU) = pad16(t) + m*(TPU + TPU/16)
    const float4* base = sm + pad16(t);
#pragma unroll
    for (int m = 0; m < 16; ++m) {
        const float4 v = base[m * (TPU + TPU / 16)];
        x[m] = C2{make_float2(v.x, v.y), make_float2(v.z, v.w)};
    }
}

// Named barrier over the `count` threads that share one exchange buffer (ids 1..15; 0 is __syncthreads).
__device__ __forceinline__ void group_bar(int id, int count)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}

// Puts the outputs of a final radix-R pass (left bit-reversed by butterfly()) back into the canonical slot map.
template <int R>
__device__ __forceinline__ void natural_order(C2 (&x)[16])
{
    constexpr int S = 16 / R;
    C2 y[16];
#pragma unroll
    for (int q = 0; q < S; ++q)
#pragma unroll
        for (int r = 0; r < R; ++r) y[q + r * S] = x[q + bitrev(r, R) * S];
#pragma unroll
    for (int m = 0; m < 16; ++m) x[m] = y[m];
}

// Full N-point transform (N = R0*R1*R2) of both lanes; unnormalised; kernel exp(SIGN*2*pi*i*k*n/N).  `after_first`
// runs once between the first barrier and the first gather (the fused kernel issues its input prefetch there).
template <int N, int R0, int R1, int R2, int SIGN, class F>
__device__ __forceinline__ void fft_pair(C2 (&x)[16], int t, float4* __restrict__ sm, const float2* __restrict__ tw,
                                         int bar_id, int bar_count, F after_first)
{
    pass_butterflies<R0, SIGN>(x);
    exchange_scatter<N, R0, 1>(x, t, sm);
    const TwSet<R1> tw1 = twiddle_prepare<N, R1, R0, SIGN>(t, tw);  // tw[m] = exp(-2*pi*i*m/N)
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
    natural_order<R2>(x);
}

}  // namespace dedisp_pair
