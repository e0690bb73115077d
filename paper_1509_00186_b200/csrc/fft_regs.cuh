// fft_regs.cuh -- register-resident pieces of the Stockham FFT used by the fused dedispersion kernel.
//
// One thread holds E complex values x[m] of an N-point sequence, always the elements  i = t + m*TPU  (t = thread index
// inside the unit, TPU = N/E threads per unit).  A radix-R pass (R | E) lets the thread run S = E/R butterflies; butterfly
// q works on registers q + r*S (r < R), i.e. on "virtual thread" jv = t + q*TPU of the classic formulation
//     v[r]  = in[jv + r*N/R] * exp(SIGN*2*pi*i*r*k/(NS*R)),   k = jv mod NS        (NS = product of earlier radices)
//     V     = DFT_R(v)
//     out[(jv - k)*R + k + r*NS] = V[r]
// After the last pass (NS*R == N) the output index is again jv + r*N/R: the spectrum lands in the same register map
// it was loaded with, so forward FFT -> chirp multiply -> inverse FFT needs no exchange in between.
#pragma once
#include <cuda_runtime.h>

namespace dedisp_fft {

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(-a.y, b.y, a.x * b.x), fmaf(a.y, b.x, a.x * b.y));
}

// d * exp(SIGN * 2*pi*i * j/16), j in [0, 8): the constant twiddles inside a radix-R (R <= 16) butterfly.
// j and SIGN are compile-time constants after unrolling; the switch folds away.
template <int SIGN>
__device__ __forceinline__ float2 mul_w16(float2 d, int j)
{
    constexpr float s = (float)SIGN;
    constexpr float C1 = 0.92387953251128674f;  // cos(pi/8)
    constexpr float S1 = 0.38268343236508977f;  // sin(pi/8)
    constexpr float H = 0.70710678118654752f;   // sqrt(1/2)
    switch (j) {
        case 0: return d;
        case 1: return make_float2(fmaf(-s * S1, d.y, C1 * d.x), fmaf(s * S1, d.x, C1 * d.y));
        case 2: return make_float2(H * (d.x - s * d.y), H * (s * d.x + d.y));
        case 3: return make_float2(fmaf(-s * C1, d.y, S1 * d.x), fmaf(s * C1, d.x, S1 * d.y));
        case 4: return make_float2(-s * d.y, s * d.x);
        case 5: return make_float2(fmaf(-s * C1, d.y, -S1 * d.x), fmaf(s * C1, d.x, -S1 * d.y));
        case 6: return make_float2(H * (-d.x - s * d.y), H * (s * d.x - d.y));
        default: return make_float2(fmaf(-s * S1, d.y, -C1 * d.x), fmaf(s * S1, d.x, -C1 * d.y));
    }
}

__host__ __device__ constexpr int bitrev(int r, int R)
{
    int o = 0;
    for (int b = 1; b < R; b <<= 1) { o = (o << 1) | (r & 1); r >>= 1; }
    return o;
}

// In-register radix-R DFT (decimation in frequency, log2 R radix-2 stages) on x[q + r*S], r < R.
// On return X[r] sits in x[q + bitrev(r)*S].
template <int R, int SIGN, int E>
__device__ __forceinline__ void butterfly(float2 (&x)[E], int q)
{
    constexpr int S = E / R;
#pragma unroll
    for (int half = R / 2; half >= 1; half >>= 1) {
#pragma unroll
        for (int g = 0; g < R; g += 2 * half) {
#pragma unroll
            for (int k = 0; k < half; ++k) {
                const float2 u = x[q + (g + k) * S], w = x[q + (g + k + half) * S];
                x[q + (g + k) * S] = cadd(u, w);
                x[q + (g + k + half) * S] = mul_w16<SIGN>(csub(u, w), k * (8 / half));
            }
        }
    }
}

// Multiply x[q + r*S] by w1^r, r = 1..R-1, w1 = exp(SIGN*2*pi*i*k/(NS*R)).  Powers by products of depth <= log2 R
// (w^r = w^hb * w^(r-hb), hb the top bit of r), so the rounding error of any power stays within ~4 ulp.
template <int R, int E>
__device__ __forceinline__ void twiddle(float2 (&x)[E], int q, float2 w1)
{
    constexpr int S = E / R;
    float2 wp[R];
    wp[1] = w1;
#pragma unroll
    for (int r = 2; r < R; ++r) {
        int hb = 1;
        while (hb * 2 <= r) hb *= 2;
        wp[r] = (r == hb) ? cmul(wp[r / 2], wp[r / 2]) : cmul(wp[hb], wp[r - hb]);
    }
#pragma unroll
    for (int r = 1; r < R; ++r) x[q + r * S] = cmul(x[q + r * S], wp[r]);
}

// smem index padding: one float2 of padding per 16 keeps both the strided writes (stride R*NS) and the contiguous
// reads of an exchange free of bank conflicts for 8-byte accesses.
__device__ __forceinline__ int pad16(int i) { return i + (i >> 4); }
__host__ __device__ constexpr int padded_len(int n) { return n + (n >> 4); }

// One pass: twiddle (skipped when NS == 1) + butterflies.  tw = exp(-2*pi*i*m/N) table in global memory.
template <int N, int R, int NS, int SIGN, int E>
__device__ __forceinline__ void pass_compute(float2 (&x)[E], int t, const float2* __restrict__ tw)
{
    constexpr int S = E / R;
    constexpr int TPU = N / E;
#pragma unroll
    for (int q = 0; q < S; ++q) {
        if (NS > 1) {
            const int k = (t + q * TPU) & (NS - 1);
            float2 w1 = __ldg(&tw[k * (N / (NS * R))]);
            if (SIGN > 0) w1.y = -w1.y;
            twiddle<R, E>(x, q, w1);
        }
        butterfly<R, SIGN, E>(x, q);
    }
}

// Exchange through shared memory: scatter the pass outputs to their Stockham positions, gather the next map.
template <int N, int R, int NS, int E>
__device__ __forceinline__ void exchange(float2 (&x)[E], int t, float2* __restrict__ sm)
{
    constexpr int S = E / R;
    constexpr int TPU = N / E;
#pragma unroll
    for (int q = 0; q < S; ++q) {
        const int jv = t + q * TPU;
        const int k = jv & (NS - 1);
        const int j0 = (jv - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) sm[pad16(j0 + r * NS)] = x[q + bitrev(r, R) * S];
    }
    __syncthreads();
#pragma unroll
    for (int m = 0; m < E; ++m) x[m] = sm[pad16(t + m * TPU)];
    __syncthreads();
}

}  // namespace dedisp_fft
