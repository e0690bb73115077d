// fft_aos.cuh -- register-resident Stockham FFT with ONE complex number per packed f32x2 register pair (re, im).
//
// The sm_100 packed instructions accept lane-swapped, per-lane-negated operands (SASS `.F32x2.LO_HI.NP`) and scalar
// broadcasts (`.F32`), so with the natural (re, im) layout
//   complex add / sub      = 1 FADD2
//   times +-i              = an operand swizzle of the consumer (no instruction)
//   a +- T b, T complex    = 3 FFMA2 (below)
// i.e. half the issue slots of scalar FADD/FMUL/FFMA at the same FP32 lane throughput, with 2 registers per element.
//
// A thread holds E elements (E = 16 or 64); N/E threads (TPU) make one transform.  Element slot m of thread t is
// i = t + m*TPU; a radix-R pass runs S = E/R butterflies per thread on slots q + r*S; after the last pass the spectrum
// is back in the same slot map, so forward FFT -> chirp -> second FFT needs no exchange in between.  E = 64 does a
// 4096-point transform in TWO radix-64 passes with ONE trip through shared memory (E = 16: three passes, two trips);
// the shared-memory data pipe is what bounds the fused kernel once the FP32 work is folded (profiles/r2b_*).
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
// instead of FMUL2 + FFMA2 + 2 FADD2, and a pass needs only log2(R) powers of w and R/2 - log2(R) products with
// constants: T for k >= M/2 is (SIGN i) T_{k - M/2}, an operand swizzle.  Measured per butterfly
// (bench.py --ubench fp32-issue): 8.3 against 9.9 SM sub-partition cycles.  In the first pass T is a compile-time
// constant; 1 and +-i cost two FADD2.
// ---------------------------------------------------------------------------------------------------------------

// cos(2 pi j / 64), j = 0..16 (sin(2 pi j / 64) = cos(2 pi (16 - j) / 64)); j is a constant after unrolling
__device__ __forceinline__ float cos64(int j)
{
    switch (j) {
        case 0: return 1.0f;
        case 1: return 0.99518472667219688624f;
        case 2: return 0.98078528040323044913f;
        case 3: return 0.95694033573220886494f;
        case 4: return 0.92387953251128675613f;
        case 5: return 0.88192126434835502971f;
        case 6: return 0.83146961230254523708f;
        case 7: return 0.77301045336273696081f;
        case 8: return 0.70710678118654752440f;
        case 9: return 0.63439328416364549822f;
        case 10: return 0.55557023301960222474f;
        case 11: return 0.47139673682599764856f;
        case 12: return 0.38268343236508977173f;
        case 13: return 0.29028467725446236764f;
        case 14: return 0.19509032201612826785f;
        case 15: return 0.09801714032956060199f;
        default: return 0.0f;
    }
}
// W_{M2}^{kb} = (cos, SIGN sin)(2 pi kb / M2), kb <= M2/4, M2 <= 64
template <int SIGN, int M2>
__device__ __forceinline__ C w_const(int kb)
{
    const int j = kb * (64 / M2);
    return make_float2(cos64(j), (float)SIGN * cos64(16 - j));
}

// 2a - u in one FFMA2.  Written in PTX on 64-bit registers: with the intrinsic, ptxas copies about a quarter of these
// results to a scratch register pair before they are stored to shared memory (MOV, MOV, STS.64 on one pair, serialised).
__device__ __forceinline__ C two_a_minus(C a, C u)
{
    unsigned long long ra, ru, rv;
    C v;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(ru) : "f"(-u.x), "f"(-u.y));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rv) : "l"(ra), "l"(0x4000000040000000ull), "l"(ru));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(v.x), "=f"(v.y) : "l"(rv));
    return v;
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
    b = two_a_minus(a, u);
    a = u;
}

// Stage M2 (2, 4, ..., R) of a radix-R DIT butterfly network on c[0..R): G_M -> G_{2M}; ws = w^{R/M2} when TW.
template <int R, int SIGN, bool TW, int M2>
__device__ __forceinline__ void dit_stage(C (&c)[R], C ws)
{
    constexpr int s2 = R / M2, M = M2 / 2, quarter = M2 >= 4 ? M2 / 4 : 1;
    C nxt[R];
#pragma unroll
    for (int kb = 0; kb < quarter; ++kb) {
        C T = make_float2(1.f, 0.f);
        if (TW) T = kb == 0 ? ws : cmul(ws, w_const<SIGN, M2>(kb));
        else if (kb > 0) T = w_const<SIGN, M2>(kb);
#pragma unroll
        for (int rot = 0; rot < M / quarter; ++rot) {
            const int k = kb + rot * quarter;
#pragma unroll
            for (int o = 0; o < s2; ++o) {
                C a = c[o + 2 * s2 * k], b = c[o + s2 + 2 * s2 * k];
                if (!TW && kb == 0) {  // T = 1 or SIGN i
                    const C tb = rot == 0 ? b : (SIGN > 0 ? mul_i(b) : make_float2(b.y, -b.x));
                    const C u = cadd(a, tb);
                    b = csub(a, tb);
                    a = u;
                } else {
                    bfly_tw<SIGN>(a, b, T, rot != 0);
                }
                nxt[o + s2 * k] = a;
                nxt[o + s2 * (k + M)] = b;
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) c[r] = nxt[r];
}

// In-register radix-R DFT of slots q + r*S (natural order in, natural order out); when TW the inputs carry the
// twiddles w^r, folded as described above.
template <int E, int R, int SIGN, bool TW>
__device__ __forceinline__ void dft_dit(C (&x)[E], int q, C w)
{
    constexpr int S = E / R;
    // powers of w by squaring: w1 = w, w2 = w^2, ... (unused ones are dead code)
    const C w1 = w, w2 = cmul(w1, w1), w4 = cmul(w2, w2), w8 = cmul(w4, w4), w16 = cmul(w8, w8), w32 = cmul(w16, w16);
    C c[R];
#pragma unroll
    for (int r = 0; r < R; ++r) c[r] = x[q + r * S];
    // stage M2 uses w^{R/M2}
    if constexpr (R >= 2) dit_stage<R, SIGN, TW, 2>(c, R == 2 ? w1 : R == 4 ? w2 : R == 8 ? w4 : R == 16 ? w8 : R == 32 ? w16 : w32);
    if constexpr (R >= 4) dit_stage<R, SIGN, TW, 4>(c, R == 4 ? w1 : R == 8 ? w2 : R == 16 ? w4 : R == 32 ? w8 : w16);
    if constexpr (R >= 8) dit_stage<R, SIGN, TW, 8>(c, R == 8 ? w1 : R == 16 ? w2 : R == 32 ? w4 : w8);
    if constexpr (R >= 16) dit_stage<R, SIGN, TW, 16>(c, R == 16 ? w1 : R == 32 ? w2 : w4);
    if constexpr (R >= 32) dit_stage<R, SIGN, TW, 32>(c, R == 32 ? w1 : w2);
    if constexpr (R >= 64) dit_stage<R, SIGN, TW, 64>(c, w1);
#pragma unroll
    for (int r = 0; r < R; ++r) x[q + r * S] = c[r];
}

// The Stockham twiddles w of one pass, one per sub-butterfly: w = exp(SIGN 2 pi i (j mod NS) / (NS R)), NS = product
// of the radices of the passes before this one; tw[m] = exp(-2 pi i m / N).  Loaded in the window between the scatter
// and the gather of the preceding exchange, so the latency of the table read hides behind the barrier.
template <int E, int R> struct TwBase { C w[E / R]; };
template <int E, int N, int R, int NS, int SIGN>
__device__ __forceinline__ TwBase<E, R> twiddle_load(int t, const float2* __restrict__ tw)
{
    constexpr int TPU = N / E;
    TwBase<E, R> s;
#pragma unroll
    for (int q = 0; q < E / R; ++q) {
        s.w[q] = __ldg(&tw[((t + q * TPU) & (NS - 1)) * (N / (NS * R))]);
        if (SIGN > 0) s.w[q].y = -s.w[q].y;
    }
    return s;
}

// One pass over all S = E/R sub-butterflies of the thread (TW = false: first pass, no twiddles).
template <int E, int R, int SIGN, bool TW>
__device__ __forceinline__ void pass_dit(C (&x)[E], const TwBase<E, R>& tb)
{
#pragma unroll
    for (int q = 0; q < E / R; ++q) dft_dit<E, R, SIGN, TW>(x, q, tb.w[q]);
}

// Exchange buffer: two 8-byte cells of padding per P cells, P = the first pass's radix.  In the first exchange thread t
// writes cells t*P .. t*P + P - 1, two at a time with STS.128: rows of P + 2 cells start 16-byte aligned, and a quarter
// warp's eight stores (served together) fall (P + 2) * 8 bytes = 16 (mod 128) apart: no bank conflict.  Every other access
// is contiguous across threads (64-bit, served 16 lanes at a time).
template <int P> __host__ __device__ constexpr int padp(int i) { return i + 2 * (i / P); }

// Exchange through shared memory, in two halves so that the caller can place its barrier (and work that only needs the
// barrier, like a prefetch) between them: scatter the pass outputs to their Stockham positions; [barrier]; gather the
// next slot map; [barrier before the buffer is written again].
template <int E, int N, int R, int NS, int P>
__device__ __forceinline__ void exchange_scatter(const C (&x)[E], int t, C* __restrict__ sm)
{
    constexpr int S = E / R;
    constexpr int TPU = N / E;
    static_assert(NS == 1 ? R == P : NS % P == 0, "padp(j0 + r*NS) must split into padp(j0) + constant");
    // NS == 1: output r of butterfly j goes to cell j*R + r, j*R a multiple of P = R; otherwise r*NS is a multiple of
    // P: either way the padded position of output r is padp(j0) plus a compile-time constant (base + immediate).
    constexpr int STEP = NS == 1 ? 1 : NS + 2 * (NS / P);
#pragma unroll
    for (int q = 0; q < S; ++q) {
        const int jv = t + q * TPU;
        const int k = jv & (NS - 1);
        C* base = sm + padp<P>((jv - k) * R + k);
        if constexpr (NS == 1) {  // adjacent cells: 16-byte stores
#pragma unroll
            for (int r = 0; r < R; r += 2)
                *reinterpret_cast<float4*>(base + r) =
                    make_float4(x[q + r * S].x, x[q + r * S].y, x[q + (r + 1) * S].x, x[q + (r + 1) * S].y);
        } else {
#pragma unroll
            for (int r = 0; r < R; ++r) base[r * STEP] = x[q + r * S];
        }
    }
}

template <int E, int N, int P>
__device__ __forceinline__ void exchange_gather(C (&x)[E], int t, const C* __restrict__ sm)
{
    constexpr int TPU = N / E;
    static_assert(TPU % P == 0 || P % TPU == 0, "padp(t + m*TPU) must be padp(t) + constant");
    const C* base = sm + padp<P>(t);  // t < TPU: padp(t + m*TPU) = padp(t) + padp(m*TPU) in both cases
#pragma unroll
    for (int m = 0; m < E; ++m) x[m] = base[padp<P>(m * TPU)];
}

// Barrier over the `count` threads that share one exchange buffer: a named barrier (ids 1..15; 0 is __syncthreads),
// or, when the threads of a transform sit in one warp, a warp barrier.
__device__ __forceinline__ void group_bar(int id, int count)
{
    if (count <= 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}

// Full N-point transform (N = R0*R1*R2*R3, trailing radices 1 when unused); unnormalised; kernel
// exp(SIGN*2*pi*i*k*n/N).  `after_first` runs once between the first barrier and the first gather (the fused kernel
// issues its input prefetch there).  Every gather is followed by a barrier, so on return the exchange buffer is free.
// PRE_BAR: the buffer is still being read by the caller on entry; a barrier is placed before the first scatter.
template <int E, int N, int R0, int R1, int R2, int R3, int SIGN, bool PRE_BAR, class F>
__device__ __forceinline__ void fft_aos(C (&x)[E], int t, C* __restrict__ sm, const float2* __restrict__ tw, int bar_id,
                                        int bar_count, F after_first)
{
    static_assert(R0 * R1 * R2 * R3 == N, "radix plan");
    pass_dit<E, R0, SIGN, false>(x, TwBase<E, R0>{});
    if (PRE_BAR) group_bar(bar_id, bar_count);  // the caller's last reads of the exchange buffer end here
    exchange_scatter<E, N, R0, 1, R0>(x, t, sm);
    const TwBase<E, R1> tw1 = twiddle_load<E, N, R1, R0, SIGN>(t, tw);
    group_bar(bar_id, bar_count);
    after_first();
    exchange_gather<E, N, R0>(x, t, sm);
    group_bar(bar_id, bar_count);
    pass_dit<E, R1, SIGN, true>(x, tw1);
    if constexpr (R2 > 1) {
            exchange_scatter<E, N, R1, R0, R0>(x, t, sm);
        const TwBase<E, R2> tw2 = twiddle_load<E, N, R2, R0 * R1, SIGN>(t, tw);
        group_bar(bar_id, bar_count);
        exchange_gather<E, N, R0>(x, t, sm);
        group_bar(bar_id, bar_count);
            pass_dit<E, R2, SIGN, true>(x, tw2);
        if constexpr (R3 > 1) {
                    exchange_scatter<E, N, R2, R0 * R1, R0>(x, t, sm);
            const TwBase<E, R3> tw3 = twiddle_load<E, N, R3, R0 * R1 * R2, SIGN>(t, tw);
            group_bar(bar_id, bar_count);
            exchange_gather<E, N, R0>(x, t, sm);
            group_bar(bar_id, bar_count);
                    pass_dit<E, R3, SIGN, true>(x, tw3);
        }
    }
}

}  // namespace dedisp_aos
