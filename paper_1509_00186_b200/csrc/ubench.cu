// ubench.cu -- FP32 issue-rate micro-benchmark of the instruction forms the fused kernel is built from
// (dedisp_ubench_fp32, `python bench.py --ubench fp32-issue`).  It exists so that the per-form cycle costs DESIGN.md
// section 6 argues with can be regenerated from the repo.  One persistent 1024-thread CTA per SM with 64 registers per
// thread, like fused_aos_kernel: 8 warps per SM sub-partition, each thread holding 8 independent (a, b) complex pairs
// in packed f32x2 registers and one per-thread twiddle (c, s).  Every form is one radix-2 butterfly on a pair; the
// kernel reports SM sub-partition cycles per butterfly (clock64 around the loop, max over the CTA's warps).
#include "dedisp_internal.h"
#include "fft_aos.cuh"

using namespace dedisp_aos;

namespace {

constexpr int UB_CTA = 1024, UB_PAIRS = 8;

template <int FORM>
__device__ __forceinline__ void bfly(C& a, C& b, float c, float s)
{
    if constexpr (FORM == 0) {         // plain butterfly: 2 FADD2
        const C u = cadd(a, b), v = csub(a, b);
        a = u; b = v;
    } else if constexpr (FORM == 1) {  // butterfly with +-i on b: 2 FADD2 with a lane-swapped operand
        const C ib = mul_i(b);
        const C u = cadd(a, ib), v = csub(a, ib);
        a = u; b = v;
    } else if constexpr (FORM == 2) {  // general twiddle, conventional: FMUL2 + FFMA2 + 2 FADD2
        const C t = crot(b, c, s);
        const C u = cadd(a, t), v = csub(a, t);
        a = u; b = v;
    } else if constexpr (FORM == 3) {  // general twiddle folded into the butterfly: 3 FFMA2 (v = 2a - u)
        const C t = __ffma2_rn(b, make_float2(c, c), a);
        const C u = __ffma2_rn(mul_i(b), make_float2(s, s), t);
        const C v = __ffma2_rn(a, make_float2(2.f, 2.f), make_float2(-u.x, -u.y));
        a = u; b = v;
    } else if constexpr (FORM == 4) {  // the same with the twiddle rotated by i: (c, s) -> (-s, c), no extra instruction
        const C t = __ffma2_rn(b, make_float2(-s, -s), a);
        const C u = __ffma2_rn(mul_i(b), make_float2(c, c), t);
        const C v = __ffma2_rn(a, make_float2(2.f, 2.f), make_float2(-u.x, -u.y));
        a = u; b = v;
    } else if constexpr (FORM == 5) {  // folded, without the 2a - u trick: 4 FFMA2
        const C t = __ffma2_rn(b, make_float2(c, c), a);
        const C u = __ffma2_rn(mul_i(b), make_float2(s, s), t);
        const C t2 = __ffma2_rn(b, make_float2(-c, -c), a);
        const C v = __ffma2_rn(mul_i(b), make_float2(-s, -s), t2);
        a = u; b = v;
    } else if constexpr (FORM == 6) {  // constant twiddle (immediates) folded: 3 FFMA2
        constexpr float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f;
        const C t = __ffma2_rn(b, make_float2(C1, C1), a);
        const C u = __ffma2_rn(mul_i(b), make_float2(S1, S1), t);
        const C v = __ffma2_rn(a, make_float2(2.f, 2.f), make_float2(-u.x, -u.y));
        a = u; b = v;
    } else {                           // constant twiddle, conventional: FMUL2 + FFMA2 (immediates) + 2 FADD2
        constexpr float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f;
        const C t = crot(b, C1, S1);
        const C u = cadd(a, t), v = csub(a, t);
        a = u; b = v;
    }
}

template <int FORM>
__global__ void __launch_bounds__(UB_CTA, 1) ubench_kernel(const float2* __restrict__ in, float2* __restrict__ out,
                                                           int iters, long long* __restrict__ cycles)
{
    C a[UB_PAIRS], b[UB_PAIRS];
    const int gid = blockIdx.x * UB_CTA + threadIdx.x;
#pragma unroll
    for (int j = 0; j < UB_PAIRS; ++j) {
        a[j] = in[(gid * 2 * UB_PAIRS + 2 * j) & 4095];
        b[j] = in[(gid * 2 * UB_PAIRS + 2 * j + 1) & 4095];
    }
    const float2 w = in[gid & 4095];
    const float c = w.x, s = w.y;
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < UB_PAIRS; ++j) bfly<FORM>(a[j], b[j], c, s);
        // rotate the pairs so that a later iteration cannot be folded into an earlier one
        const C tmp = b[0];
#pragma unroll
        for (int j = 0; j + 1 < UB_PAIRS; ++j) b[j] = b[j + 1];
        b[UB_PAIRS - 1] = tmp;
    }
    const long long t1 = clock64();
    C acc = a[0];
#pragma unroll
    for (int j = 0; j < UB_PAIRS; ++j) acc = cadd(acc, cadd(a[j], b[j]));
    out[gid] = acc;
    __shared__ long long tmax;
    if (threadIdx.x == 0) tmax = 0;
    __syncthreads();
    atomicMax(&tmax, t1 - t0);
    __syncthreads();
    if (threadIdx.x == 0) cycles[blockIdx.x] = tmax;
}

template <int FORM>
void launch(int grid, const float2* in, float2* out, int iters, long long* cyc)
{
    ubench_kernel<FORM><<<grid, UB_CTA>>>(in, out, iters, cyc);
}

}  // namespace

extern "C" int dedisp_ubench_fp32(int form, int iters, double* cycles_per_butterfly, double* ms)
{
    if (form < 0 || form >= DEDISP_UBENCH_FORMS || iters <= 0 || !cycles_per_butterfly || !ms) return DEDISP_EINVAL;
    int dev = 0, n_sm = 0;
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    DEDISP_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    float2 *d_in = nullptr, *d_out = nullptr;
    long long* d_cyc = nullptr;
    DEDISP_CUDA_TRY(cudaMalloc(&d_in, sizeof(float2) * 4096));
    DEDISP_CUDA_TRY(cudaMalloc(&d_out, sizeof(float2) * (size_t)n_sm * UB_CTA));
    DEDISP_CUDA_TRY(cudaMalloc(&d_cyc, sizeof(long long) * n_sm));
    float2* h = (float2*)malloc(sizeof(float2) * 4096);
    for (int i = 0; i < 4096; ++i) h[i] = make_float2(0.6f + 1e-4f * (i % 97), 0.8f - 1e-4f * (i % 89));
    cudaMemcpy(d_in, h, sizeof(float2) * 4096, cudaMemcpyHostToDevice);
    free(h);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    for (int rep = 0; rep < 2; ++rep) {  // first pass warms the instruction cache
        cudaEventRecord(e0);
        switch (form) {
            case 0: launch<0>(n_sm, d_in, d_out, iters, d_cyc); break;
            case 1: launch<1>(n_sm, d_in, d_out, iters, d_cyc); break;
            case 2: launch<2>(n_sm, d_in, d_out, iters, d_cyc); break;
            case 3: launch<3>(n_sm, d_in, d_out, iters, d_cyc); break;
            case 4: launch<4>(n_sm, d_in, d_out, iters, d_cyc); break;
            case 5: launch<5>(n_sm, d_in, d_out, iters, d_cyc); break;
            case 6: launch<6>(n_sm, d_in, d_out, iters, d_cyc); break;
            default: launch<7>(n_sm, d_in, d_out, iters, d_cyc); break;
        }
        cudaEventRecord(e1);
    }
    cudaError_t err = cudaDeviceSynchronize();
    float t = 0.f;
    cudaEventElapsedTime(&t, e0, e1);
    long long* hc = (long long*)malloc(sizeof(long long) * n_sm);
    cudaMemcpy(hc, d_cyc, sizeof(long long) * n_sm, cudaMemcpyDeviceToHost);
    double sum = 0.0;
    for (int i = 0; i < n_sm; ++i) sum += (double)hc[i];
    free(hc);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d_in); cudaFree(d_out); cudaFree(d_cyc);
    DEDISP_CUDA_TRY(err);
    // 8 warps per SM sub-partition, UB_PAIRS butterflies per warp and iteration
    *cycles_per_butterfly = sum / n_sm / ((double)(UB_CTA / 32 / 4) * UB_PAIRS * iters);
    *ms = t;
    return DEDISP_OK;
}
