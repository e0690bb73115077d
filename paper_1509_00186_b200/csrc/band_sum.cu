// band_sum.cu -- alignment of the coherently dedispersed sub-bands in time and band sum (P:L43,
// P:L67; reading R16):  series[d][j] = sum_c out[d][c][j + shift(d, c)].
// HBM-bound: every detected sample is read once (4 B), one float per (dm, j) is written.  A CTA owns 128 consecutive
// j of one trial DM; its 4 thread rows take every fourth channel, eight independent loads in flight per thread (the
// 32 lanes of a warp read 128 contiguous bytes of a channel row; the shift only moves the window), and the four
// partial sums meet in shared memory.  Rounding error ~sqrt(C) ulp.
#include "dedisp_internal.h"

namespace {

constexpr int TJ = 128;     // outputs per CTA
constexpr int SLICES = 4;   // channel slices per CTA
constexpr int UNROLL = 8;   // loads in flight per thread

__global__ void __launch_bounds__(TJ * SLICES) band_sum_kernel(const float* __restrict__ out, long long out_stride,
                                                               const int* __restrict__ shift, int n_chan,
                                                               float* __restrict__ series, long long series_stride,
                                                               long long n_series)
{
    __shared__ float part[SLICES][TJ];
    const int d = blockIdx.y, tx = threadIdx.x, ty = threadIdx.y;
    const long long j = (long long)blockIdx.x * TJ + tx;
    const bool live = j < n_series;  // j + shift < n_out for every live j (n_series = n_out - largest shift)
    const float* row = out + (size_t)d * n_chan * out_stride + (live ? j : 0);
    const int* sh = shift + (size_t)d * n_chan;
    float acc = 0.f;
    int c = ty;
    for (; c + (UNROLL - 1) * SLICES < n_chan; c += UNROLL * SLICES) {
        float v[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const int cc = c + u * SLICES;
            v[u] = live ? __ldg(row + (size_t)cc * out_stride + __ldg(sh + cc)) : 0.f;
        }
#pragma unroll
        for (int u = 0; u < UNROLL; u += 2) acc += v[u] + v[u + 1];
    }
    for (; c < n_chan; c += SLICES)
        if (live) acc += __ldg(row + (size_t)c * out_stride + __ldg(sh + c));
    part[ty][tx] = acc;
    __syncthreads();
    if (ty == 0 && live)
        series[(size_t)d * series_stride + j] = (part[0][tx] + part[1][tx]) + (part[2][tx] + part[3][tx]);
}

// Folding at a trial period (reading R17): bin = floor(frac((t0 + j*dt)/P) * n_bins) decided in fp64 (as the oracle
// does), sums and counts collected in a shared-memory histogram per CTA and merged with one atomic per bin and CTA.
__global__ void __launch_bounds__(256) fold_kernel(const float* __restrict__ series, long long n, double t0, double dt,
                                                   double period, int n_bins, float* __restrict__ sum,
                                                   unsigned int* __restrict__ count)
{
    extern __shared__ float sh_sum[];                                        // [n_bins] sums, then [n_bins] counts
    unsigned int* sh_cnt = reinterpret_cast<unsigned int*>(sh_sum + n_bins);
    for (int b = threadIdx.x; b < n_bins; b += blockDim.x) { sh_sum[b] = 0.f; sh_cnt[b] = 0u; }
    __syncthreads();
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) {
        // no FMA contraction: the bin must come out exactly as in plain IEEE fp64 arithmetic (the oracle's)
        const double turns = __ddiv_rn(__dadd_rn(t0, __dmul_rn((double)j, dt)), period);
        const double phase = __dadd_rn(turns, -floor(turns));
        int b = (int)__dmul_rn(phase, (double)n_bins);
        if (b > n_bins - 1) b = n_bins - 1;
        atomicAdd(&sh_sum[b], __ldg(series + j));
        atomicAdd(&sh_cnt[b], 1u);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < n_bins; b += blockDim.x) {
        if (sh_cnt[b]) { atomicAdd(&sum[b], sh_sum[b]); atomicAdd(&count[b], sh_cnt[b]); }
    }
}

}  // namespace

int dedisp_launch_fold(const float* d_series, long long n, double t0, double dt, double period, int n_bins,
                       float* d_sum, unsigned int* d_count, cudaStream_t st)
{
    DEDISP_CUDA_TRY(cudaMemsetAsync(d_sum, 0, sizeof(float) * n_bins, st));
    DEDISP_CUDA_TRY(cudaMemsetAsync(d_count, 0, sizeof(unsigned int) * n_bins, st));
    long long grid = (n + 256 * 16 - 1) / (256 * 16);  // ~16 samples per thread
    if (grid > 1184) grid = 1184;
    if (grid < 1) grid = 1;
    fold_kernel<<<(unsigned)grid, 256, sizeof(float) * 2 * n_bins, st>>>(d_series, n, t0, dt, period, n_bins, d_sum, d_count);
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}

int dedisp_launch_band_sum(const dedisp_plan_s* p, const float* d_out, long long out_stride, float* d_series,
                           long long series_stride, long long n_series, cudaStream_t st)
{
    dim3 grid((unsigned)((n_series + TJ - 1) / TJ), (unsigned)p->n_dm), block(TJ, SLICES);
    band_sum_kernel<<<grid, block, 0, st>>>(d_out, out_stride, p->d_band_shift, p->n_chan, d_series, series_stride, n_series);
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}
