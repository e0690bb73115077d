// fullband.cu -- the paper's OWN mode: full-band coherent dedispersion without sub-banding
// (Fig. 4).  The GSB spectra are inverse transformed to the real Nyquist-sampled
// voltage series, ONE long transform of N = 2^20 ... 2^28 points covers the whole band, the chirp of Eq. 3
// is applied with the lower band edge as reference, overlap-save returns the dedispersed series, which is squared and
// integrated.  Readings R19-R21; the oracle is oracle/fullband.py.
//
// B200 design (nothing of the paper's cuFFT call sequence is kept):
//   * Two real blocks ride one complex transform: z = v_b + i v_{b+1}.  The chirp is extended to all N bins with
//     Hermitian symmetry, H[N-k] = conj(H[k]), so the filter maps real series to real series and the real and the
//     imaginary part of the result ARE the two dedispersed blocks: no real-FFT split pass, no wasted half.
//   * The long transform is a four-step FFT over HBM, N = N1 x N2 with N1, N2 in {1024 ... 16384}: the row transforms
//     run in the register-resident FFT of fft_aos.cuh (64 elements per thread, radix 64 passes), so a transform of
//     2^27 points makes two passes over the data; the spectrum is left in the four-step's own order [k1][k2] -- the
//     chirp table is stored in that order and the inverse runs the steps backwards, so no reordering pass exists.
//   * forward rows -> chirp -> inverse rows is ONE kernel (the spectrum of a row never leaves the registers).
//   * HBM-bound: 7 passes of 8 B read + 8 B written per complex point (4 transposes, 3 row-transform kernels; the last
//     transpose writes 32-sample partial power sums instead of its result when n_int % 32 == 0), fp32 values, twiddles
//     and chirp from fp64 phases (the paper's fp64 requirement, concerns the phase: pin F7).
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "dedisp_internal.h"
#include "fft_aos.cuh"

using namespace dedisp_aos;

namespace {

constexpr int FB_E = 64;
// threads per CTA of the row kernels: two units where a unit is small enough -- two such CTAs share an SM and drift apart,
// so that one's loads and stores overlap the other's butterflies -- else one unit
template <int R> __host__ __device__ constexpr int fb_cta() { return R / FB_E >= 128 ? R / FB_E : 128; }
template <int N> struct FShape;
template <> struct FShape<1024>  { static constexpr int R0 = 64, R1 = 16, R2 = 1, R3 = 1; };
template <> struct FShape<2048>  { static constexpr int R0 = 64, R1 = 32, R2 = 1, R3 = 1; };
template <> struct FShape<4096>  { static constexpr int R0 = 64, R1 = 64, R2 = 1, R3 = 1; };
template <> struct FShape<8192>  { static constexpr int R0 = 64, R1 = 64, R2 = 2, R3 = 1; };
template <> struct FShape<16384> { static constexpr int R0 = 64, R1 = 64, R2 = 4, R3 = 1; };

// exp(-2 pi i p / N) for p < N from two tables: p = ph * 2^13 + pl, ta[ph] = exp(-2 pi i ph 2^13 / N), tb[pl] =
// exp(-2 pi i pl / N), both rounded from fp64 (the product is good to ~1e-7)
constexpr int TW_LO_BITS = 13;
__device__ __forceinline__ C long_twiddle(unsigned p, const float2* __restrict__ ta, const float2* __restrict__ tb)
{
    return cmul(__ldg(ta + (p >> TW_LO_BITS)), __ldg(tb + (p & ((1u << TW_LO_BITS) - 1))));
}

enum { ROWS_FWD_TWIDDLE = 0, ROWS_CHIRP = 1, ROWS_TWIDDLE_INV = 2, ROWS_GSB = 3 };

struct RowsArgs {
    const float2* in;    // [n_rows][R] (ROWS_GSB: unused)
    float2* out;         // [n_rows][R] (ROWS_GSB: unused)
    const float2* tw;    // [R] exp(-2 pi i m / R)
    const float2 *ta, *tb;  // long twiddle tables (ROWS_FWD_TWIDDLE, ROWS_TWIDDLE_INV)
    const float2* chirp; // ROWS_CHIRP: [rows_per_batch][R] in the spectrum's own order, includes 1/N
    const int8_t* gsb;   // ROWS_GSB: [n_rows][R/2][2]
    float* series;       // ROWS_GSB: [n_rows * R]
    long long n_rows;
    int rows_per_batch;  // rows of one transform (row index inside the transform = row % rows_per_batch)
    unsigned n_mask;     // N - 1
    float gsb_scale;     // 1 / R
};

// One row transform per unit of R/64 threads (256/(R/64) units per CTA); R = row length.
//   ROWS_FWD_TWIDDLE  out[row][k] = DFT(in[row])[k] * W_N^{(row in transform) * k}            (four-step, steps 1-2)
//   ROWS_CHIRP        out[row] = IDFT( DFT(in[row]) * chirp[row in transform] )                (step 3, Eq. 3, step 3')
//   ROWS_TWIDDLE_INV  out[row] = IDFT( in[row][k] * conj(W_N^{(row in transform) * k}) )       (steps 2'-1')
//   ROWS_GSB          series[row*R + n] = Re IDFT(Hermitian extension of gsb[row])[n] / R      (R19: c2r of a spectrum)
template <int R, int MODE>
__global__ void __launch_bounds__((fb_cta<R>()), (fb_cta<R>() == 128 ? 2 : 1)) fb_rows_kernel(const RowsArgs a)
{
    using Sh = FShape<R>;
    constexpr int E = FB_E, TPU = R / E, FB_CTA = fb_cta<R>(), UPS = FB_CTA / TPU, P = Sh::R0, GROUP = TPU < 32 ? 32 : TPU;
    extern __shared__ float2 smem2[];
    const int us = threadIdx.x / TPU, t = threadIdx.x % TPU;
    const int bar_id = threadIdx.x / GROUP + 1;
    C* sm = smem2 + (size_t)us * padp<P>(R);
    const long long row = (long long)blockIdx.x * UPS + us;
    const bool live = row < a.n_rows;
    const long long r = live ? row : a.n_rows - 1;  // idle unit slots redo the last row and store nothing
    const unsigned rt = (unsigned)(r % a.rows_per_batch);
    C x[E];
    if constexpr (MODE == ROWS_GSB) {
        // bins 0 .. R/2-1 are recorded (bin 0: real part only), bin R/2 is 0, the rest is the conjugate mirror (R19)
        const uint16_t* g = reinterpret_cast<const uint16_t*>(a.gsb) + r * (R / 2);  // one (re, im) byte pair per bin
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int k = t + m * TPU;
            const int ks = k < R / 2 ? k : R - k;
            const uint32_t w = __ldg(g + (ks & (R / 2 - 1)));
            const float re = (float)(int8_t)(w & 0xffu), im = (float)(int8_t)(w >> 8);
            x[m] = k == R / 2 ? make_float2(0.f, 0.f)
                              : (k == 0 ? make_float2(re, 0.f) : make_float2(re, k < R / 2 ? im : -im));
        }
    } else {
        const float2* src = a.in + r * R + t;
#pragma unroll
        for (int m = 0; m < E; ++m) x[m] = src[m * TPU];
    }
    if constexpr (MODE == ROWS_TWIDDLE_INV) {
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const C w = long_twiddle((rt * (unsigned)(t + m * TPU)) & a.n_mask, a.ta, a.tb);
            x[m] = crot(x[m], w.x, -w.y);
        }
    }
    if constexpr (MODE == ROWS_FWD_TWIDDLE || MODE == ROWS_CHIRP) {
        fft_aos<E, R, Sh::R0, Sh::R1, Sh::R2, Sh::R3, -1, false>(x, t, sm, a.tw, bar_id, GROUP, [] {});
        if constexpr (MODE == ROWS_FWD_TWIDDLE) {
#pragma unroll
            for (int m = 0; m < E; ++m)
                x[m] = cmul(x[m], long_twiddle((rt * (unsigned)(t + m * TPU)) & a.n_mask, a.ta, a.tb));
        } else {
            const float2* h = a.chirp + (size_t)rt * R + t;
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = cmul(x[m], __ldg(h + m * TPU));
        }
    }
    if constexpr (MODE != ROWS_FWD_TWIDDLE)
        fft_aos<E, R, Sh::R0, Sh::R1, Sh::R2, Sh::R3, +1, false>(x, t, sm, a.tw, bar_id, GROUP, [] {});
    if (!live) return;  // (after the last barrier of the unit's group)
    if constexpr (MODE == ROWS_GSB) {
        float* dst = a.series + r * R + t;
#pragma unroll
        for (int m = 0; m < E; ++m) dst[m * TPU] = x[m].x * a.gsb_scale;
    } else {
        float2* dst = a.out + r * R + t;
#pragma unroll
        for (int m = 0; m < E; ++m) dst[m * TPU] = x[m];
    }
}

// Batched transpose of float2 matrices [rows][cols] -> [cols][rows] through a padded 32 x 32 tile.
// PACK: the source is not a matrix but the real series: element (n1, n2) of batch p is
//       v[2p L + n] + i v[(2p+1) L + n], n = n1 cols + n2 (two overlap-save blocks in one complex transform); samples
//       past the end of the series (an odd last block, the tail of the last block) read as 0.
template <bool PACK>
__global__ void __launch_bounds__(256) fb_transpose_kernel(const float2* __restrict__ in, float2* __restrict__ out,
                                                            int rows, int cols, const float* __restrict__ series,
                                                            long long n_series, long long L, long long first_block)
{
    __shared__ float2 tile[32][33];
    const size_t batch = blockIdx.z, mat = (size_t)rows * cols;
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int j = ty; j < 32; j += 8) {
        const long long n = (long long)(r0 + j) * cols + c0 + tx;
        if (PACK) {
            const long long i0 = (first_block + 2 * (long long)batch) * L + n, i1 = i0 + L;
            tile[j][tx] = make_float2(i0 < n_series ? series[i0] : 0.f, i1 < n_series ? series[i1] : 0.f);
        } else {
            tile[j][tx] = in[batch * mat + n];
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = ty; j < 32; j += 8) out[batch * mat + (size_t)(c0 + j) * rows + r0 + tx] = tile[tx][j];
}

// The last transpose of the inverse transform fused with the detection (n_int a multiple of 32): a tile row of the
// transposed result is 32 consecutive samples n of one block pair, all inside one integration group, so instead of
// writing y the warp squares and adds them: part[batch][0/1][n / 32] = sum of re^2 (block 2 batch) / im^2 (the block
// after it).  Saves the 8 B per point store and fb_detect_kernel's 8 B per point read; fb_sum_parts_kernel adds
// n_int/32 consecutive partial sums per output in a fixed order (no atomics: results are reproducible).
__global__ void __launch_bounds__(256) fb_transpose_detect_kernel(const float2* __restrict__ in, float* __restrict__ part,
                                                                  int rows, int cols)
{
    __shared__ float2 tile[32][33];
    const size_t batch = blockIdx.z, mat = (size_t)rows * cols;
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int j = ty; j < 32; j += 8) tile[j][tx] = in[batch * mat + (size_t)(r0 + j) * cols + c0 + tx];
    __syncthreads();
#pragma unroll
    for (int j = ty; j < 32; j += 8) {
        const float2 v = tile[tx][j];  // natural-order element n = (c0 + j) * rows + r0 + tx
        float a = v.x * v.x, b = v.y * v.y;
#pragma unroll
        for (int off = 16; off; off >>= 1) {
            a += __shfl_xor_sync(0xffffffffu, a, off);
            b += __shfl_xor_sync(0xffffffffu, b, off);
        }
        if (tx == 0) {
            const size_t g = ((size_t)(c0 + j) * rows + r0) >> 5;  // group of 32 samples inside the transform
            part[(2 * batch) * (mat >> 5) + g] = a;
            part[(2 * batch + 1) * (mat >> 5) + g] = b;
        }
    }
}
__global__ void fb_sum_parts_kernel(const float* __restrict__ part, long long groups_per_block, int D, int n_int,
                                    long long outs_per_block, long long first_block, long long n_blocks_total,
                                    long long n_ids, float* __restrict__ out)
{
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= n_ids) return;
    const long long lb = id / outs_per_block, j = id - lb * outs_per_block;  // lb = block index inside this batch set
    const long long block = first_block + lb;
    if (block >= n_blocks_total) return;
    const float* p = part + lb * groups_per_block + ((long long)D + j * n_int) / 32;
    float acc = 0.f;
    for (int i = 0; i < n_int / 32; ++i) acc += p[i];
    out[block * outs_per_block + j] = acc;
}

// Overlap-save discard, detect, integrate (R20): y[batch][n] complex, re = block
// first_block + 2 batch, im = the block after it; out[block L/n_int + j] = sum_{i < n_int} part(y[D + j n_int + i])^2.
// One warp per output when n_int >= 32, one thread otherwise.
__global__ void fb_detect_kernel(const float2* __restrict__ y, long long n_fft, int D, int n_int, long long outs_per_block,
                                 long long first_block, long long n_blocks_total, float* __restrict__ out)
{
    const bool by_warp = n_int >= 32;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long id = by_warp ? gid >> 5 : gid;
    const int lane = threadIdx.x & 31;
    const long long per_batch = 2 * outs_per_block;
    const long long batch = id / per_batch, rem = id - batch * per_batch;
    const int part = (int)(rem / outs_per_block);
    const long long j = rem - part * outs_per_block;
    const long long block = first_block + 2 * batch + part;
    if (block >= n_blocks_total) return;  // (uniform over a warp when by_warp)
    const float2* p = y + batch * n_fft + D + j * n_int;
    float acc = 0.f;
    if (by_warp) {
        for (int i = lane; i < n_int; i += 32) {
            const float v = part ? p[i].y : p[i].x;
            acc = fmaf(v, v, acc);
        }
        for (int off = 16; off; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
        if (lane == 0) out[block * outs_per_block + j] = acc;
    } else {
        for (int i = 0; i < n_int; ++i) {
            const float v = part ? p[i].y : p[i].x;
            acc = fmaf(v, v, acc);
        }
        out[block * outs_per_block + j] = acc;
    }
}

// Plan-time tables (fp64 phases).
__global__ void fb_twiddle_tables_kernel(float2* ta, int n_a, float2* tb, int n_b, double n_fft)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double s, c;
    if (i < n_a) {
        sincospi(-2.0 * (double)i * (double)(1 << TW_LO_BITS) / n_fft, &s, &c);
        ta[i] = make_float2((float)c, (float)s);
    }
    if (i < n_b) {
        sincospi(-2.0 * (double)i / n_fft, &s, &c);
        tb[i] = make_float2((float)c, (float)s);
    }
}
__global__ void fb_small_twiddle_kernel(float2* tw, int n)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    double s, c;
    sincospi(-2.0 * (double)m / (double)n, &s, &c);
    tw[m] = make_float2((float)c, (float)s);
}
// chirp[k1][k2] for bin k = k1 + N1 k2 (the four-step's output order), Hermitian: bins above N/2 are the conjugates of
// their mirrors; f_l = k 2B / N above the lower band edge f_lo (R21); psi = D DM f_l^2 / ((f_l + f_lo) f_lo^2) cycles;
// the filter applied is exp(-2 pi i psi) (R1), tapered, divided by N (R7)
__global__ void fb_chirp_kernel(float2* __restrict__ chirp, int n1, int n2, double bw, double f_lo, double dm, unsigned taper)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long n = (long long)n1 * n2;
    if (idx >= n) return;
    const long long k1 = idx / n2, k2 = idx - k1 * n2;
    const long long k = k1 + (long long)n1 * k2;
    const long long km = k <= n / 2 ? k : n - k;
    const double fl = (double)km * (2.0 * bw / (double)n);
    double psi = DEDISP_D_HZ2_S * dm * fl * fl / ((fl + f_lo) * f_lo * f_lo);
    psi -= floor(psi);
    double s, c;
    sincospi(2.0 * psi, &s, &c);
    double w = 1.0 / (double)n;
    if (taper == DEDISP_TAPER_HANN) {
        const double ch = cospi((fl - 0.5 * bw) / bw);
        w *= ch * ch;
    } else if (taper == DEDISP_TAPER_WELCH) {
        const double rr = 2.0 * (fl - 0.5 * bw) / bw;
        w *= 1.0 - rr * rr;
    }
    chirp[idx] = make_float2((float)(w * c), (float)((k <= n / 2 ? -1.0 : 1.0) * w * s));
}

template <int R> constexpr size_t rows_smem() { return (size_t)(fb_cta<R>() / (R / FB_E)) * padp<FShape<R>::R0>(R) * sizeof(float2); }

template <int R, int MODE> int launch_rows_r(const RowsArgs& a, cudaStream_t st)
{
    static bool attr_set[64] = {};
    int dev = 0;
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    if (dev >= 0 && dev < 64 && !attr_set[dev]) {
        DEDISP_CUDA_TRY(cudaFuncSetAttribute(fb_rows_kernel<R, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)rows_smem<R>()));
        attr_set[dev] = true;
    }
    constexpr int FB_CTA = fb_cta<R>(), UPS = FB_CTA / (R / FB_E);
    const long long grid = (a.n_rows + UPS - 1) / UPS;
    if (grid <= 0 || grid > 0x7fffffffll) return DEDISP_EINVAL;
    fb_rows_kernel<R, MODE><<<(unsigned)grid, FB_CTA, rows_smem<R>(), st>>>(a);
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}
template <int MODE> int launch_rows(int R, const RowsArgs& a, cudaStream_t st)
{
    switch (R) {
        case 1024: return launch_rows_r<1024, MODE>(a, st);
        case 2048: return launch_rows_r<2048, MODE>(a, st);
        case 4096: return launch_rows_r<4096, MODE>(a, st);
        case 8192: return launch_rows_r<8192, MODE>(a, st);
        case 16384: return launch_rows_r<16384, MODE>(a, st);
        default: return DEDISP_EINVAL;
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------------------------------------------
struct dedisp_fullband_s {
    int n_chan, n_dm, n_int, n1, n2, D, device, max_pairs;
    long long n_fft, L;
    double bw_hz, f_lo_hz;
    unsigned flags;
    float2 *d_chirp, *d_tw1, *d_tw2, *d_twg, *d_ta, *d_tb;  // chirp [n_dm][n1][n2]; twiddles of the three row lengths
    float2* d_buf[3];                                       // [max_pairs][n_fft] each
    float* d_series;                                        // real voltage series
    long long series_cap;
};

static void fb_free(dedisp_fullband_s* p)
{
    if (!p) return;
    float2* f2[] = {p->d_chirp, p->d_tw1, p->d_tw2, p->d_twg, p->d_ta, p->d_tb, p->d_buf[0], p->d_buf[1], p->d_buf[2]};
    for (float2* q : f2)
        if (q) cudaFree(q);
    if (p->d_series) cudaFree(p->d_series);
    delete p;
}

static bool fb_row_len_ok(long long r) { return r == 1024 || r == 2048 || r == 4096 || r == 8192 || r == 16384; }

extern "C" int dedisp_fullband_framing(double bw_hz, double f_lo_hz, const double* dm, int n_dm, long long n_fft, int n_int,
                                       int* D, long long* L)
{
    if (!dm || n_dm <= 0 || !(bw_hz > 0.0) || !(f_lo_hz > 0.0) || n_fft <= 0 || n_int <= 0 || !D || !L) return DEDISP_EINVAL;
    long long d = 0;
    for (int i = 0; i < n_dm; ++i) {
        if (!isfinite(dm[i])) return DEDISP_EINVAL;
        const double f_hi = f_lo_hz + bw_hz;
        const double smear = DEDISP_D_HZ2_S * fabs(dm[i]) * (1.0 / (f_lo_hz * f_lo_hz) - 1.0 / (f_hi * f_hi));
        const long long di = (long long)ceil(smear * 2.0 * bw_hz);
        if (di > d) d = di;
    }
    d = (d + n_int - 1) / n_int * n_int;  // R20
    if (d >= n_fft || (n_fft - d) % n_int || d > 0x7fffffffll) return DEDISP_EINVAL;
    *D = (int)d;
    *L = n_fft - d;
    return DEDISP_OK;
}

extern "C" int dedisp_fullband_plan(dedisp_fullband_t* out_plan, int n_chan, double bw_hz, double f_lo_hz, const double* dm,
                                    int n_dm, long long n_fft, int n_int, unsigned flags)
{
    if (!out_plan) return DEDISP_EINVAL;
    *out_plan = nullptr;
    if ((flags & ~DEDISP_TAPER_MASK) || (flags & DEDISP_TAPER_MASK) == 3u) return DEDISP_EINVAL;
    if (n_chan <= 0 || !fb_row_len_ok(2ll * n_chan)) return DEDISP_EINVAL;          // the c2r row is 2C points
    if (n_fft < (1ll << 20) || n_fft > (1ll << 28) || (n_fft & (n_fft - 1))) return DEDISP_EINVAL;
    for (int i = 0; i < n_dm; ++i)
        if (dm && dm[i] < 0.0) return DEDISP_EINVAL;  // R20's discard end holds for DM >= 0 (the delaying filter)
    int D;
    long long L;
    int rc = dedisp_fullband_framing(bw_hz, f_lo_hz, dm, n_dm, n_fft, n_int, &D, &L);
    if (rc != DEDISP_OK) return rc;
    int lg = 0;
    while ((1ll << lg) < n_fft) ++lg;
    int l1 = lg / 2;
    if (l1 < 10) l1 = 10;
    if (lg - l1 > 14) l1 = lg - 14;
    const int n1 = 1 << l1, n2 = (int)(n_fft >> l1);
    if (!fb_row_len_ok(n1) || !fb_row_len_ok(n2)) return DEDISP_EINVAL;

    int dev = 0, n_dev = 0, major = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) {
        (void)cudaGetLastError();
        return DEDISP_ENODEV;
    }
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    DEDISP_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return DEDISP_ENODEV;

    dedisp_fullband_s* p = new (std::nothrow) dedisp_fullband_s();
    if (!p) return DEDISP_ENOMEM;
    memset(p, 0, sizeof(*p));
    p->n_chan = n_chan; p->n_dm = n_dm; p->n_int = n_int; p->n1 = n1; p->n2 = n2; p->D = D; p->L = L; p->device = dev;
    p->n_fft = n_fft; p->bw_hz = bw_hz; p->f_lo_hz = f_lo_hz; p->flags = flags;
    p->max_pairs = (int)((1ll << 27) / n_fft);  // 1 GB per buffer
    if (p->max_pairs < 1) p->max_pairs = 1;
#define FB_TRY(expr)                                                                             \
    do {                                                                                         \
        cudaError_t e__ = (expr);                                                                \
        if (e__ != cudaSuccess) {                                                                \
            g_dedisp_last_cuda = (int)e__; (void)cudaGetLastError(); fb_free(p);                 \
            return e__ == cudaErrorMemoryAllocation ? DEDISP_ENOMEM : DEDISP_ECUDA;              \
        }                                                                                        \
    } while (0)
    const int n_a = (int)(n_fft >> TW_LO_BITS), n_b = 1 << TW_LO_BITS;
    FB_TRY(cudaMalloc(&p->d_chirp, sizeof(float2) * (size_t)n_dm * n_fft));
    FB_TRY(cudaMalloc(&p->d_tw1, sizeof(float2) * n1));
    FB_TRY(cudaMalloc(&p->d_tw2, sizeof(float2) * n2));
    FB_TRY(cudaMalloc(&p->d_twg, sizeof(float2) * 2 * n_chan));
    FB_TRY(cudaMalloc(&p->d_ta, sizeof(float2) * n_a));
    FB_TRY(cudaMalloc(&p->d_tb, sizeof(float2) * n_b));
    fb_small_twiddle_kernel<<<(n1 + 255) / 256, 256>>>(p->d_tw1, n1);
    fb_small_twiddle_kernel<<<(n2 + 255) / 256, 256>>>(p->d_tw2, n2);
    fb_small_twiddle_kernel<<<(2 * n_chan + 255) / 256, 256>>>(p->d_twg, 2 * n_chan);
    fb_twiddle_tables_kernel<<<((n_a > n_b ? n_a : n_b) + 255) / 256, 256>>>(p->d_ta, n_a, p->d_tb, n_b, (double)n_fft);
    for (int d = 0; d < n_dm; ++d)
        fb_chirp_kernel<<<(unsigned)((n_fft + 255) / 256), 256>>>(p->d_chirp + (size_t)d * n_fft, n1, n2, bw_hz, f_lo_hz,
                                                                   dm[d], flags & DEDISP_TAPER_MASK);
    FB_TRY(cudaGetLastError());
    FB_TRY(cudaDeviceSynchronize());
    *out_plan = p;
    return DEDISP_OK;
}

extern "C" int dedisp_fullband_get_framing(dedisp_fullband_t p, int* D, long long* L, int* n1, int* n2)
{
    if (!p) return DEDISP_EINVAL;
    if (D) *D = p->D;
    if (L) *L = p->L;
    if (n1) *n1 = p->n1;
    if (n2) *n2 = p->n2;
    return DEDISP_OK;
}

static long long fb_n_blocks(const dedisp_fullband_s* p, long long n_spec)
{
    const long long n_v = n_spec * 2 * p->n_chan;
    return n_v < p->n_fft ? 0 : (n_v - p->D) / p->L;
}

extern "C" long long dedisp_fullband_out_samples(dedisp_fullband_t p, long long n_spec)
{
    if (!p || n_spec <= 0) return 0;
    return fb_n_blocks(p, n_spec) * (p->L / p->n_int);
}

static int fb_reserve(dedisp_fullband_s* p, long long n_v, long long pairs)
{
    if (p->series_cap < n_v) {
        if (p->d_series) { cudaFree(p->d_series); p->d_series = nullptr; p->series_cap = 0; }
        DEDISP_CUDA_TRY(cudaMalloc(&p->d_series, sizeof(float) * (size_t)n_v));
        p->series_cap = n_v;
    }
    if (!p->d_buf[0]) {
        (void)pairs;
        for (int i = 0; i < 3; ++i)
            DEDISP_CUDA_TRY(cudaMalloc(&p->d_buf[i], sizeof(float2) * (size_t)p->max_pairs * p->n_fft));
    }
    return DEDISP_OK;
}

static int fb_series(dedisp_fullband_s* p, const int8_t* d_spec, long long n_spec, cudaStream_t st)
{
    RowsArgs a{};
    a.gsb = d_spec; a.series = p->d_series; a.tw = p->d_twg; a.n_rows = n_spec; a.rows_per_batch = 1;
    a.gsb_scale = 1.0f / (2.0f * p->n_chan);
    return launch_rows<ROWS_GSB>(2 * p->n_chan, a, st);
}

extern "C" int dedisp_fullband_debug_series(dedisp_fullband_t p, const int8_t* d_spec, long long n_spec, float* d_series,
                                            void* cuda_stream)
{
    if (!p || !d_spec || !d_series || n_spec <= 0) return DEDISP_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = fb_reserve(p, n_spec * 2 * p->n_chan, 1);
    if (rc != DEDISP_OK) return rc;
    if ((rc = fb_series(p, d_spec, n_spec, st)) != DEDISP_OK) return rc;
    DEDISP_CUDA_TRY(cudaMemcpyAsync(d_series, p->d_series, sizeof(float) * (size_t)n_spec * 2 * p->n_chan,
                                    cudaMemcpyDeviceToDevice, st));
    return DEDISP_OK;
}

extern "C" int dedisp_fullband_execute(dedisp_fullband_t p, const int8_t* d_spec, long long n_spec, float* d_out,
                                       long long out_stride, void* cuda_stream)
{
    if (!p || !d_spec || !d_out || n_spec <= 0) return DEDISP_EINVAL;
    int dev = -1;
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != p->device) return DEDISP_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long n_v = n_spec * 2 * p->n_chan, nb = fb_n_blocks(p, n_spec), opb = p->L / p->n_int;
    if (nb <= 0) return DEDISP_ESHORT;
    if (out_stride < nb * opb) return DEDISP_EINVAL;
    int rc = fb_reserve(p, n_v, (nb + 1) / 2);
    if (rc != DEDISP_OK) return rc;
    if ((rc = fb_series(p, d_spec, n_spec, st)) != DEDISP_OK) return rc;  // step 1
    const int n1 = p->n1, n2 = p->n2;
    const long long pairs = (nb + 1) / 2;
    for (long long p0 = 0; p0 < pairs; p0 += p->max_pairs) {
        const int pb = (int)(pairs - p0 < p->max_pairs ? pairs - p0 : p->max_pairs);
        float2 *A = p->d_buf[0], *B = p->d_buf[1], *Cc = p->d_buf[2];
        // pack two blocks per transform and turn [n1][n2] -> [n2][n1]
        fb_transpose_kernel<true><<<dim3(n2 / 32, n1 / 32, pb), 256, 0, st>>>(nullptr, A, n1, n2, p->d_series, n_v, p->L,
                                                                              2 * p0);
        RowsArgs a{};
        a.ta = p->d_ta; a.tb = p->d_tb; a.n_mask = (unsigned)(p->n_fft - 1);
        // four-step, steps 1-2: n2 column transforms of length n1, twiddle W_N^{n2 k1}
        a.in = A; a.out = B; a.tw = p->d_tw1; a.n_rows = (long long)pb * n2; a.rows_per_batch = n2;
        if ((rc = launch_rows<ROWS_FWD_TWIDDLE>(n1, a, st)) != DEDISP_OK) return rc;
        fb_transpose_kernel<false><<<dim3(n1 / 32, n2 / 32, pb), 256, 0, st>>>(B, A, n2, n1, nullptr, 0, 0, 0);  // -> [k1][n2]
        for (int d = 0; d < p->n_dm; ++d) {
            // step 3, chirp (Eq. 3), step 3': rows k1 of length n2, the spectrum stays in registers
            a.in = A; a.out = B; a.tw = p->d_tw2; a.n_rows = (long long)pb * n1; a.rows_per_batch = n1;
            a.chirp = p->d_chirp + (size_t)d * p->n_fft;
            if ((rc = launch_rows<ROWS_CHIRP>(n2, a, st)) != DEDISP_OK) return rc;
            fb_transpose_kernel<false><<<dim3(n2 / 32, n1 / 32, pb), 256, 0, st>>>(B, Cc, n1, n2, nullptr, 0, 0, 0);  // -> [n2][k1]
            // steps 2'-1': conjugate twiddle, inverse transforms of length n1
            a.in = Cc; a.out = B; a.tw = p->d_tw1; a.n_rows = (long long)pb * n2; a.rows_per_batch = n2;
            if ((rc = launch_rows<ROWS_TWIDDLE_INV>(n1, a, st)) != DEDISP_OK) return rc;
            // back to natural order + overlap-save discard, detect, integrate
            if (p->n_int % 32 == 0) {
                float* part = reinterpret_cast<float*>(Cc);  // [pb][2][n_fft / 32]
                fb_transpose_detect_kernel<<<dim3(n1 / 32, n2 / 32, pb), 256, 0, st>>>(B, part, n2, n1);
                const long long ids = (long long)pb * 2 * opb;
                fb_sum_parts_kernel<<<(unsigned)((ids + 255) / 256), 256, 0, st>>>(part, p->n_fft / 32, p->D, p->n_int, opb,
                                                                                   2 * p0, nb, ids,
                                                                                   d_out + (size_t)d * out_stride);
            } else {
                fb_transpose_kernel<false><<<dim3(n1 / 32, n2 / 32, pb), 256, 0, st>>>(B, Cc, n2, n1, nullptr, 0, 0, 0);
                const long long ids = (long long)pb * 2 * opb * (p->n_int >= 32 ? 32 : 1);
                fb_detect_kernel<<<(unsigned)((ids + 255) / 256), 256, 0, st>>>(Cc, p->n_fft, p->D, p->n_int, opb, 2 * p0,
                                                                                nb, d_out + (size_t)d * out_stride);
            }
        }
    }
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}

extern "C" int dedisp_fullband_destroy(dedisp_fullband_t p)
{
    if (!p) return DEDISP_EINVAL;
    fb_free(p);
    return DEDISP_OK;
}
