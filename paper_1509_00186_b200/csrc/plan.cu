// plan.cu -- host side of libdedisp: validation, overlap-save framing (R9), plan-time tables, execute, debug hooks.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "dedisp_internal.h"

thread_local int g_dedisp_last_cuda = 0;

// ---------------------------------------------------------------------------------------------------------------
// Frequencies (R3, R5) -- host and device versions of the same two lines
// ---------------------------------------------------------------------------------------------------------------
__host__ __device__ static inline double chan_center_hz(double f_center_hz, double bw_hz, int n_chan, int c)
{
    // channels tile [F - B/2, F + B/2) ascending (R3)
    return f_center_hz - 0.5 * bw_hz + ((double)c + 0.5) * (bw_hz / (double)n_chan);
}

// ---------------------------------------------------------------------------------------------------------------
// Framing (R9): discard = impulse-response length = dispersion time in the band
// ---------------------------------------------------------------------------------------------------------------
static long long round_up(long long x, long long m) { return (x + m - 1) / m * m; }
static long long gcd(long long a, long long b) { return b ? gcd(b, a % b) : a; }
static long long max_ll(long long a, long long b) { return a > b ? a : b; }

int dedisp_framing_impl(int n_chan, double bw, double F, const double* dm, int n_dm, int n_fft, int n_int, int* head,
                        int* tail, int* L, double* max_smear)
{
    if (n_chan <= 0 || n_dm <= 0 || n_fft <= 0 || n_int <= 0 || !dm || !(bw > 0.0) || !(F - 0.5 * bw > 0.0))
        return DEDISP_EINVAL;
    const double dv = bw / n_chan;
    long long need_past = 0, need_future = 0;
    double smear = 0.0;
    // the delays fall with frequency, so channel 0 is the worst case; the loop over all channels costs nothing
    for (int c = 0; c < n_chan; ++c) {
        const double fc = chan_center_hz(F, bw, n_chan, c);
        const double inv_lo = 1.0 / ((fc - 0.5 * dv) * (fc - 0.5 * dv));
        const double inv_c = 1.0 / (fc * fc);
        const double inv_hi = 1.0 / ((fc + 0.5 * dv) * (fc + 0.5 * dv));
        for (int d = 0; d < n_dm; ++d) {
            if (!isfinite(dm[d])) return DEDISP_EINVAL;
            const double k = DEDISP_D_HZ2_S * fabs(dm[d]) * dv;        // seconds -> samples
            // the ISM makes the low edge lag the channel centre and the high edge lead it (delay law P:L39-41); the
            // correction (R1: the inverse of Eq. 3) holds the high edge back -- an output sample needs that much PAST
            // input -- and pulls the low edge forward -- FUTURE input; a negative DM swaps the two
            const long long n_low = (long long)ceil(k * (inv_lo - inv_c));
            const long long n_high = (long long)ceil(k * (inv_c - inv_hi));
            const bool pos = dm[d] >= 0.0;
            need_past = max_ll(need_past, pos ? n_high : n_low);
            need_future = max_ll(need_future, pos ? n_low : n_high);
            smear = fmax(smear, k * (inv_lo - inv_hi));
        }
    }
    const long long h = round_up(need_past, n_int);
    const long long dtot = round_up(h + need_future, 32 / gcd(32, n_int) * (long long)n_int);
    const long long len = (long long)n_fft - dtot;
    if (max_smear) *max_smear = smear;
    if (len <= 0 || len % n_int != 0) return DEDISP_EINVAL;
    *head = (int)h;
    *tail = (int)(dtot - h);
    *L = (int)len;
    return DEDISP_OK;
}

extern "C" int dedisp_framing(int n_chan, double bw_hz, double f_center_hz, const double* dm, int n_dm, int n_fft,
                              int n_int, int* head, int* tail, int* L)
{
    if (!head || !tail || !L) return DEDISP_EINVAL;
    return dedisp_framing_impl(n_chan, bw_hz, f_center_hz, dm, n_dm, n_fft, n_int, head, tail, L, nullptr);
}

// ---------------------------------------------------------------------------------------------------------------
// Plan-time tables, generated on the device with the phase in fp64
// ---------------------------------------------------------------------------------------------------------------
// chirp[d][c][k] = w(f_k) * exp(-2 pi i psi) / N,  psi = D DM f^2 / ((f + f_c) f_c^2) cycles: the inverse of
// the ISM's in-band term, which Eq. 3 prints as exp(+2 pi i psi); R1, R2
// (bw, F, n_chan_total describe the WHOLE band; the table holds channels chan0 .. chan0 + n_chan - 1 of it)
__global__ void chirp_table_kernel(float2* __restrict__ chirp, const double* __restrict__ dm, int n_chan, int n_fft,
                                   double bw, double F, int n_chan_total, int chan0, unsigned taper)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y, d = blockIdx.z;
    if (k >= n_fft) return;
    const double dv = bw / (double)n_chan_total;
    const double fc = chan_center_hz(F, bw, n_chan_total, chan0 + c);
    const int ks = (k < n_fft / 2) ? k : k - n_fft;  // bin N/2 is -dv/2 (R5)
    const double f = (double)ks * dv / (double)n_fft;
    double psi = DEDISP_D_HZ2_S * dm[d] * f * f / ((f + fc) * fc * fc);
    psi -= floor(psi);  // whole cycles carry no information; keeps the trig argument in [0, 2)
    double s, co;
    sincospi(2.0 * psi, &s, &co);
    double w = 1.0 / (double)n_fft;  // 1/N of the inverse transform (R7) folded in: exact, N is a power of two
    if (taper == DEDISP_TAPER_HANN) {
        const double ch = cospi(f / dv);
        w *= ch * ch;
    } else if (taper == DEDISP_TAPER_WELCH) {
        const double r = 2.0 * f / dv;
        w *= 1.0 - r * r;
    }
    chirp[((size_t)d * n_chan + c) * n_fft + k] = make_float2((float)(w * co), (float)(-(w * s)));
}

__global__ void twiddle_table_kernel(float2* __restrict__ tw, int n_fft)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n_fft) return;
    double s, co;
    sincospi(-2.0 * (double)m / (double)n_fft, &s, &co);
    tw[m] = make_float2((float)co, (float)s);
}

int dedisp_launch_chirp_table(const dedisp_plan_s* p, const double* d_dm, cudaStream_t st)
{
    dim3 grid((p->n_fft + 255) / 256, p->n_chan, p->n_dm);
    chirp_table_kernel<<<grid, 256, 0, st>>>(p->d_chirp, d_dm, p->n_chan, p->n_fft, p->bw_total_hz, p->f_center_total_hz,
                                             p->n_chan_total, p->chan0, p->flags & DEDISP_TAPER_MASK);
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}

int dedisp_launch_twiddle_table(const dedisp_plan_s* p, cudaStream_t st)
{
    twiddle_table_kernel<<<(p->n_fft + 255) / 256, 256, 0, st>>>(p->d_twiddle, p->n_fft);
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}
