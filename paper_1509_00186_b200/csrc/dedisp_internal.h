// Internal definitions shared by the translation units of libdedisp (product code; nothing here is used by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "dedisp.h"

// Dispersion constant of P:L117 ("4.148808 x 10^9" in MHz / us units) in Hz^2 s per pc cm^-3 (R8).
#define DEDISP_D_HZ2_S 4.148808e15

struct dedisp_stream_state;

struct dedisp_plan_s {
    // problem statement (observing frequency, bandwidth, DM) + channelisation and transform sizes
    int n_chan, n_dm, n_fft, n_int;
    double bw_hz, f_center_hz;  // of THIS plan's channels (a shard: its sub-band)
    // the whole band this plan's channels are cut from (dedisp_plan_shard; equal to the above for dedisp_plan): the
    // chirp and the band-alignment shifts are computed from these, so a shard's values are bit-identical to the whole plan's
    int n_chan_total, chan0;
    double bw_total_hz, f_center_total_hz;
    int in_pitch;               // channels per row of the caller's input: n_chan, or n_chan_total (DEDISP_SHARD_FULL_INPUT)
    long long time_offset;      // output samples by which this plan's time axis is ahead of the whole band's framing
    double* dm;  // host copy [n_dm]
    unsigned flags;
    // framing (R9)
    int head, tail, L;
    double max_smear_samples;
    int nfft_rule;
    int device;
    // device tables owned by the plan
    float2* d_chirp;    // [n_dm][n_chan][n_fft], taper * exp(+2 pi i psi) / n_fft
    float2* d_twiddle;  // [n_fft], exp(-2 pi i m / n_fft)
    // channel-major int8 scratch: [n_chan][xt_stride] (re,im) pairs, xt_stride samples per row
    float2* d_spec;     // [resident CTAs][units per CTA][n_fft] forward-spectrum stash shared by the trial DMs (n_dm > 1)
    int8_t* d_xt;
    long long xt_cap_samp;  // samples per row the scratch can hold
    // band alignment (R16): whole-output-sample delay of every channel, host and device copies [n_dm][n_chan]
    long long* band_shift;
    int* d_band_shift;
    long long band_max_shift;
    dedisp_stream_state* stream;
    // kernel timing (dedisp_profile_enable): 3 events per call -- before corner turn, between, after fused
    int prof_on, prof_n;
    cudaEvent_t* prof_ev;  // [DEDISP_PROF_MAX][3], created on first enable
};
#define DEDISP_PROF_MAX 256

extern thread_local int g_dedisp_last_cuda;

#define DEDISP_CUDA_TRY(expr)                     \
    do {                                          \
        cudaError_t e__ = (expr);                 \
        if (e__ != cudaSuccess) {                 \
            g_dedisp_last_cuda = (int)e__;        \
            (void)cudaGetLastError();             \
            return e__ == cudaErrorMemoryAllocation ? DEDISP_ENOMEM : DEDISP_ECUDA; \
        }                                         \
    } while (0)

// row stride (in samples) of the channel-major scratch for a call of n_samp samples: multiple of 64 samples
// (= 128 B) so every block start b*L (L % 32 == 0) stays 64 B aligned for vector / bulk loads.
static inline long long dedisp_xt_stride(long long n_samp) { return (n_samp + 63) / 64 * 64; }

// corner_turn.cu (all launchers enqueue only)
// corner turn: int8 [n_samp][n_chan][2] -> int8 [n_chan][xt_stride][2], rows t0_dst.. of the destination
// (columns chan0 .. chan0 + n_chan - 1 of rows that are in_pitch channels wide)
int dedisp_launch_corner_turn(const int8_t* d_in, long long n_samp, int n_chan, int in_pitch, int chan0, int8_t* d_xt,
                              long long xt_stride, long long dst_t0, cudaStream_t st);
// fused_aos.cu: fused unpack -> forward FFT -> chirp -> inverse FFT -> discard -> detect -> integrate over nb blocks of
// every channel (all enqueue only):  out[d][c][out_col0 + b*L/n_int + j]
// accumulate != 0: add to d_out instead of overwriting it
int dedisp_launch_aos(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, long long nb, float* d_out,
                      long long out_stride, long long out_col0, int accumulate, cudaStream_t st);
// debug: dump_unpack = 0 -> [n_dm][L] dedispersed voltages of (chan, block); 1 -> the [N] values the fused kernel holds
// in registers right after its own int8 -> fp32 conversion
int dedisp_launch_aos_debug_voltage(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, int chan,
                                    long long block, float* d_volt, int dump_unpack, cudaStream_t st);
int dedisp_aos_supported(int n_fft);
size_t dedisp_aos_spec_bytes(int n_fft);  // valid after dedisp_aos_init()
int dedisp_aos_init(void);                // sets the dynamic shared memory attributes once per process
// plan-time table generation on the device (fp64 phase)
int dedisp_launch_chirp_table(const dedisp_plan_s* p, const double* d_dm, cudaStream_t st);
int dedisp_launch_twiddle_table(const dedisp_plan_s* p, cudaStream_t st);
// framing (R9) with the largest in-band smear (samples) reported as well
int dedisp_framing_impl(int n_chan, double bw, double F, const double* dm, int n_dm, int n_fft, int n_int, int* head,
                        int* tail, int* L, double* max_smear);
// api.cu: corner turn + fused kernel on `st` with the optional profiling events around them
int dedisp_enqueue_chunk(dedisp_plan_s* p, const int8_t* d_in, long long n_rows, int8_t* d_xt, long long xt_stride,
                         long long dst_t0, long long nb, float* d_out, long long out_stride, cudaStream_t st,
                         cudaEvent_t after_corner_turn, int accumulate = 0);
long long dedisp_n_blocks(const dedisp_plan_s* p, long long n_samp);
// band_sum.cu
int dedisp_launch_band_sum(const dedisp_plan_s* p, const float* d_out, long long out_stride, float* d_series,
                           long long series_stride, long long n_series, cudaStream_t st);
int dedisp_launch_fold(const float* d_series, long long n, double t0, double dt, double period, int n_bins,
                       float* d_sum, unsigned int* d_count, cudaStream_t st);
// stream.cu
void dedisp_stream_free(dedisp_plan_s* p);
