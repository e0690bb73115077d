/*
 * dedisp.h -- C ABI of libdedisp: channelised overlap-save coherent dedispersion on one B200 (sm_100a).
 *
 * The operation is the data-parallel hot path of De & Gupta, "A Real-time Coherent Dedispersion Pipeline
 * for the GMRT" (arXiv:1509.00186).  Citations "P:L<n>" are line numbers of the paper text;
 * "R<n>" are the readings listed in DESIGN.md where the paper is silent or ambiguous.
 *
 * What one dedisp_execute() call computes, for every frequency channel c, overlap-save block b and trial DM d
 * (stage order of P:L139-145 Fig. 4):
 *   1. unpack   x[n] = (float)in[b*L+n][c].re + i*(float)in[b*L+n][c].im,  n in [0,N)      (R10)
 *   2. forward  S[k] = sum_n x[n] exp(-2*pi*i*k*n/N)
 *   3. chirp    Y[k] = S[k] * w(f_k) * exp(-2*pi*i*psi),  psi = D*DM_d*f_k^2/(f_c^2*(f_c+f_k)):  the INVERSE
 *               of the ISM's in-band term, which Eq. 3 prints as exp(+2*pi*i*psi); taper w; R1.
 *               D = 4.148808e15 Hz^2 s / (pc cm^-3), f_c = F - B/2 + (c+1/2)*B/C,
 *               f_k = k*dv/N (k < N/2) or (k-N)*dv/N, dv = B/C; baseband frequency rises with sky frequency.
 *               DM_d > 0 removes the dispersion of a pulsar at that DM; DM_d < 0 applies Eq. 3 itself.
 *   4. inverse  y[n] = (1/N) sum_k Y[k] exp(+2*pi*i*k*n/N)                                    (R7)
 *   5. discard  keep n in [head, head+L), L = N - head - tail                                (R9)
 *   6. detect + integrate  out[d][c][b*L/n_int + j] = sum_{i<n_int} |y[head + j*n_int + i]|^2 (R11)
 *
 * Pointers: every pointer argument says HOST or DEVICE.  The library never takes ownership of caller buffers.
 * Errors:   every call returns DEDISP_OK (0) or a negative DEDISP_E* code; no exceptions, no aborts, no output.
 * Threads:  a plan may be used from one host thread at a time, and its calls must be ordered on ONE stream at a time
 *           (a plan owns scratch buffers that its kernels share; two executes of one plan on two streams would race).
 *           Plans are independent of each other.
 * Devices:  a plan belongs to the device that was current in dedisp_plan(); every later call on it must be made with
 *           that device current (else DEDISP_EINVAL).  Several devices may be used from one process.
 */
#ifndef DEDISP_H
#define DEDISP_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dedisp_plan_s* dedisp_plan_t; /* opaque, owned by the library */

enum {
    DEDISP_OK = 0,
    DEDISP_EINVAL = -1, /* bad argument (see each call) */
    DEDISP_ENOMEM = -2, /* host or device allocation failed */
    DEDISP_ECUDA = -3,  /* a CUDA call failed; dedisp_last_cuda_error() gives the cudaError_t */
    DEDISP_ESHORT = -4, /* n_samp shorter than one block (n_fft samples) */
    DEDISP_ENODEV = -5, /* no sm_100 device / no CUDA driver */
    DEDISP_ETOOBIG = -6 /* dedisp_execute_static: the call needs more than DEDISP_STATIC_SCRATCH_BYTES of scratch */
};

/* flags of dedisp_plan(): taper of the chirp function (P:L123 names Hanning and Welch; R6 gives the formulas) */
enum {
    DEDISP_TAPER_NONE = 0u,  /* w = 1 (default) */
    DEDISP_TAPER_HANN = 1u,  /* w = cos^2(pi f/dv) */
    DEDISP_TAPER_WELCH = 2u, /* w = 1 - (2f/dv)^2 */
    DEDISP_TAPER_MASK = 3u
};

typedef struct {
    int n_chan, n_dm, n_fft, n_int; /* echo of the arguments */
    int head, tail, L;              /* overlap-save framing in use (R9): block b reads rows b*L .. b*L+N-1 */
    double chan_width_hz;           /* dv = bw / n_chan = complex sample rate of one channel */
    double max_smear_samples;       /* largest in-band dispersion time over channels and DMs, in samples */
    int nfft_rule;                  /* smallest power of 2 > 2*max_smear_samples (advisory) */
} dedisp_info_t;

/*
 * Overlap-save framing (pure host arithmetic, no GPU needed).  P:L121/L145: the number of samples to discard is the
 * impulse-response length = dispersion time in the band.  R9: with the channel-centre reference the applied filter
 * (DM > 0) holds the high band edge back by n_high samples (an output needs that much PAST input: `head`) and pulls
 * the low edge forward by n_low samples (FUTURE input: `tail`); one framing for all channels and DMs:
 * head = roundup(n_high, n_int), head+tail = roundup(head+n_low, lcm(32,n_int)).
 *   dm: HOST array [n_dm], pc cm^-3, negative allowed (conjugate chirp; head/tail roles swap).
 * Returns DEDISP_EINVAL if an argument is non-positive, F - B/2 <= 0, head+tail >= n_fft or L % n_int != 0.
 */
int dedisp_framing(int n_chan, double bw_hz, double f_center_hz, const double* dm, int n_dm, int n_fft, int n_int,
                   int* head, int* tail, int* L);

/*
 * Create a plan on the current CUDA device: validates, computes the framing, builds the chirp table
 * float2 [n_dm][n_chan][n_fft] (phase in fp64, value rounded to fp32, pre-scaled by 1/n_fft) and the FFT twiddles.
 *   n_fft: one of 1024, 2048, 4096, 8192, 16384 (the built kernel sizes).  dm: HOST array, copied.
 *   n_int: a power of two (R9 makes the overlap a multiple of n_int, so L % n_int == n_fft % n_int).
 * Synchronises the device once.  Errors: EINVAL, ENOMEM, ECUDA, ENODEV.
 */
int dedisp_plan(dedisp_plan_t* out_plan, int n_chan, double bw_hz, double f_center_hz, const double* dm, int n_dm,
                int n_fft, int n_int, unsigned flags);

/*
 * A plan for channels chan0 .. chan0 + n_chan - 1 of a band of n_chan_total channels (bw_hz_total, f_center_hz_total):
 * the unit of the two ways the path is partitioned over channels.  Every (channel, block) is independent, so there is
 * no exchange between shards.
 *   (a) channel-range shards on several GPUs (the paper splits the two polarisations over two hosts the
 *       same way): shard_flags = 0.  The shard uses the framing of the WHOLE band, so all shards share
 *       head/tail/L and one time axis; its chirp factors and band-alignment shifts are bit-identical to the matching
 *       rows of dedisp_plan() on the whole band.  Input: the shard's own columns, int8 [n_samp][n_chan][2].
 *   (b) per-channel-group framing on one GPU (the length to discard is the
 *       dispersion time in the band, which falls as f^-3 across a wide band): DEDISP_SHARD_OWN_FRAMING computes
 *       head/tail/L from the group's own sub-band (R18), so high-frequency groups keep more of every transform.  The
 *       group's outputs start dedisp_shard_time_offset() = (head_whole - head_group)/n_int output samples EARLIER than
 *       the whole band's: out_whole_axis[j] = out_group[j + offset].  dedisp_band_shifts() already contains the offset.
 *   DEDISP_SHARD_FULL_INPUT: d_in of dedisp_execute() is the whole band, int8 [n_samp][n_chan_total][2], and the plan
 *       reads its own columns (groups on one GPU); dedisp_stream_* is not available for such plans (EINVAL).
 * Output layout and all other calls are those of a plan with n_chan channels.  Errors as dedisp_plan, plus EINVAL for a
 * channel range outside the band.
 */
enum { DEDISP_SHARD_FULL_INPUT = 1u, DEDISP_SHARD_OWN_FRAMING = 2u };
int dedisp_plan_shard(dedisp_plan_t* out_plan, int n_chan_total, double bw_hz_total, double f_center_hz_total,
                      const double* dm, int n_dm, int n_fft, int n_int, unsigned flags, int chan0, int n_chan,
                      unsigned shard_flags);
long long dedisp_shard_time_offset(dedisp_plan_t plan); /* 0 for dedisp_plan() and for shards with the band's framing */

int dedisp_get_info(dedisp_plan_t plan, dedisp_info_t* info);

/*
 * dedisp_execute() for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): same arguments, same kernels, same outputs, but the channel-major int8 scratch
 * [n_chan][stride][2] that dedisp_execute() allocates on demand is a static device array of
 * DEDISP_STATIC_SCRATCH_BYTES here (held by every GPU that loads the library until the process exits).  The call makes
 * no cudaMalloc / cudaFree / allocating library call.
 *   Limit: 2 * n_chan * roundup(nb*L + head + tail, 64) <= DEDISP_STATIC_SCRATCH_BYTES, else DEDISP_ETOOBIG (64 MiB holds
 *   a 1 s chunk of the 32 MHz / 512-channel mode).  Feed longer inputs in pieces that overlap by head + tail samples.
 *   All plans and all calls share the array and it keeps the last call's contents (nothing in it needs to start at zero: a
 *   call reads only what its own corner turn wrote); calls that overlap on the GPU -- two streams, or two host threads
 *   -- RACE on it: order them on one stream.  The array's device address is looked up once per device, at the first
 *   call with that device current.
 */
#define DEDISP_STATIC_SCRATCH_BYTES (64u << 20)
int dedisp_execute_static(dedisp_plan_t plan, const int8_t* d_in, long long n_samp, float* d_out, long long out_stride,
                          void* cuda_stream);

/* Outputs per (dm, channel) of a one-shot call on n_samp samples per channel: nb*L/n_int with
 * nb = floor((n_samp - head - tail)/L) (R12: no zero padding, trailing partial block dropped); 0 if too short. */
long long dedisp_out_samples(dedisp_plan_t plan, long long n_samp);

/* Pre-size the plan's device scratch (the channel-major int8 copy of the input) for calls of up to n_samp samples,
 * so that dedisp_execute never allocates.  Synchronises the device if it has to grow. */
int dedisp_reserve(dedisp_plan_t plan, long long n_samp);

/*
 * Enqueue steps 1-6 on `cuda_stream` (a cudaStream_t; NULL = legacy default stream).  Never synchronises unless the
 * scratch has to grow (see dedisp_reserve).  Results are valid once the caller has synchronised the stream.
 *   d_in   DEVICE, int8 [n_samp][n_chan][2] time-major, re then im (R10); 2-byte aligned; read only.
 *   d_out  DEVICE, float [n_dm][n_chan][out_stride]; the first dedisp_out_samples() entries of each row are written.
 * Errors: EINVAL (null pointer, out_stride too small), ESHORT, ENOMEM, ECUDA.
 */
int dedisp_execute(dedisp_plan_t plan, const int8_t* d_in, long long n_samp, float* d_out, long long out_stride,
                   void* cuda_stream);

/*
 * Second polarisation.  P:L258: the two polarisations of the beam are dedispersed separately "to
 * allow one to combine the signals from the two polarisations after detection".  Same as dedisp_execute, but the
 * integrated intensities are ADDED to what d_out already holds (stream order: after an earlier dedisp_execute on the
 * same stream for the first polarisation), so that d_out ends up as the total intensity |v_1|^2 + |v_2|^2.
 */
int dedisp_execute_add(dedisp_plan_t plan, const int8_t* d_in, long long n_samp, float* d_out, long long out_stride,
                       void* cuda_stream);

/*
 * Streaming form (host->device copy, compute and device->host copy overlapped on three streams; P:L270:
 * the samples lost at a block edge are prefixed to the next block).  Push consecutive chunks of the same observation;
 * the plan keeps the unconsumed tail on the device so that the concatenated output equals a one-shot call on the
 * concatenated input (R12).
 *   h_in   HOST (pinned for overlap), int8 [n_samp][n_chan][2], n_samp <= max_chunk_samp of dedisp_stream_begin.
 *   h_out  HOST (pinned), float [n_dm][n_chan][out_stride]: receives the outputs completed by THIS chunk in columns
 *          [0, *n_out); *n_out is known when the call returns (host arithmetic), out_stride >= *n_out.
 * The call enqueues the chunk's H2D copy, kernels and D2H copy on the plan's three streams and returns.  Buffer
 * hand-back: h_in may be reused once the NEXT push (or dedisp_stream_sync) has returned; h_out holds its values once
 * the SECOND-NEXT push (or dedisp_stream_sync) has returned.  dedisp_stream_begin allocates the device double buffers
 * (2 staging chunks, 2 channel-major carries+chunks, 2 output blocks) and resets the carry; dedisp_stream_end frees
 * them.  Errors: EINVAL (no begin, chunk too long, null pointers, out_stride too small), ENOMEM, ECUDA.
 */
int dedisp_stream_begin(dedisp_plan_t plan, long long max_chunk_samp);
int dedisp_stream_push(dedisp_plan_t plan, const int8_t* h_in, long long n_samp, float* h_out, long long out_stride,
                       long long* n_out);
int dedisp_stream_sync(dedisp_plan_t plan);
int dedisp_stream_end(dedisp_plan_t plan);

/*
 * Kernel timing for the roofline report: while enabled, every dedisp_execute / dedisp_stream_push records CUDA events
 * on its compute stream around the corner-turn and the fused kernel (up to 256 calls are kept).  dedisp_profile_read
 * synchronises those events, returns the summed device times in milliseconds and the number of calls, and clears them.
 */
int dedisp_profile_enable(dedisp_plan_t plan, int on);
int dedisp_profile_read(dedisp_plan_t plan, double* ms_corner_turn, double* ms_fused, int* n_calls);

/*
 * Alignment of the coherently dedispersed sub-bands in time and band sum ("Appropriate time delays are then
 * applied to align the pulses in the separate frequency channels, which are then added to produce a dedispersed time
 * series"; "coherently dedispersing each sub-band, followed by alignment of the individual sub-bands in time").
 * Reading R16: channel c is late against the highest channel by D*DM_d*(1/f_c^2 - 1/f_top^2) seconds; in
 * whole output samples  shift(d,c) = lround(delay*dv/n_int) - min over c  (>= 0; negative DMs work too), and
 *     series[d][j] = sum_c out[d][c][j + shift(d,c)],   j in [0, n_out - max shift over all d, c).
 *   dedisp_band_samples  series length for n_out output samples per (dm, channel); 0 if n_out <= the largest shift.
 *   dedisp_band_shifts   HOST int64 [n_chan]: shift(d, .).
 *   dedisp_band_sum      d_out DEVICE float [n_dm][n_chan][out_stride] (as written by dedisp_execute), first n_out
 *                        columns valid; d_series DEVICE float [n_dm][series_stride], series_stride >= the series
 *                        length.  Enqueues one kernel on cuda_stream.  Errors: EINVAL, ESHORT (n_out too short), ECUDA.
 */
long long dedisp_band_samples(dedisp_plan_t plan, long long n_out);
int dedisp_band_shifts(dedisp_plan_t plan, int d, long long* h_shift);
int dedisp_band_sum(dedisp_plan_t plan, const float* d_out, long long out_stride, long long n_out, float* d_series,
                    long long series_stride, void* cuda_stream);

/*
 * Folding a dedispersed time series into a pulse profile (every result figure of the paper is one: Figs. 1, 8, 13, 14,
 * P:L59; the method is not described - reading R17): sample j, taken at t0_s + j*dt_s, goes
 * to phase bin floor(frac(t/period_s) * n_bins) (decided in fp64); a bin holds the SUM of its samples and their count.
 *   d_series DEVICE float [n];  d_sum DEVICE float [n_bins] and d_count DEVICE unsigned [n_bins]: both zeroed by
 *   the call, then filled (floating-point sums in an unspecified order).  1 <= n_bins <= 4096.  No plan needed.
 */
int dedisp_fold(const float* d_series, long long n, double t0_s, double dt_s, double period_s, int n_bins, float* d_sum,
                unsigned int* d_count, void* cuda_stream);

/*
 * FP32 issue-rate micro-benchmark of the packed f32x2 instruction forms the fused kernel is built from (measurement
 * support for the "alu" roofline of DESIGN.md section 6; `python bench.py --ubench fp32-issue`).  Runs one persistent
 * 1024-thread CTA per SM (64 registers per thread, 8 warps per SM sub-partition, 8 independent complex pairs per
 * thread) for `iters` iterations of radix-2 butterfly form `form` and returns the SM sub-partition cycles per
 * butterfly (clock64, mean over SMs) and the CUDA-event time of the launch.  Forms: 0 plain (2 FADD2); 1 with +-i
 * (2 FADD2, lane-swapped operand); 2 general twiddle, conventional (FMUL2 + FFMA2 + 2 FADD2); 3 general twiddle
 * folded into the butterfly (3 FFMA2, v = 2a - u); 4 form 3 with the twiddle rotated by i; 5 folded without the
 * 2a - u step (4 FFMA2); 6 form 3 with an immediate twiddle; 7 form 2 with an immediate twiddle.
 * Allocates and frees its own small device buffers; synchronises the device.  Errors: EINVAL, ENOMEM, ECUDA.
 */
#define DEDISP_UBENCH_FORMS 8
int dedisp_ubench_fp32(int form, int iters, double* cycles_per_butterfly, double* ms);

int dedisp_destroy(dedisp_plan_t plan);

const char* dedisp_strerror(int code);
int dedisp_last_cuda_error(void); /* cudaError_t of the last DEDISP_ECUDA on this thread */

/*
 * Test hooks (used by the parity tests only).
 * dedisp_debug_unpack: the framed, unpacked block (step 1) of (chan, block) as float [n_fft][2] on the DEVICE: the
 *                      values the fused kernel itself holds in registers after its int8 -> fp32 conversion (the
 *                      corner turn and the kernel's own unpack run; the kernel stores and stops before the transform).
 * dedisp_debug_chirp:  copies the chirp table row (d, chan) to HOST as float [n_fft][2] (includes the 1/n_fft scale).
 * dedisp_debug_voltage: steps 1-5 for one (chan, block): DEVICE float [n_dm][L][2] dedispersed complex voltages.
 */
int dedisp_debug_unpack(dedisp_plan_t plan, const int8_t* d_in, long long n_samp, int chan, long long block,
                        float* d_block, void* cuda_stream);
int dedisp_debug_chirp(dedisp_plan_t plan, int d, int chan, float* h_chirp);
int dedisp_debug_voltage(dedisp_plan_t plan, const int8_t* d_in, long long n_samp, int chan, long long block,
                         float* d_volt, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------------------------
 * Full-band mode: the paper's own pipeline, no sub-banding (Fig. 4; SURVEY 8(f)
 * NEXT-1; readings R19-R21; oracle: oracle/fullband.py).
 *   1. every GSB spectrum (int8 [n_chan][2]: bins 0 .. n_chan-1 of a 2 n_chan-point real FFT, R19) is inverse
 *      transformed to 2 n_chan real samples: the Nyquist-sampled voltage series v
 *   2. blocks of n_fft samples (block b reads v[b L : b L + n_fft]) go through ONE long transform
 *   3. bin k (f_l = k 2 bw / n_fft above the lower band edge f_lo, R21) is multiplied by
 *      w(f_l) exp(-2 pi i psi), psi = D DM f_l^2 / ((f_l + f_lo) f_lo^2): Eq. 3 inverted, taper P:L123
 *   4. inverse transform; 5. the first D outputs of a block are dropped (R20; D = dispersion time in samples at
 *      2 bw, rounded up to n_int), L = n_fft - D stay; 6. squared and summed in groups of n_int
 *   out[d][b L/n_int + j] = sum_{i < n_int} y_d[b][D + j n_int + i]^2
 *   n_chan: 512 ... 8192 (2 n_chan a power of two); n_fft: a power of two in 2^20 ... 2^28; dm >= 0 (HOST, copied).
 * dedisp_fullband_framing is pure host arithmetic.  execute: DEVICE pointers, enqueues on the stream, allocates its
 * scratch on first use.  Errors as above (ESHORT: fewer than n_fft samples).
 * ------------------------------------------------------------------------------------------------------------------ */
typedef struct dedisp_fullband_s* dedisp_fullband_t;
int dedisp_fullband_framing(double bw_hz, double f_lo_hz, const double* dm, int n_dm, long long n_fft, int n_int, int* D,
                            long long* L);
int dedisp_fullband_plan(dedisp_fullband_t* out_plan, int n_chan, double bw_hz, double f_lo_hz, const double* dm, int n_dm,
                         long long n_fft, int n_int, unsigned flags);
int dedisp_fullband_get_framing(dedisp_fullband_t plan, int* D, long long* L, int* n1, int* n2); /* n_fft = n1 * n2 */
long long dedisp_fullband_out_samples(dedisp_fullband_t plan, long long n_spec);
int dedisp_fullband_execute(dedisp_fullband_t plan, const int8_t* d_spec, long long n_spec, float* d_out,
                            long long out_stride, void* cuda_stream); /* d_spec [n_spec][n_chan][2], d_out [n_dm][out_stride] */
/* test hook: step 1 alone, float [n_spec * 2 n_chan] on the DEVICE */
int dedisp_fullband_debug_series(dedisp_fullband_t plan, const int8_t* d_spec, long long n_spec, float* d_series,
                                 void* cuda_stream);
int dedisp_fullband_destroy(dedisp_fullband_t plan);

#ifdef __cplusplus
}
#endif
#endif /* DEDISP_H */
