// api.cu -- plan lifecycle and the one-shot execute of libdedisp (C ABI of include/dedisp.h).
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "dedisp_internal.h"

extern "C" const char* dedisp_strerror(int code)
{
    switch (code) {
        case DEDISP_OK: return "ok";
        case DEDISP_EINVAL: return "invalid argument";
        case DEDISP_ENOMEM: return "out of memory";
        case DEDISP_ECUDA: return "CUDA error (see dedisp_last_cuda_error)";
        case DEDISP_ESHORT: return "input shorter than one transform block";
        case DEDISP_ENODEV: return "no usable sm_100 CUDA device";
        case DEDISP_ETOOBIG: return "input needs more than DEDISP_STATIC_SCRATCH_BYTES of static scratch";
        default: return "unknown dedisp status";
    }
}

extern "C" int dedisp_last_cuda_error(void) { return g_dedisp_last_cuda; }

static void free_plan(dedisp_plan_s* p)
{
    if (!p) return;
    dedisp_stream_free(p);
    if (p->d_chirp) cudaFree(p->d_chirp);
    if (p->d_twiddle) cudaFree(p->d_twiddle);
    if (p->d_xt) cudaFree(p->d_xt);
    if (p->d_spec) cudaFree(p->d_spec);
    if (p->d_band_shift) cudaFree(p->d_band_shift);
    free(p->band_shift);
    if (p->prof_ev) {
        for (int i = 0; i < DEDISP_PROF_MAX * 3; ++i) cudaEventDestroy(p->prof_ev[i]);
        free(p->prof_ev);
    }
    free(p->dm);
    delete p;
}

// dedisp_plan and dedisp_plan_shard: channels chan0 .. chan0 + n_chan - 1 of a band of n_chan_total channels.
static int plan_impl(dedisp_plan_t* out_plan, int n_chan_total, double bw_total, double F_total, const double* dm, int n_dm,
                     int n_fft, int n_int, unsigned flags, int chan0, int n_chan, unsigned shard_flags)
{
    if (!out_plan) return DEDISP_EINVAL;
    *out_plan = nullptr;
    if ((flags & ~DEDISP_TAPER_MASK) || (flags & DEDISP_TAPER_MASK) == 3u) return DEDISP_EINVAL;
    if (shard_flags & ~(DEDISP_SHARD_FULL_INPUT | DEDISP_SHARD_OWN_FRAMING)) return DEDISP_EINVAL;
    if (n_fft <= 0 || (n_fft & (n_fft - 1)) || !dedisp_aos_supported(n_fft)) return DEDISP_EINVAL;
    // R9 gives D_tot % n_int == 0, so L % n_int == n_fft % n_int: only powers of two can divide a block evenly
    if (n_int <= 0 || (n_int & (n_int - 1))) return DEDISP_EINVAL;
    if (n_chan_total <= 0 || chan0 < 0 || n_chan <= 0 || chan0 > n_chan_total - n_chan) return DEDISP_EINVAL;
    // the whole band's framing: the common time axis of all shards (R9), and the one a plain plan uses
    int head_w, tail_w, L_w;
    double smear = 0.0;
    int rc = dedisp_framing_impl(n_chan_total, bw_total, F_total, dm, n_dm, n_fft, n_int, &head_w, &tail_w, &L_w, &smear);
    if (rc != DEDISP_OK) return rc;
    const double dv_total = bw_total / n_chan_total;
    const double bw_hz = dv_total * n_chan;                                               // this plan's sub-band
    const double f_center_hz = F_total - 0.5 * bw_total + ((double)chan0 + 0.5 * n_chan) * dv_total;
    int head = head_w, tail = tail_w, L = L_w;
    if (shard_flags & DEDISP_SHARD_OWN_FRAMING) {  // per-channel-group framing: only this group's own smear (R18)
        rc = dedisp_framing_impl(n_chan, bw_hz, f_center_hz, dm, n_dm, n_fft, n_int, &head, &tail, &L, &smear);
        if (rc != DEDISP_OK) return rc;
        if (head > head_w) return DEDISP_EINVAL;  // cannot happen: a sub-band's delays are bounded by the band's
    }

    int dev = 0, n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) {
        (void)cudaGetLastError();
        return DEDISP_ENODEV;
    }
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    int major = 0;
    DEDISP_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return DEDISP_ENODEV;  // the kernels are built for sm_100a only

    dedisp_plan_s* p = new (std::nothrow) dedisp_plan_s();
    if (!p) return DEDISP_ENOMEM;
    memset(p, 0, sizeof(*p));
    p->n_chan = n_chan; p->n_dm = n_dm; p->n_fft = n_fft; p->n_int = n_int;
    p->bw_hz = bw_hz; p->f_center_hz = f_center_hz; p->flags = flags;
    p->n_chan_total = n_chan_total; p->chan0 = chan0; p->bw_total_hz = bw_total; p->f_center_total_hz = F_total;
    p->in_pitch = (shard_flags & DEDISP_SHARD_FULL_INPUT) ? n_chan_total : n_chan;
    p->time_offset = (head_w - head) / n_int;  // both are multiples of n_int (R9)
    p->head = head; p->tail = tail; p->L = L; p->device = dev;
    p->max_smear_samples = smear;
    {   // P:L139-141 length rule, advisory
        long long n = 1;
        while ((double)n <= 2.0 * smear && n < (1ll << 30)) n <<= 1;
        p->nfft_rule = (int)n;
    }
    p->dm = (double*)malloc(sizeof(double) * n_dm);
    if (!p->dm) { free_plan(p); return DEDISP_ENOMEM; }
    memcpy(p->dm, dm, sizeof(double) * n_dm);

    {   // band alignment (R16): delay of channel c against the top channel of the WHOLE band in whole output samples,
        // the whole band's minimum removed, plus this plan's time offset against the whole band's framing: the
        // shifted outputs of all shards of one band line up sample for sample
        p->band_shift = (long long*)malloc(sizeof(long long) * (size_t)n_dm * n_chan);
        if (!p->band_shift) { free_plan(p); return DEDISP_ENOMEM; }
        const double f_top = F_total + 0.5 * bw_total - 0.5 * dv_total;
        p->band_max_shift = 0;
        for (int d = 0; d < n_dm; ++d) {
            long long* sh = p->band_shift + (size_t)d * n_chan;
            long long lo = 0, hi = 0;
            for (int c = 0; c < n_chan_total; ++c) {
                const double fc = F_total - 0.5 * bw_total + ((double)c + 0.5) * dv_total;
                const double delay_s = DEDISP_D_HZ2_S * dm[d] * (1.0 / (fc * fc) - 1.0 / (f_top * f_top));
                const long long v = llround(delay_s * dv_total / (double)n_int);
                if (c == 0 || v < lo) lo = v;
                if (c == 0 || v > hi) hi = v;
                if (c >= chan0 && c < chan0 + n_chan) sh[c - chan0] = v;
            }
            for (int c = 0; c < n_chan; ++c) sh[c] += p->time_offset - lo;
            if (hi - lo + p->time_offset > p->band_max_shift) p->band_max_shift = hi - lo + p->time_offset;
        }
    }
    double* d_dm = nullptr;
    auto fail = [&](int code) { if (d_dm) cudaFree(d_dm); free_plan(p); return code; };
#define PLAN_TRY(expr)                                                                           \
    do {                                                                                         \
        cudaError_t e__ = (expr);                                                                \
        if (e__ != cudaSuccess) {                                                                \
            g_dedisp_last_cuda = (int)e__; (void)cudaGetLastError();                             \
            return fail(e__ == cudaErrorMemoryAllocation ? DEDISP_ENOMEM : DEDISP_ECUDA);        \
        }                                                                                        \
    } while (0)
    rc = dedisp_aos_init();
    if (rc != DEDISP_OK) return fail(rc);
    PLAN_TRY(cudaMalloc(&p->d_chirp, sizeof(float2) * (size_t)n_dm * n_chan * n_fft));
    PLAN_TRY(cudaMalloc(&p->d_twiddle, sizeof(float2) * (size_t)n_fft));
    if (n_dm > 1)
        PLAN_TRY(cudaMalloc(&p->d_spec, dedisp_aos_spec_bytes(n_fft)));
    if (p->band_max_shift < 0x7fffffffll) {  // device copy as int32 (a shift that large leaves no series anyway)
        int* tmp = (int*)malloc(sizeof(int) * (size_t)n_dm * n_chan);
        if (!tmp) return fail(DEDISP_ENOMEM);
        for (size_t i = 0; i < (size_t)n_dm * n_chan; ++i) tmp[i] = (int)p->band_shift[i];
        cudaError_t e1 = cudaMalloc(&p->d_band_shift, sizeof(int) * (size_t)n_dm * n_chan);
        if (e1 == cudaSuccess)
            e1 = cudaMemcpy(p->d_band_shift, tmp, sizeof(int) * (size_t)n_dm * n_chan, cudaMemcpyHostToDevice);
        free(tmp);
        PLAN_TRY(e1);
    }
    PLAN_TRY(cudaMalloc(&d_dm, sizeof(double) * n_dm));
    PLAN_TRY(cudaMemcpy(d_dm, p->dm, sizeof(double) * n_dm, cudaMemcpyHostToDevice));
    rc = dedisp_launch_chirp_table(p, d_dm, 0);
    if (rc != DEDISP_OK) return fail(rc);
    rc = dedisp_launch_twiddle_table(p, 0);
    if (rc != DEDISP_OK) return fail(rc);
    PLAN_TRY(cudaDeviceSynchronize());
    cudaFree(d_dm);
#undef PLAN_TRY
    *out_plan = p;
    return DEDISP_OK;
}

extern "C" int dedisp_plan(dedisp_plan_t* out_plan, int n_chan, double bw_hz, double f_center_hz, const double* dm,
                           int n_dm, int n_fft, int n_int, unsigned flags)
{
    return plan_impl(out_plan, n_chan, bw_hz, f_center_hz, dm, n_dm, n_fft, n_int, flags, 0, n_chan, 0u);
}

extern "C" int dedisp_plan_shard(dedisp_plan_t* out_plan, int n_chan_total, double bw_hz_total, double f_center_hz_total,
                                 const double* dm, int n_dm, int n_fft, int n_int, unsigned flags, int chan0, int n_chan,
                                 unsigned shard_flags)
{
    return plan_impl(out_plan, n_chan_total, bw_hz_total, f_center_hz_total, dm, n_dm, n_fft, n_int, flags, chan0, n_chan,
                     shard_flags);
}

extern "C" long long dedisp_shard_time_offset(dedisp_plan_t p) { return p ? p->time_offset : 0; }

extern "C" int dedisp_get_info(dedisp_plan_t p, dedisp_info_t* info)
{
    if (!p || !info) return DEDISP_EINVAL;
    info->n_chan = p->n_chan; info->n_dm = p->n_dm; info->n_fft = p->n_fft; info->n_int = p->n_int;
    info->head = p->head; info->tail = p->tail; info->L = p->L;
    info->chan_width_hz = p->bw_hz / p->n_chan;
    info->max_smear_samples = p->max_smear_samples;
    info->nfft_rule = p->nfft_rule;
    return DEDISP_OK;
}

long long dedisp_n_blocks(const dedisp_plan_s* p, long long n_samp)
{
    if (n_samp < (long long)p->n_fft) return 0;
    return (n_samp - p->head - p->tail) / p->L;
}
static long long n_blocks(const dedisp_plan_s* p, long long n_samp) { return dedisp_n_blocks(p, n_samp); }

// The two kernels of the path for one batch of rows: corner-turn n_rows input rows to d_xt at row offset dst_t0, then
// the fused kernel over the first nb blocks of d_xt.  Optional events: profiling triple, and `after_corner_turn`
// (the streaming path frees its staging buffer there).
int dedisp_enqueue_chunk(dedisp_plan_s* p, const int8_t* d_in, long long n_rows, int8_t* d_xt, long long xt_stride,
                         long long dst_t0, long long nb, float* d_out, long long out_stride, cudaStream_t st,
                         cudaEvent_t after_corner_turn, int accumulate)
{
    cudaEvent_t* ev = nullptr;
    if (p->prof_on && p->prof_n < DEDISP_PROF_MAX) ev = p->prof_ev + 3 * (p->prof_n++);
    if (ev) DEDISP_CUDA_TRY(cudaEventRecord(ev[0], st));
    int rc = dedisp_launch_corner_turn(d_in, n_rows, p->n_chan, p->in_pitch, p->in_pitch == p->n_chan ? 0 : p->chan0, d_xt,
                                       xt_stride, dst_t0, st);
    if (rc != DEDISP_OK) return rc;
    if (ev) DEDISP_CUDA_TRY(cudaEventRecord(ev[1], st));
    if (after_corner_turn) DEDISP_CUDA_TRY(cudaEventRecord(after_corner_turn, st));
    if (nb > 0) {
        rc = dedisp_launch_aos(p, d_xt, xt_stride, nb, d_out, out_stride, 0, accumulate, st);
        if (rc != DEDISP_OK) return rc;
    }
    if (ev) DEDISP_CUDA_TRY(cudaEventRecord(ev[2], st));
    return DEDISP_OK;
}

extern "C" int dedisp_profile_enable(dedisp_plan_t p, int on)
{
    if (!p) return DEDISP_EINVAL;
    if (on && !p->prof_ev) {
        p->prof_ev = (cudaEvent_t*)calloc(DEDISP_PROF_MAX * 3, sizeof(cudaEvent_t));
        if (!p->prof_ev) return DEDISP_ENOMEM;
        for (int i = 0; i < DEDISP_PROF_MAX * 3; ++i) DEDISP_CUDA_TRY(cudaEventCreate(&p->prof_ev[i]));
    }
    p->prof_on = on ? 1 : 0;
    p->prof_n = 0;
    return DEDISP_OK;
}

extern "C" int dedisp_profile_read(dedisp_plan_t p, double* ms_corner_turn, double* ms_fused, int* n_calls)
{
    if (!p || !ms_corner_turn || !ms_fused || !n_calls) return DEDISP_EINVAL;
    double a = 0.0, b = 0.0;
    for (int i = 0; i < p->prof_n; ++i) {
        cudaEvent_t* ev = p->prof_ev + 3 * i;
        float m1 = 0.f, m2 = 0.f;
        DEDISP_CUDA_TRY(cudaEventSynchronize(ev[2]));
        DEDISP_CUDA_TRY(cudaEventElapsedTime(&m1, ev[0], ev[1]));
        DEDISP_CUDA_TRY(cudaEventElapsedTime(&m2, ev[1], ev[2]));
        a += m1; b += m2;
    }
    *ms_corner_turn = a; *ms_fused = b; *n_calls = p->prof_n;
    p->prof_n = 0;
    return DEDISP_OK;
}

extern "C" long long dedisp_out_samples(dedisp_plan_t p, long long n_samp)
{
    if (!p) return DEDISP_EINVAL;
    return n_blocks(p, n_samp) * (p->L / p->n_int);
}

extern "C" int dedisp_reserve(dedisp_plan_t p, long long n_samp)
{
    if (!p || n_samp <= 0) return DEDISP_EINVAL;
    const long long stride = dedisp_xt_stride(n_samp);
    if (stride <= p->xt_cap_samp) return DEDISP_OK;
    DEDISP_CUDA_TRY(cudaDeviceSynchronize());
    if (p->d_xt) { cudaFree(p->d_xt); p->d_xt = nullptr; p->xt_cap_samp = 0; }
    DEDISP_CUDA_TRY(cudaMalloc(&p->d_xt, (size_t)stride * p->n_chan * 2));
    p->xt_cap_samp = stride;
    return DEDISP_OK;
}

static int execute_impl(dedisp_plan_t p, const int8_t* d_in, long long n_samp, float* d_out, long long out_stride,
                        void* cuda_stream, int accumulate)
{
    if (!p || !d_in || n_samp <= 0) return DEDISP_EINVAL;
    const long long nb = n_blocks(p, n_samp);
    if (nb <= 0) return DEDISP_ESHORT;
    if (!d_out) return DEDISP_EINVAL;
    if (out_stride < nb * (p->L / p->n_int)) return DEDISP_EINVAL;
    int rc = dedisp_reserve(p, n_samp);
    if (rc != DEDISP_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long stride = p->xt_cap_samp;
    // only the rows that complete blocks are needed: nb*L + head + tail
    const long long used = nb * p->L + p->head + p->tail;
    return dedisp_enqueue_chunk(p, d_in, used, p->d_xt, stride, 0, nb, d_out, out_stride, st, nullptr, accumulate);
}

extern "C" int dedisp_execute(dedisp_plan_t p, const int8_t* d_in, long long n_samp, float* d_out,
                              long long out_stride, void* cuda_stream)
{
    return execute_impl(p, d_in, n_samp, d_out, out_stride, cuda_stream, 0);
}

extern "C" int dedisp_execute_add(dedisp_plan_t p, const int8_t* d_in, long long n_samp, float* d_out,
                                  long long out_stride, void* cuda_stream)
{
    return execute_impl(p, d_in, n_samp, d_out, out_stride, cuda_stream, 1);
}

// ---------------------------------------------------------------------------------------------------------------
// sub-band alignment + band sum
// ---------------------------------------------------------------------------------------------------------------
extern "C" long long dedisp_band_samples(dedisp_plan_t p, long long n_out)
{
    if (!p) return DEDISP_EINVAL;
    return n_out > p->band_max_shift ? n_out - p->band_max_shift : 0;
}

extern "C" int dedisp_band_shifts(dedisp_plan_t p, int d, long long* h_shift)
{
    if (!p || !h_shift || d < 0 || d >= p->n_dm) return DEDISP_EINVAL;
    memcpy(h_shift, p->band_shift + (size_t)d * p->n_chan, sizeof(long long) * p->n_chan);
    return DEDISP_OK;
}

extern "C" int dedisp_band_sum(dedisp_plan_t p, const float* d_out, long long out_stride, long long n_out,
                               float* d_series, long long series_stride, void* cuda_stream)
{
    if (!p || !d_out || !d_series || n_out <= 0 || out_stride < n_out || !p->d_band_shift) return DEDISP_EINVAL;
    const long long n_ser = dedisp_band_samples(p, n_out);
    if (n_ser <= 0) return DEDISP_ESHORT;
    if (series_stride < n_ser) return DEDISP_EINVAL;
    return dedisp_launch_band_sum(p, d_out, out_stride, d_series, series_stride, n_ser, (cudaStream_t)cuda_stream);
}

extern "C" int dedisp_fold(const float* d_series, long long n, double t0_s, double dt_s, double period_s, int n_bins,
                           float* d_sum, unsigned int* d_count, void* cuda_stream)
{
    if (!d_series || !d_sum || !d_count || n <= 0 || n_bins <= 0 || n_bins > 4096 || !(dt_s > 0.0) || !(period_s > 0.0) ||
        !isfinite(t0_s))
        return DEDISP_EINVAL;
    return dedisp_launch_fold(d_series, n, t0_s, dt_s, period_s, n_bins, d_sum, d_count, (cudaStream_t)cuda_stream);
}

extern "C" int dedisp_destroy(dedisp_plan_t p)
{
    if (!p) return DEDISP_EINVAL;
    cudaDeviceSynchronize();
    (void)cudaGetLastError();
    free_plan(p);
    return DEDISP_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// test hooks
// ---------------------------------------------------------------------------------------------------------------
extern "C" int dedisp_debug_chirp(dedisp_plan_t p, int d, int chan, float* h_chirp)
{
    if (!p || !h_chirp || d < 0 || d >= p->n_dm || chan < 0 || chan >= p->n_chan) return DEDISP_EINVAL;
    const size_t row = ((size_t)d * p->n_chan + chan) * p->n_fft;
    DEDISP_CUDA_TRY(cudaMemcpy(h_chirp, p->d_chirp + row, sizeof(float2) * p->n_fft, cudaMemcpyDeviceToHost));
    return DEDISP_OK;
}

static int debug_prepare(dedisp_plan_t p, const int8_t* d_in, long long n_samp, int chan, long long block,
                         cudaStream_t st)
{
    if (!p || !d_in || chan < 0 || chan >= p->n_chan) return DEDISP_EINVAL;
    const long long nb = n_blocks(p, n_samp);
    if (nb <= 0) return DEDISP_ESHORT;
    if (block < 0 || block >= nb) return DEDISP_EINVAL;
    int rc = dedisp_reserve(p, n_samp);
    if (rc != DEDISP_OK) return rc;
    return dedisp_launch_corner_turn(d_in, nb * p->L + p->head + p->tail, p->n_chan, p->in_pitch,
                                     p->in_pitch == p->n_chan ? 0 : p->chan0, p->d_xt, p->xt_cap_samp, 0, st);
}

extern "C" int dedisp_debug_unpack(dedisp_plan_t p, const int8_t* d_in, long long n_samp, int chan, long long block,
                                   float* d_block, void* cuda_stream)
{
    if (!d_block) return DEDISP_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = debug_prepare(p, d_in, n_samp, chan, block, st);
    if (rc != DEDISP_OK) return rc;
    return dedisp_launch_aos_debug_voltage(p, p->d_xt, p->xt_cap_samp, chan, block, d_block, 1, st);
}

extern "C" int dedisp_debug_voltage(dedisp_plan_t p, const int8_t* d_in, long long n_samp, int chan, long long block,
                                    float* d_volt, void* cuda_stream)
{
    if (!d_volt) return DEDISP_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = debug_prepare(p, d_in, n_samp, chan, block, st);
    if (rc != DEDISP_OK) return rc;
    return dedisp_launch_aos_debug_voltage(p, p->d_xt, p->xt_cap_samp, chan, block, d_volt, 0, st);
}
