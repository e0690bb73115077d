// stream.cu -- step a6 of the path: real-time streaming from pinned host memory (Fig. 9: host->device copy of
// one block, compute on the previous one and device->host copy of the one before run concurrently on three CUDA streams;
// the samples lost at the edge of a block are prefixed to the next one).
//
// Device buffers (all double-buffered, allocated by dedisp_stream_begin):
//   d_stage[2]  int8 [max_chunk][n_chan][2]          time-major chunk as it arrives
//   d_xt[2]     int8 [n_chan][xt_stride][2]          channel-major: [carry | chunk]; the unconsumed tail of one push is
//                                                    copied to the front of the OTHER buffer by the next push
//   d_out[2]    float [n_dm][n_chan][max_out]        outputs of one push
// Push i uses slot i&1 of d_stage / d_out and writes the xt buffer the previous push did not.
#include <stdlib.h>
#include <string.h>

#include <new>

#include "dedisp_internal.h"

struct dedisp_stream_state {
    long long max_chunk, xt_stride, max_out;
    int8_t* d_stage[2];
    int8_t* d_xt[2];
    float* d_out[2];
    cudaStream_t s_h2d, s_comp, s_d2h;
    cudaEvent_t h2d_done[2], comp_done[2], d2h_done[2];
    bool used[2];
    int cur_xt;               // xt buffer holding the carry
    long long carry_off, carry;  // carry = rows [carry_off, carry_off + carry) of d_xt[cur_xt]
    long long n_push;
};

void dedisp_stream_free(dedisp_plan_s* p)
{
    dedisp_stream_state* s = p->stream;
    if (!s) return;
    if (s->s_h2d) cudaStreamSynchronize(s->s_h2d);
    if (s->s_comp) cudaStreamSynchronize(s->s_comp);
    if (s->s_d2h) cudaStreamSynchronize(s->s_d2h);
    for (int i = 0; i < 2; ++i) {
        if (s->d_stage[i]) cudaFree(s->d_stage[i]);
        if (s->d_xt[i]) cudaFree(s->d_xt[i]);
        if (s->d_out[i]) cudaFree(s->d_out[i]);
        if (s->h2d_done[i]) cudaEventDestroy(s->h2d_done[i]);
        if (s->comp_done[i]) cudaEventDestroy(s->comp_done[i]);
        if (s->d2h_done[i]) cudaEventDestroy(s->d2h_done[i]);
    }
    if (s->s_h2d) cudaStreamDestroy(s->s_h2d);
    if (s->s_comp) cudaStreamDestroy(s->s_comp);
    if (s->s_d2h) cudaStreamDestroy(s->s_d2h);
    (void)cudaGetLastError();
    delete s;
    p->stream = nullptr;
}

extern "C" int dedisp_stream_begin(dedisp_plan_t p, long long max_chunk_samp)
{
    if (!p || max_chunk_samp <= 0) return DEDISP_EINVAL;
    if (p->in_pitch != p->n_chan) return DEDISP_EINVAL;  // DEDISP_SHARD_FULL_INPUT plans: one-shot calls only
    if (p->stream && p->stream->max_chunk >= max_chunk_samp) {
        // a new observation on buffers that are already big enough: drain, forget the carry, keep the allocations
        int rc = dedisp_stream_sync(p);
        if (rc != DEDISP_OK) return rc;
        dedisp_stream_state* s = p->stream;
        s->used[0] = s->used[1] = false;
        s->cur_xt = 0;
        s->carry_off = s->carry = s->n_push = 0;
        return DEDISP_OK;
    }
    dedisp_stream_free(p);
    dedisp_stream_state* s = new (std::nothrow) dedisp_stream_state();
    if (!s) return DEDISP_ENOMEM;
    memset(s, 0, sizeof(*s));
    p->stream = s;
    s->max_chunk = max_chunk_samp;
    // the carry is always shorter than one transform: carry - (head+tail) < L
    const long long max_total = (long long)p->n_fft - 1 + max_chunk_samp;
    s->xt_stride = dedisp_xt_stride(max_total);
    const long long max_nb = dedisp_n_blocks(p, max_total);
    s->max_out = (max_nb > 0 ? max_nb : 1) * (long long)(p->L / p->n_int);
    auto fail = [&](cudaError_t e) {
        g_dedisp_last_cuda = (int)e;
        (void)cudaGetLastError();
        dedisp_stream_free(p);
        return e == cudaErrorMemoryAllocation ? DEDISP_ENOMEM : DEDISP_ECUDA;
    };
#define S_TRY(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) return fail(e__); } while (0)
    for (int i = 0; i < 2; ++i) {
        S_TRY(cudaMalloc(&s->d_stage[i], (size_t)max_chunk_samp * p->n_chan * 2));
        S_TRY(cudaMalloc(&s->d_xt[i], (size_t)s->xt_stride * p->n_chan * 2));
        S_TRY(cudaMalloc(&s->d_out[i], sizeof(float) * (size_t)p->n_dm * p->n_chan * s->max_out));
        S_TRY(cudaEventCreateWithFlags(&s->h2d_done[i], cudaEventDisableTiming));
        S_TRY(cudaEventCreateWithFlags(&s->comp_done[i], cudaEventDisableTiming));
        S_TRY(cudaEventCreateWithFlags(&s->d2h_done[i], cudaEventDisableTiming));
    }
    S_TRY(cudaStreamCreateWithFlags(&s->s_h2d, cudaStreamNonBlocking));
    S_TRY(cudaStreamCreateWithFlags(&s->s_comp, cudaStreamNonBlocking));
    S_TRY(cudaStreamCreateWithFlags(&s->s_d2h, cudaStreamNonBlocking));
#undef S_TRY
    return DEDISP_OK;
}

extern "C" int dedisp_stream_push(dedisp_plan_t p, const int8_t* h_in, long long n_samp, float* h_out,
                                  long long out_stride, long long* n_out)
{
    if (!p || !p->stream || !h_in || !n_out || n_samp <= 0) return DEDISP_EINVAL;
    dedisp_stream_state* s = p->stream;
    if (n_samp > s->max_chunk) return DEDISP_EINVAL;
    const long long total = s->carry + n_samp;
    const long long nb = dedisp_n_blocks(p, total);
    const long long per = p->L / p->n_int;
    const long long nout = nb * per;
    if (nout > 0 && (!h_out || out_stride < nout)) return DEDISP_EINVAL;
    const int slot = (int)(s->n_push & 1), prev = slot ^ 1;
    // hand-back points (see dedisp.h): push i-2 is complete, the H2D copy of push i-1 has left its host buffer
    if (s->used[slot]) DEDISP_CUDA_TRY(cudaEventSynchronize(s->d2h_done[slot]));
    if (s->used[prev]) DEDISP_CUDA_TRY(cudaEventSynchronize(s->h2d_done[prev]));

    // stream A: host -> device.  d_stage[slot] was last read by the corner turn of push i-2: complete.
    DEDISP_CUDA_TRY(cudaMemcpyAsync(s->d_stage[slot], h_in, (size_t)n_samp * p->n_chan * 2, cudaMemcpyHostToDevice,
                                    s->s_h2d));
    DEDISP_CUDA_TRY(cudaEventRecord(s->h2d_done[slot], s->s_h2d));

    // stream B: prefix the carry, corner-turn the chunk behind it, run the fused kernel
    DEDISP_CUDA_TRY(cudaStreamWaitEvent(s->s_comp, s->h2d_done[slot], 0));
    const int nxt = s->cur_xt ^ 1;
    if (s->carry > 0)
        DEDISP_CUDA_TRY(cudaMemcpy2DAsync(s->d_xt[nxt], (size_t)s->xt_stride * 2,
                                          s->d_xt[s->cur_xt] + s->carry_off * 2, (size_t)s->xt_stride * 2,
                                          (size_t)s->carry * 2, (size_t)p->n_chan, cudaMemcpyDeviceToDevice, s->s_comp));
    int rc = dedisp_enqueue_chunk(p, s->d_stage[slot], n_samp, s->d_xt[nxt], s->xt_stride, s->carry, nb, s->d_out[slot],
                                  s->max_out, s->s_comp, nullptr);
    if (rc != DEDISP_OK) return rc;
    DEDISP_CUDA_TRY(cudaEventRecord(s->comp_done[slot], s->s_comp));

    // stream C: device -> host
    DEDISP_CUDA_TRY(cudaStreamWaitEvent(s->s_d2h, s->comp_done[slot], 0));
    if (nout > 0)
        DEDISP_CUDA_TRY(cudaMemcpy2DAsync(h_out, sizeof(float) * (size_t)out_stride, s->d_out[slot],
                                          sizeof(float) * (size_t)s->max_out, sizeof(float) * (size_t)nout,
                                          (size_t)p->n_dm * p->n_chan, cudaMemcpyDeviceToHost, s->s_d2h));
    DEDISP_CUDA_TRY(cudaEventRecord(s->d2h_done[slot], s->s_d2h));

    s->used[slot] = true;
    s->cur_xt = nxt;
    s->carry_off = nb * p->L;
    s->carry = total - nb * p->L;
    s->n_push++;
    *n_out = nout;
    return DEDISP_OK;
}

extern "C" int dedisp_stream_sync(dedisp_plan_t p)
{
    if (!p || !p->stream) return DEDISP_EINVAL;
    DEDISP_CUDA_TRY(cudaStreamSynchronize(p->stream->s_h2d));
    DEDISP_CUDA_TRY(cudaStreamSynchronize(p->stream->s_comp));
    DEDISP_CUDA_TRY(cudaStreamSynchronize(p->stream->s_d2h));
    return DEDISP_OK;
}

extern "C" int dedisp_stream_end(dedisp_plan_t p)
{
    if (!p || !p->stream) return DEDISP_EINVAL;
    int rc = dedisp_stream_sync(p);
    dedisp_stream_free(p);
    return rc;
}
