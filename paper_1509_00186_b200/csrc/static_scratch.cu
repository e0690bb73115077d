// static_scratch.cu -- dedisp_execute_static: dedisp_execute() for callers that must not allocate (CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc).  The one piece of scratch dedisp_execute() allocates on
// demand is the channel-major int8 buffer [n_chan][stride][2] that the corner turn writes and the fused kernel reads
// (dedisp_reserve); here it is a file-scope device array of a fixed, modest size instead.  Same kernels, same
// arithmetic, same outputs as dedisp_execute(); no cudaMalloc / cudaFree / allocating library call on this path.
//
//   * The array lives in every GPU context that loads the library, until the process exits.
//   * In host code the array's NAME is a host-side stand-in, not a device address: its device address is taken once
//     per device, with that device current, with cudaGetSymbolAddress (below), and that pointer goes to the kernels.
//   * Every call (of every plan, on every stream) shares the array, and it keeps the last call's contents.  Nothing
//     in it has to start at zero: a call reads only bytes that its own corner turn wrote before (rows
//     [0, nb*L + head + tail) of every channel; idle unit slots of the fused kernel read nothing).  Two calls that
//     overlap on the GPU (different streams, or one stream from two host threads) RACE on it.
#include <mutex>

#include "dedisp_internal.h"

static __device__ __align__(256) unsigned char g_static_xt[DEDISP_STATIC_SCRATCH_BYTES];

namespace {

constexpr int MAX_DEVICES = 64;
int8_t* g_static_ptr[MAX_DEVICES];  // device address of g_static_xt on device i, nullptr until asked for
std::mutex g_static_mutex;

// once per device, with that device current
int static_scratch_ptr(int dev, int8_t** out)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void* ptr = nullptr;
        DEDISP_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_static_xt));
        if (!ptr || ((uintptr_t)ptr & 255u)) return DEDISP_ECUDA;
        g_static_ptr[dev] = static_cast<int8_t*>(ptr);
    }
    *out = g_static_ptr[dev];
    return DEDISP_OK;
}

}  // namespace

extern "C" int dedisp_execute_static(dedisp_plan_t p, const int8_t* d_in, long long n_samp, float* d_out,
                                     long long out_stride, void* cuda_stream)
{
    if (!p || !d_in || n_samp <= 0) return DEDISP_EINVAL;
    const long long nb = dedisp_n_blocks(p, n_samp);
    if (nb <= 0) return DEDISP_ESHORT;
    if (!d_out) return DEDISP_EINVAL;
    if (out_stride < nb * (p->L / p->n_int)) return DEDISP_EINVAL;
    // only the rows that complete blocks are turned: nb*L + head + tail (as dedisp_execute does)
    const long long used = nb * p->L + p->head + p->tail;
    const long long stride = dedisp_xt_stride(used);
    if (stride > (long long)DEDISP_STATIC_SCRATCH_BYTES / 2 / p->n_chan) return DEDISP_ETOOBIG;
    int dev = -1;
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != p->device || dev < 0 || dev >= MAX_DEVICES) return DEDISP_EINVAL;  // a plan belongs to its device
    int8_t* d_xt = nullptr;
    int rc = static_scratch_ptr(dev, &d_xt);
    if (rc != DEDISP_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    rc = dedisp_launch_corner_turn(d_in, used, p->n_chan, p->in_pitch, p->in_pitch == p->n_chan ? 0 : p->chan0, d_xt,
                                   stride, 0, st);
    if (rc != DEDISP_OK) return rc;
    return dedisp_launch_aos(p, d_xt, stride, nb, d_out, out_stride, 0, 0, st);
}
