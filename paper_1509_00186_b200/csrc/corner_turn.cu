// corner_turn.cu -- step 1a of the path: the GSB voltage-beam block arrives time-major, int8 [t][chan][re,im]
// (R10).  Every later step works on one channel's time series, so the block is turned once into
// channel-major int8 [chan][t][re,im] (2 B per complex sample stay 2 B: the unpack to fp32 happens in registers of the
// fused kernel).  Byte movement plus one bit flip: every byte is stored as x ^ 0x80 (= x + 128 as an unsigned byte), the
// form the fused kernel's I2F-free conversion starts from; the flip is free in this HBM-bound kernel and saves the
// fused kernel one LOP3 per sample.  HBM-bound: 2 B read + 2 B written per sample.
#include "dedisp_internal.h"

namespace {

constexpr int TILE_C = 64;   // channels per tile: 64 * 2 B = 128 B per input row
constexpr int TILE_T = 128;  // samples per tile: 128 * 2 B = 256 B per output row
constexpr int PITCH_W = 33;  // smem row pitch in 32-bit words (64 shorts + 1 word pad)

// Vector path: 16 B loads along the channel axis, 16 B stores along the time axis.
// Requires n_chan % 8 == 0, xt_stride % 8 == 0 and 16 B aligned base pointers.  Tiles are laid on the DESTINATION's
// 8-sample grid (the first tile starts dst_t0 % 8 rows before row 0), so any dst_t0 keeps the 16 B stores aligned:
// the streaming path appends chunks behind a carry of arbitrary length.
__global__ void __launch_bounds__(256) corner_turn_vec_kernel(const int8_t* __restrict__ in, long long n_samp, int n_chan,
                                                              int in_pitch, int8_t* __restrict__ xt,
                                                              long long xt_stride, long long dst_t0)
{
    __shared__ uint32_t tile[TILE_T * PITCH_W];
    const long long t0 = (long long)blockIdx.x * TILE_T - (dst_t0 & 7);
    const int c0 = blockIdx.y * TILE_C;
    const int tid = threadIdx.x;
    const uint16_t* in16 = reinterpret_cast<const uint16_t*>(in);
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const int idx = it * 256 + tid;
        const int row = idx >> 3, q = idx & 7;
        const long long t = t0 + row;
        const int c = c0 + q * 8;
        uint4 v = make_uint4(0, 0, 0, 0);
        if (t >= 0 && t < n_samp && c < n_chan)  // n_chan % 8 == 0: the 8 channels are all inside
            v = __ldg(reinterpret_cast<const uint4*>(in16 + t * in_pitch + c));
        v.x ^= 0x80808080u; v.y ^= 0x80808080u; v.z ^= 0x80808080u; v.w ^= 0x80808080u;
        uint32_t* dst = &tile[row * PITCH_W + q * 4];
        dst[0] = v.x; dst[1] = v.y; dst[2] = v.z; dst[3] = v.w;
    }
    __syncthreads();
    const int lane = tid & 31, warp = tid >> 5;
    const int tq_lo = lane & 1, c_lo = lane >> 1;
    const uint16_t* tile16 = reinterpret_cast<const uint16_t*>(tile);
    uint16_t* xt16 = reinterpret_cast<uint16_t*>(xt);
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const int combo = it * 8 + warp;
        const int c = (combo & 3) * 16 + c_lo;
        const int tq = (combo >> 2) * 2 + tq_lo;
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint32_t lo = tile16[(tq * 8 + 2 * i) * (2 * PITCH_W) + c];
            const uint32_t hi = tile16[(tq * 8 + 2 * i + 1) * (2 * PITCH_W) + c];
            w[i] = lo | (hi << 16);
        }
        const long long t = t0 + tq * 8;
        if (c0 + c >= n_chan || t >= n_samp || t + 8 <= 0) continue;
        uint16_t* dst = xt16 + (long long)(c0 + c) * xt_stride + dst_t0 + t;
        if (t >= 0 && t + 8 <= n_samp) {
            *reinterpret_cast<uint4*>(dst) = make_uint4(w[0], w[1], w[2], w[3]);
        } else {
            for (int i = 0; i < 8; ++i)
                if (t + i >= 0 && t + i < n_samp) dst[i] = (uint16_t)(w[i >> 1] >> ((i & 1) * 16));
        }
    }
}

// Scalar path for any n_chan / alignment: 32 x 32 tile of 2-byte samples.
__global__ void __launch_bounds__(256) corner_turn_scalar_kernel(const int8_t* __restrict__ in, long long n_samp,
                                                                 int n_chan, int in_pitch, int8_t* __restrict__ xt,
                                                                 long long xt_stride, long long dst_t0)
{
    __shared__ uint16_t tile[32][33];
    const uint16_t* in16 = reinterpret_cast<const uint16_t*>(in);
    uint16_t* xt16 = reinterpret_cast<uint16_t*>(xt);
    const long long t0 = (long long)blockIdx.x * 32;
    const int c0 = blockIdx.y * 32;
    const int x = threadIdx.x & 31, y = threadIdx.x >> 5;
    for (int r = y; r < 32; r += 8) {
        const long long t = t0 + r;
        const int c = c0 + x;
        tile[r][x] = (t < n_samp && c < n_chan) ? (uint16_t)(in16[t * in_pitch + c] ^ 0x8080u) : (uint16_t)0x8080u;
    }
    __syncthreads();
    for (int r = y; r < 32; r += 8) {
        const int c = c0 + r;
        const long long t = t0 + x;
        if (c < n_chan && t < n_samp) xt16[(long long)c * xt_stride + dst_t0 + t] = tile[x][r];
    }
}

}  // namespace

int dedisp_launch_corner_turn(const int8_t* d_in, long long n_samp, int n_chan, int in_pitch, int chan0, int8_t* d_xt,
                              long long xt_stride, long long dst_t0, cudaStream_t st)
{
    if (n_samp <= 0) return DEDISP_OK;
    d_in += 2 * (size_t)chan0;  // first column of this plan's channels
    const bool vec = (n_chan % 8 == 0) && (in_pitch % 8 == 0) && (xt_stride % 8 == 0) && ((uintptr_t)d_in % 16 == 0) &&
                     ((uintptr_t)d_xt % 16 == 0);
    if (vec) {
        dim3 grid((unsigned)((n_samp + (dst_t0 & 7) + TILE_T - 1) / TILE_T), (unsigned)((n_chan + TILE_C - 1) / TILE_C));
        corner_turn_vec_kernel<<<grid, 256, 0, st>>>(d_in, n_samp, n_chan, in_pitch, d_xt, xt_stride, dst_t0);
    } else {
        dim3 grid((unsigned)((n_samp + 31) / 32), (unsigned)((n_chan + 31) / 32));
        corner_turn_scalar_kernel<<<grid, 256, 0, st>>>(d_in, n_samp, n_chan, in_pitch, d_xt, xt_stride, dst_t0);
    }
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}
