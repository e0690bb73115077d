// fused.cu -- steps 1b-6 of the path in ONE kernel per call: unpack -> forward FFT -> chirp multiply -> inverse FFT ->
// overlap discard -> |v|^2 -> integrate (Fig. 4).  A complex sample is read once
// from HBM as 2 bytes and leaves as 4/n_int bytes; everything in between stays in registers / shared memory.
// The forward spectrum is computed once per (channel, block) and shared by all trial DMs.
#include "dedisp_internal.h"
#include "fft_regs.cuh"

using namespace dedisp_fft;

namespace {

// Transform shapes: N = product of the radices; E values per thread; U units (channel, block) per CTA.
template <int N> struct Shape;
template <> struct Shape<1024>  { static constexpr int E = 16, U = 4, R0 = 16, R1 = 16, R2 = 4,  R3 = 1; };
template <> struct Shape<2048>  { static constexpr int E = 16, U = 2, R0 = 16, R1 = 16, R2 = 8,  R3 = 1; };
template <> struct Shape<4096>  { static constexpr int E = 16, U = 1, R0 = 16, R1 = 16, R2 = 16, R3 = 1; };
template <> struct Shape<8192>  { static constexpr int E = 32, U = 1, R0 = 16, R1 = 16, R2 = 16, R3 = 2; };
template <> struct Shape<16384> { static constexpr int E = 32, U = 1, R0 = 16, R1 = 16, R2 = 16, R3 = 4; };

// Puts the outputs of a final radix-R pass (left bit-reversed by butterfly()) back into the canonical register map.
template <int R, int E>
__device__ __forceinline__ void natural_order(float2 (&x)[E])
{
    constexpr int S = E / R;
    float2 y[E];
#pragma unroll
    for (int q = 0; q < S; ++q)
#pragma unroll
        for (int r = 0; r < R; ++r) y[q + r * S] = x[q + bitrev(r, R) * S];
#pragma unroll
    for (int m = 0; m < E; ++m) x[m] = y[m];
}

// Full N-point transform of the register-resident sequence; unnormalised; kernel exp(SIGN*2*pi*i*k*n/N).
template <int N, int SIGN>
__device__ __forceinline__ void fft_unit(float2 (&x)[Shape<N>::E], int t, float2* __restrict__ sm,
                                         const float2* __restrict__ tw)
{
    using Sh = Shape<N>;
    constexpr int E = Sh::E, R0 = Sh::R0, R1 = Sh::R1, R2 = Sh::R2, R3 = Sh::R3;
    pass_compute<N, R0, 1, SIGN, E>(x, t, tw);
    exchange<N, R0, 1, E>(x, t, sm);
    pass_compute<N, R1, R0, SIGN, E>(x, t, tw);
    exchange<N, R1, R0, E>(x, t, sm);
    pass_compute<N, R2, R0 * R1, SIGN, E>(x, t, tw);
    if constexpr (R3 > 1) {
        exchange<N, R2, R0 * R1, E>(x, t, sm);
        pass_compute<N, R3, R0 * R1 * R2, SIGN, E>(x, t, tw);
        natural_order<R3, E>(x);
    } else {
        natural_order<R2, E>(x);
    }
}

struct FusedArgs {
    const int8_t* xt;       // [n_chan][xt_stride][2]
    long long xt_stride;    // samples
    const float2* chirp;    // [n_dm][n_chan][N], includes 1/N
    const float2* tw;       // [N]
    float* out;             // [n_dm][n_chan][out_stride]
    long long out_stride, out_col0;
    float2* spec;           // [gridDim.x][U][N] forward-spectrum stash, used when n_dm > 1
    float2* volt;           // debug: [n_dm][L] voltages of unit volt_unit, else nullptr
    long long nb;           // blocks per channel
    long long n_units;      // n_chan * nb
    long long first_unit;   // debug: process only this unit
    int n_chan, n_dm, n_int, head, L;
};

template <int N>
__global__ void __launch_bounds__(Shape<N>::U * N / Shape<N>::E) fused_dedisp_kernel(const FusedArgs a)
{
    using Sh = Shape<N>;
    constexpr int E = Sh::E, U = Sh::U, TPU = N / E;
    extern __shared__ float2 smem[];
    const int ul = threadIdx.x / TPU;  // unit inside the CTA
    const int t = threadIdx.x % TPU;   // thread inside the unit
    float2* sm = smem + (size_t)ul * padded_len(N);
    float* smf = reinterpret_cast<float*>(sm);
    const long long n_items = (a.n_units + U - 1) / U;
    const int n_out = a.L / a.n_int;

    for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
        const long long u = a.first_unit + item * U + ul;
        const bool live = u < a.first_unit + a.n_units;
        const int c = live ? (int)(u / a.nb) : 0;
        const long long b = live ? u % a.nb : 0;

        // 1b. unpack int8 (re, im) -> fp32 (exact), framed block b = rows b*L .. b*L+N-1 of channel c (R10)
        float2 x[E];
        {
            const uint16_t* src = reinterpret_cast<const uint16_t*>(a.xt) + (long long)c * a.xt_stride + b * a.L + t;
#pragma unroll
            for (int m = 0; m < E; ++m) {
                const uint32_t v = live ? (uint32_t)__ldg(src + m * TPU) : 0u;
                x[m] = make_float2((float)(int8_t)(v & 0xffu), (float)(int8_t)(v >> 8));
            }
        }
        // 2. forward FFT
        fft_unit<N, -1>(x, t, sm, a.tw);

        float2* stash = a.spec + ((size_t)blockIdx.x * U + ul) * N;
        if (a.n_dm > 1) {
#pragma unroll
            for (int m = 0; m < E; ++m) stash[t + m * TPU] = x[m];
        }
        for (int d = 0; d < a.n_dm; ++d) {
            if (d > 0) {
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = stash[t + m * TPU];  // same thread wrote it: no fence needed
            }
            // 3. chirp multiply (Eq. 3); table holds taper * exp(+2 pi i psi) / N
            {
                const float2* h = a.chirp + ((size_t)d * a.n_chan + c) * N + t;
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = cmul(x[m], __ldg(h + m * TPU));
            }
            // 4. inverse FFT (1/N already applied)
            fft_unit<N, +1>(x, t, sm, a.tw);

            if (a.volt) {  // debug hook: valid voltages of this unit
#pragma unroll
                for (int m = 0; m < E; ++m) {
                    const int i = t + m * TPU - a.head;
                    if (live && i >= 0 && i < a.L) a.volt[(size_t)d * a.L + i] = x[m];
                }
                continue;
            }
            // 5 + 6. discard the overlap, detect, integrate n_int samples (R9, R11)
            float pw[E];
#pragma unroll
            for (int m = 0; m < E; ++m) pw[m] = fmaf(x[m].x, x[m].x, x[m].y * x[m].y);
            float* dst = a.out + ((size_t)d * a.n_chan + c) * a.out_stride + a.out_col0 + b * n_out;
            {
                // n_int is a power of two (the framing admits nothing else: L = N - D_tot with D_tot % n_int == 0).
                // sums over aligned groups of g = min(n_int, 32) lanes; sample i = t + m*TPU, head % n_int == 0
                const int g = a.n_int < 32 ? a.n_int : 32;
                for (int off = 1; off < g; off <<= 1) {
#pragma unroll
                    for (int m = 0; m < E; ++m) pw[m] += __shfl_xor_sync(0xffffffffu, pw[m], off);
                }
                if ((t & (g - 1)) == 0) {
#pragma unroll
                    for (int m = 0; m < E; ++m) smf[(t + m * TPU) / g] = pw[m];
                }
                __syncthreads();
                const int per = a.n_int / g, first = a.head / g;
                for (int o = t; o < n_out; o += TPU) {
                    float acc = smf[first + o * per];
                    for (int i = 1; i < per; ++i) acc += smf[first + o * per + i];
                    if (live) dst[o] = acc;
                }
            }
            __syncthreads();  // staging area is the exchange buffer of the next transform
        }
    }
}

__global__ void debug_unpack_kernel(const int8_t* __restrict__ xt, long long xt_stride, int chan, long long row0,
                                    int n_fft, float2* __restrict__ dst)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_fft) return;
    const int8_t* p = xt + ((long long)chan * xt_stride + row0 + n) * 2;
    dst[n] = make_float2((float)p[0], (float)p[1]);
}

template <int N> constexpr size_t smem_bytes() { return sizeof(float2) * (size_t)Shape<N>::U * padded_len(N); }
template <int N> constexpr int cta_threads() { return Shape<N>::U * N / Shape<N>::E; }

struct KernelInfo { int ctas_per_sm; int n_sm; size_t spec_bytes; };
KernelInfo g_info[5];
bool g_init_done = false;

template <int N> int init_one(int slot)
{
    DEDISP_CUDA_TRY(cudaFuncSetAttribute(fused_dedisp_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem_bytes<N>()));
    int occ = 0;
    DEDISP_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fused_dedisp_kernel<N>, cta_threads<N>(),
                                                                  smem_bytes<N>()));
    int dev = 0, n_sm = 0;
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    DEDISP_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    g_info[slot].ctas_per_sm = occ > 0 ? occ : 1;
    g_info[slot].n_sm = n_sm;
    g_info[slot].spec_bytes = sizeof(float2) * (size_t)g_info[slot].ctas_per_sm * n_sm * Shape<N>::U * N;
    return DEDISP_OK;
}

int slot_of(int n_fft)
{
    switch (n_fft) {
        case 1024: return 0; case 2048: return 1; case 4096: return 2; case 8192: return 3; case 16384: return 4;
        default: return -1;
    }
}

template <int N>
int launch_one(const dedisp_plan_s* p, FusedArgs& a, cudaStream_t st)
{
    const int slot = slot_of(N);
    const long long n_items = (a.n_units + Shape<N>::U - 1) / Shape<N>::U;
    long long grid = (long long)g_info[slot].ctas_per_sm * g_info[slot].n_sm;
    if (grid > n_items) grid = n_items;
    a.spec = p->d_spec;  // sized by dedisp_fused_spec_bytes() at plan time; only touched when n_dm > 1
    fused_dedisp_kernel<N><<<(unsigned)grid, cta_threads<N>(), smem_bytes<N>(), st>>>(a);
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}

int dispatch(const dedisp_plan_s* p, FusedArgs& a, cudaStream_t st)
{
    switch (p->n_fft) {
        case 1024: return launch_one<1024>(p, a, st);
        case 2048: return launch_one<2048>(p, a, st);
        case 4096: return launch_one<4096>(p, a, st);
        case 8192: return launch_one<8192>(p, a, st);
        case 16384: return launch_one<16384>(p, a, st);
        default: return DEDISP_EINVAL;
    }
}

FusedArgs base_args(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, long long nb)
{
    FusedArgs a{};
    a.xt = d_xt; a.xt_stride = xt_stride; a.chirp = p->d_chirp; a.tw = p->d_twiddle;
    a.nb = nb; a.n_units = (long long)p->n_chan * nb; a.first_unit = 0;
    a.n_chan = p->n_chan; a.n_dm = p->n_dm; a.n_int = p->n_int; a.head = p->head; a.L = p->L;
    return a;
}

}  // namespace

int dedisp_fused_supported(int n_fft) { return slot_of(n_fft) >= 0; }

size_t dedisp_fused_spec_bytes(int n_fft)
{
    const int slot = slot_of(n_fft);
    return slot < 0 ? 0 : g_info[slot].spec_bytes;
}

int dedisp_fused_init(void)
{
    if (g_init_done) return DEDISP_OK;
    int rc;
    if ((rc = init_one<1024>(0)) || (rc = init_one<2048>(1)) || (rc = init_one<4096>(2)) || (rc = init_one<8192>(3)) ||
        (rc = init_one<16384>(4)))
        return rc;
    g_init_done = true;
    return DEDISP_OK;
}

int dedisp_launch_fused(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, long long nb, float* d_out,
                        long long out_stride, long long out_col0, cudaStream_t st)
{
    FusedArgs a = base_args(p, d_xt, xt_stride, nb);
    a.out = d_out; a.out_stride = out_stride; a.out_col0 = out_col0;
    return dispatch(p, a, st);
}

int dedisp_launch_debug_voltage(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, int chan,
                                long long block, float* d_volt, cudaStream_t st)
{
    FusedArgs a = base_args(p, d_xt, xt_stride, 0);
    // one unit: (chan, block) with the true blocks-per-channel only needed for u -> (c, b); use nb = block + 1
    a.nb = block + 1;
    a.first_unit = (long long)chan * a.nb + block;
    a.n_units = 1;
    a.volt = reinterpret_cast<float2*>(d_volt);
    return dispatch(p, a, st);
}

int dedisp_launch_debug_unpack(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, int chan,
                               long long block, float* d_block, cudaStream_t st)
{
    debug_unpack_kernel<<<(p->n_fft + 255) / 256, 256, 0, st>>>(d_xt, xt_stride, chan, block * p->L, p->n_fft,
                                                                reinterpret_cast<float2*>(d_block));
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}
