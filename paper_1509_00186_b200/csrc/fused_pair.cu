// fused_pair.cu -- steps 1b-6 of the path for N_fft <= 4096 on packed f32x2 arithmetic: every thread carries TWO
// overlap-save blocks of one channel (unit A in lane .x, unit B in lane .y of each packed register, fft_pair.cuh), so
// unpack -> forward FFT -> chirp -> inverse FFT -> |v|^2 run as FADD2/FMUL2/FFMA2 with shared twiddles, chirp values
// and index arithmetic (Fig. 4).  HBM traffic is unchanged: 2 B in, 4/n_int B out
// per complex sample.
//
// One persistent 512-thread CTA per SM = 2 groups of 256 threads; a group owns P pairs (1/2/4 for N = 4096/2048/1024),
// its exchange buffers and a named barrier, so the two groups run out of phase and fill each other's barrier and
// memory stalls.  A CTA walks a contiguous range of "super-items" (2P pairs of ONE channel):
//   * the channel's chirp row sits in shared memory and is reloaded only when the channel changes (every ~60 items);
//   * the int8 input of the NEXT super-item is prefetched with cp.async into a staging buffer while this one computes.
#include "dedisp_internal.h"
#include "fft_pair.cuh"

using namespace dedisp_pair;

namespace {

constexpr int GROUP = 256;  // threads that share a named barrier
constexpr int GROUPS = 2;   // groups per CTA

template <int N> struct PShape;  // P = pairs per group; N = R0*R1*R2
template <> struct PShape<1024> { static constexpr int P = 4, R0 = 16, R1 = 16, R2 = 4; };
template <> struct PShape<2048> { static constexpr int P = 2, R0 = 16, R1 = 16, R2 = 8; };
template <> struct PShape<4096> { static constexpr int P = 1, R0 = 16, R1 = 16, R2 = 16; };

struct PairArgs {
    const int8_t* xt;      // [n_chan][xt_stride][2]
    long long xt_stride;   // samples
    const float2* chirp;   // [n_dm][n_chan][N] (c, s), includes 1/N
    const float2* tw;      // [N] exp(-2 pi i m / N)
    float* out;            // [n_dm][n_chan][out_stride]
    long long out_stride, out_col0;
    float4* spec;          // [gridDim.x][2P][N] forward-spectrum stash, used when n_dm > 1
    float2* volt;          // debug: [n_dm][L] voltages of block volt_block, else nullptr
    int volt_block;
    int nb;                // blocks per channel
    int ppc;               // pairs per channel = ceil(nb / 2)
    int spc;               // super-items per channel = ceil(ppc / 2P)
    int n_super;           // super-items to process
    int first_super;       // debug: start here
    int n_chan, n_dm, log2_nint, head, L;
};

// 8-byte power cells (pA, pB) in shared memory; 16-byte units are XOR-swizzled so that the epilogue's LDS.128 at a
// stride of two units (four consecutive samples per lane) and the STS.64 of consecutive cells are both conflict free.
__device__ __forceinline__ int pw_cell(int cell)
{
    const int u = cell >> 1;
    return ((u ^ ((u >> 3) & 1)) << 1) | (cell & 1);
}

// byte `sel & 3` of w under the exponent byte of k = 0x4B000000: the fp32 number 2^23 + byte
__device__ __forceinline__ float byte_to_f32_biased(uint32_t w, uint32_t k, int sel)
{
    uint32_t r;
    switch (sel) {
        case 0: asm("prmt.b32 %0, %1, %2, 0x7440;" : "=r"(r) : "r"(w), "r"(k)); break;
        case 1: asm("prmt.b32 %0, %1, %2, 0x7441;" : "=r"(r) : "r"(w), "r"(k)); break;
        case 2: asm("prmt.b32 %0, %1, %2, 0x7442;" : "=r"(r) : "r"(w), "r"(k)); break;
        default: asm("prmt.b32 %0, %1, %2, 0x7443;" : "=r"(r) : "r"(w), "r"(k)); break;
    }
    return __uint_as_float(r);
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int N> constexpr size_t smem_bytes()
{
    return (size_t)GROUPS * PShape<N>::P * (sizeof(float4) * padded_len(N) + 2 * N * sizeof(uint16_t)) + sizeof(float2) * N;
}

// LGN = log2(n_int) when it is one of the specialised values (the epilogue then has no run-time geometry), else -1.
template <int N, int LGN>
__global__ void __launch_bounds__(GROUP * GROUPS, 1) fused_pair_kernel(const PairArgs a)
{
    using Sh = PShape<N>;
    constexpr int P = Sh::P, TPU = N / 16, PPS = GROUPS * P;
    extern __shared__ float4 smem4[];
    const int g = threadIdx.x / GROUP;            // group: its own barrier
    const int ps = threadIdx.x / TPU;             // pair slot inside the super-item (g*P + pair in group)
    const int t = threadIdx.x % TPU;              // thread inside the pair
    const int bar_id = g + 1;
    float4* sm = smem4 + (size_t)ps * padded_len(N);                          // exchange buffer of this pair
    float2* smp = reinterpret_cast<float2*>(sm);                              // ... reused for the power cells
    float2* chirp_s = reinterpret_cast<float2*>(smem4 + (size_t)PPS * padded_len(N));  // [N], whole CTA
    uint16_t* stage = reinterpret_cast<uint16_t*>(chirp_s + N) + (size_t)ps * 2 * N;   // [2][N] int8 pairs: A, B
    const uint16_t* xt16 = reinterpret_cast<const uint16_t*>(a.xt);

    const int lgn = LGN >= 0 ? LGN : a.log2_nint;
    const int n_out = a.L >> lgn;
    // epilogue geometry: each lane sums 2^lg_chunk consecutive samples, 2^lg_lpo lanes make one output
    const int lg_chunk = lgn < 2 ? lgn : (lgn > 7 ? lgn - 5 : 2);
    const int lg_lpo = lgn - lg_chunk;
    const int n_work = a.L >> lg_chunk;

    const int s_begin = a.first_super + (int)((long long)blockIdx.x * a.n_super / gridDim.x);
    const int s_end = a.first_super + (int)((long long)(blockIdx.x + 1) * a.n_super / gridDim.x);

    // stage the int8 rows of this thread's pair of super-item s: 2 x 16 B per unit and thread (P:L270 framing: block b
    // reads rows b*L .. b*L+N-1; consecutive blocks overlap)
    auto prefetch = [&](int s) {
        const int c = s / a.spc;
        const int pr = (s - c * a.spc) * PPS + ps;
        const int bA = 2 * pr;
        const uint16_t* src = xt16 + (long long)c * a.xt_stride + (long long)bA * a.L;
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (bA + u < a.nb) {
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int k = (j * TPU + t) * 8;  // 8 samples = 16 B
                    cp_async16(stage + u * N + k, src + (long long)u * a.L + k);
                }
            }
        }
        cp_async_commit();
    };

    int cur_chan = -1;
    if (s_begin < s_end) {
        prefetch(s_begin);
        cp_async_wait_all();
        group_bar(bar_id, GROUP);
    }

    for (int s = s_begin; s < s_end; ++s) {
        const int c = s / a.spc;
        const int pr = (s - c * a.spc) * PPS + ps;
        const int bA = 2 * pr;
        const bool live = bA < a.nb, liveB = bA + 1 < a.nb;

        if (a.n_dm == 1 && c != cur_chan) {  // both groups take this branch in the same iteration
            __syncthreads();
            const float2* row = a.chirp + (size_t)c * N;
            for (int i = threadIdx.x; i < N; i += GROUP * GROUPS) chirp_s[i] = __ldg(row + i);
            cur_chan = c;
            __syncthreads();
        }
        // (the staged rows of this super-item are complete and visible: see the barrier that ends the previous one)

        // 1b. unpack int8 (re, im) -> fp32, exact: bytes -> 0x4B0000uu (= 2^23 + u, u = x + 128) -> minus (2^23 + 128)
        C2 x[16];
#pragma unroll
        for (int m = 0; m < 16; ++m) {
            const uint32_t vA = live ? (uint32_t)stage[t + m * TPU] : 0u;
            const uint32_t vB = liveB ? (uint32_t)stage[N + t + m * TPU] : 0u;
            const uint32_t w = __byte_perm(vA, vB, 0x5410) ^ 0x80808080u;  // (A.re, A.im, B.re, B.im) + 128
            const V re = make_float2(byte_to_f32_biased(w, 0x4B000000u, 0), byte_to_f32_biased(w, 0x4B000000u, 2));
            const V im = make_float2(byte_to_f32_biased(w, 0x4B000000u, 1), byte_to_f32_biased(w, 0x4B000000u, 3));
            x[m].re = vadd(re, vdup(-8388736.0f));
            x[m].im = vadd(im, vdup(-8388736.0f));
        }
        // 2. forward FFT; once every thread of the group is past the unpack, the staging buffer is
        //    free for the next super-item's rows
        fft_pair<N, Sh::R0, Sh::R1, Sh::R2, -1>(x, t, sm, a.tw, bar_id, GROUP, [&] {
            if (s + 1 < s_end) prefetch(s + 1);
        });

        float4* stash = a.spec + ((size_t)blockIdx.x * PPS + ps) * N;
        if (a.n_dm > 1) {
#pragma unroll
            for (int m = 0; m < 16; ++m)
                stash[t + m * TPU] = make_float4(x[m].re.x, x[m].re.y, x[m].im.x, x[m].im.y);
        }
        for (int d = 0; d < a.n_dm; ++d) {
            if (d > 0) {
#pragma unroll
                for (int m = 0; m < 16; ++m) {  // same thread wrote it: no fence needed
                    const float4 v = stash[t + m * TPU];
                    x[m] = C2{make_float2(v.x, v.y), make_float2(v.z, v.w)};
                }
            }
            // 3. chirp multiply (Eq. 3): both blocks of the pair share the channel's chirp
            if (a.n_dm == 1) {
#pragma unroll
                for (int m = 0; m < 16; ++m) {
                    const float2 hv = chirp_s[t + m * TPU];
                    x[m] = cmul(x[m], C2{vdup(hv.x), vdup(hv.y)});
                }
            } else {
                const float2* h = a.chirp + ((size_t)d * a.n_chan + c) * N + t;
#pragma unroll
                for (int m = 0; m < 16; ++m) {
                    const float2 hv = __ldg(h + m * TPU);
                    x[m] = cmul(x[m], C2{vdup(hv.x), vdup(hv.y)});
                }
            }
            // 4. inverse FFT (1/N already applied)
            fft_pair<N, Sh::R0, Sh::R1, Sh::R2, +1>(x, t, sm, a.tw, bar_id, GROUP, [] {});

            if (a.volt) {  // debug hook: valid voltages of one block
                if (live && (a.volt_block >> 1) == pr) {
                    const bool second = a.volt_block & 1;
#pragma unroll
                    for (int m = 0; m < 16; ++m) {
                        const int i = t + m * TPU - a.head;
                        if (i >= 0 && i < a.L)
                            a.volt[(size_t)d * a.L + i] = second ? make_float2(x[m].re.y, x[m].im.y)
                                                                 : make_float2(x[m].re.x, x[m].im.x);
                    }
                }
                cp_async_wait_all();
                group_bar(bar_id, GROUP);
                continue;
            }
            // 5 + 6. discard the overlap, detect, integrate n_int samples (R9, R11)
            {
                float2* cell = smp + pw_cell(t);  // TPU/2 is a multiple of 16 units: pw_cell(t + m*TPU) = pw_cell(t) + m*TPU
#pragma unroll
                for (int m = 0; m < 16; ++m) cell[m * TPU] = vfma(x[m].re, x[m].re, vmul(x[m].im, x[m].im));
            }
            group_bar(bar_id, GROUP);
            float* dstA = a.out + ((size_t)d * a.n_chan + c) * a.out_stride + a.out_col0 + (long long)bA * n_out;
            float* dstB = dstA + n_out;
            for (int id = t; id - t < n_work; id += TPU) {  // uniform trip count: the shuffles need whole warps
                V acc = make_float2(0.f, 0.f);
                if (id < n_work) {
                    const int cell0 = a.head + (id << lg_chunk);
                    if (lg_chunk >= 2) {
                        for (int j = 0; j < (1 << lg_chunk); j += 4) {
                            const float4 u0 = *reinterpret_cast<const float4*>(&smp[pw_cell(cell0 + j)]);
                            const float4 u1 = *reinterpret_cast<const float4*>(&smp[pw_cell(cell0 + j + 2)]);
                            const V s0 = vadd(make_float2(u0.x, u0.y), make_float2(u0.z, u0.w));
                            const V s1 = vadd(make_float2(u1.x, u1.y), make_float2(u1.z, u1.w));
                            acc = vadd(acc, vadd(s0, s1));
                        }
                    } else if (lg_chunk == 1) {
                        const float4 u0 = *reinterpret_cast<const float4*>(&smp[pw_cell(cell0)]);
                        acc = vadd(make_float2(u0.x, u0.y), make_float2(u0.z, u0.w));
                    } else {
                        acc = smp[pw_cell(cell0)];
                    }
                }
                for (int off = 1; off < (1 << lg_lpo); off <<= 1) {
                    acc.x += __shfl_xor_sync(0xffffffffu, acc.x, off);
                    acc.y += __shfl_xor_sync(0xffffffffu, acc.y, off);
                }
                if (id < n_work && (id & ((1 << lg_lpo) - 1)) == 0) {
                    const int o = id >> lg_lpo;
                    if (live) dstA[o] = acc.x;
                    if (liveB) dstB[o] = acc.y;
                }
            }
            // one barrier for two hand-overs: the power cells live in the exchange buffer of the next transform, and the
            // rows prefetched for the next super-item (issued during this one's first exchange) are now visible
            cp_async_wait_all();
            group_bar(bar_id, GROUP);
        }
    }
}

struct KernelInfo { int ctas_per_sm; int n_sm; size_t spec_bytes; };
KernelInfo g_info[3];
bool g_init_done = false;

int slot_of(int n_fft) { return n_fft == 1024 ? 0 : n_fft == 2048 ? 1 : n_fft == 4096 ? 2 : -1; }

template <int N> int init_one(int slot)
{
    DEDISP_CUDA_TRY(cudaFuncSetAttribute(fused_pair_kernel<N, -1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem_bytes<N>()));
    DEDISP_CUDA_TRY(cudaFuncSetAttribute(fused_pair_kernel<N, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem_bytes<N>()));
    DEDISP_CUDA_TRY(cudaFuncSetAttribute(fused_pair_kernel<N, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem_bytes<N>()));
    DEDISP_CUDA_TRY(cudaFuncSetAttribute(fused_pair_kernel<N, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem_bytes<N>()));
    int occ = 0;
    DEDISP_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fused_pair_kernel<N, -1>, GROUP * GROUPS,
                                                                  smem_bytes<N>()));
    int dev = 0, n_sm = 0;
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    DEDISP_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    g_info[slot].ctas_per_sm = occ > 0 ? occ : 1;
    g_info[slot].n_sm = n_sm;
    g_info[slot].spec_bytes = sizeof(float4) * (size_t)g_info[slot].ctas_per_sm * n_sm * GROUPS * PShape<N>::P * N;
    return DEDISP_OK;
}

template <int N>
int launch_one(const dedisp_plan_s* p, PairArgs& a, cudaStream_t st)
{
    const int slot = slot_of(N);
    long long grid = (long long)g_info[slot].ctas_per_sm * g_info[slot].n_sm;
    if (grid > a.n_super) grid = a.n_super;
    a.spec = reinterpret_cast<float4*>(p->d_spec);
    const dim3 g((unsigned)grid), b(GROUP * GROUPS);
    switch (a.volt ? -1 : a.log2_nint) {  // n_int = 4, 8, 16 (the 32/16 MHz and Tiny configs) are specialised
        case 2: fused_pair_kernel<N, 2><<<g, b, smem_bytes<N>(), st>>>(a); break;
        case 3: fused_pair_kernel<N, 3><<<g, b, smem_bytes<N>(), st>>>(a); break;
        case 4: fused_pair_kernel<N, 4><<<g, b, smem_bytes<N>(), st>>>(a); break;
        default: fused_pair_kernel<N, -1><<<g, b, smem_bytes<N>(), st>>>(a); break;
    }
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}

int dispatch(const dedisp_plan_s* p, PairArgs& a, cudaStream_t st)
{
    switch (p->n_fft) {
        case 1024: return launch_one<1024>(p, a, st);
        case 2048: return launch_one<2048>(p, a, st);
        case 4096: return launch_one<4096>(p, a, st);
        default: return DEDISP_EINVAL;
    }
}

int pairs_per_super(int n_fft) { return GROUPS * (n_fft == 1024 ? 4 : n_fft == 2048 ? 2 : 1); }

int base_args(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, long long nb, PairArgs& a)
{
    const long long ppc = (nb + 1) / 2, pps = pairs_per_super(p->n_fft), spc = (ppc + pps - 1) / pps;
    if (nb > 0x3fffffff || spc * p->n_chan > 0x7fffffff) return DEDISP_EINVAL;  // 32-bit item arithmetic in the kernel
    a = PairArgs{};
    a.xt = d_xt; a.xt_stride = xt_stride; a.chirp = p->d_chirp; a.tw = p->d_twiddle;
    a.nb = (int)nb; a.ppc = (int)ppc; a.spc = (int)spc; a.n_super = (int)(spc * p->n_chan); a.first_super = 0;
    a.n_chan = p->n_chan; a.n_dm = p->n_dm; a.head = p->head; a.L = p->L;
    int lg = 0;
    while ((1 << lg) < p->n_int) ++lg;
    a.log2_nint = lg;
    return DEDISP_OK;
}

}  // namespace

int dedisp_pair_supported(int n_fft) { return slot_of(n_fft) >= 0; }

size_t dedisp_pair_spec_bytes(int n_fft)
{
    const int slot = slot_of(n_fft);
    return slot < 0 ? 0 : g_info[slot].spec_bytes;
}

int dedisp_pair_init(void)
{
    if (g_init_done) return DEDISP_OK;
    int rc;
    if ((rc = init_one<1024>(0)) || (rc = init_one<2048>(1)) || (rc = init_one<4096>(2))) return rc;
    g_init_done = true;
    return DEDISP_OK;
}

int dedisp_launch_pair(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, long long nb, float* d_out,
                       long long out_stride, long long out_col0, cudaStream_t st)
{
    PairArgs a;
    int rc = base_args(p, d_xt, xt_stride, nb, a);
    if (rc != DEDISP_OK) return rc;
    a.out = d_out; a.out_stride = out_stride; a.out_col0 = out_col0;
    return dispatch(p, a, st);
}

int dedisp_launch_pair_debug_voltage(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, int chan,
                                     long long block, float* d_volt, cudaStream_t st)
{
    // the one super-item that holds (chan, block); blocks-per-channel = block + 1 is enough to address it
    PairArgs a;
    int rc = base_args(p, d_xt, xt_stride, block + 1, a);
    if (rc != DEDISP_OK) return rc;
    a.first_super = chan * a.spc + (int)(block / 2) / pairs_per_super(p->n_fft);
    a.n_super = 1;
    a.volt = reinterpret_cast<float2*>(d_volt);
    a.volt_block = (int)block;
    return dispatch(p, a, st);
}
