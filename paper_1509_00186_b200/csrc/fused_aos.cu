// fused_aos.cu -- steps 1b-6 of the path in ONE kernel per call, for every built transform size: unpack -> forward
// FFT -> chirp -> inverse FFT -> overlap discard -> |v|^2 -> integrate (Fig. 4).
// A complex sample is read once from HBM as 2 bytes and leaves as 4/n_int bytes; everything in between stays in
// registers and shared memory.  Every complex number is one packed f32x2 register pair (fft_aos.cuh), so the arithmetic
// is FADD2/FMUL2/FFMA2.  The forward spectrum is computed once per (channel, block) and shared by all trial DMs.
//
// 64 elements per thread (128 data registers, ~190-215 in all), N/64 threads per (channel, block) unit, ONE persistent
// 256-thread CTA per SM holding 256*64/N units at a time (4 at N = 4096), each with its own exchange buffer and barrier
// (a named barrier over the unit's threads; a warp barrier when the unit fits in one warp, N <= 2048).  A 4096-point
// transform is two radix-64 passes with ONE trip through shared memory; with 16 elements per thread and 1024 threads
// (the round-1 shape) it was three passes and two trips, and the shared-memory data pipe was the first limiter
// (profiles/r2_*).  A CTA walks a contiguous range of "super-items" (consecutive blocks of ONE channel, one per unit):
//   * for N <= 4096 the channel's chirp row sits in shared memory and is reloaded only when the channel changes
//     (larger rows do not fit beside the exchange buffers and come from L2);
//   * the int8 rows of the NEXT super-item are prefetched with cp.async while this one computes;
//   * single-DM plans unpack the next super-item beside the epilogue of this one (PIPE below): with two warps per SM
//     sub-partition nothing else hides the shared-memory latency of the epilogue.
// The three control flows (one DM, several DMs, debug hooks) are separate instantiations (MODE), so the hot loop of each
// is straight-line code with the spectrum in fixed registers.
// Barrier discipline (compute-sanitizer is not available on this pool, so it is spelled out): a unit's staging rows
// are written by cp.async issued after the first barrier of the forward transform (every thread of the unit is then
// past its unpack reads: those sit before that transform in program order) and become visible at the barrier between
// the power stores and the power reads of the epilogue (PIPE; cp.async.wait_group 0 before it) or at the barrier that
// ends the super-item (otherwise); the exchange buffer is reused for the detected powers only after the last gather's
// barrier, and for the next transform's scatter only after the epilogue's closing barrier (PIPE: the barrier the
// forward transform places before its first scatter); the chirp row is rewritten between two __syncthreads() that all
// units reach in the same loop iteration.
#include <mutex>
#include <type_traits>

#include "dedisp_internal.h"
#include "fft_aos.cuh"

using namespace dedisp_aos;

namespace {

// N = R0*R1*R2*R3, E elements per thread (N/E threads per unit), CTA threads per block, GROUP = threads that share a
// barrier (a named barrier, or a warp barrier when a unit fits in a warp).
// STAGE: the int8 rows of the next super-item are prefetched into shared memory with cp.async (else read from global
// memory when the unit starts); ROW: single-DM plans keep the channel's chirp row in shared memory (else it comes from
// L2: 8 B x N does not fit beside the exchange buffers for N > 4096).
template <int N, int E> struct AShape;
template <> struct AShape<1024, 64>  { static constexpr int CTA = 256, GROUP = 32,  R0 = 64, R1 = 16, R2 = 1, R3 = 1; };
template <> struct AShape<2048, 64>  { static constexpr int CTA = 256, GROUP = 32,  R0 = 64, R1 = 32, R2 = 1, R3 = 1; };
template <> struct AShape<4096, 64>  { static constexpr int CTA = 256, GROUP = 64,  R0 = 64, R1 = 64, R2 = 1, R3 = 1; };
template <> struct AShape<8192, 64>  { static constexpr int CTA = 256, GROUP = 128, R0 = 64, R1 = 64, R2 = 2, R3 = 1; };
template <> struct AShape<16384, 64> { static constexpr int CTA = 256, GROUP = 256, R0 = 64, R1 = 64, R2 = 4, R3 = 1; };
template <int N, int E> struct Cfg {
    static constexpr int CTA = AShape<N, E>::CTA;
    static constexpr bool STAGE = true, ROW = N <= 4096;
};
constexpr int AOS_E = 64;  // elements per thread of every built size (E = 16 was measured slower on all five workloads)
template <int N, int E> __host__ __device__ constexpr int units_per_super_of() { return Cfg<N, E>::CTA / (N / E); }
template <int N> __host__ __device__ constexpr bool chirp_in_smem() { return N <= 4096; }

struct AosArgs {
    const int8_t* xt;      // [n_chan][xt_stride][2]
    long long xt_stride;   // samples
    const float2* chirp;   // [n_dm][n_chan][N] (c, s), includes 1/N
    const float2* tw;      // [N] exp(-2 pi i m / N)
    float* out;            // [n_dm][n_chan][out_stride]
    long long out_stride, out_col0;
    int accumulate;        // add to out instead of overwriting it (second polarisation)
    float2* spec;          // [gridDim.x][units per super-item][N] forward-spectrum stash, used when n_dm > 1
    float2* volt;          // debug: [n_dm][L] voltages of block volt_block, else nullptr
    int volt_block;
    int dump_unpack;       // debug (with volt != nullptr): store the registers right after unpack_int8x2 as [N] (re, im)
    int nb;                // blocks per channel
    int spc;               // super-items per channel = ceil(nb / units per super-item)
    int n_super;           // super-items to process
    int first_super;       // debug: start here
    int n_chan, n_dm, log2_nint, head, L;
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// biased int8 pair ((re ^ 0x80) | (im ^ 0x80) << 8, as the corner turn stores it: u = x + 128) -> fp32 (re, im), exact,
// without I2F: PRMT builds 0x4B0000uu = 2^23 + u, then one packed add of -(2^23 + 128)
__device__ __forceinline__ C unpack_int8x2(uint32_t w, uint32_t k /* 0x4B000000 */)
{
    uint32_t re, im;
    asm("prmt.b32 %0, %1, %2, 0x7440;" : "=r"(re) : "r"(w), "r"(k));
    asm("prmt.b32 %0, %1, %2, 0x7441;" : "=r"(im) : "r"(w), "r"(k));
    return __fadd2_rn(make_float2(__uint_as_float(re), __uint_as_float(im)), make_float2(-8388736.0f, -8388736.0f));
}
// The PRMT constant, made opaque to the compiler: left to itself it re-creates 0x4B000000 with an HFMA2 (an FP32-pipe
// instruction) before every conversion instead of keeping it in one register.
__device__ __forceinline__ uint32_t magic_2p23()
{
    uint32_t k;
    asm volatile("mov.b32 %0, 0x4B000000;" : "=r"(k));
    return k;
}

template <int N, int E> constexpr size_t smem_bytes()
{
    return (size_t)units_per_super_of<N, E>() *
               (sizeof(float2) * padp<AShape<N, E>::R0>(N) + (Cfg<N, E>::STAGE ? N * sizeof(uint16_t) : 0)) +
           (Cfg<N, E>::ROW ? sizeof(float2) * N : 0);
}

// LGN = log2(n_int) when it is one of the specialised values (the epilogue then has no run-time geometry), else -1.
// MODE: the three control flows are separate instantiations, so that the hot loop of each is straight-line code with
// the spectrum in fixed registers (a merged loop costs ~100 register moves per unit at the join points).
enum { MODE_ONE_DM = 0, MODE_MULTI_DM = 1, MODE_DEBUG = 2 };
template <int N, int E, int LGN, int MODE>
__global__ void __launch_bounds__((Cfg<N, E>::CTA), 1) fused_aos_kernel(const AosArgs a)
{
    using Sh = AShape<N, E>;
    constexpr int CTA = Cfg<N, E>::CTA, GROUP = Sh::GROUP, TPU = N / E, UPS = units_per_super_of<N, E>(), P = Sh::R0;
    constexpr bool CHIRP_SMEM = chirp_in_smem<N>();  // decides the work split (see below)
    constexpr bool STAGE = Cfg<N, E>::STAGE;
    constexpr bool ROW_SMEM = Cfg<N, E>::ROW && MODE == MODE_ONE_DM;  // the channel's chirp row is held in shared memory
    extern __shared__ float2 smem2[];
    const int us = threadIdx.x / TPU;   // unit slot inside the super-item
    const int t = threadIdx.x % TPU;    // thread inside the unit
    const int bar_id = threadIdx.x / GROUP + 1;  // the group's own named barrier
    C* sm = smem2 + (size_t)us * padp<P>(N);                             // exchange buffer of this unit
    float* smf = reinterpret_cast<float*>(sm);                           // ... reused for the detected powers
    float2* chirp_s = smem2 + (size_t)UPS * padp<P>(N);                  // [N], whole CTA (only if CHIRP_SMEM)
    uint16_t* stage = reinterpret_cast<uint16_t*>(chirp_s + (Cfg<N, E>::ROW ? N : 0)) + (size_t)us * N;  // [N] int8 pairs
    const uint16_t* xt16 = reinterpret_cast<const uint16_t*>(a.xt);

    const int lgn = LGN >= 0 ? LGN : a.log2_nint;
    const int n_out = a.L >> lgn;
    // epilogue geometry: each lane sums 2^lg_chunk consecutive samples, 2^lg_lpo lanes (inside one unit's threads and
    // one warp) make one output
    constexpr int MAX_LPO = TPU >= 32 ? 5 : 4;
    const int lg_chunk = lgn < 2 ? lgn : (lgn > 2 + MAX_LPO ? lgn - MAX_LPO : 2);
    const int lg_lpo = lgn - lg_chunk;
    const int n_work = a.L >> lg_chunk;

    // Work split.  Chirp row in shared memory: a contiguous range per CTA, so the row is reloaded only at channel
    // changes.  Chirp row from L2 (N > 4096): super-items dealt round-robin, so that at any moment all CTAs work on the
    // same one or two channels and their chirp rows (8 B x N per trial DM) stay L2-resident instead of 148 different
    // channels' worth of rows thrashing it.
    const int s_step = CHIRP_SMEM ? 1 : (int)gridDim.x;
    const int s_begin = a.first_super + (CHIRP_SMEM ? (int)((long long)blockIdx.x * a.n_super / gridDim.x) : (int)blockIdx.x);
    const int s_end = a.first_super + (CHIRP_SMEM ? (int)((long long)(blockIdx.x + 1) * a.n_super / gridDim.x) : a.n_super);

    // stage the int8 rows of this thread's unit of super-item s: E/8 x 16 B per thread (P:L270 framing: block b reads
    // rows b*L .. b*L+N-1; consecutive blocks overlap)
    auto prefetch = [&](int s) {
        if (!STAGE) return;
        const int c = s / a.spc;
        const int b = (s - c * a.spc) * UPS + us;
        if (b < a.nb) {
            const uint16_t* src = xt16 + (long long)c * a.xt_stride + (long long)b * a.L;
#pragma unroll
            for (int j = 0; j < E / 8; ++j) {
                const int k = (j * TPU + t) * 8;  // 8 samples = 16 B
                cp_async16(stage + k, src + k);
            }
        }
        cp_async_commit();
    };

    int cur_chan = -1;
    if (STAGE && s_begin < s_end) {
        prefetch(s_begin);
        cp_async_wait_all();
        group_bar(bar_id, GROUP);
    }

    // 1b. unpack int8 (re, im) -> fp32 (exact) for this thread's unit of super-item s2
    C x[E];
    const uint32_t k23 = magic_2p23();
    auto unpack = [&](int s2) {
        // (a unit slot past the channel's last block is transformed like the others -- any bytes are valid samples --
        // and only its stores are suppressed: no select per element here)
        if constexpr (STAGE) {
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = unpack_int8x2((uint32_t)stage[t + m * TPU], k23);
        } else {  // block b reads rows b*L .. b*L+N-1 (P:L270 framing)
            const int c2 = s2 / a.spc;
            const int b2 = min((s2 - c2 * a.spc) * UPS + us, a.nb - 1);
            const uint16_t* src = xt16 + (long long)c2 * a.xt_stride + (long long)b2 * a.L + t;
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = unpack_int8x2((uint32_t)__ldg(src + m * TPU), k23);
        }
    };
    // PIPE (single-DM plans): the unpack of the NEXT super-item runs beside the epilogue of this one, whose
    // shared-memory round trip (powers out, barrier, sums in) would otherwise leave the warp idle
    constexpr bool PIPE = MODE == MODE_ONE_DM && STAGE;
    if (PIPE && s_begin < s_end) unpack(s_begin);

    for (int s = s_begin; s < s_end; s += s_step) {
        const int c = s / a.spc;
        const int b = (s - c * a.spc) * UPS + us;
        const bool live = b < a.nb;

        if (ROW_SMEM && c != cur_chan) {  // all groups take this branch in the same iteration
            __syncthreads();
            const float2* row = a.chirp + (size_t)c * N;
            for (int i = threadIdx.x; i < N; i += CTA) chirp_s[i] = __ldg(row + i);
            cur_chan = c;
            __syncthreads();
        }
        // (the staged rows of this super-item are complete and visible: see the barrier that ends the previous one)

        if (!PIPE) unpack(s);
        if (MODE == MODE_DEBUG && a.dump_unpack) {  // debug hook (one super-item): what the transform is about to see
            if (live && a.volt_block == b) {
#pragma unroll
                for (int m = 0; m < E; ++m) a.volt[t + m * TPU] = x[m];
            }
            return;  // uniform over the CTA; no cp.async is in flight (the prefetch is issued in the transform)
        }
        // 2. forward FFT; once every thread of the group is past the unpack, the staging buffer is
        //    free for the next super-item's rows
        fft_aos<E, N, Sh::R0, Sh::R1, Sh::R2, Sh::R3, -1, PIPE>(x, t, sm, a.tw, bar_id, GROUP, [&] {
            if (s + s_step < s_end) prefetch(s + s_step);
        });

        // steps 3-6 for trial DM d on the spectrum in x
        auto dedisperse = [&](int d) {
            // 3. chirp multiply (Eq. 3)
            if (ROW_SMEM) {
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = cmul(x[m], chirp_s[t + m * TPU]);
            } else {
                const float2* hp = a.chirp + ((size_t)d * a.n_chan + c) * N + t;
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = cmul(x[m], __ldg(hp + m * TPU));
            }
            // 4. inverse FFT (1/N already in the chirp)
            fft_aos<E, N, Sh::R0, Sh::R1, Sh::R2, Sh::R3, +1, false>(x, t, sm, a.tw, bar_id, GROUP, [] {});

            if constexpr (MODE == MODE_DEBUG) {  // debug hook: valid voltages of one block
                if (live && a.volt_block == b) {
#pragma unroll
                    for (int m = 0; m < E; ++m) {
                        const int i = t + m * TPU - a.head;
                        if (i >= 0 && i < a.L) a.volt[(size_t)d * a.L + i] = x[m];
                    }
                }
                cp_async_wait_all();
                group_bar(bar_id, GROUP);
            } else {
            // 5 + 6. discard the overlap, detect, integrate n_int samples (R9, R11)
#pragma unroll
            for (int m = 0; m < E; ++m) {
                smf[t + m * TPU] = __fmaf_rn(x[m].y, x[m].y, x[m].x * x[m].x);  // FMUL + FFMA: 2 pipe cycles, not 3
            }
            if (PIPE) cp_async_wait_all();  // the next super-item's rows become visible at this barrier too
            group_bar(bar_id, GROUP);
            float* dst = a.out + ((size_t)d * a.n_chan + c) * a.out_stride + a.out_col0 + (long long)b * n_out;
            if constexpr (LGN >= 2) {
                // chunk id = t + i*TPU holds 4 consecutive powers (one LDS.128); 2^LPO lanes make one output, which
                // lands at (t >> LPO) + i*(TPU >> LPO): base + compile-time stride, no index arithmetic in the loop
                constexpr int LPO = LGN - 2;
                static_assert(LPO <= MAX_LPO, "the lanes of one output sit in one warp and one unit");
                const float4* p4 = reinterpret_cast<const float4*>(smf + a.head) + t;  // head % 4 == 0
                float* dt = dst + (t >> LPO);
                const bool writer = live && (t & ((1 << LPO) - 1)) == 0;
                if (PIPE && s + s_step < s_end) unpack(s + s_step);  // beside the shared-memory reads below
                const int n_full = n_work / TPU, rem = n_work - n_full * TPU;
                constexpr int QS = TPU >> LPO;  // stride of a thread's outputs
                // four chunks per trip: the loads go out together with immediate offsets, the pointers move once, the
                // stores are predicated on one loop-invariant flag; no reconvergence point inside the loop
                auto run = [&](auto acc_tag) {
                    constexpr bool ACC = decltype(acc_tag)::value;
                    const float4* pp = p4;
                    float* q = dt;
                    auto sum4 = [](const float4& u) { return (u.x + u.y) + (u.z + u.w); };
                    auto reduce = [](float v) {
#pragma unroll
                        for (int off = 1; off < (1 << LPO); off <<= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
                        return v;
                    };
                    int i = 0;
#pragma unroll 1
                    for (; i + 4 <= n_full; i += 4) {
                        const float4 u0 = pp[0], u1 = pp[TPU], u2 = pp[2 * TPU], u3 = pp[3 * TPU];
                        const float r0 = reduce(sum4(u0)), r1 = reduce(sum4(u1)), r2 = reduce(sum4(u2)),
                                    r3 = reduce(sum4(u3));
                        if (writer) {
                            if (ACC) { q[0] += r0; q[QS] += r1; q[2 * QS] += r2; q[3 * QS] += r3; }
                            else { q[0] = r0; q[QS] = r1; q[2 * QS] = r2; q[3 * QS] = r3; }
                        }
                        pp += 4 * TPU;
                        q += 4 * QS;
                    }
#pragma unroll 1
                    for (; i < n_full + (rem > 0 ? 1 : 0); ++i) {  // the last trip may be ragged: rem % 2^LPO == 0
                        const bool valid = i < n_full || t < rem;
                        const float r = reduce(valid ? sum4(pp[0]) : 0.f);
                        if (writer && valid) {
                            if (ACC) q[0] += r;
                            else q[0] = r;
                        }
                        pp += TPU;
                        q += QS;
                    }
                };
                if (a.accumulate) run(std::true_type{});
                else run(std::false_type{});
            } else {
                for (int id = t; id - t < n_work; id += TPU) {  // uniform trip count: the shuffles need whole warps
                    float acc = 0.f;
                    if (id < n_work) {
                        const float* p0 = smf + a.head + (id << lg_chunk);  // head % min(n_int, 4) == 0: aligned
                        if (lg_chunk >= 2) {
                            for (int j = 0; j < (1 << lg_chunk); j += 4) {
                                const float4 u = *reinterpret_cast<const float4*>(p0 + j);
                                acc += (u.x + u.y) + (u.z + u.w);
                            }
                        } else if (lg_chunk == 1) {
                            const float2 u = *reinterpret_cast<const float2*>(p0);
                            acc = u.x + u.y;
                        } else {
                            acc = p0[0];
                        }
                    }
                    for (int off = 1; off < (1 << lg_lpo); off <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
                    if (live && id < n_work && (id & ((1 << lg_lpo) - 1)) == 0)
                        dst[id >> lg_lpo] = a.accumulate ? dst[id >> lg_lpo] + acc : acc;
                }
                if (PIPE && s + s_step < s_end) unpack(s + s_step);
            }
            // one barrier for two hand-overs: the powers live in the exchange buffer of the next transform, and the
            // rows prefetched for the next super-item (issued during this one's first exchange) become visible
            if (!PIPE) {  // (PIPE: the forward transform places this barrier before its first scatter)
                cp_async_wait_all();
                group_bar(bar_id, GROUP);
            }
            }
        };

        if constexpr (MODE == MODE_ONE_DM) {
            dedisperse(0);
        } else {
            // the forward spectrum is computed once and shared by all trial DMs: every DM reads it back from the
            // (L2-resident) stash; the same thread wrote it, so no fence is needed
            // (the debug instantiation also serves single-DM plans, which have no stash)
            const bool use_stash = MODE == MODE_MULTI_DM || a.n_dm > 1;
            float2* stash = a.spec + ((size_t)blockIdx.x * UPS + us) * N;
            if (use_stash) {
#pragma unroll
                for (int m = 0; m < E; ++m) stash[t + m * TPU] = x[m];
            }
#pragma unroll 1
            for (int d = 0; d < a.n_dm; ++d) {
                if (use_stash) {
#pragma unroll
                    for (int m = 0; m < E; ++m) x[m] = stash[t + m * TPU];
                }
                dedisperse(d);
            }
        }
    }
}

// Per-device launch geometry.  The dynamic shared memory attribute of a kernel is a per-device setting and the SM count a
// per-device fact, so both are established once per device (under a mutex: plans may be made from several host threads).
struct KernelInfo { int ctas_per_sm; int n_sm; size_t spec_bytes; };
constexpr int MAX_DEVICES = 64;
struct DeviceInfo { bool done; KernelInfo k[5]; };
DeviceInfo g_dev[MAX_DEVICES];
std::mutex g_dev_mutex;

int slot_of(int n_fft)
{
    switch (n_fft) {
        case 1024: return 0; case 2048: return 1; case 4096: return 2; case 8192: return 3; case 16384: return 4;
        default: return -1;
    }
}

// The specialised epilogue is built for the n_int of the BASELINE.json workload of each transform size only (tiny,
// gmrt16, gmrt32, lowfreq / wideband); every other n_int runs the generic epilogue (LGN = -1).
template <int N> constexpr int special_lgn(int which) { return -1; }
template <> constexpr int special_lgn<1024>(int) { return 4; }
template <> constexpr int special_lgn<2048>(int) { return 3; }
template <> constexpr int special_lgn<4096>(int) { return 2; }
template <> constexpr int special_lgn<16384>(int which) { return which == 0 ? 5 : 6; }

template <int N, int LGN, int MODE> int set_smem()
{
    DEDISP_CUDA_TRY(cudaFuncSetAttribute(fused_aos_kernel<N, AOS_E, LGN, MODE>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<N, AOS_E>()));
    return DEDISP_OK;
}
template <int N, int LGN> int set_smem_modes()
{
    int rc;
    if ((rc = set_smem<N, LGN, MODE_ONE_DM>()) || (rc = set_smem<N, LGN, MODE_MULTI_DM>())) return rc;
    return DEDISP_OK;
}

template <int N> int init_one(KernelInfo& k, int dev)
{
    int rc;
    if ((rc = set_smem_modes<N, -1>()) || (rc = set_smem<N, -1, MODE_DEBUG>())) return rc;
    if constexpr (special_lgn<N>(0) >= 0)
        if ((rc = set_smem_modes<N, special_lgn<N>(0)>())) return rc;
    if constexpr (special_lgn<N>(1) != special_lgn<N>(0))
        if ((rc = set_smem_modes<N, special_lgn<N>(1)>())) return rc;
    int occ = 0, n_sm = 0;
    DEDISP_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fused_aos_kernel<N, AOS_E, -1, MODE_MULTI_DM>,
                                                                  Cfg<N, AOS_E>::CTA, smem_bytes<N, AOS_E>()));
    DEDISP_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    k.ctas_per_sm = occ > 0 ? occ : 1;
    k.n_sm = n_sm;
    k.spec_bytes = sizeof(float2) * (size_t)k.ctas_per_sm * n_sm * units_per_super_of<N, AOS_E>() * N;
    return DEDISP_OK;
}

template <int N, int LGN>
void launch_lgn(const AosArgs& a, int n_dm, dim3 g, cudaStream_t st)
{
    const dim3 b(Cfg<N, AOS_E>::CTA);
    constexpr size_t sb = smem_bytes<N, AOS_E>();
    if (n_dm == 1) fused_aos_kernel<N, AOS_E, LGN, MODE_ONE_DM><<<g, b, sb, st>>>(a);
    else fused_aos_kernel<N, AOS_E, LGN, MODE_MULTI_DM><<<g, b, sb, st>>>(a);
}

template <int N>
int launch_one(const dedisp_plan_s* p, AosArgs& a, cudaStream_t st)
{
    const KernelInfo& k = g_dev[p->device].k[slot_of(N)];
    long long grid = (long long)k.ctas_per_sm * k.n_sm;
    if (grid > a.n_super) grid = a.n_super;
    a.spec = p->d_spec;
    const dim3 g((unsigned)grid);
    if (a.volt) {
        fused_aos_kernel<N, AOS_E, -1, MODE_DEBUG><<<g, dim3(Cfg<N, AOS_E>::CTA), smem_bytes<N, AOS_E>(), st>>>(a);
    } else if (special_lgn<N>(0) >= 0 && a.log2_nint == special_lgn<N>(0)) {
        launch_lgn<N, special_lgn<N>(0)>(a, p->n_dm, g, st);
    } else if (special_lgn<N>(1) >= 0 && a.log2_nint == special_lgn<N>(1)) {
        launch_lgn<N, special_lgn<N>(1)>(a, p->n_dm, g, st);
    } else {
        launch_lgn<N, -1>(a, p->n_dm, g, st);
    }
    DEDISP_CUDA_TRY(cudaGetLastError());
    return DEDISP_OK;
}

int dispatch(const dedisp_plan_s* p, AosArgs& a, cudaStream_t st)
{
    // the kernels, their shared-memory attributes and the plan's tables all belong to the plan's device
    int dev = -1;
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != p->device || dev < 0 || dev >= MAX_DEVICES || !g_dev[dev].done) return DEDISP_EINVAL;
    switch (p->n_fft) {
        case 1024: return launch_one<1024>(p, a, st);
        case 2048: return launch_one<2048>(p, a, st);
        case 4096: return launch_one<4096>(p, a, st);
        case 8192: return launch_one<8192>(p, a, st);
        case 16384: return launch_one<16384>(p, a, st);
        default: return DEDISP_EINVAL;
    }
}

int units_per_super(int n_fft)
{
    switch (n_fft) {
        case 1024: return units_per_super_of<1024, AOS_E>(); case 2048: return units_per_super_of<2048, AOS_E>();
        case 4096: return units_per_super_of<4096, AOS_E>(); case 8192: return units_per_super_of<8192, AOS_E>();
        default: return units_per_super_of<16384, AOS_E>();
    }
}

int base_args(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, long long nb, AosArgs& a)
{
    const long long ups = units_per_super(p->n_fft), spc = (nb + ups - 1) / ups;
    if (nb > 0x3fffffff || spc * p->n_chan > 0x7fffffff) return DEDISP_EINVAL;  // 32-bit item arithmetic in the kernel
    a = AosArgs{};
    a.xt = d_xt; a.xt_stride = xt_stride; a.chirp = p->d_chirp; a.tw = p->d_twiddle;
    a.nb = (int)nb; a.spc = (int)spc; a.n_super = (int)(spc * p->n_chan); a.first_super = 0;
    a.n_chan = p->n_chan; a.n_dm = p->n_dm; a.head = p->head; a.L = p->L;
    int lg = 0;
    while ((1 << lg) < p->n_int) ++lg;
    a.log2_nint = lg;
    return DEDISP_OK;
}

}  // namespace

int dedisp_aos_supported(int n_fft) { return slot_of(n_fft) >= 0; }

size_t dedisp_aos_spec_bytes(int n_fft)
{
    int dev = -1;
    const int slot = slot_of(n_fft);
    if (slot < 0 || cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES || !g_dev[dev].done) return 0;
    return g_dev[dev].k[slot].spec_bytes;
}

int dedisp_aos_init(void)
{
    int dev = -1;
    DEDISP_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return DEDISP_ENODEV;
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    DeviceInfo& d = g_dev[dev];
    if (d.done) return DEDISP_OK;
    int rc;
    if ((rc = init_one<1024>(d.k[0], dev)) || (rc = init_one<2048>(d.k[1], dev)) || (rc = init_one<4096>(d.k[2], dev)) ||
        (rc = init_one<8192>(d.k[3], dev)) || (rc = init_one<16384>(d.k[4], dev)))
        return rc;
    d.done = true;
    return DEDISP_OK;
}

int dedisp_launch_aos(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, long long nb, float* d_out,
                      long long out_stride, long long out_col0, int accumulate, cudaStream_t st)
{
    AosArgs a;
    int rc = base_args(p, d_xt, xt_stride, nb, a);
    if (rc != DEDISP_OK) return rc;
    a.out = d_out; a.out_stride = out_stride; a.out_col0 = out_col0; a.accumulate = accumulate;
    return dispatch(p, a, st);
}

int dedisp_launch_aos_debug_voltage(const dedisp_plan_s* p, const int8_t* d_xt, long long xt_stride, int chan,
                                    long long block, float* d_volt, int dump_unpack, cudaStream_t st)
{
    // the one super-item that holds (chan, block); blocks-per-channel = block + 1 is enough to address it
    AosArgs a;
    int rc = base_args(p, d_xt, xt_stride, block + 1, a);
    if (rc != DEDISP_OK) return rc;
    a.first_super = chan * a.spc + (int)(block / units_per_super(p->n_fft));
    a.n_super = 1;
    a.volt = reinterpret_cast<float2*>(d_volt);
    a.volt_block = (int)block;
    a.dump_unpack = dump_unpack;
    return dispatch(p, a, st);
}
