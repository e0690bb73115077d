"""GPU parity: the CUDA path (through the C ABI / ctypes binding) against the fp64 oracle on the same seeded inputs.

Tolerances are BASELINE.json:north_star's: per output block (the L/n_int outputs of one (dm, chan, block)) relative L2
error <= 2e-5 and max |diff| <= 1e-3 * block RMS; the int8 unpack must be bit exact."""
import os

import numpy as np
import pytest

import datagen
import oracle

pytestmark = pytest.mark.gpu

REL_L2_TOL = 2e-5     # north_star
MAX_ABS_TOL = 1e-3    # x block RMS, north_star
NT = os.cpu_count() or 1


@pytest.fixture(scope="module")
def dd():
    import paper_1509_00186_b200 as m
    return m


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


def block_errors(got, ref, per):
    """got/ref [n_dm][C][n_out] -> (worst rel-L2, worst max|d|/rms) over output blocks of `per` samples."""
    g = np.asarray(got, dtype=np.float64).reshape(got.shape[0], got.shape[1], -1, per)
    r = np.asarray(ref, dtype=np.float64).reshape(g.shape)
    den = (r ** 2).sum(-1)
    rel = np.sqrt(((g - r) ** 2).sum(-1) / np.where(den > 0, den, 1.0))
    mx = np.abs(g - r).max(-1) / np.sqrt(np.where(den > 0, den / per, 1.0))
    return float(rel.max()), float(mx.max())


def assert_parity(got, ref, per):
    assert got.shape == ref.shape
    rel, mx = block_errors(got, ref, per)
    assert rel <= REL_L2_TOL, f"block rel-L2 {rel:.3e} > {REL_L2_TOL}"
    assert mx <= MAX_ABS_TOL, f"block max|d|/rms {mx:.3e} > {MAX_ABS_TOL}"
    return rel, mx


def make_plan(dd, w, **kw):
    args = dict(n_chan=w.n_chan, bw_hz=w.bw_hz, f_center_hz=w.f_center_hz, dm=w.dm_trials, n_fft=w.n_fft,
                n_int=w.n_int)
    args.update(kw)
    return dd.dedisp_plan(**args)


def ocfg(w, **kw):
    args = dict(n_chan=w.n_chan, bw_hz=w.bw_hz, f_center_hz=w.f_center_hz, dm=w.dm_trials, n_fft=w.n_fft,
                n_int=w.n_int)
    args.update(kw)
    return oracle.OracleConfig(**args)


def run_gpu(torch, plan, x):
    out = plan.execute(torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    return out.cpu().numpy()


# ----------------------------------------------------------------------------------------------------------------
# framing + chirp table
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", datagen.WORKLOAD_ORDER)
def test_plan_framing_matches_oracle(dd, name):
    w = datagen.WORKLOADS[name]
    with make_plan(dd, w) as plan:
        assert (plan.head, plan.tail, plan.L) == oracle.framing(ocfg(w))
        assert plan.info.chan_width_hz == w.bw_hz / w.n_chan


@pytest.mark.parametrize("name,taper", [("tiny", "none"), ("gmrt32", "none"), ("lowfreq", "hann"),
                                        ("wideband", "welch")])
def test_chirp_table_matches_oracle_chirp(dd, name, taper):
    """Table entries are fp32 roundings of taper*exp(2 pi i psi)/N with psi in fp64: error <= 1 ulp-ish of 1/N."""
    w = datagen.WORKLOADS[name]
    cfg = ocfg(w, taper=taper)
    with make_plan(dd, w, taper=taper) as plan:
        for d in sorted({0, plan.n_dm - 1}):
            for c in (0, w.n_chan // 2, w.n_chan - 1):
                h = plan.debug_chirp(d, c) * w.n_fft
                ref = oracle.chirp(cfg, d, c)
                assert np.abs(h - ref).max() <= 2.5e-7, (d, c, np.abs(h - ref).max())


# ----------------------------------------------------------------------------------------------------------------
# unpack + corner turn: bit exact
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_chan,n_samp", [(64, 3000), (8, 2500), (5, 2100), (520, 2049)])
def test_unpack_bit_exact_all_byte_values(dd, torch, n_chan, n_samp):
    x = datagen.uniform_int8(n_samp, n_chan, seed=11)
    x[:256, 0, 0] = np.arange(-128, 128, dtype=np.int8)   # every byte value at known places
    x[:256, n_chan - 1, 1] = np.arange(-128, 128, dtype=np.int8)[::-1]
    dm = (2.0,)
    cfg = oracle.OracleConfig(n_chan, 16e6 * n_chan / 64, 325e6, dm, 1024, 4)
    with dd.dedisp_plan(n_chan, cfg.bw_hz, 325e6, dm, 1024, 4) as plan:
        xd = torch.from_numpy(x).cuda()
        nb = plan.n_blocks(n_samp)
        assert nb == oracle.n_blocks(cfg, n_samp) and nb >= 2
        # dedisp_debug_unpack stores the registers of the FUSED kernel right after its own PRMT/FADD2 conversion
        for c in sorted({0, 1, n_chan // 2, n_chan - 1}):
            for b in range(nb):
                got = plan.debug_unpack(xd, c, b).cpu().numpy()
                ref = oracle.unpack_block(cfg, x, c, b)
                assert np.array_equal(got.astype(np.float64), ref), (c, b)
        got = plan.debug_unpack(xd, 0, 0).cpu().numpy()
        assert np.array_equal(got[:256, 0], np.arange(-128, 128, dtype=np.float32))   # -128 ... 127 at known places


@pytest.mark.parametrize("n_fft", [1024, 2048, 4096, 8192, 16384])
def test_fused_kernel_unpack_bit_exact_every_size(dd, torch, n_fft):
    """The same hook for every built transform size (each has its own staging geometry), on input that holds all 256
    byte values in both components."""
    n_chan = 8
    dm = (1.0,)
    cfg = oracle.OracleConfig(n_chan, 62.5e3 * n_chan, 325e6, dm, n_fft, 4)
    head, tail, L = oracle.framing(cfg)
    n_samp = 5 * L + head + tail + 3
    x = datagen.uniform_int8(n_samp, n_chan, seed=n_fft)
    with dd.dedisp_plan(n_chan, cfg.bw_hz, 325e6, dm, n_fft, 4) as plan:
        xd = torch.from_numpy(x).cuda()
        for c in (0, 3, 7):
            for b in range(5):
                got = plan.debug_unpack(xd, c, b).cpu().numpy()
                assert np.array_equal(got.astype(np.float64), oracle.unpack_block(cfg, x, c, b)), (c, b)


@pytest.mark.parametrize("n_fft,n_int,dm", [(1024, 4, (10.0,)), (4096, 4, (71.0, -20.0)), (16384, 32, (150.0,))])
def test_full_range_int8_input_through_the_chirp(dd, torch, n_fft, n_int, dm):
    """Uniform int8 input (every byte value, -128 included) through the whole path at a non-zero DM: the squares of a
    DM = 0 run cannot tell -128 from +128, the dedispersed voltages can."""
    n_chan = 6
    cfg = oracle.OracleConfig(n_chan, 62.5e3 * n_chan, 325e6 if n_fft < 16384 else 150e6, dm, n_fft, n_int)
    head, tail, L = oracle.framing(cfg)
    x = datagen.uniform_int8(3 * L + head + tail + 11, n_chan, seed=7 * n_fft)
    assert (x == -128).sum() > 100
    ref = oracle.dedisp(cfg, x, n_threads=NT)
    with dd.dedisp_plan(n_chan, cfg.bw_hz, cfg.f_center_hz, dm, n_fft, n_int) as plan:
        assert_parity(run_gpu(torch, plan, x), ref, L // n_int)


def test_dm_zero_is_integer_boxcar_power(dd, torch):
    """P8: DM = 0 => H = 1 => out[j] is the integer sum of re^2+im^2 over rows head + j*n_int ...; pins unpack,
    framing, block stitching, 1/N and the epilogue of the GPU path against a closed form (fp32 rounding only)."""
    n_chan, n_samp, n_int = 24, 9000, 8
    x = datagen.uniform_int8(n_samp, n_chan, seed=5)
    with dd.dedisp_plan(n_chan, 6e6, 325e6, (0.0,), 2048, n_int) as plan:
        got = run_gpu(torch, plan, x)[0]
        head, L = plan.head, plan.L
        n_out = plan.out_samples(n_samp)
    p = (x.astype(np.int64) ** 2).sum(-1)                       # [t][c]
    ref = p[head:head + n_out * n_int].reshape(n_out, n_int, n_chan).sum(1).T
    assert got.shape == ref.shape
    assert np.abs(got / ref - 1.0).max() < 5e-6


# ----------------------------------------------------------------------------------------------------------------
# whole path vs oracle
# ----------------------------------------------------------------------------------------------------------------
def test_tiny_workload_full_parity(dd, torch):
    w = datagen.WORKLOADS["tiny"]
    x = datagen.generate(w)
    ref = oracle.dedisp(ocfg(w), x, n_threads=NT)
    with make_plan(dd, w) as plan:
        got = run_gpu(torch, plan, x)
        rel, mx = assert_parity(got, ref, plan.L // plan.n_int)
    print(f"tiny: rel-L2 {rel:.2e} max/rms {mx:.2e}")


@pytest.mark.parametrize("n_fft,n_int,dm,n_chan,taper", [
    (1024, 16, (10.0,), 7, "none"),
    (1024, 1, (-10.0,), 4, "hann"),
    (2048, 8, (57.0,), 6, "none"),
    (2048, 2, (20.0,), 5, "welch"),
    (4096, 4, (71.0,), 4, "none"),
    (4096, 64, (30.0, -30.0, 0.0), 3, "none"),
    (8192, 32, (100.0,), 3, "none"),
    (16384, 32, (150.0,), 3, "none"),
    (16384, 64, (90.0, 100.0, 107.5), 2, "none"),
    (16384, 128, (50.0,), 2, "hann"),      # n_int > one warp
])
def test_small_cases_full_parity(dd, torch, n_fft, n_int, dm, n_chan, taper):
    """Several blocks + a ragged tail per channel, every built transform size, multi-DM, n_int below/above a warp."""
    bw = 62.5e3 * n_chan
    cfg = oracle.OracleConfig(n_chan, bw, 325e6 if n_fft < 16384 else 150e6, dm, n_fft, n_int, taper)
    head, tail, L = oracle.framing(cfg)
    n_samp = 3 * L + head + tail + 517        # 3 full blocks, ragged tail dropped
    x = datagen.noise_only(n_samp, n_chan, seed=n_fft + n_int)
    ref = oracle.dedisp(cfg, x, n_threads=NT)
    with dd.dedisp_plan(n_chan, bw, cfg.f_center_hz, dm, n_fft, n_int, taper) as plan:
        assert (plan.head, plan.tail, plan.L) == (head, tail, L)
        got = run_gpu(torch, plan, x)
        assert_parity(got, ref, L // n_int)


@pytest.mark.parametrize("n_fft,n_int,dm,n_chan,n_blocks", [
    (4096, 256, (5.0,), 3, 4),          # n_int > 128: the pair kernel's epilogue sums more than 4 samples per lane
    (1024, 256, (0.5,), 9, 5),          # half of every block is overlap, two outputs per block and channel
    (2048, 1, (20.0,), 2, 2),           # no integration at all
    (4096, 4, (71.0,), 1, 1),           # a single (channel, block) unit: one half-empty pair
    (1024, 16, (10.0,), 1, 17),         # one channel, an odd number of blocks, several super-items
    (16384, 1, (100.0,), 1, 1),
])
def test_degenerate_shapes_full_parity(dd, torch, n_fft, n_int, dm, n_chan, n_blocks):
    bw = 62.5e3 * n_chan
    cfg = oracle.OracleConfig(n_chan, bw, 325e6 if n_fft < 16384 else 150e6, dm, n_fft, n_int)
    head, tail, L = oracle.framing(cfg)
    n_samp = n_blocks * L + head + tail          # exactly n_blocks blocks, no tail
    x = datagen.noise_only(n_samp, n_chan, seed=3 * n_fft + n_int)
    ref = oracle.dedisp(cfg, x, n_threads=NT)
    with dd.dedisp_plan(n_chan, bw, cfg.f_center_hz, dm, n_fft, n_int) as plan:
        assert plan.n_blocks(n_samp) == n_blocks and plan.n_blocks(n_samp - 1) == n_blocks - 1
        got = run_gpu(torch, plan, x)
        assert_parity(got, ref, L // n_int)
        if n_blocks > 1:                         # one sample short of the last block: that block must not be written
            out = torch.full((len(dm), n_chan, got.shape[2]), -1.0, dtype=torch.float32, device="cuda")
            plan.execute(torch.from_numpy(x[:-1]).cuda(), out)
            torch.cuda.synchronize()
            o = out.cpu().numpy()
            per = L // n_int
            assert np.array_equal(o[:, :, : (n_blocks - 1) * per], got[:, :, : (n_blocks - 1) * per])
            assert (o[:, :, (n_blocks - 1) * per:] == -1.0).all()


def test_voltage_hook_matches_oracle_voltages(dd, torch):
    w = datagen.WORKLOADS["gmrt32"].scaled(0.2)
    chans = [0, 255, 511]
    x = datagen.generate(w)
    cfg = ocfg(w)
    with make_plan(dd, w) as plan:
        xd = torch.from_numpy(x).cuda()
        nb = plan.n_blocks(x.shape[0])
        for c in chans:
            b = nb - 1
            v = plan.debug_voltage(xd, c, b).cpu().numpy()
            _, ref = oracle.dedisp_units(cfg, x, [c], [b], want_voltage=True)
            got = v[..., 0] + 1j * v[..., 1]
            err = np.linalg.norm(got - ref[0]) / np.linalg.norm(ref[0])
            assert err < 2e-6, (c, err)


def test_errors(dd, torch):
    w = datagen.WORKLOADS["tiny"]
    with pytest.raises(dd.DedispError):
        make_plan(dd, w, n_fft=1000)
    with pytest.raises(dd.DedispError):
        make_plan(dd, w, dm=(100.0,))          # smear longer than the transform
    with pytest.raises(dd.DedispError):
        make_plan(dd, w, n_int=3)              # R9: only powers of two divide a block
    with make_plan(dd, w) as plan:
        short = torch.zeros((100, w.n_chan, 2), dtype=torch.int8, device="cuda")
        with pytest.raises(dd.DedispError) as e:
            plan.execute(short)
        assert e.value.code == -4
        assert plan.out_samples(100) == 0


# ----------------------------------------------------------------------------------------------------------------
# streaming (a6): chunked == one-shot (P10), carry across chunks of awkward lengths
# ----------------------------------------------------------------------------------------------------------------
def stream_run(torch, plan, x, chunk_lens):
    n_samp = x.shape[0]
    total_out = plan.out_samples(n_samp)
    h_out = torch.full((plan.n_dm, plan.n_chan, total_out + 8), float("nan")).pin_memory()
    plan.stream_begin(max(chunk_lens))
    col, t, i = 0, 0, 0
    keep = []
    while t < n_samp:
        n = min(chunk_lens[i % len(chunk_lens)], n_samp - t)
        h_in = torch.from_numpy(x[t:t + n]).clone().pin_memory()
        keep = (keep + [h_in])[-2:]            # h_in may be reused once the next push has returned
        col += plan.stream_push(h_in, h_out, col)
        t += n
        i += 1
    plan.stream_sync()
    plan.stream_end()
    assert col == total_out
    assert torch.isnan(h_out[:, :, total_out:]).all()          # nothing written past the outputs
    return h_out[:, :, :total_out].numpy().copy()


@pytest.mark.parametrize("n_fft,n_int,dm,n_chan,chunks", [
    (1024, 16, (10.0,), 64, (5000,)),
    (1024, 4, (10.0,), 8, (1237, 3001, 411)),          # odd lengths: carry lands on every alignment; 411 < one block
    (4096, 4, (71.0,), 16, (6250,)),                   # gmrt32's 1 s chunk / 10
    (2048, 8, (57.0,), 5, (4099, 2048)),               # n_chan % 8 != 0: scalar corner turn
    (16384, 64, (90.0, 100.0), 8, (40000, 12345)),
])
def test_streaming_equals_one_shot_bitwise(dd, torch, n_fft, n_int, dm, n_chan, chunks):
    bw = 62.5e3 * n_chan
    fc = 325e6 if n_fft < 16384 else 400e6
    with dd.dedisp_plan(n_chan, bw, fc, dm, n_fft, n_int) as plan:
        n_samp = 4 * plan.L + plan.head + plan.tail + 777 if n_fft < 16384 else 5 * plan.L + 999
        x = datagen.noise_only(n_samp, n_chan, seed=n_fft + n_chan)
        one = run_gpu(torch, plan, x)
        got = stream_run(torch, plan, x, chunks)
        assert one.shape == got.shape and one.shape[2] > 0
        assert np.array_equal(one, got)
        # and once more on the same plan: begin() resets the carry
        got2 = stream_run(torch, plan, x, chunks[::-1])
        assert np.array_equal(one, got2)


def test_streaming_against_oracle(dd, torch):
    """The streamed path on a 0.5 s cut of the 32 MHz workload in 0.1 s chunks, against the one-shot oracle."""
    w = datagen.WORKLOADS["gmrt32"].scaled(0.5)
    chans = list(range(0, 512, 16))
    x = datagen.generate(w, chans=chans)
    bw = w.chan_width_hz * len(chans)
    # a 32-channel band with the same channel width; centre chosen so the lowest channel is gmrt32's lowest
    fc = w.f_center_hz - 0.5 * w.bw_hz + 0.5 * bw
    cfg = oracle.OracleConfig(len(chans), bw, fc, w.dm_trials, w.n_fft, w.n_int)
    ref = oracle.dedisp(cfg, x, n_threads=NT)
    with dd.dedisp_plan(len(chans), bw, fc, w.dm_trials, w.n_fft, w.n_int) as plan:
        got = stream_run(torch, plan, x, (6250,))
        assert_parity(got, ref, plan.L // plan.n_int)


def test_stream_errors(dd, torch):
    w = datagen.WORKLOADS["tiny"]
    with make_plan(dd, w) as plan:
        h_in = torch.zeros((2000, w.n_chan, 2), dtype=torch.int8).pin_memory()
        h_out = torch.zeros((1, w.n_chan, 64), dtype=torch.float32).pin_memory()
        with pytest.raises(dd.DedispError):
            plan.stream_push(h_in, h_out)              # no begin
        plan.stream_begin(1000)
        with pytest.raises(dd.DedispError):
            plan.stream_push(h_in, h_out)              # chunk longer than max_chunk_samp
        plan.stream_end()
        plan.stream_begin(2000)
        with pytest.raises(dd.DedispError):
            plan.stream_push(h_in, h_out[:, :, :1].contiguous())   # out_stride too small
        plan.stream_end()


def test_profile_hooks_time_both_kernels(dd, torch):
    w = datagen.WORKLOADS["tiny"]
    x = torch.from_numpy(datagen.noise_only(w.n_samp, w.n_chan, seed=1)).cuda()
    with make_plan(dd, w) as plan:
        plan.profile_enable(True)
        for _ in range(3):
            plan.execute(x)
        a, b, n = plan.profile_read()
        assert n == 3 and a > 0.0 and b > 0.0
        assert plan.profile_read() == (0.0, 0.0, 0)
        plan.profile_enable(False)
        plan.execute(x)
        assert plan.profile_read()[2] == 0


def test_repeated_calls_are_bitwise_identical(dd, torch):
    """Every output is written by exactly one thread from values that only depend on its (dm, channel, block) unit, so
    two calls on the same input must agree bit for bit; a missing barrier or a buffer reused too early would show up
    here (compute-sanitizer is not available on this pool).  Large enough for every CTA to walk several super-items
    with all four groups busy, and to change channel inside a CTA."""
    w = datagen.WORKLOADS["gmrt32"]
    n_chan = 512
    with dd.dedisp_plan(n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int) as plan:
        n_samp = 37 * plan.L + plan.head + plan.tail + 5          # 37 blocks: super-items of 4 leave one block over
        x = torch.from_numpy(datagen.noise_only(n_samp, n_chan, seed=99)).cuda()
        a = plan.execute(x).clone()
        for _ in range(3):
            b = plan.execute(x)
            torch.cuda.synchronize()
            assert torch.equal(a, b)
        # the same blocks computed with a different block-to-group assignment (the input shifted by one block)
        c = plan.execute(x[plan.L:].contiguous())
        torch.cuda.synchronize()
        per = plan.L // plan.n_int
        assert torch.equal(a[:, :, per:], c)


@pytest.mark.parametrize("n_fft,n_int,dm,n_chan", [(4096, 4, (71.0,), 6), (1024, 16, (10.0, 5.0), 9), (16384, 32, (150.0,), 2)])
def test_two_polarisations_add_after_detection(dd, torch, n_fft, n_int, dm, n_chan):
    """SURVEY 8(f) NEXT-4, P:L258 ("combine the signals from the two polarisations after detection"):
    dedisp_execute on polarisation 1, dedisp_execute_add on polarisation 2 == oracle(pol 1) + oracle(pol 2)."""
    bw = 62.5e3 * n_chan
    cfg = oracle.OracleConfig(n_chan, bw, 325e6 if n_fft < 16384 else 150e6, dm, n_fft, n_int)
    head, tail, L = oracle.framing(cfg)
    n_samp = 3 * L + head + tail + 17
    x1 = datagen.noise_only(n_samp, n_chan, seed=1000 + n_fft)
    x2 = datagen.noise_only(n_samp, n_chan, seed=2000 + n_fft)
    ref = oracle.dedisp(cfg, x1, n_threads=NT) + oracle.dedisp(cfg, x2, n_threads=NT)
    with dd.dedisp_plan(n_chan, bw, cfg.f_center_hz, dm, n_fft, n_int) as plan:
        out = plan.execute(torch.from_numpy(x1).cuda())
        plan.execute(torch.from_numpy(x2).cuda(), out, add=True)
        torch.cuda.synchronize()
        assert_parity(out.cpu().numpy(), ref, L // n_int)


def test_execute_is_cuda_graph_capturable(dd, torch):
    """dedisp_execute only enqueues on the caller's stream (no allocation, no synchronisation once the scratch is
    reserved), so a real-time loop can capture it in a CUDA graph and replay it on new data in the same buffers."""
    w = datagen.WORKLOADS["tiny"]
    x1 = torch.from_numpy(datagen.noise_only(w.n_samp, w.n_chan, seed=7)).cuda()
    x2 = torch.from_numpy(datagen.noise_only(w.n_samp, w.n_chan, seed=8)).cuda()
    with make_plan(dd, w) as plan:
        plan.reserve(w.n_samp)
        want1 = plan.execute(x1).clone()
        want2 = plan.execute(x2).clone()
        buf = x1.clone()
        out = torch.empty_like(want1)
        g = torch.cuda.CUDAGraph()
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            plan.execute(buf, out)                       # warm-up on the capture stream
            torch.cuda.synchronize()
            with torch.cuda.graph(g, stream=s):
                plan.execute(buf, out)
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, want1)
        buf.copy_(x2)
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, want2)


def test_gpu_matches_the_frozen_oracle_case(dd, torch):
    """The stored oracle output of tests/golden (fp64, written by a script that calls only oracle/) as a second, frozen
    reference for the CUDA path: Hann taper, a positive and a negative DM, three blocks."""
    from test_oracle_pins import load_frozen_case
    mod, frozen = load_frozen_case()
    cfg, x, _ = mod.compute()
    with dd.dedisp_plan(cfg.n_chan, cfg.bw_hz, cfg.f_center_hz, cfg.dm, cfg.n_fft, cfg.n_int, cfg.taper) as plan:
        got = run_gpu(torch, plan, x)
        assert_parity(got, frozen, plan.L // plan.n_int)
