"""GPU: dedisp_execute_static, the entry point that allocates nothing (its channel-major scratch is a static 64 MiB device
array instead of a cudaMalloc'ed buffer; include/dedisp.h).  Same kernels and arithmetic as dedisp_execute, so its
output must equal the existing path's: checked with the parity tolerances of the other GPU tests AND bitwise, on two
calls in a row (the second on a SHORTER input of another seed, so stale bytes of the first call would show).
This file is named to be collected last: the suite runs with pytest -x."""
import numpy as np
import pytest

import datagen
from test_gpu_parity import assert_parity, dd, make_plan, torch  # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu

STATIC_BYTES = 64 << 20


def test_execute_static_equals_execute_on_two_calls_in_a_row(dd, torch):
    w = datagen.WORKLOADS["tiny"].scaled(0.12)
    with make_plan(dd, w) as plan:
        per = plan.L // plan.n_int
        for call, (seed, n_samp) in enumerate(((11, w.n_samp), (12, w.n_samp - 3 * plan.L - 17))):
            x = datagen.noise_only(n_samp, w.n_chan, seed=seed)
            d_in = torch.from_numpy(x).cuda()
            ref = plan.execute(d_in)                                   # the existing path (allocates its scratch)
            out = torch.full_like(ref, float("nan"))
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            plan.execute_static(d_in, out)
            torch.cuda.synchronize()
            if call == 1:                                             # (the first call may page in lazily loaded code)
                assert torch.cuda.mem_get_info()[0] >= free0          # driver-level: no cudaMalloc behind the call
            assert ref.shape[2] == plan.out_samples(n_samp) and ref.shape[2] % per == 0 and ref.shape[2] > 0
            assert_parity(out.cpu().numpy(), ref.cpu().numpy().astype(np.float64), per)
            assert torch.equal(out, ref), f"call {call}"               # same kernels, same arithmetic


def test_execute_static_multi_dm_and_size_limit(dd, torch):
    # three trial DMs (the spectrum stash belongs to the plan, not to the call)
    w = datagen.WORKLOADS["tiny"].scaled(0.06)
    x = datagen.noise_only(w.n_samp, w.n_chan, seed=13)
    d_in = torch.from_numpy(x).cuda()
    with make_plan(dd, w, dm=(9.0, 10.0, 11.0)) as plan:
        ref = plan.execute(d_in)
        out = torch.empty_like(ref)
        plan.execute_static(d_in, out)
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
    # one sample row too many for the static array: a clear error, nothing launched
    w2 = datagen.WORKLOADS["gmrt32"]
    with make_plan(dd, w2) as plan:
        n_fit = STATIC_BYTES // 2 // w2.n_chan                          # rows of 64-sample granularity that still fit
        nb_fit = (n_fit - plan.head - plan.tail) // plan.L
        n_big = (nb_fit + 1) * plan.L + plan.head + plan.tail
        d_big = torch.zeros((n_big, w2.n_chan, 2), dtype=torch.int8, device="cuda")
        d_out = torch.empty((1, w2.n_chan, plan.out_samples(n_big)), dtype=torch.float32, device="cuda")
        with pytest.raises(dd.DedispError) as e:
            plan.execute_static(d_big, d_out)
        assert e.value.code == -6 and "STATIC_SCRATCH" in str(e.value)
        n_ok = nb_fit * plan.L + plan.head + plan.tail                  # the largest input that fits
        plan.execute_static(d_big[:n_ok], d_out)
        torch.cuda.synchronize()
        assert torch.equal(d_out[:, :, : plan.out_samples(n_ok)], plan.execute(d_big[:n_ok]))
