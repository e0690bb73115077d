"""CPU-only checks of the product's host side: the C-ABI library loads without a GPU, exports every symbol that
include/dedisp.h declares, and its pure-host arithmetic (framing, R9) agrees with the oracle's independent restatement.
No compute call is made here."""
import ctypes
import os
import re

import numpy as np
import pytest

import datagen
import oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def dd():
    import __graft_entry__ as g
    g._load_build_script().build_lib()      # nvcc cross-compiles for sm_100a without a GPU
    import paper_1509_00186_b200 as m
    return m


def header_symbols():
    text = open(os.path.join(ROOT, "include", "dedisp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dedisp_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(dd):
    names = header_symbols()
    assert len(names) >= 16
    assert sorted(dd.SYMBOLS) == names, "binding.SYMBOLS and include/dedisp.h disagree"
    lib = ctypes.CDLL(dd.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"libdedisp.so does not export {n}"


def test_library_is_built_for_sm100a_only(dd):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", dd.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


@pytest.mark.parametrize("name", datagen.WORKLOAD_ORDER)
def test_framing_agrees_with_oracle(dd, name):
    w = datagen.WORKLOADS[name]
    cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    assert dd.dedisp_framing(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int) == oracle.framing(cfg)


def test_framing_agrees_with_oracle_on_random_setups(dd):
    rng = np.random.default_rng(7)
    n_ok = 0
    for _ in range(300):
        n_chan = int(rng.choice([1, 3, 64, 256, 512, 2048]))
        dv = float(rng.choice([31.25e3, 62.5e3, 125e3, 250e3]))
        F = float(rng.uniform(120e6, 1400e6))
        n_fft = int(rng.choice([1024, 2048, 4096, 8192, 16384]))
        n_int = int(rng.choice([1, 2, 4, 8, 16, 32, 64, 128]))
        dm = tuple(float(v) for v in rng.uniform(-200, 200, size=int(rng.integers(1, 4))))
        bw = dv * n_chan
        if F - bw / 2 <= 0:
            continue
        cfg = oracle.OracleConfig(n_chan, bw, F, dm, n_fft, n_int)
        try:
            ref = oracle.framing(cfg)
        except ValueError:
            with pytest.raises(dd.DedispError):
                dd.dedisp_framing(n_chan, bw, F, dm, n_fft, n_int)
            continue
        assert dd.dedisp_framing(n_chan, bw, F, dm, n_fft, n_int) == ref
        n_ok += 1
    assert n_ok > 100


def test_framing_rejects_bad_arguments(dd):
    for args in [(0, 16e6, 325e6, (10.0,), 1024, 16), (64, -1.0, 325e6, (10.0,), 1024, 16),
                 (64, 16e6, 7e6, (10.0,), 1024, 16), (64, 16e6, 325e6, (10.0,), 1024, 0),
                 (64, 16e6, 325e6, (float("nan"),), 1024, 16), (64, 16e6, 325e6, (1000.0,), 1024, 16)]:
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_framing(*args)
        assert e.value.code == -1


def test_plan_without_gpu_fails_loudly(dd):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(dd.DedispError) as e:
        dd.dedisp_plan(64, 16e6, 325e6, (10.0,), 1024, 16)
    assert e.value.code == -5      # DEDISP_ENODEV: no fallback of any kind


def test_strerror_covers_every_code(dd):
    for code in range(-5, 1):
        assert dd.lib().dedisp_strerror(code).decode() != "unknown dedisp status"
    assert dd.lib().dedisp_strerror(-99).decode() == "unknown dedisp status"
