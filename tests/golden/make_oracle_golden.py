"""Writes tests/golden/oracle_small_case.txt: the fp64 oracle's output on one small seeded case.

Calls only oracle/ and datagen/ (never the CUDA path).  The stored values guard the oracle against silent changes of
its arithmetic (a change that moves them must name the paper passage or DESIGN.md reading that justifies it in its
commit message) and give the GPU tests a second, frozen reference.
    python tests/golden/make_oracle_golden.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import datagen  # noqa: E402
import oracle  # noqa: E402

CASE = dict(n_chan=2, bw_hz=500e3, f_center_hz=325e6, dm=(10.0, -4.0), n_fft=1024, n_int=16, taper="hann")
N_BLOCKS, SEED = 3, 20240


def compute():
    cfg = oracle.OracleConfig(**CASE)
    head, tail, L = oracle.framing(cfg)
    x = datagen.noise_only(N_BLOCKS * L + head + tail + 9, CASE["n_chan"], seed=SEED)
    return cfg, x, oracle.dedisp(cfg, x)


if __name__ == "__main__":
    cfg, x, out = compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_small_case.txt")
    with open(path, "w") as fh:
        fh.write("# fp64 oracle output [n_dm][n_chan][n_out] of the case defined in make_oracle_golden.py\n")
        fh.write("# (Hann taper, DMs +10 and -4, N_fft 1024, n_int 16, 3 blocks, seeded int8 noise); row-major, one value per line\n")
        fh.write(f"# shape {out.shape[0]} {out.shape[1]} {out.shape[2]}\n")
        for v in out.reshape(-1):
            fh.write(f"{v:.17e}\n")
    print(path, out.shape)
