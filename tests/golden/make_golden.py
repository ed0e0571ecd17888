"""Writes tests/golden/oracle_checksums.json: 64-bit checksums of the seeded inputs and of the ORACLE's outputs.

    python tests/golden/make_golden.py

Calls only `oracle/` and the input generator (never the CUDA path).  The paper prints no worked numerical
example, so these are not paper values: they freeze the generator and the oracle as
pinned by tests/test_oracle_pins.py, so that a later change to either is noticed ("golden 64-bit
checksums of inputs and of oracle outputs").  A change of the oracle's arithmetic must name the passage of the
paper or the DESIGN.md reading that justifies it and regenerate this file in the same commit.
"""
import hashlib
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import oracle  # noqa: E402
from paper_2001_03389_b200 import synth  # noqa: E402


def digest(a: np.ndarray) -> str:
    return hashlib.blake2b(np.ascontiguousarray(a).tobytes(), digest_size=8).hexdigest()


def cases():
    """(name, config overrides, call) -- small enough for the CPU suite, same generator as the full configs."""
    yield "config1_td", synth.config(1), ("time", [3.0], oracle.MEAN, 0)
    yield "config2_td_beam0_64ch", synth.config(2, beams=1, channels=64), ("time", [5.0, 4.0, 3.0], oracle.MEAN, 0)
    yield "config3_fd_beam0_64ch_2000s", synth.config(3, beams=1, channels=64, samples=2000), ("freq", [4.0, 3.0], oracle.MEAN, 0)
    yield "config2_td_median_w256_16ch", synth.config(2, beams=1, channels=16), ("time", [4.0, 3.0], oracle.MEDIAN, 256)
    # (float32 inputs come from libm's log / cos on the host and are not frozen: integer-only cases only)


def compute():
    out = {}
    for name, cfg, (op, ks, policy, window) in cases():
        x = synth.fill_host(cfg)
        if op == "time":
            y, f, c = oracle.time_sigma_cut(x, ks, policy=policy, window=window)
        else:
            y, f, c = oracle.freq_sigma_cut(x, ks, policy=policy)
        out[name] = {"input": digest(x), "cleaned": digest(y), "flags": digest(f), "counts": [int(v) for v in c]}
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_checksums.json")
    with open(path, "w") as fh:
        json.dump(compute(), fh, indent=1, sort_keys=True)
        fh.write("\n")
    print(path)
