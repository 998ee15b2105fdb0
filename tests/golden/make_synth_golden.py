"""Writes tests/golden/synth_inputs_golden.txt: the first values of every seeded stream the
configs use, so the generators can never drift silently.  Calls only
synth_inputs (numpy); no oracle, no CUDA.   python tests/golden/make_synth_golden.py"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from synth_inputs import normal_bf16, stratified_rows, uniform_pm1  # noqa: E402

out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "synth_inputs_golden.txt")
with open(out, "w") as f:
    f.write("# written by tests/golden/make_synth_golden.py (numpy only)\n")
    for seed in (0, 1):
        v = uniform_pm1(seed, 8).view(np.uint32)
        f.write(f"uniform_pm1 seed={seed} " + " ".join(f"{x:08X}" for x in v) + "\n")
    v = uniform_pm1(1, 4, start=(1 << 28) - 4).view(np.uint32)
    f.write("uniform_pm1_tail seed=1 " + " ".join(f"{x:08X}" for x in v) + "\n")
    for seed, std, stream in ((2, 1.0, 0), (2, 0.02, 1), (3, 1.0, 0), (3, 0.02, 1)):
        v = normal_bf16(seed, (8,), std=std, stream=stream)
        f.write(f"normal_bf16 seed={seed} std={std} stream={stream} " + " ".join(f"{x:04X}" for x in v) + "\n")
    f.write("stratified_rows seed=3 m=4096 " + " ".join(str(x) for x in stratified_rows(3, 4096)[:8]) + "\n")
print(open(out).read())
