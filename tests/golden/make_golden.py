"""Writes tests/golden/oracle_c1_c3.txt: the ORACLE's loss and a few sampled gradient entries for two small seeded
cases.  Calls only `oracle/` and the seeded generator (never the CUDA path).  The paper prints no worked numeric
example (README.md here), so these are regression fixtures: `tests/test_golden.py` checks that the oracle still
reproduces them (-m "not gpu") and that the CUDA path matches the same stored numbers (-m gpu).

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, ".."))
sys.path.insert(0, os.path.join(HERE, "..", ".."))

from cases import make_case, oracle_grad  # noqa: E402
from paper_2505_07814_b200 import synth  # noqa: E402

CASES = [("c1A", 1, "A", 6), ("c3A", 3, "A", 3)]      # name, config, evaluation point, positions
N_SAMPLES = 12


def sample_indices(shape, seed):
    rng = np.random.default_rng(seed)
    return [tuple(int(rng.integers(0, n)) for n in shape) for _ in range(N_SAMPLES)]


def case_and_ref(c, which, B):
    cfg = synth.get_config(c)
    case = make_case(c, which, synth.minibatch(cfg, 0, cfg.B)[:B])
    return case, oracle_grad(case, workers=1)


def main():
    lines = ["# written by tests/golden/make_golden.py from oracle/ (float64); name key index... value(s)"]
    for name, c, which, B in CASES:
        case, ref = case_and_ref(c, which, B)
        lines.append(f"{name} loss {ref['loss']!r}")
        for key in ("g_object", "g_probe", "g_positions"):
            arr = np.asarray(ref[key])
            lines.append(f"{name} norm_{key} {float(np.linalg.norm(arr))!r}")
            # object samples only inside the first position's patch (elsewhere the gradient is exactly 0)
            for idx in sample_indices(arr.shape, 17 * c + len(key)):
                if key == "g_object":
                    y0, x0 = (int(np.floor(v + 0.5)) for v in case["positions"][0])
                    idx = (idx[0], y0 + idx[1] % case["cfg"].N, x0 + idx[2] % case["cfg"].N)
                v = arr[idx]
                vals = f"{float(np.real(v))!r} {float(np.imag(v))!r}" if np.iscomplexobj(arr) else f"{float(v)!r}"
                lines.append(f"{name} {key} {','.join(map(str, idx))} {vals}")
    with open(os.path.join(HERE, "oracle_c1_c3.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")
    print(f"wrote {len(lines)} lines")


if __name__ == "__main__":
    main()
