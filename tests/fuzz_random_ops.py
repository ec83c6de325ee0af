"""Fuzz campaign over tests/test_gpu_random_ops.py (a campaign driver; tests/test_gpu_fuzz.py runs a bounded, fixed-seed slice of it): N seeded random operation sequences with
random geometry (head_dim 64 / 128 / 256, GQA group, page size, rope mode) on the CUDA library and the oracle side by side.

    python tests/fuzz_random_ops.py <campaign seed> <number of sequences>        (needs a GPU)
"""
import os
import sys
import traceback

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)
import test_gpu_random_ops as R  # noqa: E402


def main(campaign_seed: int, n: int) -> int:
    rng = np.random.default_rng(campaign_seed)
    fails = 0
    for _ in range(n):
        seed = int(rng.integers(1000, 10 ** 6))
        D = int(rng.choice([64, 128, 256, 16, 48, 80, 96, 112, 160, 192, 224]))
        Hq, Hkv = [(4, 2), (4, 4), (8, 2), (2, 1), (6, 2)][int(rng.integers(5))]
        P = int(rng.choice([8, 16, 32, 64]))
        rope_mode = int(rng.integers(3))
        try:
            R.test_random_operation_sequences(seed, D, Hq, Hkv, P, rope_mode)
        except Exception as e:  # keep going: report every failing parameter set
            fails += 1
            print("FAIL", (seed, D, Hq, Hkv, P, rope_mode), repr(e)[:300], flush=True)
            traceback.print_exc()
    print(f"done: {n} sequences, {fails} failures")
    return fails


if __name__ == "__main__":
    sys.exit(1 if main(int(sys.argv[1]), int(sys.argv[2])) else 0)
