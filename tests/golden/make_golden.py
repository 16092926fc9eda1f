"""Writes tests/golden/odirect_tiny.txt from the CPU oracle only (never from the CUDA path)."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle      # noqa: E402
import workloads   # noqa: E402

N, NA, ND = 12, 7, 13


def compute():
    x = workloads.white_noise(N, 4242).astype(np.float64)
    S = oracle.forward(x, NA, ND)
    A = oracle.adjoint(S, N)
    return np.concatenate([S.ravel(), A.ravel()])


if __name__ == "__main__":
    v = compute()
    with open(os.path.join(HERE, "odirect_tiny.txt"), "w") as f:
        f.write(f"# O-direct forward ({NA}x{ND}) then adjoint ({N}x{N}) of workloads.white_noise({N}, 4242); "
                "written by make_golden.py from oracle/ only\n")
        for t in v:
            f.write(f"{t:.17e}\n")
    print("wrote", len(v), "values")
