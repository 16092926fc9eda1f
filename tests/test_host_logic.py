"""CPU-only tests: the C-ABI library loads and exports every symbol include/radon.h declares,
argument validation, and the plan-time schedule builder's invariants (no GPU compute)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1009_1380_b200 as rb
from paper_1009_1380_b200 import build as rb_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    rb_build.build()


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "radon.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(radon_[a-z0-9_]+)\s*\(", header))
    assert declared, "no declarations parsed"
    L = ctypes.CDLL(rb.lib_path())
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/radon.h but not exported"
    assert declared == set(rb.EXPORTED_SYMBOLS), declared ^ set(rb.EXPORTED_SYMBOLS)


def test_strerror_and_validation_without_gpu():
    L = rb.lib()
    assert L.radon_strerror(0) == b"ok"
    assert b"invalid" in L.radon_strerror(-1)
    h = ctypes.c_void_p(123)
    # invalid arguments are rejected before any CUDA call
    assert L.radon_plan_create(ctypes.byref(h), 4, 10, 10, 2.0, 6) == -1 and not h.value     # N < 8
    assert L.radon_plan_create(ctypes.byref(h), 64, 0, 91, 2.0, 6) == -1
    assert L.radon_plan_create(ctypes.byref(h), 64, 90, 1, 2.0, 6) == -1
    assert L.radon_plan_create(ctypes.byref(h), 64, 90, 91, 2.0, 13) == -1
    assert L.radon_plan_create(ctypes.byref(h), 65, 90, 91, 1.5, 6) == -1                   # odd sigma*N
    assert L.radon_plan_create(None, 64, 90, 91, 2.0, 6) == -1
    assert L.radon_plan_create(ctypes.byref(h), 64, 90, 91, 2.0, 10) == -5                  # W not in {4, 6, 8}: not built
    assert L.radon_plan_create(ctypes.byref(h), 56, 90, 91, 2.0, 6) == -5                   # G = 112 = 7 * 16: not built
    assert L.radon_plan_destroy(None) == 0
    assert L.radon_forward(None, None, None, None) == -1


@pytest.mark.parametrize("half", [False, True])
@pytest.mark.parametrize("shape", [(8, 5, 9), (16, 7, 12), (32, 33, 47), (64, 90, 91), (128, 64, 181),
                                   (256, 100, 256)])
def test_schedule_invariants(shape, half):
    """Every sample issued exactly once by the gather; every (sample, wrap image, tap, cell)
    incidence accumulated exactly once by the scatter; footprints of a round disjoint per row
    step; at most two lanes of a half-warp per bank pair; every grid cell written exactly once.  half: the Hermitian
    half schedules of radon_forward / radon_adjoint (samples j >= 0 plus the Nyquist ghost for
    even n_det; grid rows ky = 0 .. G/2 only, every other row untouched)."""
    rc, bad = rb.schedule_selfcheck(*shape, half=half)
    assert (rc, bad) == (0, 0)


@pytest.mark.parametrize("half", [False, True])
@pytest.mark.parametrize("shape", [(2048, 12, 40), (2048, 40, 2048), (1536, 9, 100)])
def test_schedule_invariants_with_tall_scatter_tiles(shape, half):
    """Grids of 4096 and more get 64 x 40 scatter tiles (Geometry::st_y; 64 x 32 below): the same
    invariants, and the tile count says which height the plan took (G = 4096: 64 tiles across,
    ceil(G / 40) = 103 down on the full grid against 128 with 32 rows; G = 3072 keeps 32 rows)."""
    assert rb.schedule_selfcheck(*shape, half=half) == (0, 0)
    st = rb.schedule_host_stats(*shape, half=half)
    G = 2 * shape[0]
    rows = (1 + -(-(G // 2) // (40 if G >= 4096 else 32))) if half else -(-G // (40 if G >= 4096 else 32))
    tiles = (G // 64) * rows
    assert tiles <= st["scatter_ctas"] <= tiles + st["partial_rects"], (st["scatter_ctas"], tiles)


def test_schedule_stats_config2_shape():
    st = rb.schedule_host_stats(512, 360, 725)
    M = 360 * 725
    assert st["gather_filled"] == M
    assert st["scatter_filled"] >= M                       # owner-computes duplicates at tile borders
    assert st["scatter_filled"] < 1.3 * M
    assert st["gather_filled"] / st["gather_slots"] > 0.8  # lane utilisation of the gather rounds
    assert st["scatter_max_rounds"] <= 96 and st["gather_max_rounds"] <= 64   # full schedule splits at 96
    # Hermitian half: j >= 0 of every ray plus the ghost (n even) or nothing (n odd: 725)
    sh = rb.schedule_host_stats(512, 360, 725, half=True)
    assert sh["gather_filled"] == 360 * (725 - 725 // 2)
    assert 0.5 * M <= sh["scatter_filled"] < 0.7 * M
    assert sh["scatter_max_rounds"] <= 48                                      # half schedule splits at 48
    se = rb.schedule_host_stats(512, 90, 512, half=True)
    assert se["gather_filled"] == 90 * (512 // 2 + 1)


def test_kb_polynomial_weights_match_oracle_kernel():
    """The kernels' tap weights (plan-time degree-7 polynomial pieces, fp32 Horner) against
    the oracle's directly evaluated Kaiser-Bessel kernel: |err| < 3e-7 (fp32 round-off level)."""
    import numpy as np
    import oracle

    worst = 0.0
    for delta in np.linspace(0.0, 1.0, 257):
        w = np.array(rb.kb_weights_host(float(delta)))
        ref = oracle.kb_phi(np.float32(delta).astype(np.float64) - 3.0 + np.arange(6))
        worst = max(worst, float(np.abs(w - ref).max()))
    assert worst < 3e-7, worst


@pytest.mark.parametrize("shape", [(64, 90, 91), (32, 17, 48), (16, 3, 64)])
def test_density_table_of_the_library_matches_the_oracle(shape):
    """radon_inverse's plan constant (host fp64 -> fp32) against O-density evaluated
    as printed (the O(M^2) double sum: no bucketing on the oracle's side)."""
    import oracle

    N, na, nd = shape
    D, scale = rb.density_host(N, na, nd)
    assert abs(scale / oracle.inverse_scale(nd, 2 * N) - 1) < 1e-12
    ref = oracle.density(na, nd, 2 * N, brute=True) * scale
    assert np.max(np.abs(D / ref - 1)) < 2e-7


def test_product_never_touches_the_oracle_or_work_files():
    """The CUDA path and its binding share nothing with oracle/ (and nothing committed reads
    _work/): scan the package and the C sources for any reference."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    pkg = os.path.join(root, "paper_1009_1380_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if not f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                continue
            text = open(os.path.join(dirpath, f)).read()
            assert not re.search(r"^\s*(import|from)\s+oracle\b", text, re.M), f
            assert "liboracle" not in text and "radon_oracle" not in text, f
            assert "_work/" not in text, f
    assert "oracle" not in open(os.path.join(root, "include", "radon.h")).read()


def test_bench_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the CPU oracle as the reference arm) prints one JSON line with
    the contract's keys; a tiny sample keeps this to seconds."""
    import json
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--ref-sample", "8"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-500:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                "scaling", "vs_baseline", "dtype", "data", "config", "e2e", "cpu_baseline"):
        assert key in line, key
    assert line["impl"] == "reference" and line["unit"] == "pairs/s" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["cpu_baseline"]["kind"] == "oracle"


@pytest.mark.parametrize("n,order", [(91, 3), (2048, 3), (725, 0), (64, 5), (3, 3)])
def test_filter_basis_of_the_library_spans_the_oracle_projector(n, order):
    """The plan-time basis of the sinogram filter (fp64 Gram-Schmidt -> fp32) against
    O-filter: z - Q Q^T z must be the oracle's fit-and-subtract on random lines."""
    import oracle

    q = rb.filter_basis_host(n, order).astype(np.float64)
    z = np.random.default_rng(5).standard_normal((7, n)) + np.linspace(-2, 3, n)[None, :] ** 3
    got = z - (z @ q) @ q.T
    ref = oracle.polyfilter(z, min(order, n - 1))
    assert np.linalg.norm(got - ref) / np.linalg.norm(z) < 5e-7


def test_plan_create_rejects_bad_and_unbuilt_requests_without_touching_a_gpu():
    """Error behaviour of the boundary (include/radon.h): argument checks come before any CUDA call,
    so they can be exercised on a CPU box.  EINVAL = -1, EUNSUPPORTED = -5."""
    import ctypes

    L = rb.lib()
    h = ctypes.c_void_p(123)

    def create(N, na, nd, sigma=2.0, W=6):
        return L.radon_plan_create(ctypes.byref(h), N, na, nd, ctypes.c_float(sigma), W), h.value

    assert L.radon_plan_create(None, 64, 90, 91, ctypes.c_float(2.0), 6) == -1
    for args in [(4, 90, 91), (64, 0, 91), (64, 90, 1), (64, 70000, 91), (64, 90, 65534)]:
        assert create(*args) == (-1, None), args                          # and *out is set to NULL
    assert create(64, 90, 91, sigma=1.0)[0] == -1 and create(64, 90, 91, sigma=9.0)[0] == -1
    assert create(63, 90, 91, sigma=1.5)[0] == -1                          # sigma N not an even integer
    assert create(64, 90, 91, W=1)[0] == -1 and create(64, 90, 91, W=13)[0] == -1
    assert create(64, 90, 91, W=10)[0] == -5 and create(64, 90, 91, W=5)[0] == -5     # valid, not built (4, 6, 8 are)
    assert create(56, 90, 91)[0] == -5 and create(6144, 90, 91)[0] == -5   # sigma N = 7 * 16; 3 * 4096 (sub-length > 2048)
    assert create(64, 90, 5000)[0] == -5                                   # Bluestein length > 8192
    assert b"power of two" in L.radon_strerror(-5)
    # host-only entry points
    q = (ctypes.c_float * 64)()
    assert L.radon_filter_basis_host(0, 3, q) == -1 and L.radon_filter_basis_host(8, 8, q) == -1
    assert L.radon_filter_basis_host(8, 3, None) == -1 and L.radon_filter_basis_host(8, 3, q) == 0
    w = (ctypes.c_float * 6)()
    assert L.radon_kb_weights_host(6, ctypes.c_float(2.0), ctypes.c_float(1.5), w) == -1
    assert L.radon_kb_weights_host(10, ctypes.c_float(2.0), ctypes.c_float(0.5), w) == -5
    bad = ctypes.c_longlong()
    assert L.radon_schedule_selfcheck(64, 90, 91, ctypes.c_float(2.0), 10, 0, ctypes.byref(bad)) == -5
    assert L.radon_density_host(64, 90, 91, ctypes.c_float(2.0), 6, None, None) == -1
    # a NULL plan is an argument error everywhere, never a crash
    for name in ("radon_forward", "radon_adjoint", "radon_inverse", "radon_nufft2", "radon_nufft1", "radon_interp_only",
                 "radon_grid_only", "radon_proj_ifft", "radon_proj_fft", "radon_forward_filtered", "radon_adjoint_filtered"):
        assert getattr(L, name)(None, None, None, None) == -1, name
    assert L.radon_plan_destroy(None) == 0


@pytest.mark.parametrize("W", [4, 8])
def test_other_kernel_widths_weights_and_schedules(W):
    """radon_plan_create(..., W) for the other widths the library is instantiated for: the tap
    weights against the oracle's directly evaluated Kaiser-Bessel kernel, and the host schedule
    builder's invariants with footprints of W x W cells."""
    import oracle

    beta = oracle.kb_beta(W, 2.0)
    for delta in (0.0, 0.123, 0.5, 0.77, 1.0):
        w = rb.kb_weights_host(delta, W=W)
        ref = oracle.kb_phi(delta - W / 2 + np.arange(W), W, beta)
        assert np.max(np.abs(np.array(w) - ref)) < 5e-7, (W, delta)
    for shape in [(16, 7, 12), (64, 90, 91), (128, 64, 181)]:
        for half in (False, True):
            assert rb.schedule_selfcheck(*shape, W=W, half=half) == (0, 0), (W, shape, half)
