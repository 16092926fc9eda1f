"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 CPU oracle on the
same seeded inputs.  Tolerances: BASELINE.json north_star -- relative L2 <= 1e-5 against the
oracle for radon_forward / radon_adjoint on the configs' phantoms (gate G1), <= 1e-4 for the
bare NUFFT against the direct NDFT on arbitrary inputs (gate G2); stage-level comparisons
against O-grid / plain DFTs use fp32 round-off level bounds derived in DESIGN.md section 6."""
import numpy as np
import pytest
import torch

import oracle
import workloads

pytestmark = pytest.mark.gpu

G1 = 1e-5
G2 = 1e-4


def rel(a, b):
    a = np.asarray(a).ravel(); b = np.asarray(b).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def rb():
    import paper_1009_1380_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()     # fails loudly if the extension is missing
    return m


def dev(a, dtype):
    return torch.from_numpy(np.ascontiguousarray(a)).to(dtype).cuda()


# --------------------------------------------------------------- stage level ----
@pytest.mark.parametrize("shape", [(64, 90, 91), (32, 17, 48), (128, 37, 200)])
def test_interp_only_matches_ogrid(rb, shape):
    N, na, nd = shape
    plan = rb.RadonPlan(N, na, nd)
    grid = workloads.random_complex((plan.G, plan.G), 11)
    ref = oracle.grid_interp(grid, na, nd)
    out = plan.radon_interp_only(dev(grid, torch.complex64)).cpu().numpy()
    assert rel(out, ref) < 2e-6          # LUT (S=256, linear) + fp32 accumulation


@pytest.mark.parametrize("shape", [(64, 90, 91), (32, 17, 48), (128, 37, 200)])
def test_grid_only_matches_ogrid_and_is_deterministic(rb, shape):
    N, na, nd = shape
    plan = rb.RadonPlan(N, na, nd)
    P = workloads.random_complex((na, nd), 12)
    ref = oracle.grid_grid(P, plan.G)
    dP = dev(P, torch.complex64)
    out1 = plan.radon_grid_only(dP).cpu().numpy()
    assert rel(out1, ref) < 2e-6
    out2 = plan.radon_grid_only(dP, torch.full((plan.G, plan.G), 7 + 7j, dtype=torch.complex64, device="cuda")).cpu().numpy()
    assert np.array_equal(out1.view(np.uint32), out2.view(np.uint32))    # bitwise, every cell rewritten


@pytest.mark.parametrize("nd", [16, 91, 128, 725, 1449, 2048])
def test_projection_dfts_match_plain_dft(rb, nd):
    na = 5
    plan = rb.RadonPlan(64, na, nd)
    c = nd // 2
    j = np.arange(nd) - c
    E = np.exp(-2j * np.pi * ((j[:, None] * j[None, :]) % nd) / nd)      # [k, s]
    y = np.random.default_rng(3).standard_normal((na, nd)).astype(np.float32)
    ref = (y.astype(np.float64) @ E.T) / nd
    out = plan.radon_proj_fft(dev(y, torch.float32)).cpu().numpy()
    assert rel(out, ref) < 3e-6
    P = workloads.random_complex((na, nd), 4)
    ref = np.real(P.astype(np.complex128) @ np.conj(E)) / nd
    out = plan.radon_proj_ifft(dev(P, torch.complex64)).cpu().numpy()
    assert rel(out, ref) < 3e-6


# --------------------------------------------------------------- gate G2 --------
@pytest.mark.parametrize("N,na,nd", [(8, 6, 11), (16, 9, 16), (64, 30, 91)])
def test_bare_nufft_vs_direct_ndft(rb, N, na, nd):
    plan = rb.RadonPlan(N, na, nd)
    for img in (workloads.white_noise(N, 21), workloads.delta_image(N, 0, N - 1)):
        ref = oracle.ndft2(img.astype(np.float64), na, nd)
        out = plan.radon_nufft2(dev(img, torch.float32)).cpu().numpy()
        assert rel(out, ref) < G2
    P = workloads.random_complex((na, nd), 22)
    ref = np.real(oracle.ndft1(P, N))
    out = plan.radon_nufft1(dev(P, torch.complex64)).cpu().numpy()
    assert rel(out, ref) < G2


# --------------------------------------------------------------- gate G1 --------
def test_config1_forward_adjoint_vs_odirect_full(rb):
    cfg = workloads.get_config(1)
    x = workloads.make_image(1)
    plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    S_ref = oracle.forward(x, cfg.n_angles, cfg.n_det)
    S = plan.radon_forward(dev(x, torch.float32)).cpu().numpy()
    e_f = rel(S, S_ref)
    y = S_ref.astype(np.float32)
    A_ref = oracle.adjoint(y, cfg.N)
    A = plan.radon_adjoint(dev(y, torch.float32)).cpu().numpy()
    e_a = rel(A, A_ref)
    assert e_f < G1 and e_a < G1, (e_f, e_a)
    # C8: not suspiciously below the method's fp64 algorithmic floor, and the fp32 path
    # sits within round-off of the fp64 same-algorithm oracle (O-alg)
    assert e_f > 5e-7
    assert rel(S, oracle.fast_forward(x, cfg.n_angles, cfg.n_det)) < 2e-6
    assert rel(A, oracle.fast_adjoint(y, cfg.N)) < 2e-6


def test_adjoint_identity_fp32(rb):
    cfg = workloads.get_config(1)
    plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    rng = np.random.default_rng(5)
    x = rng.standard_normal((cfg.N, cfg.N)).astype(np.float32)
    y = rng.standard_normal((cfg.n_angles, cfg.n_det)).astype(np.float32)
    Ax = plan.radon_forward(dev(x, torch.float32)).cpu().numpy().astype(np.float64)
    Aty = plan.radon_adjoint(dev(y, torch.float32)).cpu().numpy().astype(np.float64)
    lhs, rhs = np.vdot(Ax, y), np.vdot(x, Aty)
    assert abs(lhs - rhs) < 5e-6 * np.linalg.norm(Ax) * np.linalg.norm(y)


@pytest.mark.parametrize("cfg_id,n_sub", [(2, 2048), (3, 1024), (4, 384)])
def test_full_size_configs_on_sampled_outputs(rb, cfg_id, n_sub):
    """At BASELINE.json's full sizes the oracle evaluates a seeded random subset of outputs
    (each output is an independent sum, so the subset is exact)."""
    cfg = workloads.get_config(cfg_id)
    x = workloads.make_image(cfg_id)
    plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    rng = np.random.default_rng(100 + cfg_id)
    idx = rng.choice(cfg.M, n_sub, replace=False)
    S = plan.radon_forward(dev(x, torch.float32))
    ref = oracle.dirichlet_forward_subset(x, cfg.n_angles, cfg.n_det, idx)    # closed form: N^2 terms/output
    e_f = rel(S.cpu().numpy().ravel()[idx], ref)
    # adjoint on y = A x (computed by the GPU, then handed identically to both sides)
    y = S.cpu().numpy()
    pix = rng.choice(cfg.N * cfg.N, n_sub, replace=False)
    A = plan.radon_adjoint(dev(y, torch.float32)).cpu().numpy()
    ref_a = oracle.dirichlet_adjoint(y, cfg.N, pix=pix)                        # closed form: M terms/pixel
    e_a = rel(A.ravel()[pix], ref_a)
    assert e_f < G1 and e_a < G1, (cfg_id, e_f, e_a)


@pytest.mark.parametrize("cfg_id", [2, 3])
def test_repeated_calls_are_bitwise_identical(rb, cfg_id):
    """No atomics and a fixed order of every addition: forward, adjoint and the bare gridding
    kernels are bitwise reproducible from call to call (also guards the staged kernels'
    buffer reuse: a missing proxy fence showed up here as run-to-run differences)."""
    cfg = workloads.get_config(cfg_id)
    plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    rng = np.random.default_rng(40 + cfg_id)
    x = dev(rng.standard_normal((cfg.N, cfg.N)), torch.float32)
    y = dev(rng.standard_normal((cfg.n_angles, cfg.n_det)), torch.float32)
    pol = torch.view_as_complex(dev(rng.standard_normal((cfg.n_angles, cfg.n_det, 2)), torch.float32))
    grd = torch.view_as_complex(dev(rng.standard_normal((plan.G, plan.G, 2)), torch.float32))
    ref = [plan.radon_forward(x).clone(), plan.radon_adjoint(y).clone(),
           plan.radon_grid_only(pol).clone(), plan.radon_interp_only(grd).clone()]
    for _ in range(12):
        assert torch.equal(plan.radon_forward(x), ref[0])
        assert torch.equal(plan.radon_adjoint(y), ref[1])
        assert torch.equal(plan.radon_grid_only(pol), ref[2])
        assert torch.equal(plan.radon_interp_only(grd), ref[3])


def test_batch_and_host_entry_points_match_single_calls(rb):
    N, na, nd = 128, 50, 181
    plan = rb.RadonPlan(N, na, nd)
    xs = np.stack([workloads.make_batch_slice(i, N) for i in range(3)])
    dx = dev(xs, torch.float32)
    single = torch.stack([plan.radon_forward(dx[i]).clone() for i in range(3)])
    batch = plan.radon_forward_batch(dx)
    assert torch.equal(single, batch)
    hx = torch.from_numpy(xs).pin_memory()
    hs = torch.empty((3, na, nd), dtype=torch.float32).pin_memory()
    plan.radon_forward_host(hx, hs)
    assert torch.equal(hs, batch.cpu())
    back = plan.radon_adjoint_batch(batch)
    hb = torch.empty((3, N, N), dtype=torch.float32).pin_memory()
    plan.radon_adjoint_host(hs, hb)
    assert torch.equal(hb, back.cpu())
    assert rb.kernel_launch_count() > 0
