"""GPU parity of the sinogram filter and of the solver iteration.

* `radon_filter` (both axes), `radon_forward_filtered`, `radon_adjoint_filtered` against O-filter
  (least-squares polynomial fit subtracted) composed with the operator
  oracles; the filtered pair keeps <F A x, y> = <x, A^T F y>;
* `radon_solver_step` / `radon_solver_run` against O-solver (one iterative soft-thresholding step,
  PAPER.md:29-31) on the exact operator (config 1) and on O-alg (config 3), after 1 and 10
  iterations; the graph-captured loop equals the single steps bit for bit and descends.

Tolerances: G1 = 1e-5 vs the oracle (north_star); the stand-alone filter adds fp32 dot products of
n <= 2048 terms (eps sqrt(n) ~ 3e-6 on the coefficients, which are O(1) of the line's norm)."""
import numpy as np
import pytest
import torch

import oracle
import workloads

pytestmark = pytest.mark.gpu
G1 = 1e-5


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).ravel(); b = np.asarray(b, dtype=np.float64).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def rb():
    import paper_1009_1380_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def synthetic_sinogram(cfg, seed):
    """Noise plus a slowly varying background along both axes (what the filter is there to remove)."""
    rng = np.random.default_rng(seed)
    s = np.linspace(-1, 1, cfg.n_det)[None, :]; a = np.linspace(-1, 1, cfg.n_angles)[:, None]
    return (rng.standard_normal((cfg.n_angles, cfg.n_det)) + 3.0 + 2.0 * s - 1.5 * s ** 3 + a * a * (1 + s)).astype(np.float32)


@pytest.mark.parametrize("cfg_id,order", [(1, 3), (1, 0), (1, 5), (2, 3), (3, 3), (4, 3)])
def test_filter_matches_oracle_on_both_axes(rb, cfg_id, order):
    cfg = workloads.get_config(cfg_id)
    plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    plan.set_filter(order)
    y = synthetic_sinogram(cfg, 40 + cfg_id)
    for axis in (0, 1):
        got = plan.radon_filter(dev(y), axis=axis).cpu().numpy()
        ref = oracle.polyfilter(y.astype(np.float64), order, axis=1 - axis)      # oracle axis 1 = detector
        assert rel(got, ref) < G1, (axis, rel(got, ref))
        assert np.abs(got - ref).max() < 5e-5 * np.abs(ref).max()
    # in place, and idempotent to round-off
    t = dev(y)
    plan.radon_filter(t, out=t, axis=0)
    assert rel(t.cpu().numpy(), oracle.polyfilter(y.astype(np.float64), order)) < G1
    plan.close()


@pytest.mark.parametrize("cfg_id", [1, 2, 4])
def test_filtered_forward_and_adjoint_match_oracle(rb, cfg_id):
    """filter(Radon{x}) and Radon^T{filter(y)} with the filter fused into the projection DFT kernels
    (power-of-two n_det: the pair kernels; otherwise the Bluestein kernels)."""
    cfg = workloads.get_config(cfg_id)
    plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    x = workloads.make_image(cfg_id)
    y = synthetic_sinogram(cfg, 50 + cfg_id)
    got_f = plan.radon_forward_filtered(dev(x)).cpu().numpy()
    got_a = plan.radon_adjoint_filtered(dev(y)).cpu().numpy()
    if cfg_id == 1:
        ref_f = oracle.polyfilter(oracle.forward(x, cfg.n_angles, cfg.n_det), 3)
        ref_a = oracle.adjoint(oracle.polyfilter(y.astype(np.float64), 3), cfg.N)
        assert rel(got_f, ref_f) < G1 and rel(got_a, ref_a) < G1, (rel(got_f, ref_f), rel(got_a, ref_a))
    else:
        # O-alg (gated against O-direct in the pins and in test_gpu_fullsize) at the full size
        ref_f = oracle.polyfilter(oracle.fast_forward(x, cfg.n_angles, cfg.n_det), 3)
        ref_a = oracle.fast_adjoint(oracle.polyfilter(y.astype(np.float64), 3), cfg.N)
        assert rel(got_f, ref_f) < G1 and rel(got_a, ref_a) < G1, (rel(got_f, ref_f), rel(got_a, ref_a))
    # fused == separate passes of the same library, to fp32 round-off
    sep_f = plan.radon_filter(plan.radon_forward(dev(x)), axis=0).cpu().numpy()
    sep_a = plan.radon_adjoint(plan.radon_filter(dev(y), axis=0)).cpu().numpy()
    assert rel(got_f, sep_f) < 3e-6 and rel(got_a, sep_a) < 3e-6, (rel(got_f, sep_f), rel(got_a, sep_a))
    # the filtered pair is still an adjoint pair: <F A x, y> = <x, A^T F y>
    lhs = float(np.vdot(got_f.astype(np.float64), y.astype(np.float64)))
    rhs = float(np.vdot(x.astype(np.float64), got_a.astype(np.float64)))
    assert abs(lhs - rhs) <= 5e-6 * np.linalg.norm(got_f) * np.linalg.norm(y)
    # orders above 3 take the separate pass
    plan.set_filter(5)
    hi = plan.radon_forward_filtered(dev(x)).cpu().numpy()
    assert rel(hi, oracle.polyfilter(plan.radon_forward(dev(x)).cpu().numpy().astype(np.float64), 5)) < G1
    plan.close()


def _power_iteration(plan, n_it=10):
    v = torch.ones((plan.N, plan.N), dtype=torch.float32, device="cuda")
    lam = 1.0
    for _ in range(n_it):
        w = plan.radon_adjoint(plan.radon_forward(v))
        lam = float(w.norm() / v.norm())
        v = w / w.norm()
    return lam


@pytest.mark.parametrize("cfg_id,filtered", [(1, False), (1, True), (3, False), (3, True)])
def test_solver_step_matches_oracle_after_1_and_10_iterations(rb, cfg_id, filtered):
    cfg = workloads.get_config(cfg_id)
    plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    x_true = workloads.make_image(cfg_id).astype(np.float64)
    if cfg_id == 1:
        fwd = lambda u: oracle.forward(u, cfg.n_angles, cfg.n_det)
        adj = lambda y: oracle.adjoint(y, cfg.N)
    else:
        fwd = lambda u: oracle.fast_forward(u, cfg.n_angles, cfg.n_det)
        adj = lambda y: oracle.fast_adjoint(y, cfg.N)
    b = fwd(x_true)
    alpha = 1.0 / _power_iteration(plan)
    tau = 1e-3 * alpha * float(np.abs(adj(b)).max())
    order = 3 if filtered else None
    x_ref = np.zeros_like(x_true)
    x_gpu = torch.zeros((cfg.N, cfg.N), dtype=torch.float32, device="cuda")
    bd = dev(b)
    for it in range(1, 11):
        x_ref = oracle.ista_step(x_ref, b, alpha, tau, fwd, adj, order)
        plan.radon_solver_step(x_gpu, bd, alpha, tau, filtered)
        if it in (1, 10):
            e = rel(x_gpu.cpu().numpy(), x_ref)
            assert e < (G1 if it == 1 else 1e-4), (it, e)
    plan.close()


def test_solver_run_is_the_captured_step_and_descends(rb):
    """radon_solver_run (one iteration captured as a CUDA graph, launched n times) == n calls of
    radon_solver_step bit for bit; the objective (1/2)||F(Ax - b)||^2 + (tau/alpha)||x||_1 falls
    monotonically over 100 iterations; no kernel outside the library runs in the loop."""
    cfg = workloads.get_config(3)
    plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    x_true = dev(workloads.make_image(3))
    b = plan.radon_forward(x_true).clone()
    alpha = 1.0 / _power_iteration(plan)
    tau = 1e-4
    for filtered in (False, True):
        xa = torch.zeros_like(x_true); xb = torch.zeros_like(x_true)
        for _ in range(5):
            plan.radon_solver_step(xa, b, alpha, tau, filtered)
        n0 = rb.kernel_launch_count()
        plan.radon_solver_run(xb, b, alpha, tau, 5, filtered)
        torch.cuda.synchronize()
        assert rb.kernel_launch_count() - n0 == 5 * 8
        assert torch.equal(xa, xb)

        def objective(x):
            r = plan.radon_forward(x) - b
            if filtered:
                r = plan.radon_filter(r, axis=0)
            return 0.5 * float((r.double() ** 2).sum()) + tau / alpha * float(x.double().abs().sum())

        vals = [objective(xb)]
        for _ in range(10):
            plan.radon_solver_run(xb, b, alpha, tau, 10, filtered)
            vals.append(objective(xb))
        assert all(v1 <= v0 * (1 + 1e-6) for v0, v1 in zip(vals, vals[1:])), vals
        assert vals[-1] < 0.2 * vals[0]
    plan.close()
