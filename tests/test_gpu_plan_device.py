"""P3 on the device (PAPER.md:57's bins replaced by plan-time tiles and
rounds): the schedules radon_plan_create builds with CUDA kernels (plan_device.cu) must pass the
same host checker as the host builder's (every sample exactly once in the gather; every
(sample, image, tile) incidence exactly once in the scatter; no two lanes of a round on the same
cells within a row step; at most two lanes of a half-warp per bank pair; every needed cell written
exactly once), and the operators built on them must match the oracle like any other plan."""
import os

import numpy as np
import pytest
import torch

import oracle
import workloads

pytestmark = pytest.mark.gpu

SHAPES = [(64, 90, 91), (512, 360, 725), (1024, 64, 1449), (2048, 1025, 2048),          # configs 1-4
          (32, 17, 48), (8, 1, 2), (128, 37, 200), (64, 30, 92), (512, 180, 1024), (16, 5, 33)]


@pytest.fixture(scope="module")
def rb():
    import paper_1009_1380_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


@pytest.mark.parametrize("shape", SHAPES)
def test_device_built_schedules_pass_the_host_checker(rb, shape):
    plan = rb.RadonPlan(*shape)
    for half in (False, True):
        bad, on_device, ms = plan.schedule_check(half)
        assert on_device, "schedules were built by the host fallback"
        assert bad == 0, (shape, half, bad)
        st = plan.schedule_stats(half)
        assert st["scatter_filled"] > 0 and st["gather_filled"] > 0
    plan.close()


def test_device_and_host_built_plans_agree_and_match_the_oracle(rb):
    """Same geometry, both builders: the gather does not depend on the schedule at all (bitwise
    equal), the scatter differs by the order of the additions only; both within the oracle gates."""
    cfg = workloads.get_config(1)
    x = workloads.make_image(1)
    xd = torch.from_numpy(x).cuda()
    dev_plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    os.environ["RADON_PLAN_BUILDER"] = "host"
    try:
        host_plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    finally:
        del os.environ["RADON_PLAN_BUILDER"]
    assert dev_plan.schedule_check(False, verify=False)[1] and not host_plan.schedule_check(False, verify=False)[1]
    Sd, Sh = dev_plan.radon_forward(xd), host_plan.radon_forward(xd)
    assert torch.equal(Sd, Sh)
    Ad, Ah = dev_plan.radon_adjoint(Sd).cpu().numpy(), host_plan.radon_adjoint(Sh).cpu().numpy()
    assert np.linalg.norm(Ad - Ah) / np.linalg.norm(Ah) < 1e-6
    ref = oracle.adjoint(Sd.cpu().numpy().astype(np.float64), cfg.N)
    assert np.linalg.norm(Ad - ref) / np.linalg.norm(ref) < 1e-5
    # a device-built plan is the same plan every time: bitwise equal results across plan instances
    again = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    assert np.array_equal(again.radon_adjoint(Sd).cpu().numpy(), Ad)
    for p in (dev_plan, host_plan, again):
        p.close()


@pytest.mark.parametrize("shape", [(64, 90, 91), (64, 30, 92), (32, 17, 48), (128, 37, 200), (512, 360, 725)])
def test_device_built_density_table_matches_the_host_table(rb, shape):
    """D of PAPER.md:89 for radon_inverse: the CUDA kernel (one thread per sample, neighbours from the
    geometry, fp64 series of I0) against the host fp64 table (itself checked against the oracle's
    O(M^2) double sum in tests/test_host_logic.py) to fp32 round-off."""
    plan = rb.RadonPlan(*shape)
    plan.prepare_inverse()
    D, scale = plan.density()
    ref, scale_ref = rb.density_host(*shape)
    assert abs(scale / scale_ref - 1) < 1e-12
    assert np.max(np.abs(D.numpy() / ref - 1)) < 2e-7
    plan.close()
