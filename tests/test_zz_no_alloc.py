"""radon_grid_only_static (include/radon.h): gridding (D == 1) for callers that cannot
allocate.  Same kernel and schedule as radon_grid_only, with the kernel's scratch (partial rectangles
of split tiles, merge counters, the summed j = 0 samples) in file-scope device arrays of the library.

Collected last on purpose (test_zz_*): the suite runs with `pytest -x`, so a failure here must not
hide any other test.  Passes alone in a fresh process and after the other tests: it reads no state
they leave behind (each test creates its own plans; the static arrays are cleared / rewritten by the
call itself)."""
import numpy as np
import pytest
import torch

import oracle
import workloads

pytestmark = pytest.mark.gpu

RADON_ELIMIT = -6


@pytest.fixture(scope="module")
def rb():
    import paper_1009_1380_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a, dtype=np.complex128) - b) / np.linalg.norm(b))


def polar_input(shape, seed):
    na, nd = shape[1], shape[2]
    return torch.from_numpy(workloads.random_complex((na, nd), seed).astype(np.complex64)).cuda()


# split tiles + centre window (merge jobs, partial rectangles) at every shape: configs 1-4 and the
# paper's own 180 x 1024 shape (64 to ~1500 partial rectangles)
@pytest.mark.parametrize("shape", [(64, 90, 91), (512, 360, 725), (1024, 64, 1449), (2048, 1025, 2048), (512, 180, 1024)])
def test_static_scratch_gridding_matches_the_workspace_path_twice_in_a_row(rb, shape):
    plan = rb.RadonPlan(*shape)
    st = rb.schedule_host_stats(*shape, half=False)             # the host builder's count; the device builder's is close
    assert st["merge_jobs"] > 0 and 0 < st["partial_rects"] <= 2048, "the shape must use the scratch and fit the limit"
    for call, seed in enumerate((21, 22)):                      # two calls in a row, different data
        P = polar_input(shape, seed)
        ref = plan.radon_grid_only(P).clone()                    # existing path: scratch in the plan's workspace
        out = torch.full((plan.G, plan.G), 7 + 7j, dtype=torch.complex64, device="cuda")
        torch.cuda.synchronize()
        before = (plan.device_bytes(), torch.cuda.mem_get_info()[0])   # the library's own count; the driver's free bytes
        ret = plan.radon_grid_only_static(P, out)
        torch.cuda.synchronize()
        after = (plan.device_bytes(), torch.cuda.mem_get_info()[0])
        assert ret is out and after[0] == before[0]
        if call == 1:                                            # the first call on a device may load the module
            assert after[1] == before[1], "free device memory changed across the call"
        # same kernel, same schedule, fixed order of additions: bit-identical (tighter than the
        # 2e-6 relative L2 the gridding tests allow against the oracle)
        assert torch.equal(torch.view_as_real(out), torch.view_as_real(ref)), (shape, call)
    plan.close()


def test_static_scratch_gridding_matches_the_oracle_and_survives_other_plans(rb):
    """Against O-grid within the gridding tests' tolerance (2e-6), with calls of OTHER plans in
    between: the arrays keep the last call's contents and the next call must not depend on them."""
    small, other = (64, 90, 91), (128, 37, 200)
    pa, pb = rb.RadonPlan(*small), rb.RadonPlan(*other)
    Pa_np = workloads.random_complex((small[1], small[2]), 12)
    ref = oracle.grid_grid(Pa_np, pa.G)
    Pa = torch.from_numpy(Pa_np.astype(np.complex64)).cuda()
    Pb = polar_input(other, 5)
    outs = []
    for _ in range(2):
        ga = torch.empty((pa.G, pa.G), dtype=torch.complex64, device="cuda")
        gb = torch.empty((pb.G, pb.G), dtype=torch.complex64, device="cuda")
        pb.radon_grid_only_static(Pb, gb)                        # leaves its partial rectangles in the arrays
        pa.radon_grid_only_static(Pa, ga)
        assert torch.equal(torch.view_as_real(gb), torch.view_as_real(pb.radon_grid_only(Pb)))
        outs.append(ga.cpu().numpy())
    assert rel(outs[0], ref) < 2e-6
    assert np.array_equal(outs[0].view(np.uint32), outs[1].view(np.uint32))
    pa.close(); pb.close()


def test_static_scratch_limit_is_enforced_before_any_launch(rb):
    """1024^2 with 4096 x 2048 samples: ~5500 partial rectangles (host builder: 5549) against
    RADON_STATIC_SCRATCH_SLOTS = 2048."""
    shape = (1024, 4096, 2048)
    plan = rb.RadonPlan(*shape)
    P = polar_input(shape, 3)
    out = torch.full((plan.G, plan.G), 7 + 7j, dtype=torch.complex64, device="cuda")
    n0 = rb.kernel_launch_count()
    with pytest.raises(rb.RadonError) as e:
        plan.radon_grid_only_static(P, out)
    assert e.value.code == RADON_ELIMIT and "static" in str(e.value)
    assert rb.kernel_launch_count() == n0                        # nothing was launched
    torch.cuda.synchronize()
    assert bool((out == 7 + 7j).all())                           # the output was not touched
    # null arguments
    import ctypes
    L = rb.lib()
    assert L.radon_grid_only_static(None, ctypes.c_void_p(P.data_ptr()), ctypes.c_void_p(out.data_ptr()), None) == -1
    assert L.radon_grid_only_static(plan._h, None, ctypes.c_void_p(out.data_ptr()), None) == -1
    # the ordinary entry point takes the same plan
    assert torch.isfinite(torch.view_as_real(plan.radon_grid_only(P))).all()
    plan.close()
