"""ctypes binding with the same names as include/radon.h (marshalling only)."""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libradon_b200.so")
_lib = None

c_int, c_ll, c_float, c_void_p, c_size_t = (ctypes.c_int, ctypes.c_longlong, ctypes.c_float,
                                            ctypes.c_void_p, ctypes.c_size_t)
P = ctypes.POINTER

# name -> (restype, argtypes); one entry per function declared in include/radon.h
_SIGNATURES = {
    "radon_plan_create": (c_int, [P(c_void_p), c_int, c_int, c_int, c_float, c_int]),
    "radon_plan_destroy": (c_int, [c_void_p]),
    "radon_forward": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_adjoint": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_forward_batch": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_void_p]),
    "radon_adjoint_batch": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_void_p]),
    "radon_forward_host": (c_int, [c_void_p, c_void_p, c_void_p, c_int]),
    "radon_adjoint_host": (c_int, [c_void_p, c_void_p, c_void_p, c_int]),
    "radon_forward_adjoint_host": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_int]),
    "radon_nufft2": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_nufft1": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_interp_only": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_grid_only": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_grid_only_static": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_grid_only_paper_bins": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_void_p]),
    "radon_paper_bins_stats": (c_int, [c_void_p, P(c_int), P(c_ll), P(c_int), P(c_int)]),
    "radon_proj_ifft": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_proj_fft": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_plan_stage_timing": (c_int, [c_void_p, c_int]),
    "radon_plan_stage_times": (c_int, [c_void_p, P(ctypes.c_double), P(c_ll)]),
    "radon_plan_info": (c_int, [c_void_p, P(c_int), P(c_int), P(c_int), P(c_int), P(c_ll), P(c_size_t)]),
    "radon_plan_schedule_stats": (c_int, [c_void_p, c_int, P(c_ll), P(c_ll), P(c_int), P(c_ll), P(c_ll), P(c_int)]),
    "radon_plan_schedule_check": (c_int, [c_void_p, c_int, P(c_ll), P(c_int), P(ctypes.c_double)]),
    "radon_schedule_selfcheck": (c_int, [c_int, c_int, c_int, c_float, c_int, c_int, P(c_ll)]),
    "radon_schedule_host_stats": (c_int, [c_int, c_int, c_int, c_float, c_int, c_int, P(c_ll)]),
    "radon_kb_weights_host": (c_int, [c_int, c_float, c_float, P(c_float)]),
    "radon_inverse": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_plan_prepare_inverse": (c_int, [c_void_p]),
    "radon_plan_density": (c_int, [c_void_p, c_void_p, P(ctypes.c_double)]),
    "radon_density_host": (c_int, [c_int, c_int, c_int, c_float, c_int, c_void_p, P(ctypes.c_double)]),
    "radon_plan_set_filter": (c_int, [c_void_p, c_int]),
    "radon_filter": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_void_p]),
    "radon_forward_filtered": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_adjoint_filtered": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "radon_filter_basis_host": (c_int, [c_int, c_int, c_void_p]),
    "radon_solver_step": (c_int, [c_void_p, c_void_p, c_void_p, c_float, c_float, c_int, c_void_p]),
    "radon_solver_run": (c_int, [c_void_p, c_void_p, c_void_p, c_float, c_float, c_int, c_int, c_void_p]),
    "radon_kernel_launch_count": (c_ll, []),
    "radon_strerror": (ctypes.c_char_p, [c_int]),
    "radon_last_cuda_error": (ctypes.c_char_p, []),
}
EXPORTED_SYMBOLS = tuple(_SIGNATURES)


class RadonError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib().radon_strerror(code).decode()
        if code == -3:
            msg += ": " + lib().radon_last_cuda_error().decode()
        super().__init__(f"{where} failed with {code} ({msg})")


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """Load libradon_b200.so (built in-tree by build.py).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(
                f"{_LIB_PATH} is missing: run `python -m paper_1009_1380_b200.build` "
                "(or __graft_entry__.build()). There is no CPU fallback.")
        L = ctypes.CDLL(_LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(code, where):
    if code != 0:
        raise RadonError(code, where)


def density_host(N, n_angles, n_det, sigma=2.0, W=6):
    """Host-only density table of radon_inverse: (numpy float32 (n_angles, n_det) = D * scale, scale)."""
    import numpy as np

    out = np.empty((n_angles, n_det), dtype=np.float32)
    sc = ctypes.c_double()
    _check(lib().radon_density_host(N, n_angles, n_det, sigma, W, out.ctypes.data_as(c_void_p), ctypes.byref(sc)),
           "radon_density_host")
    return out, float(sc.value)


def filter_basis_host(n, order):
    """Host-only: the orthonormal discrete polynomial basis of the sinogram filter, (n, order+1) float32."""
    import numpy as np

    q = np.empty((n, order + 1), dtype=np.float32)
    _check(lib().radon_filter_basis_host(n, order, q.ctypes.data_as(c_void_p)), "radon_filter_basis_host")
    return q


def kernel_launch_count() -> int:
    return int(lib().radon_kernel_launch_count())


def schedule_selfcheck(N, n_angles, n_det, sigma=2.0, W=6, half=False):
    """Host-only check of the plan-time schedules (no GPU). Returns (rc, n_violations)."""
    bad = c_ll(-1)
    rc = lib().radon_schedule_selfcheck(N, n_angles, n_det, sigma, W, int(half), ctypes.byref(bad))
    return rc, int(bad.value)


def schedule_host_stats(N, n_angles, n_det, sigma=2.0, W=6, half=False):
    """Host-only schedule statistics (no GPU): dict of slot / CTA counts."""
    out = (c_ll * 10)()
    _check(lib().radon_schedule_host_stats(N, n_angles, n_det, sigma, W, int(half), out), "radon_schedule_host_stats")
    keys = ["gather_slots", "gather_filled", "gather_ctas", "gather_max_rounds", "scatter_slots",
            "scatter_filled", "scatter_ctas", "scatter_max_rounds", "merge_jobs", "partial_rects"]
    return dict(zip(keys, [int(v) for v in out]))


def kb_weights_host(delta, W=6, sigma=2.0):
    """The W tap weights as the kernels compute them, evaluated on the host (no GPU)."""
    out = (c_float * W)()
    _check(lib().radon_kb_weights_host(W, sigma, float(delta), out), "radon_kb_weights_host")
    return [float(v) for v in out]


def _ptr(t):
    return c_void_p(t.data_ptr())


class RadonPlan:
    """Owns a radon_plan.  Tensor arguments are CUDA tensors (fp32 / complex64, contiguous);
    outputs are allocated with torch when not supplied.  All calls are asynchronous on
    torch's current stream."""

    def __init__(self, N, n_angles, n_det, sigma=2.0, W=6):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1009_1380_b200 needs a CUDA device (sm_100a); no CPU fallback")
        self._h = c_void_p()
        _check(lib().radon_plan_create(ctypes.byref(self._h), N, n_angles, n_det, sigma, W),
               "radon_plan_create")
        n = c_int(); g = c_int(); na = c_int(); nd = c_int(); m = c_ll(); wb = c_size_t()
        _check(lib().radon_plan_info(self._h, n, g, na, nd, m, wb), "radon_plan_info")
        self.N, self.G, self.n_angles, self.n_det = n.value, g.value, na.value, nd.value
        self.M, self.workspace_bytes = m.value, wb.value

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().radon_plan_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers --------------------------------------------------------------------
    @staticmethod
    def _stream():
        import torch

        return c_void_p(torch.cuda.current_stream().cuda_stream)

    @staticmethod
    def _chk(t, dtype, numel, name):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype and t.numel() == numel):
            raise ValueError(f"{name}: need a contiguous CUDA {dtype} tensor of {numel} elements")

    def _new(self, shape, dtype):
        import torch

        return torch.empty(shape, dtype=dtype, device="cuda")

    def device_bytes(self) -> int:
        """Device bytes the plan owns now (workspaces of the batched / host calls are allocated on first use)."""
        wb = c_size_t()
        _check(lib().radon_plan_info(self._h, None, None, None, None, None, wb), "radon_plan_info")
        return int(wb.value)

    def schedule_check(self, half=False, verify=True):
        """(violations or None, built_on_device, build_ms) of the schedules this plan uses."""
        bad = c_ll(-1); dev = c_int(); ms = ctypes.c_double()
        rc = lib().radon_plan_schedule_check(self._h, int(half), ctypes.byref(bad) if verify else None,
                                             ctypes.byref(dev), ctypes.byref(ms))
        if rc not in (0, -1):
            _check(rc, "radon_plan_schedule_check")
        return (int(bad.value) if verify else None), bool(dev.value), float(ms.value)

    def schedule_stats(self, half=False):
        v = [c_ll(), c_ll(), c_int(), c_ll(), c_ll(), c_int()]
        _check(lib().radon_plan_schedule_stats(self._h, int(half), *v), "radon_plan_schedule_stats")
        k = ["gather_slots", "gather_filled", "gather_ctas", "scatter_slots", "scatter_filled", "scatter_ctas"]
        return {a: b.value for a, b in zip(k, v)}

    STAGES = ("F1_colfft", "F2_rowfft", "F3_gather", "F4_proj_ifft",
              "A1_proj_fft", "A2_scatter", "A3_rowifft", "A4_colifft")

    def stage_timing(self, enable: bool):
        _check(lib().radon_plan_stage_timing(self._h, int(enable)), "radon_plan_stage_timing")

    def stage_times(self):
        """{stage: (total_ms, launches)} accumulated since the last call (synchronises)."""
        ms = (ctypes.c_double * 8)(); n = (c_ll * 8)()
        _check(lib().radon_plan_stage_times(self._h, ms, n), "radon_plan_stage_times")
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(self.STAGES)}

    # -- the operators (same names as the C ABI) ------------------------------------------
    def radon_forward(self, x, sino=None):
        import torch

        self._chk(x, torch.float32, self.N * self.N, "x")
        sino = self._new((self.n_angles, self.n_det), torch.float32) if sino is None else sino
        self._chk(sino, torch.float32, self.M, "sino")
        _check(lib().radon_forward(self._h, _ptr(x), _ptr(sino), self._stream()), "radon_forward")
        return sino

    def radon_adjoint(self, sino, x=None):
        import torch

        self._chk(sino, torch.float32, self.M, "sino")
        x = self._new((self.N, self.N), torch.float32) if x is None else x
        self._chk(x, torch.float32, self.N * self.N, "x")
        _check(lib().radon_adjoint(self._h, _ptr(sino), _ptr(x), self._stream()), "radon_adjoint")
        return x

    def radon_inverse(self, sino, x=None):
        import torch

        self._chk(sino, torch.float32, self.M, "sino")
        x = self._new((self.N, self.N), torch.float32) if x is None else x
        self._chk(x, torch.float32, self.N * self.N, "x")
        _check(lib().radon_inverse(self._h, _ptr(sino), _ptr(x), self._stream()), "radon_inverse")
        return x

    def set_filter(self, order: int):
        _check(lib().radon_plan_set_filter(self._h, int(order)), "radon_plan_set_filter")

    def radon_filter(self, sino, out=None, axis=0):
        import torch

        self._chk(sino, torch.float32, self.M, "sino")
        out = self._new((self.n_angles, self.n_det), torch.float32) if out is None else out
        self._chk(out, torch.float32, self.M, "out")
        _check(lib().radon_filter(self._h, _ptr(sino), _ptr(out), int(axis), self._stream()), "radon_filter")
        return out

    def radon_forward_filtered(self, x, sino=None):
        import torch

        self._chk(x, torch.float32, self.N * self.N, "x")
        sino = self._new((self.n_angles, self.n_det), torch.float32) if sino is None else sino
        self._chk(sino, torch.float32, self.M, "sino")
        _check(lib().radon_forward_filtered(self._h, _ptr(x), _ptr(sino), self._stream()), "radon_forward_filtered")
        return sino

    def radon_adjoint_filtered(self, sino, x=None):
        import torch

        self._chk(sino, torch.float32, self.M, "sino")
        x = self._new((self.N, self.N), torch.float32) if x is None else x
        self._chk(x, torch.float32, self.N * self.N, "x")
        _check(lib().radon_adjoint_filtered(self._h, _ptr(sino), _ptr(x), self._stream()), "radon_adjoint_filtered")
        return x

    def radon_solver_step(self, x, b, alpha, tau, filtered=False):
        """x <- S_tau(x - alpha A^T F (A x - b)) in place."""
        import torch

        self._chk(x, torch.float32, self.N * self.N, "x")
        self._chk(b, torch.float32, self.M, "b")
        _check(lib().radon_solver_step(self._h, _ptr(x), _ptr(b), float(alpha), float(tau), int(filtered), self._stream()),
               "radon_solver_step")
        return x

    def radon_solver_run(self, x, b, alpha, tau, n_iter, filtered=False):
        import torch

        self._chk(x, torch.float32, self.N * self.N, "x")
        self._chk(b, torch.float32, self.M, "b")
        _check(lib().radon_solver_run(self._h, _ptr(x), _ptr(b), float(alpha), float(tau), int(filtered), int(n_iter),
                                      self._stream()), "radon_solver_run")
        return x

    def prepare_inverse(self):
        _check(lib().radon_plan_prepare_inverse(self._h), "radon_plan_prepare_inverse")

    def density(self):
        """(D * scale as a CPU float32 tensor of shape (n_angles, n_det), scale)."""
        import torch

        d = torch.empty((self.n_angles, self.n_det), dtype=torch.float32)
        sc = ctypes.c_double()
        _check(lib().radon_plan_density(self._h, _ptr(d), ctypes.byref(sc)), "radon_plan_density")
        return d, float(sc.value)

    def radon_forward_batch(self, x, sino=None):
        import torch

        b = x.shape[0]
        self._chk(x, torch.float32, b * self.N * self.N, "x")
        sino = self._new((b, self.n_angles, self.n_det), torch.float32) if sino is None else sino
        self._chk(sino, torch.float32, b * self.M, "sino")
        _check(lib().radon_forward_batch(self._h, _ptr(x), _ptr(sino), b, self._stream()), "radon_forward_batch")
        return sino

    def radon_adjoint_batch(self, sino, x=None):
        import torch

        b = sino.shape[0]
        self._chk(sino, torch.float32, b * self.M, "sino")
        x = self._new((b, self.N, self.N), torch.float32) if x is None else x
        self._chk(x, torch.float32, b * self.N * self.N, "x")
        _check(lib().radon_adjoint_batch(self._h, _ptr(sino), _ptr(x), b, self._stream()), "radon_adjoint_batch")
        return x

    def radon_forward_host(self, h_x, h_sino):
        """h_x, h_sino: CPU float32 tensors (pinned for overlap) of shapes (b,N,N), (b,n_angles,n_det)."""
        b = h_x.shape[0]
        assert (not h_x.is_cuda) and (not h_sino.is_cuda) and h_x.is_contiguous() and h_sino.is_contiguous()
        assert h_x.numel() == b * self.N * self.N and h_sino.numel() == b * self.M
        _check(lib().radon_forward_host(self._h, _ptr(h_x), _ptr(h_sino), b), "radon_forward_host")
        return h_sino

    def radon_adjoint_host(self, h_sino, h_x):
        b = h_sino.shape[0]
        assert (not h_x.is_cuda) and (not h_sino.is_cuda) and h_x.is_contiguous() and h_sino.is_contiguous()
        assert h_x.numel() == b * self.N * self.N and h_sino.numel() == b * self.M
        _check(lib().radon_adjoint_host(self._h, _ptr(h_sino), _ptr(h_x), b), "radon_adjoint_host")
        return h_x

    def radon_forward_adjoint_host(self, h_x, h_sino, h_xt):
        """h_sino = A h_x and h_xt = A^T h_sino per slice; CPU float32 tensors (pinned for overlap)."""
        b = h_x.shape[0]
        for t in (h_x, h_sino, h_xt):
            assert (not t.is_cuda) and t.is_contiguous()
        assert h_x.numel() == b * self.N * self.N == h_xt.numel() and h_sino.numel() == b * self.M
        _check(lib().radon_forward_adjoint_host(self._h, _ptr(h_x), _ptr(h_sino), _ptr(h_xt), b),
               "radon_forward_adjoint_host")
        return h_sino, h_xt

    def radon_nufft2(self, x, polar=None):
        import torch

        self._chk(x, torch.float32, self.N * self.N, "x")
        polar = self._new((self.n_angles, self.n_det), torch.complex64) if polar is None else polar
        self._chk(polar, torch.complex64, self.M, "polar")
        _check(lib().radon_nufft2(self._h, _ptr(x), _ptr(polar), self._stream()), "radon_nufft2")
        return polar

    def radon_nufft1(self, polar, x=None):
        import torch

        self._chk(polar, torch.complex64, self.M, "polar")
        x = self._new((self.N, self.N), torch.float32) if x is None else x
        self._chk(x, torch.float32, self.N * self.N, "x")
        _check(lib().radon_nufft1(self._h, _ptr(polar), _ptr(x), self._stream()), "radon_nufft1")
        return x

    def radon_interp_only(self, grid, polar=None):
        import torch

        self._chk(grid, torch.complex64, self.G * self.G, "grid")
        polar = self._new((self.n_angles, self.n_det), torch.complex64) if polar is None else polar
        self._chk(polar, torch.complex64, self.M, "polar")
        _check(lib().radon_interp_only(self._h, _ptr(grid), _ptr(polar), self._stream()), "radon_interp_only")
        return polar

    def radon_grid_only(self, polar, grid=None):
        import torch

        self._chk(polar, torch.complex64, self.M, "polar")
        grid = self._new((self.G, self.G), torch.complex64) if grid is None else grid
        self._chk(grid, torch.complex64, self.G * self.G, "grid")
        _check(lib().radon_grid_only(self._h, _ptr(polar), _ptr(grid), self._stream()), "radon_grid_only")
        return grid

    def radon_grid_only_static(self, polar, grid):
        """radon_grid_only with the kernel's scratch in the library's static device arrays: the call
        allocates nothing (the caller passes the output too).  RadonError -6 when the plan needs
        more than RADON_STATIC_SCRATCH_SLOTS = 2048 partial rectangles; calls that overlap on the GPU race."""
        import torch

        self._chk(polar, torch.complex64, self.M, "polar")
        self._chk(grid, torch.complex64, self.G * self.G, "grid")
        _check(lib().radon_grid_only_static(self._h, _ptr(polar), _ptr(grid), self._stream()), "radon_grid_only_static")
        return grid

    def radon_grid_only_paper_bins(self, polar, grid=None, n_bins=4096):
        """The paper's own bins / one-block-per-bin design: comparison only."""
        import torch

        self._chk(polar, torch.complex64, self.M, "polar")
        grid = self._new((self.G, self.G), torch.complex64) if grid is None else grid
        self._chk(grid, torch.complex64, self.G * self.G, "grid")
        _check(lib().radon_grid_only_paper_bins(self._h, _ptr(polar), _ptr(grid), int(n_bins), self._stream()),
               "radon_grid_only_paper_bins")
        return grid

    def paper_bins_stats(self):
        nb, ne, mx, un = c_int(), c_ll(), c_int(), c_int()
        _check(lib().radon_paper_bins_stats(self._h, nb, ne, mx, un), "radon_paper_bins_stats")
        return {"bins": nb.value, "sample_incidences": ne.value, "max_samples_per_bin": mx.value,
                "bins_not_fitting_shared_memory": un.value}

    def radon_proj_ifft(self, polar, sino=None):
        import torch

        self._chk(polar, torch.complex64, self.M, "polar")
        sino = self._new((self.n_angles, self.n_det), torch.float32) if sino is None else sino
        _check(lib().radon_proj_ifft(self._h, _ptr(polar), _ptr(sino), self._stream()), "radon_proj_ifft")
        return sino

    def radon_proj_fft(self, sino, polar=None):
        import torch

        self._chk(sino, torch.float32, self.M, "sino")
        polar = self._new((self.n_angles, self.n_det), torch.complex64) if polar is None else polar
        _check(lib().radon_proj_fft(self._h, _ptr(sino), _ptr(polar), self._stream()), "radon_proj_fft")
        return polar
