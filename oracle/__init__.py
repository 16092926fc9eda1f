"""CPU oracle for the NUFFT-Radon hot path (fp64, plain C + numpy).

TEST INFRASTRUCTURE ONLY: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package.  It shares no code with ``paper_1009_1380_b200`` and never imports it.

Functions (each cites the passage it follows; details in radon_oracle.c):

* ``forward`` / ``adjoint``      O-direct, the operator's definition
  (SURVEY.md 8(c) items 1-3).  ``idx`` / ``pix`` evaluate a subset
  of outputs (each output is an independent sum, so a subset is exact).
* ``ndft2`` / ``ndft1``          bare non-uniform DFT and its conjugate transpose.
* ``dirichlet_forward`` / ``dirichlet_forward_subset`` / ``dirichlet_adjoint``
  closed form of the same operator (periodic-sinc detector response): the second,
  independent implementation used by the pins, and -- because one output costs N^2
  (forward) or M (adjoint) terms instead of a whole radial line -- the form used for
  sampled outputs at BASELINE.json's full sizes.
* ``ray_forward``                O-ray, ray-sampled line integral (north_star).
* ``kb_*``, ``grid_interp``, ``grid_grid``  O-grid: the two sums printed with
  Fig. 5 with a directly evaluated Kaiser-Bessel kernel.
* ``fast_forward`` / ``fast_adjoint``  O-alg: the paper's fast algorithm
   step by step in fp64 -- de-apodise + zero-pad, 2-D FFT
  (numpy, a library primitive), inverse gridding (eq. :87), 1-D inverse DFT --
  used to separate algorithmic error from fp32 round-off.  Gated against
  O-direct in the pins before it is trusted.

* ``density`` / ``inverse``  O-density: D(x_i,y_i) = 1/sum_j K(x_i-x_j, y_i-y_j)
   and the density-compensated inverse Radon transform (PAPER.md:51,
  :85): weights times the exact adjoint NDFT.

* ``polyfilter``  O-filter: the sinogram filter of the paper's objective
  ("3rd order polynomial fit"; filter(Radon{x} - data), :31, :47):
  least-squares polynomial fit along one axis of the sinogram, subtracted.
* ``ista_step``   O-solver: one iteration x <- S_tau(x - alpha A^T F (A x - b)) of the
  iterative soft-thresholding stand-in for the solver loop,
  on any (forward, adjoint) pair of this module.

All pinned in tests/test_oracle_pins.py; nothing here is
"parity unpinned".
"""
import ctypes
import os

import numpy as np

from .build import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        path = _build()
        lib = ctypes.CDLL(path)
        D = ctypes.POINTER(ctypes.c_double)
        L = ctypes.POINTER(ctypes.c_longlong)
        I, LL, DBL = ctypes.c_int, ctypes.c_longlong, ctypes.c_double
        lib.oracle_num_threads.restype = I
        lib.oracle_set_num_threads.argtypes = [I]
        lib.odirect_ndft2.argtypes = [D, D, I, I, I, L, LL, D, D]
        lib.odirect_ndft1.argtypes = [D, D, I, I, I, L, LL, D, D]
        lib.odirect_forward.argtypes = [D, I, I, I, L, LL, D]
        lib.odirect_adjoint.argtypes = [D, I, I, I, L, LL, D]
        lib.odirichlet_forward.argtypes = [D, I, I, I, D]
        lib.odirichlet_forward_subset.argtypes = [D, I, I, I, L, LL, D]
        lib.odirichlet_adjoint.argtypes = [D, I, I, I, L, LL, D]
        lib.oray_forward.argtypes = [D, I, I, I, DBL, D]
        lib.okb_i0.argtypes = [DBL]; lib.okb_i0.restype = DBL
        lib.okb_beta.argtypes = [I, DBL]; lib.okb_beta.restype = DBL
        lib.okb_phi.argtypes = [DBL, I, DBL]; lib.okb_phi.restype = DBL
        lib.okb_phihat.argtypes = [DBL, I, DBL]; lib.okb_phihat.restype = DBL
        lib.ogrid_interp.argtypes = [D, D, I, I, I, I, DBL, D, D]
        lib.ogrid_grid.argtypes = [D, D, I, I, I, I, DBL, D, D]
        lib.odensity.argtypes = [I, I, I, I, DBL, I, D]
        _lib = lib
    return _lib


def _d(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _l(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _idx(idx):
    if idx is None:
        return None, 0
    idx = np.ascontiguousarray(idx, dtype=np.int64).ravel()
    return idx, idx.size


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


# ---- O-direct ---------------------------------------------------------------

def ndft2(x, n_angles, n_det, idx=None):
    """F[a,k] = sum x exp(-i (2 pi j/n)(X cos + Y sin)); x real or complex (N,N)."""
    lib = _load()
    x = np.asarray(x)
    N = x.shape[0]
    xr = _f64(x.real)
    xi = _f64(x.imag) if np.iscomplexobj(x) else None
    idx, n_idx = _idx(idx)
    cnt = n_idx if idx is not None else n_angles * n_det
    Fr = np.empty(cnt); Fi = np.empty(cnt)
    lib.odirect_ndft2(_d(xr), _d(xi) if xi is not None else None, N, n_angles, n_det,
                      _l(idx), n_idx, _d(Fr), _d(Fi))
    F = Fr + 1j * Fi
    return F if idx is not None else F.reshape(n_angles, n_det)


def ndft1(P, N, pix=None):
    """Conjugate transpose of ndft2: z[iy,ix] = sum P exp(+i ...); P complex (n_angles,n_det)."""
    lib = _load()
    P = np.asarray(P)
    n_angles, n_det = P.shape
    Pr = _f64(P.real); Pi = _f64(P.imag) if np.iscomplexobj(P) else np.zeros_like(Pr)
    pix, n_pix = _idx(pix)
    cnt = n_pix if pix is not None else N * N
    zr = np.empty(cnt); zi = np.empty(cnt)
    lib.odirect_ndft1(_d(Pr), _d(Pi), N, n_angles, n_det, _l(pix), n_pix, _d(zr), _d(zi))
    z = zr + 1j * zi
    return z if pix is not None else z.reshape(N, N)


def forward(x, n_angles, n_det, idx=None):
    """y = Radon{x} (O-direct).  Returns (n_angles,n_det) or the listed entries."""
    lib = _load()
    x = _f64(x)
    N = x.shape[0]
    idx, n_idx = _idx(idx)
    cnt = n_idx if idx is not None else n_angles * n_det
    S = np.empty(cnt)
    lib.odirect_forward(_d(x), N, n_angles, n_det, _l(idx), n_idx, _d(S))
    return S if idx is not None else S.reshape(n_angles, n_det)


def adjoint(y, N, pix=None):
    """x~ = Radon^T{y} (O-direct, exact transpose of forward)."""
    lib = _load()
    y = _f64(y)
    n_angles, n_det = y.shape
    pix, n_pix = _idx(pix)
    cnt = n_pix if pix is not None else N * N
    xt = np.empty(cnt)
    lib.odirect_adjoint(_d(y), N, n_angles, n_det, _l(pix), n_pix, _d(xt))
    return xt if pix is not None else xt.reshape(N, N)


def dirichlet_forward(x, n_angles, n_det):
    lib = _load()
    x = _f64(x)
    S = np.empty((n_angles, n_det))
    lib.odirichlet_forward(_d(x), x.shape[0], n_angles, n_det, _d(S))
    return S


def dirichlet_forward_subset(x, n_angles, n_det, idx):
    """Listed sinogram entries q = a*n_det + s by the closed form (N^2 terms each)."""
    lib = _load()
    x = _f64(x)
    idx, n_idx = _idx(idx)
    S = np.empty(n_idx)
    lib.odirichlet_forward_subset(_d(x), x.shape[0], n_angles, n_det, _l(idx), n_idx, _d(S))
    return S


def dirichlet_adjoint(y, N, pix=None):
    """Transpose by the closed form; listed pixels p = iy*N + ix (None: all), M terms each."""
    lib = _load()
    y = _f64(y)
    n_angles, n_det = y.shape
    pix, n_pix = _idx(pix)
    cnt = n_pix if pix is not None else N * N
    xt = np.empty(cnt)
    lib.odirichlet_adjoint(_d(y), N, n_angles, n_det, _l(pix), n_pix, _d(xt))
    return xt if pix is not None else xt.reshape(N, N)


def ray_forward(x, n_angles, n_det, h=0.25):
    lib = _load()
    x = _f64(x)
    L = np.empty((n_angles, n_det))
    lib.oray_forward(_d(x), x.shape[0], n_angles, n_det, float(h), _d(L))
    return L


# ---- O-grid -----------------------------------------------------------------

def kb_i0(z):
    return float(_load().okb_i0(float(z)))


def kb_beta(W=6, sigma=2.0):
    return float(_load().okb_beta(int(W), float(sigma)))


def kb_phi(u, W=6, beta=None):
    lib = _load()
    beta = kb_beta(W) if beta is None else beta
    u = np.asarray(u, dtype=np.float64)
    return np.vectorize(lambda t: lib.okb_phi(float(t), int(W), float(beta)))(u)


def kb_phihat(xi, W=6, beta=None):
    lib = _load()
    beta = kb_beta(W) if beta is None else beta
    xi = np.asarray(xi, dtype=np.float64)
    return np.vectorize(lambda t: lib.okb_phihat(float(t), int(W), float(beta)))(xi)


def grid_interp(grid, n_angles, n_det, W=6, sigma=2.0):
    """Inverse gridding.  grid: complex (G,G), centred layout."""
    lib = _load()
    grid = np.asarray(grid)
    G = grid.shape[0]
    gr = _f64(grid.real); gi = _f64(grid.imag)
    pr = np.empty(n_angles * n_det); pi = np.empty(n_angles * n_det)
    lib.ogrid_interp(_d(gr), _d(gi), G, n_angles, n_det, W, kb_beta(W, sigma), _d(pr), _d(pi))
    return (pr + 1j * pi).reshape(n_angles, n_det)


def grid_grid(polar, G, W=6, sigma=2.0):
    """Gridding, PAPER.md:85 with D == 1.  polar: complex (n_angles,n_det)."""
    lib = _load()
    polar = np.asarray(polar)
    n_angles, n_det = polar.shape
    pr = _f64(polar.real); pi = _f64(polar.imag)
    gr = np.empty(G * G); gi = np.empty(G * G)
    lib.ogrid_grid(_d(pr), _d(pi), G, n_angles, n_det, W, kb_beta(W, sigma), _d(gr), _d(gi))
    return (gr + 1j * gi).reshape(G, G)


# ---- O-alg: the paper's fast algorithm, step by step, fp64 -------------------

def _deapod(N, G, W, sigma):
    """d[X] = 1/phihat(X/G), X = -N/2 .. N/2-1 stored at index X + N//2."""
    X = np.arange(N) - N // 2
    return 1.0 / kb_phihat(X / float(G), W, kb_beta(W, sigma))


def _centered_dft_matrix(n, sign):
    """E[k,s] = exp(sign * i 2 pi (k-c)(s-c)/n), c = n//2."""
    c = n // 2
    j = (np.arange(n) - c)[:, None]
    t = (np.arange(n) - c)[None, :]
    return np.exp(sign * 2j * np.pi * ((j * t) % n) / n)


def fast_nufft2(x, n_angles, n_det, W=6, sigma=2.0):
    """Steps F1-F3: de-apodise + zero-pad, 2-D FFT, inverse gridding."""
    x = _f64(x)
    N = x.shape[0]
    G = int(round(sigma * N))
    d = _deapod(N, G, W, sigma)
    u = np.zeros((G, G))
    c = N // 2
    X = np.arange(N) - c
    u[np.ix_(X % G, X % G)] = x * d[None, :] * d[:, None]
    U = np.fft.fftshift(np.fft.fft2(u))        # centred layout, DC at (G/2,G/2)
    return grid_interp(U, n_angles, n_det, W, sigma)


def fast_forward(x, n_angles, n_det, W=6, sigma=2.0):
    """PAPER.md:51 in order: 2-D FFT, interpolate onto the polar grid (gridding,
    :53-55, eq :87), 1-D inverse transforms along the radial lines; real part."""
    F = fast_nufft2(x, n_angles, n_det, W, sigma)
    E = _centered_dft_matrix(n_det, +1)       # [k, s]
    return np.real(F @ E) / n_det


def fast_nufft1(P, N, W=6, sigma=2.0):
    """Steps A2-A4: gridding (eq :85, D==1), 2-D inverse FFT, crop, de-apodise; complex result."""
    P = np.asarray(P)
    G = int(round(sigma * N))
    grid = grid_grid(P, G, W, sigma)
    v = np.fft.ifft2(np.fft.ifftshift(grid)) * (G * G)   # unnormalised inverse
    d = _deapod(N, G, W, sigma)
    X = np.arange(N) - N // 2
    return v[np.ix_(X % G, X % G)] * d[None, :] * d[:, None]


def fast_adjoint(y, N, W=6, sigma=2.0):
    y = _f64(y)
    n_angles, n_det = y.shape
    E = _centered_dft_matrix(n_det, -1)        # [k, s]
    Yh = (y @ E.T) / n_det
    return np.real(fast_nufft1(Yh, N, W, sigma))


# ---- O-density / inverse Radon ---------------

def density(n_angles, n_det, G, W=6, sigma=2.0, brute=False):
    """D(x_i,y_i) = 1 / sum_j K(x_i - x_j, y_i - y_j) over all polar samples.
    brute=True: all M^2 terms as printed.  brute=False: the terms that are exactly zero (|dy| or
    |dx| > W/2) are skipped by a sort on the y coordinate and a scan of the band (no cell buckets:
    deliberately a different algorithm from the product's bucketed table)."""
    lib = _load()
    D = np.empty(n_angles * n_det)
    lib.odensity(n_angles, n_det, G, W, kb_beta(W, sigma), int(bool(brute)), _d(D))
    return D.reshape(n_angles, n_det)


def inverse_scale(n_det, G, W=6, sigma=2.0):
    """Quadrature weight that turns D into an area element of the image's Fourier plane:
    sum_j K ~ (samples per grid cell) * (integral of K) = rho * phihat(0)^2, so a sample owns
    D * phihat(0)^2 grid cells = D * phihat(0)^2 (2 pi / G)^2 (rad/pixel)^2, and the inverse
    Fourier integral (1/4 pi^2) int xhat e^{i w.X} d^2 w over samples xhat = n * Yhat becomes
    sum_m Yhat_m e^{...} D_m * n phihat(0)^2 / G^2.
    Pinned (tests/test_oracle_pins.py) against the polar area element the same integral gives
    directly: D * inverse_scale -> pi |j| / (n_det n_angles) in the mid band."""
    ph0 = float(kb_phihat(0.0, W, kb_beta(W, sigma)))
    return n_det * ph0 * ph0 / float(G * G)


def inverse(y, N, sigma=2.0, W=6, pix=None, brute=False):
    """Density-compensated inverse Radon transform ("inverse Radon", eq. :85 with
    the D of eq. :89): 1-D DFT of every projection, weights D, exact adjoint NDFT, real part."""
    y = _f64(y)
    n_angles, n_det = y.shape
    G = int(round(sigma * N))
    E = _centered_dft_matrix(n_det, -1)
    Yh = (y @ E.T) / n_det
    D = density(n_angles, n_det, G, W, sigma, brute=brute)
    return np.real(ndft1(Yh * D, N, pix=pix)) * inverse_scale(n_det, G, W, sigma)


# ---- O-filter / O-solver ----------------

def polyfilter(sino, order=3, axis=1):
    """filter(.) of PAPER.md:31/:47 under reading R-filter: along `axis` of
    the sinogram (1: the detector coordinate of every projection, the default; 0: the angle
    coordinate of every detector bin) fit a polynomial of degree `order` by least squares
    ("3rd order polynomial fit") and subtract it ("polynomial subtraction", :41).
    Plain normal equations on the Vandermonde matrix of t in [-1, 1], fp64."""
    z = np.moveaxis(_f64(sino), axis, -1)
    n = z.shape[-1]
    t = np.linspace(-1.0, 1.0, n) if n > 1 else np.zeros(1)
    V = np.vander(t, order + 1, increasing=True)            # n x (order + 1)
    coef = np.linalg.solve(V.T @ V, V.T @ z[..., None])     # normal equations, one right-hand side per line
    out = z - (V @ coef)[..., 0]
    return np.moveaxis(out, -1, axis)


def soft_threshold(v, tau):
    """S_tau(v) = sign(v) max(|v| - tau, 0): the proximal map of tau ||.||_1."""
    v = _f64(v)
    return np.sign(v) * np.maximum(np.abs(v) - tau, 0.0)


def ista_step(x, b, alpha, tau, fwd, adj, order=None):
    """One iteration of x <- S_tau(x - alpha A^T F (A x - b)), F = polyfilter(order) or the
    identity (order None): the gradient step on (1/2)||F(Ax - b)||^2 (F is an orthogonal
    projector: F^T F = F) followed by the l1 shrinkage, the building block a basis-pursuit
    solver repeats around y = Radon{x}.  fwd(x) / adj(y): the operator pair."""
    r = fwd(x) - _f64(b)
    if order is not None:
        r = polyfilter(r, order)
    return soft_threshold(_f64(x) - alpha * adj(r), tau)
