"""Pins for the CPU oracle (oracle/) against what the paper and mathematics fix.

None of these compares the oracle with itself or with the CUDA path: each one
ties an oracle function to a closed form, a library routine on a special case,
an invariant, or brute force written independently here (SURVEY.md 8(c) table
"What pins the oracle").
"""
import math

import numpy as np
import pytest
from scipy import integrate, special

import oracle
import workloads

RNG = np.random.default_rng(7)


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


def dirichlet_np(u, n):
    """Closed-form sum_j exp(i 2 pi j u / n)/n over j=-floor(n/2)..ceil(n/2)-1, real part."""
    u = np.asarray(u, dtype=np.float64)
    den = n * np.sin(np.pi * u / n)
    num = np.sin(np.pi * u) * (np.cos(np.pi * u / n) if n % 2 == 0 else 1.0)
    with np.errstate(divide="ignore", invalid="ignore"):
        out = num / den
    out[np.abs(den) < 1e-12] = 1.0
    return out


# ---------------------------------------------------------------- C1 delta ----
@pytest.mark.parametrize("n_det", [33, 48])        # odd and even detector counts
def test_c1_delta_pixel_is_dirichlet_kernel(n_det):
    """delta at (iy0,ix0) => S[a,s] = D_n(t_s - X0 cos - Y0 sin): pins centre,
    sign, orientation, angle direction and scale of the whole (linear) operator."""
    N, n_angles = 32, 20
    for (iy0, ix0) in [(16, 16), (3, 29), (20, 7)]:
        S = oracle.forward(workloads.delta_image(N, iy0, ix0), n_angles, n_det)
        th = np.pi * np.arange(n_angles) / n_angles
        tau = (ix0 - N // 2) * np.cos(th) + (iy0 - N // 2) * np.sin(th)
        t = np.arange(n_det) - n_det // 2
        ref = dirichlet_np(t[None, :] - tau[:, None], n_det)
        assert np.abs(S - ref).max() < 1e-12


def test_c1b_dirichlet_closed_form_function_matches_direct_sum():
    """odirichlet_forward (closed form) == odirect_forward (double sum) on noise."""
    x = RNG.standard_normal((16, 16))
    for n_det in (23, 24):
        assert np.abs(oracle.forward(x, 9, n_det) - oracle.dirichlet_forward(x, 9, n_det)).max() < 1e-11


def test_c1c_closed_form_subset_and_adjoint_match_direct_sums():
    """The closed-form subset/adjoint routines (used for sampled outputs at full sizes)
    against the by-the-definition double sums, odd and even n_det, and the dot test."""
    x = RNG.standard_normal((12, 12)); x[3, 4] = 0.0
    for n_det in (19, 20):
        y = RNG.standard_normal((7, n_det)); y[2, 5] = 0.0
        idx = RNG.choice(7 * n_det, 30, replace=False)
        assert np.abs(oracle.dirichlet_forward_subset(x, 7, n_det, idx)
                      - oracle.forward(x, 7, n_det).ravel()[idx]).max() < 1e-11
        A = oracle.adjoint(y, 12)
        assert np.abs(oracle.dirichlet_adjoint(y, 12) - A).max() < 1e-11
        pix = RNG.choice(144, 17, replace=False)
        assert np.abs(oracle.dirichlet_adjoint(y, 12, pix=pix) - A.ravel()[pix]).max() < 1e-11
        lhs = np.vdot(oracle.dirichlet_forward(x, 7, n_det), y); rhs = np.vdot(x, oracle.dirichlet_adjoint(y, 12))
        assert abs(lhs - rhs) < 1e-11 * abs(lhs)


# --------------------------------------------------- C2 axis-aligned slices ----
def test_c2_axis_rows_are_column_and_row_sums():
    N, n_angles, n_det = 24, 8, 31          # n_det >= N, even n_angles
    x = RNG.standard_normal((N, N))
    S = oracle.forward(x, n_angles, n_det)
    cd, c = n_det // 2, N // 2
    col = np.zeros(n_det); col[cd - c + np.arange(N)] = x.sum(axis=0)
    row = np.zeros(n_det); row[cd - c + np.arange(N)] = x.sum(axis=1)
    assert np.abs(S[0] - col).max() < 1e-12              # theta = 0: t = X
    assert np.abs(S[n_angles // 2] - row).max() < 1e-12  # theta = pi/2: t = Y


def test_c2b_fourier_slice_against_numpy_fft2():
    """n_det == N: the theta=0 radial line of ndft2 is the ky=0 row of fft2(x),
    the theta=pi/2 line the kx=0 column, up to the centring phase."""
    N = 16
    x = RNG.standard_normal((N, N))
    F = oracle.ndft2(x, 2, N)                     # angles 0 and pi/2
    X2 = np.fft.fft2(x)
    c = N // 2
    j = np.arange(N) - c
    phase = np.exp(2j * np.pi * j * c / N)        # image origin at pixel c
    assert np.abs(F[0] - X2[0, j % N] * phase).max() < 1e-11
    assert np.abs(F[1] - X2[j % N, 0] * phase).max() < 1e-11


def test_ndft2_on_cartesian_points_equals_fft2_everywhere():
    """Brute-force check of the 2-D phase: for n_det = N and theta in {0, pi/2} done
    above; here a complex image and the conjugate-transpose pair."""
    N = 8
    x = RNG.standard_normal((N, N)) + 1j * RNG.standard_normal((N, N))
    n_angles, n_det = 5, 9
    F = oracle.ndft2(x, n_angles, n_det)
    # brute force, written independently with a dense matrix
    c, cd = N // 2, n_det // 2
    iy, ix = np.mgrid[0:N, 0:N]
    A = np.empty((n_angles * n_det, N * N), dtype=complex)
    for a in range(n_angles):
        th = math.pi * a / n_angles
        for k in range(n_det):
            w = 2 * math.pi * (k - cd) / n_det
            A[a * n_det + k] = np.exp(-1j * w * ((ix - c) * math.cos(th) + (iy - c) * math.sin(th))).ravel()
    assert np.abs(F.ravel() - A @ x.ravel()).max() < 1e-11
    P = RNG.standard_normal((n_angles, n_det)) + 1j * RNG.standard_normal((n_angles, n_det))
    z = oracle.ndft1(P, N)
    assert np.abs(z.ravel() - A.conj().T @ P.ravel()).max() < 1e-11


# ------------------------------------------------------------ C3 Gaussian ----
def test_c3_gaussian_blob_matches_continuous_radon():
    N, n_angles, n_det, s = 64, 12, 91, 3.5
    x0, y0 = 5.25, -7.5
    S = oracle.forward(workloads.gaussian_blob(N, x0, y0, s), n_angles, n_det)
    th = np.pi * np.arange(n_angles) / n_angles
    tau0 = x0 * np.cos(th) + y0 * np.sin(th)
    t = np.arange(n_det) - n_det // 2
    ref = math.sqrt(2 * math.pi) * s * np.exp(-(t[None, :] - tau0[:, None]) ** 2 / (2 * s * s))
    assert rel(S, ref) < 1e-10
    L = oracle.ray_forward(workloads.gaussian_blob(N, x0, y0, s), n_angles, n_det)
    assert rel(L, ref) < 2e-2


# ---------------------------------------------------- C4 disk chord length ----
def test_c4_disk_chord_length_converges_like_one_over_r():
    errs_d, errs_r = [], []
    radii = [6.0, 12.0, 24.0]
    for r in radii:
        N = 64
        n_angles, n_det = 8, 91
        x0, y0 = 2.5, -1.25
        img = workloads.single_disk(N, x0, y0, r, 0.8)
        th = np.pi * np.arange(n_angles) / n_angles
        tau0 = x0 * np.cos(th) + y0 * np.sin(th)
        t = np.arange(n_det) - n_det // 2
        chord = 2 * 0.8 * np.sqrt(np.maximum(r * r - (t[None, :] - tau0[:, None]) ** 2, 0.0))
        errs_d.append(rel(oracle.forward(img, n_angles, n_det), chord))
        errs_r.append(rel(oracle.ray_forward(img, n_angles, n_det), chord))
    for errs in (errs_d, errs_r):
        for r, e in zip(radii, errs):
            assert e < 0.5 / r, (r, e)
        assert errs[2] < 0.6 * errs[0]      # shrinks with radius


# ------------------------------------------------------- C5 / C6 / C9 ----
def test_c5_mass_conservation():
    x = workloads.make_image(1).astype(np.float64)
    S = oracle.forward(x, 30, 91)
    assert np.abs(S.sum(axis=1) - x.sum()).max() < 1e-9 * abs(x.sum())


@pytest.mark.parametrize("n_det", [21, 22])
def test_c6_adjoint_identity(n_det):
    N, n_angles = 12, 7
    x = RNG.standard_normal((N, N)); y = RNG.standard_normal((n_angles, n_det))
    lhs = np.vdot(oracle.forward(x, n_angles, n_det), y)
    rhs = np.vdot(x, oracle.adjoint(y, N))
    assert abs(lhs - rhs) < 1e-12 * max(abs(lhs), 1.0)


def test_c7_dense_matrix_brute_force_and_transpose():
    """Build A from the Dirichlet closed form (independent of the C double sum) at
    N=8; forward == A x, adjoint == A^T y."""
    N, n_angles, n_det = 8, 6, 11
    c, cd = N // 2, n_det // 2
    iy, ix = np.mgrid[0:N, 0:N]
    A = np.empty((n_angles * n_det, N * N))
    for a in range(n_angles):
        th = math.pi * a / n_angles
        tau = ((ix - c) * math.cos(th) + (iy - c) * math.sin(th)).ravel()
        for s in range(n_det):
            A[a * n_det + s] = dirichlet_np((s - cd) - tau, n_det)
    x = RNG.standard_normal((N, N)); y = RNG.standard_normal((n_angles, n_det))
    assert np.abs(oracle.forward(x, n_angles, n_det).ravel() - A @ x.ravel()).max() < 1e-12
    assert np.abs(oracle.adjoint(y, N).ravel() - A.T @ y.ravel()).max() < 1e-12


def test_c9_invariances_linearity_shift_and_pi_symmetry():
    N, n_det = 16, 25
    x1 = RNG.standard_normal((N, N)); x2 = RNG.standard_normal((N, N))
    f = lambda x, na=6: oracle.forward(x, na, n_det)
    assert np.abs(f(2.0 * x1 - 0.5 * x2) - (2.0 * f(x1) - 0.5 * f(x2))).max() < 1e-11
    # theta -> theta + pi flips the detector: plan with 2*n_angles over [0, 2 pi)
    S = oracle.forward(x1, 12, n_det)[::2]         # angles 0, pi/3 ... -> need [0,2pi): use 2pi*a/12
    # angles pi*a/12 for a=0..11 cover [0,pi); emulate theta+pi by rotating the image 180 deg
    xr = np.zeros_like(x1); xr[1:, 1:] = x1[1:, 1:][::-1, ::-1]   # (X,Y)->(-X,-Y) about c=N/2
    x1m = x1.copy(); x1m[0, :] = 0; x1m[:, 0] = 0
    Sa = oracle.forward(x1m, 5, n_det); Sb = oracle.forward(xr, 5, n_det)
    assert np.abs(Sa - Sb[:, ::-1]).max() < 1e-11   # S_rot[a, s] = S[a, -s] (odd n_det: c_d symmetric)


def test_subset_evaluation_is_exact():
    x = workloads.make_image(1).astype(np.float64)
    full = oracle.forward(x, 10, 91)
    idx = RNG.choice(10 * 91, 50, replace=False)
    assert np.abs(oracle.forward(x, 10, 91, idx=idx) - full.ravel()[idx]).max() < 1e-12
    y = RNG.standard_normal((10, 91))
    fa = oracle.adjoint(y, 64)
    pix = RNG.choice(64 * 64, 40, replace=False)
    assert np.abs(oracle.adjoint(y, 64, pix=pix) - fa.ravel()[pix]).max() < 1e-12


# ------------------------------------------------ O-ray orientation pin ----
def test_oray_orientation_matches_odirect_on_offcentre_disk():
    N, n_angles, n_det = 64, 16, 91
    img = workloads.single_disk(N, 14.0, -9.0, 7.0, 1.0)
    S = oracle.forward(img, n_angles, n_det); L = oracle.ray_forward(img, n_angles, n_det)
    assert rel(L, S) < 0.08
    # peak position follows tau0 = x0 cos + y0 sin for every angle (orientation, centre)
    th = np.pi * np.arange(n_angles) / n_angles
    tau0 = 14.0 * np.cos(th) - 9.0 * np.sin(th)
    for Z in (S, L):
        com = (Z * (np.arange(n_det) - n_det // 2)[None, :]).sum(1) / Z.sum(1)
        assert np.abs(com - tau0).max() < 0.05


# ------------------------------------------------------ Kaiser-Bessel pins ----
def test_kb_i0_against_scipy_and_kernel_special_values():
    for z in (0.0, 0.3, 2.0, 13.8551, 30.0):
        assert abs(oracle.kb_i0(z) - special.i0(z)) < 1e-13 * special.i0(z)
    beta = oracle.kb_beta(6, 2.0)
    assert abs(beta - math.pi * math.sqrt(9 * 2.25 - 0.8)) < 1e-14      # 13.8551...
    assert abs(beta - 13.8551) < 1e-4
    assert abs(oracle.kb_phi(0.0) - 1.0) < 1e-15
    assert abs(oracle.kb_phi(3.0) - 1.0 / special.i0(beta)) < 1e-18
    assert oracle.kb_phi(3.0000001) == 0.0
    u = np.linspace(-3, 3, 41)
    assert np.abs(oracle.kb_phi(u) - oracle.kb_phi(-u)).max() == 0.0


def test_kb_fourier_transform_closed_form_against_quadrature():
    """phihat(xi) closed form == numerical integral of phi(u) cos(2 pi xi u)."""
    beta = oracle.kb_beta()
    for xi in (0.0, 0.1, 0.25, 0.5, 0.74, 0.9):       # incl. beyond sqrt: beta/(pi W) = 0.735
        num, _ = integrate.quad(lambda u: float(oracle.kb_phi(u)) * math.cos(2 * math.pi * xi * u),
                                -3, 3, epsabs=1e-13, epsrel=1e-13, limit=200)
        assert abs(num - float(oracle.kb_phihat(xi))) < 1e-10


# -------------------------------------------------------------- O-grid pins ----
def test_ogrid_interp_of_plane_wave_is_deapodised_exponential():
    """Inverse gridding (eq :87) of G_r[k] = exp(-i 2 pi k.X/G) returns
    phihat(X/G) phihat(Y/G) exp(-i 2 pi kappa.X/G) up to the aliasing error of the
    kernel (W=6, sigma=2: ~1e-5 relative for |X| <= G/4): ties tap selection,
    kernel, centred layout and the de-apodisation formula together."""
    G, n_angles, n_det = 64, 7, 45
    k = np.arange(G) - G // 2
    for (X, Y) in [(0, 0), (5, -3), (-16, 15), (11, 16)]:
        grid = np.exp(-2j * np.pi * (k[None, :] * X + k[:, None] * Y) / G)
        P = oracle.grid_interp(grid, n_angles, n_det)
        th = np.pi * np.arange(n_angles) / n_angles
        rho = G * (np.arange(n_det) - n_det // 2) / n_det
        kx = rho[None, :] * np.cos(th)[:, None]; ky = rho[None, :] * np.sin(th)[:, None]
        hx, hy = float(oracle.kb_phihat(X / G)), float(oracle.kb_phihat(Y / G))
        ref = hx * hy * np.exp(-2j * np.pi * (kx * X + ky * Y) / G)
        # Poisson summation: P - ref = sum over aliases phihat(X/G + p), p != 0; for
        # Kaiser-Bessel W=6, sigma=2, beta=13.855 and |X| <= G/4 that is the method's
        # design accuracy, ~1e-5 relative (1.03e-5 worst case, corner pixel)
        err = np.abs(P - ref).max() / abs(hx * hy)
        assert 1e-8 < err < 3e-5, (X, Y, err)   # 2-D corner: ~2x the 1-D 1.03e-5


def test_ogrid_grid_is_transpose_of_interp_and_brute_force():
    G, n_angles, n_det = 16, 5, 13
    grid = RNG.standard_normal((G, G)) + 1j * RNG.standard_normal((G, G))
    P = RNG.standard_normal((n_angles, n_det)) + 1j * RNG.standard_normal((n_angles, n_det))
    lhs = np.vdot(P, oracle.grid_interp(grid, n_angles, n_det))
    rhs = np.vdot(oracle.grid_grid(P, G), grid)
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    # brute force with scipy's I0 and an independently written tap loop
    beta = math.pi * math.sqrt((6 / 2.0) ** 2 * 1.5 ** 2 - 0.8)
    phi = lambda u: special.i0(beta * math.sqrt(max(1 - (u / 3) ** 2, 0))) / special.i0(beta) if abs(u) <= 3 else 0.0
    out = np.zeros((n_angles, n_det), dtype=complex)
    for a in range(n_angles):
        for kk in range(n_det):
            rho = G * (kk - n_det // 2) / n_det
            kx, ky = rho * math.cos(math.pi * a / n_angles), rho * math.sin(math.pi * a / n_angles)
            for yy in range(math.ceil(ky - 3), math.ceil(ky - 3) + 6):
                for xx in range(math.ceil(kx - 3), math.ceil(kx - 3) + 6):
                    out[a, kk] += grid[(yy + G // 2) % G, (xx + G // 2) % G] * phi(xx - kx) * phi(yy - ky)
    assert np.abs(out - oracle.grid_interp(grid, n_angles, n_det)).max() < 1e-12


# ------------------------------ O-alg gated against O-direct (error bound) ----
def test_fast_algorithm_within_kernel_error_bound_of_exact_operator():
    """'the exact result within the method's error bound': the fp64 fast algorithm
    (O-alg) must sit within the KB W=6, sigma=2 aliasing bound of O-direct -- and
    not far below it (C8: an error << 1e-6 would mean comparing a method with itself)."""
    x = workloads.make_image(1).astype(np.float64)
    S = oracle.forward(x, 90, 91)
    Sf = oracle.fast_forward(x, 90, 91)
    e = rel(Sf, S)
    assert 5e-7 < e < 1e-5
    y = S
    A = oracle.adjoint(y, 64); Af = oracle.fast_adjoint(y, 64)
    e = rel(Af, A)
    assert 5e-7 < e < 1e-5
    # bare NUFFT on white noise and a corner pixel (gate G2 inputs): <= 1e-4
    for img in (workloads.white_noise(32, 3), workloads.delta_image(32, 0, 31)):
        e = rel(oracle.fast_nufft2(img, 16, 45), oracle.ndft2(img.astype(np.float64), 16, 45))
        assert e < 1e-4
    # adjointness of the fast pair is exact (W-independent): C6 for O-alg
    x2 = RNG.standard_normal((64, 64)); y2 = RNG.standard_normal((90, 91))
    lhs = np.vdot(oracle.fast_forward(x2, 90, 91), y2); rhs = np.vdot(x2, oracle.fast_adjoint(y2, 64))
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)


def test_golden_regression_fixture():
    """tests/golden/odirect_tiny.txt (written by make_golden.py from oracle/ only) still
    matches: guards the oracle's arithmetic against accidental edits."""
    import os
    import sys

    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    sys.path.insert(0, here)
    import make_golden

    ref = np.loadtxt(os.path.join(here, "odirect_tiny.txt"))
    got = make_golden.compute()
    assert ref.shape == got.shape
    assert np.abs(ref - got).max() < 1e-12 * np.abs(ref).max()


# ---- O-density / inverse Radon -----------------
def test_density_band_scan_equals_the_double_sum_as_printed():
    """PAPER.md:89 written out as the O(M^2) double sum (every term) against the evaluation that
    skips the exactly-zero terms (sort on y, scan of the band).  Shapes: odd and even n_det,
    coincident j = 0 samples, samples at the grid edge |kappa| = G/2 (even n_det, k = 0), a
    single angle, and config 1 (90 x 91, G = 128)."""
    for (na, nd, G) in [(12, 21, 32), (9, 16, 16), (5, 33, 64), (1, 8, 16), (30, 64, 64), (90, 91, 128)]:
        Db = oracle.density(na, nd, G, brute=True)
        Df = oracle.density(na, nd, G)
        assert np.max(np.abs(Db / Df - 1)) < 1e-13, (na, nd, G)


def test_density_special_values_and_ramp():
    """All n_angles samples with j = 0 coincide at kappa = 0 and see the same neighbourhood, so
    they share one D <= 1/n_angles (K(0,0) = 1 for each of them); an isolated sample has D = 1;
    between DC and the band edge D follows the polar area element, D ~ |j| (the ramp filter)."""
    na, nd, G = 90, 91, 128
    D = oracle.density(na, nd, G, brute=True)
    c = nd // 2
    assert np.ptp(D[:, c]) < 1e-12 * D[0, c] and D[0, c] < 1.0 / na
    assert abs(oracle.density(1, 2, 64, brute=True)[0, 1] - 1.0) < 1e-12          # two samples 32 cells apart
    j = np.arange(8, 33)
    ratio = D[10, c + j] / j
    assert np.max(np.abs(ratio / ratio.mean() - 1)) < 0.01
    assert np.allclose(D[:, c + j], D[:, c - j], rtol=1e-9)            # point symmetry of the sample set


@pytest.mark.parametrize("na,nd,G", [(90, 91, 128), (180, 181, 256)])
def test_density_times_scale_is_the_polar_area_element(na, nd, G):
    """Absolute level of D * inverse_scale (reading R-scale) against a closed
    form that does not involve the kernel: the inverse Fourier integral
    x(X) = (1/4 pi^2) int xhat(w) exp(i w.X) d^2 w on the polar samples w = (2 pi j/n)(cos, sin),
    xhat = n Yhat, has the area element |w| dw dtheta = (2 pi |j|/n)(2 pi/n)(pi/n_angles), i.e. the
    weight pi |j| / (n n_angles) per sample.  Where the samples are dense against the kernel width
    (radial spacing G/n = 1.41 cells here, angular spacing below that for |j| <= n/3) eq. :89 must
    reproduce it: <= 1 % for 8 <= |j| <= n/3, every angle.  (At radial spacing 2 cells, e.g.
    n = G/2, the sum over K undersamples the kernel and eq. :89 sits 7 % below the area element:
    a property of the formula as printed, the same on both sides.)"""
    D = oracle.density(na, nd, G) * oracle.inverse_scale(nd, G)
    c = nd // 2
    j = np.arange(8, nd // 3)
    area = np.pi * j / (nd * na)
    for sgn in (+1, -1):
        ratio = D[:, c + sgn * j] / area[None, :]
        assert np.max(np.abs(ratio - 1)) < 0.01, float(np.max(np.abs(ratio - 1)))
    # and the level is not an accident of one shape: the two geometries agree on the mean ratio
    assert abs(np.mean(D[:, c + j] / area[None, :]) - 1) < 0.005


def test_inverse_recovers_a_gaussian_blob():
    """inverse(forward(x)) ~ x for a band-limited blob (filtered-back-projection quality: the
    kernel-smoothed density of eq. :89 is not the exact ramp near DC)."""
    N, na, nd = 64, 90, 91
    x = workloads.gaussian_blob(N, 5.0, -7.0, 4.0)
    xr = oracle.inverse(oracle.forward(x, na, nd), N, brute=True)
    assert rel(xr, x) < 0.10
    assert abs(xr.max() / x.max() - 1) < 0.02
    iy, ix = np.unravel_index(np.argmax(xr), xr.shape)
    assert (iy, ix) == (N // 2 - 7, N // 2 + 5)
    # a pixel subset is exact (independent sums)
    pix = np.array([5, 77, N * N - 1, (N // 2 - 7) * N + N // 2 + 5])
    assert np.allclose(oracle.inverse(oracle.forward(x, na, nd), N, pix=pix), xr.ravel()[pix], rtol=1e-12, atol=1e-14)


# ---------------------------------------------------------------- O-filter / O-solver ----
@pytest.mark.parametrize("axis", [0, 1])
def test_filter_annihilates_polynomials_and_is_an_orthogonal_projector(axis):
    """PAPER.md:27 "3rd order polynomial fit ... polynomial subtraction" (:41): whatever the
    basis used, fit-and-subtract of degree p is I - P with P the orthogonal projector onto the
    polynomials of degree <= p sampled on the line: it maps every such polynomial to zero, is
    idempotent and symmetric.  None of this uses the oracle's own Vandermonde matrix."""
    shape = (37, 53)
    n = shape[axis]
    s = np.arange(n, dtype=np.float64)
    for order in (0, 1, 3, 5):
        poly = sum(RNG.standard_normal() * (s / n - 0.3) ** d for d in range(order + 1))
        z = np.moveaxis(np.broadcast_to(poly, (shape[1 - axis], n)).copy() * RNG.standard_normal((shape[1 - axis], 1)), -1, axis)
        assert np.abs(oracle.polyfilter(z, order, axis)).max() < 1e-9 * np.abs(z).max()
        y, w = RNG.standard_normal(shape), RNG.standard_normal(shape)
        Fy = oracle.polyfilter(y, order, axis)
        assert np.abs(oracle.polyfilter(Fy, order, axis) - Fy).max() < 1e-11              # F F = F
        assert abs(np.vdot(Fy, w) - np.vdot(y, oracle.polyfilter(w, order, axis))) < 1e-10  # F^T = F
        # a polynomial of degree order + 1 is NOT annihilated (the degree is what it says)
        assert np.abs(oracle.polyfilter(np.moveaxis(np.broadcast_to(s ** (order + 1), (shape[1 - axis], n)), -1, axis),
                                        order, axis)).max() > 1e-3


def test_filter_closed_forms_and_library_fit():
    """order 0 = subtract the mean; order 1 = subtract the regression line with slope
    cov(s,z)/var(s) (textbook closed forms); any order = the residual of numpy's own
    polynomial least-squares routine (a different algorithm: QR/SVD on a scaled basis)."""
    y = RNG.standard_normal((9, 41))
    assert np.abs(oracle.polyfilter(y, 0) - (y - y.mean(axis=1, keepdims=True))).max() < 1e-12
    s = np.arange(41.0)
    sc = s - s.mean()
    slope = (y * sc).sum(axis=1, keepdims=True) / (sc * sc).sum()
    assert np.abs(oracle.polyfilter(y, 1) - (y - y.mean(axis=1, keepdims=True) - slope * sc)).max() < 1e-12
    for order in (2, 3, 4):
        c = np.polynomial.polynomial.polyfit(s, y.T, order)             # (order+1, 9)
        fit = np.polynomial.polynomial.polyval(s, c)                     # (9, 41)
        assert np.abs(oracle.polyfilter(y, order) - (y - fit)).max() < 1e-10
        assert np.abs(oracle.polyfilter(y.T, order, axis=0) - (y - fit).T).max() < 1e-10


def test_filter_leaves_fast_oscillations_alone():
    """The filter removes slowly varying background only: the alternating sequence (-1)^s has
    inner product at most ~sqrt((2d+1)/n) with the unit-norm degree-d polynomial (it only
    sees the polynomial's variation over one sample), so ||z - F z|| <= (p+1) ||z|| / sqrt(n)."""
    for n in (91, 725, 2048):
        z = ((-1.0) ** np.arange(n))[None, :]
        d = oracle.polyfilter(z, 3) - z
        assert np.linalg.norm(d) / np.linalg.norm(z) < 4.0 / np.sqrt(n)


def test_soft_threshold_and_ista_step_follow_their_definitions():
    """S_tau is the proximal map of tau |.|: it minimises (1/2)(u - v)^2 + tau |u| (checked by
    brute force on a fine grid); one ISTA step on the dense matrix of config-0-sized operator equals
    the same formula written with explicit matrices (A from the closed form D_n, pin C7)."""
    v = np.array([-2.0, -0.3, 0.0, 0.2, 1.7]); tau = 0.5
    u = np.linspace(-3, 3, 60001)
    brute = np.array([u[np.argmin(0.5 * (u - vi) ** 2 + tau * np.abs(u))] for vi in v])
    assert np.abs(oracle.soft_threshold(v, tau) - brute).max() < 2e-4
    N, n_angles, n_det = 8, 5, 9
    th = np.pi * np.arange(n_angles) / n_angles
    X = (np.arange(N) - N // 2)[None, :].repeat(N, 0).ravel(); Y = (np.arange(N) - N // 2)[:, None].repeat(N, 1).ravel()
    t = np.arange(n_det) - n_det // 2
    A = np.stack([dirichlet_np(t[k % n_det] - (X * np.cos(th[k // n_det]) + Y * np.sin(th[k // n_det])), n_det)
                  for k in range(n_angles * n_det)])
    x = RNG.standard_normal((N, N)); b = RNG.standard_normal((n_angles, n_det)); alpha, tau = 0.01, 0.05
    fwd = lambda u: oracle.forward(u, n_angles, n_det)
    adj = lambda y: oracle.adjoint(y, N)
    got = oracle.ista_step(x, b, alpha, tau, fwd, adj)
    g = A.T @ (A @ x.ravel() - b.ravel())
    w = x.ravel() - alpha * g
    ref = np.sign(w) * np.maximum(np.abs(w) - tau, 0)
    assert np.abs(got.ravel() - ref).max() < 1e-12
    # with the filter: gradient of (1/2)||F(Ax - b)||^2 by central differences
    got_f = oracle.ista_step(x, b, alpha, 0.0, fwd, adj, order=3)
    f = lambda u: 0.5 * np.sum(oracle.polyfilter((A @ u).reshape(n_angles, n_det) - b, 3) ** 2)
    e = np.zeros(N * N); grad = np.zeros(N * N)
    for i in range(N * N):
        e[:] = 0; e[i] = 1e-5
        grad[i] = (f(x.ravel() + e) - f(x.ravel() - e)) / 2e-5
    assert np.abs(got_f.ravel() - (x.ravel() - alpha * grad)).max() < 1e-8
