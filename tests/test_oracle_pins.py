"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Each test cites the passage (P:<line> = /root/reference/PAPER.md line) or the SURVEY 8(c) pin it
implements.  Nothing here re-types the oracle's own formulas: the references are closed forms,
scipy.special.sph_harm_y, mpmath at 60+ digits, numpy brute force, or dense matrices.
"""
import math
import os

import numpy as np
import pytest
from scipy.special import sph_harm_y

import oracle
from paper_2510_01785_b200 import synth


def pix_angles(nside):
    """theta, phi of every RING pixel from the oracle's ring table."""
    th, ph = [], []
    for ring in range(1, 4 * nside):
        n, start, c, s, phi0 = oracle.ring_geometry(nside, ring)
        assert start == len(th)
        th += [math.atan2(s, c)] * n
        ph += [phi0 + 2.0 * math.pi * x / n for x in range(n)]
    return np.array(th), np.array(ph)


# ----------------------------------------------------------------------------- A1 geometry

@pytest.mark.parametrize("nside", [1, 2, 4, 8, 32, 256, 4096])
def test_geometry_counts_and_offsets(nside):
    """Npix = 12 nside^2, 4 nside - 1 rings, 4 nside pixels on belt rings, 4 at the poles;
    offsets chain (RING: rings north to south)."""
    tot = 0
    for ring in range(1, 4 * nside):
        n, start, c, s, phi0 = oracle.ring_geometry(nside, ring)
        assert start == tot
        tot += n
        if nside <= ring <= 3 * nside:
            assert n == 4 * nside
        assert abs(c * c + s * s - 1.0) < 4e-16
    assert tot == 12 * nside * nside
    assert oracle.ring_geometry(nside, 1)[0] == 4 and oracle.ring_geometry(nside, 4 * nside - 1)[0] == 4
    with pytest.raises(ValueError):
        oracle.ring_geometry(nside, 0)
    with pytest.raises(ValueError):
        oracle.ring_geometry(nside, 4 * nside)
    with pytest.raises(ValueError):
        oracle.ring_geometry(3, 1)


def test_geometry_nside1_base_pixels():
    """nside = 1: the 12 base-pixel centres, z in {2/3, 0, -2/3}; phi = pi/4 + k pi/2 on z = +-2/3 and
    k pi/2 on z = 0 (Gorski et al., ref [1] P:416; SURVEY 8(c) A1 pin)."""
    th, ph = pix_angles(1)
    z = np.cos(th)
    np.testing.assert_allclose(z, [2 / 3] * 4 + [0.0] * 4 + [-2 / 3] * 4, atol=1e-15)
    k = np.arange(4)
    np.testing.assert_allclose(ph[:4], np.pi / 4 + k * np.pi / 2, atol=1e-15)
    np.testing.assert_allclose(ph[4:8], k * np.pi / 2, atol=1e-15)
    np.testing.assert_allclose(ph[8:], np.pi / 4 + k * np.pi / 2, atol=1e-15)


@pytest.mark.parametrize("nside", [2, 8, 64])
def test_geometry_equal_area_and_symmetry(nside):
    """Equal-area cells: the ring's latitude bisects the area of its own pixels, i.e.
    2 pi (1 - z_i) = (pixels in rings before i + N_i / 2) * 4 pi / Npix.  Point set invariant under
    z -> -z, phi -> phi + pi/2, phi -> -phi; belt rings alternate a half-pixel shift and the belt rule
    agrees with the cap rule at i = nside."""
    npix = 12 * nside * nside
    for ring in range(1, 4 * nside):
        n, start, c, s, phi0 = oracle.ring_geometry(nside, ring)
        assert abs((1.0 - c) - (2 * start + n) / npix * 1.0) < 1e-15 * 4
        n2, start2, c2, s2, phi02 = oracle.ring_geometry(nside, 4 * nside - ring)
        assert n2 == n and abs(c2 + c) < 1e-16 and abs(s2 - s) < 1e-16 and phi02 == phi0
        # phi -> -phi maps the ring onto itself iff 2 phi0 is a multiple of the spacing
        r = (2 * phi0) / (2 * math.pi / n)
        assert abs(r - round(r)) < 1e-12
        assert n % 4 == 0  # phi -> phi + pi/2
        assert 0.0 <= phi0 < 2 * math.pi / n  # RING: first pixel at the smallest non-negative longitude
    shifts = [oracle.ring_geometry(nside, r)[4] > 0 for r in range(nside, 3 * nside + 1)]
    assert shifts[0] and all(a != b for a, b in zip(shifts, shifts[1:]))
    assert all(oracle.ring_geometry(nside, r)[4] > 0 for r in range(1, nside))
    assert abs(oracle.ring_geometry(nside, nside)[2] - 2 / 3) < 1e-16


# ----------------------------------------------------------------------------- A2 lambda_lm

def test_lambda_closed_forms():
    """Low-degree closed forms with the Condon-Shortley phase of Eq. 15."""
    for th in [0.0, 1e-3, 0.3, 1.0, math.pi / 2, 2.2, math.pi - 1e-3]:
        c, s = math.cos(th), math.sin(th)
        pi = math.pi
        ref = {
            (0, 0): 1 / math.sqrt(4 * pi),
            (1, 0): math.sqrt(3 / (4 * pi)) * c,
            (1, 1): -math.sqrt(3 / (8 * pi)) * s,
            (2, 0): math.sqrt(5 / (16 * pi)) * (3 * c * c - 1),
            (2, 1): -math.sqrt(15 / (8 * pi)) * s * c,
            (2, 2): 0.25 * math.sqrt(15 / (2 * pi)) * s * s,
            (3, 3): -0.125 * math.sqrt(35 / pi) * s ** 3,
            (3, 1): -0.125 * math.sqrt(21 / pi) * s * (5 * c * c - 1),
        }
        for (l, m), v in ref.items():
            got = oracle.lambda_lm(3, m, th)[l]
            assert abs(got - v) < 3e-16, (l, m, th, got, v)


@pytest.mark.parametrize("lmax", [40, 500])
def test_lambda_vs_scipy(lmax):
    """lambda_lm(theta) = Y_lm(theta, 0) against scipy.special.sph_harm_y (SURVEY 8(c) A2 pin)."""
    rng = np.random.default_rng(5)
    thetas = np.concatenate([rng.uniform(0.05, math.pi - 0.05, 4), [0.01, math.pi / 2]])
    ms = sorted(set([0, 1, 2, 3, lmax // 3, lmax // 2, lmax - 1, lmax]))
    ls = np.arange(lmax + 1)
    for th in thetas:
        for m in ms:
            got = oracle.lambda_lm(lmax, m, th)
            ref = np.where(ls >= m, sph_harm_y(ls, np.minimum(m, ls), th, 0.0).real, 0.0)
            ok = np.isfinite(ref)
            # scipy evaluates from cos(theta) rounded to double: its own error is ~ eps * l / sin(theta)
            # (conditioning of P_l^m in x); the mpmath test below covers the polar regime tightly.
            tol = 5e-13 + 4e-16 * lmax / math.sin(th)
            assert np.abs(got - ref)[ok].max() < tol, (th, m)
            assert np.all(got[:m] == 0.0)


def _mp_lambda_legenp(l, m, z, dps):
    """mpmath's own Ferrers function (hypergeometric series) times the normalisation of Eq. 8."""
    import mpmath as mp

    mp.mp.dps = dps
    p = mp.legenp(l, m, z, type=2)  # includes the Condon-Shortley (-1)^m
    return mp.sqrt((2 * l + 1) / (4 * mp.pi) * mp.gammaprod([l - m + 1], [l + m + 1])) * p


def _mp_lambda_textbook(l, m, z, dps=60):
    """Independent route: the textbook UNNORMALISED recurrence (k-m) P_k^m = (2k-1) x P_(k-1)^m - (k+m-1) P_(k-2)^m
    from P_m^m = (-1)^m (2m-1)!! (1-x^2)^(m/2), in 60-digit mpmath floats (no range or conditioning issue),
    normalised at the end with Gamma functions."""
    import mpmath as mp

    mp.mp.dps = dps
    z = mp.mpf(z)
    pmm = (-1) ** m * mp.fac2(2 * m - 1) * (1 - z * z) ** (mp.mpf(m) / 2) if m > 0 else mp.mpf(1)
    p2, p1 = mp.mpf(0), pmm
    for k in range(m + 1, l + 1):
        p2, p1 = p1, ((2 * k - 1) * z * p1 - (k + m - 1) * p2) / (k - m)
    return mp.sqrt((2 * l + 1) / (4 * mp.pi) * mp.gammaprod([l - m + 1], [l + m + 1])) * p1


def _mp_ring_z(nside, ring):
    import mpmath as mp

    mp.mp.dps = 60
    ns = mp.mpf(nside)
    ip = min(ring, 4 * nside - ring)
    z = 1 - mp.mpf(ip) ** 2 / (3 * ns * ns) if ip < nside else (4 * ns - 2 * ip) / (3 * ns)
    return -z if ring > 2 * nside else z


def test_mp_textbook_recurrence_matches_mpmath_legenp():
    """Ties the arbitrary-precision reference used below to mpmath's library routine."""
    import mpmath as mp

    for (l, m, nside, ring) in [(300, 120, 256, 100), (511, 0, 256, 1), (200, 200, 64, 128), (97, 31, 64, 200)]:
        z = _mp_ring_z(nside, ring)
        a = _mp_lambda_legenp(l, m, z, 150)
        b = _mp_lambda_textbook(l, m, z)
        assert abs(a - b) <= abs(a) * mp.mpf(10) ** -40


@pytest.mark.parametrize("l,m,nside,ring", [
    (8191, 0, 4096, 1), (8191, 8191, 4096, 8192), (8191, 8190, 4096, 8000), (8000, 4000, 4096, 5000),
    (2047, 1500, 1024, 1500), (2047, 7, 1024, 3), (6000, 300, 4096, 200), (511, 200, 256, 100),
    (8191, 40, 4096, 20), (8191, 3, 4096, 16380), (4000, 4000, 4096, 4096), (8191, 1, 4096, 2),
])
def test_lambda_vs_mpmath_high_degree(l, m, nside, ring):
    """Spot values up to l = 8191 incl. polar rings and both hemispheres, against a 60-digit mpmath
    evaluation.  Exercises the exponent-scaled seeds ((8191, 8191) at the equator) and columns that start
    far below the double range near the pole."""
    z = _mp_ring_z(nside, ring)
    ref = float(_mp_lambda_textbook(l, m, z))
    got = oracle.lambda_lm_ring(nside, ring, l, m)[l]
    # The forward recurrence of Eq. 16 loses ~eps/(1-|cos theta|) near the poles in ANY working precision
    # (the restoring term of the difference equation is a cancellation of O(1) coefficients).  With the oracle's
    # 64-bit mantissa (eps = 5.4e-20) and the y-form of DESIGN.md R3 the measured errors are 6.5e-13 at ring 1 of
    # nside 4096 (y = 2e-8), 2.5e-13 at ring 2, 3.1e-13 four rings from the south pole (y = 3.2e-7) and < 1e-15 from
    # ring ~20 on.  The pin is 2e-19 / y capped at 2e-12: 2-3 x those figures and 5 x below the 1e-11 parity bar at
    # every ring (the round-1 pin, 3e-19 / y uncapped, admitted 1.5e-11 at ring 1).
    y = float(1 - abs(z))
    tol = min(2e-14 + 2e-19 / y, 2e-12)
    assert abs(got - ref) <= tol * max(abs(ref), 1e-300) + 1e-300, (got, ref, tol)


def test_reading_R3_cos_theta_rounded_to_double_is_not_enough_at_the_pole():
    """DESIGN.md R3 in numbers, independent of the oracle's code: run the three-term recurrence of Eq. 16 in
    60-digit arithmetic at ring 1 of nside 4096 once with the exact rational x = cos(theta) = 1 - 1/(3 nside^2) and once
    with x rounded to double.  The only difference is the rounding of x (1.1e-16 relative), yet lambda_l0 at l ~ 8000
    moves by ~1e-10 relative to the column's maximum -- above the 1e-11 parity bar -- because near the pole
    d(lambda)/dx ~ l^2 lambda / 2.  Forming x p as p - y p with y = 1 - x taken exactly from the ring integers (what
    the oracle and the kernels do) removes it: y rounded to double moves the result by < 1e-15."""
    import mpmath as mp

    mp.mp.dps = 60
    nside, lmax, m = 4096, 8191, 0
    y_exact = mp.mpf(1) / (3 * mp.mpf(nside) ** 2)

    def column_last(xp):  # lambda_{l,0}, l = 0..lmax, by Eq. 16 with x p supplied by `xp`
        p0 = 1 / mp.sqrt(4 * mp.pi)
        p1 = mp.sqrt(3) * xp(p0)
        big = max(abs(p0), abs(p1))
        for l in range(2, lmax + 1):
            a = mp.sqrt(mp.mpf(4 * l * l - 1) / (l * l - m * m))
            b = -mp.sqrt(mp.mpf(2 * l + 1) / (2 * l - 3) * ((l - 1) ** 2 - m * m) / (l * l - m * m))
            p0, p1 = p1, a * xp(p1) + b * p0
            big = max(big, abs(p1))
        return p1, big

    exact, big = column_last(lambda p: p - y_exact * p)
    x_double = mp.mpf(float(1 - y_exact))
    rounded_x, _ = column_last(lambda p: x_double * p)
    y_double = mp.mpf(float(y_exact))
    rounded_y, _ = column_last(lambda p: p - y_double * p)
    err_x = float(abs(rounded_x - exact) / big)
    err_y = float(abs(rounded_y - exact) / big)
    assert err_x > 2e-11, err_x   # x rounded to double alone already breaks the 1e-11 bar
    assert err_y < 1e-14, err_y   # the y-form does not
    # and the oracle (64-bit mantissa, y-form) sits with the exact column
    got = oracle.lambda_lm_ring(nside, 1, lmax, m)[lmax]
    assert abs(got - float(exact)) <= 2e-12 * float(big)


@pytest.mark.parametrize("lmax", [64, 700])
def test_lambda_addition_theorem_sign_parity(lmax):
    """sum_m |Y_lm|^2 = (2l+1)/4pi at any theta pins the normalisation of every (l,m) (Eq. 9);
    lambda_lm(pi - theta) = (-1)^(l+m) lambda_lm(theta); sign -> (-1)^m as theta -> 0+ (Eq. 15)."""
    ls = np.arange(lmax + 1)
    for th in [0.02, 0.4, 1.3, math.pi / 2]:
        tot = np.zeros(lmax + 1)
        for m in range(lmax + 1):
            lam = oracle.lambda_lm(lmax, m, th)
            lam_s = oracle.lambda_lm(lmax, m, math.pi - th)
            tot += (1 if m == 0 else 2) * lam ** 2
            sign = np.where((ls + m) % 2 == 0, 1.0, -1.0)
            np.testing.assert_allclose(lam_s, sign * lam, rtol=0, atol=1e-13 * max(1.0, np.abs(lam).max()))
        np.testing.assert_allclose(tot, (2 * ls + 1) / (4 * math.pi), rtol=2e-13)
    for m in range(0, 9):
        lam = oracle.lambda_lm(12, m, 1e-4)
        assert np.all(np.sign(lam[m:]) == (-1) ** m)


def test_lambda_orthonormal_gauss_legendre():
    """2 pi int lambda_lm lambda_l'm sin(theta) dtheta = delta_ll' (Eq. 9) by Gauss-Legendre
    quadrature, exact for lmax + lmax < 2 n."""
    lmax = 200
    x, w = np.polynomial.legendre.leggauss(lmax + 2)
    for m in [0, 1, 17, 100, 199, 200]:
        L = np.array([oracle.lambda_lm(lmax, m, math.acos(xi)) for xi in x])[:, m:]
        G = 2 * math.pi * (L * w[:, None]).T @ L
        np.testing.assert_allclose(G, np.eye(lmax + 1 - m), atol=5e-13)


# ----------------------------------------------------------------------------- A3 ring DFT

@pytest.mark.parametrize("nside,ring", [(4, 1), (4, 3), (4, 4), (4, 5), (8, 9), (8, 31), (16, 11)])
def test_ring_dft_vs_direct_sum(nside, ring):
    """F_m = sum_x p_x exp(-i m (phi0 + 2 pi x / N)) against a direct numpy cos/sin sum (Eq. 13 P:177,
    Eq. 26), including m far beyond N/2 (aliasing on polar rings)."""
    n, start, c, s, phi0 = oracle.ring_geometry(nside, ring)
    p = synth.normal(7, ring, n)
    mmax = 3 * nside + 5
    got = oracle.ring_dft(nside, ring, p, mmax)
    x = np.arange(n)
    ref = np.array([(p * np.exp(-1j * m * (phi0 + 2 * np.pi * x / n))).sum() for m in range(mmax + 1)])
    np.testing.assert_allclose(got, ref, atol=1e-13 * n)


@pytest.mark.parametrize("nside,ring", [(4, 1), (4, 2), (4, 6), (8, 13), (16, 40)])
def test_ring_synth_vs_direct_sum(nside, ring):
    """The ring synthesis sum of Eq. 24 against numpy, with m far beyond N/2."""
    n, start, c, s, phi0 = oracle.ring_geometry(nside, ring)
    mmax = 3 * nside + 3
    G = synth.white_alm(5, mmax, 0)[0][: mmax + 1].copy()
    x = np.arange(n)
    ref = G[0].real + 2 * sum((G[m] * np.exp(1j * m * (phi0 + 2 * np.pi * x / n))).real for m in range(1, mmax + 1))
    np.testing.assert_allclose(oracle.ring_synth(nside, ring, G), ref, atol=1e-13 * mmax)


def test_bluestein_identity():
    """Eq. 17-23: X(k) = h[k] sum_n (x[n] h[n]) h^-1[k-n], h[m] = W_N^(m^2/2), reproduces
    the ring DFT for a non-power-of-two ring (the identity the CUDA chirp-z kernels rely on)."""
    nside, ring = 8, 5  # N = 20
    n, start, c, s, phi0 = oracle.ring_geometry(nside, ring)
    p = synth.normal(11, 3, n)
    k = np.arange(n)
    h = np.exp(-1j * np.pi * ((k * k) % (2 * n)) / n)
    y = p * h
    w = np.array([sum(y[t] * np.conj(h[abs(kk - t)]) for t in range(n)) for kk in range(n)])
    X = w * h
    F = oracle.ring_dft(nside, ring, p, n - 1) * np.exp(1j * np.arange(n) * phi0)
    np.testing.assert_allclose(X, F, atol=1e-13 * n)


# ----------------------------------------------------------------------------- A4 operators

def dense_S(nside, lmax, mmax):
    """Npix x 2 Nalm real matrix of S built from scipy's Y_lm at the pixel centres."""
    th, ph = pix_angles(nside)
    ls, ms = synth.alm_lm(lmax, mmax)
    Y = sph_harm_y(ls[None, :], ms[None, :], th[:, None], ph[:, None])
    cm = np.where(ms == 0, 1.0, 2.0)
    Sre = cm * Y.real
    Sim = -cm * Y.imag
    Sim[:, ms == 0] = 0.0
    return np.hstack([Sre, Sim]), cm


@pytest.mark.parametrize("nside,lmax,mmax", [(1, 4, 4), (2, 8, 8), (2, 5, 3), (4, 16, 16), (4, 11, 7)])
def test_operators_vs_dense_matrices(nside, lmax, mmax):
    """S, S^T, A = D^-1 S^T W and A^T = W S D^-1 as explicit matrix products (SURVEY 8(c) A4 pin),
    lmax up to 4 nside so polar rings alias heavily; non-uniform, non-symmetric ring weights."""
    S, cm = dense_S(nside, lmax, mmax)
    na = synth.alm_count(lmax, mmax)
    npix = 12 * nside * nside
    a = synth.white_alm(3, lmax, mmax)[0]
    g = synth.normal(4, 9, npix)
    w_ring = synth.ring_weights(5, nside)
    w_pix = np.concatenate([[w_ring[r - 1]] * oracle.ring_geometry(nside, r)[0] for r in range(1, 4 * nside)])
    ms = synth.alm_lm(lmax, mmax)[1]
    v = np.concatenate([a.real, a.imag])
    tol = 2e-13 * np.abs(S).max() * math.sqrt(na)

    np.testing.assert_allclose(oracle.alm2map(nside, lmax, mmax, a), S @ v, atol=tol * np.abs(v).max())
    st = S.T @ g
    got = oracle.alm2map_adjoint(nside, lmax, mmax, g)
    np.testing.assert_allclose(np.concatenate([got.real, got.imag]), st, atol=tol * np.abs(g).max() * 10)
    assert np.all(got.imag[ms == 0] == 0.0)

    aa = (S.T @ (w_pix * g)) / np.concatenate([cm, cm])
    got = oracle.map2alm(nside, lmax, mmax, g, w_ring)
    np.testing.assert_allclose(np.concatenate([got.real, got.imag]), aa, atol=tol * np.abs(g).max())
    at = w_pix * (S @ (v / np.concatenate([cm, cm])))
    np.testing.assert_allclose(oracle.map2alm_adjoint(nside, lmax, mmax, a, w_ring), at, atol=tol)
    # default weights are 4 pi / Npix (Eq. 1)
    got = oracle.map2alm(nside, lmax, mmax, g)
    aa = (S.T @ g) * (4 * np.pi / npix) / np.concatenate([cm, cm])
    np.testing.assert_allclose(np.concatenate([got.real, got.imag]), aa, atol=tol)


@pytest.mark.parametrize("nside,lmax,n_iter", [(2, 4, 1), (2, 5, 3), (4, 8, 2)])
def test_iterative_refinement_equals_gradient_descent_form(nside, lmax, n_iter):
    """Eq. 4 against its 'equivalent gradient descent form' Eq. 5 written with the dense scipy
    matrix: a^(k+1) = (4 pi / N) S* f + (I - (4 pi / N) S* S) a^(k), S* = Y^dagger = D^-1 S^T on the stored m >= 0
    half (R4), a^(0) = (4 pi / N) S* f.  Pins the oracle's map2alm_iter (a dropped sign, A and S swapped
    or a residual formed the other way round all fail)."""
    S, cm = dense_S(nside, lmax, lmax)
    npix = 12 * nside * nside
    f = synth.normal(6, 2, npix)
    cc = np.concatenate([cm, cm])
    A = (4 * np.pi / npix) * (S.T / cc[:, None])
    v = A @ f
    for _ in range(n_iter):
        v = A @ f + (np.eye(A.shape[0]) - A @ S) @ v
    got = oracle.map2alm_iter(nside, lmax, lmax, f, n_iter)
    ms = synth.alm_lm(lmax, lmax)[1]
    ref = v[: len(ms)] + 1j * v[len(ms):]
    np.testing.assert_allclose(got, ref, atol=1e-12 * np.abs(ref).max())
    assert np.all(got.imag[ms == 0] == 0.0)


def test_iterative_refinement_converges_on_band_limited_input():
    """P:59 / P:400: 'accuracy improved by increasing the number of iterations' -- for f = S a with lmax <= 2 nside
    the error |a^(k) - a| falls with every iteration."""
    nside, lmax = 8, 12
    a = synth.powerlaw_alm(8, lmax, lmax)[0]
    f = oracle.alm2map(nside, lmax, lmax, a)
    errs = [np.abs(oracle.map2alm_iter(nside, lmax, lmax, f, k) - a).max() for k in range(4)]
    assert all(e1 < 0.5 * e0 for e0, e1 in zip(errs, errs[1:])), errs


@pytest.mark.parametrize("nside,lmax", [(8, 16), (16, 40)])
def test_adjoint_dot_product_identities(nside, lmax):
    """<S a, g> = <a, S^T g> and <A f, b> = <f, A^T b> (north_star)."""
    mmax = lmax
    a = synth.white_alm(21, lmax, mmax)[0]
    a[: lmax + 1] = a[: lmax + 1].real  # m = 0 coefficients are real in both inner products
    b = synth.white_alm(22, lmax, mmax)[0]
    b[: lmax + 1] = b[: lmax + 1].real
    f = synth.gaussian_map(23, nside)[0]
    g = synth.gaussian_map(24, nside)[0]
    w = synth.ring_weights(25, nside)

    def adot(x, y):
        return float((x.real * y.real + x.imag * y.imag).sum())

    lhs = float(oracle.alm2map(nside, lmax, mmax, a) @ g)
    rhs = adot(a, oracle.alm2map_adjoint(nside, lmax, mmax, g))
    assert abs(lhs - rhs) < 1e-13 * max(abs(lhs), 1.0) * 10
    lhs = adot(oracle.map2alm(nside, lmax, mmax, f, w), b)
    rhs = float(f @ oracle.map2alm_adjoint(nside, lmax, mmax, b, w))
    assert abs(lhs - rhs) < 1e-13 * max(abs(lhs), 1.0) * 10


def test_single_coefficient_synthesis_closed_form():
    """a_lm = 1 -> 2 lambda_lm cos(m phi); a_lm = i -> -2 lambda_lm sin(m phi); a_l0 = 1 -> lambda_l0;
    a_00 -> constant 1/sqrt(4 pi)  (Eq. 24; SURVEY 8(c) A3 pin), including m > N_i/2 on polar rings."""
    nside, lmax = 4, 14
    th, ph = pix_angles(nside)
    na = synth.alm_count(lmax, lmax)
    for (l, m, val) in [(0, 0, 1.0), (5, 0, 1.0), (5, 0, 1j), (7, 3, 1.0), (7, 3, 1j), (14, 14, 1.0), (13, 9, 1j),
                        (12, 8, 1.0), (9, 4, 1.0)]:
        a = np.zeros(na, dtype=complex)
        a[oracle.alm_index(lmax, l, m)] = val
        got = oracle.alm2map(nside, lmax, lmax, a)
        Y = sph_harm_y(l, m, th, ph)
        if m == 0:
            ref = Y.real * np.real(val)
        else:
            ref = 2 * (val * Y).real
        np.testing.assert_allclose(got, ref, atol=3e-14)
    a = np.zeros(na, dtype=complex)
    a[0] = 1.0
    np.testing.assert_allclose(oracle.alm2map(nside, lmax, lmax, a), 1 / math.sqrt(4 * math.pi), atol=1e-16)


def test_constant_map_analysis():
    """Analysing f = 1 with equal weights: a_00 = sqrt(4 pi) exactly, a_l0 = 0 for odd l, a_lm = 0 unless
    4 | m (SURVEY 8(c) A3 pin: a pure test of the alias/DC handling: ring 1 aliases m = 4 onto DC)."""
    nside, lmax = 4, 16
    a = oracle.map2alm(nside, lmax, lmax, np.ones(12 * nside * nside))
    ls, ms = synth.alm_lm(lmax, lmax)
    assert abs(a[0] - math.sqrt(4 * math.pi)) < 2e-15
    assert np.abs(a[(ms == 0) & (ls % 2 == 1)]).max() < 1e-15
    assert np.abs(a[ms % 4 != 0]).max() < 1e-15
    assert np.abs(a[(ms == 4)]).max() > 1e-4  # aliased power really is there


def test_round_trip_error_shrinks():
    """Qualitative: synth + analysis of a fixed low-degree a_lm, equal weights, lmax = 2 nside: the error
    falls monotonically with nside."""
    a8 = synth.powerlaw_alm(31, 8, 8)[0]
    errs = []
    for nside in [8, 16, 32]:
        lmax = 2 * nside
        a = np.zeros(synth.alm_count(lmax, lmax), dtype=complex)
        for l in range(9):
            for m in range(l + 1):
                a[oracle.alm_index(lmax, l, m)] = a8[oracle.alm_index(8, l, m)]
        back = oracle.map2alm(nside, lmax, lmax, oracle.alm2map(nside, lmax, lmax, a))
        errs.append(np.abs(back - a).max())
    assert errs[0] > errs[1] > errs[2]
    assert errs[2] < errs[0] / 4


def test_subset_modes_match_full():
    """Subset entry points return the same numbers as the full transforms."""
    nside, lmax, mmax = 8, 20, 17
    f = synth.gaussian_map(41, nside)[0]
    w = synth.ring_weights(42, nside)
    a = synth.white_alm(43, lmax, mmax)[0]
    full = oracle.map2alm(nside, lmax, mmax, f, w)
    full_st = oracle.alm2map_adjoint(nside, lmax, mmax, f)
    sel = [(0, 0), (20, 0), (17, 17), (20, 17), (20, 16), (9, 5), (13, 5), (6, 6)]
    sl, sm = [s[0] for s in sel], [s[1] for s in sel]
    idx = [oracle.alm_index(lmax, l, m) for l, m in sel]
    np.testing.assert_allclose(oracle.map2alm_subset(nside, lmax, mmax, f, sl, sm, w), full[idx], rtol=0, atol=1e-17)
    np.testing.assert_allclose(oracle.alm2map_adjoint_subset(nside, lmax, mmax, f, sl, sm), full_st[idx], rtol=0,
                               atol=1e-15)
    rings = [1, 7, 8, 16, 31, 22, 5]
    fm = oracle.alm2map(nside, lmax, mmax, a)
    fat = oracle.map2alm_adjoint(nside, lmax, mmax, a, w)
    pieces, pieces_t = [], []
    for r in rings:
        n, start = oracle.ring_geometry(nside, r)[:2]
        pieces.append(fm[start:start + n])
        pieces_t.append(fat[start:start + n])
    np.testing.assert_array_equal(oracle.alm2map_rings(nside, lmax, mmax, a, rings), np.concatenate(pieces))
    np.testing.assert_array_equal(oracle.map2alm_adjoint_rings(nside, lmax, mmax, a, rings, w),
                                  np.concatenate(pieces_t))


def test_bad_arguments():
    with pytest.raises(ValueError):
        oracle.lambda_lm(3, 4, 0.1)
    with pytest.raises(ValueError):
        oracle.map2alm_subset(4, 8, 8, np.zeros(192), [9], [0])


# ----------------------------------------------------------------------------- input generators

def test_synth_is_counter_based_and_sane():
    a = synth.normal(1, 2, 1000)
    b = synth.normal(1, 2, 400, offset=600)
    np.testing.assert_array_equal(a[600:], b)
    x = synth.normal(9, 1, 200000)
    assert abs(x.mean()) < 0.01 and abs(x.std() - 1) < 0.01
    alm = synth.powerlaw_alm(3, 30, 30, batch=2)
    ls, ms = synth.alm_lm(30, 30)
    assert alm.shape == (2, synth.alm_count(30, 30)) and np.all(alm[:, ms == 0].imag == 0)
    for l in range(31):
        for m in range(l + 1):
            k = oracle.alm_index(30, l, m)
            assert ls[k] == l and ms[k] == m


_SAN_SCRIPT = """
import numpy as np
import oracle
from paper_2510_01785_b200 import synth
for nside, lmax, mmax in [(1, 3, 3), (4, 11, 7), (8, 16, 16), (16, 40, 40)]:
    f = synth.gaussian_map(9, nside, 1)[0]
    a = synth.powerlaw_alm(9, lmax, mmax, 1)[0]
    w = synth.ring_weights(9, nside)
    full_s = oracle.alm2map(nside, lmax, mmax, a)
    full_a = oracle.map2alm(nside, lmax, mmax, f, w)
    full_st = oracle.alm2map_adjoint(nside, lmax, mmax, f)
    full_at = oracle.map2alm_adjoint(nside, lmax, mmax, a, w)
    rings = sorted({1, 2 * nside, 4 * nside - 1, min(3, 4 * nside - 1)})
    ls = [mmax, lmax, lmax]
    ms = [mmax, 0, min(1, mmax)]
    idx = [oracle.alm_index(lmax, l, m) for l, m in zip(ls, ms)]
    sub = oracle.alm2map_rings(nside, lmax, mmax, a, rings)
    ref = np.concatenate([full_s[s:s + n] for n, s in (oracle.ring_geometry(nside, r)[:2] for r in rings)])
    assert np.array_equal(sub, ref)
    assert np.allclose(oracle.map2alm_subset(nside, lmax, mmax, f, ls, ms, w), full_a[idx], rtol=0, atol=1e-15)
    assert np.allclose(oracle.alm2map_adjoint_subset(nside, lmax, mmax, f, ls, ms), full_st[idx], rtol=0, atol=1e-15)
    sub = oracle.map2alm_adjoint_rings(nside, lmax, mmax, a, rings, w)
    ref = np.concatenate([full_at[s:s + n] for n, s in (oracle.ring_geometry(nside, r)[:2] for r in rings)])
    assert np.array_equal(sub, ref)
    oracle.map2alm_iter(nside, lmax, mmax, f, 1, w)
    oracle.lambda_lm(lmax, mmax, 0.3)
    oracle.lambda_lm_ring(nside, 1, lmax, mmax)
    oracle.ring_dft(nside, 1, f[:4], lmax)
    oracle.ring_synth(nside, 1, a[: lmax + 1])
print("sanitized oracle ok")
"""


def test_oracle_under_asan_ubsan(tmp_path):
    """the oracle's C code (full operators and the subset entry points the cfg4 / cfg5 parity tests
    rely on) built with -fsanitize=address,undefined and run once; any out-of-bounds access, signed overflow, bad
    shift or misaligned access aborts the subprocess."""
    import subprocess
    import sys

    lib = oracle.build(sanitize=True)
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("libasan.so not found next to gcc")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, SHT_ORACLE_LIB=lib, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", PYTHONPATH=root, OMP_NUM_THREADS="2")
    res = subprocess.run([sys.executable, "-c", _SAN_SCRIPT], env=env, capture_output=True, text=True, timeout=600)
    assert res.returncode == 0, res.stderr[-3000:]
    assert "sanitized oracle ok" in res.stdout
    assert "runtime error" not in res.stderr and "AddressSanitizer" not in res.stderr, res.stderr[-3000:]
