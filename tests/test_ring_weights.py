"""Ring quadrature weights: oracle pins (CPU) and GPU parity.

The oracle (oracle/ring_weights.py) is the minimum-norm solution written out with a dense library solve; it is pinned
here against facts it does not use: exact integration of Legendre polynomials evaluated by numpy's own Legendre series,
the closed-form total area, symmetry, a KKT check of the minimum-norm property, exact recovery of zonal coefficients
through the (separately pinned) oracle transforms, and the paper's qualitative statement that ring weights beat equal
weights.
"""
import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

import oracle
from oracle import ring_weights as orw
from paper_2510_01785_b200 import synth


def _table(nside):
    z, n = orw.ring_table(nside)
    return z.astype(np.float64), n.astype(np.float64)


@pytest.mark.parametrize("nside", [1, 2, 4, 8, 16])
def test_oracle_weights_integrate_legendre_polynomials_exactly(nside):
    w = orw.ring_weights(nside)
    z, n = _table(nside)
    # sum over pixels of P_l(z) w = 2 pi int_-1^1 P_l dz = 4 pi delta_l0, for every l <= 3 nside (numpy's Legendre series)
    for l in range(0, 3 * nside + 1):
        c = np.zeros(l + 1)
        c[l] = 1.0
        got = float(np.sum(w * n * npleg.legval(z, c)))
        want = 4.0 * np.pi if l == 0 else 0.0
        assert abs(got - want) < 5e-13, (l, got)
    assert abs(float(np.sum(w * n)) - 4.0 * np.pi) < 1e-13          # total area
    assert np.abs(w - w[::-1]).max() < 1e-17 + 1e-14 * w.max()       # north / south symmetry
    assert (w > 0).all()


@pytest.mark.parametrize("nside", [2, 4, 8])
def test_oracle_weights_are_the_minimum_norm_solution(nside):
    """KKT: N (w - w0) must lie in the span of the constraint gradients N lambda_l0, i.e. w - w0 is a zonal polynomial of
    degree <= lmax_w sampled on the rings; and any feasible perturbation increases the objective."""
    w = orw.ring_weights(nside)
    z, n = _table(nside)
    w0 = 4.0 * np.pi / (12 * nside * nside)
    V = np.stack([npleg.legval(z, np.eye(3 * nside + 1)[l]) for l in range(3 * nside + 1)], axis=1)  # rings x degrees
    coef, *_ = np.linalg.lstsq(V, w - w0, rcond=None)
    assert np.abs(V @ coef - (w - w0)).max() < 1e-13 * w0 * 100
    # a feasible direction: null space of the constraints
    A = (V * n[:, None]).T
    _u, s, vt = np.linalg.svd(A)
    null = vt[(s > 1e-10 * s[0]).sum():]
    if len(null):
        d = null[0] * 1e-3 * w0
        f = lambda x: float(np.sum(n * (x - w0) ** 2))
        assert f(w + d) > f(w) and f(w - d) > f(w)


@pytest.mark.parametrize("nside", [4, 8])
def test_oracle_weights_recover_zonal_coefficients(nside):
    """alm2map then map2alm with the ring weights returns a_l0 of a zonal map band-limited to 1.5 nside to rounding,
    while equal weights do not (ring weights are the more accurate scheme)."""
    lmax = 3 * nside // 2
    alm = np.zeros(oracle.alm_count(lmax, lmax), dtype=np.complex128)
    rng = synth.powerlaw_alm(77 + nside, lmax, lmax, 1)[0]
    for l in range(lmax + 1):
        alm[oracle.alm_index(lmax, l, 0)] = rng[oracle.alm_index(lmax, l, 0)].real
    m = oracle.alm2map(nside, lmax, lmax, alm)
    back_w = oracle.map2alm(nside, lmax, lmax, m, ring_weights=orw.ring_weights(nside))
    back_e = oracle.map2alm(nside, lmax, lmax, m)
    scale = np.abs(alm).max()
    zonal = [oracle.alm_index(lmax, l, 0) for l in range(lmax + 1)]  # orders m = 4 k pick up ring aliasing, not quadrature error
    err_w = np.abs(back_w[zonal] - alm[zonal]).max() / scale
    err_e = np.abs(back_e[zonal] - alm[zonal]).max() / scale
    assert err_w < 1e-12, err_w
    assert err_e > 1e-6 and err_e > 1e3 * err_w


def test_ring_weights_improve_the_round_trip_of_a_general_map():
    """Round trip of a band-limited map with all orders m (lmax = 1.5 nside): smaller error with ring weights."""
    nside, lmax = 8, 12
    alm = synth.powerlaw_alm(5, lmax, lmax, 1)[0]
    m = oracle.alm2map(nside, lmax, lmax, alm)
    err_w = np.abs(oracle.map2alm(nside, lmax, lmax, m, ring_weights=orw.ring_weights(nside)) - alm).max()
    err_e = np.abs(oracle.map2alm(nside, lmax, lmax, m) - alm).max()
    assert err_w < err_e


@pytest.mark.gpu
@pytest.mark.parametrize("nside,lmax_w", [(1, 0), (2, 0), (8, 0), (32, 0), (32, 64), (128, 0)])
def test_gpu_ring_weights_match_oracle(nside, lmax_w):
    import torch

    from paper_2510_01785_b200 import binding as B

    got = B.ring_weights(nside, lmax_w).cpu().numpy()
    ref = orw.ring_weights(nside, lmax_w)
    assert got.shape == ref.shape
    assert np.abs(got - ref).max() / np.abs(ref).max() <= 1e-11
    assert np.abs(got - got[::-1]).max() <= 1e-14 * got.max()


@pytest.mark.gpu
def test_gpu_ring_weights_large_nside_properties():
    """nside 1024 (beyond the dense oracle): the properties that hold at any size, with numpy's Legendre recurrence on a
    sample of degrees, and use as d_ring_weights of map2alm."""
    import torch

    from paper_2510_01785_b200 import binding as B

    nside = 1024
    w = B.ring_weights(nside).cpu().numpy()
    z = np.empty(4 * nside - 1)
    n = np.empty(4 * nside - 1)
    for i in range(1, 4 * nside):
        npx, _f, ct, _p = B.cuhpx_ring_info(nside, i)
        z[i - 1], n[i - 1] = ct, npx
    assert abs(np.sum(w * n) - 4 * np.pi) < 1e-12
    assert np.abs(w - w[::-1]).max() <= 1e-14 * w.max()
    # three-term recurrence in plain numpy for P_l(z), all l up to 3 nside; check a sample of degrees
    pm, p = np.ones_like(z), z.copy()
    check = {1, 2, 3, 10, 511, 1024, 2047, 2048, 3071, 3072}
    for l in range(1, 3 * nside + 1):
        if l in check:
            assert abs(np.sum(w * n * p)) < 2e-11, l
        pm, p = p, ((2 * l + 1) * z * p - l * pm) / (l + 1)


@pytest.mark.gpu
def test_gpu_map2alm_with_ring_weights():
    """The weights plug into cuhpx_map2alm as d_ring_weights: parity with the oracle using the same weights, and the
    paper's ordering on the GPU: smaller round-trip error than equal weights for a band-limited map."""
    import torch

    from paper_2510_01785_b200 import binding as B

    nside, lmax = 32, 48
    T = B.Transform(nside, lmax, lmax, 1, torch.float64)
    w = B.ring_weights(nside)
    alm = synth.powerlaw_alm(9, lmax, lmax, 1)
    z0 = [oracle.alm_index(lmax, l, 0) for l in range(lmax + 1)]
    alm[0, z0] = alm[0, z0].real
    d_map = T.alm2map(torch.from_numpy(alm).cuda())
    got_w = torch.empty(1, T.nalm, dtype=torch.complex128, device="cuda")
    B.cuhpx_map2alm(*T.params, d_map, got_w, w, T.workspace)
    got_e = T.map2alm(d_map)
    ref_w = oracle.map2alm(nside, lmax, lmax, d_map.cpu().numpy()[0], ring_weights=w.cpu().numpy())
    assert np.abs(got_w.cpu().numpy()[0] - ref_w).max() / np.abs(ref_w).max() <= 1e-11
    err_w = np.abs(got_w.cpu().numpy()[0] - alm[0]).max()
    err_e = np.abs(got_e.cpu().numpy()[0] - alm[0]).max()
    assert err_w < err_e
