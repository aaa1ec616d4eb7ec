"""CPU oracle of the transforms on iso-latitude grids (TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline leg may import this; it shares no code with paper_2510_01785_b200/).

Same operators as oracle/sht_oracle.c (Eq. 24, Eq. 26, adjoints P:287-288 in the reading DESIGN.md R4), on
the grids of P:376-386: nlat rings (north to south) of nlon pixels at phi = 2 pi x / nlon.
  "gl": cos(theta_k) = roots of P_nlat (numpy.polynomial.legendre.leggauss), weights w_k 2 pi / nlon
  "eq": theta_k = pi (k + 1/2) / nlat, Fejer's first rule  w_k = (2 / nlat) (1 - 2 sum_{j=1}^{nlat/2} cos(2 j theta_k) / (4 j^2 - 1))
Plain dense sums in double (numpy); lambda_lm(theta) is the oracle's own recurrence (pinned in tests/test_oracle_pins.py).
"""
from __future__ import annotations

import numpy as np

import oracle


def grid_nodes(kind: str, nlat: int, nlon: int):
    """(theta_k, per-pixel quadrature weight) of every ring."""
    if kind == "gl":
        x, w = np.polynomial.legendre.leggauss(nlat)
        theta = np.arccos(x[::-1])
        w = w[::-1]
    elif kind == "eq":
        theta = np.pi * (np.arange(nlat) + 0.5) / nlat
        j = np.arange(1, nlat // 2 + 1)
        w = np.array([(2.0 / nlat) * (1.0 - 2.0 * np.sum(np.cos(2 * j * t) / (4.0 * j * j - 1.0))) for t in theta])
    else:
        raise ValueError(kind)
    return theta, w * 2.0 * np.pi / nlon


def _ylm_matrix(kind, nlat, nlon, lmax, mmax):
    """Complex matrix Y[p, idx(l, m)] = lambda_lm(theta_p) exp(i m phi_p), m >= 0, packed like alm."""
    theta, _w = grid_nodes(kind, nlat, nlon)
    nalm = oracle.alm_count(lmax, mmax)
    Y = np.zeros((nlat * nlon, nalm), dtype=np.complex128)
    phi = 2.0 * np.pi * np.arange(nlon) / nlon
    for m in range(mmax + 1):
        e = np.exp(1j * m * phi)
        for k in range(nlat):
            lam = oracle.lambda_lm(lmax, m, float(theta[k]))
            for l in range(m, lmax + 1):
                Y[k * nlon:(k + 1) * nlon, oracle.alm_index(lmax, l, m)] = lam[l] * e
    return Y


def _cm(lmax, mmax):
    c = np.empty(oracle.alm_count(lmax, mmax))
    for m in range(mmax + 1):
        for l in range(m, lmax + 1):
            c[oracle.alm_index(lmax, l, m)] = 1.0 if m == 0 else 2.0
    return c


def _zero_imag_m0(a, lmax):
    a = np.array(a, dtype=np.complex128)
    for l in range(lmax + 1):
        a[oracle.alm_index(lmax, l, 0)] = a[oracle.alm_index(lmax, l, 0)].real
    return a


def alm2map(kind, nlat, nlon, lmax, mmax, alm):
    """f_p = sum_l Re(a_l0) lambda_l0 + 2 sum_{m>=1} sum_l Re(a_lm lambda_lm e^{i m phi_p})   (Eq. 24)"""
    Y = _ylm_matrix(kind, nlat, nlon, lmax, mmax)
    a = _zero_imag_m0(alm, lmax)
    return np.real(Y @ (a * _cm(lmax, mmax)))


def map2alm(kind, nlat, nlon, lmax, mmax, fmap, ring_weights=None):
    """a_lm = sum_p w_p f_p lambda_lm e^{-i m phi_p}   (Eq. 26)"""
    Y = _ylm_matrix(kind, nlat, nlon, lmax, mmax)
    _t, w = grid_nodes(kind, nlat, nlon)
    if ring_weights is not None:
        w = np.asarray(ring_weights, dtype=np.float64)
    a = np.conj(Y).T @ (np.repeat(w, nlon) * np.asarray(fmap, dtype=np.float64))
    return _zero_imag_m0(a, lmax)


def alm2map_adjoint(kind, nlat, nlon, lmax, mmax, gmap):
    """(S^T g)_lm = c_m sum_p g_p lambda_lm e^{-i m phi_p}   (reading R4)"""
    Y = _ylm_matrix(kind, nlat, nlon, lmax, mmax)
    return _zero_imag_m0(_cm(lmax, mmax) * (np.conj(Y).T @ np.asarray(gmap, dtype=np.float64)), lmax)


def map2alm_adjoint(kind, nlat, nlon, lmax, mmax, galm, ring_weights=None):
    """(A^T b)_p = w_p [sum_l Re(b_l0) lambda_l0 + sum_{m>=1} sum_l Re(b_lm lambda_lm e^{i m phi_p})]   (reading R4)"""
    Y = _ylm_matrix(kind, nlat, nlon, lmax, mmax)
    _t, w = grid_nodes(kind, nlat, nlon)
    if ring_weights is not None:
        w = np.asarray(ring_weights, dtype=np.float64)
    b = _zero_imag_m0(galm, lmax)
    return np.repeat(w, nlon) * np.real(Y @ b)
