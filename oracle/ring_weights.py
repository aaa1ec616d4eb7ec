"""CPU oracle of the ring quadrature weights (TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg may import this; it shares no code with paper_2510_01785_b200/).

Definition (reading R11; P:340-346 names "ring weights" as cuHPX's default but takes the values from the HEALPix
data files, which are not available here): the per-ring weights w_i, i = 1 .. 4 nside - 1, closest to the equal weights
w0 = 4 pi / Npix (Eq. 1) in the pixel-weighted norm  sum_i N_i (w_i - w0)^2  among all weights for which the m = 0
quadrature of Eq. 26 is exact,
        sum_i w_i N_i lambda_l0(theta_i) = sqrt(4 pi) delta_l0          for l = 0 .. lmax_w   (default 3 nside).
Written out as the textbook minimum-norm solution of a linear system, dense, in long double:
        M[l][i] = sqrt(N_i) lambda_l0(theta_i),   r = sqrt(4 pi) e_0 - M sqrt(N) w0,
        w = w0 + N^-1/2 M^T (M M^T)^+ r
Whether these weights equal the values HEALPix tabulates is PARITY UNPINNED (the files are not available; R11);
everything the definition above states is pinned in tests/test_ring_weights.py.
lambda_l0 comes from the oracle's own recurrence (oracle/sht_oracle.c, pinned in tests/test_oracle_pins.py); the solve is
numpy's (a library primitive serving as a step).
"""
from __future__ import annotations

import numpy as np

import oracle


def ring_table(nside: int):
    """(cos theta_i, N_i) of every ring, north to south, from the oracle's geometry."""
    nr = 4 * nside - 1
    z = np.empty(nr, dtype=np.longdouble)
    n = np.empty(nr, dtype=np.longdouble)
    for i in range(1, nr + 1):
        npx, _first, ct, _st, _phi0 = oracle.ring_geometry(nside, i)
        z[i - 1] = ct
        n[i - 1] = npx
    return z, n


def zonal_matrix(nside: int, lmax_w: int) -> np.ndarray:
    """lambda_l0(theta_i) for l = 0 .. lmax_w (rows) and every ring (columns)."""
    nr = 4 * nside - 1
    lam = np.empty((lmax_w + 1, nr), dtype=np.longdouble)
    for i in range(1, nr + 1):
        lam[:, i - 1] = oracle.lambda_lm_ring(nside, i, lmax_w, 0)
    return lam


def ring_weights(nside: int, lmax_w: int = 0) -> np.ndarray:
    if lmax_w <= 0:
        lmax_w = 3 * nside
    _z, n = ring_table(nside)
    lam = zonal_matrix(nside, lmax_w)
    w0 = np.longdouble(4.0) * np.pi / np.longdouble(12 * nside * nside)
    sq = np.sqrt(n)
    M = lam * sq[None, :]
    r = -(lam * n[None, :]) @ np.full(n.shape, w0, dtype=np.longdouble)
    r[0] += np.sqrt(np.longdouble(4.0) * np.pi)
    # minimum-norm solution of M u = r (u = sqrt(N) (w - w0)); lstsq works in double: iterate on the residual in long double
    u = np.zeros(n.shape, dtype=np.longdouble)
    Md = M.astype(np.float64)
    for _ in range(4):
        res = r - M @ u
        du = np.linalg.lstsq(Md, res.astype(np.float64), rcond=1e-12)[0]
        u = u + du.astype(np.longdouble)
    return np.asarray(w0 + u / sq, dtype=np.float64)
