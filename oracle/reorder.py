"""CPU oracle for NESTED <-> RING reordering -- TEST INFRASTRUCTURE ONLY (same rules as oracle/__init__.py).

The paper states WHAT the layouts are (RING = west-to-east along iso-latitude rings, rings north to
south; NESTED = Z-order / Morton curve inside each of the 12 base faces) and that conversion goes through
(x, y, f).  It gives no formula.  This oracle therefore uses the one definition both layouts share:
a pixel IS its centre on the sphere.  For every NESTED index it
  1. de-interleaves the Morton code into (x, y) inside face f            (Fig. 4B),
  2. places the pixel centre in the HEALPix projection plane (Gorski et al., ref [1] P:416, section 4.1: the 12
     faces are unit diamonds, 4 per row; x runs along the north-east edge, y along the north-west edge from the
     southern corner), and maps plane -> sphere: equatorial zone z = 2 Y / 3, phi = pi X / 4; polar zones
     z = +-(1 - sigma^2 / 3), sigma = 2 - |Y|, phi compressed towards the face's meridian by 1 / sigma,
  3. looks the centre up in the ring table of oracle/sht_oracle.c (already pinned: tests/test_oracle_pins.py),
     nearest ring in z, nearest pixel in phi -- and insists that the match is exact to 1e-12.
Nothing here shares code or formulas with csrc/reorder.cu (which uses the integer ring / in-ring arithmetic).
"""
from __future__ import annotations

import numpy as np

from . import ring_geometry


def _deinterleave(code: np.ndarray):
    x = np.zeros_like(code)
    y = np.zeros_like(code)
    for b in range(32):
        x |= ((code >> (2 * b)) & 1) << b
        y |= ((code >> (2 * b + 1)) & 1) << b
    return x, y


def nested_centres(nside: int):
    """(z, phi) of the centre of every NESTED pixel, from the projection-plane construction."""
    npix = 12 * nside * nside
    ip = np.arange(npix, dtype=np.int64)
    f = ip // (nside * nside)
    x, y = _deinterleave(ip % (nside * nside))
    # southern corner of face f in the plane: X in units of pi/4 (0..8), Y in units where |Y| = 1 is |z| = 2/3
    row = f // 4
    col = f % 4
    cx = np.where(row == 1, 2.0 * col, 2.0 * col + 1.0)
    cy = -row.astype(np.float64)
    u = (x + 0.5) / nside  # along the north-east edge
    v = (y + 0.5) / nside  # along the north-west edge
    X = cx + u - v
    Y = cy + u + v
    z = np.empty(npix)
    phi = np.empty(npix)
    eq = np.abs(Y) <= 1.0
    z[eq] = 2.0 * Y[eq] / 3.0
    phi[eq] = X[eq] * (np.pi / 4.0)
    po = ~eq
    sigma = 2.0 - np.abs(Y[po])
    z[po] = np.sign(Y[po]) * (1.0 - sigma * sigma / 3.0)
    xm = 2.0 * col[po] + 1.0  # meridian of the polar face (and of the cap triangle above / below it)
    phi[po] = (xm + (X[po] - xm) / sigma) * (np.pi / 4.0)
    return z, np.mod(phi, 2.0 * np.pi)


def _plane_to_sphere(X, Y, col):
    """HEALPix projection plane -> (z, phi); col = column of the face (its meridian in the polar zones)."""
    z = np.empty(X.shape)
    phi = np.empty(X.shape)
    eq = np.abs(Y) <= 1.0
    z[eq] = 2.0 * Y[eq] / 3.0
    phi[eq] = X[eq] * (np.pi / 4.0)
    po = ~eq
    sigma = 2.0 - np.abs(Y[po])
    z[po] = np.sign(Y[po]) * (1.0 - sigma * sigma / 3.0)
    xm = 2.0 * col[po] + 1.0
    phi[po] = (xm + (X[po] - xm) / sigma) * (np.pi / 4.0)
    return z, np.mod(phi, 2.0 * np.pi)


def flat_centres(nside: int, corner: int, sense: int):
    """(z, phi) of the centre of every pixel of the flat layout (Fig. 3C; reading R12): face f is a
    row-major nside x nside image whose origin is the face's corner `corner` (0 S, 1 E, 2 N, 3 W) and whose fast axis
    runs along the face edge towards the counter-clockwise (sense 0: S -> E -> N -> W) or clockwise (sense 1) neighbour
    corner, the slow axis along the other edge.  Written with the corners of the face diamond in the projection plane,
    not with (x, y) index arithmetic.  The paper defines the layout only by Fig. 3C: that this reading matches the figure's
    face orientation is PARITY UNPINNED (R12); the stated geometry itself is pinned in tests/test_reorder.py."""
    npix = 12 * nside * nside
    ip = np.arange(npix, dtype=np.int64)
    f = ip // (nside * nside)
    r = ip % (nside * nside)
    row_i = r // nside
    col_i = r % nside
    frow = f // 4
    fcol = f % 4
    cx = np.where(frow == 1, 2.0 * fcol, 2.0 * fcol + 1.0)
    cy = -frow.astype(np.float64)
    corners = [(cx, cy), (cx + 1.0, cy + 1.0), (cx, cy + 2.0), (cx - 1.0, cy + 1.0)]  # S, E, N, W: counter-clockwise
    O = corners[corner]
    ccw = corners[(corner + 1) % 4]
    cw = corners[(corner - 1) % 4]
    A, B = (ccw, cw) if sense == 0 else (cw, ccw)  # fast edge, slow edge
    s = (col_i + 0.5) / nside
    t = (row_i + 0.5) / nside
    X = O[0] + s * (A[0] - O[0]) + t * (B[0] - O[0])
    Y = O[1] + s * (A[1] - O[1]) + t * (B[1] - O[1])
    return _plane_to_sphere(X, Y, fcol)


def _lookup_ring_index(nside: int, z, phi) -> np.ndarray:
    """RING index of the pixels with centres (z, phi), by matching against the (pinned) ring table."""
    nrings = 4 * nside - 1
    N = np.empty(nrings, dtype=np.int64)
    start = np.empty(nrings, dtype=np.int64)
    zr = np.empty(nrings)
    phi0 = np.empty(nrings)
    for r in range(nrings):
        n, st, c, _s, p0 = ring_geometry(nside, r + 1)
        N[r], start[r], zr[r], phi0[r] = n, st, c, p0
    pos = np.clip(np.searchsorted(-zr, -z), 1, nrings - 1)
    ring = np.where(np.abs(zr[pos - 1] - z) < np.abs(zr[pos] - z), pos - 1, pos)
    assert np.abs(zr[ring] - z).max() < 1e-12, "a pixel centre is not on any ring"
    t = (phi - phi0[ring]) * N[ring] / (2.0 * np.pi)
    k = np.rint(t)
    assert np.abs(t - k).max() < 1e-9, "a pixel centre is not a RING pixel centre"
    return start[ring] + np.mod(k.astype(np.int64), N[ring])


def flat2ring_table(nside: int, corner: int, sense: int) -> np.ndarray:
    """ring_index[ipflat] for the flat layout (corner, sense)."""
    z, phi = flat_centres(nside, corner, sense)
    return _lookup_ring_index(nside, z, phi)


def nest2ring_table(nside: int) -> np.ndarray:
    """ring_index[ipnest] for all 12 nside^2 pixels, by matching pixel centres against the ring table."""
    nrings = 4 * nside - 1
    N = np.empty(nrings, dtype=np.int64)
    start = np.empty(nrings, dtype=np.int64)
    zr = np.empty(nrings)
    phi0 = np.empty(nrings)
    for r in range(nrings):
        n, st, c, _s, p0 = ring_geometry(nside, r + 1)
        N[r], start[r], zr[r], phi0[r] = n, st, c, p0
    z, phi = nested_centres(nside)
    # rings are sorted by decreasing z
    pos = np.searchsorted(-zr, -z)
    pos = np.clip(pos, 1, nrings - 1)
    ring = np.where(np.abs(zr[pos - 1] - z) < np.abs(zr[pos] - z), pos - 1, pos)
    assert np.abs(zr[ring] - z).max() < 1e-12, "a NESTED pixel centre is not on any ring"
    t = (phi - phi0[ring]) * N[ring] / (2.0 * np.pi)
    k = np.rint(t)
    assert np.abs(t - k).max() < 1e-9, "a NESTED pixel centre is not a RING pixel centre"
    out = start[ring] + np.mod(k.astype(np.int64), N[ring])
    return out


def nest2ring(hmap_nest: np.ndarray, nside: int) -> np.ndarray:
    """Reorder [..., npix] from NESTED to RING."""
    tab = nest2ring_table(nside)
    out = np.empty_like(hmap_nest)
    out[..., tab] = hmap_nest
    return out


def ring2nest(hmap_ring: np.ndarray, nside: int) -> np.ndarray:
    """Reorder [..., npix] from RING to NESTED."""
    return hmap_ring[..., nest2ring_table(nside)]


def alm_resize(alm: np.ndarray, lmax_in: int, mmax_in: int, lmax_out: int, mmax_out: int) -> np.ndarray:
    """Truncate / zero-extend coefficients, the definition written out: every (l, m) of the output that
    the input has is copied, the others are 0.  alm: [..., nalm_in], m-major packed index m (2 lmax + 1 - m) / 2 + l."""
    nout = (mmax_out + 1) * (lmax_out + 1) - mmax_out * (mmax_out + 1) // 2
    out = np.zeros(alm.shape[:-1] + (nout,), dtype=alm.dtype)
    for m in range(mmax_out + 1):
        for l in range(m, lmax_out + 1):
            if m <= mmax_in and l <= lmax_in:
                out[..., m * (2 * lmax_out + 1 - m) // 2 + l] = alm[..., m * (2 * lmax_in + 1 - m) // 2 + l]
    return out
