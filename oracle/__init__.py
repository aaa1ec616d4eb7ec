"""CPU oracle for the HEALPix RING spherical harmonic transform -- TEST INFRASTRUCTURE ONLY.

Thin ctypes wrapper around ``oracle/sht_oracle.c`` (plain C, long double, OpenMP over rings).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this package; the product path (``paper_2510_01785_b200``) never does, and this
package never imports the product.  See the header of ``sht_oracle.c`` for what is computed and
which passage of the paper each function follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sht_oracle.c")
_LIB = os.path.join(_HERE, "libsht_oracle.so")


_LIB_SAN = os.path.join(_HERE, "libsht_oracle_san.so")


def build(force: bool = False, sanitize: bool = False) -> str:
    """Compile the oracle with gcc (idempotent). Building the checker is not using it.

    sanitize=True builds a second library with -fsanitize=address,undefined; it is loaded instead
    of the plain one when the environment variable SHT_ORACLE_LIB names it, in a process started with libasan
    preloaded (tests/test_oracle_pins.py::test_oracle_under_asan_ubsan does that in a subprocess)."""
    lib = _LIB_SAN if sanitize else _LIB
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] \
            if sanitize else ["-O2"]
        cmd = ["gcc"] + flags + ["-std=c11", "-fopenmp", "-shared", "-fPIC", "-o", lib, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return lib


_lib = None


def _load():
    global _lib
    if _lib is None:
        path = os.environ.get("SHT_ORACLE_LIB")
        if not path:
            path = build()
        _lib = ctypes.CDLL(path)
        i32, i64 = ctypes.c_int, ctypes.c_int64
        vp = ctypes.c_void_p
        _lib.oracle_alm_count.restype = i64
        _lib.oracle_alm_count.argtypes = [i32, i32]
        _lib.oracle_alm_index.restype = i64
        _lib.oracle_alm_index.argtypes = [i32, i32, i32]
        _lib.oracle_ring_geometry.argtypes = [i32, i32, vp, vp, vp, vp, vp]
        _lib.oracle_lambda.argtypes = [i32, i32, ctypes.c_double, vp]
        _lib.oracle_lambda_ring.argtypes = [i32, i32, i32, i32, vp]
        _lib.oracle_ring_dft.argtypes = [i32, i32, vp, i32, vp]
        _lib.oracle_ring_synth.argtypes = [i32, i32, vp, i32, vp]
        _lib.oracle_alm2map.argtypes = [i32, i32, i32, vp, vp]
        _lib.oracle_map2alm.argtypes = [i32, i32, i32, vp, vp, vp]
        _lib.oracle_alm2map_adjoint.argtypes = [i32, i32, i32, vp, vp]
        _lib.oracle_map2alm_adjoint.argtypes = [i32, i32, i32, vp, vp, vp]
        _lib.oracle_map2alm_subset.argtypes = [i32, i32, i32, vp, vp, i32, vp, vp, vp]
        _lib.oracle_alm2map_adjoint_subset.argtypes = [i32, i32, i32, vp, i32, vp, vp, vp]
        _lib.oracle_alm2map_rings.argtypes = [i32, i32, i32, vp, i32, vp, vp]
        _lib.oracle_map2alm_adjoint_rings.argtypes = [i32, i32, i32, vp, vp, i32, vp, vp]
        _lib.oracle_num_threads.restype = i32
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise ValueError(f"oracle {what} failed with status {rc}")


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def npix(nside: int) -> int:
    return 12 * nside * nside


def alm_count(lmax: int, mmax: int) -> int:
    return int(_load().oracle_alm_count(lmax, mmax))


def alm_index(lmax: int, l: int, m: int) -> int:
    return int(_load().oracle_alm_index(lmax, l, m))


def ring_geometry(nside: int, ring: int):
    """(N_i, start_i, cos theta_i, sin theta_i, phi0_i) of ring ``ring`` (1-based, north to south)."""
    n = ctypes.c_int64()
    st = ctypes.c_int64()
    c = ctypes.c_double()
    s = ctypes.c_double()
    p = ctypes.c_double()
    _check(_load().oracle_ring_geometry(nside, ring, ctypes.byref(n), ctypes.byref(st), ctypes.byref(c),
                                        ctypes.byref(s), ctypes.byref(p)), "ring_geometry")
    return n.value, st.value, c.value, s.value, p.value


def lambda_lm(lmax: int, m: int, theta: float) -> np.ndarray:
    """lambda_lm(theta) for l = 0..lmax (zeros for l < m)."""
    out = np.zeros(lmax + 1)
    _check(_load().oracle_lambda(lmax, m, float(theta), _ptr(out)), "lambda")
    return out


def lambda_lm_ring(nside: int, ring: int, lmax: int, m: int) -> np.ndarray:
    out = np.zeros(lmax + 1)
    _check(_load().oracle_lambda_ring(nside, ring, lmax, m, _ptr(out)), "lambda_ring")
    return out


def ring_dft(nside: int, ring: int, p, mmax: int) -> np.ndarray:
    """F_m = sum_x p_x exp(-i m (phi0 + 2 pi x / N)), m = 0..mmax, by the direct O(N mmax) sum."""
    p = _f64(p)
    out = np.zeros(mmax + 1, dtype=np.complex128)
    _check(_load().oracle_ring_dft(nside, ring, _ptr(p), mmax, _ptr(out)), "ring_dft")
    return out


def ring_synth(nside: int, ring: int, G) -> np.ndarray:
    """p_x = Re G_0 + 2 sum_{m>=1} Re(G_m exp(+i m (phi0 + 2 pi x / N))) for one ring, G = G_0..G_mmax."""
    G = _c128(G)
    out = np.zeros(ring_geometry(nside, ring)[0])
    _check(_load().oracle_ring_synth(nside, ring, _ptr(G), len(G) - 1, _ptr(out)), "ring_synth")
    return out


def alm2map(nside: int, lmax: int, mmax: int, alm) -> np.ndarray:
    alm = _c128(alm)
    assert alm.shape == (alm_count(lmax, mmax),)
    out = np.zeros(npix(nside))
    _check(_load().oracle_alm2map(nside, lmax, mmax, _ptr(alm), _ptr(out)), "alm2map")
    return out


def map2alm(nside: int, lmax: int, mmax: int, hmap, ring_weights=None) -> np.ndarray:
    hmap = _f64(hmap)
    assert hmap.shape == (npix(nside),)
    w = None if ring_weights is None else _f64(ring_weights)
    assert w is None or w.shape == (4 * nside - 1,)
    out = np.zeros(alm_count(lmax, mmax), dtype=np.complex128)
    _check(_load().oracle_map2alm(nside, lmax, mmax, _ptr(hmap), _ptr(w), _ptr(out)), "map2alm")
    return out


def alm2map_adjoint(nside: int, lmax: int, mmax: int, gmap) -> np.ndarray:
    gmap = _f64(gmap)
    assert gmap.shape == (npix(nside),)
    out = np.zeros(alm_count(lmax, mmax), dtype=np.complex128)
    _check(_load().oracle_alm2map_adjoint(nside, lmax, mmax, _ptr(gmap), _ptr(out)), "alm2map_adjoint")
    return out


def map2alm_adjoint(nside: int, lmax: int, mmax: int, galm, ring_weights=None) -> np.ndarray:
    galm = _c128(galm)
    assert galm.shape == (alm_count(lmax, mmax),)
    w = None if ring_weights is None else _f64(ring_weights)
    out = np.zeros(npix(nside))
    _check(_load().oracle_map2alm_adjoint(nside, lmax, mmax, _ptr(galm), _ptr(w), _ptr(out)), "map2alm_adjoint")
    return out


def map2alm_iter(nside: int, lmax: int, mmax: int, hmap, n_iter: int, ring_weights=None) -> np.ndarray:
    """Iterative refinement of the analysis, Eq. 4 step by step in the paper's notation:
    a^(0) = A f;  r^(k+1) = f - S a^(k);  a^(k+1) = a^(k) + A r^(k+1)."""
    f = _f64(hmap)
    a = map2alm(nside, lmax, mmax, f, ring_weights)
    for _ in range(n_iter):
        r = f - alm2map(nside, lmax, mmax, a)
        a = a + map2alm(nside, lmax, mmax, r, ring_weights)
    return a


def map2alm_subset(nside, lmax, mmax, hmap, sel_l, sel_m, ring_weights=None) -> np.ndarray:
    hmap = _f64(hmap)
    sel_l, sel_m = _i32(sel_l), _i32(sel_m)
    w = None if ring_weights is None else _f64(ring_weights)
    out = np.zeros(len(sel_l), dtype=np.complex128)
    _check(_load().oracle_map2alm_subset(nside, lmax, mmax, _ptr(hmap), _ptr(w), len(sel_l), _ptr(sel_l),
                                         _ptr(sel_m), _ptr(out)), "map2alm_subset")
    return out


def alm2map_adjoint_subset(nside, lmax, mmax, gmap, sel_l, sel_m) -> np.ndarray:
    gmap = _f64(gmap)
    sel_l, sel_m = _i32(sel_l), _i32(sel_m)
    out = np.zeros(len(sel_l), dtype=np.complex128)
    _check(_load().oracle_alm2map_adjoint_subset(nside, lmax, mmax, _ptr(gmap), len(sel_l), _ptr(sel_l),
                                                 _ptr(sel_m), _ptr(out)), "alm2map_adjoint_subset")
    return out


def _rings_len(nside, rings) -> int:
    return int(sum(ring_geometry(nside, int(r))[0] for r in rings))


def alm2map_rings(nside, lmax, mmax, alm, rings) -> np.ndarray:
    """Pixels of the selected rings (1-based), concatenated in the order given."""
    alm = _c128(alm)
    rings = _i32(rings)
    out = np.zeros(_rings_len(nside, rings))
    _check(_load().oracle_alm2map_rings(nside, lmax, mmax, _ptr(alm), len(rings), _ptr(rings), _ptr(out)),
           "alm2map_rings")
    return out


def map2alm_adjoint_rings(nside, lmax, mmax, galm, rings, ring_weights=None) -> np.ndarray:
    galm = _c128(galm)
    rings = _i32(rings)
    w = None if ring_weights is None else _f64(ring_weights)
    out = np.zeros(_rings_len(nside, rings))
    _check(_load().oracle_map2alm_adjoint_rings(nside, lmax, mmax, _ptr(galm), _ptr(w), len(rings), _ptr(rings),
                                                _ptr(out)), "map2alm_adjoint_rings")
    return out
