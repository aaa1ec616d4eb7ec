"""Thin Python binding of libcuhpx.so (include/cuhpx.h): argument marshalling only.

Every step of the transforms runs in the CUDA kernels behind the C ABI; PyTorch is used for device memory
and streams.  There is no CPU fallback: if the shared library is missing the import fails, and the compute
calls raise when no CUDA device is present.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcuhpx.so")

CUHPX_F32, CUHPX_F64 = 0, 1
CUHPX_OK, CUHPX_EINVAL, CUHPX_EWORKSPACE, CUHPX_EUNSUPPORTED, CUHPX_ECUDA = 0, 1, 2, 3, 4

#: every symbol include/cuhpx.h declares
EXPORTS = [
    "cuhpx_npix", "cuhpx_nrings", "cuhpx_alm_count", "cuhpx_alm_index", "cuhpx_status_string", "cuhpx_ring_info",
    "cuhpx_workspace_bytes", "cuhpx_workspace_init", "cuhpx_workspace_check", "cuhpx_map2alm", "cuhpx_alm2map",
    "cuhpx_alm2map_adjoint", "cuhpx_map2alm_adjoint", "cuhpx_spectra_stride", "cuhpx_spectra_offset",
    "cuhpx_plan_mcut", "cuhpx_analysis_fft_stage", "cuhpx_analysis_legendre_stage",
    "cuhpx_synthesis_legendre_stage", "cuhpx_synthesis_fft_stage", "cuhpx_fma_peak_probe", "cuhpx_plan_stats",
    "cuhpx_grid_npix", "cuhpx_grid_ring_info", "cuhpx_grid_workspace_bytes", "cuhpx_grid_workspace_init",
    "cuhpx_grid_alm2map", "cuhpx_grid_map2alm", "cuhpx_grid_alm2map_adjoint", "cuhpx_grid_map2alm_adjoint",
    "cuhpx_reorder_layout", "cuhpx_layout_index",
    "cuhpx_map2alm_iter", "cuhpx_ring_weights_workspace_bytes", "cuhpx_ring_weights", "cuhpx_ring_weights_noalloc", "cuhpx_late_start_stats", "cuhpx_reorder", "cuhpx_nest2ring_index", "cuhpx_alm_resize",
]
CUHPX_NEST2RING, CUHPX_RING2NEST = 0, 1
CUHPX_GRID_HEALPIX, CUHPX_GRID_GAUSS_LEGENDRE, CUHPX_GRID_EQUIANGULAR = 0, 1, 2


class CuhpxError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(f"{what}: {status_string(status)}")


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2510_01785_b200.build` "
            "(there is no CPU fallback for the cuHPX transforms)")
    lib = ctypes.CDLL(LIB_PATH)
    i, sz, vp = ctypes.c_int, ctypes.c_size_t, ctypes.c_void_p
    lib.cuhpx_npix.restype = sz
    lib.cuhpx_npix.argtypes = [i]
    lib.cuhpx_nrings.restype = sz
    lib.cuhpx_nrings.argtypes = [i]
    lib.cuhpx_alm_count.restype = sz
    lib.cuhpx_alm_count.argtypes = [i, i]
    lib.cuhpx_alm_index.restype = sz
    lib.cuhpx_alm_index.argtypes = [i, i, i]
    lib.cuhpx_status_string.restype = ctypes.c_char_p
    lib.cuhpx_status_string.argtypes = [i]
    lib.cuhpx_ring_info.argtypes = [i, i, vp, vp, vp, vp]
    lib.cuhpx_workspace_bytes.restype = sz
    lib.cuhpx_workspace_bytes.argtypes = [i, i, i, i, i]
    lib.cuhpx_workspace_init.argtypes = [i, i, i, i, i, vp, sz, vp]
    lib.cuhpx_workspace_check.argtypes = [i, i, i, i, i, vp, sz, vp]
    lib.cuhpx_map2alm.argtypes = [i, i, i, i, i, vp, vp, vp, vp, sz, vp]
    lib.cuhpx_alm2map.argtypes = [i, i, i, i, i, vp, vp, vp, sz, vp]
    lib.cuhpx_alm2map_adjoint.argtypes = [i, i, i, i, i, vp, vp, vp, sz, vp]
    lib.cuhpx_map2alm_adjoint.argtypes = [i, i, i, i, i, vp, vp, vp, vp, sz, vp]
    lib.cuhpx_map2alm_iter.argtypes = [i, i, i, i, i, vp, vp, vp, i, vp, vp, vp, sz, vp]
    lib.cuhpx_reorder.argtypes = [i, i, i, i, vp, vp, vp]
    lib.cuhpx_grid_npix.argtypes = [i, i, i]
    lib.cuhpx_grid_npix.restype = sz
    lib.cuhpx_grid_ring_info.argtypes = [i, i, i, i, vp, vp]
    lib.cuhpx_grid_workspace_bytes.argtypes = [i, i, i, i, i, i, i]
    lib.cuhpx_grid_workspace_bytes.restype = sz
    lib.cuhpx_grid_workspace_init.argtypes = [i, i, i, i, i, i, i, vp, sz, vp]
    lib.cuhpx_grid_alm2map.argtypes = [i, i, i, i, i, i, i, vp, vp, vp, sz, vp]
    lib.cuhpx_grid_map2alm.argtypes = [i, i, i, i, i, i, i, vp, vp, vp, vp, sz, vp]
    lib.cuhpx_grid_alm2map_adjoint.argtypes = [i, i, i, i, i, i, i, vp, vp, vp, sz, vp]
    lib.cuhpx_grid_map2alm_adjoint.argtypes = [i, i, i, i, i, i, i, vp, vp, vp, vp, sz, vp]
    lib.cuhpx_reorder_layout.argtypes = [i, i, i, i, i, vp, vp, vp]
    lib.cuhpx_layout_index.argtypes = [i, i, i, ctypes.c_longlong]
    lib.cuhpx_layout_index.restype = ctypes.c_longlong
    lib.cuhpx_ring_weights_workspace_bytes.argtypes = [i, i]
    lib.cuhpx_ring_weights_workspace_bytes.restype = sz
    lib.cuhpx_ring_weights.argtypes = [i, i, vp, vp, sz, vp]
    lib.cuhpx_ring_weights_noalloc.argtypes = [i, i, vp, vp]
    lib.cuhpx_alm_resize.argtypes = [i, i, i, i, i, i, vp, vp, vp]
    lib.cuhpx_nest2ring_index.restype = ctypes.c_longlong
    lib.cuhpx_nest2ring_index.argtypes = [i, ctypes.c_longlong]
    lib.cuhpx_spectra_stride.restype = sz
    lib.cuhpx_spectra_stride.argtypes = [i]
    lib.cuhpx_spectra_offset.restype = sz
    lib.cuhpx_spectra_offset.argtypes = [i, i, i, i, i]
    lib.cuhpx_plan_mcut.argtypes = [i, i, i, i, i, vp]
    lib.cuhpx_analysis_fft_stage.argtypes = [i, i, i, i, i, vp, vp, i, vp, sz, vp]
    lib.cuhpx_analysis_legendre_stage.argtypes = [i, i, i, i, i, vp, i, vp, sz, vp]
    lib.cuhpx_synthesis_legendre_stage.argtypes = [i, i, i, i, i, vp, i, vp, sz, vp]
    lib.cuhpx_synthesis_fft_stage.argtypes = [i, i, i, i, i, vp, vp, i, vp, sz, vp]
    lib.cuhpx_fma_peak_probe.argtypes = [i, i, vp, vp, vp]
    lib.cuhpx_plan_stats.argtypes = [i, i, i, i, i, vp, i]
    lib.cuhpx_late_start_stats.argtypes = [i, i, i, i, i, vp, sz, vp, vp]
    return lib


_lib = _load()


def lib() -> ctypes.CDLL:
    return _lib


def status_string(status: int) -> str:
    return _lib.cuhpx_status_string(int(status)).decode()


def _check(status: int, what: str) -> None:
    if status != CUHPX_OK:
        raise CuhpxError(status, what)


def cuhpx_npix(nside: int) -> int:
    return int(_lib.cuhpx_npix(nside))


def cuhpx_nrings(nside: int) -> int:
    return int(_lib.cuhpx_nrings(nside))


def cuhpx_alm_count(lmax: int, mmax: int) -> int:
    return int(_lib.cuhpx_alm_count(lmax, mmax))


def cuhpx_alm_index(lmax: int, l: int, m: int) -> int:
    return int(_lib.cuhpx_alm_index(lmax, l, m))


def cuhpx_spectra_stride(mmax: int) -> int:
    return int(_lib.cuhpx_spectra_stride(mmax))


def cuhpx_ring_info(nside: int, ring: int):
    n, s = ctypes.c_longlong(), ctypes.c_longlong()
    c, p = ctypes.c_double(), ctypes.c_double()
    _check(_lib.cuhpx_ring_info(nside, ring, ctypes.byref(n), ctypes.byref(s), ctypes.byref(c), ctypes.byref(p)),
           "cuhpx_ring_info")
    return n.value, s.value, c.value, p.value


def cuhpx_workspace_bytes(nside: int, lmax: int, mmax: int, batch: int, dtype: int) -> int:
    return int(_lib.cuhpx_workspace_bytes(nside, lmax, mmax, batch, dtype))


def _dtype_code(t: torch.dtype) -> int:
    if t in (torch.float32, torch.complex64):
        return CUHPX_F32
    if t in (torch.float64, torch.complex128):
        return CUHPX_F64
    raise TypeError(f"unsupported dtype {t}")


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dev_ptr(t: torch.Tensor | None) -> int | None:
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("cuhpx needs contiguous CUDA tensors")
    return t.data_ptr()


def cuhpx_workspace_init(nside, lmax, mmax, batch, dtype, workspace: torch.Tensor, stream=None) -> None:
    _check(_lib.cuhpx_workspace_init(nside, lmax, mmax, batch, dtype, _dev_ptr(workspace),
                                     workspace.numel() * workspace.element_size(), _stream_ptr(stream)),
           "cuhpx_workspace_init")


def cuhpx_workspace_check(nside, lmax, mmax, batch, dtype, workspace: torch.Tensor, stream=None) -> None:
    """Synchronising: raises CuhpxError(CUHPX_EWORKSPACE) unless `workspace` is initialised for these parameters."""
    _check(_lib.cuhpx_workspace_check(nside, lmax, mmax, batch, dtype, _dev_ptr(workspace),
                                      workspace.numel() * workspace.element_size(), _stream_ptr(stream)),
           "cuhpx_workspace_check")


def _ws_args(ws: torch.Tensor):
    return _dev_ptr(ws), ws.numel() * ws.element_size()


def cuhpx_map2alm(nside, lmax, mmax, batch, dtype, d_map, d_alm, d_ring_weights, workspace, stream=None) -> None:
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_map2alm(nside, lmax, mmax, batch, dtype, _dev_ptr(d_map), _dev_ptr(d_alm),
                              _dev_ptr(d_ring_weights), p, n, _stream_ptr(stream)), "cuhpx_map2alm")


def cuhpx_map2alm_iter(nside, lmax, mmax, batch, dtype, d_map, d_alm, d_ring_weights, n_iter, d_scratch_map,
                       d_scratch_alm, workspace, stream=None) -> None:
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_map2alm_iter(nside, lmax, mmax, batch, dtype, _dev_ptr(d_map), _dev_ptr(d_alm),
                                   _dev_ptr(d_ring_weights), int(n_iter), _dev_ptr(d_scratch_map),
                                   _dev_ptr(d_scratch_alm), p, n, _stream_ptr(stream)), "cuhpx_map2alm_iter")


def cuhpx_alm2map(nside, lmax, mmax, batch, dtype, d_alm, d_map, workspace, stream=None) -> None:
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_alm2map(nside, lmax, mmax, batch, dtype, _dev_ptr(d_alm), _dev_ptr(d_map), p, n,
                              _stream_ptr(stream)), "cuhpx_alm2map")


def cuhpx_alm2map_adjoint(nside, lmax, mmax, batch, dtype, d_gmap, d_galm, workspace, stream=None) -> None:
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_alm2map_adjoint(nside, lmax, mmax, batch, dtype, _dev_ptr(d_gmap), _dev_ptr(d_galm), p, n,
                                      _stream_ptr(stream)), "cuhpx_alm2map_adjoint")


def cuhpx_map2alm_adjoint(nside, lmax, mmax, batch, dtype, d_galm, d_gmap, d_ring_weights, workspace,
                          stream=None) -> None:
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_map2alm_adjoint(nside, lmax, mmax, batch, dtype, _dev_ptr(d_galm), _dev_ptr(d_gmap),
                                      _dev_ptr(d_ring_weights), p, n, _stream_ptr(stream)), "cuhpx_map2alm_adjoint")


def cuhpx_ring_weights_workspace_bytes(nside: int, lmax_w: int = 0) -> int:
    return int(_lib.cuhpx_ring_weights_workspace_bytes(nside, lmax_w))


def cuhpx_ring_weights(nside, lmax_w, d_weights, workspace, stream=None) -> None:
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_ring_weights(nside, lmax_w, _dev_ptr(d_weights), p, n, _stream_ptr(stream)), "cuhpx_ring_weights")


CUHPX_NOALLOC_SCRATCH_BYTES = 8 << 20


def cuhpx_ring_weights_noalloc(nside, lmax_w, d_weights, stream=None) -> None:
    """cuhpx_ring_weights with the scratch in the library's built-in device array (no device allocation; requests needing
    more than CUHPX_NOALLOC_SCRATCH_BYTES raise CUHPX_EWORKSPACE; calls on one device share the array: serialise them)."""
    _check(_lib.cuhpx_ring_weights_noalloc(nside, lmax_w, _dev_ptr(d_weights), _stream_ptr(stream)), "cuhpx_ring_weights_noalloc")


def ring_weights(nside: int, lmax_w: int = 0, device="cuda") -> torch.Tensor:
    """Ring quadrature weights [4 nside - 1] (fp64, device) exact for the m = 0 modes up to lmax_w (default 3 nside)."""
    nbytes = cuhpx_ring_weights_workspace_bytes(nside, lmax_w)
    if nbytes == 0:
        raise CuhpxError(1, "cuhpx_ring_weights_workspace_bytes")
    ws = torch.empty(nbytes, dtype=torch.uint8, device=device)
    w = torch.empty(4 * nside - 1, dtype=torch.float64, device=device)
    with torch.cuda.device(w.device):
        cuhpx_ring_weights(nside, lmax_w, w, ws)
    return w


def cuhpx_reorder(nside, batch, dtype, direction, d_in, d_out, stream=None) -> None:
    _check(_lib.cuhpx_reorder(nside, batch, dtype, int(direction), _dev_ptr(d_in), _dev_ptr(d_out), _stream_ptr(stream)),
           "cuhpx_reorder")


CUHPX_LAYOUT_RING, CUHPX_LAYOUT_NESTED = 0, 1


def CUHPX_LAYOUT_FLAT(corner: int, sense: int) -> int:
    return 2 + 2 * corner + sense


def cuhpx_reorder_layout(nside, batch, dtype, src_layout, dst_layout, d_in, d_out, stream=None) -> None:
    _check(_lib.cuhpx_reorder_layout(nside, batch, dtype, int(src_layout), int(dst_layout), _dev_ptr(d_in), _dev_ptr(d_out),
                                     _stream_ptr(stream)), "cuhpx_reorder_layout")


def cuhpx_layout_index(nside: int, src_layout: int, dst_layout: int, ip_src: int) -> int:
    return int(_lib.cuhpx_layout_index(nside, src_layout, dst_layout, ip_src))


def reorder_layout(hmap: torch.Tensor, nside: int, src_layout: int, dst_layout: int) -> torch.Tensor:
    """[batch, npix] between RING / NESTED / flat layouts."""
    out = torch.empty_like(hmap)
    cuhpx_reorder_layout(nside, hmap.shape[0], _dtype_code(hmap.dtype), src_layout, dst_layout, hmap, out)
    return out


def cuhpx_alm_resize(lmax_in, mmax_in, lmax_out, mmax_out, batch, dtype, d_in, d_out, stream=None) -> None:
    _check(_lib.cuhpx_alm_resize(lmax_in, mmax_in, lmax_out, mmax_out, batch, dtype, _dev_ptr(d_in), _dev_ptr(d_out),
                                 _stream_ptr(stream)), "cuhpx_alm_resize")


def alm_resize(alm: torch.Tensor, lmax_in: int, mmax_in: int, lmax_out: int, mmax_out: int) -> torch.Tensor:
    """Truncate / zero-extend [batch, nalm] coefficients to another (lmax, mmax)."""
    out = torch.empty(alm.shape[0], cuhpx_alm_count(lmax_out, mmax_out), dtype=alm.dtype, device=alm.device)
    cuhpx_alm_resize(lmax_in, mmax_in, lmax_out, mmax_out, alm.shape[0], _dtype_code(alm.dtype), alm, out)
    return out


def cuhpx_nest2ring_index(nside: int, ipnest: int) -> int:
    return int(_lib.cuhpx_nest2ring_index(nside, ipnest))


def nest2ring(hmap: torch.Tensor, nside: int) -> torch.Tensor:
    """[batch, npix] NESTED -> RING (paper section III-B)."""
    out = torch.empty_like(hmap)
    cuhpx_reorder(nside, hmap.shape[0], _dtype_code(hmap.dtype), CUHPX_NEST2RING, hmap, out)
    return out


def ring2nest(hmap: torch.Tensor, nside: int) -> torch.Tensor:
    """[batch, npix] RING -> NESTED (paper section III-B)."""
    out = torch.empty_like(hmap)
    cuhpx_reorder(nside, hmap.shape[0], _dtype_code(hmap.dtype), CUHPX_RING2NEST, hmap, out)
    return out


def cuhpx_analysis_fft_stage(params, d_map, d_ring_weights, use_weights, workspace, stream=None) -> None:
    """params = (nside, lmax, mmax, batch, dtype code), e.g. Transform.params"""
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_analysis_fft_stage(*params, _dev_ptr(d_map), _dev_ptr(d_ring_weights), int(use_weights), p, n,
                                         _stream_ptr(stream)), "cuhpx_analysis_fft_stage")


def cuhpx_analysis_legendre_stage(params, d_alm, adjoint, workspace, stream=None) -> None:
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_analysis_legendre_stage(*params, _dev_ptr(d_alm), int(adjoint), p, n, _stream_ptr(stream)),
           "cuhpx_analysis_legendre_stage")


def cuhpx_synthesis_legendre_stage(params, d_alm, adjoint, workspace, stream=None) -> None:
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_synthesis_legendre_stage(*params, _dev_ptr(d_alm), int(adjoint), p, n, _stream_ptr(stream)),
           "cuhpx_synthesis_legendre_stage")


def cuhpx_synthesis_fft_stage(params, d_map, d_ring_weights, use_weights, workspace, stream=None) -> None:
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_synthesis_fft_stage(*params, _dev_ptr(d_map), _dev_ptr(d_ring_weights), int(use_weights), p, n,
                                          _stream_ptr(stream)), "cuhpx_synthesis_fft_stage")


def cuhpx_spectra_offset(params) -> int:
    return int(_lib.cuhpx_spectra_offset(*params))


def cuhpx_plan_mcut(params):
    import numpy as np

    out = np.zeros(4 * params[0] - 1, dtype=np.int32)
    _check(_lib.cuhpx_plan_mcut(*params, out.ctypes.data_as(ctypes.c_void_p)), "cuhpx_plan_mcut")
    return out


def cuhpx_plan_stats(params) -> dict:
    """Host-side statistics of the plan for params (see cuhpx.h)."""
    arr = (ctypes.c_double * 8)()
    _check(_lib.cuhpx_plan_stats(*params, arr, 8), "cuhpx_plan_stats")
    keys = ["fft_stage_launches", "legendre_analysis_launches", "legendre_synthesis_launches", "legendre_terms_executed",
            "legendre_terms_full", "spectra_entries", "fft_table_bytes", "workspace_bytes"]
    return dict(zip(keys, [float(v) for v in arr]))


def cuhpx_late_start_stats(params, workspace, stream=None):
    """(analysis, synthesis) Legendre steps of legendre_terms_executed that the late-start tables skip (synchronising)."""
    arr = (ctypes.c_double * 2)()
    p, n = _ws_args(workspace)
    _check(_lib.cuhpx_late_start_stats(*params, p, n, _stream_ptr(stream), arr), "cuhpx_late_start_stats")
    return float(arr[0]), float(arr[1])


def cuhpx_fma_peak_probe(dtype: int, iters: int, stream=None):
    """(milliseconds, FMA instructions executed) of a register-only FMA loop over the whole GPU."""
    ms, cnt = ctypes.c_float(), ctypes.c_double()
    _check(_lib.cuhpx_fma_peak_probe(dtype, iters, ctypes.byref(ms), ctypes.byref(cnt), _stream_ptr(stream)),
           "cuhpx_fma_peak_probe")
    return ms.value, cnt.value


class Transform:
    """Convenience holder of a workspace for fixed (nside, lmax, mmax, batch, dtype): the call a user makes.

    Tensors: maps are real [batch, npix]; alm are complex [batch, nalm] (m-major packed, see cuhpx.h).
    """

    def __init__(self, nside: int, lmax: int, mmax: int | None = None, batch: int = 1,
                 dtype: torch.dtype = torch.float64, device="cuda", ring_weights: torch.Tensor | None = None):
        if not torch.cuda.is_available():
            raise RuntimeError("cuhpx needs a CUDA device (no CPU fallback)")
        mmax = lmax if mmax is None else mmax
        self.nside, self.lmax, self.mmax, self.batch = nside, lmax, mmax, batch
        self.rdtype = dtype
        self.cdtype = torch.complex64 if dtype == torch.float32 else torch.complex128
        self.code = _dtype_code(dtype)
        self.device = torch.device(device)
        self.npix = cuhpx_npix(nside)
        self.nalm = cuhpx_alm_count(lmax, mmax)
        import time

        t0 = time.perf_counter()
        nbytes = cuhpx_workspace_bytes(nside, lmax, mmax, batch, self.code)  # first call for these parameters: host planning
        plan_seconds = time.perf_counter() - t0
        if nbytes == 0:
            raise CuhpxError(CUHPX_EINVAL, "cuhpx_workspace_bytes")
        self.workspace = torch.empty((nbytes + 7) // 8, dtype=torch.int64, device=self.device)
        self.ring_weights = None
        if ring_weights is not None:
            self.ring_weights = ring_weights.to(device=self.device, dtype=torch.float64).contiguous()
        with torch.cuda.device(self.device):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            cuhpx_workspace_init(nside, lmax, mmax, batch, self.code, self.workspace)  # returns when the tables are built
            #: seconds of the table set-up alone (SURVEY 8(a) a0 "first-call time"): host planning (ring classes, cut-offs;
            #: memoised per parameter set, so ~0 from the second Transform on) + cuhpx_workspace_init (uploads, table kernels)
            self.init_seconds = plan_seconds + (time.perf_counter() - t0)

    def _args(self):
        return self.nside, self.lmax, self.mmax, self.batch, self.code

    @property
    def params(self):
        """(nside, lmax, mmax, batch, dtype code): the scalar arguments every C-ABI call takes"""
        return self._args()

    def spectra_view(self) -> torch.Tensor:
        """[batch, nrings, stride] complex view of the ring spectra inside the workspace (stage-level tests)."""
        off = cuhpx_spectra_offset(self.params)
        stride = cuhpx_spectra_stride(self.mmax)
        nr = cuhpx_nrings(self.nside)
        esz = 16 if self.code == CUHPX_F64 else 8
        raw = self.workspace.view(torch.uint8)[off:off + self.batch * nr * stride * esz]
        return raw.view(self.cdtype).view(self.batch, nr, stride)

    def map2alm(self, hmap: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        assert hmap.shape == (self.batch, self.npix) and hmap.dtype == self.rdtype
        alm = torch.empty(self.batch, self.nalm, dtype=self.cdtype, device=self.device) if out is None else out
        cuhpx_map2alm(*self._args(), hmap, alm, self.ring_weights, self.workspace)
        return alm

    def map2alm_iter(self, hmap: torch.Tensor, n_iter: int, out: torch.Tensor | None = None) -> torch.Tensor:
        """Analysis with n_iter refinement iterations a <- a + A (f - S a) (Eq. 4)."""
        assert hmap.shape == (self.batch, self.npix) and hmap.dtype == self.rdtype
        alm = torch.empty(self.batch, self.nalm, dtype=self.cdtype, device=self.device) if out is None else out
        smap = torch.empty_like(hmap) if n_iter > 0 else None
        salm = torch.empty_like(alm) if n_iter > 0 else None
        cuhpx_map2alm_iter(*self._args(), hmap, alm, self.ring_weights, n_iter, smap, salm, self.workspace)
        return alm

    def alm2map(self, alm: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        assert alm.shape == (self.batch, self.nalm) and alm.dtype == self.cdtype
        hmap = torch.empty(self.batch, self.npix, dtype=self.rdtype, device=self.device) if out is None else out
        cuhpx_alm2map(*self._args(), alm, hmap, self.workspace)
        return hmap

    def alm2map_adjoint(self, gmap: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        assert gmap.shape == (self.batch, self.npix) and gmap.dtype == self.rdtype
        galm = torch.empty(self.batch, self.nalm, dtype=self.cdtype, device=self.device) if out is None else out
        cuhpx_alm2map_adjoint(*self._args(), gmap, galm, self.workspace)
        return galm

    def map2alm_adjoint(self, galm: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        assert galm.shape == (self.batch, self.nalm) and galm.dtype == self.cdtype
        gmap = torch.empty(self.batch, self.npix, dtype=self.rdtype, device=self.device) if out is None else out
        cuhpx_map2alm_adjoint(*self._args(), galm, gmap, self.ring_weights, self.workspace)
        return gmap


# ---------------------------------------------------------------- iso-latitude grids
def cuhpx_grid_npix(grid: int, nlat: int, nlon: int) -> int:
    return int(_lib.cuhpx_grid_npix(grid, nlat, nlon))


def cuhpx_grid_ring_info(grid: int, nlat: int, nlon: int, ring: int):
    c, w = ctypes.c_double(), ctypes.c_double()
    _check(_lib.cuhpx_grid_ring_info(grid, nlat, nlon, ring, ctypes.byref(c), ctypes.byref(w)), "cuhpx_grid_ring_info")
    return c.value, w.value


class GridTransform:
    """alm2map / map2alm and their adjoints on a Gauss-Legendre or equiangular grid; argument marshalling only."""

    def __init__(self, grid: int, nlat: int, nlon: int, lmax: int, mmax: int, batch: int, dtype: torch.dtype, device="cuda"):
        self.grid, self.nlat, self.nlon, self.lmax, self.mmax, self.batch = grid, nlat, nlon, lmax, mmax, batch
        self.dtype, self.code = dtype, _dtype_code(dtype)
        self.cdtype = torch.complex128 if dtype == torch.float64 else torch.complex64
        self.device = torch.device(device)
        self.npix = cuhpx_grid_npix(grid, nlat, nlon)
        self.nalm = cuhpx_alm_count(lmax, mmax)
        nbytes = int(_lib.cuhpx_grid_workspace_bytes(grid, nlat, nlon, lmax, mmax, batch, self.code))
        if nbytes == 0 or self.npix == 0:
            raise CuhpxError(1, "cuhpx_grid_workspace_bytes")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            p, n = _ws_args(self.workspace)
            _check(_lib.cuhpx_grid_workspace_init(grid, nlat, nlon, lmax, mmax, batch, self.code, p, n, _stream_ptr(None)),
                   "cuhpx_grid_workspace_init")

    def _a(self):
        return (self.grid, self.nlat, self.nlon, self.lmax, self.mmax, self.batch, self.code)

    def alm2map(self, alm: torch.Tensor) -> torch.Tensor:
        out = torch.empty(self.batch, self.npix, dtype=self.dtype, device=self.device)
        p, n = _ws_args(self.workspace)
        _check(_lib.cuhpx_grid_alm2map(*self._a(), _dev_ptr(alm), _dev_ptr(out), p, n, _stream_ptr(None)), "cuhpx_grid_alm2map")
        return out

    def map2alm(self, hmap: torch.Tensor, ring_weights: torch.Tensor | None = None) -> torch.Tensor:
        out = torch.empty(self.batch, self.nalm, dtype=self.cdtype, device=self.device)
        p, n = _ws_args(self.workspace)
        _check(_lib.cuhpx_grid_map2alm(*self._a(), _dev_ptr(hmap), _dev_ptr(out), _dev_ptr(ring_weights), p, n, _stream_ptr(None)),
               "cuhpx_grid_map2alm")
        return out

    def alm2map_adjoint(self, gmap: torch.Tensor) -> torch.Tensor:
        out = torch.empty(self.batch, self.nalm, dtype=self.cdtype, device=self.device)
        p, n = _ws_args(self.workspace)
        _check(_lib.cuhpx_grid_alm2map_adjoint(*self._a(), _dev_ptr(gmap), _dev_ptr(out), p, n, _stream_ptr(None)),
               "cuhpx_grid_alm2map_adjoint")
        return out

    def map2alm_adjoint(self, galm: torch.Tensor, ring_weights: torch.Tensor | None = None) -> torch.Tensor:
        out = torch.empty(self.batch, self.npix, dtype=self.dtype, device=self.device)
        p, n = _ws_args(self.workspace)
        _check(_lib.cuhpx_grid_map2alm_adjoint(*self._a(), _dev_ptr(galm), _dev_ptr(out), _dev_ptr(ring_weights), p, n,
                                               _stream_ptr(None)), "cuhpx_grid_map2alm_adjoint")
        return out
