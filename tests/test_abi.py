"""CPU-side checks of the C-ABI library: it loads, exports what include/cuhpx.h declares, validates
arguments on the host before any launch, and its host helpers agree with the oracle's ring table."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
from paper_2510_01785_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "cuhpx.h")).read()
    body = hdr[hdr.index('extern "C"'):]
    declared = sorted(set(re.findall(r"\b(cuhpx_[a-z0-9_]+)\s*\(", body)))
    assert len(declared) >= 20
    lib = ctypes.CDLL(B.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in cuhpx.h but not exported"
    assert sorted(B.EXPORTS) == declared


def test_host_helpers():
    assert B.cuhpx_npix(32) == 12288 and B.cuhpx_npix(3) == 0 and B.cuhpx_npix(0) == 0
    assert B.cuhpx_nrings(256) == 1023
    assert B.cuhpx_alm_count(64, 64) == 2145 and B.cuhpx_alm_count(8191, 8191) == 33558528
    assert B.cuhpx_alm_count(4, 5) == 0 and B.cuhpx_alm_count(-1, 0) == 0
    for lmax, mmax in [(5, 5), (9, 4)]:
        k = 0
        for m in range(mmax + 1):
            for l in range(m, lmax + 1):
                assert B.cuhpx_alm_index(lmax, l, m) == k == oracle.alm_index(lmax, l, m)
                k += 1
        assert k == B.cuhpx_alm_count(lmax, mmax)
    assert B.cuhpx_spectra_stride(64) == 66 and B.cuhpx_spectra_stride(511) == 512
    assert "EINVAL" in B.status_string(B.CUHPX_EINVAL)


@pytest.mark.parametrize("nside", [1, 2, 16, 1024])
def test_ring_info_matches_oracle_geometry(nside):
    """Two independently written ring tables (library: fp80 host code in plan.cu; oracle: sht_oracle.c)."""
    rings = range(1, 4 * nside) if nside <= 16 else [1, 2, 5, nside - 1, nside, nside + 1, 2 * nside, 3 * nside,
                                                       3 * nside + 1, 4 * nside - 1]
    for ring in rings:
        n, start, c, phi0 = B.cuhpx_ring_info(nside, ring)
        on, ostart, oc, os_, ophi0 = oracle.ring_geometry(nside, ring)
        assert (n, start) == (on, ostart)
        assert abs(c - oc) < 2e-16 and abs(phi0 - ophi0) < 1e-18
    with pytest.raises(B.CuhpxError):
        B.cuhpx_ring_info(nside, 4 * nside)


def test_workspace_bytes_and_argument_validation():
    assert B.cuhpx_workspace_bytes(32, 64, 64, 1, B.CUHPX_F64) > 0
    assert B.cuhpx_workspace_bytes(33, 64, 64, 1, B.CUHPX_F64) == 0
    assert B.cuhpx_workspace_bytes(32, 64, 65, 1, B.CUHPX_F64) == 0
    assert B.cuhpx_workspace_bytes(32, 64, 64, 0, B.CUHPX_F64) == 0
    assert B.cuhpx_workspace_bytes(32, 64, 64, 1, 7) == 0
    big = B.cuhpx_workspace_bytes(4096, 8191, 8191, 1, B.CUHPX_F64)
    assert 2e9 < big < 12e9
    lib = B.lib()
    # argument errors are detected on the host before any launch: these never touch a GPU
    assert lib.cuhpx_workspace_init(3, 4, 4, 1, 1, 256, 1 << 20, None) == B.CUHPX_EINVAL
    assert lib.cuhpx_workspace_init(4, 4, 5, 1, 1, 256, 1 << 20, None) == B.CUHPX_EINVAL
    assert lib.cuhpx_workspace_init(4, 4, 4, 1, 1, None, 1 << 20, None) == B.CUHPX_EINVAL
    assert lib.cuhpx_workspace_init(4, 4, 4, 1, 1, 8, 1 << 20, None) == B.CUHPX_EINVAL  # misaligned
    assert lib.cuhpx_workspace_init(4, 4, 4, 1, 1, 256, 16, None) == B.CUHPX_EWORKSPACE  # too small
    # workspace too small -> EWORKSPACE; bad scalars / null / overlapping pointers -> EINVAL
    assert lib.cuhpx_map2alm(4, 4, 4, 1, 1, 256, 1 << 21, None, 1 << 22, 64, None) == B.CUHPX_EWORKSPACE
    assert lib.cuhpx_map2alm(5, 4, 4, 1, 1, 256, 512, None, 1024, 1 << 20, None) == B.CUHPX_EINVAL
    assert lib.cuhpx_alm2map(4, 4, 4, 1, 1, None, 512, 1024, 1 << 20, None) == B.CUHPX_EINVAL
    assert lib.cuhpx_alm2map(4, 4, 4, 1, 1, 512, 512, 1 << 22, 1 << 20, None) == B.CUHPX_EINVAL
    assert lib.cuhpx_alm2map(4, 4, 4, 1, 1, 512, 512 + 16, 1 << 22, 1 << 20, None) == B.CUHPX_EINVAL  # partial overlap
    assert lib.cuhpx_alm2map(4, 4, 4, 1, 1, 512, 1 << 22, 1 << 22, 1 << 20, None) == B.CUHPX_EINVAL  # output inside workspace
    assert lib.cuhpx_alm2map_adjoint(4, 4, 4, 1, 1, 256, 520, 1024, 1 << 20, None) == B.CUHPX_EINVAL
    assert lib.cuhpx_map2alm_adjoint(4, 4, 4, 1, 2, 256, 512, None, 1024, 1 << 20, None) == B.CUHPX_EINVAL
    assert lib.cuhpx_analysis_fft_stage(4, 4, 4, 1, 1, 256, None, 0, 1 << 22, 64, None) == B.CUHPX_EWORKSPACE
    assert lib.cuhpx_workspace_bytes(4, 4, 4, 65536, 1) == 0  # channels index a grid dimension
    assert B.cuhpx_spectra_offset((4, 4, 4, 1, 1)) > 0 and B.cuhpx_spectra_offset((3, 4, 4, 1, 1)) == 0
    assert len(B.cuhpx_plan_mcut((4, 8, 8, 1, 1))) == 15
    st = B.cuhpx_plan_stats((32, 64, 64, 1, 1))
    assert st["legendre_terms_full"] == 2145 * 64 and 0 < st["legendre_terms_executed"] <= st["legendre_terms_full"]


def test_measurement_probes_compile_for_sm100a():
    """csrc/tcgen05_probe.cu and csrc/dfma_probe.cu (profiles/r2_tcgen05_probe.md, r2_dfma_probe.md) are measurement tools
    outside the library; they must keep building with the library's toolchain (nvcc cross-compiles without a GPU)."""
    import shutil

    from paper_2510_01785_b200 import build as builder

    if shutil.which(os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")) is None:
        pytest.skip("nvcc not available")
    for exe in builder.build_probe():
        assert os.path.getsize(exe) > 0
