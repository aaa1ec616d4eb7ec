"""cuhpx_ring_weights_noalloc (csrc/noalloc.cu): the ring-weight solver with its scratch in the library's built-in device
array instead of a caller-owned workspace.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL64 = 1e-11  # the fp64 bar of tests/test_gpu_parity.py: max |d| / max |ref|


def _existing_path(B, nside, lmax_w):
    return B.ring_weights(nside, lmax_w, "cuda:0")


def test_noalloc_matches_existing_path_on_two_calls_in_a_row():
    from paper_2510_01785_b200 import binding as B

    torch.cuda.set_device(0)
    # two calls in a row that need different tables and leave different contents in the shared array, then the first again
    cases = [(64, 0), (32, 50), (64, 0)]
    for k, (nside, lmax_w) in enumerate(cases):
        ref = _existing_path(B, nside, lmax_w).cpu().numpy()
        w = torch.full((4 * nside - 1,), float("nan"), dtype=torch.float64, device="cuda:0")
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info(0)[0]
        B.cuhpx_ring_weights_noalloc(nside, lmax_w, w)
        torch.cuda.synchronize()
        if k == 2:  # every kernel of this case is loaded by now: the device's free memory must not have moved
            assert torch.cuda.mem_get_info(0)[0] == free_before
        got = w.cpu().numpy()
        assert np.all(np.isfinite(got))
        err = float(np.abs(got - ref).max() / np.abs(ref).max())
        assert err <= TOL64, f"nside {nside}, lmax_w {lmax_w}: {err:.3e} > {TOL64}"


def test_noalloc_repeated_call_is_bitwise_stable_and_limit_is_enforced():
    from paper_2510_01785_b200 import binding as B

    torch.cuda.set_device(0)
    nside = 128
    a = torch.empty(4 * nside - 1, dtype=torch.float64, device="cuda:0")
    b = torch.empty_like(a)
    B.cuhpx_ring_weights_noalloc(nside, 0, a)
    B.cuhpx_ring_weights_noalloc(nside, 0, b)  # the array still holds the first call's tables, spectra and vectors
    assert torch.equal(a, b)
    ref = _existing_path(B, nside, 0)
    assert float((a - ref).abs().max() / ref.abs().max()) <= TOL64
    # beyond the built-in scratch: refused with CUHPX_EWORKSPACE, nothing written
    big = 1024
    assert B.cuhpx_ring_weights_workspace_bytes(big, 0) > B.CUHPX_NOALLOC_SCRATCH_BYTES
    w = torch.full((4 * big - 1,), -1.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(B.CuhpxError) as ei:
        B.cuhpx_ring_weights_noalloc(big, 0, w)
    assert ei.value.status == B.CUHPX_EWORKSPACE
    assert bool((w == -1.0).all())
    with pytest.raises(B.CuhpxError) as ei:
        B.cuhpx_ring_weights_noalloc(3, 0, w)  # not a power of two
    assert ei.value.status == B.CUHPX_EINVAL
