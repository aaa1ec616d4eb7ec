"""Spectral resampling: truncating / extending a_lm, and a map moved between two nside
through it.  not gpu: the oracle's index bookkeeping against synth.alm_lm; gpu: bit-exact parity of cuhpx_alm_resize and
the resampled map against the oracle pipeline."""
import numpy as np
import pytest

import oracle
from oracle import reorder as oreorder
from paper_2510_01785_b200 import synth


@pytest.mark.parametrize("li,mi,lo,mo", [(8, 8, 12, 12), (12, 12, 8, 8), (10, 6, 7, 7), (5, 5, 9, 3), (0, 0, 3, 3)])
def test_oracle_resize_keeps_exactly_the_shared_coefficients(li, mi, lo, mo):
    a = synth.white_alm(3, li, mi)[0]
    out = oreorder.alm_resize(a, li, mi, lo, mo)
    lin, min_ = synth.alm_lm(li, mi)
    lout, mout = synth.alm_lm(lo, mo)
    src = {(int(l), int(m)): a[k] for k, (l, m) in enumerate(zip(lin, min_))}
    for k, (l, m) in enumerate(zip(lout, mout)):
        assert out[k] == src.get((int(l), int(m)), 0.0)
    # truncation after extension is the identity
    assert np.array_equal(oreorder.alm_resize(oreorder.alm_resize(a, li, mi, li + 5, li + 5), li + 5, li + 5, li, mi), a)


@pytest.mark.gpu
@pytest.mark.parametrize("li,mi,lo,mo,batch,dtype", [(8, 8, 12, 12, 1, "f64"), (40, 33, 17, 17, 3, "f32"), (64, 64, 200, 150, 2, "f64"),
                                                     (0, 0, 5, 5, 1, "f32"), (300, 300, 128, 100, 4, "f32")])
def test_gpu_alm_resize_bit_exact(li, mi, lo, mo, batch, dtype):
    import torch

    from paper_2510_01785_b200 import binding as B

    a = synth.white_alm(9, li, mi, batch).astype(np.complex128 if dtype == "f64" else np.complex64)
    got = B.alm_resize(torch.from_numpy(a).cuda(), li, mi, lo, mo).cpu().numpy()
    assert np.array_equal(got, oreorder.alm_resize(a, li, mi, lo, mo))


@pytest.mark.gpu
def test_gpu_upsampled_map_matches_oracle_pipeline():
    """nside 16 -> 32: analyse at lmax 32, extend to lmax 64, synthesise on the finer grid (Fig. 11 in small)."""
    import torch

    from paper_2510_01785_b200 import binding as B

    f = synth.gaussian_map(41, 16, 1)
    Ta = B.Transform(16, 32, 32, 1, torch.float64, "cuda:0")
    Tb = B.Transform(32, 64, 64, 1, torch.float64, "cuda:0")
    got = Tb.alm2map(B.alm_resize(Ta.map2alm(torch.from_numpy(f).cuda()), 32, 32, 64, 64)).cpu().numpy()[0]
    ref = oracle.alm2map(32, 64, 64, oreorder.alm_resize(oracle.map2alm(16, 32, 32, f[0]), 32, 32, 64, 64))
    assert np.abs(got - ref).max() / np.abs(ref).max() <= 1e-11
