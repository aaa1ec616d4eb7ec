"""NESTED <-> RING reordering (paper section III-B).
not gpu: the oracle's centre-matching table is a permutation, obeys the facts HEALPix fixes, and the library's
host index function (integer ring arithmetic, csrc/reorder.cu) reproduces it bit for bit.
gpu: cuhpx_reorder against the oracle, bit-exact, both directions, fp32 / fp64, batches, up to nside 1024."""
import numpy as np
import pytest

from oracle import reorder as oreorder
from paper_2510_01785_b200 import synth


@pytest.mark.parametrize("nside", [1, 2, 4, 8, 32])
def test_oracle_table_is_a_permutation(nside):
    tab = oreorder.nest2ring_table(nside)
    assert np.array_equal(np.sort(tab), np.arange(12 * nside * nside))


def test_oracle_nside1_is_identity():
    # the 12 base pixels: faces 0-3 on ring 1, 4-7 on ring 2 (first at phi = 0), 8-11 on ring 3 -> same numbering
    assert np.array_equal(oreorder.nest2ring_table(1), np.arange(12))


def test_oracle_children_cover_their_parent():
    """Hierarchical subdivision (Fig. 2A): the four NESTED children 4p..4p+3 at 2 nside sit around the
    centre of parent p; child 0 is the southern, 3 the northern, 1 the eastern and 2 the western one
    (x on the even Morton bits -- the reading recorded in DESIGN.md)."""
    for nside in (1, 2, 8):
        zp, pp = oreorder.nested_centres(nside)
        zc, pc = oreorder.nested_centres(2 * nside)
        zc = zc.reshape(-1, 4)
        pc = pc.reshape(-1, 4)
        assert np.all(zc[:, 0] < zp) and np.all(zc[:, 3] > zp)
        assert np.all(np.abs(zc[:, 1] - zc[:, 2]) < 1e-12)
        dphi = np.mod(pc[:, 1] - pc[:, 2] + np.pi, 2 * np.pi) - np.pi
        assert np.all(dphi > 0)  # child 1 is east of child 2
        # and they are close: within one parent pixel (angular size ~ sqrt(4 pi / npix))
        size = np.sqrt(4 * np.pi / (12 * nside * nside))
        assert np.all(np.abs(zc - zp[:, None]) < 1.5 * size)


@pytest.mark.parametrize("nside", [1, 2, 4, 8, 64, 256])
def test_library_host_index_matches_oracle(nside):
    from paper_2510_01785_b200 import binding as B

    tab = oreorder.nest2ring_table(nside)
    npix = 12 * nside * nside
    sel = np.arange(npix) if npix <= 50000 else np.unique((synth.uniform(5, 3, 4000) * npix).astype(np.int64))
    got = np.array([B.cuhpx_nest2ring_index(nside, int(p)) for p in sel])
    assert np.array_equal(got, tab[sel])
    assert B.cuhpx_nest2ring_index(nside, npix) == -1 and B.cuhpx_nest2ring_index(3, 0) == -1


@pytest.mark.gpu
@pytest.mark.parametrize("nside,batch,dtype", [(1, 1, "f64"), (2, 3, "f32"), (4, 1, "f64"), (8, 2, "f32"), (16, 1, "f32"),
                                               (32, 5, "f64"), (64, 2, "f32"), (128, 3, "f64"), (1024, 8, "f32")])
def test_gpu_reorder_bit_exact(nside, batch, dtype):
    import torch

    from paper_2510_01785_b200 import binding as B

    npix = 12 * nside * nside
    tdt = torch.float64 if dtype == "f64" else torch.float32
    src = synth.gaussian_map(900 + nside, nside, batch).astype(np.float64 if dtype == "f64" else np.float32)
    d = torch.from_numpy(src).cuda()
    tab = oreorder.nest2ring_table(nside)
    ring = B.nest2ring(d, nside)
    ref = np.empty_like(src)
    ref[:, tab] = src
    assert np.array_equal(ring.cpu().numpy(), ref)
    nest = B.ring2nest(d, nside)
    assert np.array_equal(nest.cpu().numpy(), src[:, tab])
    assert torch.equal(B.ring2nest(ring, nside), d)
    assert ring.dtype == tdt and npix == ring.shape[1]


@pytest.mark.gpu
def test_gpu_reorder_bad_arguments():
    import torch

    from paper_2510_01785_b200 import binding as B

    a = torch.zeros(1, 48, device="cuda")
    with pytest.raises(B.CuhpxError):
        B.cuhpx_reorder(3, 1, B.CUHPX_F32, B.CUHPX_NEST2RING, a, torch.empty_like(a))
    with pytest.raises(B.CuhpxError):
        B.cuhpx_reorder(2, 1, B.CUHPX_F32, 7, a, torch.empty_like(a))
    with pytest.raises(B.CuhpxError):
        B.cuhpx_reorder(2, 1, B.CUHPX_F32, B.CUHPX_NEST2RING, a, a)
