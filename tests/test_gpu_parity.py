"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances are north_star's: fp64 max|d|/max|ref| <= 1e-11, fp32 relative L2 <= 2e-5."""
import numpy as np
import pytest

import oracle
from paper_2510_01785_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL64 = 1e-11
TOL32 = 2e-5


def _binding():
    from paper_2510_01785_b200 import binding

    return binding


def err64(got, ref):
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def err32(got, ref):
    return float(np.linalg.norm((got - ref).ravel()) / np.linalg.norm(ref.ravel()))


def check(got, ref, dtype):
    if dtype == "f64":
        e = err64(got, ref)
        assert e <= TOL64, f"fp64 max-norm relative error {e:.3e} > {TOL64}"
    else:
        e = err32(got, ref)
        assert e <= TOL32, f"fp32 relative L2 error {e:.3e} > {TOL32}"
    return e


def make_transform(nside, lmax, mmax, batch, dtype, weights=None):
    B = _binding()
    tdt = torch.float64 if dtype == "f64" else torch.float32
    w = None if weights is None else torch.from_numpy(weights)
    return B.Transform(nside, lmax, mmax, batch, tdt, "cuda:0", ring_weights=w)


def to_dev(a, dtype, complex_=False):
    if complex_:
        t = torch.from_numpy(np.ascontiguousarray(a)).to(torch.complex128 if dtype == "f64" else torch.complex64)
    else:
        t = torch.from_numpy(np.ascontiguousarray(a)).to(torch.float64 if dtype == "f64" else torch.float32)
    return t.cuda()


def rounded(a, dtype, complex_=False):
    """What the oracle sees: the inputs after their one rounding to the transform's dtype."""
    if dtype == "f64":
        return a
    return a.astype(np.complex64).astype(np.complex128) if complex_ else a.astype(np.float32).astype(np.float64)


def run_all_four(nside, lmax, mmax, batch, dtype, seed, weights=None, channels_checked=None):
    """All four operators against the full oracle; returns the four error figures."""
    T = make_transform(nside, lmax, mmax, batch, dtype, weights)
    fmap = synth.gaussian_map(seed, nside, batch)
    alm = synth.powerlaw_alm(seed, lmax, mmax, batch)
    galm = synth.white_alm(seed, lmax, mmax, batch)
    chans = range(batch) if channels_checked is None else channels_checked
    out = {}

    got = T.map2alm(to_dev(fmap, dtype)).cpu().numpy().astype(np.complex128)
    ref = np.stack([oracle.map2alm(nside, lmax, mmax, rounded(fmap[c], dtype), weights) for c in chans])
    out["map2alm"] = check(got[list(chans)], ref, dtype)
    assert np.all(got[:, : lmax + 1].imag == 0.0), "Im a_l0 must be exactly zero"

    got = T.alm2map(to_dev(alm, dtype, True)).cpu().numpy().astype(np.float64)
    ref = np.stack([oracle.alm2map(nside, lmax, mmax, rounded(alm[c], dtype, True)) for c in chans])
    out["alm2map"] = check(got[list(chans)], ref, dtype)

    got = T.alm2map_adjoint(to_dev(fmap, dtype)).cpu().numpy().astype(np.complex128)
    ref = np.stack([oracle.alm2map_adjoint(nside, lmax, mmax, rounded(fmap[c], dtype)) for c in chans])
    out["alm2map_adjoint"] = check(got[list(chans)], ref, dtype)

    got = T.map2alm_adjoint(to_dev(galm, dtype, True)).cpu().numpy().astype(np.float64)
    ref = np.stack([oracle.map2alm_adjoint(nside, lmax, mmax, rounded(galm[c], dtype, True), weights) for c in chans])
    out["map2alm_adjoint"] = check(got[list(chans)], ref, dtype)
    return out


# ----------------------------------------------------------------------------- BASELINE configs 1-3

def test_cfg1_all_four_fp64():
    """configs[0]: nside 32, lmax = mmax = 64 (= equatorial Nyquist), batch 1, fp64; full oracle."""
    errs = run_all_four(32, 64, 64, 1, "f64", 101)
    print("cfg1", errs)


def test_cfg1_weighted_fp64():
    """Same with non-uniform, non-symmetric ring weights."""
    errs = run_all_four(32, 64, 64, 1, "f64", 101, weights=synth.ring_weights(101, 32))
    print("cfg1 weighted", errs)


def test_cfg2_both_directions_fp64():
    """configs[1]: nside 256, lmax = mmax = 511: alm -> map (both sides), then analysis of the ORACLE's map on
    both sides, plus the adjoint dot-product identities on the GPU results."""
    nside, lmax = 256, 511
    T = make_transform(nside, lmax, lmax, 1, "f64")
    alm = synth.powerlaw_alm(202, lmax, lmax, 1)
    ref_map = oracle.alm2map(nside, lmax, lmax, alm[0])
    got_map = T.alm2map(to_dev(alm, "f64", True)).cpu().numpy()[0]
    check(got_map, ref_map, "f64")
    ref_alm = oracle.map2alm(nside, lmax, lmax, ref_map)
    got_alm = T.map2alm(to_dev(ref_map[None], "f64")).cpu().numpy()[0]
    check(got_alm, ref_alm, "f64")
    # adjoint dot products with fresh cotangents
    g = synth.gaussian_map(203, nside, 1)
    b = synth.white_alm(204, lmax, lmax, 1)
    b[:, : lmax + 1] = b[:, : lmax + 1].real
    a = alm.copy()
    st_g = T.alm2map_adjoint(to_dev(g, "f64")).cpu().numpy()[0]
    lhs = float(got_map @ g[0])
    rhs = float((a[0].real * st_g.real + a[0].imag * st_g.imag).sum())
    assert abs(lhs - rhs) <= 1e-11 * max(abs(lhs), 1.0)
    at_b = T.map2alm_adjoint(to_dev(b, "f64", True)).cpu().numpy()[0]
    lhs = float((got_alm.real * b[0].real + got_alm.imag * b[0].imag).sum())
    rhs = float(ref_map @ at_b)
    assert abs(lhs - rhs) <= 1e-11 * max(abs(lhs), 1.0)
    check(st_g, oracle.alm2map_adjoint(nside, lmax, lmax, g[0]), "f64")
    check(at_b, oracle.map2alm_adjoint(nside, lmax, lmax, b[0]), "f64")


def test_cfg3_batched_fp32_training_step():
    """configs[2]: nside 64, lmax = mmax = 128, 256 channels fp32: map2alm forward then map2alm_adjoint backward
    with random upstream alm gradients; full oracle on every channel."""
    nside, lmax, batch = 64, 128, 256
    T = make_transform(nside, lmax, lmax, batch, "f32")
    fmap = synth.gaussian_map(303, nside, batch)
    galm = synth.white_alm(303, lmax, lmax, batch)
    got = T.map2alm(to_dev(fmap, "f32")).cpu().numpy().astype(np.complex128)
    ref = np.stack([oracle.map2alm(nside, lmax, lmax, rounded(fmap[c], "f32")) for c in range(batch)])
    e1 = check(got, ref, "f32")
    for c in (0, 17, 255):  # per-channel too: no channel hides behind the others
        check(got[c], ref[c], "f32")
    got = T.map2alm_adjoint(to_dev(galm, "f32", True)).cpu().numpy().astype(np.float64)
    ref = np.stack([oracle.map2alm_adjoint(nside, lmax, lmax, rounded(galm[c], "f32", True)) for c in range(batch)])
    e2 = check(got, ref, "f32")
    print("cfg3", e1, e2)


# ----------------------------------------------------------------------------- small, ragged and degenerate cases

@pytest.mark.parametrize("nside,lmax,batch,dtype,n_iter,weighted", [(32, 64, 1, "f64", 3, False), (16, 40, 3, "f64", 2, True),
                                                                    (64, 128, 4, "f32", 2, False), (8, 16, 1, "f64", 0, False)])
def test_map2alm_iter_matches_oracle(nside, lmax, batch, dtype, n_iter, weighted):
    """Iterative refinement (Eq. 4) through cuhpx_map2alm_iter against the oracle's step-by-step loop."""
    w = synth.ring_weights(77, nside) if weighted else None
    T = make_transform(nside, lmax, lmax, batch, dtype, w)
    fmap = synth.gaussian_map(70 + nside, nside, batch)
    got = T.map2alm_iter(to_dev(fmap, dtype), n_iter).cpu().numpy().astype(np.complex128)
    ref = np.stack([oracle.map2alm_iter(nside, lmax, lmax, rounded(fmap[c], dtype), n_iter, w) for c in range(batch)])
    check(got, ref, dtype)
    assert np.all(got[:, : lmax + 1].imag == 0.0)
    if n_iter == 0:
        assert np.array_equal(got, T.map2alm(to_dev(fmap, dtype)).cpu().numpy())


@pytest.mark.parametrize("nside,lmax,mmax,batch,dtype", [
    (1, 0, 0, 1, "f64"), (1, 3, 3, 1, "f64"), (2, 8, 8, 2, "f64"), (4, 16, 16, 1, "f64"), (4, 11, 7, 3, "f64"),
    (8, 16, 0, 1, "f64"), (16, 40, 33, 1, "f64"), (16, 47, 47, 5, "f32"), (8, 23, 23, 1, "f32"),
    (64, 200, 150, 2, "f64"), (32, 95, 95, 7, "f32"), (128, 300, 300, 1, "f64"),
    # kernel-selection corners: channel-blocked direct sums in fp64; 32-degree contraction with several ring chunks and
    # the combine kernel; 64-degree contraction accumulating in place over ring chunks with mmax < lmax and a ragged
    # channel group; packed-FMA synthesis with two channel groups, the second ragged (both CTA shapes)
    (32, 64, 64, 5, "f64"), (256, 300, 300, 6, "f32"), (256, 600, 450, 6, "f32"), (64, 128, 128, 11, "f32"),
    (128, 520, 520, 9, "f32"),
    # fp32 with few channels at sizes where the exponent-scaled seeds matter (sc < 0 on polar rings) and the
    # analysis walks several ring chunks: legendre_analysis_kernel<float, 1 / 4>, legendre_synthesis_kernel<float, 1 / 4>
    (256, 600, 600, 1, "f32"), (512, 700, 700, 4, "f32"),
    # tensor-core synthesis (batch >= 8): 16-channel groups with a ragged second group and mmax < lmax; a last stage of
    # one degree (lmax - m + 1 = 1 mod 32); more than one 128-ring tile per order with late-starting polar rings
    (32, 64, 40, 20, "f32"), (16, 32, 32, 8, "f32"), (128, 300, 300, 8, "f32"),
])
def test_small_and_ragged_cases(nside, lmax, mmax, batch, dtype):
    """mmax < lmax, lmax far above 2 nside (every polar ring aliases), batch not a multiple of the channel
    tile, lmax not a multiple of any l tile, single-coefficient transforms (lmax = 0)."""
    w = synth.ring_weights(7, nside) if (nside + batch) % 2 == 0 else None
    run_all_four(nside, lmax, mmax, batch, dtype, 1000 + nside + lmax, weights=w)


def test_fft_stage_alone_matches_ring_dft():
    """Stage-level parity: spectra written by the analysis FFT stage against the oracle's
    direct ring DFT, ring by ring, for every m the stage is required to produce."""
    B = _binding()
    nside, lmax = 16, 40
    T = make_transform(nside, lmax, lmax, 2, "f64")
    fmap = synth.gaussian_map(55, nside, 2)
    B.cuhpx_analysis_fft_stage(T.params, to_dev(fmap, "f64"), None, 0, T.workspace)
    torch.cuda.synchronize()
    mcut = B.cuhpx_plan_mcut(T.params)
    nrings = 4 * nside - 1
    spec = T.spectra_view().cpu().numpy()
    for ring in range(1, nrings + 1):
        n, start = oracle.ring_geometry(nside, ring)[:2]
        assert mcut[ring - 1] >= min(lmax, 2)  # low orders are needed on every ring
        for c in range(2):
            ref = oracle.ring_dft(nside, ring, fmap[c, start:start + n], lmax)
            mc = mcut[ring - 1]
            np.testing.assert_allclose(spec[c, ring - 1, : mc + 1], ref[: mc + 1], atol=1e-12 * n)


def test_outputs_are_overwritten_and_inputs_untouched():
    nside, lmax = 8, 16
    T = make_transform(nside, lmax, lmax, 1, "f64")
    fmap = to_dev(synth.gaussian_map(1, nside, 1), "f64")
    keep = fmap.clone()
    out = torch.full((1, T.nalm), 7.0 + 3.0j, dtype=torch.complex128, device="cuda")
    a1 = T.map2alm(fmap, out=out).clone()
    a2 = T.map2alm(fmap, out=out).clone()
    assert torch.equal(fmap, keep) and torch.equal(a1, a2)
    m1 = T.alm2map(a1, out=torch.full((1, T.npix), 5.0, dtype=torch.float64, device="cuda"))
    m2 = T.alm2map(a1)
    assert torch.equal(m1, m2)


def test_stream_ordering_and_error_codes():
    B = _binding()
    nside, lmax = 8, 16
    T = make_transform(nside, lmax, lmax, 1, "f64")
    fmap = to_dev(synth.gaussian_map(2, nside, 1), "f64")
    s = torch.cuda.Stream()
    ref = T.map2alm(fmap)
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        got = T.map2alm(fmap)
    s.synchronize()
    assert torch.equal(ref, got)
    # A workspace initialised for other parameters: the library keeps no per-workspace state, so the host cannot
    # know; every kernel checks the header, the call leaves the output untouched and marks the workspace, and
    # cuhpx_workspace_check (synchronising) reports it.  Overlapping buffers are refused on the host.
    B.cuhpx_workspace_check(*T.params, T.workspace)
    big = torch.empty(B.cuhpx_workspace_bytes(nside, lmax + 8, lmax + 8, 1, B.CUHPX_F64) // 8 + 64, dtype=torch.int64, device="cuda")
    big[: T.workspace.numel()] = T.workspace  # a moved copy of an initialised workspace works as is
    got2 = torch.empty_like(ref)
    B.cuhpx_map2alm(*T.params, fmap, got2, None, big[: T.workspace.numel()])
    assert torch.equal(ref, got2)
    nalm2 = B.cuhpx_alm_count(lmax + 8, lmax + 8)
    alm = torch.full((1, nalm2), 7.0 + 1.0j, dtype=torch.complex128, device="cuda")
    B.cuhpx_map2alm(nside, lmax + 8, lmax + 8, 1, B.CUHPX_F64, fmap, alm, None, big)  # header says (lmax, lmax)
    torch.cuda.synchronize()
    assert torch.all(alm == 7.0 + 1.0j), "a kernel trusted a workspace built for other parameters"
    with pytest.raises(B.CuhpxError) as ei:
        B.cuhpx_workspace_check(nside, lmax + 8, lmax + 8, 1, B.CUHPX_F64, big)
    assert ei.value.status == B.CUHPX_EWORKSPACE
    with pytest.raises(B.CuhpxError) as ei:  # too small for the parameters of the call
        B.cuhpx_map2alm(nside, lmax + 8, lmax + 8, 1, B.CUHPX_F64, fmap, alm, None, T.workspace)
    assert ei.value.status == B.CUHPX_EWORKSPACE
    both = torch.empty(T.npix + 2 * T.nalm, dtype=torch.float64, device="cuda")
    with pytest.raises(B.CuhpxError) as ei:  # partial overlap of input and output
        B.cuhpx_map2alm(*T.params, both[: T.npix].view(1, -1), both[T.npix - 2: T.npix - 2 + 2 * T.nalm].view(torch.complex128).view(1, -1),
                        None, T.workspace)
    assert ei.value.status == B.CUHPX_EINVAL


# ----------------------------------------------------------------------------- FFT stage at full ring sizes

def _spectra_view(B, T, batch, nside, mmax, dtype):
    return T.spectra_view()


def _class_rings(nside):
    """Rings hitting every FFT kernel family and size class present at this nside, both hemispheres."""
    picks = {1, 2, 3, 16, 63, 64, 65, 96, 127, 128, 129, 200, 255, 256, 257, 300, 511, 512, 513, 700, 1000, 1023, 1024,
             1025, 1500, 2047, 2048, 2049, 3000, 4095, 4096, 4097, 5000}
    rings = sorted(r for r in picks if r <= 2 * nside)
    rings += [nside - 1, nside, nside + 1, 2 * nside, 3 * nside, 4 * nside - 1, 4 * nside - 70, 4 * nside - 1030]
    return sorted(set(r for r in rings if 1 <= r <= 4 * nside - 1))


@pytest.mark.parametrize("nside,lmax,dtype", [(512, 1200, "f64"), (1024, 2047, "f32"), (2048, 4095, "f64"),
                                                (4096, 8191, "f64"), (4096, 8191, "f32")])
def test_fft_stages_every_size_class(nside, lmax, dtype):
    """a1 and s2 alone at full ring sizes against the oracle's direct ring sums, for rings from every
    kernel family (direct / pow2 / chirp-z) and every block-FFT size (2^8 .. 2^13), incl. the m > N/2 fold."""
    B = _binding()
    T = make_transform(nside, lmax, lmax, 1, dtype)
    mcut = B.cuhpx_plan_mcut(T.params)
    rings = _class_rings(nside)
    npix = 12 * nside * nside
    fmap = np.zeros(npix)
    for r in rings:
        n, start = oracle.ring_geometry(nside, r)[:2]
        fmap[start:start + n] = synth.normal(900 + nside, r, n)
    fmap_r = rounded(fmap, dtype)
    B.cuhpx_analysis_fft_stage(T.params, to_dev(fmap[None], dtype), None, 0, T.workspace)
    torch.cuda.synchronize()
    spec = _spectra_view(B, T, 1, nside, lmax, dtype)
    tol = 1e-12 if dtype == "f64" else 3e-6
    for r in rings:
        n, start = oracle.ring_geometry(nside, r)[:2]
        mc = int(mcut[r - 1])
        ref = oracle.ring_dft(nside, r, fmap_r[start:start + n], mc)
        got = spec[0, r - 1, : mc + 1].cpu().numpy().astype(np.complex128)
        err = np.abs(got - ref).max() / np.abs(ref).max()
        assert err < tol, f"analysis FFT stage ring {r} (N={n}, mcut={mc}): {err:.3e}"
    # synthesis: fill the spectra rows of the picked rings, run s2 alone
    spec.zero_()
    Gs = {}
    for r in rings:
        mc = int(mcut[r - 1])
        G = synth.white_alm(901 + nside, mc + 5, 0, 1, tag=r)[0][: mc + 1].copy()
        G[0] = G[0].real
        G = rounded(G, dtype, True)
        Gs[r] = G
        spec[0, r - 1, : mc + 1] = torch.from_numpy(G).to(spec.dtype).cuda()
    out = torch.empty(1, npix, dtype=torch.float64 if dtype == "f64" else torch.float32, device="cuda")
    B.cuhpx_synthesis_fft_stage(T.params, out, None, 0, T.workspace)
    torch.cuda.synchronize()
    out = out.cpu().numpy().astype(np.float64)[0]
    for r in rings:
        n, start = oracle.ring_geometry(nside, r)[:2]
        ref = oracle.ring_synth(nside, r, Gs[r])
        err = np.abs(out[start:start + n] - ref).max() / np.abs(ref).max()
        assert err < tol, f"synthesis FFT stage ring {r} (N={n}): {err:.3e}"


# ----------------------------------------------------------------------------- BASELINE configs 4 and 5 (subset oracle)

def _subset_lm(seed, lmax, mmax, n_m, per_m):
    """Seeded (l, m) sample: mandated corner cases plus n_m random orders with per_m degrees each."""
    u = synth.uniform(seed, 77, n_m * (per_m + 1))
    sel = {(0, 0), (lmax, 0), (lmax, mmax), (lmax, mmax - 1), (mmax, mmax), (lmax - 1, 5), (lmax, 7), (17, 6)}
    ms = sorted(set(int(x * (mmax + 1)) for x in u[:n_m]))
    k = n_m
    for m in ms:
        for _ in range(per_m):
            sel.add((m + int(u[k] * (lmax - m + 1)), m))
            k += 1
    sel = sorted(sel, key=lambda t: (t[1], t[0]))
    return [s[0] for s in sel], [s[1] for s in sel]


def _subset_rings(seed, nside, count):
    u = synth.uniform(seed, 78, count)
    rings = {1, 2, 3, nside - 1, nside, nside + 1, 2 * nside, 2 * nside + 1, 4 * nside - 1, 4 * nside - 5, 3 * nside + 7,
             nside // 2 + 1, 3 * nside // 4 + 3, 97}
    rings |= set(1 + int(x * (4 * nside - 1)) for x in u)
    return sorted(r for r in rings if 1 <= r <= 4 * nside - 1)


def _ring_slices(nside, rings):
    return [slice(s, s + n) for n, s in (oracle.ring_geometry(nside, r)[:2] for r in rings)]


@pytest.mark.slow
def test_cfg4_nside1024_fp32_batch8():
    """configs[3]: nside 1024, lmax = mmax = 2047, 8 channels fp32; alm -> alm2map + 0.01 noise -> map2alm; adjoints.
    Oracle: seeded subset (256+ coefficients, 40+ rings) on channels 0 and 7 (full oracle = hours of x87 work)."""
    nside, lmax, batch = 1024, 2047, 8
    T = make_transform(nside, lmax, lmax, batch, "f32")
    alm = synth.powerlaw_alm(404, lmax, lmax, batch)
    rings = _subset_rings(404, nside, 32)
    sl, sm = _subset_lm(404, lmax, lmax, 32, 8)
    sl_idx = [oracle.alm_index(lmax, l, m) for l, m in zip(sl, sm)]
    slices = _ring_slices(nside, rings)
    gmap = T.alm2map(to_dev(alm, "f32", True))
    got_map = gmap.cpu().numpy().astype(np.float64)
    noisy = got_map + 0.01 * synth.gaussian_map(405, nside, batch)
    noisy32 = noisy.astype(np.float32)
    galm = T.map2alm(torch.from_numpy(noisy32).cuda()).cpu().numpy().astype(np.complex128)
    gst = T.alm2map_adjoint(torch.from_numpy(noisy32).cuda()).cpu().numpy().astype(np.complex128)
    cot = synth.white_alm(406, lmax, lmax, batch)
    gat = T.map2alm_adjoint(to_dev(cot, "f32", True)).cpu().numpy().astype(np.float64)
    for c in (0, 7):
        a_in = rounded(alm[c], "f32", True)
        ref = oracle.alm2map_rings(nside, lmax, lmax, a_in, rings)
        got = np.concatenate([got_map[c][s] for s in slices])
        assert err32(got, ref) <= TOL32
        f_in = noisy32[c].astype(np.float64)
        ref = oracle.map2alm_subset(nside, lmax, lmax, f_in, sl, sm)
        assert err32(galm[c][sl_idx], ref) <= TOL32
        # per coefficient: nothing hides in the norm (the largest coefficients dominate it)
        assert np.abs(galm[c][sl_idx] - ref).max() <= 2e-5 * np.abs(galm[c]).max()
        ref = oracle.alm2map_adjoint_subset(nside, lmax, lmax, f_in, sl, sm)
        assert err32(gst[c][sl_idx], ref) <= TOL32
        ref = oracle.map2alm_adjoint_rings(nside, lmax, lmax, rounded(cot[c], "f32", True), rings)
        got = np.concatenate([gat[c][s] for s in slices])
        assert err32(got, ref) <= TOL32


@pytest.mark.slow
@pytest.mark.parametrize("batch", [1, 3])
def test_nside1024_fp32_few_channels(batch):
    """A single fp32 map (and three) at nside 1024, lmax = mmax = 2047: the default user configuration runs the
    few-channel fp32 kernels (multi-chunk analysis, exponent-scaled seeds), which configs[3] (batch 8) never reaches.
    Oracle: seeded subset on the first and last channel."""
    nside, lmax = 1024, 2047
    T = make_transform(nside, lmax, lmax, batch, "f32")
    alm = synth.powerlaw_alm(414, lmax, lmax, batch)
    rings = _subset_rings(414, nside, 20)
    sl, sm = _subset_lm(414, lmax, lmax, 24, 6)
    sl_idx = [oracle.alm_index(lmax, l, m) for l, m in zip(sl, sm)]
    slices = _ring_slices(nside, rings)
    got_map = T.alm2map(to_dev(alm, "f32", True)).cpu().numpy()
    galm = T.map2alm(torch.from_numpy(got_map).cuda()).cpu().numpy().astype(np.complex128)
    for c in sorted({0, batch - 1}):
        ref = oracle.alm2map_rings(nside, lmax, lmax, rounded(alm[c], "f32", True), rings)
        got = np.concatenate([got_map[c].astype(np.float64)[s] for s in slices])
        assert err32(got, ref) <= TOL32
        ref = oracle.map2alm_subset(nside, lmax, lmax, got_map[c].astype(np.float64), sl, sm)
        assert err32(galm[c][sl_idx], ref) <= TOL32
        assert np.abs(galm[c][sl_idx] - ref).max() <= 2e-5 * np.abs(ref).max()


@pytest.mark.slow
@pytest.mark.parametrize("nside,lmax,mmax,seed", [(4096, 8191, 8191, 505), (2048, 4095, 4095, 506), (2048, 5000, 3777, 507)],
                         ids=["cfg5", "nside2048", "nside2048-ragged"])
def test_cfg5_nside4096_fp64(nside, lmax, mmax, seed):
    """configs[4]: nside 4096, lmax = mmax = 8191, fp64: alm -> alm2map -> map2alm.  Oracle checked on a seeded
    subset of 512+ (l, m) and 64+ rings; the analysis is checked on the GPU's own map so both
    sides see identical input.  The nside 2048 cases run the same late-start Legendre kernels with other chunk counts,
    lmax > 2 nside and mmax < lmax."""
    T = make_transform(nside, lmax, mmax, 1, "f64")
    alm = synth.powerlaw_alm(seed, lmax, mmax, 1)
    rings = _subset_rings(seed, nside, 60)
    sl, sm = _subset_lm(seed, lmax, mmax, 60, 9)
    assert len(sl) >= 512 and len(rings) >= 64
    sl_idx = [oracle.alm_index(lmax, l, m) for l, m in zip(sl, sm)]
    slices = _ring_slices(nside, rings)
    dmap = T.alm2map(to_dev(alm, "f64", True))
    got_map = dmap.cpu().numpy()[0]
    ref = oracle.alm2map_rings(nside, lmax, mmax, alm[0], rings)
    got = np.concatenate([got_map[s] for s in slices])
    e_syn = np.abs(got - ref).max() / np.abs(ref).max()  # oracle-side maximum (of the sampled rings)
    assert e_syn <= TOL64, f"alm2map {e_syn:.3e}"
    galm = T.map2alm(dmap).cpu().numpy()[0]
    ref = oracle.map2alm_subset(nside, lmax, mmax, got_map, sl, sm)
    e_ana = np.abs(galm[sl_idx] - ref).max() / np.abs(ref).max()  # the sample holds (0, 0), the largest coefficient
    assert e_ana <= TOL64, f"map2alm {e_ana:.3e}"
    assert np.all(galm[: lmax + 1].imag == 0.0)
    # adjoints on the same subset
    gst = T.alm2map_adjoint(dmap).cpu().numpy()[0]
    ref = oracle.alm2map_adjoint_subset(nside, lmax, mmax, got_map, sl, sm)
    e_st = np.abs(gst[sl_idx] - ref).max() / np.abs(ref).max()
    assert e_st <= TOL64, f"alm2map_adjoint {e_st:.3e}"
    gat = T.map2alm_adjoint(to_dev(alm, "f64", True)).cpu().numpy()[0]
    ref = oracle.map2alm_adjoint_rings(nside, lmax, mmax, alm[0], rings)
    got = np.concatenate([gat[s] for s in slices])
    e_at = np.abs(got - ref).max() / np.abs(ref).max()
    assert e_at <= TOL64, f"map2alm_adjoint {e_at:.3e}"
    print("cfg5", e_syn, e_ana, e_st, e_at)


@pytest.mark.parametrize("nside,lmax,batch,dtype", [(32, 64, 1, "f64"), (64, 128, 16, "f32"), (128, 255, 1, "f64"),
                                                    (256, 600, 8, "f32"), (128, 200, 4, "f32")])
def test_results_are_bitwise_repeatable(nside, lmax, batch, dtype):
    """Race / uninitialised-memory screen (compute-sanitizer is not available on the GPU pool): every kernel family
    -- direct, channel-blocked direct, power-of-two, chirp-z FFT kernels; fp64, fp32 and contraction Legendre kernels
    with several ring chunks -- must give bit-identical results when the same call is repeated on a workspace that
    other calls have dirtied in between, and on a second, freshly initialised workspace."""
    T1 = make_transform(nside, lmax, lmax, batch, dtype)
    T2 = make_transform(nside, lmax, lmax, batch, dtype)
    alm = to_dev(synth.powerlaw_alm(5, lmax, lmax, batch), dtype, True)
    fmap = to_dev(synth.gaussian_map(6, nside, batch), dtype)
    ref = {"s": T1.alm2map(alm).clone(), "a": T1.map2alm(fmap).clone(), "st": T1.alm2map_adjoint(fmap).clone(),
           "at": T1.map2alm_adjoint(alm).clone()}
    for T in (T1, T2, T1):
        assert torch.equal(T.map2alm(fmap), ref["a"])
        assert torch.equal(T.alm2map_adjoint(fmap), ref["st"])
        assert torch.equal(T.alm2map(alm), ref["s"])
        assert torch.equal(T.map2alm_adjoint(alm), ref["at"])


@pytest.mark.parametrize("nside,lmax,batch,dtype", [(64, 128, 1, "f64"), (128, 255, 8, "f32"), (512, 1023, 1, "f64"),
                                                    (256, 511, 2, "f32")])
def test_cuda_graph_capture_replay(nside, lmax, batch, dtype):
    """include/cuhpx.h promises that the transform calls never synchronise and can be captured in a CUDA graph
    (the FFT stage forks part of its work onto a library stream and joins it back: exactly what breaks under capture
    if done wrong).  Capture map2alm + alm2map once, replay on three fresh inputs, compare with eager bit for bit."""
    B = _binding()
    T = make_transform(nside, lmax, lmax, batch, dtype)
    ins = [(to_dev(synth.gaussian_map(40 + k, nside, batch), dtype), to_dev(synth.powerlaw_alm(50 + k, lmax, lmax, batch), dtype, True))
           for k in range(3)]
    s_map, s_alm = ins[0][0].clone(), ins[0][1].clone()
    o_alm = torch.zeros_like(s_alm)
    o_map = torch.zeros_like(s_map)
    T.map2alm(s_map)  # warm: nothing is created lazily inside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        B.cuhpx_map2alm(*T.params, s_map, o_alm, None, T.workspace)
        B.cuhpx_alm2map(*T.params, s_alm, o_map, T.workspace)
    for fmap, alm in ins:
        s_map.copy_(fmap)
        s_alm.copy_(alm)
        o_alm.zero_()
        o_map.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(o_alm, T.map2alm(fmap)) and torch.equal(o_map, T.alm2map(alm))
    B.cuhpx_workspace_check(*T.params, T.workspace)


def test_late_start_tables_change_no_bit():
    """fp64 Legendre kernels with >= 2048 ring pairs start each (order, ring chunk) at the first tile with a significant
    ring pair, from a tabulated recurrence state (legendre.cu "late start").  The skipped steps carry no data, so the
    results must equal those of the full walk (CUHPX_LATE_START=0, its own process: plans are memoised) bit for bit."""
    import os
    import subprocess
    import sys
    import tempfile

    nside, lmax = 1024, 2047  # 2048 ring pairs: the smallest transform that plans the tables
    code = (
        "import sys, torch; sys.path.insert(0, %r)\n"
        "from paper_2510_01785_b200 import binding as B\n"
        "t = B.Transform(%d, %d, %d, 1, torch.float64)\n"
        "g = torch.Generator(device='cuda').manual_seed(5)\n"
        "m = torch.randn(1, t.npix, dtype=torch.float64, device='cuda', generator=g)\n"
        "a = t.map2alm(m); r = t.alm2map(a); ga = t.alm2map_adjoint(m); gm = t.map2alm_adjoint(a)\n"
        "torch.save({'alm': a.cpu(), 'map': r.cpu(), 'galm': ga.cpu(), 'gmap': gm.cpu(), 'ws': t.workspace.numel()}, sys.argv[1])\n"
    ) % (os.path.dirname(os.path.dirname(os.path.abspath(__file__))), nside, lmax, lmax)
    with tempfile.TemporaryDirectory() as d:
        res = {}
        for arm in ("0", "1"):
            env = dict(os.environ)
            env.pop("CUHPX_LATE_START", None)
            if arm == "0":
                env["CUHPX_LATE_START"] = "0"
            path = os.path.join(d, f"arm{arm}.pt")
            subprocess.run([sys.executable, "-c", code, path], env=env, check=True, timeout=600)
            res[arm] = torch.load(path)
    assert res["1"]["ws"] > res["0"]["ws"], "the tables were not planned"
    for k in ("alm", "map", "galm", "gmap"):
        assert torch.equal(res["0"][k], res["1"][k]), f"{k} differs between the full walk and the late start"
