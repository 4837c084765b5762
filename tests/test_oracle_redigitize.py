"""Pins of the redigitisation oracle (Alg. 1 l.104-106) -- CPU only.

The oracle (oracle/cdmt_oracle.c: oracle_redigitize) forms per-block sums of I and I^2, adds
them into per-channel mean / standard deviation, derives offset and scale (reading Q22) and
quantises in float32.  Each pin below is something other than the oracle's own formula:
numpy's two-pass mean / std, closed forms on dyadic inputs, invariants, and a brute-force
restatement of the float32 decision with numpy scalars.
"""
import numpy as np
import pytest

from oracle import cdmt_oracle as orc


def rand_fb(seed, ndm, nt, nch, mu=12.0, sd=3.0):
    rng = np.random.default_rng(seed)
    # chi-square-like, positive, channel-dependent level: what an integrated Stokes-I filterbank looks like
    lev = 1.0 + rng.random(nch)
    return ((rng.standard_normal((ndm, nt, nch)) * sd + mu) * lev).astype(np.float32)


@pytest.mark.parametrize("shape", [(1, 8, 1, 1), (3, 40, 5, 4), (2, 96, 16, 6), (4, 21, 7, 3)])
def test_R1_statistics_match_numpy_two_pass(shape):
    """mean/std from the segment sums = numpy's two-pass mean and population std (library routine
    with another formula)."""
    ndm, nt, nch, nblock = shape
    nt = nt - nt % nblock
    fb = rand_fb(1, ndm, nt, nch)
    r = orc.redigitize(fb, nblock)
    f64 = fb.astype(np.float64)
    np.testing.assert_allclose(r["mean"], f64.mean(axis=1), rtol=1e-13)
    np.testing.assert_allclose(r["std"], f64.std(axis=1), rtol=1e-9)   # E[x^2]-E[x]^2 loses digits
    seg = f64.reshape(ndm, nblock, nt // nblock, nch)
    np.testing.assert_allclose(r["segsum"][..., 0], seg.sum(axis=2), rtol=1e-13)
    np.testing.assert_allclose(r["segsum"][..., 1], (seg ** 2).sum(axis=2), rtol=1e-13)


def test_R2_closed_form_two_level_channel():
    """x alternating a-b, a+b: mean a, std b exactly -> codes qmean -+ qstd exactly (dyadic values)."""
    a, b = 40.0, 2.5
    nt = 64
    x = np.where(np.arange(nt) % 2 == 0, a - b, a + b).astype(np.float32)
    fb = np.stack([x, 4 * x + 3], axis=-1)[None]          # second channel: affine copy
    r = orc.redigitize(fb, 4, qmean=64, qstd=16)
    assert r["mean"][0, 0] == a and r["std"][0, 0] == b
    assert r["scale"][0, 0] == np.float32(b / 16) and r["offset"][0, 0] == np.float32(a - 64 * b / 16)
    assert set(r["codes"][0, :, 0]) == {48, 80}
    assert (r["codes"][0, ::2, 0] == 48).all() and (r["codes"][0, 1::2, 0] == 80).all()
    # other targets
    r = orc.redigitize(fb, 1, qmean=128, qstd=32)
    assert set(r["codes"][0, :, 0]) == {96, 160}


def test_R3_clipping_both_ends():
    """Outliers saturate at 0 and 255 (8-bit), they do not wrap."""
    nt = 4096
    x = np.where(np.arange(nt) % 2 == 0, 9.0, 11.0).astype(np.float32)
    x[7] = 1000.0      # z = +45 -> above code 255
    x[100] = -1000.0   # z = -45 -> below code 0
    r = orc.redigitize(x[None, :, None], 2)
    c = r["codes"][0, :, 0]
    assert c[7] == 255 and c[100] == 0
    assert c.dtype == np.uint8
    # a NaN sample must not crash and maps to 0
    r2 = orc.quantize(np.array([np.nan, 10.0], np.float32)[None, :, None], [[10.0]], [[1.0]])
    assert r2[0, 0, 0] == 0 and r2[0, 1, 0] == 0


def test_R4_ties_round_half_to_even():
    """(x-offset)/scale = k + 1/2 exactly -> the even neighbour (float32 rint)."""
    off, sc = np.float32(8.0), np.float32(0.25)
    ks = np.arange(0, 20)
    x = (off + sc * (ks + 0.5)).astype(np.float32)         # exact in float32
    c = orc.quantize(x[None, :, None], [[off]], [[sc]])[0, :, 0]
    want = np.where(ks % 2 == 0, ks, ks + 1)
    assert (c == want).all()


def test_R5_constant_channel():
    """std = 0 -> scale 1, every code = qmean (reading Q22)."""
    fb = np.full((2, 30, 3), 7.25, np.float32)
    r = orc.redigitize(fb, 3)
    assert (r["std"] == 0).all() and (r["scale"] == 1).all()
    assert (r["codes"] == 64).all()


def test_R6_affine_invariance():
    """Codes depend on (x - mean)/std only: scaling a channel by a power of two and shifting it by a
    dyadic constant leaves every code unchanged."""
    rng = np.random.default_rng(5)
    fb = (rng.integers(0, 4096, size=(2, 120, 4)) / 64.0).astype(np.float32)   # dyadic grid
    r0 = orc.redigitize(fb, 5)
    r1 = orc.redigitize((fb * 8.0).astype(np.float32), 5)
    assert (r0["codes"] == r1["codes"]).all()
    np.testing.assert_allclose(r1["std"], 8 * r0["std"], rtol=1e-12)
    r2 = orc.redigitize((fb * 0.5 + 16.0).astype(np.float32), 5)
    assert (np.abs(r0["codes"].astype(int) - r2["codes"].astype(int)) <= 1).all()
    assert (r0["codes"] != r2["codes"]).mean() < 0.01


def test_R7_brute_force_float32_decision():
    """The quantiser restated with numpy float32 scalars, one operation at a time."""
    fb = rand_fb(7, 2, 24, 3)
    r = orc.redigitize(fb, 2, qmean=100, qstd=20)
    for d in range(2):
        for c in range(3):
            col = fb[d, :, c].astype(np.float64)
            mu = col.sum() / col.size
            sd = np.sqrt(max(0.0, (col * col).sum() / col.size - mu * mu))
            sc = np.float32(sd / 20)
            off = np.float32(mu - 100 * (sd / 20))
            assert r["scale"][d, c] == sc and r["offset"][d, c] == off
            for t in range(24):
                q = np.float32(np.float32(fb[d, t, c] - off) / sc)
                want = int(min(255.0, max(0.0, float(np.rint(q)))))
                assert r["codes"][d, t, c] == want


def test_R8_segmentation_does_not_matter():
    """The statistics are those of the whole batch whatever the segment (block) length."""
    fb = rand_fb(8, 2, 120, 5)
    ra, rb, rc = orc.redigitize(fb, 1), orc.redigitize(fb, 8), orc.redigitize(fb, 120)
    for k in ("mean", "std"):
        np.testing.assert_allclose(ra[k], rb[k], rtol=1e-13)
        np.testing.assert_allclose(ra[k], rc[k], rtol=1e-13)
    assert (ra["codes"] == rb["codes"]).mean() > 0.999


def test_R9_code_statistics_and_volume():
    """Codes of a Gaussian channel have mean qmean and std qstd (to sampling and rounding error);
    8 bits per sample is the paper's 2.2 GB per DM for 1200 s x 10 subbands."""
    fb = rand_fb(9, 1, 20000, 2)
    r = orc.redigitize(fb, 10)
    c = r["codes"].astype(np.float64)
    assert abs(c.mean() - 64) < 0.05
    assert abs(c.std() - 16) < 0.1            # + 1/12 quantisation variance
    nbytes = 1200 * 195312.5 * 10 * r["codes"].itemsize
    assert abs(nbytes / 2 ** 30 - 2.2) < 0.05


def test_quantize_matches_redigitize_on_its_own_offsets():
    fb = rand_fb(10, 3, 50, 4)
    r = orc.redigitize(fb, 5)
    assert (orc.quantize(fb, r["offset"], r["scale"]) == r["codes"]).all()
