"""Pins of the incoherent-dedispersion oracle (second stage of the semi-coherent search,
PAPER.md:35, 141, 185) -- CPU only.

The oracle (oracle/cdmt_oracle.c: oracle_incoherent) shifts every channel by the residual delay of
a fine DM offset and sums over channels.  Pins: the delay against Eq. 2 (the separately written and
paper-pinned oracle_sweep_seconds and the paper's printed t_d), closed forms (zero offset = plain
channel sum, a dispersed pulse train adds up to nch at the matching trial only, histogram of the
mismatch at the others), antisymmetry, shift invariance, and brute-force Python loops.
"""
import os

import numpy as np
import pytest

from oracle import cdmt_oracle as orc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def golden():
    g = {}
    for ln in open(GOLDEN):
        ln = ln.split("#")[0].strip()
        if ln:
            k, v = ln.split("=")
            g[k.strip()] = float(v)
    return g


def survey_params(nsub=4, nchan=8, ndec=1, f_lo=134.9):
    fcen = f_lo + 0.1953125 * (np.arange(nsub) + 0.5)
    return orc.Params(nsub, fcen, 0.1953125, 65536, 2048 * nchan, nchan, ndec, [0.0])


def test_I0_channel_frequencies_descending_and_centred():
    p = survey_params(nsub=3, nchan=8)
    f = orc.channel_frequencies(p)
    assert f.size == 24 and np.all(np.diff(f) < 0)
    np.testing.assert_allclose(-np.diff(f), 0.1953125 / 8, rtol=1e-12)          # 24.41 kHz channels
    np.testing.assert_allclose(f.mean(), p.fcen.mean(), rtol=1e-12)


def test_I1_shifts_are_eq2_between_channel_centres():
    """shift = rint(t_d / tsamp) with t_d of Eq. 2 evaluated by oracle_sweep_seconds (its own function,
    pinned to the paper's 3.3 ms / 5.7 ms) over the band [f_j, f_0]."""
    g = golden()
    p = survey_params(nsub=10, nchan=8, f_lo=g["survey_fmin_mhz"])
    f = orc.channel_frequencies(p)
    tsamp = g["tres_us_nc8"] * 1e-6
    ddm = np.array([-0.5, -0.002, 0.0, 0.002, 0.25, 0.5])
    r = orc.incoherent(np.zeros((4, f.size), np.float32), f, tsamp, ddm, want_ts=False)
    for k, d in enumerate(ddm):
        for j in (1, 7, 40, f.size - 1):
            td = orc.sweep_seconds(0.5 * (f[0] + f[j]), f[0] - f[j], d)
            assert abs(r["shifts"][k, j] - td / tsamp) <= 0.5 + 1e-9
    assert (r["shifts"][:, 0] == 0).all() and (r["shifts"][2] == 0).all()
    assert r["smin"] == r["shifts"].min() and r["range"] == r["shifts"].max() - r["shifts"].min()
    # the paper's own number: a 24.41 kHz channel at 135 MHz sweeps 3.3 ms at DM 39.658
    fa = np.array([135.0 + 0.0244140625 / 2, 135.0 - 0.0244140625 / 2])
    one = orc.incoherent(np.zeros((2, 2), np.float32), fa, 1e-4, [g["dm_J1810"]], want_ts=False)
    assert abs(one["shifts"][0, 1] * 1e-4 * 1e3 - g["td_ms_J1810"]) < 0.06


def test_I2_zero_offset_is_the_channel_sum():
    rng = np.random.default_rng(2)
    fb = rng.random((300, 32)).astype(np.float32)
    p = survey_params()
    f = orc.channel_frequencies(p)
    r = orc.incoherent(fb, f, 40.96e-6, [0.0])
    assert r["range"] == 0
    np.testing.assert_allclose(r["ts"][0], fb.astype(np.float64).sum(axis=1), rtol=1e-6)


def test_I3_dispersed_pulses_add_up_only_at_the_matching_trial():
    """fb = unit impulses delayed by the shifts of trial k*: exactly nch at the pulse time in trial k*; in
    trial k the pulse is spread as the histogram of shift differences (closed form)."""
    p = survey_params(nsub=6, nchan=8, f_lo=120.0)
    f = orc.channel_frequencies(p)
    nch, nt, tsamp = f.size, 900, 40.96e-6
    ddm = np.round(np.arange(-0.5, 0.5001, 0.05), 6)
    sh = orc.incoherent(np.zeros((1, nch), np.float32), f, tsamp, ddm, want_ts=False)
    smin, kstar = sh["smin"], 15
    t0 = 400
    fb = np.zeros((nt, nch), np.float32)
    fb[t0 + sh["shifts"][kstar], np.arange(nch)] = 1.0
    r = orc.incoherent(fb, f, tsamp, ddm)
    ts = r["ts"]
    assert ts[kstar].max() == nch and ts[kstar].argmax() == t0 + smin
    assert (np.delete(ts[kstar], t0 + smin) == 0).all()
    for k in range(len(ddm)):
        want = np.zeros(ts.shape[1])
        np.add.at(want, t0 + smin + sh["shifts"][kstar] - sh["shifts"][k], 1.0)
        assert np.array_equal(ts[k], want.astype(np.float32))
        if k != kstar:
            assert ts[k].max() < nch
    # peak height falls monotonically away from the matching trial
    peaks = ts.max(axis=1)
    assert all(peaks[k] >= peaks[k + 1] for k in range(kstar, len(ddm) - 1))
    assert all(peaks[k] <= peaks[k + 1] for k in range(0, kstar))


def test_I4_brute_force_python_loops():
    rng = np.random.default_rng(4)
    p = survey_params(nsub=2, nchan=4, f_lo=115.0)
    f = orc.channel_frequencies(p)
    fb = rng.standard_normal((120, f.size)).astype(np.float32)
    ddm, tsamp = [-0.3, 0.1, 0.45], 20.48e-6
    r = orc.incoherent(fb, f, tsamp, ddm)
    kdm = golden()["kdm_inv_s_mhz2"]
    sh = np.array([[int(np.rint(d * (fj ** -2 - f[0] ** -2) / kdm / tsamp)) for fj in f] for d in ddm])
    assert np.array_equal(sh, r["shifts"])
    smin, rng_ = sh.min(), sh.max() - sh.min()
    assert r["ts"].shape == (3, 120 - rng_)
    for k in range(3):
        for t in range(120 - rng_):
            want = sum(float(fb[t + sh[k, j] - smin, j]) for j in range(f.size))
            assert abs(r["ts"][k, t] - want) <= 1e-6 * max(1.0, abs(want))


def test_I5_antisymmetry_and_shift_invariance():
    p = survey_params(nsub=3, nchan=8, f_lo=125.0)
    f = orc.channel_frequencies(p)
    ddm = np.array([-0.4, -0.1, 0.1, 0.4])
    rng = np.random.default_rng(5)
    fb = rng.random((400, f.size)).astype(np.float32)
    r = orc.incoherent(fb, f, 40.96e-6, ddm)
    assert np.array_equal(r["shifts"][0], -r["shifts"][3]) and np.array_equal(r["shifts"][1], -r["shifts"][2])
    # delaying the whole filterbank by m samples delays every time series by m
    m = 7
    r2 = orc.incoherent(np.roll(fb, m, axis=0), f, 40.96e-6, ddm)
    assert np.array_equal(r2["ts"][:, m:], r["ts"][:, :-m])
    # linearity
    r3 = orc.incoherent((2 * fb).astype(np.float32), f, 40.96e-6, ddm)
    np.testing.assert_allclose(r3["ts"], 2 * r["ts"], rtol=1e-6)


def test_I6_paper_trial_count():
    """80 coherent trials x (1.0 / 0.002) fine steps = 40 000 incoherent trials."""
    g = golden()
    per = round(1.0 / 0.002)
    assert 80 * per == g["incoherent_trials"]
    assert np.arange(-0.5, 0.5, 0.002).size == per
