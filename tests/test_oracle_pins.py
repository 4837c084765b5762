"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

P1..P10 are the rows of DESIGN.md "What pins the oracle".  None of these tests calls the
CUDA library; none takes an expected value from it.
"""
import os

import numpy as np
import pytest

from oracle import cdmt_oracle as orc
import cdmt_synth as synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def golden():
    vals = {}
    with open(GOLDEN) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if line:
                k, v = line.split("=")
                vals[k.strip()] = float(v)
    return vals


def params(nsub=1, fcen=(150.0,), nfft=256, noverlap=64, nchan=4, ndec=2, dm=(0.0,),
           in_dtype=orc.IN_CF32, chirp_ref=orc.REF_CHANNEL, bw=synth.BW_MHZ):
    return orc.Params(nsub, np.asarray(fcen, dtype=np.float64), bw, nfft, noverlap, nchan, ndec,
                      np.asarray(dm, dtype=np.float64), in_dtype, chirp_ref)


def noise(shape, seed):
    rng = np.random.default_rng(seed)
    return ((rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / np.sqrt(2)).astype(np.complex64)


# ------------------------------------------------------------------ P1
@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 32, 64, 128, 256, 512])
@pytest.mark.parametrize("sign", [-1, +1])
def test_p1_fft_vs_bruteforce_dft(n, sign):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    k = np.arange(n)
    W = np.exp(sign * 2j * np.pi * np.outer(k, k) / n)      # O(n^2) definition
    ref = W @ x
    got = orc.fft(x, sign)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max() * max(1, n)
    lib = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n   # library second opinion
    assert np.abs(got - lib).max() <= 1e-12 * np.abs(ref).max() * max(1, n)


def test_p1_fft_rejects_non_power_of_two():
    with pytest.raises(ValueError):
        orc.fft(np.zeros(12, dtype=np.complex128), -1)


# ------------------------------------------------------------------ P2
def test_p2_dm0_is_plain_channelisation():
    """DM = 0: mix each channel to its centre, ideal low-pass, decimate by C (time domain,
    brute force), unpad, detect, integrate, pack descending."""
    N, O, C, D, S = 256, 64, 4, 2, 2
    M, step, h = N // C, N - O, O // (2 * C)
    T = N + 2 * step + 17                      # ragged tail: 17 unused samples
    B = (T - N) // step + 1
    V = M - 2 * h
    Vd = V // D
    fcen = [140.0, 140.0 + synth.BW_MHZ]
    x = noise((S, 2, T), 11)
    p = params(S, fcen, N, O, C, D, [0.0])
    got = orc.run(p, x, want64=True)[1]
    assert got.shape == (1, B * Vd, S * C)
    n = np.arange(N)
    m = np.arange(M)
    exp = np.zeros_like(got)
    for s in range(S):
        for b in range(B):
            I = np.zeros((C, M))
            for pol in range(2):
                u = x[s, pol, b * step:b * step + N].astype(np.complex128)
                for c in range(C):
                    mix = np.exp(-2j * np.pi * (c * M + M // 2 - N // 2) * n / N)
                    t = np.arange(M)
                    lag = t[:, None] * C - n[None, :]                           # [t][n]
                    kern = np.exp(2j * np.pi * (m[None, None, :] - M // 2) * lag[:, :, None] / N).sum(-1)
                    y = kern @ (u * mix)
                    I[c] += np.abs(y) ** 2 / (N * M)
            F = I[:, h:M - h].reshape(C, Vd, D).sum(-1)                          # [c][q]
            for c in range(C):
                exp[0, b * Vd:(b + 1) * Vd, S * C - 1 - (s * C + c)] = F[c]
    assert np.abs(got - exp).max() <= 1e-10 * exp.max()


# ------------------------------------------------------------------ P3
@pytest.mark.parametrize("nblk_off", [0, 1, 2])
def test_p3_impulse_closed_form(nblk_off):
    N, O, C, D = 512, 128, 8, 4
    M, step, h = N // C, N - O, O // (2 * C)
    Vd = (M - 2 * h) // D
    T = N + 3 * step
    A = 3.0
    n0 = O // 2 + nblk_off * step + 5 * C * D + 2 * C       # multiple of C, inside kept range
    x = np.zeros((1, 2, T), dtype=np.complex64)
    x[0, :, n0] = A
    p = params(1, [150.0], N, O, C, D, [0.0])
    out = orc.run(p, x, want64=True)[1][0]                  # [tau][chan]
    tau = (n0 - O // 2) // (C * D)
    assert tau == nblk_off * Vd + 5
    exp = np.zeros_like(out)
    exp[tau, :] = 2 * A * A / C
    assert np.abs(out - exp).max() <= 1e-12 * A * A


# ------------------------------------------------------------------ P4
@pytest.mark.parametrize("s0,c0", [(0, 0), (1, 2), (2, 3)])
def test_p4_tone_lands_in_one_descending_channel_for_every_dm(s0, c0):
    N, O, C, D, S = 256, 64, 4, 2, 3
    M = N // C
    T = N + 2 * (N - O)
    a = 0.7
    m0 = M // 2 + 3                                        # a bin inside channel c0
    j0 = c0 * M + m0                                       # index in increasing-frequency order
    k0 = (j0 + N // 2) % N                                 # FFT bin (swap halves)
    x = np.zeros((S, 2, T), dtype=np.complex64)
    n = np.arange(T)
    x[s0, :, :] = (a * np.exp(2j * np.pi * k0 * n / N)).astype(np.complex64)
    fcen = 120.0 + (np.arange(S) + 0.5) * synth.BW_MHZ
    dms = [0.0, 3.0, 17.5, -8.0]
    out = orc.run(params(S, fcen, N, O, C, D, dms), x, want64=True)[1]
    exp = np.zeros_like(out)
    exp[:, :, S * C - 1 - (s0 * C + c0)] = 2 * a * a * C * D
    assert np.abs(out - exp).max() <= 1e-6 * exp.max()     # float32 tone samples limit this


def test_p4_higher_frequency_is_lower_output_index():
    """A tone nearer the top of the band must come out at a smaller channel index."""
    N, O, C, D = 256, 64, 4, 2
    T = N
    n = np.arange(T)
    outs = []
    for fbin in (-100, +100):                              # offset from centre in FFT bins
        x = np.zeros((1, 2, T), dtype=np.complex64)
        x[0, :, :] = np.exp(2j * np.pi * fbin * n / N).astype(np.complex64)
        o = orc.run(params(1, [150.0], N, O, C, D, [0.0]), x)
        outs.append(int(o[0].sum(0).argmax()))
    assert outs[0] > outs[1]


# ------------------------------------------------------------------ P5
@pytest.mark.parametrize("dm", [0.0, 5.0, 40.0])
@pytest.mark.parametrize("ref", [orc.REF_CHANNEL, orc.REF_SUBBAND])
def test_p5_parseval_before_unpad(dm, ref):
    N, C = 1024, 8
    M = N // C
    u = noise((N,), 5)
    p = params(1, [130.0], N, 256, C, 2, [dm], chirp_ref=ref)
    tot = 0.0
    for c in range(C):
        y = orc.channel_timeseries(p, 0, c, dm, u)
        tot += (np.abs(y) ** 2).sum() / (N * M)
    assert abs(tot - (np.abs(u.astype(np.complex128)) ** 2).sum()) <= 1e-12 * tot


def test_p5_noise_mean_level():
    cfg = synth.small_config(nsub=2, nsamp=16384, nfft=1024, noverlap=256, nchan=4, ndec=2,
                             dm=(0.0, 7.0))
    x = synth.generate(cfg)
    out = orc.run(orc.Params(**cfg.plan_kwargs()), x)
    # unit-variance complex noise: every (pol, channel, sample) has mean power 1 -> 2 D
    assert abs(out.mean() / (2 * cfg.ndec) - 1.0) < 0.02


# ------------------------------------------------------------------ P6
@pytest.mark.parametrize("ref", [orc.REF_CHANNEL, orc.REF_SUBBAND])
def test_p6_transfer_function_unit_modulus_and_inverse(ref):
    p = params(1, [125.0], 2048, 512, 8, 2, [33.0], chirp_ref=ref)
    for c in (0, 3, 7):
        Hp = orc.transfer_function(p, 125.0, c, 33.0)
        Hm = orc.transfer_function(p, 125.0, c, -33.0)
        assert np.abs(np.abs(Hp) - 1).max() < 1e-14
        assert np.abs(Hp * Hm - 1).max() < 1e-9
        H0 = orc.transfer_function(p, 125.0, c, 0.0)
        assert np.abs(H0 - 1).max() == 0.0


@pytest.mark.parametrize("ref", [orc.REF_CHANNEL, orc.REF_SUBBAND])
def test_p6_dispersed_then_dedispersed_is_identity(ref):
    """A block dispersed by the generator's independently typed ISM response (conjugate of
    Eq. 1 on numpy's frequency axis) and processed at +DM equals the block at DM=0."""
    N, C, dm, fc = 2048, 8, 12.5, 118.0
    u = noise((N,), 9)
    ud = synth.disperse(u, dm, fc, synth.BW_MHZ, C, ref).astype(np.complex64)
    p = params(1, [fc], N, 512, C, 2, [dm], chirp_ref=ref)
    for c in range(C):
        y0 = orc.channel_timeseries(p, 0, c, 0.0, u)
        y1 = orc.channel_timeseries(p, 0, c, dm, ud)
        assert np.abs(y1 - y0).max() <= 2e-5 * np.abs(y0).max()   # complex64 storage of ud


# ------------------------------------------------------------------ P7
def test_p7_group_delay_is_eq2_and_paper_values():
    g = golden()
    assert g["kdm_inv_s_mhz2"] == 2.41e-4
    f0 = g["td_freq_mhz"]
    cw = g["subband_bw_khz"] * 1e-3 / g["survey_nc"]
    assert abs(cw * 1e3 - g["chan_bw_khz_nc8"]) < 0.005
    assert abs(g["survey_nc"] / (synth.BW_MHZ) - g["tres_us_nc8"]) < 1e-9
    for dm, td_ms in ((g["dm_J1810"], g["td_ms_J1810"]), (g["dm_J2215"], g["td_ms_J2215"])):
        td = orc.sweep_seconds(f0, cw, dm)
        assert abs(td * 1e3 - td_ms) < 0.05                 # the paper prints one decimal
        # Eq. 1 <-> Eq. 2: the chirp's group delay -dphi/dnu swept across the channel equals t_d.
        eps = 1e-7

        def dphi(f):                                        # cycles per MHz = microseconds
            return (orc.chirp_phase_cycles(dm, f0, f + eps) - orc.chirp_phase_cycles(dm, f0, f - eps)) / (2 * eps)
        swept = (dphi(+cw / 2) - dphi(-cw / 2)) * 1e-6       # lower edge is removed by more
        assert abs(swept - td) < 1e-6 * td
        # sign of the adopted reading (Q2): H advances the low edge relative to the high edge,
        # i.e. -dphi/dnu is larger (later) at lower frequency for the ISM = conj(H)
        assert dphi(-cw / 2) < 0 < dphi(+cw / 2)


def test_p7_minimum_overlap_of_the_survey_setup():
    """n_d = r t_d / n_c for the lowest channel; the survey used n_d = 2048."""
    g = golden()
    cw = synth.BW_MHZ / g["survey_nc"]
    flo_centre = g["survey_fmin_mhz"] + cw / 2
    td = orc.sweep_seconds(flo_centre, cw, g["survey_dm_max"])
    nd = synth.BW_MHZ * 1e6 * td / g["survey_nc"]
    assert 250 < nd < 270 and nd < g["survey_nd"]
    assert g["survey_nbin"] / g["survey_nc"] == g["survey_mbin"]


def test_p7_data_volumes():
    g = golden()
    nbytes_in = g["obs_seconds"] * synth.BW_MHZ * 1e6 * 10 * 2 * 2      # 10 subbands, 2 pols, (re,im) int8
    assert abs(nbytes_in / 2 ** 30 - g["in_gb_10sub_20min"]) < 0.1
    nbytes_out = g["obs_seconds"] * synth.BW_MHZ * 1e6 * 10            # 8-bit, no averaging
    assert abs(nbytes_out / 2 ** 30 - g["out_gb_per_dm"]) < 0.05


# ------------------------------------------------------------------ P8
def test_p8_subband_vs_channel_reference_differ_by_a_pure_delay():
    N, C, dm, fc = 4096, 8, 20.0, 121.0
    M = N // C
    u = noise((N,), 21)
    pc = params(1, [fc], N, 1024, C, 2, [dm], chirp_ref=orc.REF_CHANNEL)
    ps = params(1, [fc], N, 1024, C, 2, [dm], chirp_ref=orc.REF_SUBBAND)
    kdm = 1.0 / 2.41e-4
    for c in (0, 2, 7):
        Hc = orc.transfer_function(pc, fc, c, dm)
        Hs = orc.transfer_function(ps, fc, c, dm)
        dphi = np.unwrap(np.angle(Hs * np.conj(Hc))) / (2 * np.pi)
        assert np.abs(np.diff(dphi, 2)).max() < 1e-9                   # linear in frequency
        fchan = fc + (c + 0.5 - C / 2) * synth.BW_MHZ / C
        delay_s = kdm * dm * (fc ** -2 - fchan ** -2)                   # d(phi_s - phi_c)/dnu
        slope = np.diff(dphi).mean() / (synth.BW_MHZ / N * 1e6)        # cycles per Hz = seconds
        assert abs(slope - delay_s) < 1e-6 * abs(delay_s)
        # and the time series are circularly shifted copies (up to a constant phase)
        yc = orc.channel_timeseries(pc, 0, c, dm, u)
        ys = orc.channel_timeseries(ps, 0, c, dm, u)
        Yc, Ys = np.fft.fftshift(np.fft.fft(yc)), np.fft.fftshift(np.fft.fft(ys))
        assert np.abs(np.abs(Ys) - np.abs(Yc)).max() < 1e-9 * np.abs(Yc).max()
        ratio = Ys * np.conj(Yc) / np.abs(Yc) ** 2          # unit phasors e^{i(alpha + beta k)}
        stepph = ratio[1:] * np.conj(ratio[:-1])            # e^{i beta}: the same for every bin
        assert np.abs(stepph - stepph[0]).max() < 1e-7
        # ys[t] = yc[t + delta]  <=>  FFT(ys)[k] = FFT(yc)[k] e^{+2 pi i k delta / M}
        shift_samples = np.angle(stepph[0]) * M / (2 * np.pi)
        exp_shift = delay_s * synth.BW_MHZ * 1e6 / C        # delta in channelised samples
        assert abs((shift_samples - exp_shift + M / 2) % M - M / 2) < 1e-4


# ------------------------------------------------------------------ P9
@pytest.mark.parametrize("ref", [orc.REF_CHANNEL, orc.REF_SUBBAND])
def test_p9_dispersed_impulse_recovered_only_at_matching_dm(ref):
    cfg = synth.make_config("c1")
    cfg.ndec = 1                                            # see the smear at neighbouring trials
    cfg.noise_sigma = 0.0
    if ref == orc.REF_SUBBAND:
        cfg.dm = np.array([0.0, 3.0, 4.0, 5.0])             # subband sweep is larger: closer trials
    x = synth.generate(cfg, chirp_ref=ref)
    p = orc.Params(**cfg.plan_kwargs(chirp_ref=ref))
    out = orc.run(p, x, want64=True)[1]
    imp = cfg.impulses[0]
    C, O = cfg.nchan, cfg.noverlap
    tau = (imp.n0 - O // 2) // C
    imatch = int(np.argmin(np.abs(cfg.dm - imp.dm)))
    peak = 2 * imp.amp ** 2 / C
    for d in range(cfg.ndm):
        od = out[d]
        for ch in range(cfg.nsub * C):
            assert int(od[:, ch].argmax()) in range(tau - 40, tau + 41)
        if d == imatch:
            assert (od.argmax(0) == tau).all()             # same sample in every channel
            assert np.abs(od[tau] / peak - 1).max() < 0.05   # a delta of the closed-form height
            off = np.delete(od, tau, axis=0)
            assert off.max() < 0.02 * peak
        else:
            # smeared within the channel (REF_CHANNEL) or channels misaligned (REF_SUBBAND)
            assert od.sum(1).max() < 0.7 * peak * cfg.nsub * C


def test_p9_c1_with_noise_peak_position():
    cfg = synth.make_config("c1")
    x = synth.generate(cfg)
    out = orc.run(orc.Params(**cfg.plan_kwargs()), x)
    ts = out.sum(-1)                                        # [dm][tau]
    d, tau = np.unravel_index(ts.argmax(), ts.shape)
    assert cfg.dm[d] == 4.0
    assert tau == (cfg.impulses[0].n0 - cfg.noverlap // 2) // (cfg.nchan * cfg.ndec)


# ------------------------------------------------------------------ P10
@pytest.mark.parametrize("ref", [orc.REF_CHANNEL, orc.REF_SUBBAND])
@pytest.mark.parametrize("in_dtype", [orc.IN_CF32, orc.IN_CI8])
def test_p10_bruteforce_chain_tiny(ref, in_dtype):
    """Whole chain by DFT matrices on numpy's own frequency axis, DM != 0, S=2, ragged T."""
    N, O, C, D, S = 64, 16, 4, 2, 2
    M, step, h = N // C, N - O, O // (2 * C)
    Vd = (M - 2 * h) // D
    T = N + 2 * step + 5
    B = (T - N) // step + 1
    fcen = np.array([110.0, 110.0 + synth.BW_MHZ])
    dms = np.array([0.0, 2.5, -1.0, 30.0])
    rng = np.random.default_rng(3)
    if in_dtype == orc.IN_CI8:
        xi = rng.integers(-127, 128, size=(S, 2, T, 2)).astype(np.int8)
        xc = xi[..., 0].astype(np.float64) + 1j * xi[..., 1]
        xin = xi
    else:
        xin = noise((S, 2, T), 4)
        xc = xin.astype(np.complex128)
    got = orc.run(params(S, fcen, N, O, C, D, dms, in_dtype, ref), xin, want64=True)[1]
    kN = np.arange(N)
    FN = np.exp(-2j * np.pi * np.outer(kN, kN) / N)
    kM = np.arange(M)
    BM = np.exp(+2j * np.pi * np.outer(kM, kM) / M)
    foff = np.fft.fftshift(np.fft.fftfreq(N, d=1.0 / synth.BW_MHZ))     # increasing frequency, MHz
    exp = np.zeros_like(got)
    for s in range(S):
        for b in range(B):
            for d, dm in enumerate(dms):
                I = np.zeros((C, M))
                for pol in range(2):
                    X = np.fft.fftshift(FN @ xc[s, pol, b * step:b * step + N])
                    for c in range(C):
                        sl = slice(c * M, (c + 1) * M)
                        if ref == orc.REF_SUBBAND:
                            ph = synth.ism_phase_cycles(dm, fcen[s], foff[sl])
                        else:
                            fch = foff[sl][M // 2]
                            ph = synth.ism_phase_cycles(dm, fcen[s] + fch, foff[sl] - fch)
                        Z = X[sl] * np.exp(2j * np.pi * ph)
                        y = BM @ np.fft.ifftshift(Z)
                        I[c] += np.abs(y) ** 2 / (N * M)
                F = I[:, h:M - h].reshape(C, Vd, D).sum(-1)
                for c in range(C):
                    exp[d, b * Vd:(b + 1) * Vd, S * C - 1 - (s * C + c)] = F[c]
    assert np.abs(got - exp).max() <= 1e-9 * exp.max()


def test_sizes_and_ragged_tail():
    p = params(1, [150.0], 4096, 1024, 8, 4, [0.0])
    assert p.sizes(2 ** 14) == (5, 512, 64, 96)
    assert p.sizes(2 ** 14 + 100)[0] == 5
    assert p.sizes(4096)[0] == 1
    with pytest.raises(ValueError):
        p.sizes(4095)
    with pytest.raises(ValueError):
        params(1, [150.0], 4096, 1000, 8, 4, [0.0]).sizes(2 ** 14)     # noverlap % 2C != 0


def test_units_equals_run():
    cfg = synth.small_config()
    x = synth.generate(cfg)
    p = orc.Params(**cfg.plan_kwargs())
    full = orc.run(p, x, want64=True)[1]
    B, Vd, C, S = cfg.nblock, cfg.nvalid_dec, cfg.nchan, cfg.nsub
    us = [(1, 0), (0, B - 1), (1, 1)]
    blocks = np.stack([x[s, :, b * cfg.step:b * cfg.step + cfg.nfft] for s, b in us])
    o = orc.units(p, [s for s, _ in us], blocks)
    for i, (s, b) in enumerate(us):
        ref = full[:, b * Vd:(b + 1) * Vd, :][:, :, ::-1][:, :, s * C:(s + 1) * C]
        assert np.array_equal(o[i], ref)
