"""GPU parity of cdmt_incoherent_dedisperse (semi-coherent search) against the oracle.

  * the shift table (an integer decided in fp64 on both sides) must be identical;
  * on integer-valued filterbanks every partial sum is exact in float32, so the time series must
    match the oracle BIT FOR BIT, whatever the summation order;
  * on noise-like float data the kernel adds nch float32 numbers (runs of channels that share their
    shifts first, four channels of a sample pairwise) where the oracle adds in double: |delta| <= 2e-5
    of the (positive) sums, far inside north_star's 1e-3 of the rms.
The cases cover the three launch forms: 16-byte rows with 128-sample tiles (two CTAs per SM), the same with
256-sample tiles (shift range too large for two small tiles), and the general kernel (channel count not a
multiple of 4, or a shift range beyond what two tiles can hold).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import cdmt_oracle as orc            # noqa: E402
import cdmt_synth as synth          # noqa: E402


@pytest.fixture(scope="module")
def cdmt():
    from paper_1607_00909_b200 import cdmt as m
    assert torch.cuda.is_available()
    return m


def make_plan(cdmt, nsub, nchan, ndec, ndm, f_lo=119.0):
    fcen = f_lo + 0.1953125 * (np.arange(nsub) + 0.5)
    kw = dict(nsub=nsub, fcen_mhz=fcen, bw_mhz=0.1953125, nfft=1024 * nchan, noverlap=512 * nchan, nchan=nchan,
              ndec=ndec, dm=np.arange(ndm) * 0.5)
    return cdmt.cdmt_plan_create(**kw), orc.Params(nsub, fcen, 0.1953125, 1024 * nchan, 512 * nchan, nchan, ndec, [0.0])


def gpu_incoherent(cdmt, plan, fb, ddm, pitch_pad=0):
    ndm, nt, nch = fb.shape
    q = cdmt.cdmt_incoherent_query(plan, ddm, nt)
    nout, nfine = q["nt_out"], len(ddm)
    pitch = nout + pitch_pad
    d_fb = torch.from_numpy(fb).cuda()
    d_ts = torch.full((ndm, nfine, pitch), -7.0, dtype=torch.float32, device="cuda")
    ws = torch.empty(max(256, q["workspace_bytes"]), dtype=torch.uint8, device="cuda")
    cdmt.cdmt_incoherent_dedisperse(plan, d_fb, nt * nch, nt, ddm, d_ts, nfine * pitch, pitch, ws, ws.numel())
    torch.cuda.synchronize()
    assert cdmt.cdmt_last_launch_count(plan) == 1
    ts = d_ts.cpu().numpy()
    if pitch_pad:
        assert (ts[:, :, nout:] == -7.0).all()          # nothing written past a row
    return ts[:, :, :nout], q


def oracle_incoherent(p, fb, ddm, nchan, ndec):
    f = orc.channel_frequencies(p)
    tsamp = nchan * ndec * synth.TSAMP_S
    return [orc.incoherent(fb[d], f, tsamp, ddm) for d in range(fb.shape[0])]


CASES = [
    # nsub nchan ndec ndm  nt   ddm grid                                   what
    (1, 8, 4, 2, 700, np.arange(-0.5, 0.5001, 0.02)),                      # 8 channels: one partial chunk
    (5, 8, 1, 1, 1500, np.arange(-0.5, 0.5001, 0.002)),                    # paper grid: 501 trials, 40 channels
    (36, 16, 16, 2, 600, np.arange(-0.25, 0.2501, 0.002)),                 # c3-like channels (576), time step 1.3 ms
    (3, 2, 1, 1, 2000, np.arange(-0.5, 0.5001, 0.1)),                      # 6 channels (scalar loads), coarse steps
    (7, 4, 2, 3, 1031, np.array([-0.3, -0.299, -0.1, 0.0, 0.004, 0.3])),   # 28 channels, irregular grid
    (64, 1, 1, 1, 3000, np.arange(0.0, 0.05001, 0.005)),                   # big shifts (range ~520): groups of one trial,
                                                                           # 256-sample tiles of the 16-byte kernel
    (64, 1, 1, 1, 4000, np.arange(0.0, 0.10001, 0.01)),                    # range ~1040: two tiles do not fit, general kernel
    (10, 8, 8, 1, 300, np.array([0.0])),                                   # single trial = channel sum
]


@pytest.mark.parametrize("case", CASES)
def test_incoherent_matches_oracle(cdmt, case):
    nsub, nchan, ndec, ndm, nt, ddm = case
    ddm = np.round(ddm, 9)
    plan, p = make_plan(cdmt, nsub, nchan, ndec, ndm)
    nch = nsub * nchan
    rng = np.random.default_rng(nch + nt)
    # integer-valued samples: exact in float32 -> bit-exact comparison
    fb_int = rng.integers(0, 64, size=(ndm, nt, nch)).astype(np.float32)
    ts, q = gpu_incoherent(cdmt, plan, fb_int, ddm, pitch_pad=3)
    ref = oracle_incoherent(p, fb_int, ddm, nchan, ndec)
    assert np.array_equal(cdmt.cdmt_incoherent_shifts(plan, ddm), ref[0]["shifts"])
    assert q["shift_min"] == ref[0]["smin"] and q["shift_range"] == ref[0]["range"]
    for d in range(ndm):
        assert ts[d].shape == ref[d]["ts"].shape
        assert np.array_equal(ts[d], ref[d]["ts"]), "plane %d" % d
    # noise-like float samples (integrated Stokes I: chi-square): float32 accumulation error only
    fb = (rng.chisquare(2 * 2 * ndec, size=(ndm, nt, nch)) / 2).astype(np.float32)
    ts, _ = gpu_incoherent(cdmt, plan, fb, ddm)
    ref = oracle_incoherent(p, fb, ddm, nchan, ndec)
    for d in range(ndm):
        np.testing.assert_allclose(ts[d], ref[d]["ts"], rtol=2e-5)


def test_incoherent_recovers_a_dispersed_pulse_at_the_matching_offset(cdmt):
    """Unit impulses delayed by the residual sweep of ddm = +0.118 add up to nch at that trial only."""
    nsub, nchan, ndec = 20, 8, 2
    plan, p = make_plan(cdmt, nsub, nchan, ndec, 1)
    nch, nt = nsub * nchan, 1200
    ddm = np.round(np.arange(-0.25, 0.2501, 0.002), 9)
    sh = cdmt.cdmt_incoherent_shifts(plan, ddm)
    kstar = int(np.argmin(np.abs(ddm - 0.118)))
    fb = np.zeros((1, nt, nch), np.float32)
    t0 = 500
    fb[0, t0 + sh[kstar], np.arange(nch)] = 1.0
    ts, q = gpu_incoherent(cdmt, plan, fb, ddm)
    peak = ts[0].max(axis=1)
    assert peak[kstar] == nch and ts[0, kstar].argmax() == t0 + q["shift_min"]
    assert (peak[np.arange(len(ddm)) != kstar] <= nch).all() and peak[0] < nch and peak[-1] < nch
    assert np.array_equal(ts[0], oracle_incoherent(p, fb, ddm, nchan, ndec)[0]["ts"])


def test_incoherent_after_execute_end_to_end(cdmt):
    """cdmt_execute -> cdmt_incoherent_dedisperse on the device against oracle.run -> oracle.incoherent."""
    cfg = synth.small_config(nsub=3, nsamp=2 ** 16, nfft=4096, noverlap=1024, nchan=8, ndec=4, dm=(0.0, 4.0))
    x = synth.generate(cfg)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    out = cdmt.run_on_device(plan, torch.from_numpy(x).cuda(), cfg.nsamp)
    ndm, nt, nch = out.shape
    ddm = np.round(np.arange(-0.5, 0.5001, 0.01), 9)
    q = cdmt.cdmt_incoherent_query(plan, ddm, nt)
    d_ts = torch.empty((ndm, len(ddm), q["nt_out"]), dtype=torch.float32, device="cuda")
    ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device="cuda")
    cdmt.cdmt_incoherent_dedisperse(plan, out, nt * nch, nt, ddm, d_ts, len(ddm) * q["nt_out"], q["nt_out"], ws,
                                    ws.numel())
    torch.cuda.synchronize()
    p = orc.Params(**cfg.plan_kwargs())
    fb_ref = orc.run(p, x)
    f = orc.channel_frequencies(p)
    for d in range(ndm):
        ref = orc.incoherent(fb_ref[d], f, cfg.nchan * cfg.ndec * synth.TSAMP_S, ddm)
        got = d_ts[d].cpu().numpy()
        rms = float(np.sqrt(np.mean(ref["ts"].astype(np.float64) ** 2)))
        assert np.abs(got - ref["ts"]).max() <= 1e-3 * rms


def test_incoherent_streams_over_block_groups_bit_exact(cdmt):
    """the filterbanks of a long observation are never resident at once.  execute ->
    incoherent runs group by group on a window of shift_range + nt_group rows (cdmt_incoherent_carry moves
    the halo); on integer data the concatenated series equal ONE whole-span oracle call bit for bit."""
    nsub, nchan, ndec, ndm = 12, 8, 2, 3
    plan, p = make_plan(cdmt, nsub, nchan, ndec, ndm)
    nch = nsub * nchan
    ddm = np.round(np.arange(-0.25, 0.2501, 0.004), 9)
    rng = np.random.default_rng(5)
    sizes = [700, 512, 301, 900]                       # rows per group (ragged)
    nt = sum(sizes)
    fb = rng.integers(0, 64, size=(ndm, nt, nch)).astype(np.float32)
    ref = oracle_incoherent(p, fb, ddm, nchan, ndec)
    q = cdmt.cdmt_incoherent_query(plan, ddm, nt)
    R, nfine, nout = q["shift_range"], len(ddm), q["nt_out"]
    assert 0 < R and 2 * R <= min(sizes)
    wrows = R + max(sizes)
    win = torch.zeros((ndm, wrows, nch), dtype=torch.float32, device="cuda")
    d_ts = torch.full((ndm, nfine, nout), -7.0, dtype=torch.float32, device="cuda")
    ws = torch.empty(max(256, q["workspace_bytes"]), dtype=torch.uint8, device="cuda")
    d_fb = torch.from_numpy(fb).cuda()
    row0, done = 0, 0
    for i, n in enumerate(sizes):
        win[:, R:R + n] = d_fb[:, row0:row0 + n]        # stands for cdmt_execute writing the group's rows
        first = i == 0
        src = win[:, R:] if first else win
        nt_in = n if first else R + n
        cdmt.cdmt_incoherent_dedisperse(plan, src.data_ptr(), wrows * nch, nt_in, ddm, d_ts.data_ptr() + 4 * done,
                                        nfine * nout, nout, ws, ws.numel())
        done += nt_in - R
        # the window's last R rows (rows [R + n - R, R + n) of the buffer) become its first
        cdmt.cdmt_incoherent_carry(plan, win, wrows * nch, R + n, R)
        row0 += n
    torch.cuda.synchronize()
    assert done == nout
    got = d_ts.cpu().numpy()
    for d in range(ndm):
        assert np.array_equal(got[d], ref[d]["ts"]), d
    bf, pf = cdmt.cdmt_incoherent_work(plan, ddm, nt)
    assert bf == ndm * nfine * nch * nout and pf > 0


def test_incoherent_argument_checks(cdmt):
    plan, _ = make_plan(cdmt, 2, 8, 1, 1)
    fb = torch.zeros((1, 400, 16), dtype=torch.float32, device="cuda")
    ddm = np.array([-0.1, 0.0, 0.1])
    q = cdmt.cdmt_incoherent_query(plan, ddm, 400)
    ts = torch.zeros((1, 3, q["nt_out"]), dtype=torch.float32, device="cuda")
    ws = torch.zeros(max(256, q["workspace_bytes"]), dtype=torch.uint8, device="cuda")

    def call(**o):
        a = dict(d_fb=fb, fb_stride_dm=400 * 16, nt_in=400, ddm=ddm, d_ts=ts, ts_stride_dm=3 * q["nt_out"],
                 ts_pitch=q["nt_out"], ws=ws, nws=ws.numel())
        a.update(o)
        cdmt.cdmt_incoherent_dedisperse(plan, a["d_fb"], a["fb_stride_dm"], a["nt_in"], a["ddm"], a["d_ts"],
                                        a["ts_stride_dm"], a["ts_pitch"], a["ws"], a["nws"])

    call()
    for over, status in [(dict(d_fb=None), cdmt.ERR_ARG), (dict(d_ts=None), cdmt.ERR_ARG),
                         (dict(ddm=np.array([0.1, 0.0])), cdmt.ERR_ARG), (dict(ddm=np.array([0.0, np.nan])), cdmt.ERR_ARG),
                         (dict(nt_in=q["shift_range"]), cdmt.ERR_SIZE), (dict(fb_stride_dm=100), cdmt.ERR_SIZE),
                         (dict(ts_pitch=q["nt_out"] - 1), cdmt.ERR_SIZE), (dict(nws=8), cdmt.ERR_WORKSPACE)]:
        with pytest.raises(cdmt.CdmtError) as e:
            call(**over)
        assert e.value.status == status, over
