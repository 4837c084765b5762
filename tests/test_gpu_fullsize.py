"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

c2 is compared in full.  For c3, c4 and c5 the GPU processes the whole observation (into a
NaN-filled output: every element must have been written) and the oracle recomputes a stratified
sample of (subband, block) units one by one -- units are independent, so per-unit parity is exact
evidence -- with every DM trial of each sampled unit.  The sample holds at least
one unit of every subband, every block index, both edge blocks of the lowest and highest subband
and the blocks that contain the injected impulses.  Bar: max |delta| <= 1e-3 x rms (north_star),
rms taken over the sampled oracle values of that DM; peak positions of injected signals equal.
c3 -- the bench workload -- also carries the N1 (8-bit) and N2 (incoherent) stages at the shape the
bench times.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import cdmt_oracle as orc            # noqa: E402
import cdmt_synth as synth          # noqa: E402

TOL = 1e-3


@pytest.fixture(scope="module")
def cdmt():
    from paper_1607_00909_b200 import cdmt as m
    assert torch.cuda.is_available()
    return m


def upload(cfg, subbands=None, threads=16, units=None):
    """Generate on the host subband by subband and copy to the device.  Keeps the subbands the caller asks
    for (`subbands`: None = all), or -- with `units` -- only the input blocks of those (s, b) units."""
    from concurrent.futures import ThreadPoolExecutor
    int8 = cfg.in_dtype == synth.IN_CI8
    shape = (cfg.nsub, 2, cfg.nsamp, 2) if int8 else (cfg.nsub, 2, cfg.nsamp)
    d_in = torch.empty(shape, dtype=torch.int8 if int8 else torch.complex64, device="cuda")
    keep = {}
    by_sub = {}
    for (s, b) in units or []:
        by_sub.setdefault(s, []).append(b)
    with ThreadPoolExecutor(threads) as ex:
        for s, xs in zip(range(cfg.nsub), ex.map(lambda s: synth.generate_subband(cfg, s), range(cfg.nsub))):
            d_in[s].copy_(torch.from_numpy(xs))
            if units is not None:
                for b in by_sub.get(s, []):
                    keep[(s, b)] = xs[:, b * cfg.step:b * cfg.step + cfg.nfft].copy()
            elif subbands is None or s in subbands:
                keep[s] = xs
    torch.cuda.synchronize()
    return d_in, keep


def unit_sample(cfg, pulse_subband_stride=1, seed=0):
    """Stratified (s, b) sample of SURVEY.md 8(d): at least one unit of EVERY subband, every block index,
    the four corner units (both edge blocks of the lowest and highest subband) and the units that hold an
    injected impulse (on every `pulse_subband_stride`-th subband).  Returns (units, pulse_units)."""
    S, B = cfg.nsub, cfg.nblock
    units = {(0, 0), (S - 1, B - 1), (0, B - 1), (S - 1, 0), (S // 2, B // 2)}
    rng = np.random.default_rng(seed)
    off = int(rng.integers(B))
    for i in range(max(S, B)):              # a diagonal walk: covers every subband and every block index
        units.add((i % S, (i + off) % B))
    pulse_units = []
    for imp in cfg.impulses:
        # block whose kept region holds the pulse arrival (REF_CHANNEL: the same sample in every channel)
        b = min(B - 1, max(0, (imp.n0 - cfg.noverlap // 2) // cfg.step))
        for s in sorted(set(range(0, S, pulse_subband_stride)) | {S - 1}):
            units.add((s, b))
            pulse_units.append((s, b, imp))
    units = sorted(units)
    assert {s for s, _ in units} == set(range(S)) and {b for _, b in units} == set(range(B))
    return units, pulse_units


def gpu_unit_slice(out, cfg, s, b, b0=0):
    """[ndm][Vd][C] ascending-frequency view of one unit from a filterbank that starts at block b0."""
    Vd, C, nch = cfg.nvalid_dec, cfg.nchan, cfg.nsub * cfg.nchan
    lo = nch - 1 - (s * C + C - 1)
    sl = out[:, (b - b0) * Vd:(b - b0 + 1) * Vd, lo:lo + C]
    return torch.flip(sl, dims=[2]).cpu().numpy()


def compare_units(cfg, got_units, ref_units):
    """Per DM: max |delta| over the sampled units <= TOL x rms of the sampled oracle values."""
    got = np.stack(got_units).astype(np.float64)       # [unit][dm][q][c]
    ref = np.stack(ref_units)
    worst = 0.0
    for d in range(cfg.ndm):
        rms = np.sqrt(np.mean(ref[:, d] ** 2))
        err = np.abs(got[:, d] - ref[:, d]).max()
        assert err <= TOL * rms, "DM %d: max|d| %g rms %g" % (d, err, rms)
        worst = max(worst, err / rms)
    return worst


def check_pulse_peaks(cfg, units, pulse_units, got_units, ref_units):
    """north_star: identical peak positions on injected pulses.  SURVEY Q17: per DM trial, the position of
    the first maximum over time of the power summed over the subband's channels must be the oracle's,
    wherever the oracle's maximum is clear (top-2 margin > 2e-3 x rms of that trial's row).
    Impulse configs: the units holding an impulse; pulse-train config (c3): every sampled unit.
    Returns the number of (unit, DM trial) rows whose peak position was compared."""
    idx = {u: i for i, u in enumerate(units)}
    todo = [(s, b) for (s, b, _) in pulse_units]
    if cfg.pulse_train is not None:
        todo += list(units)
    checked = 0
    for (s, b) in todo:
        g = got_units[idx[(s, b)]].sum(-1)             # [dm][q] summed over the subband's channels
        r = ref_units[idx[(s, b)]].sum(-1)
        top = np.sort(r, axis=1)
        clear = top[:, -1] - top[:, -2] > 2e-3 * np.sqrt(np.mean(r ** 2, axis=1))
        assert np.array_equal(g.argmax(axis=1)[clear], r.argmax(axis=1)[clear]), (s, b)
        checked += int(clear.sum())
    return checked


def assert_all_written(out):
    """The output was NaN-filled before the execute: every element of every plane must have been written."""
    assert not bool(torch.isnan(out).any())


def run_blocks(cdmt, plan, cfg, d_in, out, ws, b0, nb):
    esz = 2 if cfg.in_dtype == synth.IN_CI8 else 8
    ns = (nb - 1) * cfg.step + cfg.nfft
    cdmt.cdmt_execute(plan, d_in.data_ptr() + b0 * cfg.step * esz, ns, cfg.nsamp, out, out[0].numel(), ws, ws.numel())


def test_c2_full(cdmt):
    cfg = synth.make_config("c2")
    d_in, keep = upload(cfg)
    x = np.stack([keep[s] for s in range(cfg.nsub)])
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    out = cdmt.run_on_device(plan, d_in, cfg.nsamp)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    want = orc.run(orc.Params(**cfg.plan_kwargs()), x)
    for d in range(cfg.ndm):
        rms = float(np.sqrt(np.mean(want[d].astype(np.float64) ** 2)))
        assert float(np.abs(got[d] - want[d]).max()) <= TOL * rms, d
    # injected impulses: position of the channel-summed maximum near each pulse, at its nearest DM trial
    for imp in cfg.impulses:
        d = int(np.argmin(np.abs(cfg.dm - imp.dm)))
        tau = (imp.n0 - cfg.noverlap // 2) // (cfg.nchan * cfg.ndec)
        lo, hi = max(0, tau - 64), min(got.shape[1], tau + 64)
        assert int(got[d, lo:hi].sum(-1).argmax()) == int(want[d, lo:hi].sum(-1).argmax())


def oracle_units(cfg, units, keep):
    blocks = np.stack([keep[u] for u in units])
    return list(orc.units(orc.Params(**cfg.plan_kwargs()), [s for s, _ in units], blocks))


def nan_filled(shape):
    return torch.full(shape, float("nan"), dtype=torch.float32, device="cuda")


def test_c3_stratified_units_then_redigitize_and_incoherent_at_bench_shape(cdmt):
    """c3 as bench.py runs it (whole output resident): parity on a sample that holds every subband and every
    block index; peak positions of the pulse train; then N1 and N2 at the shape the bench times
    (4608 channels x 8064 samples x 96 planes, 251 fine offsets), a few planes against the oracle."""
    cfg = synth.make_config("c3")
    units, pulse_units = unit_sample(cfg, seed=11)
    assert len(units) >= cfg.nsub
    d_in, keep = upload(cfg, units=units)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
    nt, nch = q["nout_per_chan"], cfg.nsub * cfg.nchan
    out = nan_filled((cfg.ndm, nt, nch))
    segsum = torch.empty(cdmt.cdmt_redigitize_workspace_bytes(plan, cfg.nblock) // 8, dtype=torch.float64, device="cuda")
    ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device="cuda")
    cdmt.cdmt_execute_sums(plan, d_in, cfg.nsamp, cfg.nsamp, out, nt * nch, segsum, ws, ws.numel())
    torch.cuda.synchronize()
    assert_all_written(out)
    got_units = [gpu_unit_slice(out, cfg, s, b) for s, b in units]
    ref = oracle_units(cfg, units, keep)
    compare_units(cfg, got_units, ref)
    assert check_pulse_peaks(cfg, units, pulse_units, got_units, ref) >= len(units) * cfg.ndm // 2
    del d_in, ws

    # ---- N1 at the bench shape: statistics and codes of three planes against the oracle
    d_codes = torch.empty((cfg.ndm, nt, nch), dtype=torch.uint8, device="cuda")
    d_off = torch.empty((cfg.ndm, nch), dtype=torch.float32, device="cuda")
    d_sc = torch.empty((cfg.ndm, nch), dtype=torch.float32, device="cuda")
    cdmt.cdmt_redigitize_sums(plan, out, nt * nch, cfg.nblock, 64.0, 16.0, segsum, d_codes, nt * nch, d_off, d_sc)
    torch.cuda.synchronize()
    planes = [0, 42, cfg.ndm - 1]
    for d in planes:
        fb = out[d].cpu().numpy()[None]
        r = orc.redigitize(fb, cfg.nblock)
        off, sc = d_off[d].cpu().numpy()[None], d_sc[d].cpu().numpy()[None]
        np.testing.assert_allclose(sc, r["scale"], rtol=2e-7, atol=0)
        np.testing.assert_allclose(off, r["offset"], rtol=2e-7, atol=2e-7 * float(np.abs(r["mean"]).max()))
        codes = d_codes[d].cpu().numpy()[None]
        assert np.array_equal(codes, orc.quantize(fb, off, sc))                 # bit-exact decision
        diff = np.abs(codes.astype(np.int16) - r["codes"].astype(np.int16))
        assert diff.max() <= 1 and (diff != 0).mean() <= 1e-4
    del segsum

    # ---- N2 at the bench shape, bit exact: the 8-bit codes as float32 are integers, so every order of the
    #      additions gives the same sums (4608 x 255 < 2^24)
    out.copy_(d_codes)
    del d_codes
    dm_step = float(cfg.dm[1] - cfg.dm[0])
    nhalf = int(round(0.5 * dm_step / 0.002))
    ddm = np.round(np.arange(-nhalf, nhalf + 1) * 0.002, 9)
    assert len(ddm) == 251
    qi = cdmt.cdmt_incoherent_query(plan, ddm, nt)
    d_ts = nan_filled((cfg.ndm, len(ddm), qi["nt_out"]))
    iws = torch.empty(max(256, qi["workspace_bytes"]), dtype=torch.uint8, device="cuda")
    cdmt.cdmt_incoherent_dedisperse(plan, out, nt * nch, nt, ddm, d_ts, d_ts[0].numel(), qi["nt_out"], iws, iws.numel())
    torch.cuda.synchronize()
    assert_all_written(d_ts)
    p = orc.Params(**cfg.plan_kwargs())
    fch = orc.channel_frequencies(p)
    tsamp = cfg.nchan * cfg.ndec / (cfg.bw_mhz * 1e6)
    for d in (0, cfg.ndm - 1):
        r = orc.incoherent(out[d].cpu().numpy(), fch, tsamp, ddm)
        assert r["range"] == qi["shift_range"] and r["smin"] == qi["shift_min"]
        assert np.array_equal(d_ts[d].cpu().numpy(), r["ts"])


def test_c4_stratified_units(cdmt):
    """c4 (nfft 262144, M 8192, ndec 32, DM to 995): every subband, every block index, and the blocks that
    hold the three injected impulses on every subband."""
    cfg = synth.make_config("c4")
    units, pulse_units = unit_sample(cfg, seed=11)
    d_in, keep = upload(cfg, units=units)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
    out = nan_filled((cfg.ndm, q["nout_per_chan"], cfg.nsub * cfg.nchan))
    cdmt.run_on_device(plan, d_in, cfg.nsamp, out=out)
    torch.cuda.synchronize()
    assert_all_written(out)
    got_units = [gpu_unit_slice(out, cfg, s, b) for s, b in units]
    del out
    ref = oracle_units(cfg, units, keep)
    compare_units(cfg, got_units, ref)
    assert check_pulse_peaks(cfg, units, pulse_units, got_units, ref) >= len(pulse_units) * cfg.ndm // 2


def test_c5_int8_block_groups(cdmt):
    """c5's 136 GB of filterbanks do not fit: block groups run through one output buffer, as in bench.py.
    Every block index (hence every subband twice) plus the impulse blocks on every 8th subband."""
    cfg = synth.make_config("c5")
    units, pulse_units = unit_sample(cfg, pulse_subband_stride=8, seed=12)
    d_in, keep = upload(cfg, units=units)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    nb_group = 32
    nch = cfg.nsub * cfg.nchan
    out = torch.empty((cfg.ndm, nb_group * cfg.nvalid_dec, nch), dtype=torch.float32, device="cuda")
    ws = torch.empty(cdmt.cdmt_plan_query(plan, (nb_group - 1) * cfg.step + cfg.nfft)["workspace_bytes"],
                     dtype=torch.uint8, device="cuda")
    got = {}
    for b0 in range(0, cfg.nblock, nb_group):
        nb = min(nb_group, cfg.nblock - b0)
        out.fill_(float("nan"))
        run_blocks(cdmt, plan, cfg, d_in, out, ws, b0, nb)
        torch.cuda.synchronize()
        assert_all_written(out[:, :nb * cfg.nvalid_dec])
        for (s, b) in units:
            if b0 <= b < b0 + nb:
                got[(s, b)] = gpu_unit_slice(out, cfg, s, b, b0)
    got_units = [got[u] for u in units]
    ref = oracle_units(cfg, units, keep)
    compare_units(cfg, got_units, ref)
    assert check_pulse_peaks(cfg, units, pulse_units, got_units, ref) >= len(pulse_units) * cfg.ndm // 2


def test_subband_reference_mode_c2_sample(cdmt):
    """The REF_SUBBAND reading of Eq. 1 (Q3): phases of thousands of cycles."""
    cfg = synth.make_config("c2")
    units = [(0, 0), (19, 17), (7, 9), (12, 3)]
    keep = {s: synth.generate_subband(cfg, s, chirp_ref=synth.REF_SUBBAND) for s in {u[0] for u in units}}
    d_in = torch.empty((cfg.nsub, 2, cfg.nsamp), dtype=torch.complex64, device="cuda").zero_()
    for s, xs in keep.items():
        d_in[s].copy_(torch.from_numpy(xs))
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs(synth.REF_SUBBAND))
    out = cdmt.run_on_device(plan, d_in, cfg.nsamp)
    torch.cuda.synchronize()
    got_units = [gpu_unit_slice(out, cfg, s, b) for s, b in units]
    blocks = np.stack([keep[s][:, b * cfg.step:b * cfg.step + cfg.nfft] for s, b in units])
    ref = orc.units(orc.Params(**cfg.plan_kwargs(synth.REF_SUBBAND)), [s for s, _ in units], blocks)
    compare_units(cfg, got_units, list(ref))


@pytest.mark.parametrize("name", ["c3", "c4", "c5"])
def test_every_unit_of_a_config_when_asked(cdmt, name):
    """Opt-in (CDMT_FULL_PARITY=c3,c4,c5; about 11 / 13 / 80 minutes of oracle time on 16 host cores): EVERY
    (subband, block) unit of the config -- not a sample -- against the oracle, subband by subband in runs of
    up to 42 blocks, all DM trials, at north_star's 1e-3 x rms (rms over the run's units of that trial),
    with the peak positions of every clear maximum.  The whole filterbank set is resident (c5: 136 GB).
    The results of the round's runs are recorded in DESIGN.md section 3 and profiles/r2_full_parity.md."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    if name not in os.environ.get("CDMT_FULL_PARITY", "").split(","):
        pytest.skip("set CDMT_FULL_PARITY=%s to run" % name)
    cfg = synth.make_config(name)
    d_in, _ = upload(cfg, subbands=[])
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
    nt, nch = q["nout_per_chan"], cfg.nsub * cfg.nchan
    out = nan_filled((cfg.ndm, nt, nch))
    ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device="cuda")
    cdmt.cdmt_execute(plan, d_in, cfg.nsamp, cfg.nsamp, out, nt * nch, ws, ws.numel())
    torch.cuda.synchronize()
    assert_all_written(out)
    del d_in, ws
    p = orc.Params(**cfg.plan_kwargs())
    worst, nunits, npeaks = 0.0, 0, 0
    # CDMT_FULL_PARITY_SUBBANDS=a:b:step restricts the oracle side to those subbands, every block of each (a
    # GPU call on this pool is limited to an hour; c5 in full needs about 90 minutes of oracle time)
    sel = os.environ.get("CDMT_FULL_PARITY_SUBBANDS", "")
    subs = list(range(cfg.nsub))
    if sel:
        a, b, st = (int(v) for v in (sel.split(":") + ["1"])[:3])
        subs = list(range(a, min(b, cfg.nsub), st))
    with ThreadPoolExecutor(2) as ex:
        nxt = ex.submit(synth.generate_subband, cfg, subs[0])
        for i, s in enumerate(subs):
            xs = nxt.result()
            if i + 1 < len(subs):
                nxt = ex.submit(synth.generate_subband, cfg, subs[i + 1])
            for b0 in range(0, cfg.nblock, 42):
                bs = range(b0, min(cfg.nblock, b0 + 42))
                blocks = np.stack([xs[:, b * cfg.step:b * cfg.step + cfg.nfft] for b in bs])
                ref = np.stack(list(orc.units(p, [s] * len(bs), blocks)))          # [block][dm][q][c]
                got = np.stack([gpu_unit_slice(out, cfg, s, b) for b in bs]).astype(np.float64)
                rms = np.sqrt(np.mean(ref ** 2, axis=(0, 2, 3)))                   # per DM trial
                err = np.abs(got - ref).max(axis=(0, 2, 3))
                assert (err <= TOL * rms).all(), (s, b0, float((err / rms).max()))
                worst = max(worst, float((err / rms).max()))
                g, r = got.sum(-1), ref.sum(-1)                                    # [block][dm][q]
                top = np.sort(r, axis=2)
                clear = top[..., -1] - top[..., -2] > 2e-3 * np.sqrt(np.mean(r ** 2, axis=2))
                assert np.array_equal(g.argmax(axis=2)[clear], r.argmax(axis=2)[clear]), (s, b0)
                npeaks += int(clear.sum())
                nunits += len(bs)
    assert nunits == len(subs) * cfg.nblock
    print("\n%s: %s %d units x %d DM trials: max |delta| / rms = %.3g; %d peak positions equal" % (
        name, "all" if len(subs) == cfg.nsub else "every block of subbands %s:" % sel, nunits, cfg.ndm, worst, npeaks))
