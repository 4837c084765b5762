"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

c2 is compared in full.  For c3, c4 and c5 the GPU processes the whole observation and the
oracle recomputes a stratified sample of (subband, block) units one by one -- units are
independent, so per-unit parity is exact evidence -- with every DM trial of each sampled unit.
The sample always holds both edge blocks, the lowest and highest subband and, where the config
injects impulses, the blocks that contain them.  Bar: max |delta| <= 1e-3 x rms (north_star),
rms taken over the sampled oracle values of that DM; peak positions of injected pulses equal.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import cdmt_oracle as orc            # noqa: E402
from paper_1607_00909_b200 import synth          # noqa: E402

TOL = 1e-3


@pytest.fixture(scope="module")
def cdmt():
    from paper_1607_00909_b200 import cdmt as m
    assert torch.cuda.is_available()
    return m


def upload(cfg, subbands=None, threads=16):
    """Generate on the host subband by subband and copy to the device; keep what the caller asks for."""
    from concurrent.futures import ThreadPoolExecutor
    int8 = cfg.in_dtype == synth.IN_CI8
    shape = (cfg.nsub, 2, cfg.nsamp, 2) if int8 else (cfg.nsub, 2, cfg.nsamp)
    d_in = torch.empty(shape, dtype=torch.int8 if int8 else torch.complex64, device="cuda")
    keep = {}
    with ThreadPoolExecutor(threads) as ex:
        for s, xs in zip(range(cfg.nsub), ex.map(lambda s: synth.generate_subband(cfg, s), range(cfg.nsub))):
            d_in[s].copy_(torch.from_numpy(xs))
            if subbands is None or s in subbands:
                keep[s] = xs
    torch.cuda.synchronize()
    return d_in, keep


def unit_sample(cfg, n_random, seed):
    """(s, b) units: corners, impulse blocks on a few subbands, plus random ones."""
    S, B = cfg.nsub, cfg.nblock
    units = {(0, 0), (S - 1, B - 1), (0, B - 1), (S - 1, 0), (S // 2, B // 2)}
    pulse_units = []
    for imp in cfg.impulses:
        # block whose kept region holds the pulse arrival at the subband centre
        b = min(B - 1, max(0, (imp.n0 - cfg.noverlap // 2) // cfg.step))
        for s in (0, S // 3, S - 1):
            units.add((s, b))
            pulse_units.append((s, b, imp))
    rng = np.random.default_rng(seed)
    while len(units) < n_random + 5 + len(pulse_units):
        units.add((int(rng.integers(S)), int(rng.integers(B))))
    return sorted(units), pulse_units


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
    idx = {u: i for i, u in enumerate(units)}
    for (s, b, imp) in pulse_units:
        g = got_units[idx[(s, b)]].sum(-1)             # [dm][q] summed over the subband's channels
        r = ref_units[idx[(s, b)]].sum(-1)
        # compare the position of the maximum over (dm, q) where the oracle's maximum is clear
        flat = np.sort(r.ravel())
        if flat[-1] - flat[-2] > 2e-3 * np.sqrt(np.mean(r ** 2)):
            assert np.unravel_index(g.argmax(), g.shape) == np.unravel_index(r.argmax(), r.shape), (s, b, imp)


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


@pytest.mark.parametrize("name,nrand", [("c3", 20), ("c4", 6)])
def test_sampled_units_whole_output_resident(cdmt, name, nrand):
    cfg = synth.make_config(name)
    units, pulse_units = unit_sample(cfg, nrand, seed=11)
    d_in, keep = upload(cfg, subbands={s for s, _ in units})
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    out = cdmt.run_on_device(plan, d_in, cfg.nsamp)
    torch.cuda.synchronize()
    got_units = [gpu_unit_slice(out, cfg, s, b) for s, b in units]
    del out
    blocks = np.stack([keep[s][:, b * cfg.step:b * cfg.step + cfg.nfft] for s, b in units])
    ref = orc.units(orc.Params(**cfg.plan_kwargs()), [s for s, _ in units], blocks)
    compare_units(cfg, got_units, list(ref))
    check_pulse_peaks(cfg, units, pulse_units, got_units, list(ref))


def test_c5_int8_block_groups(cdmt):
    """c5's 136 GB of filterbanks do not fit: block groups run through one output buffer, as in bench.py."""
    cfg = synth.make_config("c5")
    units, pulse_units = unit_sample(cfg, 4, seed=12)
    units = units[:14]
    pulse_units = [p for p in pulse_units if (p[0], p[1]) in units]
    d_in, keep = upload(cfg, subbands={s for s, _ in units})
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    nb_group = 32
    nch = cfg.nsub * cfg.nchan
    out = torch.empty((cfg.ndm, nb_group * cfg.nvalid_dec, nch), dtype=torch.float32, device="cuda")
    ws = torch.empty(cdmt.cdmt_plan_query(plan, (nb_group - 1) * cfg.step + cfg.nfft)["workspace_bytes"],
                     dtype=torch.uint8, device="cuda")
    got = {}
    for b0 in range(0, cfg.nblock, nb_group):
        nb = min(nb_group, cfg.nblock - b0)
        if not any(b0 <= b < b0 + nb for _, b in units):
            continue
        run_blocks(cdmt, plan, cfg, d_in, out, ws, b0, nb)
        torch.cuda.synchronize()
        for (s, b) in units:
            if b0 <= b < b0 + nb:
                got[(s, b)] = gpu_unit_slice(out, cfg, s, b, b0)
    got_units = [got[u] for u in units]
    blocks = np.stack([keep[s][:, b * cfg.step:b * cfg.step + cfg.nfft] for s, b in units])
    ref = orc.units(orc.Params(**cfg.plan_kwargs()), [s for s, _ in units], blocks)
    compare_units(cfg, got_units, list(ref))
    check_pulse_peaks(cfg, units, pulse_units, got_units, list(ref))


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
