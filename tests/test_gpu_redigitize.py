"""GPU parity of cdmt_redigitize (Alg. 1 l.104-106) against the oracle.

What is compared, and how (the quantised code is an integer decided by floating point):
  * offset / scale come from fp64 block sums on both sides; the summation order differs, so
    they are compared to 2e-7 relative (float32 rounding of values equal to ~1e-15);
  * the decision itself is taken in float32 on both sides: on the offsets and scales the GPU
    reports, oracle.quantize must reproduce the GPU's codes BIT FOR BIT;
  * the whole chain against oracle.redigitize on the same float32 filterbank: codes may differ
    by one unit only where offset/scale differ in the last bit -- at most 1e-4 of the samples.
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


def plan_for(cdmt, nsub, nchan, ndm, vd=8, ndec=2):
    """A plan whose geometry gives nsub*nchan channels and Vd = vd samples per block:
    M = 512 (1024), V = vd*ndec kept samples, the rest of each block is overlap."""
    M = 512 if vd * ndec < 512 else 1024
    nfft = M * nchan
    noverlap = (M - vd * ndec) * nchan
    fcen = 120.0 + 0.1953125 * (np.arange(nsub) + 0.5)
    plan = cdmt.cdmt_plan_create(nsub=nsub, fcen_mhz=fcen, bw_mhz=0.1953125, nfft=nfft, noverlap=noverlap,
                                 nchan=nchan, ndec=ndec, dm=np.arange(ndm) * 1.0)
    assert cdmt.cdmt_plan_query(plan, nfft)["nout_per_chan"] == vd
    return plan


def gpu_redigitize(cdmt, plan, fb, nblock, qmean=64.0, qstd=16.0, pad=0):
    ndm, nt, nch = fb.shape
    d_fb = torch.zeros((ndm, nt * nch + pad), dtype=torch.float32, device="cuda")
    d_fb[:, :nt * nch] = torch.from_numpy(fb.reshape(ndm, -1)).cuda()
    d_codes = torch.full((ndm, nt * nch + pad), 255, dtype=torch.uint8, device="cuda")
    d_off = torch.empty((ndm, nch), dtype=torch.float32, device="cuda")
    d_sc = torch.empty((ndm, nch), dtype=torch.float32, device="cuda")
    nws = cdmt.cdmt_redigitize_workspace_bytes(plan, nblock)
    ws = torch.empty(max(nws, 256), dtype=torch.uint8, device="cuda")
    cdmt.cdmt_redigitize(plan, d_fb, nt * nch + pad, nblock, qmean, qstd, d_codes, nt * nch + pad, d_off, d_sc,
                         ws, ws.numel())
    torch.cuda.synchronize()
    assert cdmt.cdmt_last_launch_count(plan) == 3
    codes = d_codes.cpu().numpy()
    if pad:
        assert (codes[:, nt * nch:] == 255).all()         # nothing written past a plane
    return codes[:, :nt * nch].reshape(ndm, nt, nch), d_off.cpu().numpy(), d_sc.cpu().numpy()


def synthetic_fb(seed, ndm, nt, nch):
    """Integrated Stokes-I like samples: chi-square with 2*ndec*... degrees of freedom per channel,
    channel-dependent level, one bright pulse, one dead (constant) channel."""
    rng = np.random.default_rng(seed)
    fb = rng.chisquare(32, size=(ndm, nt, nch)) * (0.5 + rng.random(nch))
    fb[:, nt // 3, :] *= 6.0
    if nch > 2:
        fb[:, :, 2] = 3.5
    return fb.astype(np.float32)


def compare(cdmt, plan, fb, nblock, **kw):
    codes, off, sc = gpu_redigitize(cdmt, plan, fb, nblock, **kw)
    q = {k: kw[k] for k in ("qmean", "qstd") if k in kw}
    ref = orc.redigitize(fb, nblock, **q)
    np.testing.assert_allclose(sc, ref["scale"], rtol=2e-7, atol=0)
    np.testing.assert_allclose(off, ref["offset"], rtol=2e-7, atol=2e-7 * float(np.abs(ref["mean"]).max()))
    assert np.array_equal(codes, orc.quantize(fb, off, sc))                    # bit exact decision
    diff = np.abs(codes.astype(np.int16) - ref["codes"].astype(np.int16))
    assert diff.max() <= 1
    assert (diff != 0).mean() <= 1e-4
    return codes, ref


SHAPES = [
    # nsub nchan ndm nblock vd
    (1, 8, 4, 5, 96),       # c1's channel count: float4 path, two channel groups
    (3, 16, 3, 7, 24),      # 48 channels
    (40, 16, 2, 3, 40),     # 640 channels: several channel-group CTAs, ragged last one
    (3, 1, 2, 4, 16),       # 3 channels: scalar path
    (5, 2, 1, 1, 200),      # 10 channels (not a multiple of 4): scalar path, one block
    (2, 32, 5, 9, 33),      # Vd not a multiple of the row slices
]


@pytest.mark.parametrize("shape", SHAPES)
def test_redigitize_matches_oracle(cdmt, shape):
    nsub, nchan, ndm, nblock, vd = shape
    plan = plan_for(cdmt, nsub, nchan, ndm, vd=vd)
    fb = synthetic_fb(11, ndm, nblock * vd, nsub * nchan)
    codes, ref = compare(cdmt, plan, fb, nblock)
    if nsub * nchan > 2:
        assert (codes[:, :, 2] == 64).all()            # dead channel: std = 0 -> qmean


def test_redigitize_other_targets_strided_planes_and_clipping(cdmt):
    plan = plan_for(cdmt, 2, 16, 3, vd=64)
    fb = synthetic_fb(12, 3, 6 * 64, 32)
    fb[1, 100, 5] = 1e9            # saturates at 255
    fb[2, 7, 9] = -1e9             # saturates at 0
    codes, ref = compare(cdmt, plan, fb, 6, qmean=128.0, qstd=32.0, pad=64)
    assert codes[1, 100, 5] == 255 and codes[2, 7, 9] == 0
    # the bulk of a channel sits round qmean (the bright sample row is clipped, so the code std is below qstd)
    assert abs(np.median(codes[0, :, 0].astype(np.float64)) - 128) < 12


def test_redigitize_after_execute_end_to_end(cdmt):
    """cdmt_execute -> cdmt_redigitize on the device against oracle.run -> oracle.redigitize: the two
    float32 filterbanks differ by ~1e-6 relative, so codes may differ by one unit on a small fraction."""
    cfg = synth.small_config(nsub=2, nsamp=2 ** 15, nfft=4096, noverlap=1024, nchan=8, ndec=4, dm=(0.0, 2.0, 4.0))
    x = synth.generate(cfg)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    d_in = torch.from_numpy(x).cuda()
    out = cdmt.run_on_device(plan, d_in, cfg.nsamp)
    ndm, nt, nch = out.shape
    d_codes = torch.empty((ndm, nt, nch), dtype=torch.uint8, device="cuda")
    d_off = torch.empty((ndm, nch), dtype=torch.float32, device="cuda")
    d_sc = torch.empty((ndm, nch), dtype=torch.float32, device="cuda")
    ws = torch.empty(cdmt.cdmt_redigitize_workspace_bytes(plan, cfg.nblock), dtype=torch.uint8, device="cuda")
    cdmt.cdmt_redigitize(plan, out, nt * nch, cfg.nblock, 64.0, 16.0, d_codes, nt * nch, d_off, d_sc, ws, ws.numel())
    torch.cuda.synchronize()
    fb_ref = orc.run(orc.Params(**cfg.plan_kwargs()), x)
    ref = orc.redigitize(fb_ref, cfg.nblock)
    np.testing.assert_allclose(d_sc.cpu().numpy(), ref["scale"], rtol=1e-4)
    np.testing.assert_allclose(d_off.cpu().numpy(), ref["offset"], rtol=1e-4, atol=1e-4 * float(ref["mean"].max()))
    diff = np.abs(d_codes.cpu().numpy().astype(np.int16) - ref["codes"].astype(np.int16))
    assert diff.max() <= 1 and (diff != 0).mean() < 5e-3
    # and exactly the oracle's decision on the GPU's own filterbank and statistics
    assert np.array_equal(d_codes.cpu().numpy(),
                          orc.quantize(out.cpu().numpy(), d_off.cpu().numpy(), d_sc.cpu().numpy()))


def test_redigitize_argument_checks(cdmt):
    plan = plan_for(cdmt, 1, 8, 2, vd=8)
    fb = torch.zeros((2, 16, 8), dtype=torch.float32, device="cuda")
    codes = torch.zeros((2, 16, 8), dtype=torch.uint8, device="cuda")
    off = torch.zeros((2, 8), dtype=torch.float32, device="cuda")
    sc = torch.zeros((2, 8), dtype=torch.float32, device="cuda")
    ws = torch.zeros(4096, dtype=torch.uint8, device="cuda")

    def call(**o):
        a = dict(d_fb=fb, fb_stride_dm=128, nblock=2, qmean=64.0, qstd=16.0, d_codes=codes, codes_stride_dm=128,
                 d_offset=off, d_scale=sc, d_workspace=ws, workspace_bytes=ws.numel())
        a.update(o)
        cdmt.cdmt_redigitize(plan, a["d_fb"], a["fb_stride_dm"], a["nblock"], a["qmean"], a["qstd"], a["d_codes"],
                             a["codes_stride_dm"], a["d_offset"], a["d_scale"], a["d_workspace"], a["workspace_bytes"])

    call()
    for over, status in [(dict(d_fb=None), cdmt.ERR_ARG), (dict(d_codes=None), cdmt.ERR_ARG),
                         (dict(qstd=0.0), cdmt.ERR_ARG), (dict(qstd=float("nan")), cdmt.ERR_ARG),
                         (dict(nblock=0), cdmt.ERR_SIZE), (dict(fb_stride_dm=127), cdmt.ERR_SIZE),
                         (dict(codes_stride_dm=100), cdmt.ERR_SIZE), (dict(workspace_bytes=16), cdmt.ERR_WORKSPACE)]:
        with pytest.raises(cdmt.CdmtError) as e:
            call(**over)
        assert e.value.status == status, over
