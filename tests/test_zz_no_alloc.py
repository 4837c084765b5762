"""cdmt_redigitize_static: the redigitisation entry point that allocates nothing (block sums in a file-scope
device array of the library, 4 MiB) against the existing cdmt_redigitize (caller's workspace).

Both run the same three kernels on the same float32 filterbank, so codes, offsets and scales must be
IDENTICAL, bit for bit (the bar of tests/test_gpu_redigitize.py for the quantised decision).  Two calls in a
row on different data and a different shape: the array keeps the first call's contents and the second call
must not see them.  A batch beyond the fixed scratch is refused with a status, before anything is launched.

This file sorts last on purpose (pytest -x: a failure here hides nothing else) and needs
nothing from the other tests: it passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def cdmt():
    from paper_1607_00909_b200 import cdmt as m
    assert torch.cuda.is_available()
    return m


def make_plan(cdmt, nsub, nchan, ndm, vd=8, ndec=2):
    """nsub*nchan channels, Vd = vd integrated samples per block (M = 512, the rest of a block is overlap)."""
    M = 512
    fcen = 120.0 + 0.1953125 * (np.arange(nsub) + 0.5)
    plan = cdmt.cdmt_plan_create(nsub=nsub, fcen_mhz=fcen, bw_mhz=0.1953125, nfft=M * nchan,
                                 noverlap=(M - vd * ndec) * nchan, nchan=nchan, ndec=ndec, dm=np.arange(ndm) * 1.0)
    assert cdmt.cdmt_plan_query(plan, M * nchan)["nout_per_chan"] == vd
    return plan


def filterbank(seed, ndm, nt, nch):
    """Integrated Stokes-I like samples (chi-square), channel-dependent level, one bright row, one dead channel."""
    rng = np.random.default_rng(seed)
    fb = rng.chisquare(32, size=(ndm, nt, nch)) * (0.5 + rng.random(nch))
    fb[:, nt // 3, :] *= 6.0
    fb[:, :, 2] = 3.5
    return torch.from_numpy(fb.astype(np.float32)).cuda()


def outputs(ndm, nt, nch):
    return (torch.full((ndm, nt, nch), 255, dtype=torch.uint8, device="cuda"),
            torch.full((ndm, nch), float("nan"), dtype=torch.float32, device="cuda"),
            torch.full((ndm, nch), float("nan"), dtype=torch.float32, device="cuda"))


def both_paths(cdmt, plan, d_fb, nblock):
    ndm, nt, nch = d_fb.shape
    # existing path: caller's workspace
    c0, o0, s0 = outputs(ndm, nt, nch)
    nws = cdmt.cdmt_redigitize_workspace_bytes(plan, nblock)
    ws = torch.empty(max(nws, 256), dtype=torch.uint8, device="cuda")
    cdmt.cdmt_redigitize(plan, d_fb, nt * nch, nblock, 64.0, 16.0, c0, nt * nch, o0, s0, ws, ws.numel())
    # new path: the library's static scratch
    assert nws <= cdmt.cdmt_redigitize_static_max_bytes()
    c1, o1, s1 = outputs(ndm, nt, nch)
    cdmt.cdmt_redigitize_static(plan, d_fb, nt * nch, nblock, 64.0, 16.0, c1, nt * nch, o1, s1)
    torch.cuda.synchronize()
    assert cdmt.cdmt_last_launch_count(plan) == 3
    assert not bool(torch.isnan(o1).any()) and not bool(torch.isnan(s1).any())
    assert torch.equal(o0, o1) and torch.equal(s0, s1)
    assert torch.equal(c0, c1)
    assert int(c1.min()) < 255 and float(c1.float().std()) > 1.0      # real codes, not the fill value
    return c1


def test_static_scratch_matches_the_workspace_path_on_two_calls_in_a_row(cdmt):
    assert cdmt.cdmt_redigitize_static_max_bytes() == 4 << 20
    # call 1: 3 DMs x 12 blocks x 640 channels = 23040 entries (368 KB of the 4 MiB)
    plan1 = make_plan(cdmt, nsub=40, nchan=16, ndm=3)
    both_paths(cdmt, plan1, filterbank(1, 3, 12 * 8, 640), 12)
    # call 2: other data, other shape (the entries of call 1 are still in the array, laid out differently);
    # 5 x 7 x 50 channels -- not a multiple of 4: the scalar variants of the kernels
    plan2 = make_plan(cdmt, nsub=25, nchan=2, ndm=5)
    both_paths(cdmt, plan2, filterbank(2, 5, 7 * 8, 50), 7)
    # and the first shape again on new data: same plan, same stream, straight after
    both_paths(cdmt, plan1, filterbank(3, 3, 12 * 8, 640), 12)


def test_static_scratch_refuses_what_does_not_fit(cdmt):
    # 64 DMs x 40 blocks x 640 channels x 16 bytes = 26 MB > 4 MiB
    plan = make_plan(cdmt, nsub=40, nchan=16, ndm=64)
    nblock, nt, nch = 40, 40 * 8, 640
    assert cdmt.cdmt_redigitize_workspace_bytes(plan, nblock) > cdmt.cdmt_redigitize_static_max_bytes()
    d_fb = torch.zeros((64, nt, nch), dtype=torch.float32, device="cuda")
    codes, off, sc = outputs(64, nt, nch)
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_redigitize_static(plan, d_fb, nt * nch, nblock, 64.0, 16.0, codes, nt * nch, off, sc)
    assert e.value.status == cdmt.ERR_WORKSPACE
    torch.cuda.synchronize()
    assert int(codes.min()) == 255                                     # nothing was launched
    # the largest batch that fits exactly: 64 x 4 x 1024 channels x 16 bytes = 4 MiB
    plan = make_plan(cdmt, nsub=64, nchan=16, ndm=64)
    assert cdmt.cdmt_redigitize_workspace_bytes(plan, 4) == cdmt.cdmt_redigitize_static_max_bytes()
    both_paths(cdmt, plan, filterbank(4, 64, 4 * 8, 1024), 4)
