"""GPU parity: the CUDA path through the C ABI against the CPU oracle, same seeded inputs.

Tolerance (BASELINE.json north_star): max |delta| <= 1e-3 * rms of the oracle's filterbank,
per DM trial; identical peak positions on injected pulses.
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


TOL = 1e-3


def check_filterbank(got, ref, tol=TOL):
    assert got.shape == ref.shape
    worst = 0.0
    for d in range(ref.shape[0]):
        rms = float(np.sqrt(np.mean(ref[d].astype(np.float64) ** 2)))
        err = float(np.abs(got[d].astype(np.float64) - ref[d]).max())
        assert err <= tol * rms, "DM %d: max|d| = %g, rms = %g" % (d, err, rms)
        worst = max(worst, err / rms)
    return worst


def gpu_run(cdmt, cfg, x, chirp_ref=synth.REF_CHANNEL, opts=None):
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs(chirp_ref))
    for k, v in (opts or {}).items():
        cdmt.cdmt_plan_set_option(plan, k, v)
    d_in = torch.from_numpy(x).cuda()
    out = cdmt.run_on_device(plan, d_in, x.shape[2])
    torch.cuda.synchronize()
    return out.cpu().numpy(), plan


# ---------------------------------------------------------------- stage a1: unpack / segment
@pytest.mark.parametrize("in_dtype", [synth.IN_CF32, synth.IN_CI8])
def test_unpack_blocks(cdmt, in_dtype):
    cfg = synth.small_config(nsub=3, nsamp=4096 + 300, nfft=1024, noverlap=256, in_dtype=in_dtype)
    x = synth.generate(cfg)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    d_in = torch.from_numpy(x).cuda()
    B = cfg.nblock
    blocks = torch.zeros((B * cfg.nsub, 2, cfg.nfft), dtype=torch.complex64, device="cuda")
    cdmt.cdmt_unpack(plan, d_in, cfg.nsamp, cfg.nsamp, blocks)
    torch.cuda.synchronize()
    got = blocks.cpu().numpy()
    xc = x if in_dtype == synth.IN_CF32 else (x[..., 0].astype(np.float32) + 1j * x[..., 1].astype(np.float32))
    for b in range(B):
        for s in range(cfg.nsub):
            exp = xc[s, :, b * cfg.step:b * cfg.step + cfg.nfft]
            assert np.array_equal(got[b * cfg.nsub + s], exp.astype(np.complex64))   # bit exact


# ---------------------------------------------------------------- stage a2-a3: forward FFT + swap
@pytest.mark.parametrize("nfft", [256, 512, 1024, 4096, 8192, 65536, 131072, 262144])
def test_forward_spectrum(cdmt, nfft):
    nchan = 16 if nfft // 16 <= 8192 else nfft // 8192
    cfg = synth.small_config(nsub=2, nsamp=nfft + (nfft // 2) * 2, nfft=nfft, noverlap=nfft // 2,
                             nchan=nchan, ndec=1, dm=(0.0,))
    x = synth.generate(cfg)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
    B = q["nblock"]
    assert B == 3
    d_in = torch.from_numpy(x).cuda()
    spec = torch.zeros((B * cfg.nsub, 2, nfft), dtype=torch.complex64, device="cuda")
    ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device="cuda")
    cdmt.cdmt_forward_spectrum(plan, d_in, cfg.nsamp, cfg.nsamp, spec, ws, ws.numel())
    torch.cuda.synchronize()
    got = spec.cpu().numpy()
    p = orc.Params(**cfg.plan_kwargs())
    for (b, s, pol) in [(0, 0, 0), (1, 1, 1), (2, 0, 1)]:
        ref = orc.block_spectrum(p, x[s, pol], first=b * cfg.step)
        err = np.abs(got[b * cfg.nsub + s, pol] - ref).max()
        rms = np.sqrt(np.mean(np.abs(ref) ** 2))
        assert err <= 2e-6 * rms * np.log2(nfft), (nfft, err / rms)


# ---------------------------------------------------------------- whole path, small shapes
SMALL = [
    # nsub nsamp  nfft noverlap nchan ndec  (M)          comment
    (1, 2 ** 14, 4096, 1024, 8, 4),         # c1 geometry (M=512)
    (2, 4096 + 78, 1024, 256, 4, 2),        # M=256, ragged tail
    (3, 3 * 768 + 256, 1024, 256, 64, 1),   # M=16: one thread per transform
    (2, 2048, 1024, 0, 32, 4),              # M=32, no overlap
    (1, 8192, 2048, 512, 32, 3),            # M=64, ndec=3 (general decimation path); step=1536=32*3*16
    (2, 8192, 2048, 1024, 16, 8),           # M=128
    (1, 2 ** 15, 8192, 2048, 8, 16),        # M=1024
    (1, 2 ** 16, 16384, 4096, 8, 6),        # M=2048, ndec=6: step 12288 = 8*6*256
    (2, 2 ** 17, 65536, 16384, 16, 16),     # c3 geometry (M=4096)
    (1, 2 ** 17, 65536, 8192, 8, 8),        # c2 geometry (M=8192)
    (1, 2 ** 16, 32768, 2048, 4, 64),       # M=8192, ndec=64 > warp
    (1, 2 ** 13, 4096, 1024 + 16, 8, 1),    # h = 65: h % ndec irrelevant at ndec=1
    (1, 2 ** 13, 4096, 1024 + 32, 8, 2),    # h = 66, ndec = 2 ok; step 3040 = 8*2*190
    (1, 2 ** 13, 4096, 992, 8, 4),          # h = 62 -> h % ndec != 0 (general decimation path)
]


@pytest.mark.parametrize("shape", SMALL)
@pytest.mark.parametrize("ref", [synth.REF_CHANNEL, synth.REF_SUBBAND])
def test_small_shapes_full_parity(cdmt, shape, ref):
    nsub, nsamp, nfft, noverlap, nchan, ndec = shape
    if (nfft - noverlap) % (nchan * ndec) or noverlap % (2 * nchan):
        pytest.skip("shape violates the divisibility rules")
    cfg = synth.small_config(nsub=nsub, nsamp=nsamp, nfft=nfft, noverlap=noverlap, nchan=nchan,
                             ndec=ndec, dm=(0.0, 2.0, -3.5, 41.25), f_lo=121.0)
    x = synth.generate(cfg, chirp_ref=ref)
    got, _ = gpu_run(cdmt, cfg, x, ref)
    want = orc.run(orc.Params(**cfg.plan_kwargs(ref)), x)
    check_filterbank(got, want)


# ---------------------------------------------------------------- the three fused kernels agree with the oracle
X2_SHAPES = [
    # nsub nsamp     nfft  noverlap nchan ndec     M
    (2, 2 ** 17, 65536, 16384, 16, 16),   # 4096, c3 geometry
    (1, 2 ** 17, 65536, 8192, 8, 8),      # 8192, c2 / c5 geometry
    (1, 2 ** 17, 65536, 16384, 8, 32),    # 8192, ndec = 32 (c4's decimation): whole-warp groups
    (2, 2 ** 15, 16384, 4096, 8, 8),      # 2048
    (1, 2 ** 16, 32768, 8192, 16, 32),    # 2048, ndec = 32
    (1, 2 ** 17, 65536, 32768, 16, 8),    # 4096, half of every block discarded
    (1, 2 ** 17, 65536, 16384, 16, 1),    # 4096, no integration (kernel 5 only among the packed ones)
    (1, 2 ** 16, 32768, 8192, 16, 4),     # 2048, ndec = 4
]


@pytest.mark.parametrize("shape", X2_SHAPES)
@pytest.mark.parametrize("ref", [synth.REF_CHANNEL, synth.REF_SUBBAND])
def test_fused_kernel_variants(cdmt, shape, ref):
    """CDMT_OPT_FUSED_KERNEL: software-pipelined packed polarisations (5), warp-specialised packed half
    transforms with two blocks per CTA (4), packed half transforms (3), scalar fast (2) and general (1)."""
    nsub, nsamp, nfft, noverlap, nchan, ndec = shape
    cfg = synth.small_config(nsub=nsub, nsamp=nsamp, nfft=nfft, noverlap=noverlap, nchan=nchan,
                             ndec=ndec, dm=(0.0, 1.5, -3.5, 41.25, 96.0), f_lo=121.0)
    x = synth.generate(cfg, chirp_ref=ref)
    want = orc.run(orc.Params(**cfg.plan_kwargs(ref)), x)
    M = nfft // nchan
    kerns = [2, 1]
    if ndec >= 8:
        kerns.insert(0, 3)
    if M <= 4096:
        kerns.insert(0, 5)
    if M == 4096 and ndec >= 8:
        kerns.append(4)
    for kern in kerns:
        got, _ = gpu_run(cdmt, cfg, x, ref, opts={cdmt.OPT_FUSED_KERNEL: kern})
        worst = check_filterbank(got, want)
        assert worst < TOL, (kern, worst)
    if 4 in kerns:
        # kernel 4 pairs the blocks of a chunk: chunks of three blocks (the third block's CTAs run with the
        # second FFT group idle) with a DM tile that does not divide ndm, and chunks of two blocks (where
        # nblock is odd the last chunk is a lone block, which goes to kernel 3)
        for opts in ({cdmt.OPT_CHUNK_UNITS: 3 * nsub, cdmt.OPT_DM_TILE: 2}, {cdmt.OPT_CHUNK_UNITS: 2 * nsub}):
            got, _ = gpu_run(cdmt, cfg, x, ref, opts=opts)
            check_filterbank(got, want)
    # a DM tile that does not divide ndm, one unit per chunk
    got, _ = gpu_run(cdmt, cfg, x, ref, opts={cdmt.OPT_FUSED_KERNEL: kerns[0], cdmt.OPT_DM_TILE: 2,
                                             cdmt.OPT_CHUNK_UNITS: 1})
    check_filterbank(got, want)


def test_fused_kernel_choice_is_checked(cdmt):
    """Kernels 2 to 5 refuse shapes they do not cover (status, not a wrong answer)."""
    cfg = synth.small_config(nsub=1, nsamp=2 ** 13, nfft=4096, noverlap=992, nchan=8, ndec=4, dm=(0.0, 3.0))
    x = synth.generate(cfg)
    for kern in (2, 3, 4, 5):
        with pytest.raises(cdmt.CdmtError) as e:
            gpu_run(cdmt, cfg, x, opts={cdmt.OPT_FUSED_KERNEL: kern})
        assert e.value.status == cdmt.ERR_CUDA
    got, _ = gpu_run(cdmt, cfg, x)
    check_filterbank(got, orc.run(orc.Params(**cfg.plan_kwargs()), x))


def test_c1_tiny_config(cdmt):
    cfg = synth.make_config("c1")
    for ref in (synth.REF_CHANNEL, synth.REF_SUBBAND):
        x = synth.generate(cfg, chirp_ref=ref)
        got, plan = gpu_run(cdmt, cfg, x, ref)
        want = orc.run(orc.Params(**cfg.plan_kwargs(ref)), x)
        check_filterbank(got, want)
        # peak of the injected pulse: same DM trial, same sample
        gi = np.unravel_index(got.sum(-1).argmax(), got.shape[:2])
        wi = np.unravel_index(want.sum(-1).argmax(), want.shape[:2])
        assert gi == wi
        assert cfg.dm[gi[0]] == 4.0
        assert cdmt.cdmt_last_launch_count(plan) >= 3


def test_int8_input(cdmt):
    cfg = synth.small_config(nsub=2, nsamp=2 ** 15, nfft=8192, noverlap=4096, nchan=8, ndec=8,
                             dm=(0.0, 10.0, 99.9), in_dtype=synth.IN_CI8, f_lo=140.0)
    x = synth.generate(cfg)
    got, _ = gpu_run(cdmt, cfg, x)
    want = orc.run(orc.Params(**cfg.plan_kwargs()), x)
    check_filterbank(got, want)


def test_options_do_not_change_results(cdmt):
    cfg = synth.small_config(nsub=3, nsamp=2 ** 14, nfft=2048, noverlap=512, nchan=4, ndec=4,
                             dm=tuple(np.arange(7) * 1.5))
    x = synth.generate(cfg)
    base, _ = gpu_run(cdmt, cfg, x)
    want = orc.run(orc.Params(**cfg.plan_kwargs()), x)
    check_filterbank(base, want)
    for opts in ({cdmt.OPT_CHUNK_UNITS: 1}, {cdmt.OPT_CHUNK_UNITS: 5}, {cdmt.OPT_DM_TILE: 1},
                 {cdmt.OPT_DM_TILE: 3}, {cdmt.OPT_CHUNK_UNITS: 4, cdmt.OPT_DM_TILE: 2}):
        got, _ = gpu_run(cdmt, cfg, x, opts=opts)
        assert np.array_equal(got, base), opts
    acc, _ = gpu_run(cdmt, cfg, x, opts={cdmt.OPT_ACCURATE_SINCOS: 1})
    check_filterbank(acc, want)


def test_strided_input_and_output(cdmt):
    """in_stride_pol > nsamp and out_stride_dm > plane size; streaming in two calls equals one call."""
    cfg = synth.small_config(nsub=2, nsamp=8 * 768 + 256, nfft=1024, noverlap=256, nchan=4, ndec=2,
                             dm=(0.0, 5.0, 9.0))
    x = synth.generate(cfg)
    want = orc.run(orc.Params(**cfg.plan_kwargs()), x)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    d_in = torch.from_numpy(x).cuda()
    T, step = cfg.nsamp, cfg.step
    nch = cfg.nsub * cfg.nchan
    B, Vd = cfg.nblock, cfg.nvalid_dec
    out = torch.full((cfg.ndm, B * Vd + 5, nch), -1.0, dtype=torch.float32, device="cuda")
    stride_dm = (B * Vd + 5) * nch
    nb1 = 3
    ns1 = (nb1 - 1) * step + cfg.nfft
    q1 = cdmt.cdmt_plan_query(plan, ns1)
    ws = torch.empty(cdmt.cdmt_plan_query(plan, T)["workspace_bytes"], dtype=torch.uint8, device="cuda")
    assert q1["nblock"] == nb1
    cdmt.cdmt_execute(plan, d_in, ns1, T, out, stride_dm, ws, ws.numel())
    # second call: advance by nb1*step samples; output rows continue at nb1*Vd
    off = nb1 * step
    d_in2 = d_in.view(torch.float32).view(cfg.nsub, 2, T, 2)[:, :, off:, :]
    out2 = out[:, nb1 * Vd:, :]
    cdmt.cdmt_execute(plan, d_in2.data_ptr(), T - off, T, out2.data_ptr(), stride_dm, ws, ws.numel())
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    check_filterbank(got[:, :B * Vd, :], want)
    assert (got[:, B * Vd:, :] == -1.0).all()        # padding rows untouched


def test_host_path_against_the_oracle(cdmt):
    """cdmt_execute_host (pinned host buffers, double-buffered block groups) against the ORACLE, in the
    multi-group case, and bit for bit against the device-resident path."""
    cfg = synth.small_config(nsub=2, nsamp=2 ** 15, nfft=4096, noverlap=1024, nchan=8, ndec=4,
                             dm=(0.0, 3.0, 6.0))
    x = synth.generate(cfg)
    want = orc.run(orc.Params(**cfg.plan_kwargs()), x)
    dev, plan = gpu_run(cdmt, cfg, x)
    h_in = torch.from_numpy(x).pin_memory()
    h_out = torch.empty(dev.shape, dtype=torch.float32).pin_memory()
    # 10 blocks: one group; then 1, 2 and 3 blocks per group (odd/even groups, ragged last group)
    assert cdmt.cdmt_plan_query(plan, cfg.nsamp)["nblock"] == 10
    for gb in (0, 1, 2, 3):
        cdmt.cdmt_plan_set_option(plan, cdmt.OPT_HOST_GROUP_BLOCKS, gb)
        lay = cdmt.cdmt_host_layout(plan, cfg.nsamp, cdmt.OUT_F32)
        assert lay["ngroups"] == (1 if gb == 0 else -(-10 // gb))
        nbytes = cdmt.cdmt_host_scratch_bytes(plan, cfg.nsamp)
        assert nbytes == lay["scratch_bytes"]
        scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        h_out.fill_(float("nan"))
        for _ in range(2):      # the second call reuses streams and events
            cdmt.cdmt_execute_host(plan, h_in.data_ptr(), cfg.nsamp, cfg.nsamp, h_out.data_ptr(), scratch, nbytes)
        check_filterbank(h_out.numpy(), want)
        assert np.array_equal(h_out.numpy(), dev), gb


def test_host_path_async_8bit_against_the_oracle(cdmt):
    """cdmt_execute_host_async(CDMT_OUT_U8): Alg. 1 l.95-108 end to end -- 8-bit codes plus offset / scale
    per (group, DM, channel) reach the host; the call only queues work (completion = the caller's stream).
    Per group: statistics against oracle.redigitize of the float32 filterbank the same plan computes
    (2e-7), the decision bit for bit (oracle.quantize on the reported offsets / scales), and the whole
    chain against oracle.run -> oracle.redigitize (codes within one unit on a small fraction)."""
    cfg = synth.small_config(nsub=2, nsamp=2 ** 17, nfft=16384, noverlap=4096, nchan=8, ndec=8,
                             dm=(0.0, 3.0, 6.0, 12.5), in_dtype=synth.IN_CI8)
    x = synth.generate(cfg)
    fb_dev, plan = gpu_run(cdmt, cfg, x)
    fb_orc = orc.run(orc.Params(**cfg.plan_kwargs()), x)
    nb, Vd, nch = cfg.nblock, cfg.nvalid_dec, cfg.nsub * cfg.nchan
    h_in = torch.from_numpy(x).pin_memory()
    for gb in (0, 4, 3):
        cdmt.cdmt_plan_set_option(plan, cdmt.OPT_HOST_GROUP_BLOCKS, gb)
        lay = cdmt.cdmt_host_layout(plan, cfg.nsamp, cdmt.OUT_U8)
        ng, gblk = lay["ngroups"], lay["group_blocks"]
        assert lay["d2h_bytes"] == fb_dev.size + ng * 2 * cfg.ndm * nch * 4
        h_codes = torch.full(fb_dev.shape, 255, dtype=torch.uint8).pin_memory()
        h_off = torch.full((ng, cfg.ndm, nch), float("nan"), dtype=torch.float32).pin_memory()
        h_sc = torch.full((ng, cfg.ndm, nch), float("nan"), dtype=torch.float32).pin_memory()
        scratch = torch.empty(lay["scratch_bytes"], dtype=torch.uint8, device="cuda")
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            cdmt.cdmt_execute_host_async(plan, h_in.data_ptr(), cfg.nsamp, cfg.nsamp, cdmt.OUT_U8, h_codes.data_ptr(),
                                         h_off.data_ptr(), h_sc.data_ptr(), 64.0, 16.0, scratch, scratch.numel(), st)
        st.synchronize()                       # the only wait: everything was joined into the caller's stream
        codes, off, sc = h_codes.numpy(), h_off.numpy(), h_sc.numpy()
        for i in range(ng):
            b0, b1 = i * gblk, min(nb, (i + 1) * gblk)
            rows = slice(b0 * Vd, b1 * Vd)
            r = orc.redigitize(fb_dev[:, rows], b1 - b0)
            np.testing.assert_allclose(sc[i], r["scale"], rtol=2e-7, atol=0)
            np.testing.assert_allclose(off[i], r["offset"], rtol=2e-7, atol=2e-7 * float(np.abs(r["mean"]).max()))
            assert np.array_equal(codes[:, rows], orc.quantize(fb_dev[:, rows], off[i], sc[i]))
            full = orc.redigitize(fb_orc[:, rows], b1 - b0)
            diff = np.abs(codes[:, rows].astype(np.int16) - full["codes"].astype(np.int16))
            assert diff.max() <= 1 and (diff != 0).mean() < 5e-3


def test_execute_sums_are_the_block_sums_of_the_stored_filterbank(cdmt):
    """cdmt_execute_sums: (sum I, sum I^2) per (DM, block, channel) of Alg. 1 l.104, from every kernel that
    can run the shape, against the oracle's segment sums of the very float32 values the GPU stored."""
    cfg = synth.small_config(nsub=3, nsamp=2 ** 17, nfft=65536, noverlap=16384, nchan=16, ndec=16,
                             dm=(0.0, 1.5, 40.0), f_lo=121.0)
    x = synth.generate(cfg)
    d_in = torch.from_numpy(x).cuda()
    for kern in (0, 1, 2, 3, 4, 5):
        plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
        cdmt.cdmt_plan_set_option(plan, cdmt.OPT_FUSED_KERNEL, kern)
        q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
        nt, nch = q["nout_per_chan"], cfg.nsub * cfg.nchan
        out = torch.empty((cfg.ndm, nt, nch), dtype=torch.float32, device="cuda")
        sums = torch.full((cfg.ndm, cfg.nblock, nch, 2), float("nan"), dtype=torch.float64, device="cuda")
        ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device="cuda")
        cdmt.cdmt_execute_sums(plan, d_in, cfg.nsamp, cfg.nsamp, out, nt * nch, sums, ws, ws.numel())
        torch.cuda.synchronize()
        r = orc.redigitize(out.cpu().numpy(), cfg.nblock)
        np.testing.assert_allclose(sums.cpu().numpy(), r["segsum"], rtol=1e-13, atol=0, err_msg="kernel %d" % kern)


def test_subband_shards_concatenate_to_the_unsharded_filterbank(cdmt):
    """N4 / 8(e): the subbands of one observation split into contiguous ranges (bench.py --shard subband,
    PAPER.md:137) -- each range through its own plan -- give, concatenated along the (descending) channel
    axis, bit for bit the filterbank of the unsharded plan."""
    import bench
    cfg = synth.small_config(nsub=5, nsamp=2 ** 16, nfft=16384, noverlap=4096, nchan=8, ndec=8,
                             dm=(0.0, 2.5, 17.0), f_lo=133.0)
    x = synth.generate(cfg)
    whole, _ = gpu_run(cdmt, cfg, x)
    check_filterbank(whole, orc.run(orc.Params(**cfg.plan_kwargs()), x))
    for world in (2, 3):
        parts = []
        for rank in range(world):
            piece, s0 = bench.rank_piece(cfg, rank, world, "subband")
            got, _ = gpu_run(cdmt, piece, x[s0:s0 + piece.nsub])
            parts.append(got)
        # output channels descend in frequency: the highest subbands come first
        assert np.array_equal(np.concatenate(parts[::-1], axis=2), whole), world
    # --shard dm: contiguous ranges of the DM trials; the DM planes concatenate
    parts = [gpu_run(cdmt, bench.rank_piece(cfg, rank, 2, "dm")[0], x)[0] for rank in range(2)]
    assert np.array_equal(np.concatenate(parts, axis=0), whole)


def test_errors_are_codes_not_crashes(cdmt):
    cfg = synth.small_config()
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    x = torch.zeros((cfg.nsub, 2, cfg.nsamp), dtype=torch.complex64, device="cuda")
    q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
    out = torch.zeros((cfg.ndm, q["nout_per_chan"], cfg.nsub * cfg.nchan), device="cuda")
    ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device="cuda")
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_execute(plan, x, cfg.nsamp, cfg.nsamp, out, out[0].numel(), ws, ws.numel() - 1024)
    assert e.value.status == cdmt.ERR_WORKSPACE
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_execute(plan, x, cfg.nfft - 1, cfg.nsamp, out, out[0].numel(), ws, ws.numel())
    assert e.value.status == cdmt.ERR_SIZE
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_execute(plan, x.data_ptr() + 4, cfg.nsamp, cfg.nsamp, out, out[0].numel(), ws, ws.numel())
    assert e.value.status == cdmt.ERR_ARG
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_execute(plan, x, cfg.nsamp, cfg.nsamp, out, out[0].numel() - 1, ws, ws.numel())
    assert e.value.status == cdmt.ERR_SIZE
    # and the plan still works afterwards
    cdmt.cdmt_execute(plan, x, cfg.nsamp, cfg.nsamp, out, out[0].numel(), ws, ws.numel())
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0


# ---------------------------------------------------------------- repeatability (stands in for racecheck)
@pytest.mark.parametrize("kern", [4, 3, 5])
def test_fused_kernels_are_bit_reproducible(cdmt, kern):
    """compute-sanitizer's racecheck is not available on the GPU pool.  The fused kernels exchange data
    through shared memory under split mbarriers; a missing wait would show as run-to-run differences.
    Twenty executes of the same plan on the same input (a grid of several waves, every DM trial written
    into its own plane) must be bit-identical."""
    cfg = synth.small_config(nsub=24, nsamp=2 ** 18, nfft=65536, noverlap=16384, nchan=16, ndec=16,
                             dm=tuple(np.arange(24) * 1.25), f_lo=119.0)
    x = synth.generate(cfg)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    cdmt.cdmt_plan_set_option(plan, cdmt.OPT_FUSED_KERNEL, kern)
    d_in = torch.from_numpy(x).cuda()
    first = cdmt.run_on_device(plan, d_in, cfg.nsamp).clone()
    for _ in range(20):
        again = cdmt.run_on_device(plan, d_in, cfg.nsamp)
        assert torch.equal(first, again)


def test_execute_is_cuda_graph_capturable(cdmt):
    """cdmt_execute only queues kernels on the caller's stream (no host synchronisation, no allocation,
    constants uploaded through kernel parameters): it can be captured into a CUDA graph and replayed on
    new input in the same buffers."""
    cfg = synth.small_config(nsub=2, nsamp=2 ** 17, nfft=65536, noverlap=16384, nchan=16, ndec=16,
                             dm=(0.0, 3.0, 11.5))
    x1 = synth.generate(cfg)
    cfg2 = synth.small_config(nsub=2, nsamp=2 ** 17, nfft=65536, noverlap=16384, nchan=16, ndec=16,
                              dm=(0.0, 3.0, 11.5), seed=77)
    x2 = synth.generate(cfg2)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
    d_in = torch.from_numpy(x1).cuda()
    nch = cfg.nsub * cfg.nchan
    out = torch.zeros((cfg.ndm, q["nout_per_chan"], nch), dtype=torch.float32, device="cuda")
    ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device="cuda")
    eager = cdmt.run_on_device(plan, d_in, cfg.nsamp).clone()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        cdmt.cdmt_execute(plan, d_in, cfg.nsamp, cfg.nsamp, out, out[0].numel(), ws, ws.numel(), side)   # warm up
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        cdmt.cdmt_execute(plan, d_in, cfg.nsamp, cfg.nsamp, out, out[0].numel(), ws, ws.numel(),
                          torch.cuda.current_stream())
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, eager)
    d_in.copy_(torch.from_numpy(x2).cuda())
    g.replay()
    torch.cuda.synchronize()
    want = orc.run(orc.Params(**cfg2.plan_kwargs()), x2)
    check_filterbank(out.cpu().numpy(), want)


def test_multiplan_groups_against_the_oracle_on_a_common_time_grid(cdmt):
    """N4: a multiplan sizes groups of subbands from Eq. 2 and writes ONE filterbank.
    Each group's columns must equal the oracle run with that group's subbands and sizes on the input from the
    group's first sample on; an undispersed impulse must land in the same row in every group (common time
    grid); rows a group does not produce stay untouched."""
    nsub, nchan, ndec = 12, 8, 8
    fcen = 114.93 + synth.BW_MHZ * 16 * (np.arange(nsub) + 0.5)          # a wide band: the sweep falls by 5x
    dm = np.array([0.0, 20.0, 79.5])
    T = 2 ** 17 + 4096
    mp = cdmt.cdmt_multiplan_create(nsub, fcen, synth.BW_MHZ, nchan, ndec, dm, min_efficiency=0.9, max_groups=3)
    q = cdmt.cdmt_multiplan_query(mp, T)
    assert q["ngroups"] == 3
    cfg = synth.small_config(nsub=nsub, nsamp=T, nfft=32768, noverlap=4096, nchan=nchan, ndec=ndec, dm=tuple(dm))
    cfg.fcen_mhz = fcen
    x = synth.generate(cfg)
    n0 = 40000
    x[:, :, n0] += 300.0                                                  # undispersed impulse, every subband
    d_in = torch.from_numpy(x).cuda()
    nch = nsub * nchan
    out = torch.full((len(dm), q["nout_alloc"], nch), float("nan"), dtype=torch.float32, device="cuda")
    ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device="cuda")
    cdmt.cdmt_multiplan_execute(mp, d_in, T, T, out, q["nout_alloc"] * nch, ws, ws.numel())
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert cdmt.cdmt_multiplan_last_launch_count(mp) >= 3 * q["ngroups"]
    tstart = None
    for g in range(q["ngroups"]):
        gi = cdmt.cdmt_multiplan_group(mp, g, T)
        s0, s1 = gi["first_subband"], gi["first_subband"] + gi["nsub"]
        p = orc.Params(gi["nsub"], fcen[s0:s1], synth.BW_MHZ, gi["nfft"], gi["noverlap"], nchan, ndec, dm)
        want = orc.run(p, np.ascontiguousarray(x[s0:s1, :, gi["first_sample"]:]))
        assert want.shape[1] == gi["nout"]
        cols = slice((nsub - s1) * nchan, (nsub - s0) * nchan)            # descending frequency
        check_filterbank(got[:, :gi["nout"], cols], want)
        assert np.isnan(got[:, gi["nout"]:, cols]).all()                  # nothing written beyond the group's rows
        t0 = gi["first_sample"] + gi["noverlap"] // 2
        tstart = t0 if tstart is None else tstart
        assert t0 == tstart
        # the impulse: same row in every group at DM 0
        row = (n0 - tstart) // (nchan * ndec)
        assert (got[0, :q["nout_valid"], cols].sum(-1).argmax() == row)
    assert not np.isnan(got[:, :q["nout_valid"]]).any()


# ---------------------------------------------------------------- N3: planar input layouts
def planar_of(x, in_dtype):
    """[nsub][2][T] complex64 or [nsub][2][T][2] int8 (interleaved) -> [nsub][2][2 parts][T] real words."""
    if in_dtype == synth.IN_CI8:
        return np.ascontiguousarray(np.moveaxis(x, 3, 2))
    return np.ascontiguousarray(np.stack([x.real, x.imag], axis=2).astype(np.float32))


@pytest.mark.parametrize("in_dtype", [synth.IN_CF32, synth.IN_CI8])
def test_planar_input_unpack_and_parity(cdmt, in_dtype):
    """CDMT_IN_PF32 / CDMT_IN_PI8 ([S][Xre, Xim, Yre, Yim][T]): cdmt_unpack is bit exact,
    the whole path matches the oracle (which is fed the same samples interleaved) and is bit for bit the
    interleaved plan's output; also through the host path, and with a row stride that defeats the 16-byte
    loads of the int8 path."""
    cfg = synth.small_config(nsub=3, nsamp=2 ** 15 + 300, nfft=8192, noverlap=2048, nchan=8, ndec=4,
                             dm=(0.0, 7.5, 30.0), in_dtype=in_dtype)
    x = synth.generate(cfg)
    xp = planar_of(x, in_dtype)
    kw = cfg.plan_kwargs()
    want = orc.run(orc.Params(**kw), x)
    base, _ = gpu_run(cdmt, cfg, x)
    kw["in_dtype"] = cdmt.IN_PI8 if in_dtype == synth.IN_CI8 else cdmt.IN_PF32
    plan = cdmt.cdmt_plan_create(**kw)
    T = cfg.nsamp
    # unpack: bit exact
    d_in = torch.from_numpy(xp).cuda()
    B = cfg.nblock
    blocks = torch.zeros((B * cfg.nsub, 2, cfg.nfft), dtype=torch.complex64, device="cuda")
    cdmt.cdmt_unpack(plan, d_in, T, T, blocks)
    torch.cuda.synchronize()
    xc = x if in_dtype == synth.IN_CF32 else (x[..., 0].astype(np.float32) + 1j * x[..., 1].astype(np.float32))
    got = blocks.cpu().numpy()
    for b in range(B):
        for s in range(cfg.nsub):
            assert np.array_equal(got[b * cfg.nsub + s], xc[s, :, b * cfg.step:b * cfg.step + cfg.nfft].astype(np.complex64))
    # whole path, rows T words apart (T % 16 != 0: the int8 path reads word by word) and padded to 16 bytes
    for stride in (T, (T + 63) // 64 * 64):
        buf = torch.zeros((cfg.nsub, 2, 2, stride), dtype=d_in.dtype, device="cuda")
        buf[..., :T] = d_in
        out = cdmt.run_on_device(plan, buf, T)
        torch.cuda.synchronize()
        check_filterbank(out.cpu().numpy(), want)
        assert np.array_equal(out.cpu().numpy(), base), stride
    # host path
    h_in = torch.from_numpy(xp).pin_memory()
    h_out = torch.empty(base.shape, dtype=torch.float32).pin_memory()
    cdmt.cdmt_plan_set_option(plan, cdmt.OPT_HOST_GROUP_BLOCKS, 2)
    nbytes = cdmt.cdmt_host_scratch_bytes(plan, T)
    scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    cdmt.cdmt_execute_host(plan, h_in.data_ptr(), T, T, h_out.data_ptr(), scratch, nbytes)
    assert np.array_equal(h_out.numpy(), base)


def test_int8_wide_loads_equal_word_loads(cdmt):
    """The interleaved int8 path takes 16-byte loads when rows are 16-byte aligned: same bits as word loads."""
    cfg = synth.small_config(nsub=2, nsamp=2 ** 16, nfft=16384, noverlap=4096, nchan=8, ndec=8,
                             dm=(0.0, 12.0), in_dtype=synth.IN_CI8)
    x = synth.generate(cfg)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    T = cfg.nsamp
    aligned = torch.from_numpy(x).cuda()                                    # rows 2 T bytes apart: 16-byte aligned
    a = cdmt.run_on_device(plan, aligned, T).cpu().numpy()
    buf = torch.zeros((cfg.nsub, 2, T + 3, 2), dtype=torch.int8, device="cuda")   # stride T + 3 words: misaligned rows
    buf[:, :, :T] = aligned
    b = cdmt.run_on_device(plan, buf, T).cpu().numpy()
    assert np.array_equal(a, b)
    check_filterbank(a, orc.run(orc.Params(**cfg.plan_kwargs()), x))
