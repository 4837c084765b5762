"""Host-side checks of the C ABI (no GPU): the library loads, exports what include/cdmt.h
declares, validates arguments with status codes, and its block bookkeeping matches the
SURVEY.md section 8 table for the five configs."""
import ctypes
import os
import re

import numpy as np
import pytest

import cdmt_synth as synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cdmt():
    from paper_1607_00909_b200 import build
    build.build()
    from paper_1607_00909_b200 import cdmt as m
    return m


def header_functions():
    txt = open(os.path.join(ROOT, "include", "cdmt.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(cdmt_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol(cdmt):
    lib = ctypes.CDLL(cdmt.LIB_PATH)
    names = header_functions()
    assert len(names) >= 14
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(cdmt.EXPORTS) == names          # the binding covers the whole header
    for n in names:
        assert hasattr(cdmt, n), "python binding lacks %s" % n


def test_no_torch_types_in_the_abi():
    txt = open(os.path.join(ROOT, "include", "cdmt.h")).read()
    assert "torch" not in txt and "at::" not in txt and "Tensor" not in txt


# SURVEY.md section 8 table:            B    V(dec)  out samples/chan  channels
TABLE = {"c1": (5, 96, 480, 8), "c2": (18, 896, 16128, 160), "c3": (42, 192, 8064, 4608),
         "c4": (31, 128, 3968, 2048), "c5": (127, 512, 65024, 512)}


@pytest.mark.parametrize("name", synth.CONFIG_NAMES)
def test_query_matches_scope_table(cdmt, name):
    cfg = synth.make_config(name)
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
    B, Vd, nout, nch = TABLE[name]
    assert q["nblock"] == B == cfg.nblock
    assert cfg.nvalid_dec == Vd
    assert q["nout_per_chan"] == nout
    assert cfg.nsub * cfg.nchan == nch
    assert q["out_bytes"] == cfg.ndm * nout * nch * 4
    assert q["nsamp_consumed"] == (B - 1) * cfg.step + cfg.nfft <= cfg.nsamp
    assert q["workspace_bytes"] > 0
    assert cdmt.cdmt_min_overlap(plan) <= cfg.noverlap      # every config's overlap covers its sweep
    if name in ("c2", "c3", "c4", "c5"):
        ps = cdmt.cdmt_plan_create(**cfg.plan_kwargs(synth.REF_SUBBAND))
        mo = cdmt.cdmt_min_overlap(ps)
        # c4's overlap is just short of the whole-subband sweep at the top DMs
        assert (mo <= cfg.noverlap) == (name != "c4")


def test_chunk_option_changes_workspace_only(cdmt):
    cfg = synth.make_config("c3")
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    w0 = cdmt.cdmt_plan_query(plan, cfg.nsamp)["workspace_bytes"]
    cdmt.cdmt_plan_set_option(plan, cdmt.OPT_CHUNK_UNITS, 64)
    q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
    assert q["workspace_bytes"] < w0
    assert abs(q["workspace_bytes"] - 2 * 64 * 2 * cfg.nfft * 8) < 2 ** 20
    assert q["nblock"] == 42


def test_host_path_group_arithmetic(cdmt):
    """cdmt_execute_host stages groups of blocks; the overlap between groups is re-sent."""
    cfg = synth.make_config("c3")
    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    esz, rows = 8, 2 * cfg.nsub
    for gb in (1, 3, 5, 42):
        cdmt.cdmt_plan_set_option(plan, cdmt.OPT_HOST_GROUP_BLOCKS, gb)
        h2d, d2h = cdmt.cdmt_host_traffic_bytes(plan, cfg.nsamp)
        want = 0
        for b0 in range(0, 42, gb):
            nbg = min(gb, 42 - b0)
            want += ((nbg - 1) * cfg.step + cfg.nfft) * esz * rows
        assert h2d == want
        assert d2h == cdmt.cdmt_plan_query(plan, cfg.nsamp)["out_bytes"]
        assert cdmt.cdmt_host_scratch_bytes(plan, cfg.nsamp) > 0
    # one group: exactly the consumed samples once
    assert h2d == cdmt.cdmt_plan_query(plan, cfg.nsamp)["nsamp_consumed"] * esz * rows
    with pytest.raises(cdmt.CdmtError):
        cdmt.cdmt_plan_set_option(plan, cdmt.OPT_HOST_GROUP_BLOCKS, -1)


def bad(cdmt, status, **over):
    kw = dict(nsub=2, fcen_mhz=[150.0, 150.2], bw_mhz=synth.BW_MHZ, nfft=4096, noverlap=1024,
              nchan=8, ndec=4, dm=[0.0, 1.0])
    kw.update(over)
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_plan_create(**kw)
    assert e.value.status == status, over


def test_plan_create_validation(cdmt):
    S, A = cdmt.ERR_SIZE, cdmt.ERR_ARG
    bad(cdmt, S, nfft=4095)                    # not a power of two
    bad(cdmt, S, nfft=128)                     # below the supported range
    bad(cdmt, S, nfft=2 ** 21)
    bad(cdmt, S, nchan=3)
    bad(cdmt, S, nchan=512)                    # M = 8 < 16
    bad(cdmt, S, nfft=2 ** 16, nchan=4)        # M = 16384 > 8192
    bad(cdmt, S, noverlap=4096)                # >= nfft
    bad(cdmt, S, noverlap=-16)
    bad(cdmt, S, noverlap=1000)                # % (2 nchan) != 0
    bad(cdmt, S, ndec=0)
    bad(cdmt, S, ndec=5)                       # (nfft - noverlap) % (nchan ndec) != 0
    bad(cdmt, A, bw_mhz=0.0)
    bad(cdmt, A, bw_mhz=float("nan"))
    bad(cdmt, A, fcen_mhz=[0.05, 150.0])       # fcen - bw/2 <= 0
    bad(cdmt, A, dm=[0.0, float("inf")])
    bad(cdmt, A, in_dtype=7)
    bad(cdmt, A, chirp_ref=2)
    lib = ctypes.CDLL(cdmt.LIB_PATH)
    h = ctypes.c_void_p()
    assert lib.cdmt_plan_create(ctypes.byref(h), 0, None, ctypes.c_double(0.2), 4096, 1024, 8, 4, 0, None, 0, 0) == A
    assert h.value is None
    assert lib.cdmt_plan_create(None, 1, None, ctypes.c_double(0.2), 4096, 1024, 8, 4, 1, None, 0, 0) == A
    assert lib.cdmt_plan_destroy(None) == A


def test_negative_dm_and_odd_ndec_are_legal(cdmt):
    p = cdmt.cdmt_plan_create(1, [150.0], synth.BW_MHZ, 4096, 1024, 8, 3, [-5.0, 5.0])
    assert cdmt.cdmt_plan_query(p, 4096)["nblock"] == 1
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_plan_query(p, 4095)
    assert e.value.status == cdmt.ERR_SIZE
    with pytest.raises(cdmt.CdmtError):
        cdmt.cdmt_plan_set_option(p, 99, 1)
    with pytest.raises(cdmt.CdmtError):
        cdmt.cdmt_plan_set_option(p, cdmt.OPT_PROFILE, 2)
    cdmt.cdmt_plan_destroy(p)


def test_execute_rejects_null_pointers_before_touching_cuda(cdmt):
    """Argument validation happens on the host: these calls must return codes on a box with no GPU."""
    p = cdmt.cdmt_plan_create(1, [150.0], synth.BW_MHZ, 4096, 1024, 8, 4, [0.0])
    for args in [(0, 16384, 16384, 256, 10 ** 9, 256, 10 ** 9),
                 (256, 16384, 16384, 0, 10 ** 9, 256, 10 ** 9),
                 (256, 16384, 16384, 256, 10 ** 9, 0, 10 ** 9),
                 (260, 16384, 16384, 256, 10 ** 9, 256, 10 ** 9)]:      # input not aligned to one complex word
        with pytest.raises(cdmt.CdmtError) as e:
            cdmt.cdmt_execute(p, args[0], args[1], args[2], args[3], args[4], args[5], args[6], stream=0)
        assert e.value.status == cdmt.ERR_ARG
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_execute(p, 256, 16384, 8192, 256, 10 ** 9, 256, 10 ** 9, stream=0)     # stride < nsamp
    assert e.value.status == cdmt.ERR_SIZE
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_execute(p, 256, 16384, 16384, 256, 10, 256, 10 ** 9, stream=0)         # planes overlap
    assert e.value.status == cdmt.ERR_SIZE


def test_redigitize_static_checks_its_limit_on_the_host(cdmt):
    """cdmt_redigitize_static (no workspace, no allocation): null pointers, bad targets and batches beyond the
    library's fixed 4 MiB scratch are refused with a status before anything touches CUDA."""
    assert cdmt.cdmt_redigitize_static_max_bytes() == 4 << 20
    fcen = 120.0 + synth.BW_MHZ * (np.arange(40) + 0.5)
    p = cdmt.cdmt_plan_create(40, fcen, synth.BW_MHZ, 8192, 7936, 16, 2, np.arange(64.0))     # Vd = 8, 640 channels
    plane = 40 * 8 * 640
    # 64 DMs x 40 blocks x 640 channels x 16 bytes = 26 MB of block sums: more than the static array holds
    assert cdmt.cdmt_redigitize_workspace_bytes(p, 40) == 64 * 40 * 640 * 16
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_redigitize_static(p, 256, plane, 40, 64.0, 16.0, 256, plane, 256, 256, stream=0)
    assert e.value.status == cdmt.ERR_WORKSPACE
    for bad in [dict(d_fb=0), dict(d_codes=0), dict(d_offset=0), dict(d_scale=0), dict(d_fb=258), dict(qstd=0.0)]:
        a = dict(d_fb=256, d_codes=256, d_offset=256, d_scale=256, qstd=16.0)
        a.update(bad)
        with pytest.raises(cdmt.CdmtError) as e:
            cdmt.cdmt_redigitize_static(p, a["d_fb"], 8 * 640, 1, 64.0, a["qstd"], a["d_codes"], 8 * 640,
                                        a["d_offset"], a["d_scale"], stream=0)
        assert e.value.status == cdmt.ERR_ARG, bad
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_redigitize_static(p, 256, 8 * 640 - 1, 1, 64.0, 16.0, 256, 8 * 640, 256, 256, stream=0)  # short plane stride
    assert e.value.status == cdmt.ERR_SIZE


def test_sweep_seconds_eq2_against_paper_values(cdmt):
    vals = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_values.txt")):
        line = line.split("#", 1)[0].strip()
        if line:
            k, v = line.split("=")
            vals[k.strip()] = float(v)
    cw = synth.BW_MHZ / 8
    assert abs(cdmt.cdmt_sweep_seconds(135.0, cw, vals["dm_J1810"]) * 1e3 - vals["td_ms_J1810"]) < 0.05
    assert abs(cdmt.cdmt_sweep_seconds(135.0, cw, vals["dm_J2215"]) * 1e3 - vals["td_ms_J2215"]) < 0.05
    assert cdmt.cdmt_strerror(0) == "ok" and "workspace" in cdmt.cdmt_strerror(3)
    assert "sm_100a" in cdmt.cdmt_version()


def test_product_path_does_not_import_the_oracle():
    """The CUDA package must never route through oracle/ (and the oracle never imports the package)."""
    pk = os.path.join(ROOT, "paper_1607_00909_b200")
    for dirpath, _, files in os.walk(pk):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, flags=re.M), f
                assert "cdmt_oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1607_00909_b200", txt, flags=re.M), f
            assert "libcdmt" not in txt and "csrc" not in txt.replace("paper_1607_00909_b200/csrc/", ""), f


def test_suggest_sizes_follow_eq2_and_are_legal(cdmt):
    """cdmt_suggest_sizes: noverlap covers r t_d of the lowest channel at the largest
    DM (Eq. 2 via the oracle's separately written sweep), is legal for cdmt_plan_create, nfft keeps the
    requested fraction; higher subbands and lower DMs get smaller sizes (the paper's own inefficiency)."""
    from oracle import cdmt_oracle as orc
    bw, nchan = 0.1953125, 8
    lo = np.array([114.93 + bw / 2])                      # the paper's lowest survey subband
    nfft, nov = cdmt.cdmt_suggest_sizes(lo, bw, nchan, 1, 79.5)
    cw = bw / nchan
    need = orc.sweep_seconds(lo[0] - bw / 2 + cw / 2, cw, 79.5) * bw * 1e6
    assert 2071 < need < 2073                              # PAPER.md:71 / SURVEY: r t_d = 2072 input samples
    assert need <= nov < need + 2 * nchan and nov % (2 * nchan) == 0
    assert (nfft - nov) >= 0.75 * nfft and (nfft // 2 - nov) < 0.75 * (nfft // 2)
    assert (nfft, nov) == (16384, 2080)                    # against the paper's fixed 65536 / 16384
    plan = cdmt.cdmt_plan_create(nsub=1, fcen_mhz=lo, bw_mhz=bw, nfft=nfft, noverlap=nov, nchan=nchan, ndec=1,
                                 dm=[0.0, 79.5])
    assert cdmt.cdmt_min_overlap(plan) == nov
    # per-subband sizes: the top of the LOFAR band needs a quarter of the overlap
    hi = np.array([175.0])
    nfft_hi, nov_hi = cdmt.cdmt_suggest_sizes(hi, bw, nchan, 1, 79.5)
    assert nov_hi < nov / 3 and nfft_hi <= nfft
    # monotone in DM, ndec divisibility, efficiency knob
    prev = 0
    for dm in (1.0, 10.0, 40.0, 79.5):
        n, o = cdmt.cdmt_suggest_sizes(lo, bw, 16, 16, dm)
        assert o >= prev and o % (16 * 16) == 0 and (n - o) % (16 * 16) == 0
        prev = o
    n9, o9 = cdmt.cdmt_suggest_sizes(lo, bw, nchan, 1, 79.5, min_efficiency=0.9)
    assert o9 == nov and n9 > nfft and (n9 - o9) >= 0.9 * n9
    # subband-referenced chirp: the sweep of the whole subband; no supported nfft at 8 channels -> status
    with pytest.raises(cdmt.CdmtError) as e:
        cdmt.cdmt_suggest_sizes(lo, bw, nchan, 1, 79.5, cdmt.REF_SUBBAND)
    assert e.value.status == cdmt.ERR_SIZE
    n32, o32 = cdmt.cdmt_suggest_sizes(lo, bw, 32, 1, 79.5, cdmt.REF_SUBBAND, 0.5)
    assert o32 >= orc.sweep_seconds(lo[0], bw, 79.5) * bw * 1e6 and n32 // 32 <= 8192
    for bad in (dict(min_efficiency=1.0), dict(min_efficiency=0.0), dict(dm_max_abs=-1.0)):
        kw = dict(fcen_mhz=lo, bw_mhz=bw, nchan=nchan, ndec=1, dm_max_abs=79.5)
        kw.update(bad)
        with pytest.raises(cdmt.CdmtError):
            cdmt.cdmt_suggest_sizes(**kw)


def test_multiplan_partitions_the_band_from_eq2(cdmt):
    """N4: groups of subbands sized from the dispersion sweep, one common time grid.
    Host arithmetic only."""
    # the paper's survey band: 200 subbands from 114.93 MHz, 8 channels, DM <= 79.5
    fcen = 114.93 + synth.BW_MHZ * (np.arange(200) + 0.5)
    dm = 0.5 + np.arange(80)
    mp = cdmt.cdmt_multiplan_create(200, fcen, synth.BW_MHZ, 8, 1, dm, min_efficiency=0.9, max_groups=4)
    T = 2 ** 20
    q = cdmt.cdmt_multiplan_query(mp, T)
    assert 1 < q["ngroups"] <= 4
    groups = [cdmt.cdmt_multiplan_group(mp, g, T) for g in range(q["ngroups"])]
    # contiguous cover of the band, sizes that shrink (or stay) with frequency, overlap from Eq. 2 per group
    assert groups[0]["first_subband"] == 0 and sum(g["nsub"] for g in groups) == 200
    for a, b in zip(groups, groups[1:]):
        assert b["first_subband"] == a["first_subband"] + a["nsub"]
        assert b["nfft"] == a["nfft"] and b["noverlap"] < a["noverlap"]
    tstart = max(g["noverlap"] // 2 for g in groups)
    for g in groups:
        lo = fcen[g["first_subband"]]
        nfft, nov = cdmt.cdmt_suggest_sizes([lo], synth.BW_MHZ, 8, 1, 79.5, min_efficiency=0.9)
        assert g["noverlap"] == nov and g["nfft"] >= nfft and g["nfft"] == groups[0]["nfft"]
        assert g["first_sample"] == tstart - g["noverlap"] // 2          # every group's row 0 starts at tstart
        step, vd = g["nfft"] - g["noverlap"], (g["nfft"] - g["noverlap"]) // 8
        assert g["nout"] == ((T - g["first_sample"] - g["nfft"]) // step + 1) * vd
    assert q["nout_valid"] == min(g["nout"] for g in groups) and q["nout_alloc"] == max(g["nout"] for g in groups)
    kept = sum(g["nsub"] * (g["nfft"] - g["noverlap"]) / g["nfft"] for g in groups) / 200
    assert abs(q["kept_fraction"] - kept) < 1e-12
    # against the paper's one pair for the whole band (N_bin 65536, n_d 2048 x n_c 8: PAPER.md:139): 75 % kept
    assert q["kept_fraction"] > 0.9 > (65536 - 2048 * 8) / 65536
    # one group = one plan for the lowest subband's sizes
    one = cdmt.cdmt_multiplan_create(200, fcen, synth.BW_MHZ, 8, 1, dm, min_efficiency=0.9, max_groups=1)
    g1 = cdmt.cdmt_multiplan_group(one, 0, T)
    assert cdmt.cdmt_multiplan_query(one, T)["ngroups"] == 1 and g1["nsub"] == 200 and g1["first_sample"] == 0
    assert cdmt.cdmt_multiplan_query(one, T)["kept_fraction"] < q["kept_fraction"]
    with pytest.raises(cdmt.CdmtError):
        cdmt.cdmt_multiplan_create(3, [120.0, 119.0, 121.0], synth.BW_MHZ, 8, 1, dm)     # not ascending
    with pytest.raises(cdmt.CdmtError):
        cdmt.cdmt_multiplan_query(mp, 1000)                                              # shorter than a block
    cdmt.cdmt_multiplan_destroy(mp)
