"""Host-side logic of bench.py (no GPU): flop accounting, the N>1 reduction over gloo with
world_size 2, and the reference arm launched the way the driver launches it."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
import cdmt_synth as synth  # noqa: E402


def test_flop_accounting_matches_scope_table():
    # per-unit per-DM flops c2 11.08, c3 10.35, c4 43.5, c5 10.88 MF
    for name, mf in (("c2", 11.08), ("c3", 10.35), ("c4", 43.5), ("c5", 10.88)):
        got = bench.algorithmic_flops_per_unit_dm(synth.make_config(name)) / 1e6
        assert abs(got - mf) < 0.06, (name, got)
    # c3 total 12.2 TF
    c3 = synth.make_config("c3")
    tot = bench.algorithmic_flops_per_unit_dm(c3) * c3.ndm * c3.nsub * c3.nblock
    assert abs(tot / 1e12 - 12.0) < 0.3
    assert abs(bench.FP32_PEAK_TFLOPS - 74.45) < 0.01


def test_rank_workloads_differ_only_by_seed():
    a = bench.rank_workload(synth.make_config("c1"), 0, 2)
    b = bench.rank_workload(synth.make_config("c1"), 1, 2)
    assert a.seed != b.seed and a.nsub == b.nsub and a.nsamp == b.nsamp
    xa, xb = synth.generate(a), synth.generate(b)
    assert xa.shape == xb.shape and not np.array_equal(xa, xb)
    solo = bench.rank_workload(synth.make_config("c1"), 0, 1)
    assert solo.seed == synth.make_config("c1").seed


WORKER = r"""
import os, sys, json
sys.path.insert(0, %(root)r)
import torch, torch.distributed as dist
import bench
import cdmt_synth as synth
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
cfg = bench.rank_workload(synth.make_config("c1"), rank, world)
ms = 10.0 + 5.0 * rank                      # rank 1 is slower
dist.barrier()
mx = bench.max_over_ranks(ms, world)
val = bench.whole_job_value(cfg, world, mx * 1e-3)
if rank == 0:
    print(json.dumps({"max_ms": mx, "value": val, "world": world}))
dist.destroy_process_group()
"""


def _torchrun(args, timeout=600):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29517"] + args
    return subprocess.run(cmd, env=env, cwd=ROOT, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % {"root": ROOT})
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    line = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(line) == 1
    d = json.loads(line[0])
    assert d["world"] == 2 and d["max_ms"] == 15.0
    c1 = synth.make_config("c1")
    assert abs(d["value"] - 2 * c1.nsub * c1.nsamp * c1.ndm / 15e-3) < 1e-3 * d["value"]


def test_reference_arm_two_ranks_prints_one_line():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1",
                   "--config", "c1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == bench.METRIC and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["n_gpus"] == 2 and d["higher_is_better"] is True


def test_subband_sharding_partitions_the_observation():
    """--shard subband (strong scaling): the ranks' subband ranges tile [0, nsub) without
    overlap, each rank's plan sees its own centre frequencies, and the generator is indexed by the
    GLOBAL subband so that the pieces are the pieces of the one observation."""
    c3 = synth.make_config("c3")
    for world in (1, 2, 3, 8):
        rng = [bench.subband_range(c3.nsub, r, world) for r in range(world)]
        assert rng[0][0] == 0 and rng[-1][1] == c3.nsub
        assert all(rng[i][1] == rng[i + 1][0] for i in range(world - 1))
        assert max(b - a for a, b in rng) - min(b - a for a, b in rng) <= 1
    piece, s0 = bench.rank_piece(synth.make_config("c3"), 3, 8, "subband")
    assert piece.nsub == 36 and s0 == 108 and np.array_equal(piece.fcen_mhz, c3.fcen_mhz[108:144])
    assert piece.nblock == c3.nblock and piece.ndm == c3.ndm and piece.seed == c3.seed
    solo, s0 = bench.rank_piece(synth.make_config("c3"), 0, 1, "subband")
    assert solo.nsub == c3.nsub and s0 == 0
    rep, s0 = bench.rank_piece(synth.make_config("c1"), 1, 2, "replicas")
    assert rep.nsub == 1 and s0 == 0 and rep.seed != synth.make_config("c1").seed
    # a piece's data equals the slice of the whole observation
    small = synth.small_config(nsub=4, nsamp=2 ** 13, nfft=4096, noverlap=1024, nchan=8, ndec=4, dm=(0.0, 3.0))
    whole = synth.generate(small)
    pc, s0 = bench.rank_piece(small, 1, 2, "subband")
    got = np.stack([synth.generate_subband(small, s0 + s) for s in range(pc.nsub)])
    assert np.array_equal(got, whole[2:4])


def test_dm_sharding_partitions_the_trials():
    """--shard dm (few subbands -> split the DM trials): the ranks' DM ranges tile the
    list without overlap; every rank keeps all subbands, blocks and the seed of the one observation."""
    c2 = synth.make_config("c2")
    got = []
    for r in range(3):
        piece, s0 = bench.rank_piece(synth.make_config("c2"), r, 3, "dm")
        assert s0 == 0 and piece.nsub == c2.nsub and piece.nblock == c2.nblock and piece.seed == c2.seed
        assert np.array_equal(piece.fcen_mhz, c2.fcen_mhz)
        got.append(piece.dm)
    assert np.array_equal(np.concatenate(got), c2.dm)
    assert max(len(g) for g in got) - min(len(g) for g in got) <= 1
    # the whole-job metric counts the observation once
    assert bench.whole_job_value(c2, 1, 0.01) == c2.nsub * c2.nsamp * c2.ndm / 0.01
