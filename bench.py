#!/usr/bin/env python
"""bench.py -- throughput of the cdmt hot path on B200 (contract: see DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config c3] [--impl ours|reference]
                  [--shard replicas|subband|dm] [--survey]

A "step" is one pass of the whole hot path (unpack + forward FFT + fused per-DM kernel, every
block, every DM) over one synthetic observation of the named config.  Metric (BASELINE.json):
input samples x DM trials per second = nsub * T * ndm / t.  One JSON line is printed by rank 0:
`value` from device-resident input, `e2e` / `e2e_8bit_output` through cdmt_execute_host_async with
pinned host buffers, `roofline` of the fused per-DM kernel, the extra legs `redigitize` (8-bit output,
Alg. 1 l.104-106) and `incoherent` (semi-coherent search), `cpu_baseline` (the oracle).

N > 1 (torchrun): the path has no exchange step, so by default each rank runs its own observation of
the same config (another beam: other seed) on its own GPU -- weak scaling, no data-path collective;
--shard subband / dm split ONE observation over the ranks instead (strong scaling, still no collective).
torch.distributed is used for the barrier and the max-over-ranks of the device time only.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import cdmt_synth as synth  # noqa: E402

METRIC = "input_samples_x_dm_trials_per_s"
UNIT = "samples*DM/s"
# FP32 (non-tensor) peak of a B200: 148 SMs x 128 FP32 lanes x 2 flop/FMA x 1.965 GHz
# (unit counts and clocks: /opt/skills/guides/B200_PROFILING.md, MEASURED_PEAKS.json sm_max_mhz)
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of one fused-kernel launch from the committed
# `ncu --set full` capture (profiles/r2_ws_c3.md: 4.397368 + 4.865498 GB for a launch of 4032 units of c3),
# per (subband, block) unit; roofline.traffic scales it to the units of a timed launch
FUSED_TRAFFIC_BYTES_PER_UNIT = {"c3": (4397368000 + 4865498000) / 4032.0}


def algorithmic_flops_per_unit_dm(cfg: synth.Config) -> float:
    """SURVEY.md 8(d) / DESIGN.md: flops credited to one (subband, block) unit at one DM:
    2 pols x C backward FFTs of M at 5 M log2 M, a complex multiply (6) on both pols per bin,
    ~20 flops to form the chirp sample per bin, 8 per detected (kept) sample."""
    N, C, M = cfg.nfft, cfg.nchan, cfg.mbin
    V = M - 2 * cfg.half_discard
    return 2 * C * 5.0 * M * np.log2(M) + 2 * 6.0 * N + 20.0 * N + 8.0 * C * V


def shard_seed(seed: int, rank: int) -> int:
    """Rank r processes its own observation: same recipe, another seed."""
    return seed + 1000 * rank


def rank_workload(cfg: synth.Config, rank: int, world: int) -> synth.Config:
    """Weak scaling: every rank gets a full observation of the config (its own beam)."""
    if world > 1:
        cfg.seed = shard_seed(cfg.seed, rank)
    return cfg


def subband_range(nsub: int, rank: int, world: int):
    """Strong scaling (--shard subband; PAPER.md:137 runs subband groups on separate GPUs): rank r
    owns the contiguous subbands [s0, s1) of the ONE observation; no exchange step, outputs concatenate."""
    return (nsub * rank) // world, (nsub * (rank + 1)) // world


def rank_piece(cfg: synth.Config, rank: int, world: int, shard: str):
    """(config of this rank's plan, first global subband it generates)."""
    if shard == "subband" and world > 1:
        import dataclasses
        s0, s1 = subband_range(cfg.nsub, rank, world)
        if s1 <= s0:
            raise SystemExit("--shard subband needs at least one subband per rank")
        return dataclasses.replace(cfg, nsub=s1 - s0, fcen_mhz=cfg.fcen_mhz[s0:s1]), s0
    if shard == "dm" and world > 1:
        # few subbands -> split the DM trials; every rank repeats the forward FFT (a1-a3)
        # of the whole observation and runs the DM loop over its own contiguous range of trials
        import dataclasses
        d0, d1 = subband_range(cfg.ndm, rank, world)
        if d1 <= d0:
            raise SystemExit("--shard dm needs at least one DM trial per rank")
        return dataclasses.replace(cfg, dm=cfg.dm[d0:d1]), 0
    return rank_workload(cfg, rank, world), 0


def max_over_ranks(value: float, world: int, device=None) -> float:
    """MAX all-reduce of a per-rank scalar (device time); identity for one rank."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(cfg: synth.Config, world: int, sec_per_step: float) -> float:
    """Metric over all ranks: every rank processed nsub*nsamp samples x ndm trials per step."""
    return world * float(cfg.nsub) * cfg.nsamp * cfg.ndm / sec_per_step


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [t.strip() for t in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(cfg: synth.Config, nunits: int, xsubs):
    """Time the oracle, as it stands, on `nunits` (subband, block) units with every DM trial.
    xsubs: list of generated subbands 0..k; units are taken block by block, subband by subband."""
    from oracle import cdmt_oracle as orc
    p = orc.Params(**cfg.plan_kwargs())
    us = [(i // cfg.nblock, i % cfg.nblock) for i in range(nunits)]
    blocks = np.stack([xsubs[s][:, b * cfg.step:b * cfg.step + cfg.nfft] for s, b in us])
    t0 = time.perf_counter()
    orc.units(p, [s for s, _ in us], blocks)
    dt = time.perf_counter() - t0
    samples_dm = nunits / float(cfg.nsub * cfg.nblock) * cfg.nsub * cfg.nsamp * cfg.ndm
    return samples_dm / dt, dt, orc.num_threads()


def oracle_sample_size(cfg: synth.Config, ncores: int, per_core: int) -> int:
    return max(1, min(cfg.nsub * cfg.nblock, per_core * ncores))


def run_reference(args, cfg, rank, world):
    """--impl reference: the CPU oracle on the host cores, bounded sample per step."""
    if rank != 0:
        return
    from oracle import cdmt_oracle as orc
    ncores = orc.num_threads()
    nunits = oracle_sample_size(cfg, ncores, 2)
    xs = [synth.generate_subband(cfg, s) for s in range((nunits + cfg.nblock - 1) // cfg.nblock)]
    for _ in range(args.warmup):
        oracle_sample(cfg, min(nunits, ncores), xs)
    t0 = time.perf_counter()
    done = 0.0
    for _ in range(args.steps):
        rate, dt, _ = oracle_sample(cfg, nunits, xs)
        done += rate * dt
    total = time.perf_counter() - t0
    value = done / total
    sample = "%d of %d (subband, block) units of %s x all %d DMs per step" % (
        nunits, cfg.nsub * cfg.nblock, cfg.name, cfg.ndm)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": total / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg, args),
        "real_time_factor": value / (cfg.nsub * cfg.ndm) * synth.TSAMP_S,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": ncores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_survey(args):
    """--survey: the paper's pilot-survey band (200 subbands of 195.31 kHz from 114.93 MHz,
    8 channels per subband, 80 DM trials 0.5 ... 79.5) through (a) one plan with the paper's own sizes
    (N_bin 65536, n_d 2048 channelised samples = 16384 input samples for every subband), (b) a multiplan
    with one group (overlap from Eq. 2 at the lowest subband) and (c) a multiplan with four groups
    (sizes that follow the observing frequency).  The paper does not integrate in time; here
    ndec = 8 keeps the output of 2^20 samples at 8 GB.  One JSON line."""
    import torch
    from paper_1607_00909_b200 import cdmt
    dev = torch.device("cuda", 0)
    nsub, nchan, ndec, T = 200, 8, 8, 2 ** 20
    fcen = 114.93 + synth.BW_MHZ * (np.arange(nsub) + 0.5)
    dm = 0.5 + np.arange(80.0)
    g = torch.Generator(device=dev)
    g.manual_seed(5)
    d_in = torch.view_as_complex(torch.randn((nsub, 2, T, 2), generator=g, device=dev, dtype=torch.float32) * 0.7071)
    nch = nsub * nchan
    stream = torch.cuda.current_stream()

    def time_it(fn):
        for _ in range(max(args.warmup, 3)):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(args.steps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    rows = []
    plan = cdmt.cdmt_plan_create(nsub, fcen, synth.BW_MHZ, 65536, 16384, nchan, ndec, dm)
    q = cdmt.cdmt_plan_query(plan, T)
    out = torch.empty((len(dm), q["nout_per_chan"], nch), dtype=torch.float32, device=dev)
    ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device=dev)
    ms = time_it(lambda: cdmt.cdmt_execute(plan, d_in, T, T, out, out[0].numel(), ws, ws.numel(), stream))
    rows.append({"what": "one plan, the paper's sizes (nfft 65536, noverlap 16384)", "groups": 1, "kept_fraction": 0.75,
                 "ms_per_step": ms, "out_samples_per_chan": q["nout_per_chan"],
                 "output_samples_x_dm_per_s": q["nout_per_chan"] * nch * len(dm) / (ms * 1e-3)})
    del out, ws
    for G in (1, 4):
        mp = cdmt.cdmt_multiplan_create(nsub, fcen, synth.BW_MHZ, nchan, ndec, dm, min_efficiency=0.9, max_groups=G)
        q = cdmt.cdmt_multiplan_query(mp, T)
        out = torch.empty((len(dm), q["nout_alloc"], nch), dtype=torch.float32, device=dev)
        ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device=dev)
        ms = time_it(lambda: cdmt.cdmt_multiplan_execute(mp, d_in, T, T, out, out[0].numel(), ws, ws.numel(), stream))
        grp = [cdmt.cdmt_multiplan_group(mp, i, T) for i in range(q["ngroups"])]
        rows.append({"what": "multiplan, max_groups %d (nfft %d; noverlap %s)" % (G, grp[0]["nfft"], [x["noverlap"] for x in grp]),
                     "groups": q["ngroups"], "kept_fraction": q["kept_fraction"], "ms_per_step": ms,
                     "out_samples_per_chan": q["nout_valid"],
                     "output_samples_x_dm_per_s": q["nout_valid"] * nch * len(dm) / (ms * 1e-3)})
        if G != 4:
            del out, ws
    best = rows[-1]
    # ---- the paper's headline use at its own scale: every coherently dedispersed filterbank
    # is incoherently dedispersed at steps of 0.002 pc/cm3 from -0.5 to +0.5 around its DM: 80 x 501 = 40 080
    # trials.  One semi-coherent step = cdmt_multiplan_execute (four groups) + cdmt_incoherent_dedisperse on the
    # rows that are complete in every column; the filterbanks never leave the device.
    semi = None
    try:
        ddm = np.round(np.arange(-250, 251) * 0.002, 9)
        nt_in = q["nout_valid"]
        qi = cdmt.cdmt_incoherent_query(plan, ddm, nt_in)
        d_ts = torch.empty((len(dm), len(ddm), qi["nt_out"]), dtype=torch.float32, device=dev)
        d_iws = torch.empty(max(256, qi["workspace_bytes"]), dtype=torch.uint8, device=dev)

        def incoh():
            cdmt.cdmt_incoherent_dedisperse(plan, out, out[0].numel(), nt_in, ddm, d_ts, d_ts[0].numel(), qi["nt_out"],
                                            d_iws, d_iws.numel(), stream)

        def semi_step():
            cdmt.cdmt_multiplan_execute(mp, d_in, T, T, out, out[0].numel(), ws, ws.numel(), stream)
            incoh()
        ims = time_it(incoh)
        sms = time_it(semi_step)
        adds_def, adds_done = cdmt.cdmt_incoherent_work(plan, ddm, nt_in)
        semi = {"coherent_trials": len(dm), "fine_trials_per_coherent": len(ddm), "dm_trials_total": len(dm) * len(ddm),
                "fine_step": 0.002, "fine_range": [-0.5, 0.5], "shift_range": qi["shift_range"],
                "trial_groups": qi["ngroups"], "incoherent_ms": ims, "semicoherent_step_ms": sms,
                "real_time_factor": T * synth.TSAMP_S / (sms * 1e-3),
                "adds_definition": adds_def, "adds_performed": adds_done,
                "definition_tadd_s": adds_def / ims / 1e9, "out_bytes": int(d_ts.numel() * 4),
                "note": "cdmt_multiplan_execute (4 groups) + cdmt_incoherent_dedisperse over 501 fine offsets per "
                        "coherent DM on the device-resident filterbanks; 2^20 input samples = %.2f s of data" % (T * synth.TSAMP_S)}
        del d_ts, d_iws
    except Exception as e:   # never lose the survey line to the extra leg
        semi = {"error": str(e)}
    line = {"metric": METRIC, "value": float(nsub) * T * len(dm) / (best["ms_per_step"] * 1e-3), "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": best["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "survey band of PAPER.md:137-139: 200 subbands from 114.93 MHz x 2^20 samples, nchan=8 "
                                   "ndec=8, 80 DM trials 0.5..79.5, complex64 noise in; sizes per group of subbands",
                       "nsub": nsub, "nsamp": T, "nchan": nchan, "ndec": ndec, "ndm": len(dm)},
            "real_time_factor": T * synth.TSAMP_S / (best["ms_per_step"] * 1e-3), "variants": rows,
            "semicoherent_search": semi}
    print(json.dumps(line), flush=True)


def workload_config(cfg, args):
    return {"workload": "%s: %d subbands x 2^%d samples, nfft=%d noverlap=%d nchan=%d ndec=%d, %d DM trials, %s in"
            % (cfg.name, cfg.nsub, int(np.log2(cfg.nsamp)), cfg.nfft, cfg.noverlap, cfg.nchan, cfg.ndec,
               cfg.ndm, "int8" if cfg.in_dtype == synth.IN_CI8 else "complex64"),
            "nsub": cfg.nsub, "nsamp": cfg.nsamp, "nfft": cfg.nfft, "noverlap": cfg.noverlap,
            "nchan": cfg.nchan, "ndec": cfg.ndec, "ndm": cfg.ndm, "nblock": cfg.nblock,
            "parallelism": ("%s of one observation split over %d GPUs (no collective)" % (
                                {"subband": "subbands", "dm": "DM trials"}[args.shard], args.gpus))
                           if getattr(args, "shard", "replicas") in ("subband", "dm") and args.gpus > 1 else
                           "replicas x%d (one observation per GPU, no collective)" % args.gpus,
            "l2": "inputs (%.1f GB) and spectra exceed the 126 MB L2; no flush needed" % (
                cfg.nsub * 2 * cfg.nsamp * (2 if cfg.in_dtype == synth.IN_CI8 else 8) / 1e9)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="c3", choices=synth.CONFIG_NAMES)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--chunk-units", type=int, default=0)
    ap.add_argument("--dm-tile", type=int, default=0)
    ap.add_argument("--fused-kernel", type=int, default=0, help="CDMT_OPT_FUSED_KERNEL (0 = library default)")
    ap.add_argument("--gen-threads", type=int, default=0)
    ap.add_argument("--host-group-blocks", type=int, default=0,
                    help="CDMT_OPT_HOST_GROUP_BLOCKS of the end-to-end leg (0 = library default)")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "subband", "dm"],
                    help="N > 1: one observation per GPU (weak scaling, default), or ONE observation with its "
                         "subbands (output channels concatenate) or its DM trials (output planes concatenate; the "
                         "forward FFT is repeated on every rank) split over the GPUs (strong scaling); none has a "
                         "collective")
    ap.add_argument("--no-redigitize", action="store_true", help="skip the extra cdmt_redigitize timing (N1)")
    ap.add_argument("--no-incoherent", action="store_true", help="skip the extra cdmt_incoherent_dedisperse timing (N2)")
    ap.add_argument("--fine-step", type=float, default=0.002, help="fine DM step of the incoherent leg (PAPER.md:141)")
    ap.add_argument("--survey", action="store_true",
                    help="N4: the paper's survey band with the paper's sizes against per-group sizes (cdmt_multiplan)")
    args = ap.parse_args()
    if args.survey:
        run_survey(args)
        return

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    full_cfg = synth.make_config(args.config)
    if args.impl == "reference":
        cfg = rank_workload(full_cfg, rank, world)
        run_reference(args, cfg, rank, world)
        return
    cfg, sub0 = rank_piece(full_cfg, rank, world, args.shard)
    gen_cfg = full_cfg if args.shard == "subband" and world > 1 else cfg   # generator sees global subband indices
    strong = args.shard in ("subband", "dm") and world > 1

    import torch
    import torch.distributed as dist
    from paper_1607_00909_b200 import cdmt

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()

    # ---- synthetic observation -> HBM (not timed)
    nthreads = args.gen_threads or max(1, (os.cpu_count() or 1) // max(1, world))
    int8 = cfg.in_dtype == synth.IN_CI8
    if int8:
        d_in = torch.empty((cfg.nsub, 2, cfg.nsamp, 2), dtype=torch.int8, device=dev)
    else:
        d_in = torch.empty((cfg.nsub, 2, cfg.nsamp), dtype=torch.complex64, device=dev)
    want_e2e = not args.no_e2e
    h_in = None
    if want_e2e:
        h_in = torch.empty(d_in.shape, dtype=d_in.dtype).pin_memory()
    x_sub0 = None
    from concurrent.futures import ThreadPoolExecutor
    t_gen = time.perf_counter()
    with ThreadPoolExecutor(nthreads) as ex:
        for s, xs in zip(range(cfg.nsub), ex.map(lambda s: synth.generate_subband(gen_cfg, sub0 + s), range(cfg.nsub))):
            if s == 0:
                x_sub0 = xs
            t = torch.from_numpy(xs)
            if h_in is not None:
                h_in[s].copy_(t)
                d_in[s].copy_(h_in[s], non_blocking=True)
            else:
                d_in[s].copy_(t)
    torch.cuda.synchronize()
    t_gen = time.perf_counter() - t_gen

    plan = cdmt.cdmt_plan_create(**cfg.plan_kwargs())
    if args.chunk_units:
        cdmt.cdmt_plan_set_option(plan, cdmt.OPT_CHUNK_UNITS, args.chunk_units)
    if args.dm_tile:
        cdmt.cdmt_plan_set_option(plan, cdmt.OPT_DM_TILE, args.dm_tile)
    if args.fused_kernel:
        cdmt.cdmt_plan_set_option(plan, cdmt.OPT_FUSED_KERNEL, args.fused_kernel)
    if args.host_group_blocks:
        cdmt.cdmt_plan_set_option(plan, cdmt.OPT_HOST_GROUP_BLOCKS, args.host_group_blocks)
    q = cdmt.cdmt_plan_query(plan, cfg.nsamp)
    nch = cfg.nsub * cfg.nchan
    nt = q["nout_per_chan"]
    ws = torch.empty(q["workspace_bytes"], dtype=torch.uint8, device=dev)

    # output: the whole filterbank set if it fits beside the rest, else block groups through one buffer
    free_b, _ = torch.cuda.mem_get_info(dev)
    out_bytes = q["out_bytes"]
    groups = 1
    while out_bytes / groups > 0.6 * free_b:
        groups += 1
    nb_total = q["nblock"]
    nb_group = (nb_total + groups - 1) // groups
    out = torch.empty((cfg.ndm, nb_group * cfg.nvalid_dec, nch), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        """One pass of the whole hot path over the observation (block groups share `out`)."""
        launches = 0
        b0 = 0
        while b0 < nb_total:
            nb = min(nb_group, nb_total - b0)
            ns = (nb - 1) * cfg.step + cfg.nfft
            off = b0 * cfg.step
            esz = 2 if int8 else 8
            cdmt.cdmt_execute(plan, d_in.data_ptr() + off * esz, ns, cfg.nsamp, out, out[0].numel(),
                              ws, ws.numel(), stream)
            launches += cdmt.cdmt_last_launch_count(plan)
            b0 += nb
        return launches

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    # ---- timed region: K steps, device time, max over ranks
    cdmt.cdmt_plan_set_option(plan, cdmt.OPT_PROFILE, 1)
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    e0.record(stream)
    launches = 0
    for _ in range(args.steps):
        launches += step()
    e1.record(stream)
    torch.cuda.synchronize()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    prof = cdmt.cdmt_profile_read(plan)
    cdmt.cdmt_plan_set_option(plan, cdmt.OPT_PROFILE, 0)
    ms = max_over_ranks(ms, world, dev)
    sec_per_step = ms * 1e-3 / args.steps
    samples_dm = float(cfg.nsub) * cfg.nsamp * cfg.ndm
    # weak: every rank processed a whole observation; strong: the ranks share one
    value = whole_job_value(full_cfg, 1, sec_per_step) if strong else whole_job_value(cfg, world, sec_per_step)

    # ---- roofline of the dominant kernel (fused per-DM kernel): ALU bound
    units_per_step = cfg.nsub * nb_total
    flops_per_launch = algorithmic_flops_per_unit_dm(cfg) * cfg.ndm * units_per_step * args.steps / max(1, prof["n_fused"])
    ms_per_launch = prof["ms_fused"] / max(1, prof["n_fused"])
    achieved = flops_per_launch / (ms_per_launch * 1e-3) / 1e12
    scratch = torch.empty(148 * 2 * 1024, dtype=torch.float32, device=dev)
    fma_peak = cdmt.cdmt_measure_fp32_peak(scratch, scratch.numel() * 4, 3)
    roofline = {"bound": "alu", "kernel": "k_fused", "achieved": achieved, "peak": FP32_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": achieved / FP32_PEAK_TFLOPS,
                "traffic": (FUSED_TRAFFIC_BYTES_PER_UNIT[cfg.name] * units_per_step * args.steps / max(1, prof["n_fused"]))
                           if cfg.name in FUSED_TRAFFIC_BYTES_PER_UNIT and not args.dm_tile else None,
                "traffic_source": "profiles/r2_ws_c3.md (ncu --set full, one launch of 4032 units, scaled to this launch's units)",
                "peak_source": "derived: 148 SM x 128 lanes x 2 x 1.965 GHz",
                "fma_peak_measured_tflops": fma_peak,
                "ms_per_launch": ms_per_launch, "launches_timed": prof["n_fused"],
                "flops_per_launch": flops_per_launch,
                "share_of_step": prof["ms_fused"] / ms,
                "forward_fft_ms_per_step": prof["ms_forward"] / args.steps}

    # ---- extra (not part of `value`): Alg. 1 l.104-106, 8-bit redigitisation of the filterbanks.  The block
    # sums come out of the fused kernel (cdmt_execute_sums), so the redigitisation proper reads the float32
    # filterbank once: 4 bytes read + 1 byte written per sample.  Timed on the last block group of the step
    # (the whole observation when the output is resident), and the whole device path with 8-bit output.
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm = float(peaks.get("hbm_gbs", 0)) or None
    redig = None
    if not args.no_redigitize:
        try:
            nb_last = nb_total - (groups - 1) * nb_group
            b0_last = (groups - 1) * nb_group
            nws = cdmt.cdmt_redigitize_workspace_bytes(plan, nb_group)
            d_codes = torch.empty((cfg.ndm, nb_group * cfg.nvalid_dec, nch), dtype=torch.uint8, device=dev)
            d_off = torch.empty((cfg.ndm, nch), dtype=torch.float32, device=dev)
            d_sc = torch.empty((cfg.ndm, nch), dtype=torch.float32, device=dev)
            d_sums = torch.empty(nws // 8, dtype=torch.float64, device=dev)
            esz = 2 if int8 else 8

            def group_8bit(b0, nb):
                ns = (nb - 1) * cfg.step + cfg.nfft
                cdmt.cdmt_execute_sums(plan, d_in.data_ptr() + b0 * cfg.step * esz, ns, cfg.nsamp, out, out[0].numel(),
                                       d_sums, ws, ws.numel(), stream)
                cdmt.cdmt_redigitize_sums(plan, out, out[0].numel(), nb, 64.0, 16.0, d_sums, d_codes,
                                          d_codes[0].numel(), d_off, d_sc, stream)

            group_8bit(b0_last, nb_last)          # leaves the last group's filterbank and sums in place
            r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = 3
            r0.record(stream)
            for _ in range(reps):
                cdmt.cdmt_redigitize_sums(plan, out, out[0].numel(), nb_last, 64.0, 16.0, d_sums, d_codes,
                                          d_codes[0].numel(), d_off, d_sc, stream)
            r1.record(stream)
            torch.cuda.synchronize()
            rms = r0.elapsed_time(r1) / reps
            rbytes = 5.0 * cfg.ndm * nb_last * cfg.nvalid_dec * nch
            # the whole device path with 8-bit output: every group through execute_sums + redigitize_sums
            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ksteps = max(1, min(args.steps, 3))
            s0.record(stream)
            for _ in range(ksteps):
                for b0 in range(0, nb_total, nb_group):
                    group_8bit(b0, min(nb_group, nb_total - b0))
            s1.record(stream)
            torch.cuda.synchronize()
            step8 = s0.elapsed_time(s1) / ksteps
            redig = {"ms_per_call": rms, "bytes": rbytes, "achieved_gbs": rbytes / rms / 1e6,
                     "peak_gbs": hbm, "frac": (rbytes / rms / 1e6 / hbm) if hbm else None,
                     "peak_source": "MEASURED_PEAKS.json hbm_gbs" if hbm else "unavailable",
                     "launches": int(cdmt.cdmt_last_launch_count(plan)), "blocks": int(nb_last),
                     "step_ms_8bit_output": step8,
                     "value_8bit_output": whole_job_value(full_cfg, 1, step8 * 1e-3) if strong else
                                          whole_job_value(cfg, world, step8 * 1e-3),
                     "note": "cdmt_redigitize_sums (channel statistics + quantisation; block sums taken inside the "
                             "fused kernel) on the last block group of the step; step_ms_8bit_output = the whole "
                             "device-resident path with 8-bit output (cdmt_execute_sums + cdmt_redigitize_sums per "
                             "group); neither is part of `value`"}
            del d_codes, d_sums
        except Exception as e:   # never lose the headline line to the extra leg
            redig = {"error": str(e)}

    # ---- extra (not part of `value`): incoherent dedispersion of every coherent filterbank over fine DM
    # offsets spanning the coherent DM step at PAPER.md:141's 0.002 pc/cm3 (semi-coherent search), streamed
    # group by group: execute writes each block group behind the shift_range rows carried over from the
    # previous one, so the stage also runs where the filterbanks are never resident at once (c5).
    incoh = None
    if not args.no_incoherent:
        try:
            dm_step = float(cfg.dm[1] - cfg.dm[0]) if cfg.ndm > 1 else 1.0
            nhalf = int(round(0.5 * dm_step / args.fine_step))
            ddm = np.round(np.arange(-nhalf, nhalf + 1) * args.fine_step, 9)
            qi = cdmt.cdmt_incoherent_query(plan, ddm, nt)
            R, nout = qi["shift_range"], qi["nt_out"]
            rows_g = nb_group * cfg.nvalid_dec
            del out
            torch.cuda.empty_cache()
            win = torch.empty((cfg.ndm, R + rows_g, nch), dtype=torch.float32, device=dev)
            out = win[:, R:]                               # where cdmt_execute writes a group
            d_ts = torch.empty((cfg.ndm, len(ddm), nout), dtype=torch.float32, device=dev)
            d_iws = torch.empty(max(256, qi["workspace_bytes"]), dtype=torch.uint8, device=dev)
            esz = 2 if int8 else 8
            wstride = win[0].numel()

            def semicoherent_step(timers=None):
                done = 0
                for gi, b0 in enumerate(range(0, nb_total, nb_group)):
                    nb = min(nb_group, nb_total - b0)
                    ns = (nb - 1) * cfg.step + cfg.nfft
                    cdmt.cdmt_execute(plan, d_in.data_ptr() + b0 * cfg.step * esz, ns, cfg.nsamp, out.data_ptr(),
                                      wstride, ws, ws.numel(), stream)
                    n = nb * cfg.nvalid_dec
                    nt_in = n if gi == 0 else R + n
                    src = out.data_ptr() if gi == 0 else win.data_ptr()
                    if timers is not None:
                        ev = torch.cuda.Event(enable_timing=True); ev.record(stream); timers.append(ev)
                    cdmt.cdmt_incoherent_dedisperse(plan, src, wstride, nt_in, ddm, d_ts.data_ptr() + 4 * done,
                                                    d_ts[0].numel(), nout, d_iws, d_iws.numel(), stream)
                    if b0 + nb < nb_total:
                        cdmt.cdmt_incoherent_carry(plan, win, wstride, R + n, R, stream)
                    if timers is not None:
                        ev = torch.cuda.Event(enable_timing=True); ev.record(stream); timers.append(ev)
                    done += nt_in - R
                return done

            assert semicoherent_step() == nout             # warm-up
            reps = 2
            i0, i1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            timers = []
            i0.record(stream)
            for _ in range(reps):
                semicoherent_step(timers)
            i1.record(stream)
            torch.cuda.synchronize()
            step_ms = i0.elapsed_time(i1) / reps
            ims = sum(timers[2 * k].elapsed_time(timers[2 * k + 1]) for k in range(len(timers) // 2)) / reps
            adds_def, adds_done = cdmt.cdmt_incoherent_work(plan, ddm, nt)
            peak_add = 148 * 128 * 1.965e9 / 1e12
            # shared-memory bound: every addition the kernel performs reads at most one 4-byte word; the
            # register window makes it (8 + spread) words per 8 (1 + spread) additions
            incoh = {"ms_per_step": ims, "groups": groups, "fine_trials": len(ddm), "fine_step": args.fine_step,
                     "trial_groups": qi["ngroups"], "shift_range": R,
                     "adds_definition": adds_def, "adds_performed": adds_done,
                     "speedup_over_definition": adds_def / adds_done,
                     "bound": "alu", "achieved_tadd_s": adds_done / ims / 1e9, "peak_tadd_s": peak_add,
                     "frac": adds_done / ims / 1e9 / peak_add,
                     "definition_tadd_s": adds_def / ims / 1e9,
                     # every addition into a run sum reads one 4-byte word from shared memory: 32 words per
                     # clock and SM; the time those reads alone take (the bound of this formulation)
                     "smem_floor_ms": adds_done * 4.0 / 128.0 / (148 * 1.965e9) * 1e3,
                     "frac_of_smem_floor": adds_done * 4.0 / 128.0 / (148 * 1.965e9) * 1e3 / ims,
                     "peak_source": "derived: 148 SM x 128 FP32 lanes x 1.965 GHz (one FADD per lane and clock)",
                     "out_bytes": int(d_ts.numel() * 4), "semicoherent_step_ms": step_ms,
                     "note": "cdmt_incoherent_dedisperse (+ cdmt_incoherent_carry) on every block group of the step, "
                             "streamed through a window of shift_range + group rows; not included in value; `frac` "
                             "counts the additions the kernel performs (runs of channels that share their shifts are "
                             "summed once per distinct shift), `definition_tadd_s` those of the brute-force "
                             "definition; semicoherent_step_ms = execute + incoherent for the whole observation"}
            del d_ts, d_iws, win
            out = None
        except Exception as e:
            incoh = {"error": str(e)}

    # ---- end to end through the host-buffer entry point (pinned host memory, copies timed): float32
    # filterbanks (the output `value` is measured on) and the paper's 8-bit product (Alg. 1 l.104-108)
    e2e = None
    e2e_u8 = None
    if want_e2e:
        out = None
        torch.cuda.empty_cache()
        ksteps = max(1, min(args.steps, 3))

        def host_leg(kind):
            lay = cdmt.cdmt_host_layout(plan, cfg.nsamp, kind)
            u8 = kind == cdmt.OUT_U8
            h_out = torch.empty((cfg.ndm, nt, nch), dtype=torch.uint8 if u8 else torch.float32).pin_memory()
            h_off = torch.empty((lay["ngroups"], cfg.ndm, nch), dtype=torch.float32).pin_memory() if u8 else None
            h_sc = torch.empty((lay["ngroups"], cfg.ndm, nch), dtype=torch.float32).pin_memory() if u8 else None
            d_scr = torch.empty(lay["scratch_bytes"], dtype=torch.uint8, device=dev)

            def call():
                cdmt.cdmt_execute_host_async(plan, h_in.data_ptr(), cfg.nsamp, cfg.nsamp, kind, h_out.data_ptr(),
                                             h_off.data_ptr() if u8 else 0, h_sc.data_ptr() if u8 else 0, 64.0, 16.0,
                                             d_scr, d_scr.numel(), stream)
                stream.synchronize()
            call()
            barrier()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(ksteps):
                call()
            torch.cuda.synchronize()
            dt = (time.perf_counter() - t0) / ksteps
            dt = max_over_ranks(dt, world, dev)
            return {"value": whole_job_value(full_cfg, 1, dt) if strong else whole_job_value(cfg, world, dt),
                    "unit": UNIT, "h2d_bytes_per_step": int(lay["h2d_bytes"]), "d2h_bytes_per_step": int(lay["d2h_bytes"]),
                    "ms_per_step": dt * 1e3, "steps": ksteps, "groups": lay["ngroups"],
                    "api": "cdmt_execute_host_async(%s) + stream synchronize (pinned host in/out, double-buffered "
                           "copy streams)" % ("CDMT_OUT_U8" if u8 else "CDMT_OUT_F32")}

        e2e = host_leg(cdmt.OUT_F32)
        torch.cuda.empty_cache()
        try:
            e2e_u8 = host_leg(cdmt.OUT_U8)
        except Exception as e:
            e2e_u8 = {"error": str(e)}

    # ---- CPU baseline: the oracle, as it stands, on a bounded sample (rank 0, N=1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        from oracle import cdmt_oracle as orc
        ncores = orc.num_threads()
        nun = oracle_sample_size(cfg, ncores, 14)       # about 10-30 s of CPU work
        xs = [x_sub0] + [synth.generate_subband(cfg, s) for s in range(1, (nun + cfg.nblock - 1) // cfg.nblock)]
        rate, dt, ncores = oracle_sample(cfg, nun, xs)
        cpu = {"value": rate, "unit": UNIT, "cores": ncores, "kind": "oracle", "seconds": dt,
               "sample": "%d of %d (subband, block) units of %s x all %d DMs" % (
                   nun, cfg.nsub * cfg.nblock, cfg.name, cfg.ndm)}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": sec_per_step * 1e3, "higher_is_better": True,
            "scaling": "strong" if strong else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(full_cfg if strong else cfg, args),
            "real_time_factor": cfg.nsamp * synth.TSAMP_S / sec_per_step,
            "clocks": clocks, "e2e": e2e, "e2e_8bit_output": e2e_u8, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu, "redigitize": redig, "incoherent": incoh,
            "gen_seconds": t_gen, "out_groups": groups,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
