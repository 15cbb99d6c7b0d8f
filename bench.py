#!/usr/bin/env python
"""bench.py — site-update throughput of the KPZ/ASEP hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config all|1|2|3|4|5|4-aux-i|4-aux-ii|2d-512|2d-1024|2d-2048|2d-32768|2-fill|3-fill|paper-...]
                    [--impl reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: reset to the
initial state (a1), run the configuration's full number of MCS with its record times (a2-a7 / a9), records left in
device memory.

Default (`--config all`): BASELINE.json's `metric` names no configuration, so the headline (top-level `value`,
`ms_per_step`, `config.workload`, `roofline`, `cpu_baseline`, `e2e`, `clocks`) is the LARGEST single-GPU configuration,
config 3 (512 rings x 16384 sites x 10^5 MCS = 8.39e11 site updates), and the same line carries one full sub-record
per other BASELINE configuration (1, 2, 4, 5), for the two auxiliary streamed runs of SURVEY §8(d) (4-aux-i: L=2^28
ring in L2; 4-aux-ii: L=2^32, the HBM roofline case) and for the 2+1D workloads 2d-512 / 2d-1024 under `"per_config"`, each timed with its own K steps after W
warm-up steps.  `--config X` runs one workload only.

value      site updates / s (GSU/s) of the whole job, device-timed (CUDA events on the launching stream), inputs
           resident in HBM when the timed region starts.
e2e        same metric through the C ABI with HOST buffers: pinned initial lattice -> device, kpz_set_lattice,
           kpz_run, kpz_roughness (records -> host) and the final lattice -> pinned host, all inside the timed region.
roofline   the dominant kernel against the bound DESIGN.md §6 derives for it: `frac` = ALGORITHMIC slots (or bytes) per
           second / peak.  `traffic` and `measured` (ncu pipe / issue utilisation of the same launch shape) are read from
           the committed capture table profiles/ncu_counters.csv (`traffic_source` names the row's capture) or are null.
cpu_baseline  the oracle (oracle/, as it stands) on one host core over a bounded sample of the same workload.

N > 1 (torchrun): every rank runs the same workloads on its own samples (first_sample = rank * S): weak scaling, no
collective on the data path; time = max over ranks.

--impl reference times the CPU oracle (there is no reference implementation to install: /root/reference holds only
the paper's text) on the headline workload (or on --config X).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "site_updates_per_sec"
UNIT = "GSU/s"


# ---------------------------------------------------------------------------------------------------------------
# roofline model: algorithmic cost per site-update of the dominant kernel of each workload
# ---------------------------------------------------------------------------------------------------------------
# alu-pipe slots per site update of the on-chip / blocked sweeps and the two-lane kernel: one slot =
# one LOP3 / SHF / IMAD.WIDE lane-instruction; the pipe takes 0.5 warp-instructions per clock and SMSP (measured).
#   Philox call = 34 slots per 128 elements and plane; pair logic 3 LOP3 per 32 pairs and pass; 4 SHF per MCS.
ALU_SLOTS_PER_SU = {
    1: (2 * 4 * 3 + 4) / 256,                       # p=1, q=0: no plane, logic only
    2: (2 * 2 * 34 + 2 * 4 * 3 + 4) / 256,          # 2 planes
    3: (2 * 1 * 34 + 2 * 4 * 3 + 4) / 256,          # 1 plane (slow sites only)
    4: (2 * 7.33 * (34 + 12) + 2 * 4 * 3 + 4) / 256,  # 32-plane thresholds: log2(64)+1.33 planes per unit and pass
    5: (2 * 2.0 * 34 + 2 * 2 * 4 * 5 + 2 * 4 * 4) / 256,  # two-lane: lane changes dominate
    "2-fill": (2 * 2 * 34 + 2 * 4 * 3 + 4) / 256,
    "3-fill": (2 * 1 * 34 + 2 * 4 * 3 + 4) / 256,
    "4-aux-i": (2 * 2 * 34 + 2 * 4 * 3 + 4) / 256,
    "4-aux-ii": (2 * 2 * 34 + 2 * 4 * 3 + 4) / 256,
    "4-aux-i-blocked": (2 * 2 * 34 + 2 * 4 * 3 + 4) / 256,
    # paper parameter sets (p = 0.8: a 30-plane threshold, ~26 forward-active pairs per unit: log2(26)+1.33 planes;
    # offsets alternate, so the frame changes twice per MCS)
    "paper-1024x30": (2 * 6.0 * (34 + 12) + 2 * 4 * 3 + 8) / 256,
    "paper-1024-fill": (2 * 6.0 * (34 + 12) + 2 * 4 * 3 + 8) / 256,
    "paper-qtasep-16384": (2 * 6.0 * (34 + 12) + 2 * 4 * 3 + 8) / 256,
    "paper-qssep-4096": (2 * 7.0 * (34 + 12) + 2 * 4 * 3 + 8) / 256,
    # paper two-lane model: per 128 sites of both lanes and MCS: in-lane p = 0.5 (1 plane per lane and pass, pair streams
    # cover 256 sites per call: 2 lanes x 2 passes x 0.5 call) + crossings 2 steps x (log2(32 live)+1.33 planes) x (34+12)
    "paper-lanes-4096": (2 * 34 + 2 * 6.33 * (34 + 12) + 2 * 2 * 4 * 5 + 2 * 4 * 4) / 256,
}
# 2+1D generalisation: per Philox supergroup (128 elements = the active half of 256 sites of a row) and
# colour pass: p = 0.75 needs 2 planes (2 x 34 slots); per 32-site word 3 LOP3/SHF for the two-pair eligibility, 1 for the
# acceptance, 2 for the flips of sx (the sy flips are memory operations); 2 passes per MCS over Lx Ly / 256 supergroups
ALU_SLOTS_PER_SU["2d-2048"] = ALU_SLOTS_PER_SU["2d-1024"] = ALU_SLOTS_PER_SU["2d-512"] = ALU_SLOTS_PER_SU["2d-512-cluster"] = 2 * (2 * 34 + 8 * 6) / 256
for _L in (512, 1024, 2048, 4096, 8192, 16384, 32768):   # the paper's size scan: same rates and schedule as paper-1024x30
    ALU_SLOTS_PER_SU[f"paper-scan-{_L}"] = ALU_SLOTS_PER_SU["paper-1024x30"]
# default run: the headline first, then the other BASELINE configs and the auxiliary streamed runs of SURVEY §8(d)
HEADLINE = 3
DEFAULT_SET = [3, 1, 2, 4, 5, "4-aux-i", "4-aux-ii", "2d-512", "2d-1024"]   # the last two: SURVEY 8(f)-4, not BASELINE configs
ALU_SLOTS_PER_CLK_SMSP = 0.5
# streamed sweep: one read + one write of the bit-packed ring per sub-lattice pass = 2 passes * 2 * 1/8 B
STREAM_BYTES_PER_SU = 0.5
PATH_NAMES = {1: "on-chip K1", 2: "streamed K3 (one launch per pass)", 3: "blocked stream K3T (32 MCS per launch)"}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            with open(path) as f:
                d = json.load(f)
            return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
        except Exception:
            pass
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def ncu_counters(cfg_key):
    """Row of profiles/ncu_counters.csv for this workload (written from `ncu --set full` captures of one launch of the
    dominant kernel in the launch shape bench.py times; the row names its capture), or None."""
    path = os.path.join(ROOT, "profiles", "ncu_counters.csv")
    if not os.path.exists(path):
        return None
    import csv
    with open(path) as f:
        for row in csv.DictReader(r for r in f if not r.startswith("#")):
            if row.get("config_key") == str(cfg_key):
                return row
    return None


# ---------------------------------------------------------------------------------------------------------------
# clock sampling during the timed region (NVML; nvidia-smi as a fallback)
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        self._h = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            phys = index
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            if vis:
                try:
                    phys = int(vis.split(",")[index])
                except Exception:
                    phys = index
            self._h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._h = None

    def _loop(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                for bit, name in self.REASONS.items():
                    if r & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.004)

    def start(self):
        if self._h is not None:
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()

    def stop(self):
        if self._thread is not None:
            self._stop.set()
            self._thread.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unsampled"]}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


# ---------------------------------------------------------------------------------------------------------------
# CPU oracle legs
# ---------------------------------------------------------------------------------------------------------------
def _oracle_sim(cfg, nsamples, first_sample=0):
    from oracle import kpzref as R  # test infrastructure: only the cpu_baseline / reference legs load it
    if cfg["kind"] == "lanes":
        return R.LanesRef(cfg["L"], nsamples, cfg["p_a"], cfg["p_b"], cfg["rho0"], cfg["turn_prob"], cfg["turn_period"],
                          cfg["omega"], seed=cfg["seed"], first_sample=first_sample,
                          offset_mode=cfg.get("offset_mode", 0), w_unflagged=cfg.get("w_unflagged"),
                          independent=cfg.get("independent", 0))
    if cfg["kind"] == "kpz2d":
        return R.Kpz2dRef(cfg["Lx"], cfg["Ly"], nsamples, cfg["p"], cfg["q"], seed=cfg["seed"], first_sample=first_sample,
                          offset_mode=cfg.get("offset_mode", 0))
    return R.KpzRef(cfg["L"], nsamples, cfg["p"], cfg["q"], disorder=cfg["disorder"], seed=cfg["seed"],
                    first_sample=first_sample, offset_mode=cfg.get("offset_mode", 0))


def oracle_sample_shape(cfg, target_su):
    """A bounded sample of the workload: whole samples first, then a prefix of the MCS; about target_su site updates."""
    per_mcs = (2 if cfg["kind"] == "lanes" else 1) * cfg["L"]
    if cfg["kind"] == "kpz2d":
        target_su //= 10   # the 2+1D oracle assembles every uniform on its own (32 Philox calls per site): ~2 MSU/s
    n_mcs = int(max(1, min(cfg["n_mcs"], target_su // per_mcs)))
    nsamp = int(max(1, min(cfg["S"], target_su // (per_mcs * n_mcs))))
    return nsamp, n_mcs


def time_oracle(cfg, nsamp, n_mcs, first_sample=0):
    sim = _oracle_sim(cfg, nsamp, first_sample)
    sim.set_record_times([t for t in cfg["record_times"] if t <= n_mcs])
    t0 = time.perf_counter()
    sim.run(n_mcs)
    if cfg["kind"] == "lanes":
        sim.currents()
    else:
        sim.roughness()
    dt = time.perf_counter() - t0
    sim.close()
    return workloads.site_updates(cfg, n_mcs, nsamp) / dt / 1e9, dt


def run_reference(args, cfg, cfg_key):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    nsamp, n_mcs = oracle_sample_shape(cfg, 8_000_000)   # ~1 s of one host core per step
    for w in range(args.warmup):
        time_oracle(cfg, nsamp, n_mcs, first_sample=w)
    t_total, su = 0.0, 0
    for k in range(args.steps):
        _, dt = time_oracle(cfg, nsamp, n_mcs, first_sample=args.warmup + k)
        t_total += dt
        su += workloads.site_updates(cfg, n_mcs, nsamp)
    value = su / t_total / 1e9
    sample = f"{nsamp} sample(s) x {n_mcs} MCS of {cfg['name']} per step (of {cfg['S']} x {cfg['n_mcs']})"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_total / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": cfg["name"], "config_key": str(cfg_key), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------------------------
# CUDA path
# ---------------------------------------------------------------------------------------------------------------
def make_sim(pkg, cfg, first_sample):
    nrec = len(cfg["record_times"])
    if cfg["kind"] == "lanes":
        sim = pkg.LanesSim(cfg["L"], cfg["S"], cfg["p_a"], cfg["p_b"], cfg["rho0"], cfg["turn_prob"], cfg["turn_period"],
                           cfg["omega"], seed=cfg["seed"], first_sample=first_sample, max_records=nrec,
                           offset_mode=cfg.get("offset_mode", 0), w_unflagged=cfg.get("w_unflagged"),
                           independent=cfg.get("independent", 0))
    elif cfg["kind"] == "kpz2d":
        sim = pkg.Kpz2dSim(cfg["Lx"], cfg["Ly"], cfg["S"], cfg["p"], cfg["q"], seed=cfg["seed"], first_sample=first_sample,
                           max_records=nrec, offset_mode=cfg.get("offset_mode", 0), path=cfg.get("path", 0))
    else:
        sim = pkg.KpzSim(cfg["L"], cfg["S"], cfg["p"], cfg["q"], disorder=cfg["disorder"], seed=cfg["seed"],
                         first_sample=first_sample, max_records=nrec, path=cfg.get("path", 0),
                         offset_mode=cfg.get("offset_mode", 0))
    sim.set_record_times(cfg["record_times"])
    return sim


class Ctx:
    """Process-wide state of the CUDA arm: device, ranks, the L2-flush buffer."""

    def __init__(self):
        import torch
        import torch.distributed as dist

        import paper_1012_0385_b200 as pkg

        self.torch, self.dist, self.pkg = torch, dist, pkg
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        if not torch.cuda.is_available():
            raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
        torch.cuda.set_device(self.local_rank)
        self.dev = torch.device("cuda", self.local_rank)
        if self.world > 1:
            dist.init_process_group("nccl", device_id=self.dev)
        pkg.load_library()
        self.sm_count = int(torch.cuda.get_device_properties(self.dev).multi_processor_count)
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)   # > 126 MB L2
        self.peaks = measured_peaks()

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def max_over_ranks(self, values):
        t = self.torch.tensor(list(values), dtype=self.torch.float64, device=self.dev)
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return [float(x) for x in t]

    def close(self):
        if self.world > 1:
            self.dist.destroy_process_group()


def bench_one(ctx, args, cfg_key, with_cpu):
    """K timed steps of one workload after W warm-up steps; returns the record of that workload (on every rank)."""
    torch, pkg = ctx.torch, ctx.pkg
    cfg = dict(workloads.CONFIGS[cfg_key])
    n_mcs = cfg["n_mcs"] if args.mcs is None else args.mcs
    if args.mcs is not None:
        cfg = workloads.truncated(cfg, n_mcs)
    if args.samples is not None:
        cfg["S"] = args.samples
    su_step = workloads.site_updates(cfg)
    from paper_1012_0385_b200 import shard
    sim = make_sim(pkg, cfg, first_sample=shard.weak_first_sample(cfg["S"], ctx.rank))   # global sample indices
    stream = torch.cuda.current_stream()
    world = ctx.world

    def step(ev=None):
        if ev:
            ev[0].record(stream)
        sim.reset()
        if ev:
            ev[1].record(stream)
        sim.run(n_mcs)
        if ev:
            ev[2].record(stream)

    for _ in range(args.warmup):
        ctx.flush.fill_(1)
        step()
    ctx.barrier()

    sampler = ClockSampler(ctx.local_rank)
    events = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    launches0 = pkg.kernel_launches()
    sampler.start()
    wall0 = time.perf_counter()
    for k in range(args.steps):
        ctx.flush.fill_(k & 0xFF)          # L2 flush between timed iterations (outside the events)
        step(events[k])
    ctx.barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    launches = pkg.kernel_launches() - launches0
    t_step = [e[0].elapsed_time(e[2]) for e in events]       # ms, reset + run
    t_run = [e[1].elapsed_time(e[2]) for e in events]        # ms, kpz_run / lanes_run only
    ms_total, ms_run_total = ctx.max_over_ranks([sum(t_step), sum(t_run)])
    value = world * su_step * args.steps / (ms_total * 1e-3) / 1e9
    e2e = time_e2e(ctx, args, cfg, sim, n_mcs, su_step)
    path = sim.path if cfg["kind"] == "kpz" else 1
    path_name = {"kpz": PATH_NAMES.get(path), "lanes": "two-lane K4", "kpz2d": "2+1D checkerboard K5"}[cfg["kind"]]
    if cfg["kind"] == "kpz2d":
        path_name += {1: " (K5S: a sample in the shared memory of a CTA, one launch per run)",
                      3: " (K5C: a sample over the shared memories of a thread-block cluster, one launch per run)"
                      }.get(sim.path, " (K5: one launch per colour pass)")
    ms_run = ms_run_total / args.steps
    roof = roofline(ctx, cfg, cfg_key, path, n_mcs, su_step, ms_run, sim_path=sim.path if cfg["kind"] == "kpz2d" else 0)
    cpu = None
    if cfg.get("no_cpu_baseline"):
        cpu = {"value": None, "unit": UNIT, "cores": 0, "kind": "oracle", "sample": f"not run: {cfg['no_cpu_baseline']}"}
    elif with_cpu and ctx.rank == 0 and world == 1 and not args.no_cpu_baseline:
        nsamp, nm = oracle_sample_shape(cfg, args.cpu_su)
        v, dt = time_oracle(cfg, nsamp, nm)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "sample": f"{nsamp} sample(s) x {nm} MCS of {cfg['name']} (of {cfg['S']} x {cfg['n_mcs']})"}
    sim.close()
    return {
        "value": value, "unit": UNIT, "ms_per_step": ms_total / args.steps, "ms_run_per_step": ms_run,
        # only "paper-1024x30" is a workload the paper quotes a number for (another machine: context)
        "vs_baseline": (value / cfg["paper_gsu"]) if (cfg.get("paper_gsu") and world == 1 and args.mcs is None
                                                      and args.samples is None) else None,
        "config": {"workload": cfg["name"], "config_key": str(cfg_key), "L": cfg["L"], "samples_per_gpu": cfg["S"],
                   "n_mcs": n_mcs, "records": len(cfg["record_times"]),
                   "path": path_name,
                   "l2": "flushed between timed steps (256 MiB fill)", "parallelism": f"samples x{world}"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": cpu,
        "wall_s_timed_region": wall,
    }


def time_e2e(ctx, args, cfg, sim, n_mcs, su_step):
    """The same metric end to end through the public API with HOST buffers inside the timed region."""
    torch = ctx.torch
    if cfg["kind"] == "kpz":
        import numpy as np
        nw = cfg["L"] // 32
        h_in = torch.from_numpy(np.full((cfg["S"], nw), 0xAAAAAAAA, dtype=np.uint32).view(np.int32)).pin_memory()
        h_out = torch.empty((cfg["S"], nw), dtype=torch.int32).pin_memory()
        d_in = torch.empty((cfg["S"], nw), dtype=torch.int32, device=ctx.dev)
        d_out = torch.empty((cfg["S"], nw), dtype=torch.int32, device=ctx.dev)

        def e2e_step():
            sim.reset()
            d_in.copy_(h_in, non_blocking=True)
            sim.set_lattice(d_in)
            sim.run(n_mcs)
            sim.lattice(out=d_out)
            h_out.copy_(d_out, non_blocking=True)
            return sim.roughness()        # syncs; records -> host

        e2e_step()
        ctx.barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            rec = e2e_step()
        ctx.barrier()
        dt, = ctx.max_over_ranks([time.perf_counter() - t0])
        rec_bytes = int(rec["sum_h"].nbytes + rec["sum_h2"].nbytes)
        return {"value": ctx.world * su_step * args.steps / dt / 1e9, "unit": UNIT,
                "h2d_bytes_per_step": int(h_in.numel() * 4), "d2h_bytes_per_step": int(h_out.numel() * 4) + rec_bytes}

    if cfg["kind"] == "kpz2d":
        import numpy as np
        rw, Ly = cfg["Lx"] // 32, cfg["Ly"]
        flat = np.empty((cfg["S"], Ly, rw), dtype=np.uint32)
        flat[:, 0::2, :] = 0xAAAAAAAA
        flat[:, 1::2, :] = 0x55555555
        h_in = torch.from_numpy(flat.view(np.int32)).pin_memory()
        h_out = [torch.empty((cfg["S"], Ly, rw), dtype=torch.int32).pin_memory() for _ in range(2)]
        d_in = torch.empty((cfg["S"], Ly, rw), dtype=torch.int32, device=ctx.dev)

        def e2e_step2d():
            sim.reset()
            d_in.copy_(h_in, non_blocking=True)
            sim.set_slopes(d_in, d_in)
            sim.run(n_mcs)
            sx, sy = sim.slopes()
            h_out[0].copy_(sx, non_blocking=True)
            h_out[1].copy_(sy, non_blocking=True)
            return sim.roughness()        # syncs; records -> host

        e2e_step2d()
        ctx.barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            rec = e2e_step2d()
        ctx.barrier()
        dt, = ctx.max_over_ranks([time.perf_counter() - t0])
        rec_bytes = int(rec["sum_h"].nbytes + rec["sum_h2"].nbytes)
        return {"value": ctx.world * su_step * args.steps / dt / 1e9, "unit": UNIT,
                "h2d_bytes_per_step": int(h_in.numel() * 4), "d2h_bytes_per_step": int(2 * h_in.numel() * 4) + rec_bytes}

    def e2e_step():
        sim.reset()
        sim.run(n_mcs)
        a, b, _ = sim.state()
        ha, hb = a.cpu(), b.cpu()
        return sim.currents(), ha, hb

    e2e_step()
    ctx.barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        cur, ha, hb = e2e_step()
    ctx.barrier()
    dt, = ctx.max_over_ranks([time.perf_counter() - t0])
    return {"value": ctx.world * su_step * args.steps / dt / 1e9, "unit": UNIT, "h2d_bytes_per_step": 0,
            "d2h_bytes_per_step": int(ha.numel() * 4 + hb.numel() * 4 + 4 * cur["j_a"].nbytes),
            "note": "the two-lane initial state is generated on the device from the seed; no host input exists"}


def roofline(ctx, cfg, cfg_key, path, n_mcs, su_step, ms_run, sim_path=0):
    """The dominant kernel against its bound.  `achieved` uses the ALGORITHMIC slots / bytes of the method
    and the device time of kpz_run / lanes_run measured in this run; `traffic` and `measured` come from the committed ncu
    capture table (one launch of the same kernel and launch shape), never from this run."""
    peaks = ctx.peaks
    row = ncu_counters(cfg_key)

    def num(name):
        try:
            return float(row[name]) if row and row.get(name) not in (None, "") else None
        except ValueError:
            return None

    traffic = None
    if row and num("dram_bytes_read") is not None and num("dram_bytes_write") is not None:
        traffic = num("dram_bytes_read") + num("dram_bytes_write")
    measured = None
    if row:
        measured = {k: num(k) for k in ("issue_active_pct", "pipe_alu_pct", "pipe_fma_pct", "pipe_fmaheavy_pct_of_elapsed",
                                        "warps_active_per_smsp", "registers", "gpu_time_us") if num(k) is not None} or None
    src = (f"profiles/ncu_counters.csv row {cfg_key}: {row.get('capture', '')}" if row else None)
    if path == 2 and 2 * cfg["S"] * cfg["L"] / 8 > 126e6:
        # streamed sweep of a ring beyond the L2 (ping-pong pair of S * L / 8 bytes each; a pair that fits the 126 MB L2
        # never reaches HBM and is measured against the alu-slot roofline below): 2*n_mcs pass kernels per run; per
        # launch one read + one write of the ring
        n_launch = 2 * n_mcs
        bytes_launch = 2 * cfg["S"] * cfg["L"] / 8
        achieved = bytes_launch * n_launch / (ms_run * 1e-3) / 1e9
        return {"bound": "hbm", "kernel": "kpz_k3_pass_jit", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": achieved / peaks["hbm_gbs"], "traffic": traffic, "traffic_source": src, "measured": measured,
                "peak_source": peaks["source"], "launches_per_step": n_launch, "algorithmic_bytes_per_launch": bytes_launch}
    if cfg["kind"] == "kpz2d" and sim_path == 2 and cfg["S"] * cfg["L"] / 4 > 126e6:
        # 2+1D streamed beyond the L2 (4 planes of S * Lx * Ly / 16 bytes): per colour pass every plane word is read once
        # and written once (DESIGN.md §5 K5)
        n_launch = 2 * n_mcs
        bytes_launch = cfg["S"] * cfg["L"] / 2
        achieved = bytes_launch * n_launch / (ms_run * 1e-3) / 1e9
        return {"bound": "hbm", "kernel": "kpz2d_k5_pass_jit", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": achieved / peaks["hbm_gbs"], "traffic": traffic, "traffic_source": src, "measured": measured,
                "peak_source": peaks["source"], "launches_per_step": n_launch, "algorithmic_bytes_per_launch": bytes_launch}
    slots = ALU_SLOTS_PER_SU.get(cfg_key)
    kname = {1: "kpz_k1_sweep_jit", 2: "kpz_k3_pass_jit", 3: "kpz_k3t_sweep_jit"}.get(path, "kpz_k1_sweep_jit") if cfg["kind"] == "kpz" \
        else ({1: "kpz2d_k5s_jit", 3: "kpz2d_k5c_jit"}.get(sim_path, "kpz2d_k5_pass_jit") if cfg["kind"] == "kpz2d"
              else "lanes_k4_sweep_jit")
    if slots is None:
        return {"bound": "alu", "kernel": kname, "achieved": None, "peak": None, "unit": "Tslot/s", "frac": None,
                "traffic": traffic, "reason": f"no algorithmic slot count is modelled for workload key {cfg_key!r}"}
    peak = ctx.sm_count * 4 * ALU_SLOTS_PER_CLK_SMSP * 32 * peaks["sm_max_mhz"] * 1e6 / 1e12   # T lane-slots/s
    achieved = slots * su_step / (ms_run * 1e-3) / 1e12
    return {"bound": "alu", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "Tslot/s",
            "frac": achieved / peak, "traffic": traffic, "traffic_source": src, "measured": measured,
            "frac_definition": "algorithmic alu-pipe slots of the method (DESIGN.md 6.1) per second / alu-pipe slot peak; "
                               "`measured` holds the ncu pipe / issue utilisation of the same kernel",
            "peak_source": f"{ctx.sm_count} SM (queried) x 4 SMSP x 0.5 alu-pipe warp-instr/clk (measured, "
                           f"profiles/r01_pipe_rates.md) x 32 lanes x {peaks['sm_max_mhz']:.0f} MHz "
                           f"({peaks['source']} max clock)",
            "algorithmic_slots_per_site_update": slots}


def run_cuda(args, keys):
    ctx = Ctx()
    records = {}
    for i, key in enumerate(keys):
        records[str(key)] = bench_one(ctx, args, key, with_cpu=True)
    if ctx.rank != 0:
        ctx.close()
        return 0
    head = records[str(keys[0])]
    line = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": ctx.world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": head["vs_baseline"], "dtype": "u32", "data": "synthetic", "config": head["config"],
        "clocks": head["clocks"], "e2e": head["e2e"],
        "gpu_launches": int(sum(r["gpu_launches"] for r in records.values())),
        "roofline": head["roofline"], "cpu_baseline": head["cpu_baseline"], "ms_run_per_step": head["ms_run_per_step"],
        "wall_s_timed_region": head["wall_s_timed_region"], "sm_count": ctx.sm_count,
    }
    if len(keys) > 1:
        line["per_config"] = records
        line["headline"] = (f"config {keys[0]}: BASELINE.json's metric names no configuration, so the top-level keys are "
                            f"the largest single-GPU configuration; every other workload is a full sub-record in per_config")
    print(json.dumps(line), flush=True)
    ctx.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", default="all")
    ap.add_argument("--mcs", type=int, default=None, help="truncate the run to this many MCS (diagnostics only)")
    ap.add_argument("--samples", type=int, default=None, help="override the sample count (diagnostics only)")
    ap.add_argument("--debug-config", default=None, help="kpz_debug_config string (kernel tuning knobs; diagnostics only)")
    ap.add_argument("--cpu-su", type=int, default=250_000_000, help="site updates of the cpu_baseline sample per workload")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.config == "all":
        keys = list(DEFAULT_SET)
    else:
        keys = [int(k) if k.isdigit() else k for k in args.config.split(",")]
    if args.impl == "reference":
        return run_reference(args, dict(workloads.CONFIGS[keys[0]]), keys[0])
    if args.debug_config:
        import paper_1012_0385_b200 as pkg
        pkg.debug_config(args.debug_config)
    return run_cuda(args, keys)


if __name__ == "__main__":
    sys.exit(main())
