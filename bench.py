#!/usr/bin/env python
"""bench.py -- throughput of the whole Delphes-chain hot path.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pd_simulate call over one batch: every event of the workload, inputs resident in
HBM.  Default workload: BASELINE.json configs[2] (CMS-like PU200-like pile-up, 10,000 events x ~4,060
particles), the largest config, on which north_star states the bandwidth target.  Prints ONE JSON line.

  value      truth particles/s, whole job (all ranks), device-timed with CUDA events, max over ranks
  e2e        same metric through pd_simulate_host: pinned HOST buffers in and out, copies timed
  roofline   algorithmic HBM bytes of one step (three launches) / its CUDA-event duration, against the
             measured copy bandwidth in MEASURED_PEAKS.json
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on a bounded sample of the same workload:
             one host core, and all host cores (events sharded over worker processes); CPU model stated

N > 1 (torchrun): events are independent, so every rank runs the same-size batch with its own
event_base (weak scaling, no data-path collective); rank 0 prints.
--impl reference: the oracle on the host cores, bounded sample per step (rank 0 only).
"""
import argparse
import importlib
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

wl = importlib.import_module("workloads.generate")

METRIC = "truth particles/sec through Delphes chain"
UNIT = "particles/s"
SAMPLE_PARTICLES = 8_000_000  # cpu_baseline sample: ~10-15 s of one core


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def _traffic(cfg):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed ncu --set full
    capture of this config, if one exists: last matching row of profiles/dram_traffic.csv."""
    val = None
    try:
        with open(os.path.join(ROOT, "profiles", "dram_traffic.csv")) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) >= 2 and c[0] == "cfg%d" % cfg:
                    val = float(c[1])
    except Exception:
        return None
    return val


def _inst_count(cfg):
    """Warp instructions per launch (smsp__inst_executed.sum) from the committed ncu --set full capture of this
    config, if one exists: last matching row of profiles/inst_count.csv."""
    val = None
    try:
        with open(os.path.join(ROOT, "profiles", "inst_count.csv")) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) >= 2 and c[0] == "cfg%d" % cfg:
                    val = float(c[1])
    except Exception:
        return None
    return val


def _sample_events(ev, max_particles):
    """Leading events of the workload holding at most max_particles particles."""
    k = int(np.searchsorted(ev.offsets, max_particles, side="right") - 1)
    k = max(1, min(k, ev.n_events))
    return wl.slice_events(ev, 0, k), k


def _cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def _oracle_warm(cfg):
    from oracle import pdo

    pdo.Card(wl.config_card(cfg))
    return 0


def _oracle_worker(job):
    """One shard of the all-cores oracle run: its own process, its own copy of the oracle library."""
    cfg, seed, e0, arrays = job
    from oracle import pdo

    ev = wl.Events(**arrays)
    card = pdo.Card(wl.config_card(cfg))
    t0 = time.perf_counter()
    pdo.simulate(card, ev, seed, event_base=e0, debug=False)
    return time.perf_counter() - t0, int(ev.n_particles)


def _oracle_rate_all_cores(cfg, ev, seed, per_worker=1_500_000):
    """The same oracle, events sharded over os.cpu_count() worker processes (events are independent and the RNG is keyed by
    the global event index, so the shards reproduce the single run).  Returns particles/s over the wall time of the pool."""
    import multiprocessing as mp

    cores = os.cpu_count() or 1
    sample, k = _sample_events(ev, min(int(ev.n_particles), per_worker * cores))
    bounds = np.linspace(0, k, cores + 1).astype(int)
    jobs = []
    for w in range(cores):
        a, b = int(bounds[w]), int(bounds[w + 1])
        if b <= a:
            continue
        sub = wl.slice_events(sample, a, b)
        jobs.append((cfg, seed, a, {f: getattr(sub, f) for f in ("offsets", "pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")}))
    ctx = mp.get_context("fork")
    with ctx.Pool(len(jobs)) as pool:
        pool.map(_oracle_warm, [cfg] * len(jobs))  # every worker has the library and the card loaded
        t0 = time.perf_counter()
        res = pool.map(_oracle_worker, jobs)
        wall = time.perf_counter() - t0
    n = sum(r[1] for r in res)
    what = "first %d events (%d particles) of %s over %d worker processes" % (k, n, wl.CONFIGS[cfg]["name"], len(jobs))
    return n / wall, len(jobs), what


def _oracle_rate(cfg, ev, seed, steps=1, warmup=0):
    from oracle import pdo

    card = pdo.Card(wl.config_card(cfg))
    sample, k = _sample_events(ev, SAMPLE_PARTICLES)
    for _ in range(warmup):
        pdo.simulate(card, wl.slice_events(sample, 0, max(1, k // 50)), seed, debug=False)
    t0 = time.perf_counter()
    for _ in range(steps):
        pdo.simulate(card, sample, seed, debug=False)
    dt = (time.perf_counter() - t0) / steps
    what = "first %d events (%d particles) of %s" % (k, sample.n_particles, wl.CONFIGS[cfg]["name"])
    return sample.n_particles / dt, dt, what


class _Clocks:
    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.QUERY,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])), mx.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}
        return out


def run_reference(args, rank, world):
    if rank != 0:
        return
    cfg = args.config
    seed = wl.CONFIGS[cfg]["seed"]
    # the oracle only sees a bounded sample: generate just enough events
    avg = {0: 60, 1: 250, 2: 4060, 3: 40, 4: 30}[cfg]
    ne = min(wl.CONFIGS[cfg]["n_events"], max(1, int(1.05 * SAMPLE_PARTICLES / avg) + 2))
    ev = wl.generate(cfg, ne)
    rate, dt, what = _oracle_rate(cfg, ev, seed, steps=max(1, args.steps), warmup=min(args.warmup, 1))
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": wl.CONFIGS[cfg]["name"], "card": wl.config_card(cfg), "sample": what},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": what},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_ours(args, rank, world, local_rank):
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    import paper_2606_26089_b200 as pd

    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    cfg = args.config
    seed = wl.CONFIGS[cfg]["seed"]
    ev = wl.generate(cfg, args.events)
    n, ne = ev.n_particles, ev.n_events
    event_base = rank * ne  # shard r of a world x ne event job (weak scaling)
    card = pd.Card(wl.config_card(cfg))
    dev = pd.DeviceEvents(ev)
    out = pd.DeviceOutputs(card, ne, n, debug=False)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    launches = 0
    for _ in range(args.warmup):
        pd.simulate(card, dev, out, seed, event_base)
    torch.cuda.synchronize()
    status = pd.last_status(out)
    if status != 0:
        raise SystemExit("bench.py: device-side status %d" % status)
    totals = [int(out.trk["offsets"][-1]), int(out.tow["offsets"][-1]), int(out.efl["offsets"][-1])]

    # ---- device-timed region: K steps, per-launch events on the launching stream
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    clocks = _Clocks(local_rank) if rank == 0 else None
    time.sleep(0.25 if clocks else 0.0)
    barrier()
    evs[0].record(stream)
    for k in range(args.steps):
        pd.simulate(card, dev, out, seed, event_base)
        launches += pd.last_launch_count()
        evs[k + 1].record(stream)
    barrier()
    clk = clocks.stop() if clocks else None
    per_launch_ms = [evs[k].elapsed_time(evs[k + 1]) for k in range(args.steps)]
    total_ms = evs[0].elapsed_time(evs[args.steps])
    t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms_max = float(t.item())
    value = world * n * args.steps / (total_ms_max * 1e-3)

    # ---- end-to-end: pinned host buffers through pd_simulate_host, copies inside the timed region
    hb = pd.HostBuffers(ev)
    pd.simulate_host(card, hb, seed, event_base)
    e2e_steps = max(1, min(args.steps, 3))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        pd.simulate_host(card, hb, seed, event_base)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_value = world * n / float(t.item())
    h2d, d2h = hb.h2d_bytes(), hb.d2h_bytes()

    # ---- the next step after the hot path: event features + lepton isolation on the EFlow
    # collection the chain just produced (device-resident).  Reported beside the step, not part of it.
    feat = pd.DeviceFeatures(ne, 2 * max(n, 1))
    for _ in range(2):
        pd.event_features(out, feat)
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    f_steps = max(1, min(args.steps, 5))
    f0.record(stream)
    for _ in range(f_steps):
        pd.event_features(out, feat)
    f1.record(stream)
    barrier()
    feat_ms = f0.elapsed_time(f1) / f_steps
    del feat
    # ---- the particle filter (pT > 0.5 GeV and |eta| < 2.5, AND) on the same EFlow collection
    conds = [{"field": "pt", "op": ">", "value": 0.5}, {"field": "eta", "op": "<", "value": 2.5, "abs": True}]
    dst = pd.DeviceEFlow(ne, 2 * max(n, 1))
    ws_keep = pd.filter_eflow(out, dst, conds, "all")
    pd.filter_eflow(out, dst, conds, "all", workspace=ws_keep)
    barrier()
    f0.record(stream)
    for _ in range(f_steps):
        pd.filter_eflow(out, dst, conds, "all", workspace=ws_keep)
    f1.record(stream)
    barrier()
    filt_ms = f0.elapsed_time(f1) / f_steps
    kept = int(dst.t["offsets"][-1])
    del dst, ws_keep
    # ---- impact parameters d0, z0 and their errors for the step's tracks
    imp = pd.DeviceImpact(max(n, 1))
    ip_res = ((20e-6, 40e-6), (30e-6, 60e-6))
    for _ in range(2):
        pd.track_impact(card, dev, out, imp, *ip_res, seed=seed, event_base=event_base)
    barrier()
    f0.record(stream)
    for _ in range(f_steps):
        pd.track_impact(card, dev, out, imp, *ip_res, seed=seed, event_base=event_base)
    f1.record(stream)
    barrier()
    imp_ms = f0.elapsed_time(f1) / f_steps
    del imp
    # the same values from the chain itself (pd_options.impact: kernel P computes them while the particle is on chip): what the
    # step costs with the option on; its difference to ms_per_step replaces the stand-alone kernel's time
    out_f = pd.DeviceOutputs(card, ne, n, debug=False, impact=ip_res)
    for _ in range(3):
        pd.simulate(card, dev, out_f, seed, event_base)
    barrier()
    f0.record(stream)
    for _ in range(f_steps):
        pd.simulate(card, dev, out_f, seed, event_base)
    f1.record(stream)
    barrier()
    step_imp_ms = f0.elapsed_time(f1) / f_steps
    del out_f
    # ---- H_T and E_T^miss of the truth collection (the step's input)
    tfeat = pd.DeviceFeatures(ne, 1)
    tws = pd.truth_features(dev, tfeat)
    pd.truth_features(dev, tfeat, workspace=tws)
    barrier()
    f0.record(stream)
    for _ in range(f_steps):
        pd.truth_features(dev, tfeat, workspace=tws)
    f1.record(stream)
    barrier()
    truth_ms = f0.elapsed_time(f1) / f_steps
    del tfeat, tws

    # ---- pile-up merging, the step right before the hot path: 5,000 cfg0-like hard-scatter
    # events, a pool of 20,000 cfg3-like minimum-bias events, mean pile-up 50 (Table C.9 defaults otherwise)
    hs_ev, pool_ev = wl.generate(0, 5000), wl.generate(3, 20000)
    d_hs, d_pool = pd.DeviceEvents(hs_ev), pd.DeviceEvents(pool_ev)
    merged = pd.DeviceMerged(hs_ev.n_events, int(hs_ev.n_particles + hs_ev.n_events * 80 * 48))
    for _ in range(2):
        pd.pileup_merge(d_hs, d_pool, merged, 50.0, seed=seed)
    barrier()
    f0.record(stream)
    for _ in range(f_steps):
        pd.pileup_merge(d_hs, d_pool, merged, 50.0, seed=seed)
    f1.record(stream)
    barrier()
    pu_ms = f0.elapsed_time(f1) / f_steps
    pu_total = merged.total()
    assert pd.pileup_status(merged) == 0
    del merged, d_hs, d_pool

    if dist is not None:
        # CSR rebasing of shard outputs: one all-gather of three int64 per rank, outside the data path
        from paper_2606_26089_b200 import shard

        shard.exchange_totals(totals, rank, world, dist, device="cuda")
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the chain.  A step is three launches on the stream -- pd_tile_events_kernel (~10 us), pd_particle_kernel
    # (kernel P) and pd_tower_kernel (kernel T) -- that split the algorithmic bytes between them (P reads the particles and
    # writes nothing that counts, T writes the three collections), so the roofline is taken over the step: algorithmic
    # bytes of one pd_simulate / its CUDA-event duration.  The per-kernel times of the same command are in the committed
    # ncu launch list (profiles/r02*_launches.*).
    alg_bytes = 33 * n + 8 * (ne + 1) + 33 * totals[0] + 28 * totals[1] + 21 * totals[2] + 3 * 8 * (ne + 1)
    kern_ms = float(np.mean(per_launch_ms))
    peak, peak_src = _peaks()
    achieved = alg_bytes / (kern_ms * 1e-3) / 1e9
    # the ALU-side reading of the same launch: warp instructions (from the committed ncu capture)
    # against the issue peak 148 SMs x 4 schedulers x SM clock
    inst = _inst_count(cfg)
    sm_mhz = (clk or {}).get("sm_mhz") or 1965.0
    alu_view = None
    if inst:
        issue_peak = 148 * 4 * sm_mhz * 1e6
        alu_view = {"warp_instructions_per_launch": inst, "warp_instructions_per_particle": inst / max(n, 1),
                    "achieved_warp_inst_per_s": inst / (kern_ms * 1e-3), "issue_peak_warp_inst_per_s": issue_peak,
                    "frac_of_issue_peak": inst / (kern_ms * 1e-3) / issue_peak,
                    "note": "instruction count of the two kernels from profiles/ (ncu), time live; the path is bound by instruction issue and on-chip synchronisation, not by HBM"}
    cpu_rate, cpu_dt, cpu_what = _oracle_rate(cfg, ev, seed)
    try:
        all_rate, all_cores, all_what = _oracle_rate_all_cores(cfg, ev, seed)
    except Exception as exc:  # the baseline is context, never a reason to lose the line
        all_rate, all_cores, all_what = None, 0, "failed: %r" % (exc,)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": wl.CONFIGS[cfg]["name"], "card": wl.config_card(cfg), "events_per_gpu": ne, "particles_per_gpu": n,
                   "tracks": totals[0], "towers": totals[1], "eflow": totals[2], "events_per_s": world * ne * args.steps / (total_ms_max * 1e-3),
                   "l2": "inputs+outputs (%.2f GB) larger than L2, no flush" % (alg_bytes / 1e9), "parallelism": "event sharding x%d" % world,
                   "input_sha256": ev.sha256()[:16], "numpy": np.__version__},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": _traffic(cfg), "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                     "bytes_per_particle": alg_bytes / max(n, 1), "kernel_ms": kern_ms,
                     "kernel": "pd_simulate = pd_tile_events_kernel + pd_particle_kernel + pd_tower_kernel (one step)",
                     "frac_of_8TBs_nominal": achieved / 8000.0, "alu_view": alu_view},
        "cpu_baseline": {"value": cpu_rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": cpu_what, "cpu_model": _cpu_model(),
                         "all_cores": {"value": all_rate, "unit": UNIT, "cores": all_cores, "host_cores": os.cpu_count(), "sample": all_what}},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3},
        "gpu_launches": launches, "clocks": clk,
        "next": {"event_features": {"ms": feat_ms, "objects_per_s": totals[2] / (feat_ms * 1e-3), "kernel": "pd_features_kernel",
                                    "algorithmic_bytes": 29 * totals[2] + 24 * ne,
                                    "hbm_frac": (29 * totals[2] + 24 * ne) / (feat_ms * 1e-3) / 1e9 / peak,
                                    "note": "H_T, MET, lepton isolation (Eq. 1) on the step's EFlow output; rank 0, not in value"},
                 "pileup_merge": {"ms": pu_ms, "merged_particles_per_s": pu_total / (pu_ms * 1e-3), "merged_particles": pu_total,
                                  "kernels": "pd_pileup_count/scan/fill_kernel", "algorithmic_bytes": 67 * pu_total + 20 * hs_ev.n_events,
                                  "hbm_frac": (67 * pu_total + 20 * hs_ev.n_events) / (pu_ms * 1e-3) / 1e9 / peak,
                                  "note": "5,000 cfg0-like events + Poisson(50) of 20,000 cfg3-like min-bias events; 3 launches; rank 0, not in value"},
                 "truth_features": {"ms": truth_ms, "particles_per_s": n / (truth_ms * 1e-3), "kernels": "pd_truth_sum_kernel + pd_truth_finish_kernel",
                                    "algorithmic_bytes": 12 * n + 8 * (ne + 1) + 16 * ne,
                                    "hbm_frac": (12 * n + 8 * (ne + 1) + 16 * ne) / (truth_ms * 1e-3) / 1e9 / peak,
                                    "note": "H_T, MET of the truth collection (neutrinos left out); 2 launches + a memset; rank 0, not in value"},
                 "track_impact": {"ms": imp_ms, "tracks_per_s": totals[0] / (imp_ms * 1e-3), "kernel": "pd_impact_kernel",
                                  "algorithmic_bytes": 45 * totals[0] + 16 * (ne + 1),
                                  "hbm_frac": (45 * totals[0] + 16 * (ne + 1)) / (imp_ms * 1e-3) / 1e9 / peak,
                                  "step_ms_with_impact_option": step_imp_ms, "extra_ms_in_chain": step_imp_ms - total_ms / args.steps,
                                  "note": "d0, z0 and errors (a (+) b/pT) for the step's tracks; stand-alone kernel: truth particles gathered through trk.src, 1 launch; or from the chain itself (pd_options.impact): the whole step then takes step_ms_with_impact_option; rank 0, not in value"},
                 "particle_filter": {"ms": filt_ms, "objects_per_s": totals[2] / (filt_ms * 1e-3), "kept": kept, "kernel": "pd_filter_kernel",
                                     "algorithmic_bytes": 21 * totals[2] + 21 * kept + 16 * (ne + 1),
                                     "hbm_frac": (21 * totals[2] + 21 * kept + 16 * (ne + 1)) / (filt_ms * 1e-3) / 1e9 / peak,
                                     "note": "pT > 0.5 and |eta| < 2.5 on the step's EFlow output; 2 launches; rank 0, not in value"}},
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--events", type=int, default=None, help="override the config's event count (debugging)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
