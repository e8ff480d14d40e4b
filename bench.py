#!/usr/bin/env python
"""bench.py -- throughput of the U(1) multilevel hot path on B200 (BASELINE.json config 5).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One STEP = one pass of the whole hot path over a 64^4 lattice (beta = 0.98, hot start seed 5):
    ul_sweep(1 HB, 4 OR)                      full compound sweep          (rows a2-a5)
    ul_multilevel(d=2, n_sub=24, r_max=16)    n_sub x {slab-masked compound sub-update (1 HB + 4 OR)
                                              + T^(2) accumulation}, slab product, reduction (a6, a7, a10, a13)
    ul_plaquette()                                                          (row a11)
metric = link updates per second (full + masked updates) over the whole step, inputs resident in HBM.
`e2e` = the same step through the C ABI with HOST link buffers (ul_set_links_async / _commit + step + ul_get_links_async: the copies of neighbouring steps overlap the work).
`roofline` = the overrelaxation sub-step kernel (4 of every 5 sweeps), timed with CUDA events inside
the timed region, against its algorithmic 36 B per link update.
`cpu_baseline` = the oracle (oracle/ulo.cpp, single thread) on a bounded sample of the same workload: one slab-masked
sub-update + one accumulation on a 64^3 x 2 sub-lattice; `--impl reference` times the same sample per step.

N > 1 (torchrun): every rank runs an independent lattice (seed 5 + rank), no data-path collective;
times are the max over ranks ("weak" scaling).
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

WORKLOAD = dict(name="cfg5_64^4", Ns=64, Nt=64, beta=0.98, seed=5, n_hb=1, n_or=4, slab_d=2, n_sub=24, r_max=16)
METRIC = "link_updates_per_s"
UNIT = "link updates/s"
BYTES_PER_UPDATE_OR = 36.0     # DESIGN.md / SURVEY 8(d): 3V + V/2 + V/2 reads, V/2 writes per V/2 updates, fp32


def updates_per_step(w):
    V = w["Ns"] ** 3 * w["Nt"]
    sweeps = w["n_hb"] + w["n_or"]
    full = sweeps * 4 * V
    d = w["slab_d"]
    masked = sweeps * (V + 3 * V * (d - 1) // d)
    return full + w["n_sub"] * masked, full, masked


def rank_seed(base_seed, rank):
    """Independent problems per rank (weak scaling): rank r runs the lattice seeded base + r."""
    return int(base_seed) + int(rank)


def distributed_max(value, dist, device=None):
    """max over ranks of a python float through torch.distributed (nccl on GPUs, gloo in CPU tests)."""
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.02):
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def measured_peak_hbm():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic():
    """DRAM bytes per launch of the dominant kernel (dram__bytes_read.sum + dram__bytes_write.sum of its
    `ncu --set full` capture), from the committed summary profiles/roofline_traffic.txt, or None."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.txt")
    try:
        for line in open(p):
            f = line.split()
            if len(f) >= 2 and f[0] == "k_update_or_dram_bytes_per_launch":
                return float(f[1])
    except Exception:
        pass
    return None


# ------------------------------------------------------------------------------------------- oracle arm
ORACLE_SAMPLE_NT = 2     # the oracle's bounded sample: one slab of the workload lattice (same in both arms)


def oracle_sample(w, ns=0):
    """Times the oracle, as it stands, on a bounded sample of the workload (SURVEY 8(d) "Oracle timing"): a
    Ns^3 x 2 sub-lattice (one slab at d = 2; same Ns, beta, seed, hot start), one slab-masked compound sub-update
    (n_hb heatbath + n_or overrelaxation sweeps) followed by one T^(2) accumulation at r <= r_max.  Returns a dict:
    link updates/s over update + accumulation (the step's own mix), the update-only rate, seconds."""
    from oracle import ulo
    Ns, nt, d = (ns or w["Ns"]), ORACLE_SAMPLE_NT, w["slab_d"]
    o = ulo.Oracle(Ns, nt, w["beta"], w["seed"])
    V = Ns ** 3 * nt
    n_upd = (w["n_hb"] + w["n_or"]) * (V + 3 * V * (d - 1) // d)
    t0 = time.perf_counter()
    for kind, n in ((0, w["n_hb"]), (1, w["n_or"])):
        for _ in range(n):
            for parity in (0, 1):
                for mu in range(4):
                    o.substep(kind, parity, mu, d)
    t_upd = time.perf_counter() - t0
    o.measure_begin(d, w["r_max"])
    t0 = time.perf_counter()
    o.accumulate()
    t_acc = time.perf_counter() - t0
    o.close()
    return {"value": n_upd / (t_upd + t_acc), "update_only": n_upd / t_upd, "seconds": t_upd + t_acc, "t_update_s": t_upd,
            "t_accumulate_s": t_acc,
            "sample": f"{Ns}^3x{nt} sub-lattice of the workload (hot start), one slab-masked sub-update ({w['n_hb']} HB + {w['n_or']} OR sweeps, "
                      f"d={d}) = {n_upd} link updates in {t_upd:.2f} s + one T^(2) accumulation r<={w['r_max']} "
                      f"({3 * w['r_max'] * (nt // d) * Ns ** 3} entries) in {t_acc:.2f} s"}


def run_reference(args, rank, world):
    if rank != 0:
        return
    w = WORKLOAD
    vals, secs, last = [], [], None
    for i in range(args.steps + args.warmup):
        last = oracle_sample(w, args.sample_ns)
        if i >= args.warmup:
            vals.append(last["value"])
            secs.append(last["seconds"])
    value = sum(vals) / len(vals)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / len(secs), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w["name"], "lattice": f"{w['Ns']}^3x{w['Nt']}", "beta": w["beta"], "seed": w["seed"],
                   "note": "oracle (single-threaded C++, fp64) on a bounded sample per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": last["sample"],
                         "update_only_link_updates_per_s": last["update_only"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------- our arm
def run_ours(args, rank, local_rank, world):
    import torch
    from paper_1309_3859_b200 import build, ul
    if rank == 0:
        build.build()
    dist = None
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    w = WORKLOAD
    Ns, Nt = w["Ns"], w["Nt"]
    V = Ns ** 3 * Nt
    ws = ul.workspace_bytes(Ns, Nt, w["slab_d"], 0, w["r_max"], 0)
    lat = ul.Lattice(Ns, Nt, w["beta"], rank_seed(w["seed"], rank), workspace_bytes=ws, device=dev)
    lat.set_subupdate(w["n_hb"], w["n_or"], 1)
    n_upd, n_full, n_masked = updates_per_step(w)

    ev_or = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]

    def step(i=None):
        lat.sweep(w["n_hb"], 0)
        if i is not None:
            ev_or[i][0].record()
        lat.sweep(0, w["n_or"])
        if i is not None:
            ev_or[i][1].record()
        lat.multilevel(w["slab_d"], w["n_sub"], w["r_max"])
        return lat.plaquette()[0]

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    l0 = lat.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(args.steps):
        plaq = step(i)
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = lat.launch_count() - l0
    ms = e0.elapsed_time(e1)
    or_ms = sum(a.elapsed_time(b) for a, b in ev_or) / args.steps          # 4 OR sweeps = 32 launches per step
    if dist is not None:
        ms = distributed_max(ms, dist, dev)
    ms_per_step = ms / args.steps
    value = world * n_upd / (ms_per_step * 1e-3)

    # ---- e2e: host buffers through the C ABI, copies inside the timed region
    host_in = torch.empty(4 * V, dtype=torch.float32).pin_memory()
    host_out = torch.empty(4 * V, dtype=torch.float32).pin_memory()
    lat.get_links(host_in)
    e2e_steps = max(2, min(args.steps, 20))
    # every step: its links host -> device (pinned), the step, its links device -> host and the correlators; the read-back is
    # ul_get_links_async, so that it shares the host link with the next step's ul_set_links (the last one is waited for inside
    # the timed region)
    # the upload of a step's links is ul_set_links_async + ul_set_links_commit: the copy of step i + 1 is started before step i
    # runs (on the library's upload stream) and committed when step i is over, so e2e_steps + 1 uploads are inside the timed
    # region for e2e_steps steps
    for _ in range(2):
        lat.set_links(host_in); step(); lat.get_links_async(host_out)
    lat.get_links_wait()
    barrier()
    t0 = time.perf_counter()
    lat.set_links_async(host_in)
    for _ in range(e2e_steps):
        lat.set_links_commit()
        lat.set_links_async(host_in)                  # the next step's input
        step()
        lat.read_correlators()                        # before the read-back of the links: a small copy queues behind a large one
        lat.get_links_async(host_out)
    lat.get_links_wait()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    if dist is not None:
        e2e_ms = distributed_max(e2e_ms, dist, dev)
    e2e_value = world * n_upd / (e2e_ms / e2e_steps * 1e-3)

    # ---- auxiliary figures (the timed region above is over; every rank runs them, rank 0 reports)
    def ev_time(fn, n=5):
        fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n * 1e-3

    def masked_compound():                               # one slab-masked compound sub-update, no accumulation (S8(d) cfg 5 (i))
        for kind, n in ((0, w["n_hb"]), (1, w["n_or"])):
            for _ in range(n):
                for parity in (0, 1):
                    for mu in range(4):
                        lat.substep(kind, parity, mu, w["slab_d"])

    t_hb, t_or = ev_time(lambda: lat.sweep(1, 0)), ev_time(lambda: lat.sweep(0, 1))
    t_masked = ev_time(masked_compound, 3)
    t_ml = ev_time(lambda: lat.multilevel(w["slab_d"], w["n_sub"], w["r_max"]), 2)      # (ii): sub-updates with accumulation
    lat.set_subupdate(0, 0, 1)
    t_meas = ev_time(lambda: lat.multilevel(w["slab_d"], w["n_sub"], w["r_max"]), 2)    # tables + accumulation + slab product only
    lat.set_subupdate(w["n_hb"], w["n_or"], 1)
    lat.set_update_algorithm(1, 1.2)
    t_met = ev_time(lambda: lat.sweep(1, 0))
    lat.set_update_algorithm(0)
    lat.close()
    l2 = [l2_resident(ul, torch, dev, *cfg) for cfg in ((24, 8, 1.00, 3, 1, 3), (32, 32, 1.00, 4, 1, 4))] if rank == 0 else []
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    peak, peak_src = measured_peak_hbm()
    n_or_launches = 8 * w["n_or"]
    or_launch_s = or_ms * 1e-3 / n_or_launches
    or_bytes = BYTES_PER_UPDATE_OR * (V / 2)
    achieved = or_bytes / or_launch_s / 1e9
    cpu = oracle_sample(w)
    d = w["slab_d"]
    n_slab = Nt // d
    E = 3 * w["r_max"] * n_slab * Ns ** 3                                                  # accumulator entries
    kb = 8                                                                                 # batch depth (DESIGN 4)
    n_pass = (w["n_sub"] + kb - 1) // kb
    # algorithmic bytes of the measurement part of one multilevel call (DESIGN 5): per configuration the temporal links read
    # (4 B x V) and the U table written and read once (2 x 16 B per slab and site); per pass the accumulators written, and
    # read except in the first pass (16 B each way per entry); the slab product reads them once
    meas_bytes = w["n_sub"] * (4 * V + 32 * n_slab * Ns ** 3) + (2 * n_pass - 1) * 16 * E + 16 * E
    masked_updates = (w["n_hb"] + w["n_or"]) * (V + 3 * V * (d - 1) // d)
    masked_bytes = (w["n_hb"] * 39.2 + w["n_or"] * 43.2) * (V + 3 * V * (d - 1) // d)    # S8(d): masked d=2 HB 39.2, OR 43.2 B per update
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": w["name"], "lattice": f"{Ns}^3x{Nt}", "beta": w["beta"], "seed": w["seed"],
                   "step": f"ul_sweep({w['n_hb']},{w['n_or']}) + ul_multilevel(d={w['slab_d']}, n_sub={w['n_sub']}, "
                           f"r_max={w['r_max']}) with sub-update ({w['n_hb']} HB + {w['n_or']} OR) + ul_plaquette",
                   "link_updates_per_step": n_upd, "slab_sweeps_per_step": w["n_sub"],
                   "l2": "inputs larger than L2 (links 268 MB + accumulators 6.4 GB vs 126 MB L2)",
                   "parallelism": f"replicas x{world}, independent seeds, no collective"},
        "slab_sweeps_per_s": world * w["n_sub"] / (ms_per_step * 1e-3),
        "plaquette": plaq,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 16 * V, "d2h_bytes_per_step": 16 * V + 8 * (2 * w["r_max"] + 12 + 3),
                "steps": e2e_steps},
        "gpu_launches": int(launches),
        "roofline": {"kernel": "k_update<OR> (overrelaxation sub-step, 32 launches per step)", "bound": "hbm",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": ncu_traffic(),
                     "algorithmic_bytes_per_launch": or_bytes, "avg_launch_us": or_launch_s * 1e6,
                     "link_updates_per_s": (V / 2) / or_launch_s, "peak_source": peak_src},
        "cpu_baseline": {"value": cpu["value"], "unit": UNIT, "cores": 1, "kind": "oracle", "sample": cpu["sample"],
                         "update_only_link_updates_per_s": cpu["update_only"]},
        # whole sweeps on the same lattice, CUDA events, against S8(d)'s algorithmic bytes (HB 32, OR 36 B per update; masked d=2:
        # HB 39.2, OR 43.2 B per update)
        "sweeps": {"hb_sweep_ms": t_hb * 1e3, "or_sweep_ms": t_or * 1e3, "metropolis_sweep_ms": t_met * 1e3,
                   "hb_sweep_frac_of_hbm_peak": 32 * 4 * V / t_hb / 1e9 / peak,
                   "or_sweep_frac_of_hbm_peak": 36 * 4 * V / t_or / 1e9 / peak,
                   "compound_1hb_4or_frac_of_hbm_peak": (32 + 4 * 36) * 4 * V / (t_hb + 4 * t_or) / 1e9 / peak,
                   "compound_1hb_4or_link_updates_per_s": 5 * 4 * V / (t_hb + 4 * t_or),
                   "paper_recipe_1metropolis_3or_frac_of_hbm_peak": 4 * 36 * 4 * V / (t_met + 3 * t_or) / 1e9 / peak,
                   "masked_compound_ms": t_masked * 1e3,
                   "masked_compound_frac_of_hbm_peak": masked_bytes / t_masked / 1e9 / peak,
                   "masked_compound_link_updates_per_s": masked_updates / t_masked,
                   "multilevel_ms_per_sub_update_with_accumulation": t_ml * 1e3 / w["n_sub"],
                   "measurement_only_ms_per_multilevel_call": t_meas * 1e3,
                   "measurement_only_ms_per_sub_update": t_meas * 1e3 / w["n_sub"],
                   "measurement_frac_of_hbm_peak": meas_bytes / t_meas / 1e9 / peak},
        "l2_resident": l2,
    }
    print(json.dumps(line), flush=True)


L2_BYTES_PER_CLK = 6300.0      # full-chip L2 (LTS) throughput cap measured in B300_MICROARCH.md "L2 cache"; x SM clock = peak


def l2_resident(ul, torch, dev, Ns, Nt, beta, seed, n_hb, n_or):
    """Compound sweep on a lattice that lives in L2 (BJ configs 3 and 4; quote the L2-bandwidth fraction there):
    microseconds per compound sweep, link updates/s, algorithmic bytes/s against the L2 peak (6300 B/clk x max SM clock)."""
    lat = ul.Lattice(Ns, Nt, beta, seed, device=dev)
    for _ in range(20):
        lat.sweep(n_hb, n_or)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n = 50
    a.record()
    for _ in range(n):
        lat.sweep(n_hb, n_or)
    b.record()
    torch.cuda.synchronize()
    lat.close()
    t = a.elapsed_time(b) / n * 1e-3
    V = Ns ** 3 * Nt
    try:
        sm_mhz = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["sm_max_mhz"])
    except Exception:
        sm_mhz = 1965.0
    l2_peak = L2_BYTES_PER_CLK * sm_mhz * 1e6 / 1e9
    gbs = (32 * n_hb + 36 * n_or) * 4 * V / t / 1e9
    return {"lattice": f"{Ns}^3x{Nt}", "recipe": f"{n_hb} HB + {n_or} OR", "compound_sweep_us": t * 1e6,
            "link_updates_per_s": (n_hb + n_or) * 4 * V / t, "algorithmic_GBps": gbs, "l2_peak_GBps": l2_peak,
            "frac_of_l2_peak": gbs / l2_peak, "link_bytes": 16 * V}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sample-ns", type=int, default=0, help="reference arm: spatial extent of the oracle sample (0 = the workload's; tests shrink it)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
