#!/usr/bin/env python
"""bench.py -- active-cell CTU updates/s of the GBEES prediction step on B200 (BASELINE.json metric).

A bench "step" = one complete propagation job of the workload (default: BASELINE config 2, the
6-D Lorenz '96 headline: init -> t = 0.5, CFL 0.9, prune every 5 steps), i.e. one pass of the whole
hot path (grow, dt, CTU flux, update, normalise, prune/compact/rehash) over one synthetic input.
`value` = sum over integration steps of the active-cell count / device time of the jobs
(init_gaussian and export outside the timed region); `e2e` = the same jobs timed through the C ABI
with HOST buffers: init_gaussian(host mean/cov) + run + export into pinned host arrays.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg3|cfg3s|cfg0|cfg1|cfg4] [--impl reference]
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "active-cell CTU updates/sec (grow+flux+update+prune) at 6-D"
UNIT = "cell-updates/s"


def workload(name):
    from paper_2508_13986_b200 import workloads as W
    if name == "cfg0":
        return W.config0()
    if name == "cfg1":
        return W.config1()
    if name == "cfg2":
        return W.config2()
    if name == "cfg3":
        return W.config3()
    if name == "cfg3s":  # 1/10-scale twin of config 3
        c = W.config3(dx=0.5)
        c.update(name="cfg3_linear_6d_tenth_scale", max_cells=1 << 25)
        return c
    raise SystemExit(f"unknown workload {name}")


def algo_bytes(stats, n, alpha):
    """Algorithmic bytes of a job, SURVEY.md 8(d) / DESIGN.md: N*(40+8n) + N_new*(28+8n) + N_prune*(45+8/alpha)."""
    return (stats["cell_updates"] * (40 + 8 * n) + stats["cells_inserted"] * (28 + 8 * n)
            + stats["cells_prune_scanned"] * (45 + 8 / alpha))


# per-phase share of the model above (bytes per cell handled by that phase)
def phase_bytes(stats, n, alpha):
    U, I, S = stats["cell_updates"], stats["cells_inserted"], stats["cells_prune_scanned"]
    return {"grow": 16 * U + (28 + 8 * n) * I, "link": 0, "passA": (16 + 8 * n) * U, "passB": 8 * U,
            "mark": 17 * S, "compact": 16 * S, "rebuild": (8 / alpha + 12) * S, "relink": 0, "sum": 0, "correct": 0}


class ClockSampler(threading.Thread):
    """Samples SM clock + throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz = index, False, [], set(), None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
                     0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown"}
            while not self.stop_flag:
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
                time.sleep(0.02)
        except Exception as e:  # noqa: BLE001
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def result(self):
        self.stop_flag = True
        self.join(timeout=2)
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.sm)}


def drive(g, cfg):
    """One propagation job on an initialised context (the timed call sequence)."""
    if cfg.get("t_meas"):
        for tm, z in zip(cfg["t_meas"], cfg["z"]):
            g.run(tm, prune_every=cfg["prune_every"])
            g.correct(z, cfg["R"])
            g.prune()
    elif cfg.get("t_end") is not None:
        g.run(cfg["t_end"], prune_every=cfg["prune_every"])
    else:
        g.run(1e300, max_steps=cfg["steps"], prune_every=cfg["prune_every"])


def drive_oracle(o, cfg, budget_s):
    """Same call sequence on the CPU oracle, stopped after budget_s seconds. Returns (updates, seconds)."""
    t0, upd, k = time.perf_counter(), 0, 0
    t_end = cfg.get("t_end") if cfg.get("t_end") is not None else (cfg["t_meas"][-1] if cfg.get("t_meas") else 1e300)
    max_steps = cfg.get("steps") or 1 << 62
    while o.time() < t_end and k < max_steps and time.perf_counter() - t0 < budget_s:
        o.step(t_end - o.time() if t_end < 1e299 else 0.0)
        upd += o.count()
        k += 1
        if cfg["prune_every"] and k % cfg["prune_every"] == 0:
            o.prune()
    return upd, time.perf_counter() - t0, k


def aggregate(ms, upd, device="cpu"):
    """Replicas-only multi-GPU: time = max over ranks, work = sum over ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return ms, upd
    dist.barrier()
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([upd], dtype=torch.float64, device=device)
    dist.all_reduce(u)
    return t.item(), u.item()


def make_oracle(cfg):
    from oracle.binding import Oracle
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    o.init_gaussian(cfg["mean"], cfg["cov"])
    return o


def run_reference(args, cfg):
    """--impl reference: the CPU oracle as it stands, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    budget = 6.0
    upd_tot, sec_tot, ksteps = 0, 0.0, 0
    for it in range(args.warmup + args.steps):
        o = make_oracle(cfg)
        upd, sec, k = drive_oracle(o, cfg, budget)
        if it >= args.warmup:
            upd_tot, sec_tot, ksteps = upd_tot + upd, sec_tot + sec, k
    val = upd_tot / sec_tot
    sample = f"first {ksteps} integration steps of {cfg['name']} from its initial state (<= {budget:.0f} s of CPU per bench step)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sec_tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": {"workload": cfg["name"], "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


def cfg4_rows(key_counts, alphas):
    """BASELINE config 4: hashtable / compaction microbench (probes/op against PAPER.md:192, M ops/s,
    modelled GB/s: 16 B slot + 8 B key per insert / successful probe chain, 8 + 1 + 8 B per compacted key)."""
    import torch
    from paper_2508_13986_b200 import HashTable, workloads as W
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback"
    rows = []

    def timed(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); e0.record(); r = fn(); e1.record(); e1.synchronize()
        return r, e0.elapsed_time(e1) * 1e-3

    for K in key_counts:
        keys = W.config4_keys(K)
        rng = np.random.default_rng(W.S0 + 42)
        dele = torch.from_numpy((rng.random(K) < 0.3).astype(np.uint8)).cuda()
        unit = np.uint64(1) << (np.uint64(10) * np.arange(6, dtype=np.uint64))
        sub = keys[:max(K // 12, 1)]
        q = torch.from_numpy(np.concatenate([sub + u for u in unit] + [sub - u for u in unit]).view(np.int64)).cuda()
        for alpha in alphas:
            kt = torch.from_numpy(keys.view(np.int64)).cuda()
            ht = HashTable(int(np.ceil(K / alpha)))
            idx = torch.empty(K, dtype=torch.int32, device="cuda")
            qo = torch.empty(q.numel(), dtype=torch.int32, device="cuda")
            p_ins, t_ins = timed(lambda: ht.insert(kt, idx))
            p_hit, t_hit = timed(lambda: ht.lookup(kt, idx))
            p_nb, t_nb = timed(lambda: ht.lookup(q, qo))
            coop = {}
            for wdt in (4, 32):
                pc, tc = timed(lambda: ht.lookup_coop(q, qo, wdt))
                ph, th = timed(lambda: ht.lookup_coop(kt, idx, wdt))
                coop[f"w{wdt}"] = {"neighbours_Mops": q.numel() / tc / 1e6, "hit_Mops": K / th / 1e6,
                                   "probes_equal_scalar": bool(pc == p_nb and ph == p_hit)}
            kept, t_cmp = timed(lambda: ht.compact(kt, dele))
            ht.close()
            rows.append({"keys": K, "alpha": alpha,
                         "insert": {"probes_per_op": p_ins / K, "Mops": K / t_ins / 1e6, "GBps": K * (8 + 16 * p_ins / K + 16) / t_ins / 1e9},
                         "lookup_hit": {"probes_per_op": p_hit / K, "Mops": K / t_hit / 1e6, "GBps": K * (8 + 16 * p_hit / K + 4) / t_hit / 1e9},
                         "lookup_neighbours": {"probes_per_op": p_nb / q.numel(), "Mops": q.numel() / t_nb / 1e6,
                                               "GBps": q.numel() * (8 + 16 * p_nb / q.numel() + 4) / t_nb / 1e9},
                         "cooperative_probing": coop,
                         "delete30_compact_rebuild": {"survivors": kept, "Mkeys_per_s": K / t_cmp / 1e6}})
    return rows


def run_cfg4(args):
    rows = cfg4_rows([int(k) for k in args.cfg4_keys.split(",")], (0.3, 0.4, 0.5, 0.6, 0.7, 0.8))
    print(json.dumps({"metric": "hashtable / compaction microbench (BASELINE config 4)", "unit": "probes/op, M ops/s, GB/s",
                      "n_gpus": 1, "data": "synthetic", "config": {"workload": "cfg4_hashtable", "keys": args.cfg4_keys},
                      "expected_probes": "PAPER.md:192: hit (1+1/(1-a))/2, miss (1+1/(1-a)^2)/2", "rows": rows}))


KERNEL_OF_PHASE = {"grow": "k_detect + k_grow<{n},{d},skip>", "link": "k_link<{n},false>", "passA": "k_flux1<{n},{d},true>",
                   "passB": "k_flux2<{n}>", "mark": "k_mark<{n},{d}>", "compact": "k_prune_scan + k_prune_move + k_zero_tail",
                   "rebuild": "k_clear_table + k_prune_tail<{n},{d}>", "relink": "k_link_finish<{n}>", "correct": "k_correct<{n}>",
                   "run": "k_run_small<{n},{d},true>"}


def load_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return json.load(open(path))["hbm_gbs"], "measured"
    return 6650.0, "fallback"


def measure(cfg, steps, warmup, local, stream, run_mode, flush, alpha=0.5, with_phases=True):
    """Time `steps` jobs of one workload on the device (CUDA events on the launching stream, L2 flushed
    between jobs); optionally one more job with per-phase event timing. Returns the context too."""
    import torch
    from paper_2508_13986_b200 import Gbees
    n = cfg["n"]
    g = Gbees(n, cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"],
              load_factor=alpha, device=local, stream=stream.cuda_stream, run_mode=run_mode)

    def job(profile=False):
        g.init_gaussian(cfg["mean"], cfg["cov"])
        flush.zero_()
        g.profile(profile)
        l0 = g.stats()["launches"]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        drive(g, cfg)
        e1.record(stream)
        e1.synchronize()
        st = g.stats()
        st["launches"] -= l0
        return e0.elapsed_time(e1), st

    for _ in range(warmup):
        job()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    ms_tot, upd_tot, launches, st = 0.0, 0, 0, None
    for _ in range(steps):
        ms, st = job()
        ms_tot, upd_tot, launches = ms_tot + ms, upd_tot + st["cell_updates"], launches + st["launches"]
    torch.cuda.synchronize()
    clocks = sampler.result()
    out = {"g": g, "job": job, "ms_tot": ms_tot, "upd_tot": upd_tot, "launches": launches, "stats": st, "clocks": clocks}
    if with_phases:
        _, st_prof = job(profile=True)
        prof = g.profile(False)
        pb = phase_bytes(st_prof, n, alpha)
        out["phases"] = {k: {"ms": round(v[0], 4), "launches": v[1],
                             "algo_GBps": (pb.get(k, 0) / (v[0] * 1e-3) / 1e9 if v[0] > 0 else None)}
                         for k, v in prof.items() if v[1]}
        out["phase_bytes"], out["st_prof"] = pb, st_prof
    return out


def extra_workloads(local, stream, run_mode, flush, peak, skip):
    """The other BASELINE configs, 3 timed jobs each after 1 warm-up (north_star: throughput on the five
    synthetic workloads). Short records: value, ms per job, whole-job roofline fraction, clocks."""
    import torch
    out = {}
    for name in ("cfg0", "cfg1", "cfg3s", "cfg3"):
        if name in skip:
            continue
        cfg = workload(name)
        r = measure(cfg, 3, 1, local, stream, run_mode, flush, with_phases=False)
        st, ms = r["stats"], r["ms_tot"] / 3
        gbps = algo_bytes(st, cfg["n"], 0.5) / (ms * 1e-3) / 1e9
        out[name] = {"workload": cfg["name"], "value": r["upd_tot"] / (r["ms_tot"] * 1e-3), "unit": UNIT, "ms_per_job": ms,
                     "jobs": 3, "integration_steps_per_job": st["steps"], "prunes_per_job": st["prunes"],
                     "cell_updates_per_job": st["cell_updates"], "final_cells": st["n_cells"],
                     "whole_job_algo_GBps": gbps, "whole_job_frac": gbps / peak, "gpu_launches": r["launches"],
                     "clocks": r["clocks"]}
        r["g"].close()
        del r
        torch.cuda.empty_cache()
    if "cfg4" not in skip:
        out["cfg4"] = cfg4_rows([1000000, 10000000], (0.5,))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the short records of the other workloads (\"workloads\" in the JSON line)")
    ap.add_argument("--cfg4-keys", default="1000000,10000000", help="key counts of the cfg4 microbench (1e8 needs ~25 GB)")
    ap.add_argument("--run-mode", type=int, default=0, help="gbees_run: 0 = device-side step control (no host round trip per step), 1 = host loop of gbees_step/gbees_prune")
    args = ap.parse_args()
    if args.workload == "cfg4":
        return run_cfg4(args)
    cfg = workload(args.workload)
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import torch.distributed as dist
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    n, alpha = cfg["n"], 0.5
    stream = torch.cuda.Stream()
    peak, peak_src = load_peak()
    with torch.cuda.stream(stream):
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
        if world > 1:
            dist.barrier()
        r = measure(cfg, args.steps, max(args.warmup, 3), local, stream, args.run_mode, flush, alpha)
        g, st, ms_tot, clocks, launches = r["g"], r["stats"], r["ms_tot"], r["clocks"], r["launches"]
        ms_max, upd_all = aggregate(ms_tot, r["upd_tot"], "cuda")
        phases, pb, st_prof = r["phases"], r["phase_bytes"], r["st_prof"]
        dom = max(phases, key=lambda k: phases[k]["ms"])
        job_GBps = algo_bytes(st, n, alpha) / (ms_tot / args.steps * 1e-3) / 1e9
        dom_GBps = phases[dom]["algo_GBps"] or 0.0
        # DRAM traffic of the dominant kernel: bytes per cell-update from the committed ncu --set full capture
        # (profiles/traffic.json, a static figure) times the live cell count
        traffic, traffic_src = None, None
        tpath = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tpath):
            tj = json.load(open(tpath))
            if tj.get("phase") == dom and tj.get("workload") == cfg["name"]:
                traffic = tj["dram_bytes_per_cell_update"] * st_prof["cell_updates"] / max(phases[dom]["launches"], 1)
                traffic_src = "profiles/traffic.json (static: ncu capture of an earlier run x live cell count)"
        kname = KERNEL_OF_PHASE.get(dom, dom).format(n=n, d=cfg["dyn"])
        roofline = {"bound": "hbm", "kernel": kname, "phase": dom, "achieved": dom_GBps, "peak": peak, "unit": "GB/s",
                    "frac": dom_GBps / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                    "algo_bytes_per_launch": pb.get(dom, 0) / max(phases[dom]["launches"], 1),
                    "timing": "CUDA events around every launch of the phase in one extra job (event timing switches the programmatic dependent launch overlap off, so the phases add up to more than ms_per_step)",
                    "whole_job": {"achieved": job_GBps, "frac": job_GBps / peak,
                                  "frac_of_8TBps": job_GBps / 8000.0, "algo_bytes_per_job": algo_bytes(st, n, alpha)},
                    "phases": phases}

        # e2e: host buffers in, host buffers out, every job
        nmax = cfg["max_cells"]
        hk = torch.empty((nmax, n), dtype=torch.int32).pin_memory() if nmax * n * 4 < (4 << 30) else None
        import ctypes as C
        from paper_2508_13986_b200.binding import lib
        e2e_ms, e2e_upd, d2h = 0.0, 0, 0
        if hk is not None:
            hp = torch.empty(nmax, dtype=torch.float64).pin_memory()
            for it in range(2 + args.steps):
                flush.zero_(); torch.cuda.synchronize()
                t0 = time.perf_counter()
                g.init_gaussian(np.asarray(cfg["mean"], dtype=np.float64), np.asarray(cfg["cov"], dtype=np.float64))
                drive(g, cfg)
                cnt = C.c_int64()
                rc = lib().gbees_export(g._h, hk.data_ptr(), hp.data_ptr(), nmax, C.byref(cnt))
                assert rc == 0
                dt_ = time.perf_counter() - t0
                if it >= 2:
                    e2e_ms += 1e3 * dt_; e2e_upd += g.stats()["cell_updates"]; d2h = cnt.value * (4 * n + 8)
            del hk, hp
        e2e = {"value": (e2e_upd / (e2e_ms * 1e-3) * world) if e2e_ms else None, "unit": UNIT,
               "h2d_bytes_per_step": 8 * (n + n * n), "d2h_bytes_per_step": d2h,
               "ms_per_step": e2e_ms / args.steps if e2e_ms else None}
        g.close()
        workloads = None
        if rank == 0 and world == 1 and not args.no_extra:
            workloads = extra_workloads(local, stream, args.run_mode, flush, peak, skip={args.workload})

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        o = make_oracle(cfg)
        upd, sec, k = drive_oracle(o, cfg, 15.0)
        cpu = {"value": upd / sec, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"first {k} integration steps of {cfg['name']} ({upd} cell-updates, {sec:.1f} s, 1 thread of {os.cpu_count()} host cores)"}
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": upd_all / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "n": n, "dx": cfg["dx"][0], "threshold": cfg["thresh"],
                       "integration_steps_per_job": st["steps"], "prunes_per_job": st["prunes"],
                       "cell_updates_per_job": st["cell_updates"], "final_cells": st["n_cells"],
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "run_mode": args.run_mode,
                       "l2": "256 MiB memset between jobs (flush)"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
            "workloads": workloads}))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
