#!/usr/bin/env python
"""bench.py -- one JSON line for the OTOO force path on B200.

A step = one pass of the whole hot path (tree build + fused walk/gravity) over one batch of
synthetic particles already resident in HBM.  metric = gravity interactions/s (R11 count / device time of the
whole step).  BASELINE.json's metric names no config, so the headline workload is the largest single-GPU one,
C5 (uniform cube, N = 33 554 432, theta = 0.5, G = 256); C2, C3 and C4 (with its SPH rows) ride in `per_config`
of the same line.  `roofline` is for the dominant kernel (walk_gravity_ws_kernel) against the non-tensor FP32
peak; `e2e` goes through the host-buffer C-ABI call; `cpu_baseline` is the fp64 oracle timed on this box's host
cores on a bounded sample.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--theta 0.5] [--no-per-config]
    python bench.py --impl reference ...      # times the oracle (CPU) on the same workload
    python bench.py --probe ffma2|sumloop|rank|sort   # the microbenchmarks behind DESIGN.md's ceilings
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from workloads import generators as gen  # noqa: E402

METRIC = "gravity_interactions_per_s"
UNIT = "interactions/s"
FLOPS_PER_INTERACTION = 20
BUILD_BYTES_PER_PARTICLE = 370      # algorithmic HBM bytes of the tree build per particle
SM_LANES = 128                      # FP32 lanes per SM
NOMINAL_SM_MHZ = 1965.0
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")
ORACLE_SAMPLE_S = 15.0              # target CPU seconds of the oracle's sampled walk + sums
# instruction-counted flops of the SPH kernels (DESIGN.md section 6 "SPH"; fma = 2): per candidate pair test of pass 1
# (3 sub, 1 mul, 2 fma, 1 sub; the force adds a max), per true neighbour pair of pass 2 (spline + sums)
SPH_FLOP_TEST = {"density": 9, "force": 10}
SPH_FLOP_HIT = {"density": 21, "force": 56}


def hbm_peak_gbs():
    """measured HBM copy bandwidth of this pool (driver-written MEASURED_PEAKS.json), else the guide's fallback"""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json (measured copy bandwidth)"
    except Exception:
        return 6650.0, "fallback of B200_PROFILING.md"


def committed_traffic(key: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on workload `key`, from the committed
    `ncu --set full` summary profiles/r2_dram_traffic.csv (a number from a profiler run, never typed in here);
    (None, why) if that file has no row for this workload."""
    try:
        with open(TRAFFIC_CSV) as f:
            for row in csv.DictReader(f):
                if row["workload"] == key and row["kernel"] == kernel:
                    return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]), row.get("report", "")
    except Exception as e:  # noqa: BLE001
        return None, f"{os.path.relpath(TRAFFIC_CSV, ROOT)} unreadable: {e}"
    return None, f"no row for ({key}, {kernel}) in {os.path.relpath(TRAFFIC_CSV, ROOT)}"


def workload(name: str, theta, seed: int, n=None):
    cfg = dict(gen.CONFIGS[name])
    if theta is not None:
        cfg["theta"] = theta
    if n is not None:
        cfg["n"] = int(n)
    pm = gen.make(cfg["kind"], cfg["n"], seed)
    return cfg, pm


def workload_text(name, cfg, mac_txt, key_order, group_distance):
    return (f"{name}: {cfg['kind']} N={cfg['n']} eps={cfg['eps']} {mac_txt} n_crit={cfg['n_crit']} group={cfg['group']} "
            f"order={key_order} distance={group_distance}")


class ClockSampler(threading.Thread):
    """nvidia-smi style clock/throttle sampling during the timed region (via NVML)."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.samples, self.reasons, self.stop_flag = [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        while not self.stop_flag:
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.02)

    def result(self):
        self.stop_flag = True
        if self.nv is None or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": []}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


# ------------------------------------------------------------------ the oracle on the host cores (bounded sample)
def oracle_sample(args, name, cfg, pm, delta, m_limit, repeats=1, budget_s=ORACLE_SAMPLE_S):
    """The oracle as it stands: full tree build (timed once), then walk + fp64 sums on a seeded sample of groups sized
    for about `budget_s` seconds, scaled to all groups (SURVEY 8(d) allows exactly this for the large configs).
    Returns a list of per-repeat dicts (ms_per_step estimate, interactions/s) and a description of the sample."""
    from oracle import oracle
    n, G, n_crit = cfg["n"], cfg["group"], cfg["n_crit"]
    eps, theta = float(np.float32(cfg["eps"])), float(np.float32(cfg["theta"]))
    t0 = time.perf_counter()
    t = oracle.Tree(pm, n_crit, key_order=1 if args.key_order == "hilbert" else 0)
    t.set_dist_kind({"box": 0, "exact": 1, "split": 2}[args.group_distance])
    rb2 = t.rb2_delta(delta, m_limit) if args.mac == "delta" else None
    t_build = time.perf_counter() - t0
    ng = t.n_groups(G)
    rng = np.random.default_rng(args.seed)
    # pilot: 16 groups tell the cost per group; then the sample that fits the budget (at most all groups)
    pilot = np.sort(rng.choice(ng, size=min(16, ng), replace=False)).astype(np.int64)
    t0 = time.perf_counter()
    t.gravity(eps, theta, G, groups=pilot, rb2=rb2)
    per_group = (time.perf_counter() - t0) / len(pilot)
    n_s = int(min(ng, max(16, budget_s / max(per_group, 1e-6))))
    whole = n_s >= ng
    res = []
    for r in range(repeats):
        sel = None if whole else np.sort(rng.choice(ng, size=n_s, replace=False)).astype(np.int64)
        t0 = time.perf_counter()
        out = t.gravity(eps, theta, G, groups=sel, rb2=rb2)
        dt = time.perf_counter() - t0
        scale = 1.0 if whole else ng / n_s
        inter_total = out["interactions"] * scale          # estimate of the whole workload's R11 count
        step_s = t_build + dt * scale
        res.append(dict(ms_per_step=1e3 * step_s, value=inter_total / step_s, sample_s=dt, interactions_est=inter_total))
    what = (f"tree build on all N = {n} particles ({t_build:.1f} s, once) + walk and fp64 sums on "
            + ("ALL" if whole else f"a seeded {n_s} of") + f" {ng} groups ({np.mean([x['sample_s'] for x in res]):.1f} s per step"
            + ("" if whole else f", scaled by {ng / n_s:.1f}") + "); value = estimated interactions / (build + scaled walk and sums)")
    return res, what, oracle.max_threads()


def run_reference(args, rank):
    """The reference arm of this tier: the oracle as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    cfg, pm = workload(args.workload, args.theta, args.seed, args.n)
    delta = float(np.float32(args.delta if args.delta is not None else cfg.get("delta", 0.01)))
    m_limit = float(np.float32(args.m_limit if args.m_limit is not None else cfg.get("m_limit", 0.05)))
    steps = args.warmup + args.steps
    res, what, cores = oracle_sample(args, args.workload, cfg, pm, delta, m_limit, repeats=steps,
                                     budget_s=max(2.0, 120.0 / steps))
    res = res[args.warmup:]
    ms = float(np.mean([r["ms_per_step"] for r in res]))
    val = float(np.mean([r["interactions_est"] for r in res])) / (ms * 1e-3)
    mac_txt = f"theta={cfg['theta']}" if args.mac == "theta" else f"Delta-MAC delta={delta:g} m_limit={m_limit:g}"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_text(args.workload, cfg, mac_txt, args.key_order, args.group_distance)},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ one workload on the GPU
def measure(args, name, theta, seed, steps, warmup, local, world, n=None, e2e=True, sampler=None, accuracy=False):
    import torch
    import torch.distributed as dist
    from paper_1206_1199_b200 import binding, replicas

    cfg, pm = workload(name, theta, seed, n)
    n, G, n_crit = cfg["n"], cfg["group"], cfg["n_crit"]
    eps, theta = float(np.float32(cfg["eps"])), float(np.float32(cfg["theta"]))
    delta = float(np.float32(args.delta if args.delta is not None else cfg.get("delta", 0.01)))
    m_limit = float(np.float32(args.m_limit if args.m_limit is not None else cfg.get("m_limit", 0.05)))
    o = binding.Otoo(max_particles=n, device=local)
    o.otoo_set_option("key_order", 1 if args.key_order == "hilbert" else 0)
    o.otoo_set_option("group_distance", {"box": 0, "exact": 1, "split": 2}[args.group_distance])
    d_pm = torch.from_numpy(pm).cuda()
    out = torch.empty((n, 4), dtype=torch.float32, device="cuda")
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step():
        flush_buf.fill_(1)                      # L2 flush between steps, outside the timed events
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        e[0].record()
        o.otoo_build_tree(d_pm, n_crit)
        e[1].record()
        if args.mac == "delta":
            o.otoo_gravity_delta(eps, delta, m_limit, G, out=out)
        else:
            o.otoo_gravity(eps, theta, G, out=out)
        e[2].record()
        return e

    # at least max(W, 3) warm-up steps, and at least a second of them: the first runs on a fresh box are 0.2-0.3 % slower
    # (81.35 against 81.15 ms per walk kernel at C5) until the GPU has been busy for about a second
    n_warm, t_warm = 0, time.perf_counter()
    while n_warm < max(warmup, 3) or (time.perf_counter() - t_warm < 1.0 and n_warm < 64):
        step()
        torch.cuda.synchronize()
        n_warm += 1
    o.otoo_build_tree(d_pm, n_crit)
    launches_build = o.otoo_last_stats()["launches"]
    step()
    st = o.otoo_last_stats()
    launches_step = launches_build + st["launches"]          # kernels of libotoo.so per step (counted inside the library)
    inter = st["sum_interactions"]
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler is not None:
        sampler.start()
    evs, kern_ms, prep_ms, phases, sm_mhz = [], [], [], [], []
    for _ in range(steps):
        evs.append(step())
        s = o.otoo_last_stats()      # synchronises: the kernel's own event pair and the build's phase events of THIS step
        kern_ms.append(s["ms_walk_force"]); prep_ms.append(s["ms_walk_prep"]); phases.append(s["ms_build"]); sm_mhz.append(s["walk_sm_mhz"])
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.result() if sampler is not None else None
    o.otoo_set_option("walk_profile", 1)          # one more step, outside the timed region, with the instrumented kernel
    step()
    s = o.otoo_last_stats()
    o.otoo_set_option("walk_profile", 0)
    t_build = np.array([e[0].elapsed_time(e[1]) for e in evs])
    t_grav = np.array([e[1].elapsed_time(e[2]) for e in evs])
    ms_step = float((t_build + t_grav).mean())
    ms_max, inter_all = replicas.aggregate(ms_step, float(inter), device="cuda")   # max over ranks, sum over ranks
    res = dict(cfg=cfg, n=n, G=G, inter=inter, inter_all=inter_all, ms_step=ms_max, value=inter_all / (ms_max * 1e-3),
               build_ms=float(t_build.mean()), call_ms=float(t_grav.mean()), kernel_ms=float(np.mean(kern_ms)),
               prep_ms=float(np.mean(prep_ms)), kernel_sm_mhz=float(np.mean(sm_mhz)), launches_step=launches_step, clocks=clocks, delta=delta, m_limit=m_limit,
               phases={k: float(np.mean([p[k] for p in phases])) for k in phases[0]}, pm=pm, o=o, stats=st, n_warm=n_warm,
               warp_time={k: float(s[k]) for k in ("eval_wait_frac", "walker_wait_frac", "walker_idle_frac")},
               walk={k: int(st[k]) for k in ("sum_tests", "sum_steps", "sum_tasks", "sum_flushes", "n_groups")})

    if e2e:   # ---- end to end through the host-buffer C-ABI call (pinned host memory)
        h_in = torch.from_numpy(pm).pin_memory()
        h_out = torch.empty((n, 4), dtype=torch.float32).pin_memory()
        e2e_t = []
        for it in range(2 + min(steps, 5)):
            flush_buf.fill_(1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            if args.mac == "delta":
                o.otoo_gravity_delta_host(h_in.numpy(), n_crit, eps, delta, m_limit, G, out=h_out.numpy())
            else:
                o.otoo_gravity_host(h_in.numpy(), n_crit, eps, theta, G, out=h_out.numpy())
            dt = time.perf_counter() - t0
            if it >= 2:
                e2e_t.append(dt)
        e2e_ms, _ = replicas.aggregate(1e3 * float(np.mean(e2e_t)), float(inter), device="cuda")
        res["e2e_ms"] = e2e_ms
        del h_in, h_out

    if accuracy:   # the method's error against the O(N^2) definition on a seeded subsample (oracle, fp64)
        from oracle import oracle
        tg = np.sort(np.random.default_rng(4096).choice(n, size=min(1024, n), replace=False)).astype(np.int64)
        ref = oracle.direct_sum(pm, eps, tg)
        got = out.cpu().numpy().astype(np.float64)[tg]
        e = np.linalg.norm(got[:, :3] - ref[:, :3], axis=1) / np.linalg.norm(ref[:, :3], axis=1)
        res["accuracy"] = {"targets": int(len(tg)), "median_rel_err": float(np.median(e)), "p99_rel_err": float(np.percentile(e, 99)),
                           "against": "oracle fp64 direct sum over all N sources"}

    if cfg["kind"] in ("wd_pair", "cold_sphere") and world == 1:
        # BASELINE config 4 / the paper's cold collapse: the SPH rows (H11-H13) on the same tree, timed like the gravity step
        w = (gen.wd_pair if cfg["kind"] == "wd_pair" else gen.cold_sphere)(n, seed)
        d_h, d_u, d_v = (torch.from_numpy(w[k]).cuda() for k in ("h", "u", "vel"))
        Gs = args.group_sph if args.group_sph else cfg.get("group_sph", 64)
        ts, ks = [], []
        for it in range(3 + steps):
            flush_buf.fill_(1)
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            ev[0].record()
            o.otoo_set_option("sph_reuse_walk", 0 if args.no_sph_reuse_walk else 1)   # stage 1 records the leaves each group opens ...
            rho, nn = o.otoo_sph_density(d_h, Gs)
            P = o.otoo_eos_ideal(rho, d_u, 5.0 / 3.0)
            ev[1].record()
            s1 = o.otoo_last_stats()
            k1 = s1["ms_walk_force"]
            o.otoo_set_option("sph_reuse_radii", 1)     # h is fixed within a step: stage 2 keeps stage 1's Eq. 5 radii
            o.otoo_sph_force(d_h, rho, P, Gs, vel=d_v)  # ... and stage 2 starts from them (same MAC, same radii: the same leaves)
            o.otoo_set_option("sph_reuse_radii", 0)
            o.otoo_set_option("sph_reuse_walk", 0)
            ev[2].record()
            s2 = o.otoo_last_stats()
            k2 = s2["ms_walk_force"]
            torch.cuda.synchronize()
            if it >= 3:
                ts.append((ev[0].elapsed_time(ev[1]), ev[1].elapsed_time(ev[2])))
                ks.append((k1, k2))
        cand = o.otoo_last_stats()["sum_interactions"]
        td, tf = float(np.mean([x[0] for x in ts])), float(np.mean([x[1] for x in ts]))
        kd, kf = float(np.mean([x[0] for x in ks])), float(np.mean([x[1] for x in ks]))
        pairs = int(nn.sum().item())
        sm_count = torch.cuda.get_device_properties(local).multi_processor_count
        peak = sm_count * SM_LANES * 2 * NOMINAL_SM_MHZ * 1e6 / 1e12
        # pair tests actually made: the candidates left after the walk-time cull (otoo_stats_t.sum_evaluated), not the
        # paper's whole list -- the flops of skipped tests are not counted as achieved
        ev_d, ev_f = s1["sum_evaluated"], s2["sum_evaluated"]
        ops_d = SPH_FLOP_TEST["density"] * ev_d + SPH_FLOP_HIT["density"] * pairs
        ops_f = SPH_FLOP_TEST["force"] * ev_f + SPH_FLOP_HIT["force"] * pairs
        res["sph"] = {"group": Gs, "stage2_walk": "full walk" if args.no_sph_reuse_walk else "replays the leaves stage 1 opened (option sph_reuse_walk)",
                      "density_eos_ms": td, "force_dudt_ms": tf, "density_kernel_ms": kd, "force_kernel_ms": kf,
                      "candidate_pairs_per_pass": cand, "evaluated_pair_tests": {"density": ev_d, "force_dudt": ev_f}, "neighbour_pairs": pairs, "candidate_pairs_per_s": 2 * cand / ((td + tf) * 1e-3),
                      "roofline": {"bound": "alu", "peak": peak, "unit": "TFLOP/s",
                                   "density": {"achieved": ops_d / (kd * 1e-3) / 1e12, "frac": ops_d / (kd * 1e-3) / 1e12 / peak},
                                   "force_dudt": {"achieved": ops_f / (kf * 1e-3) / 1e12, "frac": ops_f / (kf * 1e-3) / 1e12 / peak},
                                   "flops": f"instruction-counted: {SPH_FLOP_TEST['density']} / {SPH_FLOP_TEST['force']} flop per pair test made "
                                            f"(candidates left after the walk-time cull) + {SPH_FLOP_HIT['density']} / "
                                            f"{SPH_FLOP_HIT['force']} per neighbour pair (density / force + du/dt)",
                                   "paper_convention_200flop_tflops": 200.0 * 2 * pairs / ((kd + kf) * 1e-3) / 1e12,
                                   "note": "the paper's 200 flop per SPH interaction (L254) counts its viscosity and overstates these kernels"}}
    del d_pm, out, flush_buf
    return res


def roofline_block(res, key, peak_tflops, peak_measured, sm_count):
    achieved = FLOPS_PER_INTERACTION * res["inter"] / (res["kernel_ms"] * 1e-3) / 1e12
    traffic, src = committed_traffic(key, "walk_gravity_ws_kernel")
    return {"bound": "alu", "kernel": "walk_gravity_ws_kernel", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
            "frac": achieved / peak_tflops, "traffic": traffic, "traffic_source": src,
            "peak_source": f"derived: {sm_count} SMs x 128 FP32 lanes x 2 flop x {NOMINAL_SM_MHZ:.0f} MHz (DESIGN.md section 6); "
                           "MEASURED_PEAKS.json holds no FP32 figure",
            "peak_measured_ffma": peak_measured, "frac_of_measured": achieved / peak_measured if peak_measured else None,
            "flops_per_interaction": FLOPS_PER_INTERACTION, "interactions_per_launch": res["inter"],
            "kernel_ms": res["kernel_ms"], "kernel_ms_source": "CUDA events around the kernel launch alone, on its stream (otoo_last_stats.ms_walk_force), mean over the timed steps",
            "otoo_gravity_call_ms": res["call_ms"], "prep_ms": res["prep_ms"],
            "kernel_sm_mhz": res["kernel_sm_mhz"], "kernel_sm_mhz_source": "clock64 ticks per globaltimer ns inside the kernel (otoo_last_stats.walk_sm_mhz)",
            "interactions_per_s_kernel": res["inter"] / (res["kernel_ms"] * 1e-3),
            "warp_time": res["warp_time"], "walk": res["walk"]}


def build_block(res):
    hbm, hbm_src = hbm_peak_gbs()
    gbs = BUILD_BYTES_PER_PARTICLE * res["n"] / (res["build_ms"] * 1e-3) / 1e9
    return {"ms": res["build_ms"], "bound": "hbm", "algorithmic_bytes": BUILD_BYTES_PER_PARTICLE * res["n"],
            "bytes_per_particle": BUILD_BYTES_PER_PARTICLE, "achieved_gbs": gbs, "peak_gbs": hbm, "frac": gbs / hbm,
            "peak_source": hbm_src, "phases_ms": res["phases"]}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="otoo", choices=["otoo", "reference"])
    ap.add_argument("--workload", default="C5", choices=sorted(gen.CONFIGS))
    ap.add_argument("--theta", type=float, default=None)
    ap.add_argument("--mac", default="theta", choices=["theta", "delta"],
                    help="delta: the paper's absolute-error MAC (otoo_gravity_delta) instead of BASELINE's theta criterion")
    ap.add_argument("--key-order", default="morton", choices=["morton", "hilbert"],
                    help="hilbert: the paper's ordering (L131) instead of BASELINE's Morton-contiguous groups")
    ap.add_argument("--group-distance", default="split", choices=["box", "exact", "split"],
                    help="split (default, R25): minimum over the boxes of the group's pieces between its coarsest key boundaries; "
                         "box: one bounding box per group (R8); exact: the paper's minimum over the members' distances (L163)")
    ap.add_argument("--delta", type=float, default=None)
    ap.add_argument("--m-limit", type=float, default=None)
    ap.add_argument("--seed", type=int, default=1206)
    ap.add_argument("--n", type=int, default=None, help="override the workload's particle count (scaling runs, e.g. Fig. 9)")
    ap.add_argument("--group-sph", type=int, default=None, help="group size of the SPH rows (C4 / COLD; default: the workload's, 64)")
    ap.add_argument("--no-sph-reuse-walk", action="store_true", help="SPH rows: stage 2 walks the tree again instead of starting from the leaves stage 1 opened")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the C2 / C3 / C4 blocks of the default line")
    ap.add_argument("--probe", default=None, choices=["ffma2", "sumloop", "rank", "sort"],
                    help="run a microbenchmark of the library (otoo_probe) instead of the bench and print its table as JSON")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_1206_1199_b200 import binding, replicas   # fails loudly if libotoo.so is missing

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if args.probe:
        o = binding.Otoo(max_particles=1 << (25 if args.probe == "sort" else 20), device=local)
        print(json.dumps({"probe": args.probe, "rows": o.otoo_probe(args.probe)}), flush=True)
        return
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    # replicas only: every rank runs the same workload with its own seed
    seed = replicas.replica_seed(args.seed, rank)
    sampler = ClockSampler(local)
    res = measure(args, args.workload, args.theta, seed, args.steps, args.warmup, local, world, n=args.n, sampler=sampler)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    o = res["o"]
    peak_measured = o.otoo_measure_fp32_peak()      # FFMA2-only kernel on this GPU, at the clock it holds
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    peak_tflops = sm_count * SM_LANES * 2 * NOMINAL_SM_MHZ * 1e6 / 1e12
    cfg, n = res["cfg"], res["n"]
    custom = args.theta is not None or args.n is not None or args.mac != "theta" or args.key_order != "morton" or args.group_distance != "split"
    key = args.workload if not custom else f"{args.workload}:custom"
    mac_txt = f"theta={cfg['theta']}" if args.mac == "theta" else f"Delta-MAC delta={res['delta']:g} m_limit={res['m_limit']:g}"
    line = {"metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "warmup_steps_run": res["n_warm"], "ms_per_step": res["ms_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_text(args.workload, cfg, mac_txt, args.key_order, args.group_distance),
                       "l2": "flushed between steps (256 MiB write, outside the timed events)",
                       "parallelism": "replicas" if world > 1 else "single"},
            "gflops": FLOPS_PER_INTERACTION * res["value"] / 1e9,
            "interactions_per_step": res["inter_all"], "clocks": res["clocks"],
            "e2e": {"value": res["inter_all"] / (res["e2e_ms"] * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 16 * n,
                    "d2h_bytes_per_step": 16 * n, "ms_per_step": res["e2e_ms"]},
            "gpu_launches": int(res["launches_step"] * args.steps),
            "roofline": roofline_block(res, key, peak_tflops, peak_measured, sm_count), "build": build_block(res)}
    if "sph" in res:
        line["sph"] = res["sph"]
    pm_head = res.pop("pm")
    del res["o"]
    o.close()

    if not args.no_per_config and world == 1 and not custom and args.workload == "C5":
        # the other BASELINE configs in the same line (fewer steps; same timing rules); C4 carries the SPH rows
        per = {}
        for nm in ("C2", "C3", "C4"):
            r = measure(args, nm, None, args.seed, 5, 3, local, 1, e2e=False, accuracy=(nm == "C2"))
            blk = {"workload": workload_text(nm, r["cfg"], f"theta={r['cfg']['theta']}", args.key_order, args.group_distance),
                   "value": r["value"], "ms_per_step": r["ms_step"], "interactions_per_step": r["inter_all"],
                   "roofline": roofline_block(r, nm, peak_tflops, peak_measured, sm_count), "build": build_block(r)}
            for k in ("sph", "accuracy"):
                if k in r:
                    blk[k] = r[k]
            per[nm] = blk
            r["o"].close()
            del r
        line["per_config"] = per

    if not args.no_cpu_baseline and world == 1:
        rs, what, cores = oracle_sample(args, args.workload, cfg, pm_head, res["delta"], res["m_limit"])
        line["cpu_baseline"] = {"value": rs[0]["value"], "unit": UNIT, "cores": cores, "kind": "oracle",
                                "ms_per_step": rs[0]["ms_per_step"], "sample": what}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
