#!/usr/bin/env python
"""bench.py -- one JSON line for the OTOO force path on B200.

A step = one pass of the whole hot path (tree build + fused walk/gravity)
over one batch of synthetic particles already resident in HBM.  metric = gravity
interactions/s (R11 count / device time of the whole step).  `roofline` is for the dominant
kernel (walk_gravity_kernel) against the non-tensor FP32 peak; `e2e` goes through the host-buffer
C-ABI call; `cpu_baseline` is the fp64 oracle timed on this box's host cores.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--theta 0.6]
    python bench.py --impl reference ...      # times the oracle (CPU) on the same workload
"""
from __future__ import annotations

import argparse
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
BUILD_BYTES_PER_PARTICLE = 390      # algorithmic HBM bytes of the tree build per particle


def hbm_peak_gbs():
    """measured HBM copy bandwidth of this pool (driver-written MEASURED_PEAKS.json), else the guide's fallback"""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json"
    except Exception:
        return 6650.0, "fallback of B200_PROFILING.md"
SM_LANES = 128                      # FP32 lanes per SM
NOMINAL_SM_MHZ = 1965.0


def workload(name: str, theta, seed: int, n=None):
    cfg = dict(gen.CONFIGS[name])
    if theta is not None:
        cfg["theta"] = theta
    if n is not None:
        cfg["n"] = int(n)
    pm = gen.make(cfg["kind"], cfg["n"], seed)
    return cfg, pm


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


def run_reference(args, rank):
    """The reference arm of this tier: the oracle as it stands, on the host cores."""
    if rank != 0:
        return
    from oracle import oracle
    cfg, pm = workload(args.workload, args.theta, args.seed, args.n)
    eps, theta = float(np.float32(cfg["eps"])), float(np.float32(cfg["theta"]))
    times, inter = [], 0
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        t = oracle.Tree(pm, cfg["n_crit"], key_order=1 if args.key_order == "hilbert" else 0)
        t.set_dist_kind(1 if args.group_distance == "exact" else 0)
        rb2 = None
        if args.mac == "delta":
            rb2 = t.rb2_delta(float(np.float32(args.delta if args.delta is not None else cfg.get("delta", 0.01))),
                              float(np.float32(args.m_limit if args.m_limit is not None else cfg.get("m_limit", 0.05))))
        r = t.gravity(eps, theta, cfg["group"], rb2=rb2)
        dt = time.perf_counter() - t0
        inter = r["interactions"]
        del t
        if it >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    val = inter / (ms * 1e-3)
    cores = oracle.max_threads()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload}: {cfg['kind']} N={cfg['n']} eps={cfg['eps']} theta={cfg['theta']} "
                                   f"n_crit={cfg['n_crit']} group={cfg['group']}"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": "whole workload, tree build + walk + fp64 sums per step"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="otoo", choices=["otoo", "reference"])
    ap.add_argument("--workload", default="C2", choices=sorted(gen.CONFIGS))
    ap.add_argument("--theta", type=float, default=None)
    ap.add_argument("--mac", default="theta", choices=["theta", "delta"],
                    help="delta: the paper's absolute-error MAC (otoo_gravity_delta) instead of BASELINE's theta criterion")
    ap.add_argument("--key-order", default="morton", choices=["morton", "hilbert"],
                    help="hilbert: the paper's ordering (L131) instead of BASELINE's Morton-contiguous groups")
    ap.add_argument("--group-distance", default="box", choices=["box", "exact"],
                    help="exact: the paper's minimum over the members' distances (L163) instead of the group box distance")
    ap.add_argument("--delta", type=float, default=None)
    ap.add_argument("--m-limit", type=float, default=None)
    ap.add_argument("--seed", type=int, default=1206)
    ap.add_argument("--n", type=int, default=None, help="override the workload's particle count (scaling runs, e.g. Fig. 9)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
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
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    # replicas only: every rank runs the same workload with its own seed
    cfg, pm = workload(args.workload, args.theta, replicas.replica_seed(args.seed, rank), args.n)
    n, G, n_crit = cfg["n"], cfg["group"], cfg["n_crit"]
    eps, theta = float(np.float32(cfg["eps"])), float(np.float32(cfg["theta"]))
    delta = float(np.float32(args.delta if args.delta is not None else cfg.get("delta", 0.01)))
    m_limit = float(np.float32(args.m_limit if args.m_limit is not None else cfg.get("m_limit", 0.05)))
    o = binding.Otoo(max_particles=n, device=local)
    o.otoo_set_option("key_order", 1 if args.key_order == "hilbert" else 0)
    o.otoo_set_option("group_distance", 1 if args.group_distance == "exact" else 0)
    d_pm = torch.from_numpy(pm).cuda()
    out = torch.empty((n, 4), dtype=torch.float32, device="cuda")
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step(timed):
        flush_buf.fill_(1)                      # L2 flush between steps, outside the timed events
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        e[0].record()
        o.otoo_build_tree(d_pm, n_crit)
        l1 = o.otoo_last_stats()["launches"] if not timed else 0
        e[1].record()
        if args.mac == "delta":
            o.otoo_gravity_delta(eps, delta, m_limit, G, out=out)
        else:
            o.otoo_gravity(eps, theta, G, out=out)
        e[2].record()
        return e, l1

    launches_build = 0
    for _ in range(max(args.warmup, 3)):
        _, launches_build = step(False)
    torch.cuda.synchronize()
    st = o.otoo_last_stats()
    launches_step = launches_build + st["launches"]
    inter = st["sum_interactions"]
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    evs = [step(True)[0] for _ in range(args.steps)]
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.result()
    t_build = np.array([e[0].elapsed_time(e[1]) for e in evs])
    t_grav = np.array([e[1].elapsed_time(e[2]) for e in evs])
    ms_step = float((t_build + t_grav).mean())
    ms_max, inter_all = replicas.aggregate(ms_step, float(inter), device="cuda")   # max over ranks, sum over ranks
    value = inter_all / (ms_max * 1e-3)

    # ---- end to end through the host-buffer C-ABI call (pinned host memory)
    h_in = torch.from_numpy(pm).pin_memory()
    h_out = torch.empty((n, 4), dtype=torch.float32).pin_memory()
    e2e_t = []
    for it in range(2 + min(args.steps, 5)):
        flush_buf.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        if args.mac == "delta":      # same public calls on pinned host buffers (there is no host form of the Delta entry point)
            d_in = h_in.cuda(non_blocking=True)
            o.otoo_build_tree(d_in, n_crit)
            h_out.copy_(o.otoo_gravity_delta(eps, delta, m_limit, G, out=out), non_blocking=True)
            torch.cuda.synchronize()
        else:
            o.otoo_gravity_host(h_in.numpy(), n_crit, eps, theta, G, out=h_out.numpy())
        dt = time.perf_counter() - t0
        if it >= 2:
            e2e_t.append(dt)
    e2e_ms, _ = replicas.aggregate(1e3 * float(np.mean(e2e_t)), float(inter), device="cuda")
    e2e_val = inter_all / (e2e_ms * 1e-3)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak_measured = o.otoo_measure_fp32_peak()      # FFMA2-only kernel on this GPU, at the clock it holds
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    peak_tflops = sm_count * SM_LANES * 2 * NOMINAL_SM_MHZ * 1e6 / 1e12
    grav_ms = float(t_grav.mean())
    achieved = FLOPS_PER_INTERACTION * inter / (grav_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": "walk_gravity_ws_kernel", "achieved": achieved, "peak": peak_tflops,
                "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                # dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the committed capture
                # profiles/r1_walk_gravity_full.md (C2, theta=0.6 only); the kernel is ALU-bound, DRAM < 1 %
                "traffic": 53.70e6 if (args.workload == "C2" and args.theta is None and args.n is None and args.mac == "theta"
                                       and args.key_order == "morton" and args.group_distance == "box") else None,
                "peak_source": f"derived: {sm_count} SMs x 128 FP32 lanes x 2 flop x {NOMINAL_SM_MHZ:.0f} MHz (DESIGN.md)",
                "peak_measured_ffma": peak_measured, "frac_of_measured": achieved / peak_measured,
                "flops_per_interaction": FLOPS_PER_INTERACTION, "interactions_per_launch": inter,
                "kernel_ms": grav_ms, "interactions_per_s_kernel": inter / (grav_ms * 1e-3),
                "build_ms": float(t_build.mean())}

    mac_txt = f"theta={cfg['theta']}" if args.mac == "theta" else f"Delta-MAC delta={delta:g} m_limit={m_limit:g}"
    hbm, hbm_src = hbm_peak_gbs()
    build_ms = float(t_build.mean())
    build_gbs = BUILD_BYTES_PER_PARTICLE * n / (build_ms * 1e-3) / 1e9
    build_info = {"ms": build_ms, "bound": "hbm", "algorithmic_bytes": BUILD_BYTES_PER_PARTICLE * n, "achieved_gbs": build_gbs,
                  "peak_gbs": hbm, "frac": build_gbs / hbm, "peak_source": hbm_src}
    sph_info = None
    if cfg["kind"] in ("wd_pair", "cold_sphere") and world == 1:
        # BASELINE config 4 / the paper's cold collapse: the SPH rows (H11-H13) on the same tree, timed like the gravity step
        w = (gen.wd_pair if cfg["kind"] == "wd_pair" else gen.cold_sphere)(n, replicas.replica_seed(args.seed, rank))
        d_h, d_u, d_v = (torch.from_numpy(w[k]).cuda() for k in ("h", "u", "vel"))
        Gs = cfg.get("group_sph", 64)
        ts = []
        for it in range(3 + args.steps):
            flush_buf.fill_(1)
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            ev[0].record()
            rho, nn = o.otoo_sph_density(d_h, Gs)
            P = o.otoo_eos_ideal(rho, d_u, 5.0 / 3.0)
            ev[1].record()
            o.otoo_sph_force(d_h, rho, P, Gs, vel=d_v)
            ev[2].record()
            torch.cuda.synchronize()
            if it >= 3:
                ts.append((ev[0].elapsed_time(ev[1]), ev[1].elapsed_time(ev[2])))
        cand = o.otoo_last_stats()["sum_interactions"]
        td, tf = float(np.mean([x[0] for x in ts])), float(np.mean([x[1] for x in ts]))
        sph_info = {"group": Gs, "density_eos_ms": td, "force_dudt_ms": tf, "candidate_pairs_per_pass": cand,
                    "neighbour_pairs": int(nn.sum().item()), "candidate_pairs_per_s": 2 * cand / ((td + tf) * 1e-3)}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_max, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{args.workload}: {cfg['kind']} N={n} eps={cfg['eps']} {mac_txt} "
                                   f"n_crit={n_crit} group={G} order={args.key_order} distance={args.group_distance}",
                       "l2": "flushed between steps (256 MiB write, outside the timed events)",
                       "parallelism": "replicas" if world > 1 else "single"},
            "gflops": FLOPS_PER_INTERACTION * value / 1e9,
            "interactions_per_step": inter_all, "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 16 * n,
                    "ms_per_step": e2e_ms},
            "gpu_launches": int(launches_step * args.steps), "roofline": roofline, "build": build_info}
    if sph_info:
        line["sph"] = sph_info

    if not args.no_cpu_baseline and world == 1:
        from oracle import oracle
        t0 = time.perf_counter()
        t = oracle.Tree(pm, n_crit, key_order=1 if args.key_order == "hilbert" else 0)
        t.set_dist_kind(1 if args.group_distance == "exact" else 0)
        r = t.gravity(eps, theta, G, forces=True, rb2=t.rb2_delta(delta, m_limit) if args.mac == "delta" else None)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": r["interactions"] / dt, "unit": UNIT, "cores": oracle.max_threads(),
                                "kind": "oracle", "ms_per_step": 1e3 * dt,
                                "sample": "whole workload, one step: tree build + walk + fp64 sums"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
