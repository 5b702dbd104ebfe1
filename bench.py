#!/usr/bin/env python
"""bench.py — energy+force atom-steps/s of the Allegro MD hot path on B200 (BASELINE.json metric).

One "step" = one allegro_md_step(dt, n_md) call = n_md velocity-Verlet steps (neighbour rebuilds on skin
violation included) of BASELINE.json configs[1] (4,096-atom SiO2-like box, lmax=2, 2 layers, 16 channels)
unless --config says otherwise.  value = atoms * n_md * steps / device time (CUDA events, max over ranks).
`e2e` repeats it through the same C-ABI calls with HOST buffers: pinned host -> device copies of the inputs,
allegro_md_init, allegro_md_step, allegro_get_state and device -> host copies of the results inside the
timed region.  N > 1 GPUs: independent replicas (the path does not shard in this build).

--impl reference times the fp64 CPU oracle (oracle/, as it stands) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "energy+force atom-steps/s"
UNIT = "atom-steps/s"
FP32_LANES_PER_SM = 128


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--log2n", type=int, default=15, help="size for --config 4")
    ap.add_argument("--md-steps", type=int, default=0, help="MD steps per bench step (default: the config's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sample-atoms", type=int, default=0, help="reference arm: centre atoms per step")
    return ap.parse_args()


def load_workload(args):
    from paper_2502_06073_b200 import workloads as WL
    w = WL.get(args.config, log2_n=args.log2n) if args.config == 4 else WL.get(args.config)
    n_md = args.md_steps or w.n_steps
    return WL, w, n_md


def config_dict(w, n_md, extra=None):
    hp = w.hp
    d = {"workload": w.name, "n_atoms": w.n_atoms, "md_steps_per_step": n_md, "dt_fs": w.dt_fs, "skin": w.skin,
         "r_cut": hp["r_cut"], "lmax": hp["lmax"], "n_layers": hp["n_layers"], "n_channels": hp["n_channels"],
         "latent": hp["latent_dims"], "two_body": hp["two_body_dims"], "notes": w.notes,
         "cache": "inputs larger than L2: the per-step activation working set (about 1.4 GB for cfg 1) exceeds the 126 MB L2; no explicit flush"}
    if extra:
        d.update(extra)
    return d


# ------------------------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the oracle as it stands, on the host cores
# ------------------------------------------------------------------------------------------------------------
def oracle_setup(w):
    from oracle import allegro_oracle as O
    from paper_2502_06073_b200 import workloads as WL
    weights = WL.make_weights(O.weight_layout(w.hp), w.hp, w.weight_seed)
    model = O.AllegroOracle(w.hp, weights)
    nbr = O.neighbors_binned(w.pos, w.cell, w.hp["r_cut"] + w.skin)
    return O, model, nbr


def oracle_time_sample(w, model, nbr, centres):
    t0 = time.perf_counter()
    model.energy_forces(w.pos, w.species, w.cell, nbr, centres=centres)
    return time.perf_counter() - t0


def cores_used():
    try:
        import threadpoolctl
        n = max([p["num_threads"] for p in threadpoolctl.threadpool_info()] + [1])
    except Exception:
        n = 1
    return min(n, len(os.sched_getaffinity(0)))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    WL, w, n_md = load_workload(args)
    O, model, nbr = oracle_setup(w)
    rng = np.random.default_rng(123)
    ns = args.sample_atoms or min(w.n_atoms, 512)
    centres = np.sort(rng.choice(w.n_atoms, ns, replace=False))
    for _ in range(args.warmup):
        oracle_time_sample(w, model, nbr, centres)
    t = [oracle_time_sample(w, model, nbr, centres) for _ in range(args.steps)]
    tot = sum(t)
    val = ns * args.steps / tot
    sample = (f"each step = one oracle energy+force evaluation (fp64 numpy) for {ns} seeded centre atoms of {w.name} "
              f"with their full neighbourhoods; the integrator's cost is negligible beside it")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_dict(w, n_md),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores_used(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, dev):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={dev}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if not self.p:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill(); out = ""
        sm, mx, reasons = [], [], set()
        for ln in out.strip().splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def max_over_ranks(values, world, device="cpu"):
    """Device times of a multi-replica run are the MAX over ranks (one process per GPU, replicas only: there is no
    data-path collective, this all-reduce of a few timings is the only communication)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_value(world, n_atoms, n_md, steps, ms):
    """atom-steps/s of the whole job: every replica advances its own n_atoms system (weak scaling)."""
    return world * n_atoms * n_md * steps / (ms * 1e-3)


def roofline_for(prof, stats, clocks, peaks, n_sm):
    """`roofline` object of the JSON line for the dominant kernel class of the profiled step."""
    sm_max = (clocks or {}).get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
    fp32_peak = n_sm * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    tot_ms = sum(v["ms"] for v in prof.values()) or 1.0
    dom = max(prof, key=lambda k: prof[k]["ms"])
    E_act = stats["active_edges"]
    shares = {k: round(v["ms"] / tot_ms, 4) for k, v in prof.items() if v["launches"]}
    names = {"gemm": "k_gemm_chain", "tp_fwd": "k_tp_fwd3", "tp_bwd": "k_tp_bwd3"}
    roof = {"kernel": names.get(dom, dom), "shares": shares}
    traffic = None
    try:
        tr = json.load(open(os.path.join(ROOT, "profiles", "r1_traffic.json")))
        traffic = tr.get(roof["kernel"], {}).get("dram_bytes_per_launch")
    except Exception:
        pass
    if dom in ("gemm", "tp_fwd", "tp_bwd"):
        # algorithmic flop of all launches of the class: `work` sums flop per edge over launches, and every launch
        # covers one atom chunk, i.e. active_edges / chunks edges on average
        flops = prof[dom]["work"] * E_act / max(1, stats.get("chunks", 1))
        ach = flops / (prof[dom]["ms"] * 1e-3) / 1e12
        common = {"achieved": ach, "unit": "TFLOP/s", "traffic": traffic, "launches": prof[dom]["launches"],
                  "avg_launch_ms": prof[dom]["ms"] / max(1, prof[dom]["launches"]),
                  "algorithmic_flop_per_launch": flops / max(1, prof[dom]["launches"])}
        if dom == "gemm":
            bf16 = peaks.get("bf16_tflops_sustained") or peaks.get("bf16_tflops") or 1413.0
            tf32 = bf16 * (1.1 / 2.25)                                  # guide's nominal TF32 : BF16 dense ratio
            peak = tf32 / 3.0                                           # fp32-accurate product = 3 TF32 passes
            roof.update({"bound": "tensor", "peak": peak, "frac": ach / peak, **common,
                         "peak_source": ("MEASURED_PEAKS.json bf16_tflops_sustained x 1.1/2.25 (nominal TF32:BF16) / 3 "
                                         "(3-pass hi/lo TF32 split needed for the 1e-4 x RMS force gate)") if peaks else
                                        "fallback 1413 TF bf16 sustained x 1.1/2.25 / 3",
                         "peak_tf32_dense": tf32})
        else:
            roof.update({"bound": "alu", "peak": fp32_peak, "frac": ach / fp32_peak, **common,
                         "peak_source": "148 SM x 128 FP32 lanes x 2 x clocks.max.sm (DESIGN.md)"})
    else:
        hbm = peaks.get("hbm_gbs", 6650.0)
        roof.update({"bound": "hbm", "achieved": None, "peak": hbm, "unit": "GB/s", "frac": None, "traffic": traffic,
                     "peak_source": "MEASURED_PEAKS.json" if peaks else "fallback"})
    return roof


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2502_06073_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    WL, w, n_md = load_workload(args)
    N = w.n_atoms
    weights = B.build_weights(w.hp, w.weight_seed)
    model = B.Allegro(weights, w.hp)
    vel0 = WL.maxwell_boltzmann(w.mass, w.temperature, w.vel_seed)
    dev = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).cuda()
    pos_d, vel_d, mass_d, sp_d = dev(w.pos, np.float64), dev(vel0, np.float64), dev(w.mass, np.float64), dev(w.species, np.int32)
    rc, skin = w.hp["r_cut"], w.skin

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: state lives in the handle; inputs already in HBM
    model.md_init(pos_d, vel_d, mass_d, sp_d, w.cell, rc, skin)
    for _ in range(args.warmup):
        model.md_step(w.dt_fs, n_md)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    rebuilds = 0
    ev0.record()
    for _ in range(args.steps):
        model.md_step(w.dt_fs, n_md)
        st = model.get_stats()
        launches += st["launches"]; rebuilds += st["rebuilds"]
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if sampler else None
    stats = model.get_stats()
    Ep = torch.zeros(1, dtype=torch.float64, device="cuda"); Ek = torch.zeros(1, dtype=torch.float64, device="cuda")
    model.get_state(E_pot=Ep, E_kin=Ek)

    # ---- end to end through the C-ABI with host buffers
    pin = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).pin_memory()
    h_pos, h_vel, h_mass, h_sp = pin(w.pos, np.float64), pin(vel0, np.float64), pin(w.mass, np.float64), pin(w.species, np.int32)
    o_pos = torch.empty((N, 3), dtype=torch.float64).pin_memory(); o_vel = torch.empty_like(o_pos).pin_memory()
    o_F = torch.empty_like(o_pos).pin_memory(); o_E = torch.empty(2, dtype=torch.float64).pin_memory()
    d_pos, d_vel, d_F = torch.empty_like(pos_d), torch.empty_like(pos_d), torch.empty_like(pos_d)
    d_mass, d_sp = torch.empty_like(mass_d), torch.empty_like(sp_d)
    d_E = torch.zeros(2, dtype=torch.float64, device="cuda")
    h2d = h_pos.numel() * 8 + h_vel.numel() * 8 + h_mass.numel() * 8 + h_sp.numel() * 4
    d2h = 3 * o_pos.numel() * 8 + 16

    def e2e_step():
        d_pos.copy_(h_pos, non_blocking=True); d_vel.copy_(h_vel, non_blocking=True)
        d_mass.copy_(h_mass, non_blocking=True); d_sp.copy_(h_sp, non_blocking=True)
        model.md_init(d_pos, d_vel, d_mass, d_sp, w.cell, rc, skin)
        model.md_step(w.dt_fs, n_md)
        model.get_state(d_pos, d_vel, d_F, d_E[0:1], d_E[1:2])
        o_pos.copy_(d_pos, non_blocking=True); o_vel.copy_(d_vel, non_blocking=True)
        o_F.copy_(d_F, non_blocking=True); o_E.copy_(d_E, non_blocking=True)
        torch.cuda.synchronize()

    e2e_step()
    barrier()
    k_e2e = max(1, min(args.steps, 3))
    ev0.record()
    for _ in range(k_e2e):
        e2e_step()
    ev1.record()
    barrier()
    ms_e2e = ev0.elapsed_time(ev1)

    # ---- per-kernel-class times for the roofline line (separate pass, CUDA events around every launch)
    model.md_init(pos_d, vel_d, mass_d, sp_d, w.cell, rc, skin)
    model.md_step(w.dt_fs, n_md)
    model.profile(True)
    model.md_step(w.dt_fs, n_md)
    prof = model.get_profile()
    model.profile(False)

    ms, ms_e2e = max_over_ranks([ms, ms_e2e], world, "cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = whole_job_value(world, N, n_md, args.steps, ms)
    e2e_val = whole_job_value(world, N, n_md, k_e2e, ms_e2e)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    E_act = stats["active_edges"]
    roof = roofline_for(prof, stats, clocks, peaks, n_sm)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": config_dict(w, n_md, {"parallelism": "replicas" if world > 1 else "single",
                                            "active_edges": E_act, "list_edges": stats["list_edges"],
                                            "rebuilds_in_timed_region": rebuilds}),
            "ns_per_day": value / (world * N) * w.dt_fs * 1e-6 * 86400.0,
            "us_per_atom_step": 1e6 / value,
            "E_pot": float(Ep.item()), "E_kin": float(Ek.item()),
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": k_e2e, "ms_per_step": ms_e2e / k_e2e,
                    "includes": "pinned H2D of pos/vel/mass/species, allegro_md_init (list build + first force call), "
                                "allegro_md_step, allegro_get_state, D2H of pos/vel/F/E"},
            "gpu_launches": launches,
            "roofline": roof}

    if not args.no_cpu_baseline:
        O, omodel, nbr = oracle_setup(w)
        rng = np.random.default_rng(123)
        ns = min(N, 512)
        centres = np.sort(rng.choice(N, ns, replace=False))
        oracle_time_sample(w, omodel, nbr, centres[:32])
        reps, tsum = 0, 0.0
        while tsum < 10.0 and reps < 20:
            tsum += oracle_time_sample(w, omodel, nbr, centres); reps += 1
        line["cpu_baseline"] = {"value": ns * reps / tsum, "unit": UNIT, "cores": cores_used(), "kind": "oracle",
                                "sample": f"{reps} oracle energy+force evaluations (fp64 numpy, as it stands) over {ns} seeded centre "
                                          f"atoms of {w.name} with their full neighbourhoods, {tsum:.1f} s of CPU work"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
