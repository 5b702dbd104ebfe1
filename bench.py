#!/usr/bin/env python
"""bench.py — energy+force atom-steps/s of the Allegro MD hot path on B200 (BASELINE.json metric).

One "step" = one allegro_md_step(dt, n_md) call = n_md velocity-Verlet steps (neighbour rebuilds on skin
violation included).  Default workload: BASELINE.json configs[3], the largest single-GPU configuration and the one
north_star sets the roofline target on (262,144 atoms, lmax=3, 3 layers, 64 channels, 512-wide MLPs), with
n_md = 1 so that the driver's --steps/--warmup fit its window; --config 0|1|2|4 select the others and --sweep
runs the configs[4] size sweep.  value = atoms * n_md * steps / device time (CUDA events, max over ranks).
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
# MD steps per bench step when --md-steps is not given: sized so that the driver's --steps 20 --warmup 5 stays within minutes
DEFAULT_MD_STEPS = {0: 10, 1: 100, 2: 10, 3: 1, 4: 10}
# centre atoms of one oracle evaluation in the cpu_baseline / reference legs (seconds of host work, bounded memory)
ORACLE_SAMPLE = {0: 64, 1: 512, 2: 256, 3: 96, 4: 512}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--sweep", default="", help="configs[4] size sweep: comma-separated log2 N (e.g. 15,17,19,21,23)")
    ap.add_argument("--log2n", type=int, default=15, help="size for --config 4")
    ap.add_argument("--md-steps", type=int, default=0, help="MD steps per bench step (default: the config's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--decomp", action="store_true",
                    help="N > 1: ONE system decomposed over the ranks (paper_2502_06073_b200/distributed.py, strong scaling) instead of "
                         "the default independent replicas")
    ap.add_argument("--sample-atoms", type=int, default=0, help="reference arm: centre atoms per step")
    return ap.parse_args()


def load_workload(args):
    from paper_2502_06073_b200 import workloads as WL
    w = WL.get(args.config, log2_n=args.log2n) if args.config == 4 else WL.get(args.config)
    n_md = args.md_steps or DEFAULT_MD_STEPS[args.config]
    return WL, w, n_md


def config_dict(w, n_md, extra=None):
    hp = w.hp
    d = {"workload": w.name, "n_atoms": w.n_atoms, "md_steps_per_step": n_md, "dt_fs": w.dt_fs, "skin": w.skin,
         "r_cut": hp["r_cut"], "lmax": hp["lmax"], "n_layers": hp["n_layers"], "n_channels": hp["n_channels"],
         "latent": hp["latent_dims"], "two_body": hp["two_body_dims"], "notes": w.notes,
         "cache": "inputs larger than L2: every MD step streams its activation working set (GBs; >= 1.4 GB already for cfg 1) "
                  "through the 126 MB L2, so no step starts warm; no explicit flush"}
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


class CpuMeter:
    """Average number of busy threads of this process between start() and stop() (user + system CPU time / wall time)."""

    def start(self):
        self.t0, self.c0 = time.perf_counter(), sum(os.times()[:2])
        return self

    def stop(self):
        wall = time.perf_counter() - self.t0
        cpu = sum(os.times()[:2]) - self.c0
        return max(1, int(round(cpu / max(wall, 1e-9)))), wall


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    WL, w, n_md = load_workload(args)
    O, model, nbr = oracle_setup(w)
    rng = np.random.default_rng(123)
    ns = args.sample_atoms or min(w.n_atoms, ORACLE_SAMPLE[args.config])
    centres = np.sort(rng.choice(w.n_atoms, ns, replace=False))
    for _ in range(args.warmup):
        oracle_time_sample(w, model, nbr, centres)
    meter = CpuMeter().start()
    t = [oracle_time_sample(w, model, nbr, centres) for _ in range(args.steps)]
    cores, _ = meter.stop()
    tot = sum(t)
    val = ns * args.steps / tot
    sample = (f"each step = one oracle energy+force evaluation (fp64 numpy) for {ns} seeded centre atoms of {w.name} "
              f"with their full neighbourhoods; the integrator's cost is negligible beside it")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_dict(w, n_md),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "cores_available": len(os.sched_getaffinity(0)),
                             "kind": "oracle", "sample": sample},
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
        sm, mx, pw, reasons = [], [], [], set()
        for ln in out.strip().splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            try:
                pw.append(float(f[3]))
            except ValueError:
                pass
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "power_w": statistics.median(pw) if pw else None}


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


def roofline_for(prof, stats, clocks, peaks, n_sm, n_atoms, ms_md_step):
    """`roofline` object of the JSON line: the dominant kernel class of the profiled MD step against the peak of the pipe that
    bounds it, and the per-step fraction t_roof / t_step of SURVEY.md 8d with its three terms (tensor, FP32 ALU, HBM)."""
    sm_max = (clocks or {}).get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
    sm_now = (clocks or {}).get("sm_mhz") or sm_max
    at_max = sm_now >= 0.97 * sm_max
    # dense 16-bit tensor peak: the burst figure when the SM clock stayed at its maximum over the timed region, else the sustained one
    t16 = (peaks.get("bf16_tflops") if at_max else peaks.get("bf16_tflops_sustained")) or peaks.get("bf16_tflops_sustained") or 1413.0
    t16_src = ("MEASURED_PEAKS.json bf16_tflops (burst: clocks.sm stayed at max)" if at_max else
               "MEASURED_PEAKS.json bf16_tflops_sustained (clocks.sm below max under load)") if peaks else "fallback 1413 TF"
    peak_f16s = t16 / 3.0                           # split-fp16 product = 3 kind::f16 passes (gemm_f16s.cu; fp16 rate = bf16 rate)
    peak_tf32x3 = t16 * (1.1 / 2.25) / 3.0          # 3 x TF32 passes (gemm_tc.cu); TF32 : BF16 nominal ratio of the guide
    fp32_peak = n_sm * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    hbm = peaks.get("hbm_gbs", 6650.0)
    tot_ms = sum(v["ms"] for v in prof.values()) or 1.0
    dom = max((k for k in prof if k not in ("tp_mix", "tp_mix16")), key=lambda k: prof[k]["ms"])
    E_act, E_list = stats["active_edges"], stats["list_edges"]
    chunks = max(1, stats.get("chunks", 1))
    shares = {k: round(v["ms"] / tot_ms, 4) for k, v in prof.items() if v["launches"] and k not in ("tp_mix", "tp_mix16")}
    names = {"gemm": "k_gemm_chain", "gemm_f16s": "k_gemm_f16s", "tp_fwd": "k_tp_fwd3 / k_tpmix_fwd / k_tpo_fwd", "tp_bwd": "k_tp_bwd3 / k_tpo_bwd_ring"}
    roof = {"kernel": names.get(dom, dom), "shares": shares}
    flops = {k: prof[k]["work"] * E_act / chunks for k in ("gemm", "gemm_f16s", "tp_fwd", "tp_bwd", "tp_mix", "tp_mix16") if k in prof}
    traffic, traffic_src = None, None
    try:
        tr = json.load(open(os.path.join(ROOT, "profiles", "r2_traffic.json")))
        ent = tr.get(roof["kernel"], {})
        traffic, traffic_src = ent.get("dram_bytes_per_launch"), ent.get("source")
    except Exception:
        pass
    if dom in flops:
        n_l = prof[dom].get("launches_per_md_step", prof[dom]["launches"])
        ach = flops[dom] / (prof[dom]["ms"] * 1e-3) / 1e12
        peak = {"gemm": peak_tf32x3, "gemm_f16s": peak_f16s}.get(dom, fp32_peak)
        roof.update({"bound": "tensor" if dom.startswith("gemm") else "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                     "frac": ach / peak, "traffic": traffic, "traffic_source": traffic_src, "launches_per_md_step": n_l,
                     "avg_launch_ms": prof[dom]["ms"] / max(1, n_l),
                     "algorithmic_flop_per_launch": flops[dom] / max(1, n_l),
                     "peak_source": {"gemm": t16_src + " x 1.1/2.25 (nominal TF32:BF16) / 3 passes (3xTF32 split, gemm_tc.cu)",
                                     "gemm_f16s": t16_src + " / 3 passes (split-fp16 product hi*hi + hi*lo + lo*hi, gemm_f16s.cu)"}.get(
                                         dom, "148 SM x 128 FP32 lanes x 2 x clocks.max.sm (DESIGN.md)")})
    else:
        roof.update({"bound": "hbm", "achieved": None, "peak": hbm, "unit": "GB/s", "frac": None, "traffic": traffic,
                     "peak_source": "MEASURED_PEAKS.json" if peaks else "fallback"})
    # the tensor-product kernels against the FP32 ALU peak (their coupling arithmetic only: the channel mixing some of them also
    # run on tensor cores is counted in the tensor term below)
    roof["tensor_product"] = {k: {"kernel": names[k], "bound": "alu", "achieved": flops[k] / (prof[k]["ms"] * 1e-3) / 1e12, "peak": fp32_peak,
                                  "unit": "TFLOP/s", "frac": flops[k] / (prof[k]["ms"] * 1e-3) / 1e12 / fp32_peak, "share_of_step": shares.get(k)}
                              for k in ("tp_fwd", "tp_bwd") if k in flops and prof[k]["ms"] > 0}
    # ---- per MD step: t_roof = max(F_gemm / P_tc, F_alu / P_fp32, B_alg / BW_hbm)
    t_tensor = ((flops.get("gemm", 0.0) + flops.get("tp_mix", 0.0)) / (peak_tf32x3 * 1e12) + (flops.get("gemm_f16s", 0.0) + flops.get("tp_mix16", 0.0)) / (peak_f16s * 1e12)) * 1e3
    t_alu = (flops.get("tp_fwd", 0.0) + flops.get("tp_bwd", 0.0)) / (fp32_peak * 1e12) * 1e3
    b_alg = 52.0 * n_atoms + 8.0 * E_list + 96.0 * n_atoms
    t_hbm = b_alg / (hbm * 1e9) * 1e3
    t_roof = max(t_tensor, t_alu, t_hbm)
    roof["per_step"] = {"t_step_ms": ms_md_step, "t_roof_ms": t_roof, "frac": t_roof / ms_md_step,
                        "t_tensor_ms": t_tensor, "t_alu_ms": t_alu, "t_hbm_ms": t_hbm,
                        "gemm_flop": flops.get("gemm", 0.0) + flops.get("gemm_f16s", 0.0) + flops.get("tp_mix", 0.0) + flops.get("tp_mix16", 0.0),
                        "alu_flop": flops.get("tp_fwd", 0.0) + flops.get("tp_bwd", 0.0), "algorithmic_bytes": b_alg,
                        "peaks": {"tensor_f16_split_tflops": peak_f16s, "tensor_tf32x3_tflops": peak_tf32x3, "fp32_tflops": fp32_peak,
                                  "hbm_gbs": hbm, "tensor_peak_kind": "burst" if at_max else "sustained"},
                        "note": "algorithmic flop of one MD step (one force evaluation: forward + input-gradient backward), counted "
                                "once per product whatever the number of tensor passes; the tensor term uses the peak of the kind "
                                "each GEMM runs in divided by its passes"}
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
    for v in prof.values():                       # per MD step: the profiled call ran n_md of them
        v["ms"] /= n_md; v["work"] /= n_md; v["launches_per_md_step"] = v["launches"] / n_md

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
    roof = roofline_for(prof, stats, clocks, peaks, n_sm, N, ms / args.steps / n_md)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 (dense linears: split-fp16 x3 or TF32 x3 tensor-core products, fp32 accumulation)", "data": "synthetic",
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
        ns = min(N, ORACLE_SAMPLE[args.config])
        centres = np.sort(rng.choice(N, ns, replace=False))
        oracle_time_sample(w, omodel, nbr, centres[: max(8, ns // 8)])
        meter = CpuMeter().start()
        reps, tsum = 0, 0.0
        while tsum < 10.0 and reps < 20:
            tsum += oracle_time_sample(w, omodel, nbr, centres); reps += 1
        cores, _ = meter.stop()
        line["cpu_baseline"] = {"value": ns * reps / tsum, "unit": UNIT, "cores": cores, "cores_available": len(os.sched_getaffinity(0)),
                                "kind": "oracle",
                                "sample": f"{reps} oracle energy+force evaluations (fp64 numpy, as it stands) over {ns} seeded centre "
                                          f"atoms of {w.name} with their full neighbourhoods, {tsum:.1f} s of wall time; cores = CPU time / wall time"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_decomp(args):
    """--decomp: one system, spatially decomposed over the ranks.  value = atoms * n_md * steps / time (strong
    scaling: total work fixed).  The one collective of a step is the all-reduce of the force array over NCCL."""
    import torch
    import torch.distributed as dist
    from paper_2502_06073_b200 import binding as B
    from paper_2502_06073_b200.distributed import DistributedAllegro
    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    WL, w, n_md = load_workload(args)
    N = w.n_atoms
    d = DistributedAllegro(B.build_weights(w.hp, w.weight_seed), w.hp, w.cell, rank=rank, world=world)
    vel0 = WL.maxwell_boltzmann(w.mass, w.temperature, w.vel_seed)
    dev = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).cuda()
    pos, vel, mass, sp = dev(w.pos, np.float64), dev(vel0, np.float64), dev(w.mass, np.float64), dev(w.species, np.int32)
    F = torch.zeros((N, 3), dtype=torch.float64, device="cuda")
    d.energy_forces(pos, sp, F)
    for _ in range(args.warmup):
        d.md_step(pos, vel, mass, sp, F, w.dt_fs, n_md)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        E = d.md_step(pos, vel, mass, sp, F, w.dt_fs, n_md)
    ev1.record()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ms, = max_over_ranks([ev0.elapsed_time(ev1)], world, "cuda")
    if rank == 0:
        value = N * n_md * args.steps / (ms * 1e-3)
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                          "dtype": "f32", "data": "synthetic",
                          "config": config_dict(w, n_md, {"parallelism": "spatial decomposition %dx%dx%d, replicated coordinates, one force "
                                                                         "all-reduce per step" % d.grid,
                                                          "owned_atoms_rank0": d.n_owned, "local_atoms_rank0": d.n_local}),
                          "E_pot": float(E.item())}))
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """BASELINE.json configs[4]: the config-1 network on tiled 2.2 g/cc SiO2-like boxes, N = 2^k.  One JSON line with one entry per
    size (atom-steps/s, ms per MD step, per-step roofline fraction, device memory in use); sizes that do not fit end the sweep."""
    import torch
    from paper_2502_06073_b200 import binding as B
    from paper_2502_06073_b200 import workloads as WL
    torch.cuda.set_device(0)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    out = []
    for k in [int(x) for x in args.sweep.split(",")]:
        ent = {"log2_n": k}
        try:
            w = WL.get(4, log2_n=k)
            n_md = args.md_steps or (10 if k <= 21 else 3)
            N = w.n_atoms
            model = B.Allegro(B.build_weights(w.hp, w.weight_seed), w.hp)
            vel0 = WL.maxwell_boltzmann(w.mass, w.temperature, w.vel_seed)
            dev = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).cuda()
            model.md_init(dev(w.pos, np.float64), dev(vel0, np.float64), dev(w.mass, np.float64), dev(w.species, np.int32), w.cell,
                          w.hp["r_cut"], w.skin)
            model.md_step(w.dt_fs, 2)
            torch.cuda.synchronize()
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record()
            for _ in range(args.steps):
                model.md_step(w.dt_fs, n_md)
            ev1.record(); torch.cuda.synchronize()
            ms = ev0.elapsed_time(ev1) / (args.steps * n_md)
            st = model.get_stats()
            model.profile(True); model.md_step(w.dt_fs, 2); prof = model.get_profile(); model.profile(False)
            for v in prof.values():
                v["ms"] /= 2.0; v["work"] /= 2.0
            roof = roofline_for(prof, st, None, peaks, n_sm, N, ms)
            free_b, total_b = torch.cuda.mem_get_info()
            ent.update({"n_atoms": N, "active_edges": st["active_edges"], "list_edges": st["list_edges"], "chunks": st["chunks"],
                        "ms_per_md_step": ms, "atom_steps_per_s": N / (ms * 1e-3), "per_step_roofline_frac": roof["per_step"]["frac"],
                        "t_roof_ms": roof["per_step"]["t_roof_ms"], "device_mem_used_gb": (total_b - free_b) / 1e9})
            del model
            torch.cuda.empty_cache()
        except Exception as e:   # out of memory (host or device) ends the sweep
            ent["error"] = str(e)[:200]
            out.append(ent)
            break
        out.append(ent)
    print(json.dumps({"metric": METRIC, "unit": UNIT, "sweep": "BASELINE.json configs[4] (config-1 network, tiled SiO2-like boxes)",
                      "n_gpus": 1, "data": "synthetic", "entries": out}))


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    elif args.sweep:
        run_sweep(args)
    elif args.decomp:
        run_decomp(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
