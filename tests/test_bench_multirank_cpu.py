"""N > 1 path of bench.py on CPU: one process per replica, gloo backend, world_size 2.

The hot path does not shard in this build ("replicas only"): the only communication of a
multi-GPU run is the MAX over ranks of the device-timed milliseconds, and `value` is the whole-job throughput of
all replicas.  This test runs that host logic with two gloo ranks."""
import os
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, ms_e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 20.0 - 3.0 * rank], world, "cpu")
    out.put((rank, ms, ms_e2e, bench.whole_job_value(world, 4096, 100, 5, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29731, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, ms_e2e, value in res:
        assert ms == 15.0 and ms_e2e == 20.0                       # MAX over ranks, identical on every rank
        assert abs(value - 2 * 4096 * 100 * 5 / 15e-3) < 1e-6 * value


def test_roofline_object_shape():
    sys.path.insert(0, ROOT)
    import bench
    prof = {"gemm_f16s": dict(ms=2.0, launches=10, work=1.0e5), "gemm": dict(ms=0.2, launches=2, work=1.0e4),
            "tp_fwd": dict(ms=0.5, launches=2, work=3.0e4), "md": dict(ms=0.1, launches=4, work=0.0)}
    stats = {"active_edges": 100000, "list_edges": 130000, "chunks": 1}
    peaks = {"bf16_tflops": 1668.6, "bf16_tflops_sustained": 1361.0, "hbm_gbs": 6548.8}
    roof = bench.roofline_for(prof, stats, {"sm_max_mhz": 1965.0, "sm_mhz": 1965.0}, peaks, 148, 4096, 3.0)
    assert roof["bound"] == "tensor" and roof["unit"] == "TFLOP/s" and roof["kernel"] == "k_gemm_f16s"
    assert abs(roof["achieved"] - 1.0e5 * 1e5 / 2e-3 / 1e12) < 1e-9
    assert abs(roof["peak"] - 1668.6 / 3.0) < 1e-9                       # burst peak: the clock stayed at max; 3 fp16 passes
    assert abs(roof["frac"] - roof["achieved"] / roof["peak"]) < 1e-12
    assert abs(sum(roof["shares"].values()) - 1.0) < 1e-3
    ps = roof["per_step"]
    t_tensor = (1.0e4 * 1e5 / (1668.6 * (1.1 / 2.25) / 3 * 1e12) + 1.0e5 * 1e5 / (1668.6 / 3 * 1e12)) * 1e3
    assert abs(ps["t_tensor_ms"] - t_tensor) < 1e-9
    assert abs(ps["t_alu_ms"] - 3.0e4 * 1e5 / (148 * 128 * 2 * 1965e6) * 1e3) < 1e-9
    assert abs(ps["t_hbm_ms"] - (148.0 * 4096 + 8 * 130000) / 6548.8e9 * 1e3) < 1e-12
    assert ps["t_roof_ms"] == max(ps["t_tensor_ms"], ps["t_alu_ms"], ps["t_hbm_ms"]) and abs(ps["frac"] - ps["t_roof_ms"] / 3.0) < 1e-12
    # below-max clocks select the sustained peak
    roof2 = bench.roofline_for(prof, stats, {"sm_max_mhz": 1965.0, "sm_mhz": 1500.0}, peaks, 148, 4096, 3.0)
    assert abs(roof2["peak"] - 1361.0 / 3.0) < 1e-9
