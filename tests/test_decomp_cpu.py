"""SURVEY.md 8f-3 on CPU: the decomposition scheme of paper_2502_06073_b200/distributed.py with two gloo ranks.

The CUDA selection kernel cannot run here, so the local sets are built with numpy from the module's own brick arithmetic
(rank_grid / rank_coord / brick_bounds), the fp64 oracle evaluates each rank's owned atoms (its `centres=` mode is exactly
allegro_energy_forces_owned), the per-rank force arrays are all-reduced over gloo, and the result must equal the
single-domain oracle to round-off: energies add up, ghost forces land on their owners."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _local_set(pos, cell, grid, coord, r_halo):
    """numpy restatement of allegro_decomp_select: owned first, then ghost images, ascending atom index."""
    from paper_2502_06073_b200.distributed import brick_bounds
    L = np.diag(cell)
    lo, hi = brick_bounds(cell, grid, coord)
    dec = [g > 1 for g in grid]
    w = pos.copy()
    for d in range(3):
        if dec[d]:
            w[:, d] -= np.floor(w[:, d] / L[d]) * L[d]
    owned = np.ones(len(pos), bool)
    for d in range(3):
        if dec[d]:
            owned &= (w[:, d] >= lo[d]) & (w[:, d] < hi[d])
    own_idx = np.nonzero(owned)[0]
    g_src, g_pos = [], []
    rng = [(-1, 0, 1) if dec[d] else (0,) for d in range(3)]
    for i in range(len(pos)):
        for sx in rng[0]:
            for sy in rng[1]:
                for sz in rng[2]:
                    if owned[i] and (sx, sy, sz) == (0, 0, 0):
                        continue
                    c = w[i] + np.array([sx, sy, sz]) * L
                    if all((not dec[d]) or (lo[d] - r_halo <= c[d] < hi[d] + r_halo) for d in range(3)):
                        g_src.append(i); g_pos.append(c)
    origin = np.array([lo[d] - r_halo if dec[d] else 0.0 for d in range(3)])
    lpos = np.concatenate([w[own_idx], np.array(g_pos).reshape(-1, 3)]) - origin
    lsrc = np.concatenate([own_idx, np.array(g_src, dtype=np.int64)])
    lcell = np.diag([(hi[d] - lo[d]) + 3 * r_halo + 1.0 if dec[d] else L[d] for d in range(3)])
    return len(own_idx), lpos, lsrc.astype(np.int64), lcell


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    from oracle import allegro_oracle as O
    from paper_2502_06073_b200 import workloads as WL
    from paper_2502_06073_b200.distributed import rank_coord, rank_grid
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    hp = WL.hparams(2, 2, 2, 4, [16, 12], [16, 12], [8], 3.0, 12.0)
    model = O.AllegroOracle(hp, WL.make_weights(O.weight_layout(hp), hp, 5))
    pos, sp, cell = WL.small_periodic(6, 2.3, 0.35, 2, seed=51)          # box 13.8 = 2 bricks of 6.9 >= 2 r_c
    pos = pos + np.array([20.0, -7.0, 3.0])                              # unwrapped input
    grid = rank_grid(world)
    n_owned, lpos, lsrc, lcell = _local_set(pos, cell, grid, rank_coord(rank, grid), hp["r_cut"])
    E, Fl, _ = model.energy_forces(lpos, sp[lsrc], lcell, O.neighbors_bruteforce(lpos, lcell, hp["r_cut"]), centres=np.arange(n_owned))
    assert len(set(lsrc.tolist())) == len(lsrc)                           # every atom at most once per rank
    F = np.zeros_like(pos)
    F[lsrc] = Fl
    tF, tE, tn = torch.from_numpy(F), torch.tensor([E], dtype=torch.float64), torch.tensor([n_owned])
    dist.all_reduce(tF); dist.all_reduce(tE); dist.all_reduce(tn)
    Eo, Fo, _ = model.energy_forces(pos, sp, cell, O.neighbors_bruteforce(pos, cell, hp["r_cut"]))
    q.put((rank, int(tn.item()), float(abs(tE.item() - Eo) / abs(Eo)), float(np.abs(tF.numpy() - Fo).max() / np.abs(Fo).max()), n_owned, len(lsrc)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_decomposition_equals_single_domain():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29741, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, n_total, dE, dF, n_owned, n_local in res:
        assert n_total == 216                                             # every atom owned exactly once
        assert dE < 1e-12 and dF < 1e-11, (dE, dF)
        assert 0 < n_owned < 216 and n_local > n_owned                    # a real split with ghosts


def test_rank_grid_and_bricks():
    sys.path.insert(0, ROOT)
    from paper_2502_06073_b200.distributed import brick_bounds, rank_coord, rank_grid
    assert rank_grid(1) == (1, 1, 1) and rank_grid(2) == (2, 1, 1) and rank_grid(4) == (2, 2, 1) and rank_grid(8) == (2, 2, 2)
    assert rank_grid(6) == (3, 2, 1)
    cell = np.diag([10.0, 12.0, 14.0])
    for world in (2, 4, 8, 6):
        g = rank_grid(world)
        coords = {rank_coord(r, g) for r in range(world)}
        assert len(coords) == world
        vol = 0.0
        for c in coords:
            lo, hi = brick_bounds(cell, g, c)
            assert np.all(hi > lo)
            vol += float(np.prod(hi - lo))
        assert abs(vol - 10 * 12 * 14) < 1e-9                             # the bricks tile the cell
