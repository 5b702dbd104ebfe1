"""SURVEY.md 8f-3 on one GPU: every rank of a 2-, 4- and 8-rank decomposition is evaluated in turn by the same process (the
ranks do not wait on one another, so running them one after the other is exact); the summed energies and force arrays —
what the all-reduce of paper_2502_06073_b200/distributed.py produces — must equal the single-domain GPU result and the
fp64 oracle; allegro_energy_forces_owned alone is checked against the oracle's `centres=` mode."""
import math

import numpy as np
import pytest

from oracle import allegro_oracle as O
from paper_2502_06073_b200 import workloads as WL

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_energy_forces_owned_matches_oracle_centres(lib):
    import torch
    hp = WL.hparams(3, 2, 2, 16, [24, 32], [48, 32], [12], 4.0, 18.0, n_bessel=6)
    w = lib.build_weights(hp, 61)
    g, o = lib.Allegro(w, hp), O.AllegroOracle(hp, w)
    pos, sp, cell = WL.small_periodic(5, 2.2, 0.4, 3, seed=62)            # 125 atoms, box 11
    n_owned = 70
    p, s = _dev(pos), _dev(sp.astype(np.int32))
    E = torch.zeros(1, dtype=torch.float64, device="cuda"); F = torch.zeros((125, 3), dtype=torch.float64, device="cuda")
    Ea = torch.zeros(125, dtype=torch.float32, device="cuda")
    g.build_neighbors(p, s, cell, 4.0, 0.3)
    g.energy_forces_owned(p, s, cell, n_owned, E, F, Ea)
    Eo, Fo, Eao = o.energy_forces(pos, sp, cell, O.neighbors_bruteforce(pos, cell, 4.0), centres=np.arange(n_owned))
    rms = math.sqrt((Fo ** 2).mean())
    assert abs(float(E.item()) - Eo) <= 1e-5 * abs(Eo)
    assert np.abs(F.cpu().numpy() - Fo).max() <= 1e-4 * rms
    np.testing.assert_allclose(Ea.cpu().numpy()[:n_owned], Eao[:n_owned], rtol=2e-5, atol=2e-5)
    assert np.all(Ea.cpu().numpy()[n_owned:] == 0)
    # and the full evaluation still works on the same handle afterwards
    g.energy_forces(p, s, cell, E, F)
    Eo2, Fo2, _ = o.energy_forces(pos, sp, cell, O.neighbors_bruteforce(pos, cell, 4.0))
    assert abs(float(E.item()) - Eo2) <= 1e-5 * abs(Eo2) and np.abs(F.cpu().numpy() - Fo2).max() <= 1e-4 * math.sqrt((Fo2 ** 2).mean())


@pytest.mark.parametrize("world", [2, 4, 8])
def test_decomposed_sum_equals_single_domain(lib, world):
    import torch
    from paper_2502_06073_b200.distributed import DistributedAllegro
    w = WL.get(1)                                                         # 4,096 atoms, box 39.6 >= 2 bricks + halos
    wts = lib.build_weights(w.hp, w.weight_seed)
    pos = w.pos + np.array([50.0, -30.0, 7.0])                            # unwrapped
    p, s = _dev(pos), _dev(w.species.astype(np.int32))
    N = w.n_atoms
    Fsum = torch.zeros((N, 3), dtype=torch.float64, device="cuda"); Esum = 0.0
    owned_total = 0
    for rank in range(world):
        d = DistributedAllegro(wts, w.hp, w.cell, rank=rank, world=world)
        Fr = torch.empty((N, 3), dtype=torch.float64, device="cuda")
        Er = d.local_energy_forces(p, s, Fr)
        Fsum += Fr; Esum += float(Er.item()); owned_total += d.n_owned
        assert d.n_owned < N and d.n_local > d.n_owned
        del d
    assert owned_total == N
    g = lib.Allegro(wts, w.hp)
    E1, F1 = g.compute(pos, w.species, w.cell, skin=0.0)
    rms = math.sqrt((F1 ** 2).mean())
    assert abs(Esum - E1) <= 2e-6 * abs(E1)
    assert np.abs(Fsum.cpu().numpy() - F1).max() <= 2e-5 * rms              # same kernels, different edge order inside the rows
    o = O.AllegroOracle(w.hp, wts)
    Eo, Fo, _ = o.energy_forces(w.pos, w.species, w.cell, O.neighbors_binned(w.pos, w.cell, w.hp["r_cut"]))
    assert abs(Esum - Eo) <= 1e-5 * abs(Eo) and np.abs(Fsum.cpu().numpy() - Fo).max() <= 1e-4 * math.sqrt((Fo ** 2).mean())


def test_distributed_md_world1_matches_library_md(lib):
    """The replicated-state integrator (allegro_kick_drift around DistributedAllegro.energy_forces) against allegro_md_step."""
    import torch
    from paper_2502_06073_b200.distributed import DistributedAllegro
    w = WL.config0()
    wts = lib.build_weights(w.hp, w.weight_seed)
    vel = WL.maxwell_boltzmann(w.mass, w.temperature, w.vel_seed)
    d = DistributedAllegro(wts, w.hp, w.cell, rank=0, world=1)
    p, v, mss, s = _dev(w.pos), _dev(vel), _dev(w.mass.astype(np.float64)), _dev(w.species.astype(np.int32))
    F = torch.zeros((w.n_atoms, 3), dtype=torch.float64, device="cuda")
    d.energy_forces(p, s, F)
    d.md_step(p, v, mss, s, F, w.dt_fs, 10)
    g = lib.Allegro(wts, w.hp)
    g.md_init(_dev(w.pos), _dev(vel), mss, s, w.cell, w.hp["r_cut"], 0.0)
    g.md_step(w.dt_fs, 10)
    q = torch.empty((w.n_atoms, 3), dtype=torch.float64, device="cuda")
    g.get_state(pos=q)
    # world = 1: no decomposed dimension, the local set is the system itself in the same order -> same arithmetic
    assert np.abs(p.cpu().numpy() - q.cpu().numpy()).max() <= 1e-9
