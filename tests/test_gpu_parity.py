"""GPU parity: the CUDA path through the C-ABI against the fp64 oracle on the same seeded inputs.

Gates (BASELINE.json north_star): neighbour lists bit-exact after canonical (i, j, shift) sort;
|dE|/|E| <= 1e-5; every force component within 1e-4 x RMS(F) (fp32 GPU vs fp64 oracle)."""
import math

import numpy as np
import pytest

from oracle import allegro_oracle as O
from paper_2502_06073_b200 import workloads as WL

pytestmark = pytest.mark.gpu

E_RTOL = 1e-5
F_TOL_RMS = 1e-4


def _torch():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


def _gpu_list(model, lib, pos, species, cell, cutoff, skin):
    torch = _torch()
    p = torch.from_numpy(np.ascontiguousarray(pos)).cuda()
    s = torch.from_numpy(np.ascontiguousarray(species, dtype=np.int32)).cuda()
    model.build_neighbors(p, s, cell, cutoff, skin)
    rp, col, sh = model.get_neighbors()
    return rp.cpu().numpy(), col.cpu().numpy(), sh.cpu().numpy().astype(np.int32)


def _model(lib, hp, seed):
    w = lib.build_weights(hp, seed)
    return lib.Allegro(w, hp), O.AllegroOracle(hp, w)


def _check_ef(E, F, Eo, Fo, Ea=None, Eao=None):
    rms = math.sqrt((Fo ** 2).mean())
    assert abs(E - Eo) <= E_RTOL * abs(Eo), (E, Eo)
    err = np.abs(F - Fo).max()
    assert err <= F_TOL_RMS * rms, (err, rms, err / rms)
    if Ea is not None:
        np.testing.assert_allclose(Ea, Eao, rtol=2e-5, atol=2e-5)
    return err / rms


# ------------------------------------------------------------------------------------------------ a-1
@pytest.mark.parametrize("case", ["cfg0", "cfg0_skin", "noncubic_unwrapped", "one_cell", "empty"])
def test_neighbor_list_bit_exact_small(lib, case):
    w = WL.config0()
    g, _ = _model(lib, w.hp, 0)
    pos, cell, skin = w.pos, w.cell, 0.0
    if case == "cfg0_skin":
        skin = 0.7
    elif case == "noncubic_unwrapped":
        rng = np.random.default_rng(5)
        cell = np.diag([9.0, 13.0, 17.5])
        pos = rng.uniform(-20, 40, (150, 3))
        skin = 0.5
    elif case == "one_cell":
        cell = np.diag([4.5, 5.0, 6.0])                       # r_c+skin = 4.4: one cell per axis, many self images
        pos = np.random.default_rng(6).uniform(0, 4.5, (11, 3))
        skin = 0.4
    elif case == "empty":
        pos = np.zeros((0, 3))
    species = np.zeros(pos.shape[0], np.int32)
    rp, col, sh = _gpu_list(g, lib, pos, species, cell, w.hp["r_cut"], skin)
    rpo, colo, sho = O.neighbors_bruteforce(pos, cell, w.hp["r_cut"] + skin) if pos.shape[0] else (np.zeros(1, np.int64), np.zeros(0, np.int32), np.zeros((0, 3), np.int32))
    assert np.array_equal(rp, rpo) and np.array_equal(col, colo) and np.array_equal(sh, sho)


def test_neighbor_list_bit_exact_cfg1(lib):
    w = WL.config1()
    g, _ = _model(lib, w.hp, w.weight_seed)
    rp, col, sh = _gpu_list(g, lib, w.pos, w.species, w.cell, w.hp["r_cut"], w.skin)
    rpo, colo, sho = O.neighbors_binned(w.pos, w.cell, w.hp["r_cut"] + w.skin)
    assert np.array_equal(rp, rpo) and np.array_equal(col, colo) and np.array_equal(sh, sho)
    assert rp[-1] > 150_000


def test_errors(lib):
    torch = _torch()
    w = WL.config0()
    g, _ = _model(lib, w.hp, 0)
    p = torch.from_numpy(w.pos).cuda(); s = torch.from_numpy(w.species).cuda()
    E = torch.zeros(1, dtype=torch.float64, device="cuda"); F = torch.zeros((64, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(lib.AllegroError) as ei:
        g.energy_forces(p, s, w.cell, E, F)
    assert ei.value.code == -8                                 # no list yet
    with pytest.raises(lib.AllegroError) as ei:
        g.build_neighbors(p, s, np.diag([3.0, 8.0, 8.0]), 4.0, 0.0)
    assert ei.value.code == -6                                 # r_c + skin > box (A17)
    with pytest.raises(lib.AllegroError) as ei:
        g.build_neighbors(p, s, np.array([[8.0, 0, 0], [7.5, 3.9, 0], [0, 0, 8.0]]), 4.0, 0.0)
    assert ei.value.code == -6                                 # triclinic: r_c + skin > a perpendicular width
    with pytest.raises(lib.AllegroError) as ei:
        g.build_neighbors(p, s, -w.cell, 4.0, 0.0)
    assert ei.value.code == -1                                 # left-handed cell
    g.build_neighbors(p, s, w.cell, 4.0, 0.3)
    p2 = p.clone(); p2[5, 0] += 0.2
    with pytest.raises(lib.AllegroError) as ei:
        g.energy_forces(p2, s, w.cell, E, F)
    assert ei.value.code == -4                                 # stale list
    s2 = s.clone(); s2[3] = 7
    with pytest.raises(lib.AllegroError) as ei:
        g.energy_forces(p, s2, w.cell, E, F)
    assert ei.value.code == -7
    g.energy_forces(p, s, w.cell, E, F)                        # and it recovers


# ------------------------------------------------------------------------------------------------ a-2..a-5
def test_energy_forces_cfg0(lib):
    w = WL.config0()
    g, o = _model(lib, w.hp, w.weight_seed)
    E, F, Ea = g.compute(w.pos, w.species, w.cell, skin=w.skin, want_atom=True)
    Eo, Fo, Eao = o.energy_forces(w.pos, w.species, w.cell, O.neighbors_bruteforce(w.pos, w.cell, w.hp["r_cut"]))
    _check_ef(E, F, Eo, Fo, Ea, Eao)
    assert g.get_stats()["active_edges"] == int(O.neighbors_bruteforce(w.pos, w.cell, w.hp["r_cut"])[0][-1])


@pytest.mark.parametrize("net", [(1, 1, 8), (2, 2, 8), (3, 3, 8), (3, 2, 4), (2, 3, 12), (3, 3, 16), (2, 2, 64), (3, 3, 64),
                                 (2, 2, 128)])
@pytest.mark.parametrize("full_o3", [1, 0])
def test_energy_forces_small_nets(lib, net, full_o3):
    """All (lmax, NL) plans incl. the unnatural-parity irreps of 3-layer full O(3); ragged widths; skin list."""
    lmax, NL, n = net
    hp = WL.hparams(3, lmax, NL, n, [24, 20, 28], [36, 28], [12, 8], 4.0, 18.0, n_bessel=6, full_o3=full_o3)
    g, o = _model(lib, hp, 40 + lmax)
    pos, sp, cell = WL.small_periodic(4, 2.2, 0.4, 3, seed=31)       # 64 atoms, box 8.8
    E, F, Ea = g.compute(pos, sp, cell, skin=0.4, want_atom=True)
    Eo, Fo, Eao = o.energy_forces(pos, sp, cell, O.neighbors_bruteforce(pos, cell, 4.0))
    _check_ef(E, F, Eo, Fo, Ea, Eao)


def test_energy_forces_cfg1(lib):
    w = WL.config1()
    g, o = _model(lib, w.hp, w.weight_seed)
    E, F, Ea = g.compute(w.pos, w.species, w.cell, skin=w.skin, want_atom=True)
    Eo, Fo, Eao = o.energy_forces(w.pos, w.species, w.cell, O.neighbors_binned(w.pos, w.cell, w.hp["r_cut"]))
    rel = _check_ef(E, F, Eo, Fo, Ea, Eao)
    st = g.get_stats()
    assert st["active_edges"] == int(O.neighbors_binned(w.pos, w.cell, w.hp["r_cut"])[0][-1])
    print("cfg1 max|dF|/rms =", rel, "dE/E =", abs(E - Eo) / abs(Eo), st)


def test_isolated_atom_and_dimer(lib):
    """Degenerate rows: an atom with no neighbour has E_i = mu; a dimer's forces are equal and opposite."""
    hp = WL.hparams(2, 2, 2, 8, [16, 16], [16, 16], [8], 4.0, 10.0)
    g, o = _model(lib, hp, 9)
    cell = np.diag([30.0, 30.0, 30.0])
    pos = np.array([[5.0, 5.0, 5.0], [7.1, 5.5, 4.6], [20.0, 20.0, 20.0]])
    sp = np.array([0, 1, 1], np.int32)
    E, F, Ea = g.compute(pos, sp, cell, skin=0.5, want_atom=True)
    Eo, Fo, Eao = o.energy_forces(pos, sp, cell, O.neighbors_bruteforce(pos, cell, 4.0))
    _check_ef(E, F, Eo, Fo, Ea, Eao)
    assert abs(Ea[2] - o.W["mu"][1]) < 1e-6 and np.all(F[2] == 0)
    np.testing.assert_allclose(F[0], -F[1], atol=1e-7)


# ------------------------------------------------------------------------------------------------ a-6
def _md_gpu(lib, g, w, vel, n_steps, dt=None, skin=None):
    torch = _torch()
    dev = lambda a, dt=None: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    skin = w.skin if skin is None else skin
    g.md_init(dev(w.pos), dev(vel), dev(w.mass.astype(np.float64)), dev(w.species.astype(np.int32)), w.cell, w.hp["r_cut"], skin)
    g.md_step(w.dt_fs if dt is None else dt, n_steps)
    N = w.pos.shape[0]
    pos = torch.empty((N, 3), dtype=torch.float64, device="cuda"); v = torch.empty_like(pos); F = torch.empty_like(pos)
    Ep = torch.empty(1, dtype=torch.float64, device="cuda"); Ek = torch.empty_like(Ep)
    nreb = g.get_state(pos, v, F, Ep, Ek)
    return pos.cpu().numpy(), v.cpu().numpy(), F.cpu().numpy(), float(Ep.item()), float(Ek.item()), nreb


def test_md_cfg0_stepwise_parity(lib):
    w = WL.config0()
    g, o = _model(lib, w.hp, w.weight_seed)
    vel = WL.maxwell_boltzmann(w.mass, w.temperature, w.vel_seed)
    pos, v, F, Ep, Ek, nreb = _md_gpu(lib, g, w, vel, w.n_steps)
    ref = O.md_run(o, w.pos, vel, w.mass, w.species, w.cell, w.skin, w.dt_fs, w.n_steps)
    assert np.abs(pos - ref["pos"]).max() <= 1e-4
    assert np.abs(v - ref["vel"]).max() <= 1e-5
    assert abs(Ep - ref["E_pot"]) <= E_RTOL * abs(ref["E_pot"])
    assert abs(Ek - ref["E_kin"]) <= 1e-5 * abs(ref["E_kin"])
    assert nreb == ref["n_rebuilds"] == w.n_steps


def test_md_skin_rebuilds_match_oracle(lib):
    """Hot small system so that the skin test fires a few times; rebuild count and trajectory match."""
    hp = WL.hparams(2, 2, 2, 8, [16, 16], [16, 16], [8], 3.5, 14.0)
    g, o = _model(lib, hp, 3)
    pos, sp, cell = WL.small_periodic(4, 2.2, 0.3, 2, seed=33)
    mass = np.where(sp == 0, 28.0, 16.0)
    vel = WL.maxwell_boltzmann(mass, 4000.0, 5)
    w = WL.Workload("hot", pos, sp, mass, cell, hp, skin=0.3, dt_fs=1.0, n_steps=25)
    p, v, F, Ep, Ek, nreb = _md_gpu(lib, g, w, vel, 25)
    ref = O.md_run(o, pos, vel, mass, sp, cell, 0.3, 1.0, 25)
    assert 0 < ref["n_rebuilds"] < 25 and nreb == ref["n_rebuilds"]
    assert np.abs(p - ref["pos"]).max() <= 1e-4
    # list after MD equals the oracle's list at the last rebuild positions? -> at least symmetric & consistent E
    assert abs(Ep - ref["E_pot"]) <= E_RTOL * abs(ref["E_pot"])


# ------------------------------------------------------------------------------------------------ fused forward layer (tp_mix.cu)
@pytest.mark.parametrize("net", [(2, 2, 64, [40, 32]), (3, 3, 64, [36, 28])])
def test_fused_tensor_product_and_mixing_equals_the_unfused_path(lib, net):
    """n = 64: k_tpmix_fwd (T on chip) against k_tpo_fwd + per-irrep GEMMs (T in HBM), and both against the oracle."""
    lmax, NL, n, lat = net
    hp = WL.hparams(3, lmax, NL, n, [24, lat[-1]], lat, [12], 4.0, 18.0, n_bessel=6)
    g, o = _model(lib, hp, 77)
    pos, sp, cell = WL.small_periodic(5, 2.2, 0.4, 3, seed=31)         # 125 atoms: several 16-edge tiles and a ragged one
    Eo, Fo, Eao = o.energy_forces(pos, sp, cell, O.neighbors_bruteforce(pos, cell, 4.0))
    out = {}
    for fused in (True, False):
        g.debug_set_fusion(fused)
        E, F, Ea = g.compute(pos, sp, cell, skin=0.3, want_atom=True)
        _check_ef(E, F, Eo, Fo, Ea, Eao)
        out[fused] = (E, F, Ea)
    rms = math.sqrt((Fo ** 2).mean())
    assert abs(out[True][0] - out[False][0]) <= 2e-7 * abs(Eo)
    assert np.abs(out[True][1] - out[False][1]).max() <= 5e-6 * rms
