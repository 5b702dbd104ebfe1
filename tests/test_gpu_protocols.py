"""GPU parity for the SURVEY.md 8f-1 rows: virial / stress, Berendsen NVT with a temperature ramp (reading A25), affine
deformation (A26), checkpoint / resume (allegro_set_state) and the list-capacity recovery path of allegro_md_step."""
import math

import numpy as np
import pytest

from oracle import allegro_oracle as O
from paper_2502_06073_b200 import workloads as WL

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _state(g, N):
    import torch
    pos = torch.empty((N, 3), dtype=torch.float64, device="cuda"); vel = torch.empty_like(pos); F = torch.empty_like(pos)
    Ep = torch.empty(1, dtype=torch.float64, device="cuda"); Ek = torch.empty_like(Ep)
    nreb = g.get_state(pos, vel, F, Ep, Ek)
    return pos.cpu().numpy(), vel.cpu().numpy(), F.cpu().numpy(), float(Ep.item()), float(Ek.item()), nreb


def _pair(lib, hp, seed):
    w = lib.build_weights(hp, seed)
    return lib.Allegro(w, hp), O.AllegroOracle(hp, w)


@pytest.mark.parametrize("net", [(1, 1, 8, [32, 32]), (2, 2, 16, [48, 32]), (3, 3, 64, [36, 28])])
def test_virial_matches_oracle(lib, net):
    import torch
    lmax, NL, n, lat = net
    hp = WL.hparams(3, lmax, NL, n, [24, lat[-1]], lat, [12], 4.0, 18.0, n_bessel=6)
    g, o = _pair(lib, hp, 50 + lmax)
    pos, sp, cell = WL.small_periodic(4, 2.2, 0.4, 3, seed=41)
    E, F = g.compute(pos, sp, cell, skin=0.4)
    W = g.virial(_dev(pos))
    Eo, Fo, _, Wo = o.energy_forces(pos, sp, cell, O.neighbors_bruteforce(pos, cell, 4.0), virial=True)
    # the per-edge gradients are fp32: same gate as the forces, 1e-4 of the RMS per-edge-summed scale
    scale = math.sqrt((Fo ** 2).mean()) * math.sqrt(pos.shape[0]) * 4.0
    assert np.abs(W - Wo).max() <= 1e-4 * scale, (np.abs(W - Wo).max(), scale)
    assert np.abs(W - Wo).max() <= 2e-5 * np.abs(Wo).max()
    np.testing.assert_allclose(W, W.T, atol=2e-5 * np.abs(Wo).max())


def test_nvt_ramp_cfg0_stepwise_parity(lib):
    w = WL.config0()
    g, o = _pair(lib, w.hp, w.weight_seed)
    vel = WL.maxwell_boltzmann(w.mass, w.temperature, w.vel_seed)
    g.md_init(_dev(w.pos), _dev(vel), _dev(w.mass.astype(np.float64)), _dev(w.species.astype(np.int32)), w.cell, w.hp["r_cut"], 0.3)
    th = dict(T0=300.0, T1=600.0, n_ramp=8, tau=5.0)
    g.md_step_nvt(w.dt_fs, 12, th["T0"], th["T1"], th["n_ramp"], th["tau"])
    pos, v, F, Ep, Ek, nreb = _state(g, w.n_atoms)
    ref = O.md_run(o, w.pos, vel, w.mass, w.species, w.cell, 0.3, w.dt_fs, 12, thermostat=th)
    assert np.abs(pos - ref["pos"]).max() <= 1e-4
    assert np.abs(v - ref["vel"]).max() <= 1e-5
    assert abs(Ek - ref["E_kin"]) <= 1e-5 * abs(ref["E_kin"])
    assert nreb == ref["n_rebuilds"]
    # the thermostat did something: NVE from the same start ends colder
    nve = O.md_run(o, w.pos, vel, w.mass, w.species, w.cell, 0.3, w.dt_fs, 12)
    assert ref["E_kin"] > 1.05 * nve["E_kin"]


def test_deform_then_md_matches_oracle(lib):
    hp = WL.hparams(2, 2, 2, 8, [16, 16], [16, 16], [8], 3.5, 14.0)
    g, o = _pair(lib, hp, 3)
    pos, sp, cell = WL.small_periodic(4, 2.2, 0.3, 2, seed=43)
    mass = np.where(sp == 0, 28.0, 16.0)
    vel = WL.maxwell_boltzmann(mass, 300.0, 5)
    g.md_init(_dev(pos), _dev(vel), _dev(mass), _dev(sp.astype(np.int32)), cell, 3.5, 0.3)
    g.md_step(0.5, 4)
    cell2 = np.diag(np.diag(cell) * np.array([1.0, 1.0, 1.02]))       # 2 % tensile strain along z
    g.md_deform(cell2)
    p1, v1, F1, Ep1, _, _ = _state(g, pos.shape[0])
    W = g.virial()
    ref = O.md_run(o, pos, vel, mass, sp, cell, 0.3, 0.5, 4)
    p_ref, c_ref = O.md_deform(ref["pos"], cell, cell2)
    assert np.abs(p1 - p_ref).max() <= 1e-4
    Eo, Fo, _, Wo = o.energy_forces(p1, sp, cell2, O.neighbors_bruteforce(p1, cell2, 3.5), virial=True)   # oracle on the GPU's snapshot
    rms = math.sqrt((Fo ** 2).mean())
    assert abs(Ep1 - Eo) <= 1e-5 * abs(Eo) and np.abs(F1 - Fo).max() <= 1e-4 * rms
    assert np.abs(W - Wo).max() <= 5e-5 * np.abs(Wo).max()
    g.md_step(0.5, 4)                                                   # and the integrator carries on in the new cell
    p2, _, _, Ep2, _, _ = _state(g, pos.shape[0])
    ref2 = O.md_run(o, p1, v1, mass, sp, cell2, 0.3, 0.5, 4)
    assert np.abs(p2 - ref2["pos"]).max() <= 1e-4 and abs(Ep2 - ref2["E_pot"]) <= 1e-5 * abs(ref2["E_pot"])


def test_set_state_resumes_identically(lib):
    w = WL.config0()
    g, _ = _pair(lib, w.hp, w.weight_seed)
    vel = WL.maxwell_boltzmann(w.mass, w.temperature, w.vel_seed)
    args = (_dev(w.mass.astype(np.float64)), _dev(w.species.astype(np.int32)), w.cell, w.hp["r_cut"], 0.0)
    g.md_init(_dev(w.pos), _dev(vel), *args)
    g.md_step(w.dt_fs, 5)
    p5, v5, _, _, _, _ = _state(g, w.n_atoms)
    g.md_step(w.dt_fs, 5)
    p10, v10, _, E10, _, _ = _state(g, w.n_atoms)
    g.set_state(_dev(p5), _dev(v5))                                    # resume from the checkpoint (skin 0: list rebuilt every step anyway)
    g.md_step(w.dt_fs, 5)
    q10, u10, _, E10b, _, _ = _state(g, w.n_atoms)
    assert np.array_equal(q10, p10) and np.array_equal(u10, v10) and E10b == E10


def test_list_capacity_recovery_keeps_the_trajectory(lib):
    """A contracting open cluster: the list grows at every device-side rebuild, so with zero slack the first rebuild overflows
    it; the call must still return the trajectory of a roomy list (and say that it recovered)."""
    hp = WL.hparams(2, 2, 2, 8, [16, 16], [16, 16], [8], 3.5, 14.0)
    pos, sp, _ = WL.small_periodic(4, 2.2, 0.3, 2, seed=33)
    cell = np.diag([30.0, 30.0, 30.0])
    pos = pos + 10.0
    mass = np.where(sp == 0, 28.0, 16.0)
    vel = -0.004 * (pos - pos.mean(0))                                  # homogeneous contraction, ~15 % over the run
    out = []
    for slack in [(0.125, 4096), (0.0, 0)]:
        g, _ = _pair(lib, hp, 3)
        g.debug_set_list_slack(*slack)
        g.md_init(_dev(pos), _dev(vel), _dev(mass), _dev(sp.astype(np.int32)), cell, 3.5, 0.3)
        g.md_step(1.0, 40)
        st = g.get_stats()
        out.append(_state(g, pos.shape[0]) + (st["recoveries"], st["force_evals"]))
    roomy, tight = out
    assert roomy[6] == 0 and tight[6] >= 1, (roomy[6], tight[6])
    assert tight[7] == 40
    assert np.array_equal(tight[0], roomy[0]) and np.array_equal(tight[1], roomy[1])
    assert tight[5] == roomy[5]                                         # same number of rebuilds
