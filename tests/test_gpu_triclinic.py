"""GPU parity on general (triclinic) cells, SURVEY.md 8f-4 / reading A27: the CUDA path through the C-ABI against the fp64 oracle
(pinned on such cells in tests/test_oracle_triclinic.py).  Same gates as the orthorhombic tests: lists bit-exact, |dE|/|E| <=
1e-5, every force component within 1e-4 x RMS(F)."""
import math

import numpy as np
import pytest

from oracle import allegro_oracle as O
from paper_2502_06073_b200 import workloads as WL

pytestmark = pytest.mark.gpu

TRI = np.array([[9.2, 0.0, 0.0], [2.1, 8.8, 0.0], [-1.3, 1.7, 9.5]])


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _pair(lib, hp, seed):
    w = lib.build_weights(hp, seed)
    return lib.Allegro(w, hp), O.AllegroOracle(hp, w)


def _tri_system(H, n_side, seed, jitter=0.3, n_species=3, unwrap=2):
    rng = np.random.default_rng(seed)
    g = (np.stack(np.meshgrid(*[np.arange(n_side)] * 3, indexing="ij"), -1).reshape(-1, 3) + 0.5) / n_side
    pos = g @ H + rng.uniform(-jitter, jitter, (g.shape[0], 3))
    if unwrap:
        pos += rng.integers(-unwrap, unwrap + 1, (g.shape[0], 3)) @ H
    return pos, rng.integers(0, n_species, g.shape[0]).astype(np.int32)


def _gpu_list(g, pos, sp, H, cutoff, skin):
    g.build_neighbors(_dev(pos), _dev(sp), H, cutoff, skin)
    rp, col, sh = g.get_neighbors()
    return rp.cpu().numpy(), col.cpu().numpy(), sh.cpu().numpy().astype(np.int32)


@pytest.mark.parametrize("case", ["one_bin", "three_bins", "rotated", "random_cloud"])
def test_neighbor_list_bit_exact_triclinic(lib, case):
    w = WL.config0()
    g, _ = _pair(lib, w.hp, 0)
    rc, skin = w.hp["r_cut"], 0.4
    if case == "one_bin":                                       # widths ~8.6: one bin per axis, self images
        H = TRI; pos, sp = _tri_system(H, 4, 3)
    elif case == "three_bins":
        H = np.array([[17.0, 0.0, 0.0], [5.0, 16.0, 0.0], [-3.0, 4.0, 18.5]]); pos, sp = _tri_system(H, 7, 4)
        assert np.floor(O.cell_widths(H) / (rc + skin)).min() >= 3
    elif case == "rotated":                                     # a full 3x3 matrix
        q, r = np.linalg.qr(np.random.default_rng(2).normal(size=(3, 3))); q = q * np.sign(np.diag(r))
        if np.linalg.det(q) < 0: q[:, 0] = -q[:, 0]
        H = np.diag([13.0, 9.5, 15.0]) @ q; pos, sp = _tri_system(H, 6, 5)
    else:
        H = TRI * 1.7; rng = np.random.default_rng(9)
        pos = rng.uniform(-1.5, 2.5, (700, 3)) @ H; sp = np.zeros(700, np.int32)
    rp, col, sh = _gpu_list(g, pos, sp, H, rc, skin)
    rpo, colo, sho = O.neighbors_bruteforce(pos, H, rc + skin)
    assert np.array_equal(rp, rpo) and np.array_equal(col, colo) and np.array_equal(sh, sho)
    assert rp[-1] > 1000


@pytest.mark.parametrize("net", [(1, 1, 8, [32, 32]), (2, 2, 16, [48, 32]), (3, 3, 64, [36, 28])])
def test_energy_forces_virial_triclinic(lib, net):
    import torch
    lmax, NL, n, lat = net
    hp = WL.hparams(3, lmax, NL, n, [24, lat[-1]], lat, [12], 4.0, 18.0, n_bessel=6)
    g, o = _pair(lib, hp, 60 + lmax)
    H = TRI * 0.97
    pos, sp = _tri_system(H, 4, 11, jitter=0.35)
    E, F, Ea = g.compute(pos, sp, H, skin=0.3, want_atom=True)
    W = g.virial(_dev(pos))
    Wn = torch.empty(9, dtype=torch.float64, device="cuda")
    g.virial_noalloc(Wn, _dev(pos)); torch.cuda.synchronize()
    Eo, Fo, Eao, Wo = o.energy_forces(pos, sp, H, O.neighbors_bruteforce(pos, H, 4.0), virial=True)
    rms = math.sqrt((Fo ** 2).mean())
    assert abs(E - Eo) <= 1e-5 * abs(Eo), (E, Eo)
    assert np.abs(F - Fo).max() <= 1e-4 * rms, np.abs(F - Fo).max() / rms
    np.testing.assert_allclose(Ea, Eao, rtol=2e-5, atol=2e-5)
    assert np.abs(W - Wo).max() <= 2e-5 * np.abs(Wo).max()
    assert np.abs(Wn.cpu().numpy().reshape(3, 3) - W).max() <= 1e-12 * np.abs(W).max()


def test_md_deform_md_triclinic_matches_oracle(lib):
    hp = WL.hparams(2, 2, 2, 8, [16, 16], [16, 16], [8], 3.5, 14.0)
    g, o = _pair(lib, hp, 3)
    H = TRI * 0.9
    pos, sp = _tri_system(H, 4, 21, jitter=0.2, n_species=2)
    mass = np.where(sp == 0, 28.0, 16.0)
    vel = WL.maxwell_boltzmann(mass, 600.0, 5)
    g.md_init(_dev(pos), _dev(vel), _dev(mass), _dev(sp.astype(np.int32)), H, 3.5, 0.3)
    g.md_step(0.5, 12)
    N = pos.shape[0]
    p = torch_state(g, N)
    ref = O.md_run(o, pos, vel, mass, sp, H, 0.3, 0.5, 12)
    assert np.abs(p["pos"] - ref["pos"]).max() <= 1e-4 and np.abs(p["vel"] - ref["vel"]).max() <= 1e-5
    assert abs(p["E_pot"] - ref["E_pot"]) <= 1e-5 * abs(ref["E_pot"]) and p["n_rebuilds"] == ref["n_rebuilds"]
    # a shear + tensile increment, then the integrator carries on in the new cell
    H2 = H @ (np.eye(3) + np.array([[0.0, 0.015, 0.0], [0.0, 0.0, 0.0], [0.0, 0.0, 0.02]]))
    g.md_deform(H2)
    p1 = torch_state(g, N)
    p_ref, _ = O.md_deform(p["pos"], H, H2)
    assert np.abs(p1["pos"] - p_ref).max() <= 1e-9
    Eo, Fo, _ = o.energy_forces(p1["pos"], sp, H2, O.neighbors_bruteforce(p1["pos"], H2, 3.5))
    rms = math.sqrt((Fo ** 2).mean())
    assert abs(p1["E_pot"] - Eo) <= 1e-5 * abs(Eo) and np.abs(p1["F"] - Fo).max() <= 1e-4 * rms
    g.md_step(0.5, 6)
    p2 = torch_state(g, N)
    ref2 = O.md_run(o, p1["pos"], p1["vel"], mass, sp, H2, 0.3, 0.5, 6)
    assert np.abs(p2["pos"] - ref2["pos"]).max() <= 1e-4 and abs(p2["E_pot"] - ref2["E_pot"]) <= 1e-5 * abs(ref2["E_pot"])


def torch_state(g, N):
    import torch
    pos = torch.empty((N, 3), dtype=torch.float64, device="cuda"); vel = torch.empty_like(pos); F = torch.empty_like(pos)
    Ep = torch.empty(1, dtype=torch.float64, device="cuda"); Ek = torch.empty_like(Ep)
    nreb = g.get_state(pos, vel, F, Ep, Ek)
    return dict(pos=pos.cpu().numpy(), vel=vel.cpu().numpy(), F=F.cpu().numpy(), E_pot=float(Ep.item()), E_kin=float(Ek.item()), n_rebuilds=nreb)


def test_rotated_cell_gives_the_orthorhombic_energy_on_the_gpu(lib):
    hp = WL.hparams(2, 2, 2, 16, [32, 32], [32, 32], [8], 4.0, 16.0)
    g, _ = _pair(lib, hp, 8)
    pos, sp, cell = WL.small_periodic(4, 2.3, 0.35, 2, seed=17)
    q, r = np.linalg.qr(np.random.default_rng(12).normal(size=(3, 3))); q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0: q[:, 0] = -q[:, 0]
    E0, F0 = g.compute(pos, sp, cell, skin=0.2)
    E1, F1 = g.compute(pos @ q, sp, cell @ q, skin=0.2)
    rms = math.sqrt((F0 ** 2).mean())
    assert abs(E1 - E0) <= 2e-6 * abs(E0)
    assert np.abs(F1 - F0 @ q).max() <= 5e-5 * rms


def test_decomposition_still_needs_an_orthorhombic_cell(lib):
    import torch
    w = WL.config0()
    g, _ = _pair(lib, w.hp, 0)
    pos, sp = _tri_system(TRI * 2, 4, 1)
    lp = torch.empty((4096, 3), dtype=torch.float64, device="cuda"); ls = torch.empty(4096, dtype=torch.int32, device="cuda")
    lsrc = torch.empty(4096, dtype=torch.int64, device="cuda")
    with pytest.raises(lib.AllegroError) as ei:
        g.decomp_select(_dev(pos), _dev(sp), TRI * 2, (2, 1, 1), (0, 0, 0), 4.0, lp, ls, lsrc)
    assert ei.value.code == -2
