"""Pins for the oracle's network, gradient, neighbour search and integrator.

Invariants the model fixes (north_star): forces = central finite differences of E (h=1e-5 A, rel
<= 1e-6); E invariant under rotation / inversion / translation / same-species permutation to 1e-12;
forces covariant; net force zero to 1e-10; neighbour set = brute-force search.  Plus: strict
locality, supercell replication, skin invariance, continuity across r_c, the
pair-potential special case (c_new = 0) checked by 1-D differentiation, and the plan's path counts.
"""
import json
import math
import os

import numpy as np
import pytest

from oracle import allegro_oracle as O
from paper_2502_06073_b200 import workloads as WL

GOLD = os.path.join(os.path.dirname(__file__), "golden")
NETS = {  # (lmax, NL): small widths so every pin runs in well under a second
    "l1": dict(lmax=1, NL=1), "l2": dict(lmax=2, NL=2), "l3": dict(lmax=3, NL=3)}


def make_model(lmax, NL, n=4, S=2, rc=4.0, seed=5, navg=10.0, full_o3=1, c_new=None):
    hp = WL.hparams(S, lmax, NL, n, [16, 12], [16, 12], [8], rc, navg, full_o3=full_o3)
    lay = O.weight_layout(hp)
    w = WL.make_weights(lay, hp, seed)
    if c_new is not None:                                   # overwrite every c_new in the blob
        off = 0
        for kind, r, c in lay:
            if kind == WL.WK_RESIDUAL:
                w[off + 1] = c_new
            off += r * c
    return O.AllegroOracle(hp, w), hp


def ef(model, pos, sp, cell, radius=None):
    radius = model.hp["r_cut"] if radius is None else radius
    return model.energy_forces(pos, sp, cell, O.neighbors_bruteforce(pos, cell, radius))


# ---------------------------------------------------------------- plan
def test_plan_path_counts_golden():
    g = json.load(open(os.path.join(GOLD, "plan_paths.json")))
    for row in g["rows"]:
        hp = WL.hparams(2, row["lmax"], row["n_layers"], 4, [8], [8], [4], 4.0, 10.0)
        plan = O.build_plan(hp)
        assert [len(p) for p in plan.paths] == row["n_paths"]
        nnz = [sum(np.count_nonzero(O.coupling_tensor(a[0], l2, c[0])) for a, l2, c in pl) for pl in plan.paths]
        assert nnz == row["cg_nnz"]
        for L, outs in enumerate(row["outputs"]):
            got = {}
            for a, l2, c in plan.paths[L]:
                key = "%d%s" % (c[0], "e" if c[1] == 1 else "o")
                got[key] = got.get(key, 0) + 1
            assert got == outs


def test_plan_full_o3_differs_only_from_three_layers():
    for lmax, NL in [(2, 2), (3, 2)]:
        a = O.build_plan(WL.hparams(2, lmax, NL, 4, [8], [8], [4], 4.0, 10.0, full_o3=1))
        b = O.build_plan(WL.hparams(2, lmax, NL, 4, [8], [8], [4], 4.0, 10.0, full_o3=0))
        assert a.paths == b.paths
    a = O.build_plan(WL.hparams(2, 3, 3, 4, [8], [8], [4], 4.0, 10.0, full_o3=1))
    b = O.build_plan(WL.hparams(2, 3, 3, 4, [8], [8], [4], 4.0, 10.0, full_o3=0))
    assert len(a.paths[0]) > len(b.paths[0])


def test_table1_parameter_counts_weakly():
    """PAPER.md Table 1 (:97-104): 44.4 K / 690 K / 2.6 M parameters.  The reading of the MLP shapes
    (A5, A6) must land within 20 % (the table cannot discriminate sub-variants)."""
    for n, lat, tb, ed, ref in [(16, [64] * 3, [16, 32, 64], [64], 44.4e3),
                                (64, [256] * 3, [64, 128, 256], [128], 690e3),
                                (128, [512] * 3, [128, 256, 512], [128], 2.6e6)]:
        hp = WL.hparams(89, 2, 2, n, tb, lat, ed, 5.2, 40.0)
        cnt = sum(r * c for k, r, c in O.weight_layout(hp) if k == WL.WK_MATRIX)
        assert abs(cnt - ref) / ref < 0.20, (cnt, ref)


# ---------------------------------------------------------------- invariances
@pytest.mark.parametrize("net", list(NETS))
def test_energy_invariances_and_force_covariance(net):
    from scipy.spatial.transform import Rotation
    model, hp = make_model(**NETS[net])
    pos, sp, cell = WL.cluster(8, 2, seed=21)
    E, F, _ = ef(model, pos, sp, cell)
    c = cell[0, 0] / 2
    R = Rotation.random(random_state=3).as_matrix()
    E2, F2, _ = ef(model, (pos - c) @ R.T + c, sp, cell)
    assert abs(E2 - E) <= 1e-12 * abs(E)
    np.testing.assert_allclose(F2, F @ R.T, atol=1e-12 * np.abs(F).max() + 1e-13)
    E3, F3, _ = ef(model, -(pos - c) + c, sp, cell)                     # inversion (full O(3))
    assert abs(E3 - E) <= 1e-12 * abs(E)
    np.testing.assert_allclose(F3, -F, atol=1e-12)
    M = np.diag([1.0, -1.0, 1.0])                                       # a mirror
    E4, F4, _ = ef(model, (pos - c) @ M + c, sp, cell)
    assert abs(E4 - E) <= 1e-12 * abs(E)
    np.testing.assert_allclose(F4, F @ M, atol=1e-12)
    E5, F5, _ = ef(model, pos + np.array([1.7, -0.3, 9.1]), sp, cell)   # translation (crosses the box)
    assert abs(E5 - E) <= 1e-12 * abs(E)
    np.testing.assert_allclose(F5, F, atol=1e-11)
    perm = np.random.default_rng(0).permutation(pos.shape[0])
    E6, F6, _ = ef(model, pos[perm], sp[perm], cell)
    assert abs(E6 - E) <= 1e-12 * abs(E)
    np.testing.assert_allclose(F6, F[perm], atol=1e-12)


@pytest.mark.parametrize("net", list(NETS))
def test_forces_match_finite_differences(net):
    model, hp = make_model(**NETS[net])
    pos, sp, cell = WL.small_periodic(3, 2.3, 0.35, 2, seed=12)        # 27 atoms, box 6.9 > r_c
    E, F, _ = ef(model, pos, sp, cell)
    rms = math.sqrt((F ** 2).mean())
    h = 1e-5
    rng = np.random.default_rng(1)
    for a, k in zip(rng.integers(0, pos.shape[0], 8), rng.integers(0, 3, 8)):
        pp = pos.copy(); pp[a, k] += h
        pm = pos.copy(); pm[a, k] -= h
        fd = -(model.energy(pp, sp, cell) - model.energy(pm, sp, cell)) / (2 * h)
        assert abs(fd - F[a, k]) <= 1e-6 * rms
    assert np.abs(F.sum(0)).max() <= 1e-10                             # net force
    # zero net torque for a non-periodic cluster
    pos, sp, cell = WL.cluster(8, 2, seed=22)
    E, F, _ = ef(model, pos, sp, cell)
    assert np.abs(np.cross(pos - pos.mean(0), F).sum(0)).max() <= 1e-10


def test_supercell_replication():
    model, hp = make_model(2, 2)
    pos, sp, cell = WL.small_periodic(3, 2.3, 0.35, 2, seed=13)
    E, F, _ = ef(model, pos, sp, cell)
    L = cell[0, 0]
    offs = np.array([(a, b, c) for a in (0, 1) for b in (0, 1) for c in (0, 1)], dtype=np.float64) * L
    pos8 = (pos[None] + offs[:, None]).reshape(-1, 3)
    E8, F8, _ = ef(model, pos8, np.tile(sp, 8), 2 * cell)
    assert abs(E8 - 8 * E) <= 1e-11 * abs(E8)
    np.testing.assert_allclose(F8, np.tile(F, (8, 1)), atol=1e-11)


def test_strict_locality_and_skin_invariance():
    model, hp = make_model(2, 2)
    pos, sp, cell = WL.cluster(9, 2, seed=23, spread=3.0)
    E, F, Ea = ef(model, pos, sp, cell)
    # atom k farther than r_c from atom 0 (under PBC, box is 40 A): moving it leaves E_0 bit-identical
    d = np.linalg.norm(pos - pos[0], axis=1)
    far = [k for k in range(1, 9) if d[k] > hp["r_cut"] + 0.6]
    assert far, "fixture must contain an atom beyond r_c of atom 0"
    p2 = pos.copy(); p2[far[0]] += np.array([0.2, -0.1, 0.15])
    assert np.linalg.norm(p2[far[0]] - p2[0]) > hp["r_cut"]
    _, _, Ea2 = ef(model, p2, sp, cell)
    assert Ea2[0] == Ea[0]
    # a list built with a skin gives identical E, F (inactive edges contribute exactly zero, A11)
    pos, sp, cell = WL.small_periodic(3, 2.3, 0.35, 2, seed=12)
    E0, F0, _ = ef(model, pos, sp, cell)
    E1, F1, _ = ef(model, pos, sp, cell, radius=hp["r_cut"] + 0.7)
    assert E1 == E0 and np.array_equal(F0, F1)


def test_energy_continuous_across_cutoff():
    """A pair crossing r_c changes E by O(delta^3) (u, u', u'' vanish at r_c)."""
    model, hp = make_model(2, 2)
    rc = hp["r_cut"]
    cell = np.diag([30.0, 30.0, 30.0])
    sp = np.array([0, 1, 0], np.int32)
    base = np.array([[10.0, 10.0, 10.0], [8.2, 10.4, 9.7], [10.0 + rc, 10.0, 10.0]])
    def E(delta):
        p = base.copy(); p[2, 0] += delta
        return model.energy(p, sp, cell)
    e_out = E(+1e-3)
    d1, d2 = abs(E(-1e-3) - e_out), abs(E(-2e-3) - e_out)
    assert d1 < 1e-6 and d2 < 1e-5
    assert 4.0 < d2 / d1 < 16.0                                        # ~ delta^3 scaling (8x)


def test_pair_potential_special_case():
    """c_new = 0 in every layer => E = sum_e sigma eps(x0_e): a pure pair potential phi_{ZiZj}(r).
    Check (a) E of a configuration = sum over ordered pairs of the dimer curve, and (b) forces =
    -sum phi'(r) rhat with phi' from 1-D numerical differentiation of the dimer energy alone."""
    model, hp = make_model(2, 2, c_new=0.0)
    cell = np.diag([40.0] * 3)
    mu = model.W["mu"]

    def phi(zi, zj, r):
        """sigma_zi * eps for the ordered edge i->j, from a dimer: E_dimer - mu terms, centre i only."""
        p = np.array([[20.0, 20.0, 20.0], [20.0 + r, 20.0, 20.0]])
        sp = np.array([zi, zj], np.int32)
        _, _, Ea = ef(model, p, sp, cell)
        return Ea[0] - mu[zi]

    pos, sp, _ = WL.cluster(6, 2, seed=24, spread=2.0)
    E, F, _ = ef(model, pos, sp, cell)
    Eref = mu[sp].sum()
    Fref = np.zeros_like(F)
    h = 1e-5
    for i in range(6):
        for j in range(6):
            if i == j:
                continue
            rv = pos[j] - pos[i]; r = np.linalg.norm(rv)
            if r >= hp["r_cut"]:
                continue
            Eref += phi(sp[i], sp[j], r)
            dphi = (phi(sp[i], sp[j], r + h) - phi(sp[i], sp[j], r - h)) / (2 * h)
            Fref[i] += dphi * rv / r                                    # -d/dr_i phi(|r_j-r_i|)
            Fref[j] -= dphi * rv / r
    assert abs(E - Eref) <= 1e-12 * abs(E)
    np.testing.assert_allclose(F, Fref, atol=1e-6 * math.sqrt((F ** 2).mean()) + 1e-9)


# ---------------------------------------------------------------- neighbours
def test_neighbors_bruteforce_vs_naive_python_loops():
    """Brute force on a tiny box against literal triple loops over (i, j, all images in +-2)."""
    rng = np.random.default_rng(3)
    L = np.array([5.0, 6.0, 7.0]); cell = np.diag(L)
    pos = rng.uniform(-3, 9, (9, 3))                                   # unwrapped, outside the box too
    R = 4.5
    rp, col, sh = O.neighbors_bruteforce(pos, cell, R)
    got = {(i, int(col[e]), *map(int, sh[e])) for i in range(9) for e in range(rp[i], rp[i + 1])}
    want = set()
    for i in range(9):
        for j in range(9):
            base = -np.round((pos[j] - pos[i]) / L).astype(int)
            for a in range(-2, 3):
                for b in range(-2, 3):
                    for c in range(-2, 3):
                        s = base + np.array([a, b, c])
                        if i == j and not s.any():
                            continue
                        d = (pos[j] - pos[i]) + s * L
                        if d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < R * R:
                            want.add((i, j, int(s[0]), int(s[1]), int(s[2])))
    assert got == want
    # symmetry: every edge has its reverse
    assert all((j, i, -a, -b, -c) in got for (i, j, a, b, c) in got)


@pytest.mark.parametrize("radius", [4.0, 3.3])
def test_neighbors_binned_equals_bruteforce(radius):
    w = WL.config0()
    pos = w.pos + np.array([13.0, -21.0, 3.0]) * (np.arange(64) % 3 == 0)[:, None]   # some unwrapped atoms
    a = O.neighbors_bruteforce(pos, w.cell, radius)
    b = O.neighbors_binned(pos, w.cell, radius)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    # density estimate: count ~ rho * 4/3 pi R^3
    est = 64 / 8.0 ** 3 * 4 / 3 * math.pi * radius ** 3
    assert abs(a[0][-1] / 64 - est) / est < 0.15


# ---------------------------------------------------------------- integrator
def test_md_reversibility_momentum_and_dt2():
    w = WL.config0()
    lay = O.weight_layout(w.hp)
    model = O.AllegroOracle(w.hp, WL.make_weights(lay, w.hp, w.weight_seed))
    vel = WL.maxwell_boltzmann(w.mass, w.temperature, w.vel_seed)
    assert np.abs((w.mass[:, None] * vel).sum(0)).max() < 1e-12
    fw = O.md_run(model, w.pos, vel, w.mass, w.species, w.cell, w.skin, 0.5, 6)
    bw = O.md_run(model, fw["pos"], -fw["vel"], w.mass, w.species, w.cell, w.skin, 0.5, 6)
    np.testing.assert_allclose(bw["pos"], w.pos, atol=1e-10)
    np.testing.assert_allclose(-bw["vel"], vel, atol=1e-11)
    assert np.abs((w.mass[:, None] * fw["vel"]).sum(0)).max() < 1e-11   # COM momentum conserved
    assert fw["n_rebuilds"] == 6                                       # skin 0 => every step (A22)

    def fluct(dt, n):
        e = O.md_run(model, w.pos, vel, w.mass, w.species, w.cell, w.skin, dt, n)["energies"].sum(1)
        return np.abs(e - e[0]).max()
    f1, f2 = fluct(1.0, 8), fluct(0.5, 16)
    assert 2.5 < f1 / f2 < 6.5                                         # total-energy error ~ dt^2


def test_md_skin_list_equals_rebuild_every_step():
    """With a skin the trajectory is identical to rebuilding every step (inactive edges are exact zeros)."""
    model, hp = make_model(1, 1, rc=3.0)
    pos, sp, cell = WL.small_periodic(3, 2.3, 0.35, 2, seed=14)
    mass = np.where(sp == 0, 28.0, 16.0)
    vel = WL.maxwell_boltzmann(mass, 3000.0, 7)
    a = O.md_run(model, pos, vel, mass, sp, cell, 0.0, 1.0, 12)
    b = O.md_run(model, pos, vel, mass, sp, cell, 0.4, 1.0, 12)
    assert b["n_rebuilds"] < a["n_rebuilds"]
    np.testing.assert_allclose(a["pos"], b["pos"], atol=1e-12)
