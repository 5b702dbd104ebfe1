"""Pins for the oracle on general (triclinic) cells, reading A27: H rows = lattice vectors, image
shift s_1 a_1 + s_2 a_2 + s_3 a_3, cutoff + skin <= smallest perpendicular width.  Every pin ties the general-cell code to
something it does not compute itself: the orthorhombic results (pinned in test_oracle_model.py) through a rigid rotation, the
lattice (not its basis) through a unimodular change of basis, a supercell, a wide explicit image enumeration, finite differences,
and the textbook plane-spacing formula."""
import itertools
import math

import numpy as np
import pytest

from oracle import allegro_oracle as O
from paper_2502_06073_b200 import workloads as WL

TRI = np.array([[9.2, 0.0, 0.0], [2.1, 8.8, 0.0], [-1.3, 1.7, 9.5]])       # a sheared cell, widths ~ 8.7, 8.6, 9.5


def _model(lmax=2, NL=2, n=4, S=2, rc=4.0, seed=5, navg=12.0):
    hp = WL.hparams(S, lmax, NL, n, [16, 12], [16, 12], [8], rc, navg)
    return O.AllegroOracle(hp, WL.make_weights(O.weight_layout(hp), hp, seed)), hp


def _rotation(seed):
    q, r = np.linalg.qr(np.random.default_rng(seed).normal(size=(3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def _tri_system(n_side=4, seed=3, jitter=0.3):
    """atoms on a jittered lattice of fractional sites of TRI, unwrapped by a few images"""
    rng = np.random.default_rng(seed)
    g = (np.stack(np.meshgrid(*[np.arange(n_side)] * 3, indexing="ij"), -1).reshape(-1, 3) + 0.5) / n_side
    pos = g @ TRI + rng.uniform(-jitter, jitter, (g.shape[0], 3))
    pos += rng.integers(-2, 3, (g.shape[0], 3)) @ TRI
    return pos, rng.integers(0, 2, g.shape[0]).astype(np.int32), TRI.copy()


def test_cell_widths_are_the_lattice_plane_spacings():
    H = TRI
    V = abs(np.linalg.det(H))
    ref = np.array([V / np.linalg.norm(np.cross(H[1], H[2])), V / np.linalg.norm(np.cross(H[2], H[0])), V / np.linalg.norm(np.cross(H[0], H[1]))])
    np.testing.assert_allclose(O.cell_widths(H), ref, rtol=1e-13)
    np.testing.assert_array_equal(O.cell_widths(np.diag([3.0, 4.0, 5.0])), [3.0, 4.0, 5.0])
    with pytest.raises(ValueError):
        O.neighbors_bruteforce(np.zeros((1, 3)), H, ref.min() * 1.001)
    with pytest.raises(ValueError):
        O.neighbors_bruteforce(np.zeros((1, 3)), -H, 1.0)                      # left-handed


def test_neighbours_match_a_wide_explicit_image_enumeration():
    pos, sp, H = _tri_system(3, seed=8)
    R = 4.3
    rp, col, sh = O.neighbors_bruteforce(pos, H, R)
    got = set()
    for i in range(pos.shape[0]):
        for k in range(rp[i], rp[i + 1]):
            got.add((i, int(col[k]), *map(int, sh[k])))
    want = set()
    f = pos @ np.linalg.inv(H)
    for i in range(pos.shape[0]):
        for j in range(pos.shape[0]):
            base = -np.round(f[j] - f[i]).astype(int)
            for t in itertools.product(range(-3, 4), repeat=3):                 # far beyond the +-1 the search tries
                s = base + np.array(t)
                d = pos[j] - pos[i] + s[0] * H[0] + s[1] * H[1] + s[2] * H[2]
                if d @ d < R * R and not (i == j and not s.any()):
                    want.add((i, j, *map(int, s)))
    assert got == want and len(got) > 250
    # symmetric list: (i, j, s) <-> (j, i, -s)
    assert all((j, i, -a, -b, -c) in got for (i, j, a, b, c) in got)


def test_binned_equals_bruteforce_triclinic_three_or_more_cells():
    rng = np.random.default_rng(4)
    H = np.array([[17.0, 0.0, 0.0], [5.0, 16.0, 0.0], [-3.0, 4.0, 18.5]])
    radius = 4.4
    assert np.floor(O.cell_widths(H) / radius).min() >= 3
    pos = rng.uniform(-1.5, 2.5, (450, 3)) @ H
    a, b = O.neighbors_binned(pos, H, radius), O.neighbors_bruteforce(pos, H, radius)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    assert a[0][-1] > 4000


def test_rotated_orthorhombic_cell_gives_the_orthorhombic_result():
    """x -> x Q, H -> diag(L) Q: a full 3x3 cell that describes the same crystal.  E is unchanged, F and W rotate; the list is the
    same list.  The left-hand side runs the general-cell code, the right-hand side the orthorhombic code pinned elsewhere."""
    model, hp = _model()
    pos, sp, cell = WL.small_periodic(4, 2.3, 0.35, 2, seed=17)
    Q = _rotation(2)
    nbr = O.neighbors_bruteforce(pos, cell, hp["r_cut"])
    E, F, Ea, W = model.energy_forces(pos, sp, cell, nbr, virial=True)
    posr, Hr = pos @ Q, cell @ Q
    assert np.abs(Hr - np.diag(np.diag(Hr))).max() > 1.0
    nbr_r = O.neighbors_bruteforce(posr, Hr, hp["r_cut"])
    for x, y in zip(nbr, nbr_r):
        assert np.array_equal(x, y)
    Er, Fr, Ear, Wr = model.energy_forces(posr, sp, Hr, nbr_r, virial=True)
    assert abs(Er - E) <= 1e-12 * abs(E)
    np.testing.assert_allclose(Ear, Ea, atol=1e-12)
    np.testing.assert_allclose(Fr, F @ Q, atol=1e-11)
    np.testing.assert_allclose(Wr, Q.T @ W @ Q, atol=1e-10)
    # the transposed matrix is a different crystal: a code that mixed up rows and columns would pass neither
    assert abs(model.energy(posr, sp, Hr.T.copy() if np.linalg.det(Hr.T) > 0 else Hr) - E) > 1e-6 * abs(E)


def test_change_of_lattice_basis_leaves_energy_and_forces_unchanged():
    model, hp = _model(seed=9)
    pos, sp, H = _tri_system(4, seed=5)
    U = np.array([[1, 0, 0], [-1, 1, 0], [0, -1, 1]])                              # unimodular: same lattice, other basis
    assert round(np.linalg.det(U)) == 1
    H2 = U @ H
    assert hp["r_cut"] <= O.cell_widths(H2).min()
    E1, F1, _ = model.energy_forces(pos, sp, H, O.neighbors_bruteforce(pos, H, hp["r_cut"]))
    n2 = O.neighbors_bruteforce(pos, H2, hp["r_cut"])
    E2, F2, _ = model.energy_forces(pos, sp, H2, n2)
    assert abs(E1 - E2) <= 1e-12 * abs(E1)
    np.testing.assert_allclose(F1, F2, atol=1e-11)


def test_supercell_of_a_triclinic_cell():
    model, hp = _model(seed=11)
    pos, sp, H = _tri_system(4, seed=6)
    E1, F1, _ = model.energy_forces(pos, sp, H, O.neighbors_bruteforce(pos, H, hp["r_cut"]))
    reps = (2, 1, 2)
    H2 = H * np.array(reps)[:, None]
    pp, ss = [], []
    for t in itertools.product(*[range(r) for r in reps]):
        pp.append(pos + np.array(t) @ H); ss.append(sp)
    pos2, sp2 = np.concatenate(pp), np.concatenate(ss)
    E2, F2, _ = model.energy_forces(pos2, sp2, H2, O.neighbors_bruteforce(pos2, H2, hp["r_cut"]))
    assert abs(E2 - 4 * E1) <= 1e-11 * abs(E2)
    np.testing.assert_allclose(F2, np.tile(F1, (4, 1)), atol=1e-11)


def test_forces_and_virial_against_finite_differences_triclinic():
    model, hp = _model(seed=13)
    pos, sp, H = _tri_system(3, seed=7)
    H = H * 0.95
    pos = pos * 0.95
    assert hp["r_cut"] <= O.cell_widths(H).min()
    E, F, _, W = model.energy_forces(pos, sp, H, O.neighbors_bruteforce(pos, H, hp["r_cut"]), virial=True)
    h = 1e-5
    for (i, d) in [(0, 0), (5, 1), (11, 2), (20, 0)]:
        p1, p2 = pos.copy(), pos.copy()
        p1[i, d] += h; p2[i, d] -= h
        fd = -(model.energy(p1, sp, H) - model.energy(p2, sp, H)) / (2 * h)
        assert abs(fd - F[i, d]) <= 1e-6 * max(1.0, np.abs(F).max()), (i, d, fd, F[i, d])
    # dE/d eps_ab = -W_ab under r -> r (1 + eps), H -> H (1 + eps)
    for (a, b) in [(0, 0), (1, 1), (2, 2), (0, 1), (2, 0), (1, 2)]:
        eps = np.zeros((3, 3)); eps[a, b] = h
        Ep = model.energy(pos @ (np.eye(3) + eps), sp, H @ (np.eye(3) + eps))
        Em = model.energy(pos @ (np.eye(3) - eps), sp, H @ (np.eye(3) - eps))
        assert abs((Ep - Em) / (2 * h) + W[a, b]) <= 2e-6 * max(1.0, np.abs(W).max()), (a, b)
    np.testing.assert_allclose(W, W.T, atol=1e-9 * np.abs(W).max())
    np.testing.assert_allclose(O.stress(W, H), -W / np.linalg.det(H), rtol=1e-15)


def test_deform_keeps_fractional_coordinates_triclinic():
    pos, sp, H = _tri_system(3, seed=9)
    Hn = H @ (np.eye(3) + np.array([[0.02, 0.01, 0.0], [0.0, -0.01, 0.015], [0.0, 0.0, 0.03]]))
    p2, H2 = O.md_deform(pos, H, Hn)
    np.testing.assert_allclose(p2 @ np.linalg.inv(Hn), pos @ np.linalg.inv(H), atol=1e-12)
    np.testing.assert_array_equal(H2, Hn)
    # orthorhombic pair: the A26 expression x L'/L exactly
    p3, H3 = O.md_deform(pos, np.diag([9.0, 9.0, 9.0]), np.diag([9.9, 9.0, 8.1]))
    np.testing.assert_array_equal(p3, pos * (np.array([9.9, 9.0, 8.1]) / 9.0))


def test_md_in_a_triclinic_cell_conserves_energy_and_momentum():
    model, hp = _model(seed=15)
    pos, sp, H = _tri_system(3, seed=10, jitter=0.15)
    mass = np.where(sp == 0, 28.0855, 15.999)
    vel = WL.maxwell_boltzmann(mass, 300.0, 4)
    out = O.md_run(model, pos, vel, mass, sp, H, 0.4, 0.5, 30)
    Etot = out["energies"].sum(axis=1)
    assert np.abs(Etot - Etot[0]).max() <= 2e-4 * out["energies"][0, 1] + 1e-6    # dt^2 error, a small fraction of E_kin
    p = (mass[:, None] * out["vel"]).sum(0)
    assert np.abs(p).max() <= 1e-9
