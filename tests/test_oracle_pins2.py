"""Round-2 pins for the oracle: the subset / multi-chunk evaluation every large-config parity test relies on, the
binned neighbour search at >= 3 cells per axis, SiLU itself, the virial against central finite
differences of E under strain, the Berendsen thermostat (reading A25) and the affine deformation (A26)."""
import math

import numpy as np
import pytest

from oracle import allegro_oracle as O
from paper_2502_06073_b200 import workloads as WL


def _model(lmax=2, NL=2, n=4, S=2, rc=4.0, seed=5, navg=12.0):
    hp = WL.hparams(S, lmax, NL, n, [16, 12], [16, 12], [8], rc, navg)
    return O.AllegroOracle(hp, WL.make_weights(O.weight_layout(hp), hp, seed)), hp


# ---------------------------------------------------------------- silu: closed forms, not its own formula
def test_silu_closed_forms():
    z = np.linspace(-9, 9, 181)
    assert O.silu(np.array([0.0]))[0] == 0.0
    np.testing.assert_allclose(O.silu(z) - O.silu(-z), z, atol=1e-15)                  # z s(z) + z s(-z) = z
    np.testing.assert_allclose(O.silu(np.array([1.0]))[0], 1.0 / (1.0 + math.exp(-1.0)), rtol=1e-15)
    np.testing.assert_allclose(O.silu(z), 0.5 * z * (1.0 + np.tanh(0.5 * z)), atol=1e-14)  # logistic = (1 + tanh(z/2)) / 2
    assert O.silu_deriv(np.array([0.0]))[0] == 0.5
    np.testing.assert_allclose(O.silu_deriv(z) + O.silu_deriv(-z), 1.0, atol=1e-15)
    h = 1e-5
    fd = (O.silu(z + h) - O.silu(z - h)) / (2 * h)
    np.testing.assert_allclose(O.silu_deriv(z), fd, atol=1e-9)


# ---------------------------------------------------------------- neighbours at >= 3 cells per axis
@pytest.mark.parametrize("box", [(16.0, 16.0, 16.0), (14.0, 19.0, 24.5)])
def test_binned_equals_bruteforce_three_or_more_cells(box):
    rng = np.random.default_rng(21)
    cell = np.diag(box)
    pos = rng.uniform(-10.0, 40.0, (400, 3))                      # unwrapped, several images away
    radius = 4.4
    nc = np.floor(np.array(box) / radius).astype(int)
    assert nc.min() >= 3
    a, b = O.neighbors_binned(pos, cell, radius), O.neighbors_bruteforce(pos, cell, radius)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    assert a[0][-1] > 4000
    # the row-sampled form of the brute-force search is the same loop restricted to those centres
    rows = np.array([7, 0, 399, 123])
    rp, col, sh = O.neighbors_bruteforce(pos, cell, radius, rows=rows)
    for q, i in enumerate(rows):
        assert np.array_equal(col[rp[q]:rp[q + 1]], b[1][b[0][i]:b[0][i + 1]]) and np.array_equal(sh[rp[q]:rp[q + 1]], b[2][b[0][i]:b[0][i + 1]])


# ---------------------------------------------------------------- subset and chunked evaluation
def test_subset_with_closure_equals_full_evaluation():
    model, hp = _model()
    pos, sp, cell = WL.small_periodic(4, 2.3, 0.35, 2, seed=17)     # 64 atoms, box 9.2
    nbr = O.neighbors_bruteforce(pos, cell, hp["r_cut"])
    E, F, Ea = model.energy_forces(pos, sp, cell, nbr)
    rp, col, _ = nbr
    T = np.array([3, 17, 40])
    closure = set(T.tolist())
    for i in T:
        closure.update(col[rp[i]:rp[i + 1]].tolist())
    cen = np.array(sorted(closure))
    assert cen.size < 64                                            # a real subset
    Es, Fs, Eas = model.energy_forces(pos, sp, cell, nbr, centres=cen)
    np.testing.assert_allclose(Eas[cen], Ea[cen], rtol=0, atol=1e-13)
    np.testing.assert_allclose(Fs[T], F[T], rtol=0, atol=1e-12 * np.abs(F).max())
    assert abs(Es - Ea[cen].sum()) < 1e-11
    # without the closure the forces on the targets are NOT complete (the pin would notice a wrong gather)
    _, Fw, _ = model.energy_forces(pos, sp, cell, nbr, centres=T)
    assert np.abs(Fw[T] - F[T]).max() > 1e-3 * np.abs(F).max()


def test_chunked_evaluation_equals_single_chunk():
    model, hp = _model(lmax=3, NL=3)
    pos, sp, cell = WL.small_periodic(4, 2.3, 0.35, 2, seed=18)
    nbr = O.neighbors_bruteforce(pos, cell, hp["r_cut"])
    E, F, Ea, W = model.energy_forces(pos, sp, cell, nbr, virial=True)
    E2, F2, Ea2, W2 = model.energy_forces(pos, sp, cell, nbr, max_edges_per_chunk=300, virial=True)
    assert nbr[0][-1] > 1200                                        # several chunks
    np.testing.assert_allclose(Ea2, Ea, rtol=0, atol=1e-13)
    np.testing.assert_allclose(F2, F, rtol=0, atol=1e-12 * np.abs(F).max())
    np.testing.assert_allclose(W2, W, rtol=0, atol=1e-11 * np.abs(W).max())
    assert abs(E2 - E) < 1e-11 * abs(E)


# ---------------------------------------------------------------- virial / stress
def test_virial_periodic_diagonal_strain_fd():
    """dE/d eps_aa by central differences of E under a homogeneous stretch of cell and positions along a."""
    model, hp = _model()
    pos, sp, cell = WL.small_periodic(3, 2.9, 0.3, 2, seed=19)      # box 8.7 >= 2 r_c
    nbr = O.neighbors_bruteforce(pos, cell, hp["r_cut"])
    _, _, _, W = model.energy_forces(pos, sp, cell, nbr, virial=True)
    h = 1e-6
    for a in range(3):
        Es = []
        for sgn in (+1, -1):
            s = np.ones(3); s[a] += sgn * h
            p2, c2 = O.md_deform(pos, cell, np.diag(np.diag(cell) * s))
            Es.append(model.energy(p2, sp, c2))
        dE = (Es[0] - Es[1]) / (2 * h)
        assert abs(dE - (-W[a, a])) <= 2e-6 * max(1.0, abs(W).max()), (a, dE, -W[a, a])
    sig = O.stress(W, cell)
    np.testing.assert_allclose(sig, -W / 8.7 ** 3)
    np.testing.assert_allclose(W, W.T, atol=1e-10 * np.abs(W).max())          # rotation invariance of E


def test_virial_cluster_shear_strain_fd():
    """All six components on an open cluster (no edge crosses the box): r -> (1 + eps) r with eps symmetric."""
    model, hp = _model(lmax=3, NL=2)
    pos, sp, cell = WL.cluster(8, 2, seed=23, spread=2.0)
    c0 = pos.mean(0)
    nbr = O.neighbors_bruteforce(pos, cell, hp["r_cut"])
    _, _, _, W = model.energy_forces(pos, sp, cell, nbr, virial=True)
    h = 1e-6
    for a in range(3):
        for b in range(a, 3):
            eps = np.zeros((3, 3)); eps[a, b] += 0.5; eps[b, a] += 0.5
            Es = [model.energy(c0 + (pos - c0) @ (np.eye(3) + sgn * h * eps).T, sp, cell) for sgn in (+1, -1)]
            dE = (Es[0] - Es[1]) / (2 * h)
            ref = -0.5 * (W[a, b] + W[b, a])
            assert abs(dE - ref) <= 2e-6 * max(1.0, np.abs(W).max()), (a, b, dE, ref)
    F = model.energy_forces(pos, sp, cell, nbr)[1]
    # W = -sum_e r_e (x) g_e equals sum_i r_i (x) F_i for an open cluster (each edge enters F_i and F_j with opposite signs)
    np.testing.assert_allclose(W, np.einsum("ia,ib->ab", pos - c0, F), atol=1e-10 * np.abs(W).max())


# ---------------------------------------------------------------- thermostat and deformation
def test_berendsen_limits_and_relaxation():
    model, hp = _model(lmax=1, NL=1, rc=3.5)
    pos, sp, cell = WL.small_periodic(3, 2.6, 0.2, 2, seed=29)
    mass = np.where(sp == 0, 28.0, 16.0)
    vel = WL.maxwell_boltzmann(mass, 300.0, 3)
    nve = O.md_run(model, pos, vel, mass, sp, cell, 0.3, 0.5, 20)
    weak = O.md_run(model, pos, vel, mass, sp, cell, 0.3, 0.5, 20, thermostat=dict(T0=300.0, T1=300.0, n_ramp=0, tau=1e30))
    np.testing.assert_allclose(weak["pos"], nve["pos"], atol=1e-12)             # tau -> infinity is NVE
    # tau = dt rescales to the target exactly: T after every step = T_target (ramp 300 -> 900 K over 10 steps)
    hot = O.md_run(model, pos, vel, mass, sp, cell, 0.3, 0.5, 10, thermostat=dict(T0=300.0, T1=900.0, n_ramp=10, tau=0.5))
    T_end = 2.0 * hot["E_kin"] / ((3 * pos.shape[0] - 3) * O.KB_EV)
    assert abs(T_end - 900.0) < 1e-9 * 900.0
    mid = O.md_run(model, pos, vel, mass, sp, cell, 0.3, 0.5, 5, thermostat=dict(T0=300.0, T1=900.0, n_ramp=10, tau=0.5))
    assert abs(2.0 * mid["E_kin"] / ((3 * pos.shape[0] - 3) * O.KB_EV) - 600.0) < 1e-9 * 600.0
    # the COM momentum stays zero under a uniform velocity scaling
    assert np.abs((mass[:, None] * hot["vel"]).sum(0)).max() < 1e-12


def test_deform_is_affine_and_energy_consistent():
    model, hp = _model()
    pos, sp, cell = WL.small_periodic(3, 2.9, 0.3, 2, seed=31)
    p2, c2 = O.md_deform(pos, cell, np.diag([8.7 * 1.01, 8.7, 8.7 * 0.98]))
    np.testing.assert_allclose(p2 / pos, np.array([[1.01, 1.0, 0.98]]) * np.ones_like(pos), rtol=1e-15)
    # fractional coordinates are unchanged: the neighbour topology at a scaled cutoff is the same set of (i, j, s)
    a = O.neighbors_bruteforce(pos, cell, 3.0)
    b = O.neighbors_bruteforce(p2 * np.array([1 / 1.01, 1.0, 1 / 0.98]), cell, 3.0)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
