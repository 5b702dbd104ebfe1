"""Precision study behind reading R4: which tensor-core product kinds keep the forces inside the 1e-4 x RMS gate.

north_star allows tensor cores "only in a precision that stays inside the stated tolerance".  Every dense linear runs as a
split product with `passes` tensor-core passes: 3 = hi*hi + hi*lo + lo*hi (the default of both kernels: 3xTF32 in gemm_tc.cu,
split fp16 in gemm_f16s.cu), 2 = only the activations split (weights rounded to 11 bits), 1 = a single TF32 / fp16 pass.
The test measures max|dF|/RMS(F) and |dE|/|E| against the fp64 oracle for each kind on configs[1] (chained 3xTF32 kernels,
full-system oracle) and configs[3] (split-fp16 kernel, cached oracle subset) and asserts what the committed table
profiles/r2_precision.md states: 3 passes pass both gates with a wide margin, 1 and 2 passes fail the force gate."""
import math
import os

import numpy as np
import pytest

from oracle import allegro_oracle as O
from paper_2502_06073_b200 import workloads as WL

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _errs(E, F, Eo, Fo, idx=None):
    Fs = F if idx is None else F[idx]
    rms = math.sqrt((Fo ** 2).mean())
    return np.abs(Fs - Fo).max() / rms, (abs(E - Eo) / abs(Eo) if Eo is not None else float("nan"))


def test_precision_kinds_cfg1_chained_tf32(lib):
    w = WL.get(1)
    wts = lib.build_weights(w.hp, w.weight_seed)
    o = O.AllegroOracle(w.hp, wts)
    Eo, Fo, _ = o.energy_forces(w.pos, w.species, w.cell, O.neighbors_binned(w.pos, w.cell, w.hp["r_cut"]))
    res = {}
    for passes in (1, 2, 3):
        g = lib.Allegro(wts, w.hp)
        g.debug_set_precision(passes)
        E, F = g.compute(w.pos, w.species, w.cell, skin=w.skin)
        res[passes] = _errs(E, F, Eo, Fo)
        print("cfg1 TF32 passes=%d: max|dF|/RMS = %.3e  |dE|/|E| = %.3e" % ((passes,) + res[passes]))
    assert res[3][0] <= 1e-4 and res[3][1] <= 1e-5
    assert res[3][0] <= 0.2e-4                                 # margin: 5x inside the gate
    assert res[1][0] > 1e-4 and res[2][0] > 1e-4                # fewer passes do not survive the force gate


def test_precision_kinds_cfg3_split_fp16(lib):
    gold = np.load(os.path.join(GOLD, "cfg3_subset.npz"))
    w = WL.get(3)
    wts = lib.build_weights(w.hp, w.weight_seed)
    T, cen = gold["targets"], gold["centres"]
    res = {}
    for passes in (1, 2, 3):
        g = lib.Allegro(wts, w.hp)
        g.debug_set_precision(passes)
        E, F, Ea = g.compute(w.pos, w.species, w.cell, skin=w.skin, want_atom=True)
        dF, _ = _errs(E, F, None, gold["F_targets"], T)
        dEa = np.abs(Ea[cen] - gold["E_atom"]).max()
        res[passes] = (dF, dEa)
        print("cfg3 fp16 passes=%d: max|dF|/RMS = %.3e  max|dE_i| = %.3e eV" % (passes, dF, dEa))
        del g
    assert res[3][0] <= 1e-4 and res[3][1] <= 2e-5 * 10
    assert res[3][0] <= 0.2e-4
    assert res[1][0] > 1e-4 and res[2][0] > 1e-4
