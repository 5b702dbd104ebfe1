"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/allegro.h
declares, and its host-side logic (plan, weight layout, coupling tables) agrees with the oracle's
independently written one.  No compute call is made (there is no GPU here)."""
import os
import re

import numpy as np
import pytest

from oracle import allegro_oracle as O
from paper_2502_06073_b200 import workloads as WL

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "allegro.h")).read()
    declared = set(re.findall(r"\b(allegro_[a-z_]+)\s*\(", hdr))
    assert declared == set(lib.EXPORTS)
    for name in declared:
        assert hasattr(lib._lib, name), name


@pytest.mark.parametrize("cfg", [0, 1, 3])
def test_weight_layout_matches_oracle(lib, cfg):
    hp = {0: WL.config0().hp, 1: WL._cfg1_hp(), 3: WL.hparams(89, 3, 3, 64, [128, 256, 512], [512] * 3, [128], 6.0, 73.4)}[cfg]
    assert lib.allegro_weight_layout(hp) == [tuple(t) for t in O.weight_layout(hp)]


def test_coupling_tables_match_oracle(lib):
    for l1 in range(4):
        for l2 in range(4):
            for l3 in range(abs(l1 - l2), min(3, l1 + l2) + 1):
                np.testing.assert_allclose(lib.allegro_debug_coupling(l1, l2, l3), O.coupling_tensor(l1, l2, l3), atol=1e-13)


def test_path_counts_match_oracle(lib):
    for lmax, NL, full in [(1, 1, 1), (2, 2, 1), (3, 3, 1), (3, 3, 0), (2, 3, 1)]:
        hp = WL.hparams(2, lmax, NL, 4, [8, 8], [8, 8], [4], 4.0, 10.0, full_o3=full)
        plan = O.build_plan(hp)
        for L in range(1, NL + 1):
            assert lib.allegro_debug_num_paths(hp, L) == len(plan.paths[L - 1])


def test_bad_hparams_are_rejected(lib):
    hp = WL.hparams(2, 5, 1, 4, [8, 8], [8, 8], [4], 4.0, 10.0)
    with pytest.raises(lib.AllegroError):
        lib.allegro_weight_layout(hp)
    hp = WL.hparams(2, 2, 1, 4, [8, 8], [8, 12], [4], 4.0, 10.0)          # D mismatch (A10)
    with pytest.raises(lib.AllegroError):
        lib.allegro_weight_layout(hp)


def test_create_fails_loudly_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    hp = WL.config0().hp
    w = lib.build_weights(hp, 0)
    with pytest.raises(lib.AllegroError) as ei:
        lib.Allegro(w, hp)
    assert ei.value.code == -3                                             # ALLEGRO_ERR_CUDA: no CPU fallback
