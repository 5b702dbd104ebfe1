"""Thin ctypes binding over the C-ABI of include/allegro.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of liballegro_b200.so; torch is used here only
for device memory and streams.  There is no CPU fallback: importing this module raises if the shared
library has not been built (``python -m paper_2502_06073_b200.build``), and every compute call raises
``AllegroError`` when the library reports an error (e.g. no CUDA device).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liballegro_b200.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2502_06073_b200.build` "
                      "(the CUDA extension is required; there is no CPU fallback)")
_lib = C.CDLL(LIB_PATH)

ERR_NAMES = {0: "OK", -1: "INVALID", -2: "UNSUPPORTED", -3: "CUDA", -4: "STALE_LIST", -5: "NONFINITE", -6: "CUTOFF",
             -7: "SPECIES", -8: "NO_LIST", -9: "ALLOC"}
EXPORTS = ["allegro_weight_layout", "allegro_create", "allegro_destroy", "allegro_build_neighbors",
           "allegro_energy_forces", "allegro_md_init", "allegro_md_step", "allegro_md_step_nvt", "allegro_md_deform",
           "allegro_set_state", "allegro_virial", "allegro_virial_noalloc", "allegro_debug_set_fusion", "allegro_debug_set_list_slack", "allegro_energy_forces_owned",
           "allegro_decomp_select", "allegro_decomp_scatter", "allegro_kick_drift", "allegro_get_state",
           "allegro_get_neighbors", "allegro_get_stats", "allegro_profile", "allegro_get_profile",
           "allegro_debug_coupling", "allegro_debug_num_paths", "allegro_debug_set_precision", "allegro_debug_gemm", "allegro_debug_forget_weights",
           "allegro_last_error"]
VIRIAL_NOALLOC_MAX_ATOMS = 1048576   # ALLEGRO_VIRIAL_NOALLOC_MAX_ATOMS of include/allegro.h
PROFILE_CLASSES = ["gemm", "tp_fwd", "tp_bwd", "gamma", "gammabar", "active_edges", "edge_misc", "neighbor", "md",
                   "force_gather", "gemm_f16s", "tp_mix", "tp_mix16"]


class HParams(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_bessel", C.c_int32), ("poly_p", C.c_int32), ("lmax", C.c_int32),
                ("n_layers", C.c_int32), ("n_channels", C.c_int32), ("full_o3", C.c_int32),
                ("two_body_nl", C.c_int32), ("two_body_dims", C.c_int32 * 8),
                ("latent_nl", C.c_int32), ("latent_dims", C.c_int32 * 8),
                ("edge_nl", C.c_int32), ("edge_dims", C.c_int32 * 8),
                ("r_cut", C.c_double), ("avg_num_neighbors", C.c_double)]


class AllegroError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"allegro error {code} ({ERR_NAMES.get(code, '?')}): {msg}")
        self.code = code


_vp, _i64, _dbl = C.c_void_p, C.c_int64, C.c_double
_lib.allegro_weight_layout.argtypes = [C.POINTER(HParams), _vp, _vp, _vp, C.c_int]
_lib.allegro_create.argtypes = [_vp, C.c_size_t, C.POINTER(HParams), C.POINTER(_vp)]
_lib.allegro_destroy.argtypes = [_vp]
_lib.allegro_build_neighbors.argtypes = [_vp, _vp, _vp, _i64, _vp, _dbl, _dbl, _vp]
_lib.allegro_energy_forces.argtypes = [_vp, _vp, _vp, _i64, _vp, _vp, _vp, _vp, _vp]
_lib.allegro_md_init.argtypes = [_vp, _vp, _vp, _vp, _vp, _i64, _vp, _dbl, _dbl, _vp]
_lib.allegro_md_step.argtypes = [_vp, _dbl, _i64, _vp]
_lib.allegro_md_step_nvt.argtypes = [_vp, _dbl, _i64, _dbl, _dbl, _i64, _dbl, _vp]
_lib.allegro_md_deform.argtypes = [_vp, _vp, _vp]
_lib.allegro_set_state.argtypes = [_vp, _vp, _vp, _vp]
_lib.allegro_virial.argtypes = [_vp, _vp, _vp, _vp]
_lib.allegro_virial_noalloc.argtypes = [_vp, _vp, _vp, _vp]
_lib.allegro_debug_set_fusion.argtypes = [_vp, C.c_int]
_lib.allegro_debug_forget_weights.argtypes = [_vp]
_lib.allegro_debug_set_list_slack.argtypes = [_vp, _dbl, _i64]
_lib.allegro_energy_forces_owned.argtypes = [_vp, _vp, _vp, _i64, _vp, _i64, _vp, _vp, _vp, _vp]
_lib.allegro_decomp_select.argtypes = [_vp, _vp, _vp, _i64, _vp, _vp, _vp, _dbl, _i64, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.allegro_decomp_scatter.argtypes = [_vp, _vp, _i64, _vp, _i64, _vp]
_lib.allegro_kick_drift.argtypes = [_vp, _vp, _vp, _vp, _i64, _dbl, C.c_int, _vp]
_lib.allegro_get_state.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.allegro_get_neighbors.argtypes = [_vp, _vp, _vp, _vp, _vp]
_lib.allegro_get_stats.argtypes = [_vp, _vp]
_lib.allegro_profile.argtypes = [_vp, C.c_int]
_lib.allegro_get_profile.argtypes = [_vp, _vp, _vp, _vp, C.c_int]
_lib.allegro_debug_coupling.argtypes = [C.c_int, C.c_int, C.c_int, _vp]
_lib.allegro_debug_num_paths.argtypes = [C.POINTER(HParams), C.c_int]
_lib.allegro_debug_set_precision.argtypes = [_vp, C.c_int]
_lib.allegro_debug_gemm.argtypes = [_vp, _i64, _i64, _vp, C.c_int, C.c_int, _vp, C.c_int, C.c_int, _vp, C.c_int, C.c_int, C.c_int,
                                    C.c_int, C.c_int, _vp, C.c_int, _vp, _vp, C.c_int, _vp, C.c_int, C.c_int, C.c_float, C.c_float, _vp]
_lib.allegro_last_error.argtypes = [_vp]
_lib.allegro_last_error.restype = C.c_char_p
for _n in EXPORTS[:-1]:
    getattr(_lib, _n).restype = C.c_int


def make_hparams(hp: dict) -> HParams:
    h = HParams()
    for k in ("n_species", "n_bessel", "poly_p", "lmax", "n_layers", "n_channels", "full_o3"):
        setattr(h, k, int(hp[k]))
    for name in ("two_body", "latent", "edge"):
        dims = list(hp[name + "_dims"])
        if len(dims) > 8:
            raise ValueError("at most 8 layers per MLP")
        setattr(h, name + "_nl", len(dims))
        arr = getattr(h, name + "_dims")
        for i, d in enumerate(dims):
            arr[i] = int(d)
    h.r_cut = float(hp["r_cut"])
    h.avg_num_neighbors = float(hp["avg_num_neighbors"])
    return h


def _last_error(handle=None) -> str:
    s = _lib.allegro_last_error(handle)
    return s.decode() if s else ""


def allegro_weight_layout(hp: dict):
    """-> list of (kind, rows, cols) in blob order."""
    h = make_hparams(hp)
    n = _lib.allegro_weight_layout(C.byref(h), None, None, None, 0)
    if n < 0:
        raise AllegroError(n, _last_error())
    kind = np.zeros(n, np.int32); rows = np.zeros(n, np.int64); cols = np.zeros(n, np.int64)
    _lib.allegro_weight_layout(C.byref(h), kind.ctypes.data, rows.ctypes.data, cols.ctypes.data, n)
    return [(int(k), int(r), int(c)) for k, r, c in zip(kind, rows, cols)]


def allegro_debug_coupling(l1, l2, l3) -> np.ndarray:
    out = np.zeros((2 * l1 + 1, 2 * l2 + 1, 2 * l3 + 1))
    rc = _lib.allegro_debug_coupling(l1, l2, l3, out.ctypes.data)
    if rc < 0:
        raise AllegroError(rc, "bad (l1,l2,l3)")
    return out


def allegro_debug_num_paths(hp: dict, layer: int) -> int:
    h = make_hparams(hp)
    rc = _lib.allegro_debug_num_paths(C.byref(h), layer)
    if rc < 0:
        raise AllegroError(rc, _last_error())
    return rc


def _ptr(t):
    return None if t is None else t.data_ptr()


def _stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


class Allegro:
    """One model handle.  Methods mirror the C entry points one to one."""

    def __init__(self, weights: np.ndarray, hp: dict):
        w = np.ascontiguousarray(weights, dtype=np.float32)
        self.hp = dict(hp)
        self._h = _vp()
        h = make_hparams(hp)
        rc = _lib.allegro_create(w.ctypes.data, w.size, C.byref(h), C.byref(self._h))
        if rc != 0:
            raise AllegroError(rc, _last_error())

    def _check(self, rc):
        if rc != 0:
            raise AllegroError(rc, _last_error(self._h))

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:   # _lib is None during interpreter shutdown
            _lib.allegro_destroy(self._h)
            self._h = None

    __del__ = close

    @staticmethod
    def _cell_host(cell):
        return np.ascontiguousarray(np.asarray(cell, dtype=np.float64).reshape(3, 3))

    def build_neighbors(self, pos, species, cell, cutoff, skin):
        c = self._cell_host(cell)
        self._n_atoms = pos.shape[0]
        self._check(_lib.allegro_build_neighbors(self._h, _ptr(pos), _ptr(species), pos.shape[0], c.ctypes.data,
                                                 float(cutoff), float(skin), _stream()))

    def energy_forces(self, pos, species, cell, E_out, F_out, E_atom_out=None):
        c = self._cell_host(cell)
        self._check(_lib.allegro_energy_forces(self._h, _ptr(pos), _ptr(species), pos.shape[0], c.ctypes.data,
                                               _ptr(E_out), _ptr(F_out), _ptr(E_atom_out), _stream()))

    def energy_forces_owned(self, pos, species, cell, n_owned, E_out, F_out, E_atom_out=None):
        c = self._cell_host(cell)
        self._check(_lib.allegro_energy_forces_owned(self._h, _ptr(pos), _ptr(species), pos.shape[0], c.ctypes.data, int(n_owned),
                                                     _ptr(E_out), _ptr(F_out), _ptr(E_atom_out), _stream()))

    def decomp_select(self, pos, species, cell, grid, coord, r_halo, local_pos, local_species, local_src):
        """-> (n_owned, n_local, local_cell [3,3]); the local arrays are caller tensors with capacity local_pos.shape[0]."""
        c = self._cell_host(cell)
        g = np.ascontiguousarray(grid, dtype=np.int32); k = np.ascontiguousarray(coord, dtype=np.int32)
        counts = np.zeros(2, np.int64); lc = np.zeros((3, 3))
        self._check(_lib.allegro_decomp_select(self._h, _ptr(pos), _ptr(species), pos.shape[0], c.ctypes.data, g.ctypes.data, k.ctypes.data,
                                               float(r_halo), int(local_pos.shape[0]), _ptr(local_pos), _ptr(local_species), _ptr(local_src),
                                               counts.ctypes.data, lc.ctypes.data, _stream()))
        return int(counts[0]), int(counts[1]), lc

    def md_init(self, pos, vel, mass, species, cell, cutoff, skin):
        c = self._cell_host(cell)
        self._n_atoms = pos.shape[0]
        self._check(_lib.allegro_md_init(self._h, _ptr(pos), _ptr(vel), _ptr(mass), _ptr(species), pos.shape[0],
                                         c.ctypes.data, float(cutoff), float(skin), _stream()))

    def md_step(self, dt_fs, n_steps):
        self._check(_lib.allegro_md_step(self._h, float(dt_fs), int(n_steps), _stream()))

    def md_step_nvt(self, dt_fs, n_steps, T0, T1, n_ramp, tau_fs):
        self._check(_lib.allegro_md_step_nvt(self._h, float(dt_fs), int(n_steps), float(T0), float(T1), int(n_ramp), float(tau_fs), _stream()))

    def md_deform(self, cell_new):
        c = self._cell_host(cell_new)
        self._check(_lib.allegro_md_deform(self._h, c.ctypes.data, _stream()))

    def set_state(self, pos, vel):
        self._check(_lib.allegro_set_state(self._h, _ptr(pos), _ptr(vel), _stream()))

    def virial(self, pos=None):
        """-> numpy [3,3]; pos = the positions of the last force evaluation (torch CUDA fp64) or None for the MD state."""
        import torch
        W = torch.zeros(9, dtype=torch.float64, device="cuda")
        self._check(_lib.allegro_virial(self._h, _ptr(pos), _ptr(W), _stream()))
        return W.cpu().numpy().reshape(3, 3)

    def virial_noalloc(self, W_out, pos=None):
        """allegro_virial_noalloc: writes the virial into W_out (torch CUDA fp64, 9 elements, the caller's buffer) on the current
        stream without allocating or synchronising; at most VIRIAL_NOALLOC_MAX_ATOMS atoms; calls that overlap on the GPU race."""
        self._check(_lib.allegro_virial_noalloc(self._h, _ptr(pos), _ptr(W_out), _stream()))

    def debug_set_fusion(self, on: bool):
        self._check(_lib.allegro_debug_set_fusion(self._h, int(bool(on))))

    def debug_set_list_slack(self, frac, extra):
        self._check(_lib.allegro_debug_set_list_slack(self._h, float(frac), int(extra)))

    def get_state(self, pos=None, vel=None, F=None, E_pot=None, E_kin=None):
        nreb = C.c_int64(0)
        self._check(_lib.allegro_get_state(self._h, _ptr(pos), _ptr(vel), _ptr(F), _ptr(E_pot), _ptr(E_kin),
                                           C.addressof(nreb), _stream()))
        return int(nreb.value)

    def get_neighbors(self):
        """-> (rowptr int64 [N+1], col int32 [E], shift int8 [E,3]) as torch CUDA tensors."""
        import torch
        E = C.c_int64(0)
        self._check(_lib.allegro_get_neighbors(self._h, None, None, None, C.addressof(E)))
        n = self._n_atoms
        rowptr = torch.empty(n + 1, dtype=torch.int64, device="cuda")
        col = torch.empty(max(E.value, 1), dtype=torch.int32, device="cuda")
        shift = torch.empty((max(E.value, 1), 3), dtype=torch.int8, device="cuda")
        torch.cuda.synchronize()
        self._check(_lib.allegro_get_neighbors(self._h, _ptr(rowptr), _ptr(col), _ptr(shift), C.addressof(E)))
        return rowptr, col[: E.value], shift[: E.value]

    def get_stats(self) -> dict:
        s = np.zeros(8, np.int64)
        self._check(_lib.allegro_get_stats(self._h, s.ctypes.data))
        return dict(active_edges=int(s[0]), list_edges=int(s[1]), launches=int(s[2]), rebuilds=int(s[3]),
                    force_evals=int(s[4]), chunks=max(1, int(s[5])), recoveries=int(s[6]))

    def profile(self, enable: bool):
        self._check(_lib.allegro_profile(self._h, 1 if enable else 0))

    def get_profile(self) -> dict:
        ms = np.zeros(16); ln = np.zeros(16, np.int64); wk = np.zeros(16)
        n = _lib.allegro_get_profile(self._h, ms.ctypes.data, ln.ctypes.data, wk.ctypes.data, 16)
        if n < 0:
            self._check(n)
        return {PROFILE_CLASSES[k]: dict(ms=float(ms[k]), launches=int(ln[k]), work=float(wk[k])) for k in range(n)}

    def debug_set_precision(self, passes: int):
        self._check(_lib.allegro_debug_set_precision(self._h, int(passes)))

    def debug_forget_weights(self):
        self._check(_lib.allegro_debug_forget_weights(self._h))

    def debug_gemm(self, M, rows_cap, A0, K0, W, N, C_out, A1=None, K1=0, wtrans=0, ldw=None, pro=0, epi=0, aux=None, geo=None,
                   C2=None, split=0, c_old=0.0, c_new=1.0):
        """One launch of the split-fp16 GEMM kernel on torch CUDA fp32 tensors (row-major, leading dimension = shape[1])."""
        ld = lambda t: 0 if t is None else int(t.shape[1])
        self._check(_lib.allegro_debug_gemm(self._h, int(M), int(rows_cap), _ptr(A0), ld(A0), int(K0), _ptr(A1), ld(A1), int(K1),
                                            _ptr(W), int(ldw if ldw is not None else W.shape[1]), int(wtrans), int(N), int(pro), int(epi),
                                            _ptr(aux), ld(aux), _ptr(geo), _ptr(C_out), ld(C_out), _ptr(C2), ld(C2), int(split),
                                            float(c_old), float(c_new), _stream()))

    # convenience wrappers (allocation + marshalling only) ---------------------------------------
    def compute(self, pos_np, species_np, cell, skin=0.0, want_atom=False):
        """Host arrays in, host arrays out: build list + one energy/force evaluation."""
        import torch
        pos = torch.from_numpy(np.ascontiguousarray(pos_np, dtype=np.float64)).cuda()
        sp = torch.from_numpy(np.ascontiguousarray(species_np, dtype=np.int32)).cuda()
        self._n_atoms = pos.shape[0]
        E = torch.zeros(1, dtype=torch.float64, device="cuda")
        F = torch.zeros((pos.shape[0], 3), dtype=torch.float64, device="cuda")
        Ea = torch.zeros(pos.shape[0], dtype=torch.float32, device="cuda") if want_atom else None
        self.build_neighbors(pos, sp, cell, self.hp["r_cut"], skin)
        self.energy_forces(pos, sp, cell, E, F, Ea)
        out = (float(E.item()), F.cpu().numpy())
        return out + ((Ea.cpu().numpy(),) if want_atom else ())


def decomp_scatter(F_local, local_src, n_local, F_global):
    rc = _lib.allegro_decomp_scatter(_ptr(F_local), _ptr(local_src), int(n_local), _ptr(F_global), F_global.shape[0], _stream())
    if rc != 0:
        raise AllegroError(rc, "allegro_decomp_scatter")


def kick_drift(pos, vel, F, mass, dt_fs, drift):
    rc = _lib.allegro_kick_drift(_ptr(pos), _ptr(vel), _ptr(F), _ptr(mass), pos.shape[0], float(dt_fs), 1 if drift else 0, _stream())
    if rc != 0:
        raise AllegroError(rc, "allegro_kick_drift")


def build_weights(hp: dict, seed: int) -> np.ndarray:
    """Random-init blob (A24) using the layout reported by the library."""
    from . import workloads
    return workloads.make_weights(allegro_weight_layout(hp), hp, seed)
