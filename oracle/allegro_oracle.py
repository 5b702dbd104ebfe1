"""fp64 CPU oracle for the Allegro energy + force hot path.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this module.  It shares no code with the CUDA path (``paper_2502_06073_b200/csrc``);
the only module both sides use is the seeded input generator ``paper_2502_06073_b200.workloads``,
which holds none of the method's arithmetic.

What it computes: the Allegro network energy E(r) exactly as SURVEY.md §8c writes it out from
PAPER.md:93 (architecture hyper-parameters), Table 1, PAPER.md:29/:142 (the
architecture is that of the paper's ref. 22) and PAPER.md:9 (strictly local, E(3)-equivariant), and
forces from its own hand-written analytic gradient (steps B1-B12), all in numpy float64, in the
paper's order and notation (F1-F12), with no blocking or fusion beyond processing centre atoms in
chunks (exact, because the model is strictly local).  ``numpy.matmul``/``einsum`` serve as the
library primitive for each linear step.

Pins (tests/test_oracle_*.py, ``-m "not gpu"``): closed forms for the envelope and Bessel basis,
scipy's spherical harmonics, sympy's exact Wigner-3j symbols for the coupling tensors, the worked
coupling values of SURVEY.md §8c, rotation/inversion/translation/permutation invariance, central
finite differences for the forces, net force / torque, supercell replication, strict locality, the
pair-potential special case (c_new = 0), brute-force neighbours, velocity-Verlet reversibility.

PARITY UNPINNED: the absolute energies/forces of the paper's *trained* Allegro-FM model on any
structure (no weights and no worked numbers are printed in PAPER.md), and the equivalence of this
spherical-harmonic basis with e3nn's (needed only to import trained weights).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

ACC_CONV = 9.648533212e-3   # A20: a[A/fs^2] = ACC_CONV * F[eV/A] / m[amu]
KB_EV = 8.617333262e-5      # A20: eV/K

WK_MATRIX, WK_RESIDUAL, WK_SIGMA, WK_MU = 0, 1, 2, 3


# ================================================================================================
# F1/F2: envelope and radial basis                                                  (A1, A2)
# ================================================================================================
def envelope(x, p):
    """F1: u(x) = 1 - (p+1)(p+2)/2 x^p + p(p+2) x^(p+1) - p(p+1)/2 x^(p+2) for x<1, else 0."""
    x = np.asarray(x, dtype=np.float64)
    u = 1.0 - 0.5 * (p + 1) * (p + 2) * x ** p + p * (p + 2) * x ** (p + 1) - 0.5 * p * (p + 1) * x ** (p + 2)
    return np.where(x < 1.0, u, 0.0)


def envelope_deriv(x, p):
    """B10: u'(x) = -(p(p+1)(p+2)/2) x^(p-1) (1-x)^2 for x<1, else 0."""
    x = np.asarray(x, dtype=np.float64)
    du = -0.5 * p * (p + 1) * (p + 2) * x ** (p - 1) * (1.0 - x) ** 2
    return np.where(x < 1.0, du, 0.0)


def bessel_raw(r, r_cut, n_bessel):
    """B_n(r) = (2/r_c) sin(n pi r / r_c) / r, n = 1..N_b  (without the envelope)."""
    r = np.asarray(r, dtype=np.float64)[..., None]
    n = np.arange(1, n_bessel + 1, dtype=np.float64)
    return (2.0 / r_cut) * np.sin(n * math.pi * r / r_cut) / r


def bessel_raw_deriv(r, r_cut, n_bessel):
    """dB_n/dr = (2/r_c) (k_n cos(k_n r)/r - sin(k_n r)/r^2), k_n = n pi / r_c."""
    r = np.asarray(r, dtype=np.float64)[..., None]
    k = np.arange(1, n_bessel + 1, dtype=np.float64) * math.pi / r_cut
    return (2.0 / r_cut) * (k * np.cos(k * r) / r - np.sin(k * r) / r ** 2)


# ================================================================================================
# F3: real spherical harmonics, component normalised, m = -l..l, polar axis z        (A3)
# ================================================================================================
def spherical_harmonics(n, lmax):
    """Y_lm(n) for unit vectors n [...,3] -> list over l of arrays [..., 2l+1] (formulas F3)."""
    n = np.asarray(n, dtype=np.float64)
    x, y, z = n[..., 0], n[..., 1], n[..., 2]
    s3, s5, s7, s15 = math.sqrt(3.0), math.sqrt(5.0), math.sqrt(7.0), math.sqrt(15.0)
    out = [np.ones(n.shape[:-1] + (1,))]
    if lmax >= 1:
        out.append(np.stack([s3 * y, s3 * z, s3 * x], -1))
    if lmax >= 2:
        out.append(np.stack([s15 * x * y, s15 * y * z, 0.5 * s5 * (3 * z * z - 1), s15 * x * z,
                             0.5 * s15 * (x * x - y * y)], -1))
    if lmax >= 3:
        a, b, c = math.sqrt(35.0 / 8.0), math.sqrt(105.0), math.sqrt(21.0 / 8.0)
        out.append(np.stack([a * y * (3 * x * x - y * y), b * x * y * z, c * y * (5 * z * z - 1),
                             0.5 * s7 * (5 * z ** 3 - 3 * z), c * x * (5 * z * z - 1),
                             0.5 * b * (x * x - y * y) * z, a * x * (x * x - 3 * y * y)], -1))
    if lmax >= 4:
        raise ValueError("lmax <= 3")
    return out


def spherical_harmonics_grad(n, lmax):
    """Gradients w.r.t. (x,y,z) of the polynomials F3 exactly as written -> list of [..., 2l+1, 3].
    Used only inside the tangential projector of B11, so the off-sphere extension is irrelevant."""
    n = np.asarray(n, dtype=np.float64)
    x, y, z = n[..., 0], n[..., 1], n[..., 2]
    o, zero = np.ones_like(x), np.zeros_like(x)
    s3, s5, s7, s15 = math.sqrt(3.0), math.sqrt(5.0), math.sqrt(7.0), math.sqrt(15.0)

    def vec(gx, gy, gz):
        return np.stack([gx, gy, gz], -1)

    out = [np.zeros(n.shape[:-1] + (1, 3))]
    if lmax >= 1:
        out.append(np.stack([vec(zero, s3 * o, zero), vec(zero, zero, s3 * o), vec(s3 * o, zero, zero)], -2))
    if lmax >= 2:
        out.append(np.stack([
            vec(s15 * y, s15 * x, zero),
            vec(zero, s15 * z, s15 * y),
            vec(zero, zero, 3 * s5 * z),
            vec(s15 * z, zero, s15 * x),
            vec(s15 * x, -s15 * y, zero)], -2))
    if lmax >= 3:
        a, b, c = math.sqrt(35.0 / 8.0), math.sqrt(105.0), math.sqrt(21.0 / 8.0)
        out.append(np.stack([
            vec(a * 6 * x * y, a * (3 * x * x - 3 * y * y), zero),
            vec(b * y * z, b * x * z, b * x * y),
            vec(zero, c * (5 * z * z - 1), c * 10 * y * z),
            vec(zero, zero, 0.5 * s7 * (15 * z * z - 3)),
            vec(c * (5 * z * z - 1), zero, c * 10 * x * z),
            vec(b * x * z, -b * y * z, 0.5 * b * (x * x - y * y)),
            vec(a * (3 * x * x - 3 * y * y), -a * 6 * x * y, zero)], -2))
    return out


# ================================================================================================
# coupling tensors C^(l1 l2 l3) in the F3 basis                                       (A9)
# ================================================================================================
def _clebsch_gordan_complex(j1, m1, j2, m2, j3, m3):
    """<j1 m1 j2 m2 | j3 m3> by Racah's formula (integer j)."""
    if m1 + m2 != m3 or not (abs(j1 - j2) <= j3 <= j1 + j2):
        return 0.0
    f = math.factorial
    pref = math.sqrt((2 * j3 + 1) * f(j3 + j1 - j2) * f(j3 - j1 + j2) * f(j1 + j2 - j3) / f(j1 + j2 + j3 + 1))
    pref *= math.sqrt(f(j3 + m3) * f(j3 - m3) * f(j1 - m1) * f(j1 + m1) * f(j2 - m2) * f(j2 + m2))
    s = 0.0
    for k in range(0, j1 + j2 - j3 + 1):
        d = [k, j1 + j2 - j3 - k, j1 - m1 - k, j2 + m2 - k, j3 - j2 + m1 + k, j3 - j1 - m2 + k]
        if min(d) < 0:
            continue
        s += (-1.0) ** k / np.prod([float(f(v)) for v in d])
    return pref * s


def _real_from_complex(l):
    """U^l with Y^real_m = sum_mu U[m,mu] Y^complex_mu; index m,mu = -l..l stored at +l offset."""
    U = np.zeros((2 * l + 1, 2 * l + 1), dtype=np.complex128)
    r2 = 1.0 / math.sqrt(2.0)
    for m in range(-l, l + 1):
        if m > 0:
            U[m + l, m + l] = (-1.0) ** m * r2
            U[m + l, -m + l] = r2
        elif m == 0:
            U[l, l] = 1.0
        else:
            mu = -m
            U[m + l, -mu + l] = 1j * r2
            U[m + l, mu + l] = -1j * (-1.0) ** mu * r2
    return U


_CG_CACHE: dict = {}


def coupling_tensor(l1, l2, l3):
    """Real O(3)-invariant 3-tensor for (l1,l2,l3): Frobenius norm sqrt(2 l3+1), first nonzero entry in
    lexicographic (m1,m2,m3) order positive (A9).  Shape [2l1+1, 2l2+1, 2l3+1]."""
    key = (l1, l2, l3)
    if key in _CG_CACHE:
        return _CG_CACHE[key]
    cg = np.zeros((2 * l1 + 1, 2 * l2 + 1, 2 * l3 + 1))
    for m1 in range(-l1, l1 + 1):
        for m2 in range(-l2, l2 + 1):
            m3 = m1 + m2
            if abs(m3) <= l3:
                cg[m1 + l1, m2 + l2, m3 + l3] = _clebsch_gordan_complex(l1, m1, l2, m2, l3, m3)
    R = np.einsum("am,bn,co,mno->abc", _real_from_complex(l1), _real_from_complex(l2),
                  np.conj(_real_from_complex(l3)), cg.astype(np.complex128))
    C = R.real if (l1 + l2 + l3) % 2 == 0 else R.imag
    other = R.imag if (l1 + l2 + l3) % 2 == 0 else R.real
    assert np.abs(other).max() < 1e-12
    C = C * (math.sqrt(2 * l3 + 1) / np.linalg.norm(C))
    C[np.abs(C) < 1e-12] = 0.0
    first = C.ravel()[np.flatnonzero(C.ravel())[0]]
    if first < 0:
        C = -C
    _CG_CACHE[key] = C
    return C


# ================================================================================================
# plan: irreps and paths per layer                                                     (A8)
# ================================================================================================
def _irrep_sort_key(ir):
    l, p = ir
    return (l, 0 if p == (-1) ** l else 1)   # l ascending, natural parity before unnatural


@dataclass
class Plan:
    hp: dict
    G: list                 # env irreps [(l, (-1)^l)]
    K: list                 # K[L] = kept irreps of V^L, L = 0..NL-1
    paths: list             # paths[L-1] = list of (ir1, l2, ir_out) for layer L = 1..NL
    out_irreps: list        # out_irreps[L-1] = targets of layer L: [(0,+1)] + K[L] (if L<NL)

    @property
    def n_scalars(self):
        return self.hp["n_channels"] * (self.hp["lmax"] + 1)


def build_plan(hp) -> Plan:
    lmax, NL, full = hp["lmax"], hp["n_layers"], hp.get("full_o3", 1)
    G = [(l, (-1) ** l) for l in range(lmax + 1)]

    def allowed(ir1, ir2, lo):
        ok = abs(ir1[0] - ir2[0]) <= lo <= min(ir1[0] + ir2[0], lmax)
        if not full:
            ok = ok and (ir1[0] + ir2[0] + lo) % 2 == 0
        return ok

    R = [list(G)]
    for L in range(1, NL + 1):
        nxt = set()
        for ir1 in R[-1]:
            for ir2 in G:
                for lo in range(0, lmax + 1):
                    if allowed(ir1, ir2, lo):
                        nxt.add((lo, ir1[1] * ir2[1]))
        R.append(sorted(nxt, key=_irrep_sort_key))
    targets = {NL: [(0, 1)]}
    K = [None] * NL
    for L in range(NL - 1, -1, -1):
        keep = []
        for ir1 in R[L]:
            hit = any(allowed(ir1, ir2, lo) and (lo, ir1[1] * ir2[1]) in targets[L + 1]
                      for ir2 in G for lo in range(lmax + 1))
            if hit:
                keep.append(ir1)
        K[L] = sorted(keep, key=_irrep_sort_key)
        targets[L] = sorted(set(K[L]) | {(0, 1)}, key=_irrep_sort_key)
    paths, outs = [], []
    for L in range(1, NL + 1):
        pl = []
        for ir1 in K[L - 1]:                       # l1 ascending, natural parity first
            for ir2 in G:                          # l2 ascending
                for lo in range(lmax + 1):         # l_out ascending
                    iro = (lo, ir1[1] * ir2[1])
                    if allowed(ir1, ir2, lo) and iro in targets[L]:
                        pl.append((ir1, ir2[0], iro))
        paths.append(pl)
        outs.append(list(targets[L]))
    assert K[0] == G, "V^0 carries exactly the natural-parity irreps"
    return Plan(hp=hp, G=G, K=K, paths=paths, out_irreps=outs)


def weight_layout(hp):
    """Blob order of SURVEY.md §8b: list of (kind, rows, cols)."""
    plan = build_plan(hp)
    S, Nb, n, lmax, NL = hp["n_species"], hp["n_bessel"], hp["n_channels"], hp["lmax"], hp["n_layers"]
    D = hp["two_body_dims"][-1]
    assert hp["latent_dims"][-1] == D
    lay = []
    fan = 2 * S + Nb
    for h in hp["two_body_dims"]:
        lay.append((WK_MATRIX, h, fan)); fan = h
    lay.append((WK_MATRIX, n * (lmax + 1), D))                       # W_init
    for L in range(1, NL + 1):
        lay.append((WK_MATRIX, n * (lmax + 1), D))                   # W_env^L
        fan = D + n * (lmax + 1)
        for h in hp["latent_dims"]:
            lay.append((WK_MATRIX, h, fan)); fan = h
        lay.append((WK_RESIDUAL, 1, 2))                              # c_old^L, c_new^L
        if L < NL:
            for iro in plan.K[L]:
                P = sum(1 for p in plan.paths[L - 1] if p[2] == iro)
                lay.append((WK_MATRIX, n, P * n))                    # W_lin^{L,(l,p)}
    fan = D
    for h in hp["edge_dims"]:
        lay.append((WK_MATRIX, h, fan)); fan = h
    lay.append((WK_MATRIX, 1, fan))
    lay.append((WK_SIGMA, 1, S))
    lay.append((WK_MU, 1, S))
    return lay


def unpack_weights(hp, blob):
    """Split the flat fp32 blob into fp64 arrays following weight_layout()."""
    blob = np.asarray(blob, dtype=np.float32)
    lay = weight_layout(hp)
    assert blob.size == sum(r * c for _, r, c in lay), "weight blob size mismatch"
    it, off = [], 0
    for kind, r, c in lay:
        it.append(blob[off: off + r * c].astype(np.float64).reshape(r, c)); off += r * c
    it = iter(it)
    plan = build_plan(hp)
    W = {"two_body": [next(it) for _ in hp["two_body_dims"]], "init": next(it), "layers": []}
    for L in range(1, hp["n_layers"] + 1):
        lw = {"env": next(it), "latent": [next(it) for _ in hp["latent_dims"]]}
        c = next(it).ravel()
        lw["c_old"], lw["c_new"] = float(c[0]), float(c[1])
        lw["lin"] = {iro: next(it) for iro in plan.K[L]} if L < hp["n_layers"] else {}
        W["layers"].append(lw)
    W["edge"] = [next(it) for _ in range(len(hp["edge_dims"]) + 1)]
    W["sigma"] = next(it).ravel()
    W["mu"] = next(it).ravel()
    return W


# ================================================================================================
# neighbours                                                                         (A16, A17)
# ================================================================================================
def _cell_matrix(cell):
    """H [3,3], rows = lattice vectors a_1, a_2, a_3 (reading A27): a periodic image is x + s_1 a_1 + s_2 a_2 + s_3 a_3."""
    H = np.asarray(cell, dtype=np.float64).reshape(3, 3)
    if not np.linalg.det(H) > 0.0:
        raise ValueError("cell must be right-handed with positive volume")
    return H


def _is_diag(H):
    return np.abs(H - np.diag(np.diag(H))).max() == 0.0


def _image_shift(s, H):
    """Cartesian shift of image s [..., 3]: (s_1 a_1 + s_2 a_2) + s_3 a_3, in this order (A27).  For a diagonal H the two
    added terms are exact zeros, so the value is s_d L_d bit for bit, the expression of A16."""
    s = np.asarray(s, dtype=np.float64)
    return (s[..., 0:1] * H[0] + s[..., 1:2] * H[1]) + s[..., 2:3] * H[2]


def cell_widths(cell):
    """Perpendicular widths of the cell: the distance between the lattice planes f_d = 0 and f_d = 1 of the fractional
    coordinate f = x H^-1, w_d = 1 / |column d of H^-1|.  For an orthorhombic cell these are the box lengths."""
    H = _cell_matrix(cell)
    if _is_diag(H):
        return np.diag(H).copy()
    Hinv = np.linalg.inv(H)
    return 1.0 / np.sqrt((Hinv * Hinv).sum(axis=0))


def _fractional(x, H):
    """x H^-1 (x / L for a diagonal H, the expression the orthorhombic pins were made with)."""
    if _is_diag(H):
        return x / np.diag(H)
    return x @ np.linalg.inv(H)


def neighbors_bruteforce(pos, cell, radius, rows=None):
    """All ordered (i, j, s) with |r_j + s.cell - r_i| < radius, (i,j,s) != (i,i,0): O(N^2 * 27).

    A16: d^2 = dx^2+dy^2+dz^2 in fp64 with dx = (x_j - x_i) + s_x L_x, compared as d^2 < radius^2.
    A17: requires radius <= min(L); the three images nearest to the rounded minimum image are tried
    per axis, which then covers every image inside the sphere.  Returns CSR (rowptr int64, col int32,
    shift int32 [E,3]) with each row sorted by (j, sx, sy, sz).  ``rows``: only these centre atoms (CSR over
    them, in the given order) - the same loop body, used to sample rows of systems too large for N^2."""
    pos = np.asarray(pos, dtype=np.float64)
    H = _cell_matrix(cell)
    if radius > cell_widths(cell).min():
        raise ValueError("radius exceeds the smallest box length (perpendicular width of the cell)")
    N = pos.shape[0]
    R2 = radius * radius
    centres = np.arange(N) if rows is None else np.asarray(rows)
    rows_j, rows_s, counts = [], [], np.zeros(centres.size, np.int64)
    trip = np.array([(a, b, c) for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1)], dtype=np.int64)
    for q, i in enumerate(centres):
        d0 = pos - pos[i]                                   # x_j - x_i
        n0 = -np.round(_fractional(d0, H)).astype(np.int64)  # image bringing j closest to i (in fractional coordinates)
        s = n0[:, None, :] + trip[None, :, :]               # [N,27,3]
        dx = d0[:, None, :] + _image_shift(s, H)            # (x_j - x_i) + s L   (A16; A27 for a general cell)
        d2 = dx[..., 0] * dx[..., 0] + dx[..., 1] * dx[..., 1] + dx[..., 2] * dx[..., 2]
        ok = d2 < R2
        ok[i] &= np.any(s[i] != 0, axis=1)                  # drop (i,i,0)
        jj, tt = np.nonzero(ok)
        ss = s[jj, tt]
        order = np.lexsort((ss[:, 2], ss[:, 1], ss[:, 0], jj))
        rows_j.append(jj[order]); rows_s.append(ss[order]); counts[q] = jj.size
    rowptr = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    col = np.concatenate(rows_j).astype(np.int32) if centres.size else np.zeros(0, np.int32)
    shift = np.concatenate(rows_s).astype(np.int32) if centres.size else np.zeros((0, 3), np.int32)
    return rowptr, col, shift


def neighbors_binned(pos, cell, radius):
    """Same set as neighbors_bruteforce, with candidates from a coarse grid (for the larger configs).
    The accept test is the identical fp64 expression; only the candidate enumeration differs."""
    pos = np.asarray(pos, dtype=np.float64)
    H = _cell_matrix(cell)
    Ld = cell_widths(cell)
    if radius > Ld.min():
        raise ValueError("radius exceeds the smallest box length (perpendicular width of the cell)")
    N = pos.shape[0]
    R2 = radius * radius
    nc = np.maximum(1, np.floor(Ld / (radius * (1 + 1e-9))).astype(np.int64))
    if _is_diag(H):
        h = Ld / nc
        w = np.floor(pos / Ld).astype(np.int64)
        xt = pos - w * Ld
        ci = np.clip((xt / h).astype(np.int64), 0, nc - 1)
    else:                                                     # bins in fractional coordinates: every point within radius of x
        f = _fractional(pos, H)                               # has |delta f_d| <= radius / width_d <= 1 / nc_d
        w = np.floor(f).astype(np.int64)
        ci = np.clip(((f - w) * nc).astype(np.int64), 0, nc - 1)
    cid = (ci[:, 0] * nc[1] + ci[:, 1]) * nc[2] + ci[:, 2]
    order = np.argsort(cid, kind="stable")
    start = np.searchsorted(cid[order], np.arange(nc.prod() + 1))
    ii_all, jj_all, ss_all = [], [], []
    for off in [(a, b, c) for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1)]:
        nb = ci + np.array(off)
        img = np.floor_divide(nb, nc)                        # -1, 0, +1 image of the neighbour cell
        nbw = nb - img * nc
        nbid = (nbw[:, 0] * nc[1] + nbw[:, 1]) * nc[2] + nbw[:, 2]
        lo, hi = start[nbid], start[nbid + 1]
        cnt = hi - lo
        i_rep = np.repeat(np.arange(N), cnt)
        k = np.arange(cnt.sum()) - np.repeat(np.cumsum(cnt) - cnt, cnt)
        j = order[np.repeat(lo, cnt) + k]
        s = img[i_rep] + w[i_rep] - w[j]
        dx = (pos[j] - pos[i_rep]) + _image_shift(s, H)
        d2 = dx[:, 0] * dx[:, 0] + dx[:, 1] * dx[:, 1] + dx[:, 2] * dx[:, 2]
        ok = (d2 < R2) & ~((i_rep == j) & np.all(s == 0, axis=1))
        ii_all.append(i_rep[ok]); jj_all.append(j[ok]); ss_all.append(s[ok])
    ii, jj, ss = np.concatenate(ii_all), np.concatenate(jj_all), np.concatenate(ss_all)
    o = np.lexsort((ss[:, 2], ss[:, 1], ss[:, 0], jj, ii))
    ii, jj, ss = ii[o], jj[o], ss[o]
    rowptr = np.concatenate([[0], np.cumsum(np.bincount(ii, minlength=N))]).astype(np.int64)
    return rowptr, jj.astype(np.int32), ss.astype(np.int32)


# ================================================================================================
# the network: forward F1-F12 and analytic backward B1-B12
# ================================================================================================
def silu(z):
    return z / (1.0 + np.exp(-z))


def silu_deriv(z):
    s = 1.0 / (1.0 + np.exp(-z))
    return s * (1.0 + z * (1.0 - s))


def _segment_sum(a, seg, nseg):
    out = np.zeros((nseg,) + a.shape[1:], dtype=np.float64)
    np.add.at(out, seg, a)
    return out


def _mlp_forward(Ws, h):
    """linear, SiLU, linear, ..., linear (no activation after the last, no bias) (A5)."""
    zs = []
    for W in Ws[:-1]:
        z = h @ W.T
        zs.append(z)
        h = silu(z)
    return h @ Ws[-1].T, zs


def _mlp_backward(Ws, zs, ybar):
    g = ybar @ Ws[-1]
    for W, z in zip(Ws[-2::-1], zs[::-1]):
        g = (g * silu_deriv(z)) @ W
    return g


class AllegroOracle:
    """E(r), F(r) of the Allegro network of SURVEY.md §8c in float64."""

    def __init__(self, hp, weights):
        self.hp = dict(hp)
        self.plan = build_plan(self.hp)
        self.W = unpack_weights(self.hp, weights)
        self.C = {}
        for pl in self.plan.paths:
            for (ir1, l2, iro) in pl:
                self.C[(ir1[0], l2, iro[0])] = coupling_tensor(ir1[0], l2, iro[0])

    # ------------------------------------------------------------------------------------------
    def _chunk(self, pos, species, cell, ci, cj, cs, centre_local, n_centres, taps=None):
        """Forward + backward for a set of edges whose centre atoms are all inside the chunk.
        ci, cj: global atom indices per edge; centre_local: row index within the chunk.
        Returns (E_i over the chunk's centres [n_centres], g_e = dE/d rvec_e [E,3], per-edge W_e)."""
        hp, plan, W = self.hp, self.plan, self.W
        S, Nb, n, lmax, NL, p = hp["n_species"], hp["n_bessel"], hp["n_channels"], hp["lmax"], hp["n_layers"], hp["poly_p"]
        rc, navg = hp["r_cut"], hp["avg_num_neighbors"]
        inv_sqrt_n = 1.0 / math.sqrt(navg)
        rvec = (pos[cj] - pos[ci]) + _image_shift(cs, _cell_matrix(cell))
        r = np.sqrt(rvec[:, 0] * rvec[:, 0] + rvec[:, 1] * rvec[:, 1] + rvec[:, 2] * rvec[:, 2])
        Ne = r.shape[0]
        rhat = rvec / r[:, None]
        x = r / rc
        # F1, F2, F3
        u = envelope(x, p)
        B = bessel_raw(r, rc, Nb)
        b = B * u[:, None]
        Y = spherical_harmonics(rhat, lmax)
        # F4
        oh_i = np.zeros((Ne, S)); oh_i[np.arange(Ne), species[ci]] = 1.0
        oh_j = np.zeros((Ne, S)); oh_j[np.arange(Ne), species[cj]] = 1.0
        in2b = np.concatenate([oh_i, oh_j, b], axis=1)
        y0, zs0 = _mlp_forward(W["two_body"], in2b)
        xl = u[:, None] * y0
        # F5
        winit = (xl @ W["init"].T).reshape(Ne, n, lmax + 1)
        V = {(l, (-1) ** l): winit[:, :, l, None] * Y[l][:, None, :] for l in range(lmax + 1)}
        saved = []
        for L in range(1, NL + 1):
            lw = W["layers"][L - 1]
            # F6, F7
            w = (xl @ lw["env"].T).reshape(Ne, n, lmax + 1)
            Gam = [inv_sqrt_n * _segment_sum(w[:, :, l, None] * Y[l][:, None, :], centre_local, n_centres)
                   for l in range(lmax + 1)]
            Gam_e = [g[centre_local] for g in Gam]
            # F8
            T = [np.einsum("abc,eia,eib->eic", self.C[(ir1[0], l2, iro[0])], V[ir1], Gam_e[l2])
                 for (ir1, l2, iro) in plan.paths[L - 1]]
            # F9: scalar paths in enumeration order, path-major then channel
            sc = [k for k, pth in enumerate(plan.paths[L - 1]) if pth[2] == (0, 1)]
            s = np.concatenate([T[k][:, :, 0] for k in sc], axis=1)
            # F10
            lat_in = np.concatenate([xl, s], axis=1)
            y, zs = _mlp_forward(lw["latent"], lat_in)
            x_new = lw["c_old"] * xl + lw["c_new"] * u[:, None] * y
            # F11
            V_new = {}
            if L < NL:
                for iro in plan.K[L]:
                    ks = [k for k, pth in enumerate(plan.paths[L - 1]) if pth[2] == iro]
                    Tcat = np.concatenate([T[k] for k in ks], axis=1)          # [E, P*n, 2l+1]
                    V_new[iro] = np.einsum("dk,ekm->edm", lw["lin"][iro], Tcat)
            saved.append(dict(w=w, Gam_e=Gam_e, V=V, zs=zs, y=y, x_prev=xl, sc=sc))
            if taps is not None:
                taps.setdefault("Gamma", []).append(Gam); taps.setdefault("s", []).append(s)
                taps.setdefault("x", []).append(x_new); taps.setdefault("V", []).append(V_new)
            xl, V = x_new, V_new
        # F12
        eps = xl
        for We in W["edge"]:
            eps = eps @ We.T
        eps = eps[:, 0]
        zi_c = np.zeros(n_centres, dtype=np.int64)
        zi_c[centre_local] = species[ci]
        has = np.zeros(n_centres, dtype=bool); has[centre_local] = True
        E_i = W["sigma"][zi_c] * _segment_sum(eps, centre_local, n_centres)   # mu added by the caller
        if taps is not None:
            taps.update(u=u, b=b, Y=Y, x0=saved[0]["x_prev"] if saved else xl, eps=eps, r=r, winit=winit)

        # ---------------- backward ----------------
        # B1
        g = W["sigma"][species[ci]][:, None]                          # eps_bar_e = sigma_{Z_i}
        for We in W["edge"][::-1]:
            g = g @ We
        xbar = g                                                        # [E, D]
        ubar = np.zeros(Ne)
        Ybar = [np.zeros_like(Yl) for Yl in Y]
        Vbar = {}                                                       # adjoint of V^L (empty at L=NL)
        for L in range(NL, 0, -1):
            lw, sv = W["layers"][L - 1], saved[L - 1]
            pl = plan.paths[L - 1]
            Tbar = [None] * len(pl)
            # B2
            if L < NL:
                for iro in plan.K[L]:
                    ks = [k for k, pth in enumerate(pl) if pth[2] == iro]
                    Tcat_bar = np.einsum("dk,edm->ekm", lw["lin"][iro], Vbar[iro])
                    for q, k in enumerate(ks):
                        Tbar[k] = Tcat_bar[:, q * n:(q + 1) * n, :]
            # B3
            ybar = lw["c_new"] * u[:, None] * xbar
            ubar += lw["c_new"] * np.sum(xbar * sv["y"], axis=1)
            xbar_prev = lw["c_old"] * xbar
            # B4
            gin = _mlp_backward(lw["latent"], sv["zs"], ybar)
            D = xbar.shape[1]
            xbar_prev = xbar_prev + gin[:, :D]
            sbar = gin[:, D:]
            for q, k in enumerate(sv["sc"]):
                t = np.zeros((Ne, n, 1)); t[:, :, 0] = sbar[:, q * n:(q + 1) * n]
                Tbar[k] = t if Tbar[k] is None else Tbar[k] + t
            # B5
            Vbar_prev = {ir: np.zeros_like(v) for ir, v in sv["V"].items()}
            Gbar_e = [np.zeros((Ne, n, 2 * l + 1)) for l in range(lmax + 1)]
            for k, (ir1, l2, iro) in enumerate(pl):
                if Tbar[k] is None:
                    continue
                C = self.C[(ir1[0], l2, iro[0])]
                Vbar_prev[ir1] += np.einsum("abc,eic,eib->eia", C, Tbar[k], sv["Gam_e"][l2])
                Gbar_e[l2] += np.einsum("abc,eic,eia->eib", C, Tbar[k], sv["V"][ir1])
            Gbar = [_segment_sum(ge, centre_local, n_centres)[centre_local] for ge in Gbar_e]
            # B6
            wbar = np.zeros((Ne, n, lmax + 1))
            for l in range(lmax + 1):
                wbar[:, :, l] = inv_sqrt_n * np.einsum("eim,em->ei", Gbar[l], Y[l])
                Ybar[l] += inv_sqrt_n * np.einsum("ei,eim->em", sv["w"][:, :, l], Gbar[l])
            # B7
            xbar_prev = xbar_prev + wbar.reshape(Ne, -1) @ lw["env"]
            xbar, Vbar = xbar_prev, Vbar_prev
        # B8
        wibar = np.zeros((Ne, n, lmax + 1))
        for l in range(lmax + 1):
            ir = (l, (-1) ** l)
            wibar[:, :, l] = np.einsum("eim,em->ei", Vbar[ir], Y[l])
            Ybar[l] += np.einsum("ei,eim->em", winit[:, :, l], Vbar[ir])
        xbar = xbar + wibar.reshape(Ne, -1) @ W["init"]
        # B9
        y0bar = u[:, None] * xbar
        ubar += np.sum(xbar * y0, axis=1)
        bbar = _mlp_backward(W["two_body"], zs0, y0bar)[:, 2 * S:]
        # B10
        du = envelope_deriv(x, p) / rc
        dB = bessel_raw_deriv(r, rc, Nb)
        rbar = np.sum(bbar * (dB * u[:, None] + B * du[:, None]), axis=1) + ubar * du
        # B11
        dY = spherical_harmonics_grad(rhat, lmax)
        t = np.zeros((Ne, 3))
        for l in range(lmax + 1):
            t += np.einsum("em,emk->ek", Ybar[l], dY[l])
        t_perp = t - rhat * np.sum(t * rhat, axis=1, keepdims=True)
        g_e = rbar[:, None] * rhat + t_perp / r[:, None]
        return E_i, has, g_e

    # ------------------------------------------------------------------------------------------
    def energy_forces(self, pos, species, cell, nbr, centres=None, max_edges_per_chunk=200_000, taps=None, virial=False):
        """E = sum_i E_i and F_i = -dE/dr_i (B12), using the neighbour list ``nbr`` =
        (rowptr, col, shift).  Edges with r >= r_cut contribute exactly zero and are skipped (A11).

        ``centres``: optional array of centre atoms; then only their E_i are summed and F is the
        gradient of that partial sum (used for subset parity on large configs).

        ``virial=True`` appends W[a][b] = -sum_e (rvec_e)_a (g_e)_b [eV] (the stress the
        paper's tensile test reads, is -W / V, see ``stress``)."""
        pos = np.asarray(pos, dtype=np.float64)
        species = np.asarray(species)
        rowptr, col, shift = nbr
        N = pos.shape[0]
        H = _cell_matrix(cell)
        rc2 = self.hp["r_cut"] ** 2
        centres = np.arange(N) if centres is None else np.asarray(centres)
        E_atom = np.zeros(N)
        F = np.zeros((N, 3))
        Wvir = np.zeros((3, 3))
        mu = self.W["mu"]
        k = 0
        while k < centres.size:
            k1, ne = k, 0
            while k1 < centres.size and (k1 == k or ne + (rowptr[centres[k1] + 1] - rowptr[centres[k1]]) <= max_edges_per_chunk):
                ne += rowptr[centres[k1] + 1] - rowptr[centres[k1]]; k1 += 1
            cc = centres[k:k1]
            idx = np.concatenate([np.arange(rowptr[a], rowptr[a + 1]) for a in cc]) if cc.size else np.zeros(0, np.int64)
            loc = np.repeat(np.arange(cc.size), [rowptr[a + 1] - rowptr[a] for a in cc])
            ci = np.repeat(cc, [rowptr[a + 1] - rowptr[a] for a in cc])
            cj = col[idx].astype(np.int64)
            cs = shift[idx].astype(np.float64)
            dx = (pos[cj] - pos[ci]) + _image_shift(cs, H)
            d2 = dx[:, 0] * dx[:, 0] + dx[:, 1] * dx[:, 1] + dx[:, 2] * dx[:, 2]
            act = d2 < rc2
            ci, cj, cs, loc, dxa = ci[act], cj[act], cs[act], loc[act], dx[act]
            E_atom[cc] = mu[species[cc]]
            if ci.size:
                E_i, has, g_e = self._chunk(pos, species, cell, ci, cj, cs, loc, cc.size, taps=taps)
                E_atom[cc] += E_i
                # B12: F_i = sum_{e in row(i)} g_e - sum_{e: j(e)=i} g_e
                np.add.at(F, ci, g_e)
                np.subtract.at(F, cj, g_e)
                Wvir -= dxa.T @ g_e
            k = k1
        if virial:
            return float(np.sum(E_atom[centres])), F, E_atom, Wvir
        return float(np.sum(E_atom[centres])), F, E_atom

    def energy(self, pos, species, cell, radius=None):
        """Convenience: rebuild the (brute-force) list at r_cut and return E only (for FD pins)."""
        radius = self.hp["r_cut"] if radius is None else radius
        nbr = neighbors_bruteforce(pos, cell, radius)
        return self.energy_forces(pos, species, cell, nbr)[0]


def stress(virial, cell):
    """Cauchy stress of the potential part [eV/A^3]: sigma_ab = (1/V) dE/d eps_ab = -W_ab / V for the homogeneous
    strain r -> (1 + eps) r, cell -> (1 + eps) cell (PAPER.md:69 tensile test, :93/:112 stress in the training loss)."""
    return -np.asarray(virial) / float(np.linalg.det(_cell_matrix(cell)))


def md_deform(pos, cell, cell_new):
    """A26: affine remap of the (unwrapped) positions from ``cell`` to ``cell_new``: the fractional coordinates are kept,
    x' = x H^-1 H'  (x' = x L'_x / L_x when both cells are orthorhombic).  The applied strain of PAPER.md:69 is a sequence of
    such increments between MD segments."""
    H, Hn = _cell_matrix(cell), _cell_matrix(cell_new)
    pos = np.asarray(pos, dtype=np.float64)
    if _is_diag(H) and _is_diag(Hn):
        return pos * (np.diag(Hn) / np.diag(H)), np.diag(np.diag(Hn))
    A = np.linalg.inv(H) @ Hn
    return (pos[:, 0:1] * A[0] + pos[:, 1:2] * A[1]) + pos[:, 2:3] * A[2], Hn.copy()


# ================================================================================================
# a-6: velocity-Verlet NVE with skin-triggered rebuilds                               (A20, A22)
# ================================================================================================
def kinetic_energy(vel, mass):
    return float(0.5 * np.sum(mass[:, None] * vel * vel) / ACC_CONV)


def md_run(model: AllegroOracle, pos, vel, mass, species, cell, skin, dt, n_steps, neighbor_fn=neighbors_bruteforce,
           thermostat=None):
    """Kick-drift-kick; rebuild when max_i |r_i - r_i^build| > skin/2, tested after the drift and
    before the force call; skin = 0 rebuilds every step.  Returns a dict with the final state.

    ``thermostat`` = dict(T0, T1, n_ramp, tau) switches to the canonical ensemble the paper runs (PAPER.md:49,
    :116 "NVT", :75 heating 300 -> 1200 K), reading A25: Berendsen weak coupling applied after the second half-kick
    of step k (1-based): T_inst = 2 E_kin / ((3N - 3) k_B), T_target = T0 + (T1 - T0) min(1, k / n_ramp),
    v <- v sqrt(1 + (dt / tau) (T_target / T_inst - 1))."""
    pos, vel = np.array(pos, dtype=np.float64), np.array(vel, dtype=np.float64)
    radius = model.hp["r_cut"] + skin
    nbr = neighbor_fn(pos, cell, radius)
    r_build = pos.copy()
    E, F, _ = model.energy_forces(pos, species, cell, nbr)
    n_rebuilds = 0
    traj_E = [(E, kinetic_energy(vel, mass))]
    for _ in range(n_steps):
        vel += 0.5 * dt * ACC_CONV * F / mass[:, None]
        pos += dt * vel
        d = pos - r_build
        dmax2 = np.max(d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1] + d[:, 2] * d[:, 2])
        if skin == 0.0 or dmax2 > (0.5 * skin) ** 2:
            nbr = neighbor_fn(pos, cell, radius)
            r_build = pos.copy()
            n_rebuilds += 1
        E, F, _ = model.energy_forces(pos, species, cell, nbr)
        vel += 0.5 * dt * ACC_CONV * F / mass[:, None]
        if thermostat is not None:
            k = len(traj_E)                                   # 1-based step index
            T_inst = 2.0 * kinetic_energy(vel, mass) / ((3 * pos.shape[0] - 3) * KB_EV)
            frac = min(1.0, k / thermostat["n_ramp"]) if thermostat.get("n_ramp", 0) > 0 else 1.0
            T_tgt = thermostat["T0"] + (thermostat["T1"] - thermostat["T0"]) * frac
            vel *= math.sqrt(1.0 + (dt / thermostat["tau"]) * (T_tgt / T_inst - 1.0))
        traj_E.append((E, kinetic_energy(vel, mass)))
    return dict(pos=pos, vel=vel, F=F, E_pot=E, E_kin=kinetic_energy(vel, mass), n_rebuilds=n_rebuilds,
                energies=np.array(traj_E))
