"""GPU unit test of the split-fp16 tcgen05 GEMM (csrc/gemm_f16s.cu) through the C-ABI test hook, against a plain
numpy fp64 product with the same fused prologue / epilogue, over several tiles, a ragged row tail, ragged K and N."""
import numpy as np
import pytest

from paper_2502_06073_b200 import workloads as WL

pytestmark = pytest.mark.gpu

PRO_NONE, PRO_SILU, PRO_SCALE_U = 0, 1, 2
EPI_STORE, EPI_GATHER2, EPI_Y_X, EPI_RESIDUAL, EPI_DSILU, EPI_ACCUM, EPI_SPLIT_RES = range(7)


def _silu(z):
    return z / (1.0 + np.exp(-z))


def _dsilu(z):
    s = 1.0 / (1.0 + np.exp(-z))
    return s * (1.0 + z * (1.0 - s))


@pytest.fixture(scope="module")
def handle(lib):
    w = WL.config0()
    return lib.Allegro(lib.build_weights(w.hp, 0), w.hp)


CASES = [
    # M, K0, K1, N, pro, epi, wtrans
    (1000, 64, 0, 64, PRO_NONE, EPI_STORE, 0),
    (37, 8, 0, 128, PRO_NONE, EPI_STORE, 0),
    (5000, 512, 256, 512, PRO_NONE, EPI_STORE, 0),
    (3333, 512, 0, 512, PRO_SILU, EPI_RESIDUAL, 0),
    (2049, 256, 0, 512, PRO_SILU, EPI_Y_X, 0),
    (4097, 512, 0, 768, PRO_SCALE_U, EPI_DSILU, 1),
    (1500, 512, 0, 768, PRO_NONE, EPI_SPLIT_RES, 1),
    (1200, 256, 0, 512, PRO_NONE, EPI_ACCUM, 1),
    (700, 36, 0, 28, PRO_SILU, EPI_STORE, 0),
    (129, 100, 0, 300, PRO_NONE, EPI_STORE, 1),
    (0, 64, 0, 64, PRO_NONE, EPI_STORE, 0),
]


@pytest.mark.parametrize("case", CASES)
def test_gemm_f16s_matches_fp64(lib, handle, case):
    import torch
    M, K0, K1, N, pro, epi, wtrans = case
    rng = np.random.default_rng(hash(case) % (2 ** 31))
    cap = M + 77
    K = K0 + K1
    A0 = rng.standard_normal((cap, K0)).astype(np.float32) * rng.choice([1e-3, 0.2, 1.0, 4.0], size=(cap, 1)).astype(np.float32)
    A1 = rng.standard_normal((cap, max(K1, 4))).astype(np.float32)
    Wm = (rng.standard_normal((N, K)) / np.sqrt(K)).astype(np.float32)          # B(k, n) = Wm[n, k]
    Wdev = np.ascontiguousarray(Wm.T) if wtrans else Wm
    geo = np.zeros((cap, 8), np.float32); geo[:, 4] = rng.uniform(0.05, 1.0, cap)
    aux_w = N if epi != EPI_SPLIT_RES else 512
    aux = rng.standard_normal((cap, aux_w)).astype(np.float32)
    c_old, c_new = 0.6, 0.8
    split = 512 if epi == EPI_SPLIT_RES else 0
    Cw = split if epi == EPI_SPLIT_RES else N
    C0 = rng.standard_normal((cap, Cw)).astype(np.float32)
    C2w = (N - split) if epi == EPI_SPLIT_RES else N
    t = lambda a: torch.from_numpy(a).cuda()
    dA0, dA1, dW, dgeo, daux, dC, dC2 = t(A0), t(A1), t(Wdev), t(geo), t(aux), t(C0.copy()), t(np.zeros((cap, C2w), np.float32))
    handle.debug_forget_weights()      # dW is a fresh matrix that may sit at a previous case's address
    handle.debug_gemm(M, cap, dA0, K0, dW, N, dC, A1=dA1 if K1 else None, K1=K1, wtrans=wtrans, pro=pro, epi=epi,
                      aux=(dC if epi == EPI_ACCUM else daux) if epi in (EPI_RESIDUAL, EPI_DSILU, EPI_ACCUM, EPI_SPLIT_RES) else None,
                      geo=dgeo, C2=dC2 if epi in (EPI_Y_X, EPI_RESIDUAL, EPI_SPLIT_RES) else None, split=split, c_old=c_old, c_new=c_new)
    C, C2 = dC.cpu().numpy().astype(np.float64), dC2.cpu().numpy().astype(np.float64)
    # ---- fp64 reference
    A = np.concatenate([A0[:, :K0], A1[:, :K1]], axis=1).astype(np.float64)[:M]
    u = geo[:M, 4:5].astype(np.float64)
    if pro == PRO_SILU:
        A = _silu(A)
    elif pro == PRO_SCALE_U:
        A = A * (c_new * u)
    V = A @ Wm.astype(np.float64).T
    x = aux[:M].astype(np.float64)
    # fp32 accumulation over K <= 768 products: a few 1e-6 of the row's RMS; a dropped correction pass would be ~1e-3
    row_rms = np.sqrt((V ** 2).mean(axis=1, keepdims=True)) if M else np.ones((0, 1))
    tol = 2e-5 * np.maximum(row_rms, 1e-30)

    def close(got, ref, scale=1.0):
        err = np.abs(got - ref)
        lim = tol * scale + 4e-7 * np.abs(ref)          # + fp32 rounding of the stored result itself
        assert np.all(err <= lim), float((err / lim).max())

    if M == 0:
        return
    if epi == EPI_STORE:
        close(C[:M], V)
    elif epi == EPI_Y_X:
        close(C[:M], V); close(C2[:M], u * V)
    elif epi == EPI_RESIDUAL:
        close(C[:M], V); close(C2[:M], c_old * x + c_new * u * V, 1.0 + np.abs(x).max() * 1e-1)
    elif epi == EPI_DSILU:
        close(C[:M], V * _dsilu(x), 2.0)
    elif epi == EPI_ACCUM:
        close(C[:M], C0[:M].astype(np.float64) + V, 1.0 + np.abs(C0).max() * 1e-1)
    elif epi == EPI_SPLIT_RES:
        close(C[:M], c_old * x[:, :split] + V[:, :split], 1.0 + np.abs(x).max() * 1e-1)
        close(C2[:M], V[:, split:])
    # rows past the last 128-row tile are never written (rows between M and the end of that tile are don't-care)
    Mt = (M + 127) // 128 * 128
    assert np.array_equal(dC.cpu().numpy()[Mt:], C0[Mt:])
