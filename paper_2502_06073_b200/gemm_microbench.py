import sys, os, time
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))  # repo root
import numpy as np, torch
from paper_2502_06073_b200 import binding as B, workloads as WL
w = WL.config0()
h = B.Allegro(B.build_weights(w.hp, 0), w.hp)
M = int(sys.argv[1]) if len(sys.argv) > 1 else 300000
h.debug_set_precision(int(sys.argv[2]) if len(sys.argv) > 2 else 3)
shapes = [(8, 128, 0, 0), (512, 512, 0, 0), (512, 512, 1, 3), (768, 512, 0, 0), (512, 256, 0, 0), (704, 64, 0, 0), (256, 512, 1, 2), (128, 256, 1, 0)]
sel = [int(x) for x in sys.argv[3].split(',')] if len(sys.argv) > 3 else range(len(shapes))
for (K, N, pro, epi) in [shapes[i] for i in sel]:
    A = torch.randn(M, K, device="cuda"); W = torch.randn(N, K, device="cuda") / K ** 0.5
    C = torch.zeros(M, N, device="cuda"); C2 = torch.zeros(M, N, device="cuda"); aux = torch.randn(M, N, device="cuda")
    geo = torch.rand(M, 8, device="cuda")
    kw = dict(pro=pro, epi=epi, geo=geo, aux=aux if epi in (3, 4) else None, C2=C2 if epi in (2, 3) else None, c_old=0.7, c_new=0.7)
    h.debug_forget_weights()           # W is a new matrix (the packed copy is cached by address and shape)
    for _ in range(2):
        h.debug_gemm(M, M, A, K, W, N, C, **kw)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 5
    e0.record()
    for _ in range(reps):
        h.debug_gemm(M, M, A, K, W, N, C, **kw)
    e1.record(); torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    fl = 2.0 * M * K * N
    tiles = ((M + 127) // 128) * ((N + 255) // 256)
    print(f"K={K:4d} N={N:4d} pro={pro} epi={epi}: {ms*1e3:8.1f} us  {fl/ms/1e9:7.1f} TFLOP/s (1-pass equiv)  {ms*1e6/ (tiles/148):8.0f} ns/tile  {ms*1e6*1.9/(tiles/148)/max(1,(K+31)//32):7.0f} cyc/stage")
