"""The paper's largest timed configuration on one B200: ntg = [160^3, 160^3], lts = 500
(Table 4 lower: 521.970 s per time step on a Tesla V100), fp32.

    python paper_2104_05426_b200/examples/paper_table4_160.py [n] [T]

The history (32.8 GB raw, 65.7 GB packed) is generated on the device (uniform [-1,1], seeded);
dx = 0.1, c dt = 0.05 as in BASELINE.json configs[4], so the longest lag (551 steps) exceeds the
stored history as in that config.  Prints the pre-pass and jefi_fields times (CUDA events) and
cross-checks a slab of 4096 outputs of the tiled kernel against the per-point kernel.
Measured (profiles/r01_paper_160.md): 16.43 s per evaluation = 1.02e12 pairs/s.
"""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import numpy as np, torch
import paper_2104_05426_b200 as jb
n, T = int(sys.argv[1]) if len(sys.argv) > 1 else 160, int(sys.argv[2]) if len(sys.argv) > 2 else 500
dx, dt = 0.1, 0.05
org = tuple([-(n - 1) / 2 * dx] * 3)
torch.cuda.set_device(0)
print("free GB", torch.cuda.mem_get_info()[0] / 1e9, flush=True)
ctx = jb.Jefi((n, n, n), org, (dx,) * 3, dt=dt, c=1.0, nsteps=T, dtype="f32", n_obs=(n, n, n), origin_obs=org, spacing_obs=(dx,) * 3)
print("ctx device bytes GB", jb.jefi_device_bytes(ctx.ctx) / 1e9, flush=True)
g = torch.Generator(device="cuda"); g.manual_seed(160)
rho = torch.empty((T, n, n, n), dtype=torch.float32, device="cuda")
J = torch.empty((T, 3, n, n, n), dtype=torch.float32, device="cuda")
for m in range(T):
    rho[m].uniform_(-1, 1, generator=g); J[m].uniform_(-1, 1, generator=g)
torch.cuda.synchronize()
ev = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
s = torch.cuda.current_stream()
ev[0].record(s); ctx.upload_history(rho, J, s); ev[1].record(s)
E = torch.empty((3, n ** 3), dtype=torch.float32, device="cuda"); B = torch.empty_like(E)
ctx.fields(T - 1, E, B, stream=s); ev[2].record(s)
ctx.fields(T - 1, E, B, stream=s); ev[3].record(s)
torch.cuda.synchronize()
pairs = float(n ** 3) ** 2
print("prepass ms", ev[0].elapsed_time(ev[1]), "GB/s", (rho.nbytes + J.nbytes) * 3 / ev[0].elapsed_time(ev[1]) / 1e6)
for a, b in ((1, 2), (2, 3)):
    ms = ev[a].elapsed_time(ev[b]); print("fields ms", ms, "pairs/s %.4g" % (pairs / ms * 1e3), "frac of FP32 peak %.4f" % (pairs * 52 / ms * 1e3 / 74.44992e12), flush=True)
print("launches", ctx.launches)
# cross-check a slab of points against the per-point kernel
begin, count = (n // 2) * n * n + 37 * n, 4096
ctx.set_kernel(1)
E1 = torch.empty((3, count), dtype=torch.float32, device="cuda"); B1 = torch.empty_like(E1)
ctx.fields(T - 1, E1, B1, begin, count); torch.cuda.synchronize()
for nm, a, b in (("E", E[:, begin:begin + count], E1), ("B", B[:, begin:begin + count], B1)):
    print(nm, "rel-L2 tiled vs point", [float((a[c] - b[c]).norm() / b[c].norm()) for c in range(3)])
ctx.close()
