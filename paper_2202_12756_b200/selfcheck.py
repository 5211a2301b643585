"""`python -m paper_2202_12756_b200.selfcheck --shape 64 64 64 --dtype f64 --slabs 4 --variants 0 2 3`

One R2C + C2R pair per kernel variant on cuda:0 through the C ABI, checked by its round trip, by Parseval's identity and
by agreement between the variants -- no oracle involved, so an installed copy of the library can check itself, and small
enough to run under `compute-sanitizer` (the memcheck / racecheck / synccheck summaries under profiles/ were made with
exactly this command).  `--static` adds the allocation-free entry point fft3d_r2c_static where the grid fits its scratch.
Exits non-zero on any failure."""
from __future__ import annotations

import argparse
import math
import sys

import torch

from . import binding as B
from . import inputs


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--shape", type=int, nargs=3, default=[64, 64, 64])
    ap.add_argument("--dtype", choices=["f32", "f64"], default="f32")
    ap.add_argument("--slabs", type=int, default=4)
    ap.add_argument("--variants", type=int, nargs="+", default=[0, 2, 3, 1])
    ap.add_argument("--static", action="store_true")
    a = ap.parse_args(argv)
    if not torch.cuda.is_available():
        print("selfcheck needs a CUDA device (there is no CPU fallback)")
        return 2
    torch.cuda.set_device(0)
    shape = tuple(a.shape)
    dtype = torch.float32 if a.dtype == "f32" else torch.float64
    n = shape[0] * shape[1] * shape[2]
    bound = (2e-6 if a.dtype == "f32" else 1e-13) * math.log2(n)
    f = inputs.uniform_grid(shape, dtype, seed=0, device="cuda")
    rows_per_chunk = max(1, (1 << 26) // (shape[1] * shape[2]))          # x-planes per chunk: no array-sized temporaries
    energy = sum(float(f[x:x + rows_per_chunk].double().pow(2).sum()) for x in range(0, shape[0], rows_per_chunk))
    fmax = max(float(f[x:x + rows_per_chunk].abs().max()) for x in range(0, shape[0], rows_per_chunk))
    Mp1 = shape[2] // 2 + 1
    w = torch.full((Mp1,), 2.0, dtype=torch.float64, device="cuda")
    w[0] = w[-1] = 1.0
    keep_first = len(a.variants) > 1 or a.static
    ok, first = True, None
    for v in a.variants:
        plan = B.Plan(*shape, dtype=dtype, virtual_slabs=a.slabs)
        plan.set_variant(v)
        work = plan.empty_workspace("cuda")               # one workspace for both directions
        spec = plan.r2c(f, work=work)
        back = plan.c2r(spec, work=work)
        torch.cuda.synchronize()
        del work
        rt = max(float((back[x:x + rows_per_chunk] - f[x:x + rows_per_chunk]).abs().max())
                 for x in range(0, shape[0], rows_per_chunk)) / fmax
        del back
        rows = spec.reshape(-1, Mp1)
        step = max(1, (1 << 26) // Mp1)
        tot = sum(float((torch.view_as_real(rows[r:r + step]).double().pow(2).sum(dim=2) * w).sum())
                  for r in range(0, rows.shape[0], step))
        pars = abs(tot / n - energy) / energy
        if not keep_first:
            good = rt <= bound and pars <= 10 * bound
            ok = ok and good
            print("variant %d  %s | %s: round trip %.2e, Parseval %.2e (bound %.2e) %s"
                  % (v, " ".join(plan.launch_impls(0)), " ".join(plan.launch_impls(1)), rt, pars, bound, "ok" if good else "FAILED"))
            plan.close()
            continue
        nat = plan.to_natural(spec)
        dev = 0.0 if first is None else float((nat - first).abs().max()) / float(first.abs().max())
        first = nat.clone() if first is None else first
        good = rt <= bound and pars <= 10 * bound and dev <= 10 * bound
        ok = ok and good
        print("variant %d  %s | %s: round trip %.2e, Parseval %.2e, vs first variant %.2e (bound %.2e) %s"
              % (v, " ".join(plan.launch_impls(0)), " ".join(plan.launch_impls(1)), rt, pars, dev, bound, "ok" if good else "FAILED"))
        plan.close()
    if a.static:
        out = torch.empty(shape[0] * shape[1] * (shape[2] // 2 + 1), dtype=first.dtype, device="cuda")
        try:
            for _ in range(2):
                B.r2c_static(f, out, virtual_slabs=a.slabs)
            torch.cuda.synchronize()
            L = shape[1] // a.slabs
            nat = out.reshape(a.slabs, shape[0], L, shape[2] // 2 + 1).permute(1, 0, 2, 3).reshape(first.shape)
            dev = float((nat - first).abs().max()) / float(first.abs().max())
            good = dev <= 10 * bound
            ok = ok and good
            print("fft3d_r2c_static: vs first variant %.2e %s" % (dev, "ok" if good else "FAILED"))
        except B.Fft3dError as e:
            print("fft3d_r2c_static: %s" % e)
            ok = ok and e.status == 5
    print("selfcheck %s" % ("passed" if ok else "FAILED"))
    return 0 if ok else 1


if __name__ == "__main__":
    sys.exit(main())
