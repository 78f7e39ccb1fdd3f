#!/usr/bin/env python
"""Writes the stored expected values of the full-size parity tests (tests/test_gpu_golden.py) — calls ONLY oracle/ and
workloads/ (never the CUDA path).

The fp64 oracle needs minutes (config 3) to hours (config 4, per source) for a whole multigroup solve to the 1e-5
tolerance, so its result is computed once here and a sample is stored:

  python tests/golden/make_goldens.py cfg3                whole config 3 (128x128x64, S16, P3, 19 groups), closure 1
  python tests/golden/make_goldens.py cfg4 --source 0     config 4 (256x256x128, S8, P3, 47 groups), one of its 8 sources
  python tests/golden/make_goldens.py cfg4 --source 3     (source 0 is axis-aligned, source 3 sits at 135 degrees)
  python tests/golden/make_goldens.py cfg4 --source 0 --closure 0   (pure diamond difference, reported beside the gate)

Stored per (config, source) in tests/golden/<name>.npz, everything straight from oracle.solve (BASELINE.json configs[3],
[4]; readings R8-R10 of DESIGN.md: the sweep counts K[g] are replayed on the GPU):
  iters [G], residual [G], balance [G][3], phi0_max [G], phi0_min [G], n_negative [G]
  stride_idx [S]                 cell indices i + nx (j + ny k) of a fixed stride sample (prime stride)
  stride_phi [G][nm_s][S]        all moments (float32-rounded) of the collided flux there (--lean: the scalar flux only)
  stride_phi_u [G][S]            uncollided flux there
  small_idx / small_phi0 [G][T]  the T smallest in-mask cells (phi0 > 1e-6 max phi0) of every group and their scalar flux:
                                 the relative error of an fp32 path peaks there
  large_idx / large_phi0 [G][U]  the U largest cells of every group
Config 4 holds the moments of finished groups in float32 (oracle.solve store_dtype: 50 GB per source otherwise).
"""
import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle            # noqa: E402
from workloads import make_config    # noqa: E402

STRIDE = {3: 1021, 4: 4099}          # primes: the sample walks through every x, y, z residue
N_SMALL, N_LARGE = 2048, 256


def golden_name(cfg, source, closure=1):
    return "cfg%d_src%d_closure%d.npz" % (cfg, source, closure)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=["cfg3", "cfg4"])
    ap.add_argument("--source", type=int, default=0)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--lean", action="store_true", help="store only the scalar flux on the stride sample (1.1 MB instead of 6.4 MB per "
                    "config-4 source): used for the sources beyond 0, 3 and 5")
    ap.add_argument("--closure", type=int, default=1, help="1 = diamond difference + set-to-zero fix-up (reading R2, the gate of "
                    "configs 2-4); 0 = pure diamond difference (PAPER.md:287), stored beside it as a finding")
    args = ap.parse_args()
    cfg = int(args.config[3])
    wl = make_config(cfg)
    if not 0 <= args.source < len(wl.sources):
        raise SystemExit("config %d has %d source(s)" % (cfg, len(wl.sources)))
    wl.sources = [wl.sources[args.source]]                    # independent problems (mode 0): one at a time
    threads = args.threads or oracle.default_threads()
    oracle.build()
    t0 = time.time()

    def progress(p, g, k, delta):
        print("  group %2d  sweeps %2d  delta %.3e  [%.0f s]" % (g, k, delta, time.time() - t0), flush=True)

    print("%s source %d: oracle.solve, closure %d, tol %g, %d threads" % (wl.name, args.source, args.closure, wl.tol, threads), flush=True)
    res = oracle.solve(wl, closure=args.closure, threads=threads, progress=progress,
                       store_dtype=np.float32 if cfg == 4 else np.float64)
    phi, phi_u = res["phi"][0], res["phi_u"][0]               # [G][nm][cells], [G][cells]
    G = wl.G
    sidx = np.arange(0, wl.cells, STRIDE[cfg], dtype=np.int64)
    out = dict(iters=res["iters"][0].astype(np.int32), residual=res["residual"][0], balance=res["balance"][0],
               phi0_max=np.array([phi[g, 0].max() for g in range(G)]), phi0_min=np.array([phi[g, 0].min() for g in range(G)]),
               n_negative=np.array([(phi[g, 0] < 0).sum() for g in range(G)], dtype=np.int64),
               stride_idx=sidx.astype(np.int32),
               stride_phi=np.stack([phi[g][:1 if args.lean else None, sidx] for g in range(G)]).astype(np.float32),
               stride_phi_u=np.stack([phi_u[g][sidx] for g in range(G)]).astype(np.float32),
               mesh=np.array([wl.nx, wl.ny, wl.nz], dtype=np.int32), source=np.int32(args.source),
               seconds=np.array([res["seconds"][k] for k in ("raytrace", "fixed_source", "sweep")]),
               threads=np.int32(threads))
    small_idx, small_phi, large_idx, large_phi = [], [], [], []
    for g in range(G):
        p0 = np.asarray(phi[g, 0], dtype=np.float64)
        inmask = np.flatnonzero(p0 > 1e-6 * np.abs(p0).max())
        order = inmask[np.argsort(p0[inmask], kind="stable")]
        lo, hi = order[:N_SMALL], order[-N_LARGE:]
        lo = np.pad(lo, (0, N_SMALL - len(lo)), mode="edge") if len(lo) else np.zeros(N_SMALL, dtype=np.int64)
        hi = np.pad(hi, (0, N_LARGE - len(hi)), mode="edge") if len(hi) else np.zeros(N_LARGE, dtype=np.int64)
        small_idx.append(lo); small_phi.append(p0[lo]); large_idx.append(hi); large_phi.append(p0[hi])
    out.update(small_idx=np.stack(small_idx).astype(np.int32), small_phi0=np.stack(small_phi).astype(np.float32),
               large_idx=np.stack(large_idx).astype(np.int32), large_phi0=np.stack(large_phi).astype(np.float32))
    path = os.path.join(HERE, golden_name(cfg, args.source, args.closure))
    np.savez_compressed(path, **out)
    print("wrote %s (%.1f KB) after %.0f s; sweeps per group %s" % (path, os.path.getsize(path) / 1024.0, time.time() - t0,
                                                                    out["iters"].tolist()), flush=True)


if __name__ == "__main__":
    main()
