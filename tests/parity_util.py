"""Helpers shared by the GPU parity tests, smoke() and bench.py: run a Workload through the
C ABI and compare with an oracle result.  Holds no transport arithmetic."""
import numpy as np

from workloads import Workload, SourceSpec, make_xs
from workloads.configs import DENSITY, BASE_SEED, cell_centres
from workloads.rng import uniform01


def masked_rel_err(gpu, ref, floor=1e-6):
    """max |gpu - ref| / |ref| where ref > floor * max(ref)  (north_star's mask), plus the mask size."""
    ref = np.asarray(ref, dtype=np.float64)
    gpu = np.asarray(gpu, dtype=np.float64)
    mx = np.abs(ref).max()
    if mx == 0.0:
        return float(np.abs(gpu).max()), 0
    m = ref > floor * mx
    if not m.any():
        return 0.0, 0
    return float((np.abs(gpu[m] - ref[m]) / np.abs(ref[m])).max()), int(m.sum())


def run_gpu(wl, closure=0, fixed_iters=None, **opts):
    """Solve `wl` through the C ABI; returns (problem handle, info dict)."""
    import paper_1910_11335_b200 as pkg
    p = pkg.problem_from_workload(wl)
    info = p.solve(tol=wl.tol, max_iters=wl.max_iters, fixed_iters=fixed_iters, closure=closure, **opts)
    return p, info


def compare_workload(wl, ref, closure=0, replay=True, check_unc=True, verbose=False, **opts):
    """GPU vs oracle on every (problem, group): scalar flux inside the mask.  With replay the GPU runs
    exactly the oracle's sweep counts (reading R10).  Returns the worst relative error."""
    fi = ref["iters"] if replay else None
    p, info = run_gpu(wl, closure=closure, fixed_iters=fi, **opts)
    worst = 0.0
    nprob, G = ref["iters"].shape
    shape = (wl.nz, wl.ny, wl.nx)
    for q in range(nprob):
        for g in range(G):
            got = p.get_flux_moments(q, g, 0)[0]
            e, n = masked_rel_err(got, ref["phi"][q, g, 0].reshape(shape))
            worst = max(worst, e)
            if verbose:
                print("  prob %d g %2d iters %3d/%3d  err %.3e  (mask %d)" % (q, g, info["iters"][q, g], ref["iters"][q, g], e, n))
    if check_unc:
        for s, src in enumerate(wl.sources):
            if src.kind == 0:
                continue
            for g in range(G):
                got = p.get_uncollided_flux(s, g)
                e, _ = masked_rel_err(got, ref["phi_u"][s, g].reshape(shape))
                worst = max(worst, e)
                if verbose and e > 1e-5:
                    print("  phi_u src %d g %d err %.3e" % (s, g, e))
    p.close()
    return worst


def tiny_p3_case(nx=12, ny=10, nz=9, G=3, sn=8, L=3, seed=7, kind=1):
    """Small ragged heterogeneous mesh with all four materials, P_L scattering, a point or cone source."""
    E, st, ss = make_xs(BASE_SEED + 100 + seed, G, L, 30.0, 100.0)
    c = np.arange(nx * ny * nz, dtype=np.uint64)
    mat = (uniform01(seed * 8 + 5, c) * 4).astype(np.uint8).reshape(nz, ny, nx)
    # blocky materials rather than white noise: coarsen by 3
    mat = mat[::3, ::3, ::3].repeat(3, 0).repeat(3, 1).repeat(3, 2)[:nz, :ny, :nx].copy()
    rho = (DENSITY[mat] * (1.0 + 0.05 * (2.0 * uniform01(seed * 8 + 6, c).reshape(nz, ny, nx) - 1.0))).astype(np.float32)
    d = 0.7
    if kind == 1:
        src = [SourceSpec(kind=1, pos=(-nx * d, 0.13, 0.21), spectrum=np.full(G, 1.0 / G))]
    else:
        src = [SourceSpec(kind=2, pos=(-nx * d, 0.13, 0.21), axis=(1.0, 0.0, 0.0), half_angle=np.deg2rad(25.0),
                          spectrum=np.full(G, 1.0 / G))]
    return Workload("tiny_%dx%dx%d_S%dP%d" % (nx, ny, nz, sn, L), nx, ny, nz, d, d * 1.1, d * 0.9, mat, rho, 4, G, L, sn,
                    st, ss, src, energies=E)
