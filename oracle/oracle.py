"""ORACLE — test infrastructure, not product code.

fp64 CPU implementation of the DOCTORS hot path written from PAPER.md and the
readings R1-R16.  Shares no code with the CUDA library; only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import it.  The heavy loops (sweep, ray trace, schedule) are plain C in
sweep.c; everything else is numpy, step by step in the paper's order.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): quadrature moment identities and
tabulated mu_1 / S8 weights, addition theorem, Eq. (9) = enumeration = brute
force, Table 1 rows, 1-D closed-form attenuation ((1-h)/(1+h))^n -> exp(-sigma L),
per-sweep particle balance, sweep-order independence (bitwise), cube symmetry,
moment form vs discrete-to-discrete form of Eq. (2), linearity, homogeneous-mesh
ray-trace closed form.  Absolute flux values on the five configs: parity unpinned
by the paper (it prints none) — see DESIGN.md.
"""
import ctypes
import os
import subprocess
import math
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


def build(force=False):
    """Compile sweep.c -> liboracle.so with gcc (fp64, no fast-math)."""
    src = os.path.join(_HERE, "sweep.c")
    out = os.path.join(_HERE, "liboracle.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC",
                               "-ffp-contract=off", "-o", out, src, "-lm"])
    return out


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(build())
        _LIB.orc_wavefront_size.restype = ctypes.c_int64
    return _LIB


def _p(a, t=ctypes.c_double):
    return a.ctypes.data_as(ctypes.POINTER(t))


def default_threads():
    return max(1, len(os.sched_getaffinity(0)))


# --------------------------------------------------------------------------------------
# Quadrature: level-symmetric LQ_N (PAPER.md:39-42, :208 give only N(N+2); rule = DESIGN.md App. A)
# --------------------------------------------------------------------------------------
def _lq_classes(N, mu1sq):
    n = N // 2
    step = 2.0 * (1.0 - 3.0 * mu1sq) / (N - 2) if N > 2 else 0.0
    mu = np.sqrt(mu1sq + np.arange(n) * step)                      # levels
    pts = [(i, j, n + 2 - i - j) for i in range(1, n + 1) for j in range(1, n + 1)
           if 1 <= n + 2 - i - j <= n]
    classes = sorted(set(tuple(sorted(p)) for p in pts))
    return mu, pts, classes


def _lq_weights(N, mu1sq):
    """Class weights (octant-normalised) from the even one-axis moments k = 0..N/2-1,
    plus for N = 16 the mixed moment mu^4 eta^4 xi^4 = 1/5005; returns also the k = N/2 residual."""
    from numpy.linalg import lstsq
    mu, pts, classes = _lq_classes(N, mu1sq)
    n = N // 2
    A = np.zeros((n + 1, len(classes)))
    for p in pts:
        c = classes.index(tuple(sorted(p)))
        for k in range(n + 1):
            A[k, c] += mu[p[0] - 1] ** (2 * k)
    b = np.array([1.0 / (2 * k + 1) for k in range(n + 1)])
    Aa, bb = A[:n], b[:n]
    if N == 16:
        r = np.zeros(len(classes))
        for p in pts:
            r[classes.index(tuple(sorted(p)))] += (mu[p[0] - 1] * mu[p[1] - 1] * mu[p[2] - 1]) ** 4
        Aa, bb = np.vstack([Aa, r]), np.append(bb, 1.0 / 5005.0)
    wc = lstsq(Aa, bb, rcond=None)[0]
    return wc, float(A[n] @ wc - b[n]), mu, pts, classes


def level_symmetric(N):
    """omega [N(N+2)][3], w [N(N+2)] with sum w = 4 pi; octant-major, octant bit0/1/2 = -x/-y/-z."""
    from scipy.optimize import brentq
    if N == 2:
        mu1sq = 1.0 / 3.0
    else:
        f = lambda x: _lq_weights(N, x)[1]
        xs = np.linspace(1e-3, 1.0 / 3.0 - 1e-4, 2000)
        vals = [f(x) for x in xs]
        mu1sq = None
        for a, b, fa, fb in zip(xs[:-1], xs[1:], vals[:-1], vals[1:]):
            if fa * fb < 0:
                r = brentq(f, a, b, xtol=1e-17, rtol=1e-15)
                if _lq_weights(N, r)[0].min() > 0:                 # reject the negative-weight root (S6)
                    mu1sq = r
        assert mu1sq is not None
    wc, _, mu, pts, classes = _lq_weights(N, mu1sq)
    M = len(pts)
    base = np.array([[mu[p[0] - 1], mu[p[1] - 1], mu[p[2] - 1]] for p in pts])
    wb = np.array([wc[classes.index(tuple(sorted(p)))] for p in pts]) * (4.0 * math.pi / 8.0)
    omega = np.zeros((8 * M, 3))
    w = np.zeros(8 * M)
    for o in range(8):
        sgn = np.array([-1.0 if o & 1 else 1.0, -1.0 if o & 2 else 1.0, -1.0 if o & 4 else 1.0])
        omega[o * M:(o + 1) * M] = base * sgn
        w[o * M:(o + 1) * M] = wb
    return omega, w


# --------------------------------------------------------------------------------------
# Real spherical harmonics (reading R4) and the projection tables of Eq. (2)/(3)
# --------------------------------------------------------------------------------------
def real_sph_harm(L, omega):
    """Y [n][(L+1)^2], index lm = l^2 + l + m.  Y_l0 = P_l(xi);
    Y_l,+-m = sqrt(2 (l-m)!/(l+m)!) P_l^m(xi) {cos, sin}(m phi), no Condon-Shortley phase."""
    omega = np.atleast_2d(np.asarray(omega, dtype=np.float64))
    mu, eta, xi = omega[:, 0], omega[:, 1], omega[:, 2]
    phi = np.arctan2(eta, mu)
    s = np.sqrt(np.maximum(0.0, 1.0 - xi * xi))
    Y = np.zeros((omega.shape[0], (L + 1) ** 2))
    P = {}
    for m in range(L + 1):
        dfact = 1.0
        for t in range(1, 2 * m, 2):
            dfact *= t                                              # (2m-1)!!
        P[(m, m)] = dfact * s ** m
        if m + 1 <= L:
            P[(m + 1, m)] = xi * (2 * m + 1) * P[(m, m)]
        for l in range(m + 2, L + 1):
            P[(l, m)] = ((2 * l - 1) * xi * P[(l - 1, m)] - (l + m - 1) * P[(l - 2, m)]) / (l - m)
    for l in range(L + 1):
        Y[:, l * l + l] = P[(l, 0)]
        for m in range(1, l + 1):
            nrm = math.sqrt(2.0 * math.factorial(l - m) / math.factorial(l + m))
            Y[:, l * l + l + m] = nrm * P[(l, m)] * np.cos(m * phi)
            Y[:, l * l + l - m] = nrm * P[(l, m)] * np.sin(m * phi)
    return Y


def l_of_lm(L):
    return np.array([l for l in range(L + 1) for _ in range(2 * l + 1)])


def projection_tables(L, omega, w):
    """Mtab [n][nm] = (2l+1)/(4 pi) Y_lm(Omega_n)  (moment -> direction, Eq. 2 rhs in moment form R3/R5)
       Dtab [nm][n] = w_n Y_lm(Omega_n)            (direction -> moment, Eq. 3)"""
    Y = real_sph_harm(L, omega)
    ll = l_of_lm(L)
    Mtab = Y * ((2 * ll + 1) / (4.0 * math.pi))[None, :]
    Dtab = (Y * w[:, None]).T.copy()
    return np.ascontiguousarray(Mtab), np.ascontiguousarray(Dtab)


# --------------------------------------------------------------------------------------
# Schedule
# --------------------------------------------------------------------------------------
def wavefront_size(nx, ny, nz, S):
    """P(S), Eqs. (9)-(22), straight from the formulas (python ints)."""
    tri = lambda d: d * (d + 1) // 2
    pos = lambda v: max(v, 0)
    return (tri(S + 1) - tri(pos(S + 1 - nx)) - tri(pos(S + 1 - ny)) - tri(pos(S + 1 - nz))
            + tri(pos(S + 1 - nx - ny)) + tri(pos(S + 1 - ny - nz)) + tri(pos(S + 1 - nx - nz)))


def schedule(nx, ny, nz, octant):
    """plane_offset [planes+1], cell_of [cells] (int32) in Table 1 order, mirrored per octant."""
    planes = nx + ny + nz - 2
    off = np.zeros(planes + 1, dtype=np.int32)
    cell_of = np.zeros(nx * ny * nz, dtype=np.int32)
    _lib().orc_schedule(nx, ny, nz, octant, _p(off, ctypes.c_int32), _p(cell_of, ctypes.c_int32))
    for S in range(planes):                                        # Eq. (9) asserted against Eq. (8)
        assert off[S + 1] - off[S] == _lib().orc_wavefront_size(nx, ny, nz, S)
    return off, cell_of


# --------------------------------------------------------------------------------------
# Sweep and ray trace (C)
# --------------------------------------------------------------------------------------
def sweep(nx, ny, nz, dx, dy, dz, sigt, Q, omega, w, Mtab, Dtab, closure=0, order=0,
          want_psi=False, threads=None):
    """One sweep of Eq. (2) over all directions.  Q, returned phi: [nm][cells] float64."""
    cells = nx * ny * nz
    nm = Q.shape[0]
    ndir = omega.shape[0]
    sigt = np.ascontiguousarray(sigt, dtype=np.float64).reshape(-1)
    Q = np.ascontiguousarray(Q, dtype=np.float64).reshape(nm, cells)
    phi = np.zeros((nm, cells))
    leak = ctypes.c_double(0.0)
    nfix = ctypes.c_int64(0)
    psi = np.zeros((ndir, cells)) if want_psi else None
    _lib().orc_sweep(nx, ny, nz, ctypes.c_double(dx), ctypes.c_double(dy), ctypes.c_double(dz),
                     _p(sigt), _p(Q), nm, ndir, _p(np.ascontiguousarray(omega)), _p(np.ascontiguousarray(w)),
                     _p(Mtab), _p(Dtab), closure, order, _p(phi), ctypes.byref(leak),
                     _p(psi) if want_psi else None, ctypes.byref(nfix),
                     threads or default_threads())
    return phi, leak.value, psi, nfix.value


def raytrace(wl, src, want_areal=False, threads=None):
    """phi_u [G][cells] for one point / cone / fan source (Eq. 4; readings R11, R12, R18)."""
    cells = wl.cells
    phi_u = np.zeros((wl.G, cells))
    areal = np.zeros((wl.n_materials, cells)) if want_areal else None
    rho = np.ascontiguousarray(wl.density, dtype=np.float64).reshape(-1)
    mat = np.ascontiguousarray(wl.material, dtype=np.uint8).reshape(-1)
    pos = np.array(src.pos, dtype=np.float64)
    axis = np.array(src.axis, dtype=np.float64)
    spec = np.ascontiguousarray(src.spectrum, dtype=np.float64)
    fan_n, sin_half2 = np.zeros(3), 0.0
    if src.kind == 3:
        # unit normal of the fan plane: the part of `up` perpendicular to the beam axis
        a = axis / np.linalg.norm(axis)
        up = np.array(src.up, dtype=np.float64)
        fan_n = up - np.dot(up, a) * a
        fan_n = fan_n / np.linalg.norm(fan_n)
        sin_half2 = math.sin(src.half_angle2)
    _lib().orc_raytrace(wl.nx, wl.ny, wl.nz, ctypes.c_double(wl.dx), ctypes.c_double(wl.dy), ctypes.c_double(wl.dz),
                        _p(mat, ctypes.c_uint8), _p(rho), wl.n_materials, wl.G,
                        _p(np.ascontiguousarray(wl.sigma_t, dtype=np.float64)),
                        src.kind, _p(pos), _p(axis), ctypes.c_double(math.cos(src.half_angle)),
                        _p(spec), _p(phi_u), _p(areal) if want_areal else None,
                        threads or default_threads(), _p(np.ascontiguousarray(fan_n)), ctypes.c_double(sin_half2))
    return (phi_u, areal) if want_areal else phi_u


def unit_dirs_from(wl, pos):
    """u_c = (r_c - r_s)/|r_c - r_s| for every cell centre, [cells][3]."""
    x = (np.arange(wl.nx) + 0.5) * wl.dx - wl.nx * wl.dx / 2.0
    y = (np.arange(wl.ny) + 0.5) * wl.dy - wl.ny * wl.dy / 2.0
    z = (np.arange(wl.nz) + 0.5) * wl.dz - wl.nz * wl.dz / 2.0
    Z, Yc, X = np.meshgrid(z, y, x, indexing="ij")
    d = np.stack([X.reshape(-1) - pos[0], Yc.reshape(-1) - pos[1], Z.reshape(-1) - pos[2]], axis=1)
    return d / np.linalg.norm(d, axis=1, keepdims=True)


# --------------------------------------------------------------------------------------
# Multigroup source iteration (PAPER.md:34 Eq. 2, :44-62 Eqs. 4-7, :149, :183)
# --------------------------------------------------------------------------------------
def solve(wl, closure=0, fixed_iters=None, threads=None, keep_history=False, order=0, store_dtype=np.float64, progress=None,
          raytrace_threads=None):
    """Whole hot path for a Workload.  Returns a dict:
         phi     [n_prob][G][nm][cells]  collided flux moments (float64)
         phi_u   [n_src][G][cells]       uncollided scalar flux (zeros for kind 0)
         iters   [n_prob][G], residual [n_prob][G], balance [n_prob][G][3] (source, collision, leakage
                 of the LAST sweep: sum Q_00 V = sum sigt phi_0 V + leakage)
         seconds dict: wall time spent in the ray trace, the fixed-source assembly and the sweeps (for bench.py)
       n_prob = n_src (mode 0) or 1 (mode 1, sources summed: linearity of Eq. 4-6).
       fixed_iters: None -> wl.fixed_iters (0 = run to wl.tol); int or [n_prob][G] array -> replay.
       store_dtype: type in which the moments of FINISHED groups are held (they feed the downscatter source of the
       groups below).  float64 everywhere except the config-4 goldens (tests/golden/make_goldens.py), where 47 groups
       x 16 moments x 8.4 M cells would take 50 GB per source: float32 there (relative rounding 6e-8, three orders
       below the 1e-4 gate; the iteration of the current group is always float64).
       progress: None or a callable (problem, group, sweeps, delta) called after every finished group (logging only).
       raytrace_threads: threads of the ray trace alone (default = threads; bench.py times the sweeps on one thread
       without waiting for a one-thread ray trace; results do not depend on any thread count)."""
    import time
    cells, G, L = wl.cells, wl.G, wl.L
    nm = (L + 1) ** 2
    ll = l_of_lm(L)
    omega, w = level_symmetric(wl.sn)
    Mtab, Dtab = projection_tables(L, omega, w)
    rho = np.ascontiguousarray(wl.density, dtype=np.float64).reshape(-1)
    mat = np.ascontiguousarray(wl.material).reshape(-1).astype(np.int64)
    V = wl.dx * wl.dy * wl.dz
    n_src = len(wl.sources)
    probs = [[s] for s in range(n_src)] if wl.mode == 0 else [list(range(n_src))]
    if fixed_iters is None:
        fixed_iters = wl.fixed_iters
    fi = np.broadcast_to(np.asarray(fixed_iters), (len(probs), G))
    seconds = dict(raytrace=0.0, fixed_source=0.0, sweep=0.0)

    # step 4: uncollided flux per source (Eq. 4) and its direction moments Y_lm(u_c)
    t0 = time.perf_counter()
    phi_u = np.zeros((n_src, G, cells))
    Yu = [None] * n_src
    for s, src in enumerate(wl.sources):
        if src.kind in (1, 2, 3):
            phi_u[s] = raytrace(wl, src, threads=raytrace_threads or threads)
            Yu[s] = real_sph_harm(L, unit_dirs_from(wl, src.pos)).T.copy()        # [nm][cells]
    seconds["raytrace"] = time.perf_counter() - t0

    out_phi = np.zeros((len(probs), G, nm, cells), dtype=store_dtype)
    iters = np.zeros((len(probs), G), dtype=np.int64)
    resid = np.zeros((len(probs), G))
    balance = np.zeros((len(probs), G, 3))
    history = [[[] for _ in range(G)] for _ in probs]
    lm_of = [slice(l * l, (l + 1) * (l + 1)) for l in range(L + 1)]              # moments lm of degree l
    for p, members in enumerate(probs):
        for g in range(G):                                                      # high -> low energy (R7)
            t0 = time.perf_counter()
            sigt = rho * wl.sigma_t[mat, g]
            # step 5 / row a2: fixed source = external + first-collision (Eq. 5) + downscatter (Eq. 2 rhs, g' < g),
            # moment lm of degree l:  rho(c) s_l[mat(c)][g' -> g] * {phi_u^{g'}(c) Y_lm(u_c)  |  phi_lm^{g'}(c)}
            fixed = np.zeros((nm, cells))
            for s in members:
                src = wl.sources[s]
                if src.kind == 0:
                    fixed[0] += np.asarray(src.volume[g], dtype=np.float64).reshape(-1)
                else:
                    for gp in range(g + 1):
                        ru = rho * phi_u[s, gp]
                        for l in range(L + 1):
                            fixed[lm_of[l]] += (ru * wl.sigma_s[:, l, gp, g][mat])[None, :] * Yu[s][lm_of[l]]
            for gp in range(g):
                for l in range(L + 1):
                    fixed[lm_of[l]] += (rho * wl.sigma_s[:, l, gp, g][mat])[None, :] * out_phi[p, gp, lm_of[l]]
            s_self = rho[None, :] * wl.sigma_s[:, :, g, g][mat][:, ll].T          # [nm][cells]
            seconds["fixed_source"] += time.perf_counter() - t0
            # step 6 / row a6: source iteration from phi = 0 (R9)
            phi = np.zeros((nm, cells))
            k = 0
            while True:
                k += 1
                Q = s_self * phi + fixed
                t0 = time.perf_counter()
                phi_new, leak, _, _ = sweep(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, sigt, Q,
                                            omega, w, Mtab, Dtab, closure, order, threads=threads)
                seconds["sweep"] += time.perf_counter() - t0
                mx = np.abs(phi_new[0]).max()
                delta = 0.0 if mx == 0.0 else np.abs(phi_new[0] - phi[0]).max() / mx   # R8
                phi = phi_new
                if keep_history:
                    history[p][g].append(delta)
                if mx == 0.0:
                    break
                if fi[p, g] > 0:
                    if k >= fi[p, g]:
                        break
                elif delta < wl.tol or k >= wl.max_iters:
                    break
            out_phi[p, g] = phi
            iters[p, g] = k
            resid[p, g] = delta
            balance[p, g] = (Q[0].sum() * V, (sigt * phi[0]).sum() * V, leak)
            if progress is not None:
                progress(p, g, k, delta)
    res = dict(phi=out_phi, phi_u=phi_u, iters=iters, residual=resid, balance=balance,
               omega=omega, w=w, seconds=seconds)
    if keep_history:
        res["history"] = history
    return res


def response(res, wl, problem, resp, include_uncollided=True):
    """Post-processing hook ("conversion of photon fluence to an absorbed dose"): a response per
    group folded with the scalar fluence of one problem of `res` = solve(wl, ...):
        D(cell) = sum_g resp[g] * (phi_00,g(cell) + sum over the problem's sources of phi_u,g(cell)).
    The total fluence of the first-collision method is collided + uncollided.  Written out as the
    definition: one term per group, in group order, float64.  Pins (tests/test_oracle_sweep.py): a unit response returns
    the group's fluence itself, linearity in the response, and in a mode-1 (summed sources) problem the uncollided part is
    the sum over all sources."""
    resp = np.asarray(resp, dtype=np.float64)
    nsrc = len(wl.sources)
    srcs = range(nsrc) if wl.mode == 1 else [problem]
    out = np.zeros(res["phi"].shape[-1], dtype=np.float64)
    for g in range(wl.G):
        f = res["phi"][problem, g, 0].copy()
        if include_uncollided:
            for s_ in srcs:
                f += res["phi_u"][s_, g]
        out += resp[g] * f
    return out

