"""The five BASELINE.json configs as concrete arrays.

Everything here is an INPUT a DOCTORS user supplies through the GUI tabs
(PAPER.md:155-165): mesh + material map + density, multigroup sigma_t and P_l
scattering tables (per unit density, g = 0 is the highest energy), S_N order,
sources.  No transport arithmetic lives here.
"""
from dataclasses import dataclass, field
import numpy as np
from .rng import uniform01, normal01

BASE_SEED = 1910113350
CONFIG_NAMES = ["cfg0_8c_S2P0", "cfg1_32c_sphere_S8P3", "cfg2_64c_cyl_S8P3",
                "cfg3_128x128x64_S16P3", "cfg4_256x256x128_S8P3_8src"]

# materials: 0 air, 1 lung, 2 water, 3 bone
DENSITY = np.array([0.0012, 0.3, 1.0, 1.85])
A0 = np.array([4468.0, 4468.0, 4468.0, 22000.0])     # keV^3 cm^2/g  (photo-electric-like)
B0 = np.array([0.1605, 0.1605, 0.1605, 0.170])       # cm^2/g        (scatter-like)


@dataclass
class SourceSpec:
    kind: int                       # 0 volume (isotropic), 1 point (isotropic), 2 cone, 3 fan
    pos: tuple = (0.0, 0.0, 0.0)
    axis: tuple = (1.0, 0.0, 0.0)
    half_angle: float = 0.0         # radians (kind 2: cone half angle; kind 3: azimuthal half angle in the fan plane)
    spectrum: np.ndarray = None     # [G] photons per group (kinds 1, 2, 3)
    volume: np.ndarray = None       # [G][nz][ny][nx] float32 photons/cm^3 (kind 0)
    up: tuple = (0.0, 0.0, 1.0)     # kind 3: a vector out of the fan plane
    half_angle2: float = 0.0        # kind 3: polar half angle out of the fan plane


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    material: np.ndarray            # uint8 [nz][ny][nx]
    density: np.ndarray             # float32 [nz][ny][nx]
    n_materials: int
    G: int
    L: int
    sn: int
    sigma_t: np.ndarray             # float64 [n_mat][G], per unit density
    sigma_s: np.ndarray             # float64 [n_mat][L+1][G_from][G_to], per unit density
    sources: list = field(default_factory=list)
    mode: int = 0                   # 0 independent (batched), 1 summed into one problem
    tol: float = 1e-5
    max_iters: int = 100
    fixed_iters: int = 0            # >0: exactly this many sweeps per (source, group)
    energies: np.ndarray = None     # [G] keV bin midpoints (informational)

    @property
    def cells(self):
        return self.nx * self.ny * self.nz

    @property
    def n_dir(self):
        return self.sn * (self.sn + 2)


def cell_centres(n, d):
    """Mesh centred on the origin: x_i = (i + 1/2) d - n d / 2."""
    return (np.arange(n) + 0.5) * d - n * d / 2.0


def energy_grid(G, e_lo, e_hi):
    """G equal bins on [e_lo, e_hi]; midpoints; g = 0 is the top bin."""
    w = (e_hi - e_lo) / G
    return e_hi - (np.arange(G) + 0.5) * w


def make_xs(seed, G, L, e_lo, e_hi, n_mat=4):
    """sigma_t = a E^-3 + b with seeded 5 % jitter; downscatter-only P_L matrix."""
    E = energy_grid(G, e_lo, e_hi)
    m = np.arange(n_mat, dtype=np.uint64)
    a = A0[:n_mat] * (1.0 + 0.05 * (2.0 * uniform01(seed * 8 + 1, 2 * m) - 1.0))
    b = B0[:n_mat] * (1.0 + 0.05 * (2.0 * uniform01(seed * 8 + 1, 2 * m + np.uint64(1)) - 1.0))
    sig_t = a[:, None] * E[None, :] ** -3 + b[:, None]                       # [m][g]
    if G > 1:
        c = 0.3 + 0.6 * (E - E[-1]) / (E[0] - E[-1])                         # [g'] rises with energy
    else:
        c = np.array([0.6])
    sig_s = np.zeros((n_mat, L + 1, G, G))
    for gp in range(G):
        d = np.arange(G - gp)
        wgt = 0.5 ** d
        wgt = wgt / wgt.sum()
        for l in range(L + 1):
            sig_s[:, l, gp, gp:] = (0.3 ** l) * c[gp] * sig_t[:, gp, None] * wgt[None, :]
    return E, sig_t, sig_s


def _cyl_phantom(nx, ny, nz, d):
    """Config 2/3: water cylinder r=12 with two bone (r=2) and one lung (r=3) inserts, along z."""
    x = cell_centres(nx, d)[None, :]
    y = cell_centres(ny, d)[:, None]
    mat2 = np.zeros((ny, nx), dtype=np.uint8)
    mat2[x ** 2 + y ** 2 <= 12.0 ** 2] = 2
    mat2[(x + 6.0) ** 2 + y ** 2 <= 2.0 ** 2] = 3
    mat2[(x - 4.0) ** 2 + (y - 6.0) ** 2 <= 2.0 ** 2] = 3
    mat2[(x - 3.0) ** 2 + (y + 5.0) ** 2 <= 3.0 ** 2] = 1
    return np.broadcast_to(mat2[None], (nz, ny, nx)).copy()


def _grf_phantom(seed, nx, ny, nz):
    """Config 4: thresholded, periodically blurred white noise (sigma = 6 voxels, +-24 taps)."""
    from scipy.ndimage import convolve1d
    f = normal01(seed * 8 + 3, nx * ny * nz).reshape(nz, ny, nx)
    t = np.arange(-24, 25, dtype=np.float64)
    k = np.exp(-0.5 * (t / 6.0) ** 2)
    k /= k.sum()
    for axis in (2, 1, 0):                       # x, y, z
        f = convolve1d(f, k, axis=axis, mode="wrap")
    f = (f - f.mean()) / f.std()
    mat = np.full(f.shape, 3, dtype=np.uint8)
    mat[f < 1.2] = 2
    mat[f < 0.0] = 1
    mat[f < -0.5] = 0
    return mat


def make_config(idx, n_sources=None):
    """Workload for BASELINE.json configs[idx]."""
    seed = BASE_SEED + idx
    if idx == 0:
        n = 8
        mat = np.zeros((n, n, n), dtype=np.uint8)
        rho = np.ones((n, n, n), dtype=np.float32)
        vol = np.zeros((1, n, n, n), dtype=np.float32)
        vol[0, 3:5, 3:5, 3:5] = 1.0
        return Workload(CONFIG_NAMES[0], n, n, n, 1.0, 1.0, 1.0, mat, rho, 1, 1, 0, 2,
                        np.array([[0.20]]), np.array([[[[0.18]]]]),
                        [SourceSpec(kind=0, volume=vol)], fixed_iters=10,
                        energies=np.array([50.0]))
    if idx == 1:
        n, d, G, L = 32, 0.5, 19, 3
        E, st, ss = make_xs(seed, G, L, 10.0, 100.0)
        x = cell_centres(n, d)
        r2 = x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2
        mat = np.where(r2 <= 36.0, 2, 0).astype(np.uint8)
        rho = DENSITY[mat].astype(np.float32)
        src = [SourceSpec(kind=1, pos=(-20.0, 0.0, 0.0), spectrum=np.full(G, 1.0 / G))]
        return Workload(CONFIG_NAMES[1], n, n, n, d, d, d, mat, rho, 4, G, L, 8, st, ss, src, energies=E)
    if idx in (2, 3):
        G, L = 19, 3
        E, st, ss = make_xs(seed, G, L, 10.0, 120.0)
        if idx == 2:
            nx, ny, nz, d, sn = 64, 64, 64, 0.5, 8
        else:
            nx, ny, nz, d, sn = 128, 128, 64, 0.25, 16
        mat = _cyl_phantom(nx, ny, nz, d)
        rho64 = DENSITY[mat]
        if idx == 3:
            c = np.arange(nx * ny * nz, dtype=np.uint64)
            rho64 = rho64 * (1.0 + 0.05 * (2.0 * uniform01(seed * 8 + 2, c).reshape(nz, ny, nx) - 1.0))
        src = [SourceSpec(kind=2, pos=(-50.0, 0.0, 0.0), axis=(1.0, 0.0, 0.0),
                          half_angle=np.deg2rad(15.0), spectrum=np.full(G, 1.0 / G))]
        return Workload(CONFIG_NAMES[idx], nx, ny, nz, d, d, d, mat, rho64.astype(np.float32),
                        4, G, L, sn, st, ss, src, energies=E)
    if idx == 4:
        nx, ny, nz, G, L = 256, 256, 128, 47, 3
        d = 50.0 / 256.0
        E, st, ss = make_xs(seed, G, L, 10.0, 140.0)
        mat = _grf_phantom(seed, nx, ny, nz)
        rho = DENSITY[mat].astype(np.float32)
        ns = 8 if n_sources is None else n_sources
        src = []
        for s in range(ns):
            th = 2.0 * np.pi * s / 8.0
            p = (50.0 * np.cos(th), 50.0 * np.sin(th), 0.0)
            src.append(SourceSpec(kind=2, pos=p, axis=(-np.cos(th), -np.sin(th), 0.0),
                                  half_angle=np.deg2rad(15.0), spectrum=np.full(G, 1.0 / G)))
        return Workload(CONFIG_NAMES[4], nx, ny, nz, d, d, d, mat, rho, 4, G, L, 8, st, ss, src, energies=E)
    raise ValueError("config index 0..4")


def single_sweep_case(idx, groups=(0, 1), n_sources=1, fixed_iters=2):
    """Full-size mesh of config idx restricted to a few groups and a fixed sweep count.

    Used for parity at BASELINE's full sizes where the whole multigroup oracle
    run would take hours: the sweep kernel sees the full mesh, quadrature and
    launch configuration; only the group list is shortened.
    """
    w = make_config(idx, n_sources=n_sources) if idx == 4 else make_config(idx)
    g = np.asarray(groups)
    w.sigma_t = np.ascontiguousarray(w.sigma_t[:, g])
    w.sigma_s = np.ascontiguousarray(w.sigma_s[:, :, g][:, :, :, g])
    w.energies = w.energies[g]
    w.G = len(g)
    for s in w.sources:
        if s.spectrum is not None:
            s.spectrum = np.ascontiguousarray(s.spectrum[g])
        if s.volume is not None:
            s.volume = np.ascontiguousarray(s.volume[g])
    w.sources = w.sources[:n_sources]
    w.fixed_iters = fixed_iters
    w.name += "_g" + "_".join(str(int(i)) for i in g) + "_k%d" % fixed_iters
    return w


def paper_shaped(fine=False, ct=False, G=90):
    """the paper's own workload shape.

    50 x 50 x 12.5 cm box, 35 cm water cylinder, 64x64x16 (or 256x256x64) voxels,
    G groups of 1 keV on 10-100 keV, S6 P0.  Single projection: isotropic point
    source above the phantom.  CT scan: 16 cone beams (30 deg full angle) on a
    ring, summed into ONE problem (mode 1).  Synthetic XS (the 90-group NJOY
    library is not in the container).
    """
    seed = BASE_SEED + 10
    nx, ny, nz = (256, 256, 64) if fine else (64, 64, 16)
    d = 50.0 / nx
    E, st, ss = make_xs(seed, G, 0, 10.0, 100.0)
    x = cell_centres(nx, d)[None, :]
    y = cell_centres(ny, d)[:, None]
    mat2 = np.where(x ** 2 + y ** 2 <= 17.5 ** 2, 2, 0).astype(np.uint8)
    mat = np.broadcast_to(mat2[None], (nz, ny, nx)).copy()
    rho = DENSITY[mat].astype(np.float32)
    spec = np.full(G, 1.0 / G)
    if not ct:
        src = [SourceSpec(kind=1, pos=(0.0, 30.0, 0.0), spectrum=spec)]
        mode = 0
    else:
        src = []
        for s in range(16):
            th = 2.0 * np.pi * s / 16.0
            src.append(SourceSpec(kind=2, pos=(30.0 * np.cos(th), 30.0 * np.sin(th), 0.0),
                                  axis=(-np.cos(th), -np.sin(th), 0.0),
                                  half_angle=np.deg2rad(15.0), spectrum=spec))
        mode = 1
    name = "paper_%s_%s_S6P0" % ("fine" if fine else "coarse", "ct16" if ct else "single")
    return Workload(name, nx, ny, nz, d, d, d, mat, rho, 4, G, 0, 6, st, ss, src, mode=mode, energies=E)
