"""Thin ctypes binding of include/doctors_b200.h — argument marshalling only.

Every step of the path (ray trace, fixed source, sweep, projections, source iteration,
convergence) runs inside libdoctors_b200.so; this module converts numpy arrays to pointers,
asks torch for the device workspace and the stream, and unpacks the info struct.  There is no
CPU fallback: if the library is missing or no CUDA device is present, calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdoctors_b200.so")

OK, INVALID_ARG, BAD_STATE, ALLOC, CUDA, NOT_CONVERGED, NOT_RETAINED = range(7)
STATUS_NAMES = ["OK", "INVALID_ARG", "BAD_STATE", "ALLOC", "CUDA", "NOT_CONVERGED", "NOT_RETAINED"]

EXPORTS = [
    "doctors_version", "doctors_abi_sizes", "doctors_create_problem", "doctors_destroy_problem", "doctors_last_error",
    "doctors_set_mesh_materials", "doctors_set_xs", "doctors_set_quadrature", "doctors_set_quadrature_points",
    "doctors_get_quadrature", "doctors_set_source", "doctors_n_problems", "doctors_workspace_bytes",
    "doctors_set_workspace", "doctors_solve", "doctors_get_flux_moments", "doctors_get_uncollided_flux", "doctors_get_response",
    "doctors_debug_schedule_dims", "doctors_debug_get_schedule", "doctors_debug_device_brick_steps", "doctors_wavefront_size", "doctors_debug_get_tables",
    "doctors_host_level_symmetric", "doctors_host_schedule", "doctors_host_projection_tables",
    "doctors_host_pl_exceeds_quadrature", "doctors_convergence_delta_no_alloc",
]


class DoctorsError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("%s: %s" % (STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else status, text))
        self.status = status


class CSource(C.Structure):
    _fields_ = [("kind", C.c_int), ("pos", C.c_double * 3), ("axis", C.c_double * 3),
                ("half_angle_rad", C.c_double), ("spectrum", C.POINTER(C.c_double)),
                ("volume", C.POINTER(C.c_float)), ("up", C.c_double * 3), ("half_angle2_rad", C.c_double)]


class CSolveOpts(C.Structure):
    _fields_ = [("tol", C.c_double), ("max_iters", C.c_int), ("fixed_iters", C.POINTER(C.c_int)),
                ("closure", C.c_int), ("deterministic", C.c_int), ("source_chunk", C.c_int),
                ("sweep_mode", C.c_int), ("brick", C.c_int * 3), ("ctas_per_sm", C.c_int),
                ("check_window", C.c_int), ("projection", C.c_int)]


class CSolveInfo(C.Structure):
    _fields_ = [("iters", C.POINTER(C.c_int)), ("residual", C.POINTER(C.c_double)),
                ("balance", C.POINTER(C.c_double)),
                ("ms_raytrace", C.c_double), ("ms_fixed_source", C.c_double), ("ms_sweep", C.c_double),
                ("ms_iterate", C.c_double), ("ms_total", C.c_double),
                ("updates", C.c_ulonglong), ("sweep_launches", C.c_ulonglong), ("kernel_launches", C.c_ulonglong),
                ("n_chunks", C.c_int), ("brick", C.c_int * 3), ("ctas_per_sm", C.c_int),
                ("sweep_kernel", C.c_int), ("projection_mtiles", C.c_int),
                ("timed_sweeps", C.c_ulonglong), ("pl_exceeds_quadrature", C.c_int)]


_lib = None


def load_library():
    """dlopen the in-tree library and declare the signatures.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libdoctors_b200.so is not built: run `python -m paper_1910_11335_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, ip, dp, fp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double), C.POINTER(C.c_float)
    L.doctors_version.restype = C.c_char_p
    L.doctors_abi_sizes.argtypes = [C.POINTER(C.c_int)]
    L.doctors_abi_sizes.restype = None
    sizes = (C.c_int * 3)()
    L.doctors_abi_sizes(sizes)
    mine = (C.sizeof(CSource), C.sizeof(CSolveOpts), C.sizeof(CSolveInfo))
    if tuple(sizes) != mine:
        raise ImportError("libdoctors_b200.so was built from another include/doctors_b200.h: struct sizes %s, binding %s"
                          % (tuple(sizes), mine))
    L.doctors_create_problem.argtypes = [C.c_int, vp, C.POINTER(vp)]
    L.doctors_destroy_problem.argtypes = [vp]
    L.doctors_destroy_problem.restype = None
    L.doctors_last_error.argtypes = [vp]
    L.doctors_last_error.restype = C.c_char_p
    L.doctors_set_mesh_materials.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                             C.POINTER(C.c_uint8), fp, C.c_int]
    L.doctors_set_xs.argtypes = [vp, C.c_int, C.c_int, C.c_int, dp, dp]
    L.doctors_set_quadrature.argtypes = [vp, C.c_int]
    L.doctors_set_quadrature_points.argtypes = [vp, C.c_int, dp, dp]
    L.doctors_get_quadrature.argtypes = [vp, ip, dp, dp]
    L.doctors_set_source.argtypes = [vp, C.c_int, C.POINTER(CSource), C.c_int]
    L.doctors_n_problems.argtypes = [vp]
    L.doctors_workspace_bytes.argtypes = [vp, C.POINTER(CSolveOpts)]
    L.doctors_workspace_bytes.restype = C.c_size_t
    L.doctors_set_workspace.argtypes = [vp, vp, C.c_size_t]
    L.doctors_solve.argtypes = [vp, C.POINTER(CSolveOpts), C.POINTER(CSolveInfo)]
    L.doctors_get_flux_moments.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, C.c_int]
    L.doctors_get_uncollided_flux.argtypes = [vp, C.c_int, C.c_int, vp, C.c_int]
    L.doctors_get_response.argtypes = [vp, C.c_int, dp, C.c_int, vp, C.c_int]
    L.doctors_debug_schedule_dims.argtypes = [vp, C.POINTER(CSolveOpts), C.c_int, ip]
    L.doctors_debug_get_schedule.argtypes = [vp, C.POINTER(CSolveOpts), C.c_int, C.c_int,
                                             C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    L.doctors_debug_device_brick_steps.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int32)]
    L.doctors_wavefront_size.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int]
    L.doctors_wavefront_size.restype = C.c_longlong
    L.doctors_debug_get_tables.argtypes = [vp, C.c_int, dp, dp]
    L.doctors_host_level_symmetric.argtypes = [C.c_int, dp, dp]
    L.doctors_host_schedule.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    L.doctors_host_projection_tables.argtypes = [C.c_int, C.c_int, dp, dp, dp, dp]
    L.doctors_host_pl_exceeds_quadrature.argtypes = [C.c_int, C.c_int, dp, dp, dp]
    L.doctors_convergence_delta_no_alloc.argtypes = [vp, vp, vp, C.c_longlong, C.c_longlong, C.c_int, vp]
    _lib = L
    return L


def _ptr(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def wavefront_size(nx, ny, nz, S):
    return int(load_library().doctors_wavefront_size(nx, ny, nz, S))


def host_level_symmetric(N):
    """The library's built-in LQ_N generator (host code, no device needed)."""
    n = N * (N + 2)
    omega, w = np.zeros((n, 3)), np.zeros(n)
    rc = load_library().doctors_host_level_symmetric(N, _ptr(omega, C.c_double), _ptr(w, C.c_double))
    if rc != OK:
        raise DoctorsError(rc, "unsupported S_N order %d" % N)
    return omega, w


def host_schedule(nx, ny, nz, octant):
    """The library's sub-sweep schedule generator (host code)."""
    off = np.zeros(nx + ny + nz - 1, dtype=np.int32)
    cells = np.zeros(nx * ny * nz, dtype=np.int32)
    rc = load_library().doctors_host_schedule(nx, ny, nz, octant, _ptr(off, C.c_int32), _ptr(cells, C.c_int32))
    if rc != OK:
        raise DoctorsError(rc, "bad schedule arguments")
    return off, cells


def host_projection_tables(L, omega, w):
    omega = np.ascontiguousarray(omega, dtype=np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    nm = (L + 1) ** 2
    M, D = np.zeros((len(w), nm)), np.zeros((len(w), nm))
    rc = load_library().doctors_host_projection_tables(L, len(w), _ptr(omega, C.c_double), _ptr(w, C.c_double),
                                                       _ptr(M, C.c_double), _ptr(D, C.c_double))
    if rc != OK:
        raise DoctorsError(rc, "bad table arguments")
    return M, D


def host_pl_exceeds_quadrature(L, omega, w):
    """(flag, defect): does P_L ask for more than the quadrature integrates exactly?  (host code)"""
    omega = np.ascontiguousarray(omega, dtype=np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    d = C.c_double()
    rc = load_library().doctors_host_pl_exceeds_quadrature(L, len(w), _ptr(omega, C.c_double), _ptr(w, C.c_double), C.byref(d))
    if rc < 0:
        raise DoctorsError(INVALID_ARG, "bad arguments")
    return bool(rc), d.value


class Problem:
    """One doctors_problem handle.  Method names follow the C ABI (doctors_<name>)."""

    def __init__(self, device=0, stream=None):
        import torch
        self._torch = torch
        self._L = load_library()
        if not torch.cuda.is_available():
            raise DoctorsError(CUDA, "no CUDA device: this library has no CPU path")
        self.device = device
        torch.cuda.set_device(device)
        if stream is None:
            stream = torch.cuda.current_stream(device)
        self._stream = stream
        h = C.c_void_p()
        rc = self._L.doctors_create_problem(device, C.c_void_p(stream.cuda_stream), C.byref(h))
        if rc != OK:
            raise DoctorsError(rc, "doctors_create_problem failed")
        self._h = h
        self._ws = None
        self._keep = []
        self.G = self.L = 0
        self.shape = None

    def close(self):
        if getattr(self, "_h", None):
            self._L.doctors_destroy_problem(self._h)
            self._h = None
        self._ws = None

    __del__ = close

    def _check(self, rc, allow=()):
        if rc != OK and rc not in allow:
            raise DoctorsError(rc, self._L.doctors_last_error(self._h).decode())
        return rc

    # ---- set_* ------------------------------------------------------------------------------
    def set_mesh_materials(self, material, density, pitch, n_materials):
        material = np.ascontiguousarray(material, dtype=np.uint8)
        nz, ny, nx = material.shape
        dens_p = None
        if density is not None:
            density = np.ascontiguousarray(density, dtype=np.float32)
            assert density.shape == material.shape
            dens_p = _ptr(density, C.c_float)
        self._check(self._L.doctors_set_mesh_materials(self._h, nx, ny, nz, pitch[0], pitch[1], pitch[2],
                                                       _ptr(material, C.c_uint8), dens_p, n_materials))
        self.shape = (nz, ny, nx)

    def set_xs(self, sigma_t, sigma_s):
        sigma_t = np.ascontiguousarray(sigma_t, dtype=np.float64)
        sigma_s = np.ascontiguousarray(sigma_s, dtype=np.float64)
        n_mat, G = sigma_t.shape
        L = sigma_s.shape[1] - 1
        assert sigma_s.shape == (n_mat, L + 1, G, G)
        self._check(self._L.doctors_set_xs(self._h, n_mat, G, L, _ptr(sigma_t, C.c_double), _ptr(sigma_s, C.c_double)))
        self.G, self.L = G, L

    def set_quadrature(self, sn_order):
        self._check(self._L.doctors_set_quadrature(self._h, sn_order))

    def set_quadrature_points(self, omega, w):
        omega = np.ascontiguousarray(omega, dtype=np.float64)
        w = np.ascontiguousarray(w, dtype=np.float64)
        self._check(self._L.doctors_set_quadrature_points(self._h, len(w), _ptr(omega, C.c_double), _ptr(w, C.c_double)))

    def get_quadrature(self):
        n = C.c_int()
        self._check(self._L.doctors_get_quadrature(self._h, C.byref(n), None, None))
        omega = np.zeros((n.value, 3))
        w = np.zeros(n.value)
        self._check(self._L.doctors_get_quadrature(self._h, C.byref(n), _ptr(omega, C.c_double), _ptr(w, C.c_double)))
        return omega, w

    def set_source(self, sources, mode=0):
        """sources: iterable of objects with kind, pos, axis, half_angle, spectrum, volume (workloads.SourceSpec)."""
        arr = (CSource * len(sources))()
        keep = []
        for i, s in enumerate(sources):
            arr[i].kind = int(s.kind)
            arr[i].pos = (C.c_double * 3)(*[float(v) for v in s.pos])
            arr[i].axis = (C.c_double * 3)(*[float(v) for v in s.axis])
            arr[i].half_angle_rad = float(s.half_angle)
            arr[i].up = (C.c_double * 3)(*[float(v) for v in getattr(s, "up", (0.0, 0.0, 1.0))])
            arr[i].half_angle2_rad = float(getattr(s, "half_angle2", 0.0))
            if s.spectrum is not None:
                sp = np.ascontiguousarray(s.spectrum, dtype=np.float64)
                keep.append(sp)
                arr[i].spectrum = _ptr(sp, C.c_double)
            if s.volume is not None:
                vol = np.ascontiguousarray(s.volume, dtype=np.float32)
                keep.append(vol)
                arr[i].volume = _ptr(vol, C.c_float)
        self._check(self._L.doctors_set_source(self._h, len(sources), arr, mode))

    def n_problems(self):
        return int(self._L.doctors_n_problems(self._h))

    # ---- solve ------------------------------------------------------------------------------
    def _opts(self, tol=1e-5, max_iters=100, fixed_iters=None, closure=0, deterministic=0, source_chunk=0,
              sweep_mode=0, brick=None, ctas_per_sm=0, check_window=0, projection=0):
        o = CSolveOpts()
        o.tol, o.max_iters, o.closure, o.deterministic = tol, max_iters, closure, deterministic
        o.source_chunk, o.sweep_mode, o.ctas_per_sm, o.check_window = source_chunk, sweep_mode, ctas_per_sm, check_window
        o.projection = projection
        if brick is not None:
            o.brick = (C.c_int * 3)(*brick)
        fi = None
        if fixed_iters is not None:
            fi = np.ascontiguousarray(np.broadcast_to(np.asarray(fixed_iters, dtype=np.int32),
                                                      (self.n_problems(), self.G)))
            o.fixed_iters = _ptr(fi, C.c_int)
        return o, fi

    def workspace_bytes(self, **kw):
        o, _fi = self._opts(**kw)
        n = int(self._L.doctors_workspace_bytes(self._h, C.byref(o)))
        if n == 0:
            raise DoctorsError(BAD_STATE, self._L.doctors_last_error(self._h).decode())
        return n

    def set_workspace(self, nbytes):
        """Ask torch for the device memory (torch owns it) and hand it to the library."""
        torch = self._torch
        if self._ws is None or self._ws.numel() < nbytes:
            self._ws = None
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda:%d" % self.device)
        self._check(self._L.doctors_set_workspace(self._h, C.c_void_p(self._ws.data_ptr()), self._ws.numel()))

    def solve(self, **kw):
        """doctors_solve.  Returns a dict with iters, residual, balance and the info scalars."""
        o, fi = self._opts(**kw)
        need = self.workspace_bytes(**kw)
        if self._ws is None or self._ws.numel() < need:
            self.set_workspace(need)
        npb, G = self.n_problems(), self.G
        iters = np.zeros((npb, G), dtype=np.int32)
        resid = np.zeros((npb, G))
        bal = np.zeros((npb, G, 3))
        info = CSolveInfo()
        info.iters, info.residual, info.balance = _ptr(iters, C.c_int), _ptr(resid, C.c_double), _ptr(bal, C.c_double)
        rc = self._check(self._L.doctors_solve(self._h, C.byref(o), C.byref(info)), allow=(NOT_CONVERGED,))
        return dict(status=rc, iters=iters, residual=resid, balance=bal,
                    ms_raytrace=info.ms_raytrace, ms_fixed_source=info.ms_fixed_source, ms_sweep=info.ms_sweep,
                    ms_iterate=info.ms_iterate, ms_total=info.ms_total, updates=int(info.updates),
                    sweep_launches=int(info.sweep_launches), kernel_launches=int(info.kernel_launches),
                    n_chunks=info.n_chunks, brick=tuple(info.brick), ctas_per_sm=info.ctas_per_sm,
                    projection_mtiles=info.projection_mtiles, sweep_kernel=info.sweep_kernel,
                    timed_sweeps=int(info.timed_sweeps), pl_exceeds_quadrature=int(info.pl_exceeds_quadrature))

    # ---- get_* ------------------------------------------------------------------------------
    def get_flux_moments(self, problem, group, l_max=0, out=None):
        """Host numpy [(l_max+1)^2][nz][ny][nx] float32, or fill a torch CUDA tensor passed as `out`."""
        nm = (l_max + 1) ** 2
        if out is None:
            host = np.empty((nm,) + self.shape, dtype=np.float32)
            self._check(self._L.doctors_get_flux_moments(self._h, problem, group, l_max, C.c_void_p(host.ctypes.data), 0))
            return host
        if isinstance(out, np.ndarray):
            assert out.dtype == np.float32 and out.flags.c_contiguous and out.size == nm * int(np.prod(self.shape))
            self._check(self._L.doctors_get_flux_moments(self._h, problem, group, l_max, C.c_void_p(out.ctypes.data), 0))
            return out
        assert out.is_cuda and out.is_contiguous() and out.numel() == nm * int(np.prod(self.shape))
        self._check(self._L.doctors_get_flux_moments(self._h, problem, group, l_max, C.c_void_p(out.data_ptr()), 1))
        return out

    def get_flux_moments_into(self, problem, group, l_max, host_ptr):
        """Raw-pointer variant (pinned host buffers of the bench's e2e leg)."""
        self._check(self._L.doctors_get_flux_moments(self._h, problem, group, l_max, C.c_void_p(host_ptr), 0))

    def get_uncollided_flux(self, source, group):
        host = np.empty(self.shape, dtype=np.float32)
        self._check(self._L.doctors_get_uncollided_flux(self._h, source, group, C.c_void_p(host.ctypes.data), 0))
        return host

    def get_response(self, problem, response, include_uncollided=True):
        """doctors_get_response: sum_g response[g] * fluence_g of one problem, dense [nz][ny][nx] fp32."""
        r = np.ascontiguousarray(response, dtype=np.float64)
        if r.shape != (self.G,):
            raise ValueError("response must have G = %d entries" % self.G)
        host = np.empty(self.shape, dtype=np.float32)
        self._check(self._L.doctors_get_response(self._h, problem, _ptr(r, C.c_double), int(bool(include_uncollided)),
                                                 C.c_void_p(host.ctypes.data), 0))
        return host

    def convergence_delta_no_alloc(self, phi_new_ptr, phi_old_ptr, n_cells, problem_stride, n_problems, out_ptr):
        """doctors_convergence_delta_no_alloc: raw DEVICE pointers in and out (e.g. tensor.data_ptr()); enqueues on the
        handle's stream, allocates nothing, does not synchronise."""
        self._check(self._L.doctors_convergence_delta_no_alloc(self._h, C.c_void_p(phi_new_ptr), C.c_void_p(phi_old_ptr),
                                                               int(n_cells), int(problem_stride), int(n_problems), C.c_void_p(out_ptr)))

    # ---- test hooks -------------------------------------------------------------------------
    def debug_schedule(self, octant, level, brick=None):
        o, _ = self._opts(brick=brick)
        dims = (C.c_int * 3)()
        self._check(self._L.doctors_debug_schedule_dims(self._h, C.byref(o), level, dims))
        d = tuple(dims)
        off = np.zeros(d[0] + d[1] + d[2] - 1, dtype=np.int32)
        cells = np.zeros(d[0] * d[1] * d[2], dtype=np.int32)
        self._check(self._L.doctors_debug_get_schedule(self._h, C.byref(o), octant, level,
                                                       _ptr(off, C.c_int32), _ptr(cells, C.c_int32)))
        return d, off, cells

    def debug_device_brick_steps(self, brick, octant):
        """Step at which the sweep kernel updates each cell of one full brick: int32 [bz][by][bx]."""
        bx, by, bz = brick
        out = np.full(bx * by * bz, -1, dtype=np.int32)
        self._check(self._L.doctors_debug_device_brick_steps(self._h, bx, by, bz, octant, _ptr(out, C.c_int32)))
        return out.reshape(bz, by, bx)

    def debug_tables(self, pl_order):
        om, w = self.get_quadrature()
        nm = (pl_order + 1) ** 2
        M = np.zeros((len(w), nm))
        D = np.zeros((len(w), nm))
        self._check(self._L.doctors_debug_get_tables(self._h, pl_order, _ptr(M, C.c_double), _ptr(D, C.c_double)))
        return M, D


def problem_from_workload(wl, device=0, stream=None):
    """Feed a workloads.Workload through the set_* calls."""
    p = Problem(device, stream)
    p.set_mesh_materials(wl.material, wl.density, (wl.dx, wl.dy, wl.dz), wl.n_materials)
    p.set_xs(wl.sigma_t, wl.sigma_s)
    p.set_quadrature(wl.sn)
    p.set_source(wl.sources, wl.mode)
    return p
