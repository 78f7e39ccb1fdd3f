"""doctors_convergence_delta_no_alloc — the allocation-free entry point (scratch in a static __device__ array) against the
existing path (`-m gpu`; collected last on purpose: the suite runs with pytest -x).

Existing path: doctors_solve evaluates delta_k = max|phi0^k - phi0^(k-1)| / max|phi0^k| on the device after every sweep (k_check,
scratch in the caller's workspace) and reports the last one as info["residual"].  Here the same two iterates are fetched through
the public API — a solve that replays K sweeps of group g and one that replays K - 1, in deterministic mode, which is
bit-reproducible — handed to the new entry point as device tensors, and its delta must equal the solver's own, on two calls in a
row (two groups), then on a third, batched call; the static scratch keeps the previous call's contents in between.
"""
import numpy as np
import pytest

from tests.parity_util import tiny_p3_case

pytestmark = pytest.mark.gpu
TOL = 1e-4          # the gate of the parity tests; the two paths do the same fp32 arithmetic, so they agree far inside it
K = 5


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1910_11335_b200 import build
    build.build()
    import paper_1910_11335_b200 as p
    p.load_library()
    return p


def _solve(pkg, wl, fixed):
    p = pkg.problem_from_workload(wl)
    info = p.solve(tol=wl.tol, max_iters=wl.max_iters, fixed_iters=np.asarray(fixed, dtype=np.int32)[None, :], closure=1,
                   deterministic=1)
    phi0 = [p.get_flux_moments(0, g, 0)[0].copy() for g in range(wl.G)]
    return p, info, phi0


def test_no_alloc_delta_matches_the_solver_on_consecutive_calls(pkg):
    import torch
    wl = tiny_p3_case(kind=2)
    assert wl.G == 3
    p, info, new = _solve(pkg, wl, [K, K, K])
    want = info["residual"][0]                                   # the solver's own delta_K per group (existing path)
    assert (want > 0).all() and (want < 1.0).all()
    old = []
    for g in (0, 1):                                             # phi0^(K-1) of group g: same history above g, one sweep less in g
        fixed = [K, K, K]
        fixed[g] = K - 1
        q, _, ph = _solve(pkg, wl, fixed)
        old.append(ph[g])
        q.close()
    n = wl.cells
    out = torch.full((3,), -1.0, dtype=torch.float32, device="cuda")
    got = []
    for g in (0, 1):                                             # two calls in a row on the shared static scratch
        a = torch.from_numpy(new[g].reshape(-1)).cuda()
        b = torch.from_numpy(old[g].reshape(-1)).cuda()
        p.convergence_delta_no_alloc(a.data_ptr(), b.data_ptr(), n, n, 1, out.data_ptr())
        torch.cuda.synchronize()
        res = out.cpu().numpy().astype(np.float64)
        got.append(res)
        assert abs(res[0] - want[g]) <= 1e-6 * want[g] and abs(res[0] - want[g]) < TOL * want[g], (g, res, want[g])
        d = np.abs(new[g].astype(np.float64) - old[g].astype(np.float64)).max()
        m = np.abs(new[g]).max()
        assert abs(res[1] - d) <= 1e-6 * d and res[2] == np.float32(m), (g, res, d, m)
    assert got[0][0] != got[1][0]                                # two different answers: nothing carried over
    # third call, batched: both problems at once (stride > n_cells), results in one go
    stride = n + 7
    A = torch.zeros(2 * stride, dtype=torch.float32, device="cuda")
    B = torch.zeros(2 * stride, dtype=torch.float32, device="cuda")
    for g in (0, 1):
        A[g * stride:g * stride + n] = torch.from_numpy(new[g].reshape(-1)).cuda()
        B[g * stride:g * stride + n] = torch.from_numpy(old[g].reshape(-1)).cuda()
    out2 = torch.full((6,), -1.0, dtype=torch.float32, device="cuda")
    p.convergence_delta_no_alloc(A.data_ptr(), B.data_ptr(), n, stride, 2, out2.data_ptr())
    torch.cuda.synchronize()
    r2 = out2.cpu().numpy().astype(np.float64).reshape(2, 3)
    assert np.array_equal(r2[0], got[0]) and np.array_equal(r2[1], got[1])
    # identical inputs -> 0; all-zero input -> 0 (no source reaches the group, reading R8)
    p.convergence_delta_no_alloc(A.data_ptr(), A.data_ptr(), n, stride, 2, out2.data_ptr())
    torch.cuda.synchronize()
    assert (out2.cpu().numpy().reshape(2, 3)[:, :2] == 0).all()
    Z = torch.zeros(n, dtype=torch.float32, device="cuda")
    p.convergence_delta_no_alloc(Z.data_ptr(), Z.data_ptr(), n, n, 1, out.data_ptr())
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == 0).all()
    # beyond the stated maximum: refused with a clear error, nothing launched
    with pytest.raises(pkg.DoctorsError) as e:
        p.convergence_delta_no_alloc(A.data_ptr(), B.data_ptr(), 16, 16, 65, out2.data_ptr())
    assert e.value.status == pkg.INVALID_ARG and "at most 64" in str(e.value)
    with pytest.raises(pkg.DoctorsError):
        p.convergence_delta_no_alloc(0, B.data_ptr(), n, n, 1, out.data_ptr())
    p.close()
