"""bie_gmres_noalloc (include/bie.h): the stored-matrix GMRES solve whose workspace is a static device array inside the
library, for callers that must not call cudaMalloc.  Checked against the existing path (bie_gmres with a caller-supplied
workspace) on two calls in a row, with the tolerances of tests/test_gpu_parity.py.  Collected last on purpose (the name):
the suite runs with pytest -x.
"""
import numpy as np
import pytest

from paper_2108_01786_b200 import inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_X = 1e-10          # GMRES solutions, tests/test_gpu_parity.py
BIE_ERR_NOALLOC_SIZE = -9


@pytest.fixture(scope="module")
def ctx():
    from paper_2108_01786_b200 import bie
    assert torch.cuda.is_available(), "the gpu tests need a B200"
    c = bie.Context(0)
    yield c
    c.close()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def build(ctx, g):
    n = g.n
    A = torch.empty((n, n + (n & 1)), dtype=torch.float64, device="cuda")
    ctx.bie_build(g.counts, g.kinds, dev(g.zeta), dev(g.dzeta), dev(g.d2zeta), A)
    return A


def outputs(n):
    return (torch.empty(n + (n & 1), dtype=torch.float64, device="cuda"),
            torch.full((2,), -7, dtype=torch.int32, device="cuda"),
            torch.full((1,), -7.0, dtype=torch.float64, device="cuda"))


def reference(ctx, A, b, P):
    """the existing path: bie_gmres with a workspace the caller allocated"""
    from paper_2108_01786_b200 import bie
    n = b.numel()
    ws = torch.empty(bie.Context.bie_gmres_workspace_bytes(n, P.restart), dtype=torch.uint8, device="cuda")
    x, oi, of = outputs(n)
    ctx.bie_gmres(A, b, x[:n], P.tol, P.restart, P.max_iters, ws, oi, of)
    torch.cuda.synchronize()
    return x[:n].cpu().numpy(), int(oi[0]), int(oi[1]), float(of[0])


def test_noalloc_matches_bie_gmres_on_two_calls_in_a_row(ctx):
    from paper_2108_01786_b200 import bie
    # config 3 (n = 4608, restart 50, 76 iterations: one restart) then config 1 (n = 640): the second call finds the
    # larger solve's contents in the shared scratch array
    cases = []
    for c in (3, 1):
        P = inputs.make_config(c)
        g = P.geometry
        assert bie.Context.bie_gmres_workspace_bytes(g.n, P.restart) <= bie.Context.bie_gmres_noalloc_max_bytes()
        A = build(ctx, g)
        b = dev(P.rhs[0])
        cases.append((P, A, b, reference(ctx, A, b, P), outputs(g.n)))
    # warm-up call: the first launch on a device loads the module and looks the array's address up
    P, A, b, _, (x, oi, of) = cases[1]
    ctx.bie_gmres_noalloc(A, b, x[:b.numel()], P.tol, P.restart, P.max_iters, oi, of)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    # the two calls, back to back on one stream, nothing in between
    for P, A, b, _, (x, oi, of) in cases:
        ctx.bie_gmres_noalloc(A, b, x[:b.numel()], P.tol, P.restart, P.max_iters, oi, of)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "the no-alloc entry point took device memory"
    for P, A, b, (xr, itr, str_, rrr), (x, oi, of) in cases:
        n = b.numel()
        xs = x[:n].cpu().numpy()
        assert int(oi[1]) == 0 and str_ == 0
        assert int(oi[0]) == itr                      # same kernel, same plan, fixed-order reductions
        assert np.linalg.norm(xs - xr) / np.linalg.norm(xr) <= TOL_X
        assert float(of[0]) <= 10 * P.tol and rrr <= 10 * P.tol


def test_noalloc_rejects_sizes_beyond_the_scratch(ctx):
    from paper_2108_01786_b200 import bie
    L = bie.lib()
    n, restart = 16384, 100                            # 13 MB of workspace: beyond the 4 MiB array
    assert bie.Context.bie_gmres_workspace_bytes(n, restart) > bie.Context.bie_gmres_noalloc_max_bytes()
    d = torch.zeros(16, dtype=torch.float64, device="cuda")      # never touched: the size check comes first
    oi = torch.full((2,), -7, dtype=torch.int32, device="cuda")
    rc = L.bie_gmres_noalloc(ctx._h, n, d.data_ptr(), n, d.data_ptr(), 1e-13, restart, 10, d.data_ptr(), oi.data_ptr(),
                             None, oi.data_ptr() + 4, None)
    torch.cuda.synchronize()
    assert rc == BIE_ERR_NOALLOC_SIZE
    assert oi.tolist() == [-7, -7]                     # nothing was launched
    assert b"static scratch" in L.bie_strerror(rc)
    with pytest.raises(bie.BieError):
        # through the binding
        P = inputs.make_config(2)
        A = build(ctx, P.geometry)
        b = dev(P.rhs[0])
        x, oi2, of = outputs(b.numel())
        # restart far beyond what fits: the Krylov basis alone would need n * (restart + 1) * 8 bytes
        ctx.bie_gmres_noalloc(A, b, x[:b.numel()], P.tol, 2000, 10, oi2, of)
