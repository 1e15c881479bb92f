"""pimpc_rprim2_noalloc (include/pimpc.h): the allocation-free entry point against the existing path
(pimpc_get -> pimpc_result.r_prim2).  Collected last on purpose (the suite runs with `pytest -x`);
passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_2601_14414_b200 import workloads as wl

pytestmark = pytest.mark.gpu

RTOL = 1e-12          # the tolerance the result-record tests use for sums of the same double-accumulated terms
NP = {"f64": np.float64, "f32": np.float32}


@pytest.fixture(scope="module")
def pimpc():
    from paper_2601_14414_b200 import pimpc as m
    m.load()
    return m


def _existing_path(pimpc, p, dtype, engine, iters):
    """Solve with the handle API; returns pimpc_result.r_prim2 and the device copies of everything the new call reads."""
    import torch
    s = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype=dtype, engine=engine, rho=p.rho)
    s.set_problem(p)
    s.solve(iters, 0.0)
    _, _, _, res = s.get()
    st = {n: s.get_state(n) for n in ("X", "DU", "Z", "V") + (("D",) if p.du_lo is not None else ())}
    s.close()
    dev = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a, NP[dtype])).cuda()
    args = dict(A=dev(p.A), B=dev(p.B), e=dev(p.e), x0=dev(p.x0), u_prev=dev(p.u_prev), X=dev(st["X"]), DU=dev(st["DU"]),
                Z=dev(st["Z"]), V=dev(st["V"]), D=dev(st.get("D")))
    return res["r_prim2"].copy(), args


def _call(pimpc, p, dtype, a, out):
    pimpc.rprim2_noalloc(dtype, p.nx, p.nu, p.N, p.batch, a["A"], a["B"], a["e"], a["x0"], a["u_prev"], a["X"], a["DU"],
                         a["Z"], a["V"], a["D"], p.rho, out)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_rprim2_noalloc_matches_pimpc_get_on_calls_in_a_row(pimpc, dtype):
    import torch
    # problem 1: 2 partial sums per instance (N (nx+nu) = 4800 rows), Delta-u box; problem 2: one partial, no box, no e
    p1 = wl.random_ltv(12, 4, 300, 3, seed=7, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5)
    p2 = wl.random_ltv(5, 3, 9, 2, seed=8, affine=False, u_prev=False, bounds=0.6)
    ref1, a1 = _existing_path(pimpc, p1, dtype, "auto", 60)
    ref2, a2 = _existing_path(pimpc, p2, dtype, "staged", 40)
    assert (ref1 > 0).all() and (ref2 > 0).all()
    o1 = torch.full((p1.batch,), float("nan"), dtype=torch.float64, device="cuda")
    o2 = torch.full((p2.batch,), float("nan"), dtype=torch.float64, device="cuda")
    o3 = torch.full((p1.batch,), float("nan"), dtype=torch.float64, device="cuda")
    _call(pimpc, p2, dtype, a2, o2)          # first use in the process: the driver loads the module (and the array) now
    torch.cuda.synchronize()
    o2.fill_(float("nan"))
    free0 = torch.cuda.mem_get_info()[0]
    _call(pimpc, p1, dtype, a1, o1)          # back to back on one stream: the shared scratch still holds the
    _call(pimpc, p2, dtype, a2, o2)          # partials of the call before
    _call(pimpc, p1, dtype, a1, o3)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0             # nothing was allocated on the device by the three calls
    np.testing.assert_allclose(o1.cpu().numpy(), ref1, rtol=RTOL, atol=0.0)
    np.testing.assert_allclose(o2.cpu().numpy(), ref2, rtol=RTOL, atol=0.0)
    assert torch.equal(o1, o3)               # same launch shape, same order: the same bits


def test_rprim2_noalloc_chunks_capped_by_the_static_scratch(pimpc):
    """batch x partials beyond PIMPC_NOALLOC_MAX_PARTS: fewer partials per instance, same sums (against the definition
    of the consensus residuals, written with torch fp64 ops on the same arrays)."""
    import torch
    nx, nu, N, batch, rho = 2, 1, 1400, 20000, 0.7          # 4200 rows -> 2 partials wanted, 40000 > 32768 -> 1
    nb = nx + nu
    assert batch * ((N * nb) // 2048) > pimpc.NOALLOC_MAX_PARTS >= batch
    g = torch.Generator(device="cuda").manual_seed(5)
    r = lambda *s: torch.randn(*s, generator=g, device="cuda", dtype=torch.float32)
    A, B, e, x0, up = r(batch, N, nx, nx), r(batch, N, nx, nu), r(batch, N, nx), r(batch, nx), r(batch, nu)
    X, Z, V, DU, D = r(batch, N, nb), r(batch, N, nb), r(batch, N, nb), r(batch, N, nu), r(batch, N, nu)
    out = torch.full((batch,), float("nan"), dtype=torch.float64, device="cuda")
    pimpc.rprim2_noalloc("f32", nx, nu, N, batch, A, B, e, x0, up, X, DU, Z, V, D, rho, out)
    d = lambda t: t.double()
    xprev = torch.cat([torch.cat([d(x0), d(up)], 1)[:, None, :], d(X)[:, :-1, :]], 1)           # xbar_k, k = 0..N-1
    Abar = torch.cat([torch.cat([d(A), d(B)], 3),
                      torch.cat([torch.zeros(batch, N, nu, nx, device="cuda", dtype=torch.float64),
                                 torch.eye(nu, device="cuda", dtype=torch.float64).expand(batch, N, nu, nu)], 3)], 2)
    axk = torch.einsum("bkij,bkj->bki", Abar, xprev)
    axk[:, :, :nx] += d(e)
    bdu = torch.cat([torch.einsum("bkij,bkj->bki", d(B), d(DU)), d(DU)], 2)
    tot = ((d(X) - d(Z)) ** 2).sum((1, 2)) + ((bdu - d(V)) ** 2).sum((1, 2)) + ((d(Z) - axk - d(V)) ** 2).sum((1, 2)) \
        + ((d(DU) - d(D)) ** 2).sum((1, 2))
    torch.cuda.synchronize()
    np.testing.assert_allclose(out.cpu().numpy(), (rho * tot).cpu().numpy(), rtol=1e-11, atol=0.0)


def test_rprim2_noalloc_rejects_sizes_beyond_the_scratch_and_bad_arguments(pimpc):
    import torch
    t = torch.zeros(64, dtype=torch.float64, device="cuda")
    big = pimpc.NOALLOC_MAX_PARTS + 1
    with pytest.raises(pimpc.PimpcError) as ei:              # rejected before anything is launched or dereferenced
        pimpc.rprim2_noalloc("f64", 2, 1, 4, big, t, t, None, t, None, t, t, t, t, None, 1.0, t)
    assert ei.value.code == pimpc.EINVAL and "PIMPC_NOALLOC_MAX_PARTS" in str(ei.value)
    with pytest.raises(pimpc.PimpcError) as ei:
        pimpc.rprim2_noalloc("f64", 2, 1, 4, 1, t, t, None, t, None, t, t, None, t, None, 1.0, t)     # Z missing
    assert ei.value.code == pimpc.EINVAL
    with pytest.raises(pimpc.PimpcError) as ei:
        pimpc.rprim2_noalloc(7, 2, 1, 4, 1, t, t, None, t, None, t, t, t, t, None, 1.0, t)            # dtype
    assert ei.value.code == pimpc.EINVAL
    torch.cuda.synchronize()
