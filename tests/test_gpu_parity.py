"""GPU parity tests: libpimpc (through the C ABI / ctypes binding) vs the CPU oracle, element by
element on the same seeded inputs (tests/parity.py).  Every test here needs a B200: `-m gpu`."""
import os

import numpy as np
import pytest

from paper_2601_14414_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu

ENGINES_SMALL = ["staged", "auto"]


@pytest.fixture(scope="module")
def pimpc():
    from paper_2601_14414_b200 import pimpc as m
    m.load()
    return m


def _golden():
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "p_tiny.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            out[k] = np.array([float(t) for t in v])
    return out


# ---- the paper-independent golden numbers, directly against the CUDA path ---------------------
@pytest.mark.parametrize("engine", ENGINES_SMALL)
def test_p_tiny_golden_numbers_on_gpu(pimpc, engine):
    g = _golden()
    r = parity.gpu_run(pimpc, wl.p_tiny(False), "f64", engine=engine, iters=10, tol=0.0)
    np.testing.assert_allclose(r["c_hist"][0], g["c_nodu"], rtol=1e-10)
    assert list(r["acc_hist"][0]) == [int(v) for v in g["acc_nodu"]]
    np.testing.assert_allclose(r["DU"].ravel(), g["du10_nodu"], atol=2e-11)
    np.testing.assert_allclose(r["Z"][0, 0], g["z0_10_nodu"], atol=2e-11)
    r = parity.gpu_run(pimpc, wl.p_tiny(True), "f64", engine=engine, iters=5, tol=0.0)
    np.testing.assert_allclose(r["c_hist"][0], g["c_du"], rtol=1e-10)


# ---- the five configs of BASELINE.json ----------------------------------------------------------
@pytest.mark.parametrize("engine", ENGINES_SMALL)
def test_config1_fp64_500_iterations(oracle, pimpc, engine):
    p = wl.config1()
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine=engine)
    assert int(g["res"]["iters"][0]) == 500
    parity.check_properties(p, "f64", g)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("engine", ENGINES_SMALL)
def test_config2_full(oracle, pimpc, dtype, engine):
    p = wl.config2()                      # N=100, tol 1e-4 or 2000 iterations (hits the cap)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine=engine)
    parity.check_properties(p, dtype, g)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2_tol_path_stops_early(oracle, pimpc, dtype):
    p = wl.quadrotor_ltv(10, 1, iters=2000, tol=1e-4, rho=10.0, name="C2-tol")
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype)
    assert int(g["res"]["converged"][0]) == 1 and int(g["res"]["iters"][0]) < 2000


@pytest.mark.parametrize("N", [10, 100, 1000])
def test_config3_horizons_fp32(oracle, pimpc, N):
    p = wl.config3(N)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f32")
    parity.check_properties(p, "f32", g)


@pytest.mark.parametrize("N", [4000, 10000])
def test_config3_long_horizons_fp32(oracle, pimpc, N):
    p = wl.config3(N)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f32")
    parity.check_properties(p, "f32", g)


def test_config4_full_batch_sampled_instances(oracle, pimpc):
    """Full 4096-instance batch in the launch configuration bench.py times; the oracle checks a
    seeded sample of instances one by one (instances are independent), properties cover the rest."""
    p = wl.config4()
    g = parity.gpu_run(pimpc, p, "f32")
    assert np.all(g["res"]["iters"] == 200)
    parity.check_properties(p, "f32", g)
    sample = np.random.default_rng(4).choice(p.batch, size=48, replace=False)
    sample = sorted(set(sample.tolist()) | {0, 147, 148, p.batch - 1})
    nrep = 0
    for b in sample:
        w, r = parity.check_instance(oracle, p, "f32", g, b)
        nrep += int(r)
    assert nrep <= 4


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config5_small_all_instances(oracle, pimpc, dtype):
    p = wl.config5(N=37, batch=3)         # several tiles + ragged tail of the wide-state shape
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype)
    parity.check_properties(p, dtype, g)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config5_full_size_sampled(oracle, pimpc, dtype):
    p = wl.config5()                      # N=2000, batch=64, 500 iterations
    g = parity.gpu_run(pimpc, p, dtype)
    assert np.all(g["res"]["iters"] == 500)
    parity.check_properties(p, dtype, g)
    for b in (0, 63):
        parity.check_instance(oracle, p, dtype, g, b)


# ---- STREAM engine (persistent cooperative grid, bulk-copy ring): ranges that split instances ------
@pytest.fixture
def stream_grid(monkeypatch):
    def set_(n):
        if n:
            monkeypatch.setenv("PIMPC_STREAM_GRID", str(n))
        else:
            monkeypatch.delenv("PIMPC_STREAM_GRID", raising=False)
    return set_


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [0, 1, 3, 7])
@pytest.mark.parametrize("shape", [(48, 12, 37, 3), (12, 4, 41, 2), (4, 2, 23, 5)])
def test_stream_engine_all_options(oracle, pimpc, stream_grid, shape, grid, dtype):
    """grid = 0: one or two steps per CTA (every step a halo); 1: one CTA owns everything; 3, 7: ranges
    start inside instances and span several of them."""
    nx, nu, N, batch = shape
    stream_grid(grid)
    p = wl.random_ltv(nx, nu, N, batch, seed=nx * 10 + N, affine=True, u_prev=True, full_cost=True, wdu=True,
                      qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="stream", iters=120, tol=0.0)
    assert g["info"]["engine"] == pimpc.ENGINE_STREAM
    parity.check_properties(p, dtype, g)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [0, 3])
@pytest.mark.parametrize("shape", [(10, 3, 17, 2), (20, 6, 9, 2), (30, 10, 7, 1), (50, 15, 5, 2)])
def test_stream_engine_paper_table1_shapes(oracle, pimpc, stream_grid, shape, grid, dtype):
    """The (n, m) of the paper's Table I, odd nb included (circulant storage of H without a
    self-paired diagonal); AUTO must pick STREAM for them."""
    nx, nu, N, batch = shape
    stream_grid(grid)
    p = wl.random_ltv(nx, nu, N, batch, seed=nx * 7 + N, affine=True, u_prev=True, full_cost=True, wdu=True,
                      qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="auto", iters=100, tol=0.0)
    assert g["info"]["engine"] == pimpc.ENGINE_STREAM
    parity.check_properties(p, dtype, g)


@pytest.mark.parametrize("grid", [0, 5])
def test_stream_engine_unbounded_and_plain_admm(oracle, pimpc, stream_grid, grid):
    stream_grid(grid)
    p = wl.random_ltv(4, 2, 9, 2, seed=77, affine=True, bounds=None, du_bound=None)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="stream", iters=300, tol=0.0)
    assert "D" not in g
    p = wl.quadrotor_ltv(12, 2, iters=120, tol=0.0)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="stream", eta=0.0)
    assert np.all(g["res"]["restarts"] == 120)


@pytest.mark.parametrize("grid", [0, 4])
def test_stream_engine_early_stop_and_warm_start(oracle, pimpc, stream_grid, grid):
    stream_grid(grid)
    p = wl.quadrotor_ltv(8, 6, iters=3000, tol=1e-4, rho=10.0, name="tolbatch")
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="stream")
    assert len(set(g["res"]["iters"].tolist())) > 1 and np.all(g["res"]["converged"] == 1)
    p = wl.quadrotor_ltv(9, 2, iters=40, tol=0.0)
    s = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f64", engine="stream")
    s.set_problem(p); s.solve(40)
    warm = {k: s.get_state(k) for k in ("Z", "V", "TH", "BE", "LA", "D", "DE")}
    s.solve(25)
    z2 = s.get_state("Z")
    for b in range(p.batch):
        o = parity.oracle_run(oracle, p, "f64", b, iters=25, tol=0.0, warm=warm)
        assert parity.relerr(z2[b], o.Z) <= 1e-9


# ---- COOP engine (batch 1, horizon spread over the SMs, tagged-word exchange instead of grid barriers) ------
@pytest.fixture
def coop_env(monkeypatch):
    def set_(grid=0, spg=0, cluster=None):
        for name, v in (("PIMPC_COOP_GRID", grid), ("PIMPC_COOP_SPG", spg)):
            if v:
                monkeypatch.setenv(name, str(v))
            else:
                monkeypatch.delenv(name, raising=False)
        if cluster is None:                       # default: one cluster (DSMEM exchange) for short horizons
            monkeypatch.delenv("PIMPC_COOP_CLUSTER", raising=False)
        else:                                     # 0: exchange through L2 (the long-horizon path); n: cluster of n CTAs
            monkeypatch.setenv("PIMPC_COOP_CLUSTER", str(cluster))
    return set_


@pytest.mark.parametrize("cluster", [None, 0, 8])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [0, 1, 2, 7])
@pytest.mark.parametrize("shape", [(12, 4, 41), (4, 2, 23), (12, 4, 150), (4, 2, 1), (12, 4, 2)])
def test_coop_engine_all_options(oracle, pimpc, coop_env, shape, grid, dtype, cluster):
    """grid = 0: one stage per CTA while N <= 148 (every stage has two ghosts); 1: a single CTA, no exchange;
    2, 7: ragged ranges.  All optional terms on."""
    nx, nu, N = shape
    if N > 100 and grid in (1, 2):
        grid += 4                         # 150 stages of (12, 4) do not fit one or two CTAs' shared memory: 5, 6 CTAs
    coop_env(grid, cluster=cluster)
    p = wl.random_ltv(nx, nu, N, 1, seed=nx * 10 + N, affine=True, u_prev=True, full_cost=True, wdu=True,
                      qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="coop", iters=120, tol=0.0)
    assert g["info"]["engine"] == pimpc.ENGINE_COOP
    parity.check_properties(p, dtype, g)


@pytest.mark.parametrize("cluster", [None, 0])
@pytest.mark.parametrize("grid", [3, 0])
def test_coop_engine_two_stages_per_group_fp32(oracle, pimpc, coop_env, grid, cluster):
    coop_env(grid, spg=2, cluster=cluster)
    p = wl.random_ltv(12, 4, 100, 1, seed=5, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f32", engine="coop", iters=150, tol=0.0)
    assert g["info"]["engine"] == pimpc.ENGINE_COOP


@pytest.mark.parametrize("cluster", [None, 0])
@pytest.mark.parametrize("grid", [0, 5])
def test_coop_engine_unbounded_plain_admm_early_stop_warm_start(oracle, pimpc, coop_env, grid, cluster):
    coop_env(grid, cluster=cluster)
    p = wl.random_ltv(4, 2, 9, 1, seed=77, affine=True, bounds=None, du_bound=None)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="coop", iters=300, tol=0.0)
    assert "D" not in g
    p = wl.quadrotor_ltv(12, 1, iters=120, tol=0.0)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="coop", eta=0.0)
    assert np.all(g["res"]["restarts"] == 120)
    p = wl.quadrotor_ltv(10, 1, iters=2000, tol=1e-4, rho=10.0, name="C2-tol")
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="coop")
    assert int(g["res"]["converged"][0]) == 1 and int(g["res"]["iters"][0]) < 2000
    p = wl.quadrotor_ltv(30, 1, iters=40, tol=0.0)
    s = pimpc.Solver(p.nx, p.nu, p.N, 1, dtype="f64", engine="coop")
    s.set_problem(p); s.solve(40)
    warm = {k: s.get_state(k) for k in ("Z", "V", "TH", "BE", "LA", "D", "DE")}
    s.solve(25)
    o = parity.oracle_run(oracle, p, "f64", 0, iters=25, tol=0.0, warm=warm)
    assert parity.relerr(s.get_state("Z")[0], o.Z) <= 1e-9


# ---- NEXT row f1: receding-horizon stepping with shift warm start ----------------
@pytest.mark.parametrize("engine", ["auto", "coop", "stream", "staged"])
def test_closed_loop_cstr_shift_warm_start(oracle, pimpc, engine):
    """Four MPC steps of the online-linearised CSTR: per step new stage data (set_stages + a0), pimpc_shift(1) of the
    previous iterates, K iterations; the plant advances with the oracle's u_0.  The CUDA path runs the (2, 1)
    problem embedded in the (4, 2) shape (workloads.pad_problem), the oracle the original one."""
    N, K, T = 60, 120, 4
    x = np.array(wl.CSTR["x_init"]); u = np.array([wl.CSTR["u_init"]]); t = 0.0
    s = pimpc.Solver(4, 2, N, 1, dtype="f64", engine=engine, history=K)
    real = [0, 1, 4]
    warm = None
    for step in range(T):
        p = wl.cstr_problem(x, u, t, N, iters=K)
        s.set_problem(wl.pad_problem(p, 4, 2))
        if step:
            s.shift(1)
        s.solve(K)
        o = oracle.solve(**p.instance(0), max_iters=K, tol=0.0, warm=None if warm is None else oracle.shift_warm(warm, 1))
        c, acc = s.get_history()
        assert list(acc[0]) == list(o.acc_hist)
        np.testing.assert_allclose(c[0], o.c_hist, rtol=1e-7)
        for name in ("Z", "V", "TH", "BE", "LA", "X"):
            g = s.get_state(name)[0]
            assert parity.relerr(g[:, real], getattr(o, name)) <= 1e-9, (step, name)
            assert float(np.max(np.abs(np.delete(g, real, axis=1)))) == 0.0          # the embedding stays exactly zero
        xg, ug, dug, res = s.get()
        assert parity.relerr(ug[0, :, :1], o.u) <= 1e-9 and parity.relerr(dug[0, :, :1], o.DU) <= 1e-9
        warm = dict(Z=o.Z, V=o.V, TH=o.TH, BE=o.BE, LA=o.LA)
        u = o.u[0].copy()
        x = wl.cstr_plant_step(x, u, t); t += wl.CSTR["Ts"]
    assert x[0] < wl.CSTR["x_init"][0]                    # the loop moves C_A towards the reference


def test_shift_argument_validation_and_identity(pimpc):
    p = wl.quadrotor_ltv(12, 2, iters=30, tol=0.0)
    s = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f32"); s.set_problem(p); s.solve(30)
    z = s.get_state("Z"); th = s.get_state("TH"); d = s.get_state("D")
    s.shift(0)
    np.testing.assert_array_equal(s.get_state("Z"), z)
    s.shift(3)
    idx = np.minimum(np.arange(p.N) + 3, p.N - 1)
    np.testing.assert_array_equal(s.get_state("Z"), z[:, idx])
    np.testing.assert_array_equal(s.get_state("TH"), th[:, idx])
    np.testing.assert_array_equal(s.get_state("D"), d[:, idx])
    for bad in (-1, p.N):
        with pytest.raises(pimpc.PimpcError) as e:
            s.shift(bad)
        assert e.value.code == pimpc.EINVAL


# ---- odd shapes, optional terms, edge cases -----------------------------------------------------
@pytest.mark.parametrize("engine", ENGINES_SMALL)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", [(1, 1, 1, 1), (2, 1, 2, 3), (3, 2, 7, 5), (5, 3, 33, 2), (7, 2, 65, 1),
                                   (12, 4, 19, 9), (4, 2, 129, 2), (20, 6, 11, 2)])
def test_random_ltv_all_options(oracle, pimpc, engine, dtype, shape):
    nx, nu, N, batch = shape
    p = wl.random_ltv(nx, nu, N, batch, seed=nx * 100 + N, affine=True, u_prev=True, full_cost=True, wdu=True,
                      qbar=True, bounds=0.8, du_bound=0.5)
    parity.check(oracle, pimpc, p, dtype, engine=engine, iters=150, tol=0.0)


@pytest.mark.parametrize("engine", ENGINES_SMALL)
def test_unbounded_is_exactly_alg1_and_matches(oracle, pimpc, engine):
    p = wl.random_ltv(4, 2, 9, 2, seed=77, affine=True, bounds=None, du_bound=None)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine=engine, iters=300, tol=0.0)
    assert "D" not in g


@pytest.mark.parametrize("engine", ENGINES_SMALL)
def test_plain_admm_eta_zero(oracle, pimpc, engine):
    p = wl.quadrotor_ltv(12, 2, iters=120, tol=0.0)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine=engine, eta=0.0)
    assert np.all(g["res"]["restarts"] == 120)
    c = g["c_hist"]
    assert np.all(c[:, 1:] <= c[:, :-1] * (1 + 1e-12))          # Lemma 2 on the device


@pytest.mark.parametrize("engine", ENGINES_SMALL)
def test_per_instance_early_stop(oracle, pimpc, engine):
    """tol mode with batch > 1: instances stop at different iterations (step 5 per instance)."""
    p = wl.quadrotor_ltv(8, 6, iters=3000, tol=1e-4, rho=10.0, name="tolbatch")
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine=engine)
    it = g["res"]["iters"]
    assert len(set(it.tolist())) > 1 and np.all(g["res"]["converged"] == 1)


@pytest.mark.parametrize("engine", ENGINES_SMALL)
def test_warm_start_second_solve(oracle, pimpc, engine):
    """a second pimpc_solve continues from the returned iterates with hats = iterates."""
    p = wl.quadrotor_ltv(9, 2, iters=40, tol=0.0)
    s = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f64", engine=engine, history=40)
    s.set_problem(p)
    s.solve(40)
    warm = {k: s.get_state(k) for k in ("Z", "V", "TH", "BE", "LA", "D", "DE")}
    s.solve(25)
    z2 = s.get_state("Z")
    for b in range(p.batch):
        o = parity.oracle_run(oracle, p, "f64", b, iters=25, tol=0.0, warm=warm)
        assert parity.relerr(z2[b], o.Z) <= 1e-9
    # set_state on a fresh handle reproduces the same continuation
    s2 = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f64", engine=engine)
    s2.set_problem(p)
    for k, v in warm.items():
        s2.set_state(k, v)
    s2.solve(25)
    np.testing.assert_allclose(s2.get_state("Z"), z2, rtol=0, atol=1e-13)
    # reset = cold start
    s.reset(); s.solve(40)
    for k, v in warm.items():
        np.testing.assert_array_equal(s.get_state(k), v)


def test_set_stage_equals_bulk_setters(pimpc):
    p = wl.random_ltv(3, 2, 4, 2, seed=5, affine=True, bounds=0.7)
    a = pimpc.Solver(3, 2, 4, 2, dtype="f64"); a.set_problem(p); a.solve(30)
    b = pimpc.Solver(3, 2, 4, 2, dtype="f64")
    b.set_cost(p.Q, p.R, p.P, p.Wdu, p.qbar)
    for i in range(2):
        for k in range(4):
            b.set_stage(i, k, p.A[i, k], p.B[i, k], p.e[i, k], None, None, np.stack([p.lo, p.hi]), p.x0[i])
    b.set_x0(p.x0, p.u_prev)
    b.solve(30)
    np.testing.assert_array_equal(a.get_state("Z"), b.get_state("Z"))


def test_cache_matches_oracle_cache(oracle, pimpc):
    p = wl.random_ltv(5, 3, 6, 2, seed=11, full_cost=True, wdu=True, du_bound=0.5)
    for dtype, tol in (("f64", 1e-12), ("f32", 2e-6)):
        s = pimpc.Solver(5, 3, 6, 2, dtype=dtype, rho=0.7); s.set_problem(p); s.solve(0)
        M, H = s.get_cache()
        q = p.rounded(dtype)
        for b in range(2):
            Mo, Ho = oracle.cache(q.A[b], q.B[b], q.Q, q.R, P=q.P, Wdu=q.Wdu, has_du=True, rho=0.7)
            assert parity.relerr(M[b], Mo) <= tol and parity.relerr(H[b], Ho) <= tol


def test_device_pointers_and_torch_stream(pimpc):
    import torch
    p = wl.quadrotor_ltv(20, 3, iters=50, tol=0.0)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        s = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f32")
        A = torch.tensor(p.A, dtype=torch.float32, device="cuda"); B = torch.tensor(p.B, dtype=torch.float32, device="cuda")
        s.set_stages(A, B)
        s.set_cost(p.Q, p.R); s.set_bounds(p.lo, p.hi, p.du_lo, p.du_hi); s.set_x0(p.x0)
        s.solve(50)
        x = torch.empty(p.batch, p.N, p.nx, device="cuda"); u = torch.empty(p.batch, p.N, p.nu, device="cuda")
        s.get(x, u, torch.empty(p.batch, p.N, p.nu, device="cuda"))
    ref = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f32"); ref.set_problem(p); ref.solve(50)
    xr, ur, _, _ = ref.get()
    np.testing.assert_array_equal(x.cpu().numpy(), xr)
    np.testing.assert_array_equal(u.cpu().numpy(), ur)


def test_error_paths(pimpc):
    with pytest.raises(pimpc.PimpcError) as e:
        pimpc.Solver(0, 1, 1, 1)
    assert e.value.code == pimpc.EINVAL
    with pytest.raises(pimpc.PimpcError):
        pimpc.Solver(100, 60, 4, 1)                      # nx+nu > 128
    s = pimpc.Solver(2, 1, 3, 1, history=5)
    with pytest.raises(pimpc.PimpcError) as e:
        s.set_bounds(np.array([1.0, 0, 0]), np.array([0.0, 1, 1]))          # lo > hi
    assert e.value.code == pimpc.EINVAL
    with pytest.raises(pimpc.PimpcError):
        s.solve(6)                                       # exceeds history capacity
    with pytest.raises(pimpc.PimpcError):
        s.set_state("X", np.zeros((1, 3, 3)))            # X is an output
    A = np.tile(np.eye(2), (1, 3, 1, 1)); A[0, 1, 0, 0] = np.nan
    s.set_stages(A, np.ones((1, 3, 2, 1)))
    s.solve(2)
    with pytest.raises(pimpc.PimpcError) as e:
        s.sync()                                         # deferred device-side error
    assert e.value.code == pimpc.EINVAL
    A[0, 1, 0, 0] = 1.0
    s.set_stages(A, np.ones((1, 3, 2, 1))); s.solve(2); s.sync()      # the handle recovers
