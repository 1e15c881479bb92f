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


def test_config4_full_batch_every_instance(oracle, pimpc):
    """Full 4096-instance batch in the launch configuration bench.py times; EVERY instance is compared with the
    oracle (819 200 accept / restart decisions; the oracle calls run on a thread pool, ctypes releases the GIL)."""
    from concurrent.futures import ThreadPoolExecutor
    p = wl.config4()
    g = parity.gpu_run(pimpc, p, "f32")
    assert np.all(g["res"]["iters"] == 200)
    parity.check_properties(p, "f32", g)
    with ThreadPoolExecutor(os.cpu_count() or 4) as ex:
        out = list(ex.map(lambda b: parity.check_instance(oracle, p, "f32", g, b, label="C4/f32/auto"), range(p.batch)))
    nrep = sum(int(r == 1) for _, r in out)
    st = parity.STATS["C4/f32/auto"]
    print(f"C4: worst {st['worst']:.2e}, c_rel {st['c_rel']:.2e}, replays {nrep} of {p.batch}, widest flip margin {st['flip_margin']}")
    print(f"    band of the widest flip {st['flip_band']}")
    assert nrep <= parity.replay_bound("f32", 200 * p.batch)


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
def _tune(**kw):
    """Solver keyword arguments with launch-shape overrides (pimpc_opts.tune)."""
    return {"tune": {k: v for k, v in kw.items() if v}}


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [0, 1, 3, 7])
@pytest.mark.parametrize("shape", [(48, 12, 37, 3), (12, 4, 41, 2), (4, 2, 23, 5)])
def test_stream_engine_all_options(oracle, pimpc, shape, grid, dtype):
    """grid = 0: one or two steps per CTA (every step a halo); 1: one CTA owns everything; 3, 7: ranges
    start inside instances and span several of them."""
    nx, nu, N, batch = shape
    p = wl.random_ltv(nx, nu, N, batch, seed=nx * 10 + N, affine=True, u_prev=True, full_cost=True, wdu=True,
                      qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="stream", iters=120, tol=0.0, opts=_tune(grid=grid))
    assert g["info"]["engine"] == pimpc.ENGINE_STREAM
    parity.check_properties(p, dtype, g)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [0, 3])
@pytest.mark.parametrize("shape", [(10, 3, 17, 2), (20, 6, 9, 2), (30, 10, 7, 1), (50, 15, 5, 2)])
def test_stream_engine_paper_table1_shapes(oracle, pimpc, shape, grid, dtype):
    """The (n, m) of the paper's Table I, odd nb included (circulant storage of H without a
    self-paired diagonal); AUTO must pick a fused engine for them (the register-resident one for (10, 3) in fp32)."""
    nx, nu, N, batch = shape
    p = wl.random_ltv(nx, nu, N, batch, seed=nx * 7 + N, affine=True, u_prev=True, full_cost=True, wdu=True,
                      qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="stream", iters=100, tol=0.0, opts=_tune(grid=grid))
    assert g["info"]["engine"] == pimpc.ENGINE_STREAM
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="auto", iters=100, tol=0.0)
    assert g["info"]["engine"] != pimpc.ENGINE_STAGED         # a fused engine serves every Table-I shape up to (50, 15)
    parity.check_properties(p, dtype, g)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [0, 3])
@pytest.mark.parametrize("shape", [(3, 1, 19, 3), (7, 4, 13, 2), (13, 2, 11, 2), (16, 4, 9, 2), (25, 8, 7, 2), (41, 13, 5, 1)])
def test_stream_engine_any_shape_inside_a_container(oracle, pimpc, shape, grid, dtype):
    """Shapes without an instantiation of their own run INSIDE the smallest container that holds them ((12, 4), (20, 6),
    (30, 10), (50, 15); template flag PAD): padded blobs and on-chip vectors, real-shape records and caller vectors.  All
    optional terms on; AUTO must not fall back to the five-launches-per-iteration STAGED engine for them."""
    nx, nu, N, batch = shape
    p = wl.random_ltv(nx, nu, N, batch, seed=nx * 5 + N, affine=True, u_prev=True, full_cost=True, wdu=True,
                      qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="stream", iters=100, tol=0.0, opts=_tune(grid=grid))
    assert g["info"]["engine"] == pimpc.ENGINE_STREAM
    parity.check_properties(p, dtype, g)
    if nx > 12 or nu > 4:                                 # (beyond the register / shared-memory resident engines' shapes)
        g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="auto", iters=100, tol=0.0)
        assert g["info"]["engine"] == pimpc.ENGINE_STREAM


def test_stream_engine_container_early_stop_warm_start_and_no_bounds(oracle, pimpc):
    p = wl.random_ltv(9, 5, 12, 3, seed=91, affine=True, bounds=None, du_bound=None)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="stream", iters=200, tol=0.0)
    assert "D" not in g
    p = wl.random_ltv(14, 3, 10, 2, seed=92, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5)
    p.iters, p.tol = 400, 3e-2                          # stops early on some instances (the oracle's iteration counts are compared)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="stream")
    assert np.any(g["res"]["converged"] == 1)
    s = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f64", engine="stream")
    s.set_problem(p); s.solve(40)
    warm = {k: s.get_state(k) for k in ("Z", "V", "TH", "BE", "LA", "D", "DE")}
    s.solve(25)
    for b in range(p.batch):
        o = parity.oracle_run(oracle, p, "f64", b, iters=25, tol=0.0, warm=warm)
        assert parity.relerr(s.get_state("Z")[b], o.Z) <= 1e-9


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", [(48, 12, 160, 6), (30, 10, 90, 3), (20, 6, 70, 4)])
def test_stream_engine_repeated_runs_are_bit_identical(pimpc, shape, dtype):
    """Two runs of the same solve on the same launch shape (several stage steps per CTA, ranges that split instances, every
    ring slot reused many times): every iterate, the primal step and the history of c bit for bit.  The stage step reuses
    its shared-memory vectors across phases (the H h partials overlay the column-product partials) and slots across
    steps: a missing barrier or a copy landing early would show here as a difference between runs."""
    nx, nu, N, batch = shape
    p = wl.random_ltv(nx, nu, N, batch, seed=N, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5)
    s = pimpc.Solver(nx, nu, N, batch, dtype=dtype, engine="stream", rho=p.rho, history=60)
    s.set_problem(p)
    runs = []
    for _ in range(3):
        s.reset()
        s.solve(60, 0.0)
        runs.append(({k: s.get_state(k).copy() for k in ("X", "DU", "Z", "V", "TH", "BE", "LA", "D", "DE")}, s.get_history()[0].copy()))
    assert s.get_info()["engine"] == pimpc.ENGINE_STREAM
    s.close()
    for st, hist in runs[1:]:
        for k, v in st.items():
            np.testing.assert_array_equal(v, runs[0][0][k], err_msg=k)
        np.testing.assert_array_equal(hist, runs[0][1])
    assert np.isfinite(runs[0][1]).all() and (runs[0][1][:, -1] < runs[0][1][:, 0]).all()


@pytest.mark.parametrize("grid", [0, 5])
def test_stream_engine_unbounded_and_plain_admm(oracle, pimpc, grid):
    p = wl.random_ltv(4, 2, 9, 2, seed=77, affine=True, bounds=None, du_bound=None)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="stream", iters=300, tol=0.0, opts=_tune(grid=grid))
    assert "D" not in g
    p = wl.quadrotor_ltv(12, 2, iters=120, tol=0.0)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="stream", eta=0.0, opts=_tune(grid=grid))
    assert np.all(g["res"]["restarts"] == 120)


@pytest.mark.parametrize("grid", [0, 4])
def test_stream_engine_early_stop_and_warm_start(oracle, pimpc, grid):
    p = wl.quadrotor_ltv(8, 6, iters=3000, tol=1e-4, rho=10.0, name="tolbatch")
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="stream", opts=_tune(grid=grid))
    assert len(set(g["res"]["iters"].tolist())) > 1 and np.all(g["res"]["converged"] == 1)
    p = wl.quadrotor_ltv(9, 2, iters=40, tol=0.0)
    s = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f64", engine="stream", **_tune(grid=grid))
    s.set_problem(p); s.solve(40)
    warm = {k: s.get_state(k) for k in ("Z", "V", "TH", "BE", "LA", "D", "DE")}
    s.solve(25)
    z2 = s.get_state("Z")
    for b in range(p.batch):
        o = parity.oracle_run(oracle, p, "f64", b, iters=25, tol=0.0, warm=warm)
        assert parity.relerr(z2[b], o.Z) <= 1e-9


# ---- COOP engine (batch 1, horizon spread over the SMs, tagged-word exchange instead of grid barriers) ------
def _coop(grid=0, spg=0, cluster=None, lookahead=0):
    """cluster None: automatic (one cluster for short horizons); 0: exchange through L2 (the long-horizon path); n: cluster of n.
    lookahead -1: every thread waits for the accept / restart decision instead of predicting it."""
    return _tune(grid=grid, stages_per_group=spg, cluster=(0 if cluster is None else (-1 if cluster == 0 else cluster)),
                 lookahead=lookahead)


@pytest.mark.parametrize("cluster", [None, 0, 8])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [0, 1, 2, 7])
@pytest.mark.parametrize("shape", [(12, 4, 41), (4, 2, 23), (12, 4, 150), (4, 2, 1), (12, 4, 2)])
def test_coop_engine_all_options(oracle, pimpc, shape, grid, dtype, cluster):
    """grid = 0: one stage per CTA while N <= 148 (every stage has two ghosts); 1: a single CTA, no exchange;
    2, 7: ragged ranges.  All optional terms on."""
    nx, nu, N = shape
    if N > 100 and grid in (1, 2):
        grid += 4                         # 150 stages of (12, 4) do not fit one or two CTAs' shared memory: 5, 6 CTAs
    if (nx, N, grid, dtype) == (12, 41, 1, "f64"):
        grid = 3                          # 41 fp64 stages of (12, 4) no longer fit ONE CTA (parity copies of xbar, lane partials of c)
    p = wl.random_ltv(nx, nu, N, 1, seed=nx * 10 + N, affine=True, u_prev=True, full_cost=True, wdu=True,
                      qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="coop", iters=120, tol=0.0, opts=_coop(grid, cluster=cluster))
    assert g["info"]["engine"] == pimpc.ENGINE_COOP
    parity.check_properties(p, dtype, g)


@pytest.mark.parametrize("cluster", [None, 0])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape,grid", [((20, 6, 31), 0), ((20, 6, 90), 7), ((16, 8, 25), 3), ((13, 5, 40), 0), ((20, 8, 12), 1),
                                        ((20, 6, 200), 0)])
def test_coop_engine_wide_shapes_inside_20_8(oracle, pimpc, shape, grid, dtype, cluster):
    """Shapes with 12 < nx <= 20 or 4 < nu <= 8 -- the (20, 6) of the paper's Table I among them -- run
    inside the (20, 8) instantiation of the COOP engine (one row per lane: 28 of the 32 lanes of a stage).  All optional
    terms on; AUTO must pick COOP for them at batch 1.  N = 200 in fp64 is longer than the ranges 16 CTAs of a cluster hold:
    the automatic plan then takes more CTAs exchanging through L2."""
    nx, nu, N = shape
    if (N, grid, dtype) == (90, 7, "f64"):
        grid = 12                         # 13 fp64 stages of (20, 8) do not fit one CTA's shared memory
    p = wl.random_ltv(nx, nu, N, 1, seed=nx * 3 + N, affine=True, u_prev=True, full_cost=True, wdu=True,
                      qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="coop", iters=120, tol=0.0, opts=_coop(grid, cluster=cluster))
    assert g["info"]["engine"] == pimpc.ENGINE_COOP
    parity.check_properties(p, dtype, g)
    if grid == 0 and cluster is None:
        g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="auto", iters=120, tol=0.0)
        assert g["info"]["engine"] == pimpc.ENGINE_COOP


@pytest.mark.parametrize("cluster", [None, 0])
@pytest.mark.parametrize("grid", [3, 0])
def test_coop_engine_two_stages_per_group_fp32(oracle, pimpc, grid, cluster):
    p = wl.random_ltv(12, 4, 100, 1, seed=5, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f32", engine="coop", iters=150, tol=0.0, opts=_coop(grid, 2, cluster))
    assert g["info"]["engine"] == pimpc.ENGINE_COOP


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("cluster", [None, 0])
@pytest.mark.parametrize("shape,grid", [((12, 4, 41), 0), ((12, 4, 150), 7), ((4, 2, 23), 2)])
def test_coop_decision_predicted_or_waited_for(oracle, pimpc, shape, grid, cluster, dtype):
    """by default the compute warps PREDICT the accept / restart decision and run phases A-C of the next
    iteration while the partial sums of c travel (a wrong prediction repeats them); tune.lookahead = -1 makes them wait.
    Both orders must give the oracle's iterates and decision sequence; 400 iterations reach the all-restart tail, so that
    accept-predicted-restart, restart-predicted-accept and the right predictions all occur."""
    nx, nu, N = shape
    p = wl.random_ltv(nx, nu, N, 1, seed=nx * 7 + N, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5)
    res = {}
    for la in (0, -1):
        g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="coop", iters=400, tol=0.0,
                                      opts=_coop(grid, cluster=cluster, lookahead=la))
        assert g["info"]["engine"] == pimpc.ENGINE_COOP
        res[la] = g
    for name in ("Z", "V", "TH", "BE", "LA", "X", "DU"):
        assert np.array_equal(res[0][name], res[-1][name]), name       # same arithmetic in both orders: bit-identical
    assert np.array_equal(res[0]["acc_hist"], res[-1]["acc_hist"])
    assert 0 < int(res[0]["res"]["restarts"][0]) < 400


@pytest.mark.parametrize("cluster", [None, 0])
@pytest.mark.parametrize("grid", [0, 5])
def test_coop_engine_unbounded_plain_admm_early_stop_warm_start(oracle, pimpc, grid, cluster):
    o = _coop(grid, cluster=cluster)
    p = wl.random_ltv(4, 2, 9, 1, seed=77, affine=True, bounds=None, du_bound=None)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="coop", iters=300, tol=0.0, opts=o)
    assert "D" not in g
    p = wl.quadrotor_ltv(12, 1, iters=120, tol=0.0)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="coop", eta=0.0, opts=o)
    assert np.all(g["res"]["restarts"] == 120)
    p = wl.quadrotor_ltv(10, 1, iters=2000, tol=1e-4, rho=10.0, name="C2-tol")
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="coop", opts=o)
    assert int(g["res"]["converged"][0]) == 1 and int(g["res"]["iters"][0]) < 2000
    p = wl.quadrotor_ltv(30, 1, iters=40, tol=0.0)
    s = pimpc.Solver(p.nx, p.nu, p.N, 1, dtype="f64", engine="coop", **o)
    s.set_problem(p); s.solve(40)
    warm = {k: s.get_state(k) for k in ("Z", "V", "TH", "BE", "LA", "D", "DE")}
    s.solve(25)
    o = parity.oracle_run(oracle, p, "f64", 0, iters=25, tol=0.0, warm=warm)
    assert parity.relerr(s.get_state("Z")[0], o.Z) <= 1e-9


# ---- NEXT row f1: receding-horizon stepping with shift warm start ----------------
@pytest.mark.parametrize("engine,native", [("auto", True), ("coop", True), ("staged", True), ("resident", True),
                                           ("stream", False), ("auto", False), ("coop", False)])
def test_closed_loop_cstr_shift_warm_start(oracle, pimpc, engine, native):
    """Four MPC steps of the online-linearised CSTR: per step new stage data (set_stages + a0), pimpc_shift(1) of the
    previous iterates, K iterations; the plant advances with the oracle's u_0.  native: the CUDA path runs the paper's
    own (n, m) = (2, 1) shape (the fused engines hold it inside their padded (4, 4) instantiation);
    else the problem is embedded in the (4, 2) shape by workloads.pad_problem (STREAM has no smaller instantiation)."""
    N, K, T = (56 if engine == "resident" else 60), 120, 4      # fp64 RESIDENT: 7 stage warps of 8 stages + the reducer warp
    x = np.array(wl.CSTR["x_init"]); u = np.array([wl.CSTR["u_init"]]); t = 0.0
    s = pimpc.Solver(2, 1, N, 1, dtype="f64", engine=engine, history=K) if native else \
        pimpc.Solver(4, 2, N, 1, dtype="f64", engine=engine, history=K)
    real = [0, 1, 2] if native else [0, 1, 4]
    warm = None
    for step in range(T):
        p = wl.cstr_problem(x, u, t, N, iters=K)
        s.set_problem(p if native else wl.pad_problem(p, 4, 2))
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
            if not native:
                assert float(np.max(np.abs(np.delete(g, real, axis=1)))) == 0.0      # the embedding stays exactly zero
        xg, ug, dug, res = s.get()
        assert parity.relerr(ug[0, :, :1], o.u) <= 1e-9 and parity.relerr(dug[0, :, :1], o.DU) <= 1e-9
        warm = dict(Z=o.Z, V=o.V, TH=o.TH, BE=o.BE, LA=o.LA)
        u = o.u[0].copy()
        x = wl.cstr_plant_step(x, u, t); t += wl.CSTR["Ts"]
    if native and engine != "staged":
        assert s.get_info()["engine"] != pimpc.ENGINE_STAGED      # a fused engine runs the native shape
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


# ---- RESIDENT engine: every instantiation AUTO can reach ---------------------------------
@pytest.mark.parametrize("N,batch,rows", [(57, 3, 0), (60, 2, 0), (64, 5, 0), (48, 3, 0), (49, 2, 0), (50, 3, 1), (23, 2, 1), (61, 2, 1)])
def test_resident_fp32_quadrotor_one_row_per_lane(oracle, pimpc, N, batch, rows):
    """fp32 (12, 4): horizons 45..60 run k_res2 with G_k in shared memory (12..15 stage warps + the reducer warp), 61..64
    and tune.rows_per_lane = 1 the one-row-per-lane kernel (k_resident<float,12,4,1,800|1024>)."""
    p = wl.quadrotor_ltv(N, batch, iters=150, tol=0.0)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f32", engine="resident", opts=_tune(rows_per_lane=rows))
    assert g["info"]["engine"] == pimpc.ENGINE_RESIDENT
    assert g["info"]["block"] == 32 * ((N + 1) // 2 if rows == 1 or N > 60 else (N + 3) // 4 + 1)
    parity.check_properties(p, "f32", g)


@pytest.mark.parametrize("N,batch", [(1, 3), (23, 4), (120, 2)])
@pytest.mark.parametrize("engine", ["auto", "resident"])
def test_resident_fp32_small_shape_all_options(oracle, pimpc, engine, N, batch):
    """fp32 (4, 2), N <= 120 (15 stage warps of 8 stages + the reducer warp): k_res2<float,4,4>, all optional terms on."""
    p = wl.random_ltv(4, 2, N, batch, seed=400 + N, affine=True, u_prev=True, full_cost=True, wdu=True, qbar=True,
                      bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f32", engine=engine, iters=150, tol=0.0)
    assert g["info"]["engine"] == pimpc.ENGINE_RESIDENT


# ---- boundary: e-only updates, partial cache refresh, caller workspace, residual halves ------------------------
@pytest.mark.parametrize("engine,shape", [("staged", (5, 3, 9, 2)), ("resident", (4, 2, 23, 3)), ("coop", (12, 4, 41, 1)),
                                          ("stream", (12, 4, 41, 2)), ("stream", (48, 12, 11, 2))])
def test_affine_term_only_update_between_solves(oracle, pimpc, engine, shape):
    """solve, change ONLY e (bulk and per-stage setter), solve again == a fresh handle with the new e.
    Also an e supplied for the first time after a solve."""
    nx, nu, N, batch = shape
    p = wl.random_ltv(nx, nu, N, batch, seed=31, affine=True, bounds=0.8, du_bound=0.5)
    e2 = -1.7 * p.e + 0.05
    for first_e in (p.e, None):
        s = pimpc.Solver(nx, nu, N, batch, dtype="f64", engine=engine)
        s.set_stages(p.A, p.B, first_e); s.set_cost(p.Q, p.R); s.set_bounds(p.lo, p.hi, p.du_lo, p.du_hi)
        s.set_x0(p.x0, p.u_prev)
        s.solve(30); s.reset()
        s.set_stages(None, None, e2)
        s.set_stage(batch - 1, N // 2, None, None, 3.0 * e2[batch - 1, N // 2])
        s.solve(60)
        e3 = e2.copy(); e3[batch - 1, N // 2] *= 3.0
        q = wl.random_ltv(nx, nu, N, batch, seed=31, affine=True, bounds=0.8, du_bound=0.5); q.e = e3
        for b in range(batch):
            o = parity.oracle_run(oracle, q, "f64", b, iters=60, tol=0.0)
            for name in ("Z", "V", "TH", "X"):
                assert parity.relerr(s.get_state(name)[b], getattr(o, name)) <= 1e-9, (engine, name, first_e is None)
        s.close()


def test_set_stage_refreshes_only_the_touched_cache_entries(oracle, pimpc):
    """pimpc_set_stage on a few stages re-inverts only H_{k-1}, M_k, H_k of those stages; the
    result equals a handle that was given the final data at once."""
    p = wl.random_ltv(12, 4, 19, 3, seed=8, affine=True, bounds=0.8, du_bound=0.5)
    for dtype, tol in (("f64", 1e-12), ("f32", 2e-6)):
        s = pimpc.Solver(12, 4, 19, 3, dtype=dtype); s.set_problem(p); s.solve(5)
        q = wl.random_ltv(12, 4, 19, 3, seed=8, affine=True, bounds=0.8, du_bound=0.5)
        for (b, k) in ((0, 0), (1, 7), (2, 18), (1, 8)):
            q.A[b, k] = 0.9 * q.A[b, k] + 0.01; q.B[b, k] = 1.1 * q.B[b, k]
            s.set_stage(b, k, q.A[b, k], q.B[b, k])
        s.reset(); s.solve(40)
        assert s.get_info()["setup_ms"] > 0.0
        M, H = s.get_cache()
        qr = q.rounded(dtype)
        for b in range(3):
            Mo, Ho = oracle.cache(qr.A[b], qr.B[b], qr.Q, qr.R, has_du=True, rho=1.0)
            assert parity.relerr(M[b], Mo) <= tol and parity.relerr(H[b], Ho) <= tol
        f = pimpc.Solver(12, 4, 19, 3, dtype=dtype); f.set_problem(q); f.solve(40)
        np.testing.assert_array_equal(s.get_state("Z"), f.get_state("Z"))


def test_caller_provided_workspace(pimpc):
    import torch
    p = wl.quadrotor_ltv(20, 3, iters=50, tol=0.0)
    need = pimpc.workspace_bytes(p.nx, p.nu, p.N, p.batch, dtype="f32", history=50)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    s = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f32", history=50, workspace=ws)
    assert s.get_info()["device_bytes"] == 0                  # nothing allocated by the library so far
    s.set_problem(p); s.solve(50)
    ref = pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f32", history=50); ref.set_problem(p); ref.solve(50)
    np.testing.assert_array_equal(s.get_state("Z"), ref.get_state("Z"))
    np.testing.assert_array_equal(s.get_history()[0], ref.get_history()[0])
    s.close()
    with pytest.raises(pimpc.PimpcError) as e:
        pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f32", workspace=ws[:need // 2])
    assert e.value.code == pimpc.EINVAL
    with pytest.raises(pimpc.PimpcError):
        pimpc.Solver(p.nx, p.nu, p.N, p.batch, dtype="f32", workspace=ws[8:])      # misaligned


@pytest.mark.parametrize("engine,dtype,shape", [("staged", "f64", (5, 3, 9, 2)), ("auto", "f32", (12, 4, 50, 7)),
                                                ("coop", "f64", (12, 4, 41, 1)), ("stream", "f32", (48, 12, 11, 2))])
def test_result_record_primal_and_dual_residual_halves(oracle, pimpc, engine, dtype, shape):
    """pimpc_result.r_prim2 / r_dual2 against the oracle's halves of c."""
    nx, nu, N, batch = shape
    p = wl.random_ltv(nx, nu, N, batch, seed=61, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5)
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine=engine, iters=80, tol=0.0)
    for b in range(batch):
        o = parity.oracle_run(oracle, p, dtype, b, iters=80, tol=0.0)
        r = g["res"][b]
        assert abs(r["r_prim2"] + r["r_dual2"] - r["c"]) <= 1e-12 * r["c"]
        assert abs(r["r_prim2"] - o.r_prim2) <= parity.TOL_C[dtype] * o.r_prim2
        assert abs(r["r_dual2"] - o.r_dual2) <= parity.TOL_C[dtype] * o.c_last


def test_large_shape_of_the_papers_table1(oracle, pimpc):
    """(n, m) = (100, 30), the largest shape of Table I: nb = 130 runs on the generic engines."""
    p = wl.paper_random(100, 30, 6, iters=40)
    g, worst, nrep = parity.check(oracle, pimpc, p, "f64", engine="auto", iters=40, tol=0.0)


# ---- general convex sets, per-stage terms, the tracking cost ----------
SETS_GPU = {"halfspace": ("halfspace", 1, [1.0, 0.6, -0.8, 0.5], 0.1), "hyperplane": ("hyperplane", 2, [1.0, -2.0, 0.7], 0.05),
            "soc": ("soc", 5, 3, None), "l1ball": ("l1ball", 5, 3, 0.35), "l1ball-wide": ("l1ball", 0, 8, 1.2)}


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("kind", list(SETS_GPU))
@pytest.mark.parametrize("engine,grid", [("staged", 0), ("stream", 0), ("stream", 3), ("auto", 0)])
def test_general_convex_sets(oracle, pimpc, engine, grid, kind, dtype):
    """z_{k+1} = Proj onto box x {halfspace, hyperplane, second-order cone, l1 ball} (Thm 1), with
    per-stage boxes on the other components and per-stage linear terms; (nx, nu) = (5, 3), N = 17, batch 2.  The set is
    active (checked on the oracle's iterate: the projection moved at least one stage)."""
    nx, nu, N, batch = 5, 3, 17, 2
    p = wl.random_ltv(nx, nu, N, batch, seed=166, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5, scale=0.2)
    rng = np.random.default_rng([2601, 14414, 8, 2])
    p.cset = SETS_GPU[kind]
    p.lo_k = -rng.uniform(0.3, 0.9, size=(N, nx + nu)); p.hi_k = rng.uniform(0.3, 0.9, size=(N, nx + nu))
    p.qbar_k = 0.3 * rng.normal(size=(N, nx + nu))
    if engine == "stream":
        if (nx, nu) == (5, 3):                            # STREAM has no (5, 3) instantiation: the same test on (12, 4)
            nx, nu = 12, 4
            p = wl.random_ltv(nx, nu, N, batch, seed=166, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5, scale=0.2)
            p.cset = SETS_GPU[kind]
            p.lo_k = -rng.uniform(0.3, 0.9, size=(N, nx + nu)); p.hi_k = rng.uniform(0.3, 0.9, size=(N, nx + nu))
            p.qbar_k = 0.3 * rng.normal(size=(N, nx + nu))
    g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine=engine, iters=150, tol=0.0, opts=_tune(grid=grid))
    assert g["info"]["engine"] in (pimpc.ENGINE_STAGED, pimpc.ENGINE_STREAM)
    k_, i0, a, b = p.cset
    n = a if isinstance(a, int) else len(a)
    Zs = g["Z"][..., i0:i0 + n].astype(np.float64)
    if k_ == "halfspace":
        val = Zs @ np.asarray(a); assert np.all(val <= b + 1e-5) and np.any(val >= b - 1e-5)
    elif k_ == "hyperplane":
        assert np.max(np.abs(Zs @ np.asarray(a) - b)) <= 1e-5
    elif k_ == "soc":
        gap = Zs[..., -1] - np.linalg.norm(Zs[..., :-1], axis=-1); assert np.all(gap >= -1e-5) and np.any(gap <= 1e-5)
    else:
        l1 = np.sum(np.abs(Zs), axis=-1); assert np.all(l1 <= b + 1e-5) and np.any(l1 >= b - 1e-5)
    out = np.delete(g["Z"], np.arange(i0, i0 + n), axis=-1)
    assert np.all(out >= np.delete(p.lo_k, np.arange(i0, i0 + n), axis=-1).astype(out.dtype))
    assert np.all(out <= np.delete(p.hi_k, np.arange(i0, i0 + n), axis=-1).astype(out.dtype))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("engine", ["staged", "auto", "stream", "coop"])
def test_tracking_entry_point_afti16(oracle, pimpc, engine, dtype):
    """pimpc_set_tracking(C, W_y, W_u, r_y, r_u) forms Q = C'W_y C, R = W_u, qbar on the device; the
    oracle forms them with its own routine.  Problem: the AFTI-16 model with its output constraints -0.5 <= y_1 <= 0.5
    (PAPER.md:321-329), N = 5 as in the paper and N = 23."""
    for N, batch in ((5, 3), (23, 1)):
        if engine == "coop" and batch != 1:
            continue
        p, trk = wl.afti16(N, batch, iters=300)
        pr = p.rounded(dtype)
        r32 = (lambda a: np.asarray(a, np.float32).astype(np.float64)) if dtype == "f32" else (lambda a: a)
        Q, R, qbar = oracle.tracking(r32(trk["C"]), r32(trk["Wy"]), r32(trk["Wu"]), r32(trk["ry"]), r32(trk["ru"]))
        s = pimpc.Solver(4, 2, N, batch, dtype=dtype, engine=engine, rho=p.rho, history=300)
        s.set_stages(p.A, p.B); s.set_bounds(p.lo, p.hi); s.set_x0(p.x0)
        s.set_cost(np.eye(4), np.eye(2), None, p.Wdu)                    # Wdu stays; Q, R, qbar are replaced below
        s.set_tracking(trk["C"], trk["Wy"], trk["Wu"], trk["ry"], trk["ru"])
        s.solve(300)
        c, acc = s.get_history()
        for b in range(batch):
            a = pr.instance(b); a.update(Q=Q, R=R, qbar=qbar)
            o = oracle.solve(**a, max_iters=300, tol=0.0)
            assert list(acc[b]) == list(o.acc_hist) or dtype == "f32"
            if list(acc[b]) != list(o.acc_hist):
                o = oracle.solve(**a, max_iters=300, tol=0.0, forced=acc[b])
            for name in ("Z", "V", "TH", "X"):
                assert parity.relerr(s.get_state(name)[b], getattr(o, name)) <= parity.TOL[dtype], (engine, N, name)
        y1 = s.get_state("Z")[..., 1]
        assert np.all(np.abs(y1) <= 0.5)
        s.close()


@pytest.mark.parametrize("engine", ["staged", "stream"])
def test_tracking_with_time_varying_references(oracle, pimpc, engine):
    """per_stage references r_y[k], r_u[k]: qbar differs per stage (STAGED / STREAM)."""
    nx, nu, N = 12, 4, 21
    p = wl.random_ltv(nx, nu, N, 2, seed=9, affine=True, u_prev=True, bounds=0.8, du_bound=0.5, scale=0.2)
    rng = np.random.default_rng([2601, 14414, 197, 2])
    C = rng.normal(size=(3, nx)); Wy = np.diag([2.0, 1.0, 0.5]); Wu = 0.1 * np.eye(nu)
    ry = 0.3 * rng.normal(size=(N, 3)); ru = 0.05 * rng.normal(size=(N, nu))
    s = pimpc.Solver(nx, nu, N, 2, dtype="f64", engine=engine, history=120)
    s.set_problem(p)
    s.set_tracking(C, Wy, Wu, ry, ru, per_stage=True)
    s.solve(120)
    qk = np.stack([oracle.tracking(C, Wy, Wu, ry[k], ru[k])[2] for k in range(N)])
    Q, R, _ = oracle.tracking(C, Wy, Wu, None, None)
    for b in range(2):
        a = p.instance(b); a.update(Q=Q, R=R, qbar=None, P=None, qbar_k=qk)
        o = oracle.solve(**a, max_iters=120, tol=0.0)
        for name in ("Z", "V", "TH", "X"):
            assert parity.relerr(s.get_state(name)[b], getattr(o, name)) <= 1e-9, (engine, name)


def test_resident_pad_stages_with_a_box_that_excludes_zero(oracle, pimpc):
    """A horizon that does not fill the last warp leaves pad stages in the CTA; they must stay exactly zero even when
    the box excludes 0 (their constants are a block of zeros, not the instance's bounds)."""
    for dtype, shape in (("f32", (12, 4, 50, 3)), ("f64", (4, 2, 9, 2)), ("f32", (4, 2, 61, 2))):
        nx, nu, N, batch = shape
        p = wl.random_ltv(nx, nu, N, batch, seed=77, affine=True, u_prev=True, bounds=0.9, du_bound=0.5, scale=0.2)
        p.lo = p.lo.copy(); p.lo[1] = 0.15; p.lo[nx] = 0.1            # x_2 >= 0.15, u_1 >= 0.1
        g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine="resident", iters=120, tol=0.0)


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
        pimpc.Solver(100, 61, 4, 1)                      # nx+nu > 160
    with pytest.raises(pimpc.PimpcError):
        pimpc.Solver(2, 1, 3, 65536)                     # batch > 65535
    with pytest.raises(pimpc.PimpcError):
        pimpc.Solver(2, 1, 3, 1, tune={"cluster": 17})
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


def test_measure_peaks_on_chip_rates_and_latencies(pimpc):
    """pimpc_measure_peaks (SURVEY 8(d) "measure both with an FMA-chain microbenchmark"): the pipe rates bench.py reports
    the RESIDENT engine against, and the latencies of a dependent instruction that DESIGN.md section 6 argues with.  Wide
    sanity bands only (any Blackwell part): the numbers are measured, not asserted to be B200's."""
    pk = pimpc.measure_peaks()
    assert pk["sm_count"] >= 1
    assert 10.0 < pk["ffma_tflops"] < 200.0 and 10.0 < pk["ffma2_tflops"] < 200.0
    assert 0.5 < pk["dfma_tflops"] < 100.0
    assert 5e3 < pk["smem_gbs"] < 1e5
    assert 2.0 <= pk["lat_ffma2_cycles"] <= 12.0
    assert pk["lat_ffma2_cycles"] < pk["lat_dadd_cycles"] <= 80.0
    assert 10.0 <= pk["lat_shfl_cycles"] <= 60.0 and 15.0 <= pk["lat_lds_cycles"] <= 60.0
    assert 1.0 <= pk["lds128_bcast_cycles"] <= 4.5           # between the 128 B/clk of distinct data and a full 4-wavefront load


@pytest.mark.parametrize("iters", [1, 2, 3, 4, 7])
@pytest.mark.parametrize("engine,dtype,shape", [("resident", "f32", (12, 4, 50, 3)), ("resident", "f32", (12, 4, 9, 2)),
                                                ("resident", "f64", (4, 2, 20, 2)), ("coop", "f32", (12, 4, 40, 1)),
                                                ("coop", "f64", (4, 2, 23, 1))])
def test_predicted_decision_short_runs(oracle, pimpc, engine, dtype, shape, iters):
    """The engines that predict the accept / restart decision unroll their loop by two and resolve a decision one phase
    late: every exit (odd / even counts, the first iterations, a pending decision at the end) must return the oracle's
    iterate, primal step, history and counters."""
    nx, nu, N, batch = shape
    p = wl.random_ltv(nx, nu, N, batch, seed=nx + N + iters, affine=True, u_prev=True, qbar=True, bounds=0.8, du_bound=0.5)
    for opts in ((None,) if engine == "resident" else (None, _coop(cluster=0), _coop(lookahead=-1))):
        g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine=engine, iters=iters, tol=0.0, opts=opts)
        assert np.all(g["res"]["iters"] == iters)


@pytest.mark.parametrize("engine,dtype,shape", [("resident", "f32", (12, 4, 50, 4)), ("resident", "f64", (4, 2, 20, 3)),
                                                ("coop", "f64", (12, 4, 40, 1)), ("coop", "f32", (4, 2, 23, 1))])
def test_predicted_decision_stop_at_every_early_iteration(oracle, pimpc, engine, dtype, shape):
    """Early stop (step 5) right at iterations 1, 2, 3, ...: the tolerance is set just above the oracle's c of that
    iteration, so the stop is found while the next iteration's phases already run on a predicted momentum."""
    nx, nu, N, batch = shape
    p = wl.random_ltv(nx, nu, N, batch, seed=17 + nx, affine=True, u_prev=True, bounds=0.8, du_bound=0.5)
    o = parity.oracle_run(oracle, p, dtype, 0, iters=12, tol=0.0)
    for stop_at in (1, 2, 3, 5, 8):
        c = np.asarray(o.c_hist)
        if not (c[stop_at - 1] < np.min(c[:stop_at - 1], initial=np.inf)):
            continue                                      # c must fall below the tolerance for the first time there
        p.iters, p.tol = 12, float(c[stop_at - 1]) * 1.0005
        g, worst, nrep = parity.check(oracle, pimpc, p, dtype, engine=engine)
        assert int(g["res"]["iters"][0]) == stop_at and int(g["res"]["converged"][0]) == 1
