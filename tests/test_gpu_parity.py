"""GPU-vs-oracle parity through the C-ABI (include/fredopt.h) on the same seeded inputs.

Tolerances (BASELINE.json north_star): per SpMV relative error <= 1e-5; after 20 iterations relative L2
error in w <= 1e-4 and an IDENTICAL constraint-violation count.  Transposed passes carry signed
coefficients, so they are judged element-wise relative to sum_i |A_ij r_i| (parity rule).
"""
import os

import numpy as np
import pytest
import torch

from paper_2509_20012_b200 import plangen as pg

pytestmark = pytest.mark.gpu

TOL_SPMV = 1e-5
TOL_X20 = 1e-4


@pytest.fixture(scope="module")
def fredopt():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2509_20012_b200 import fredopt as f
    return f


def _oracle(plan):
    from oracle import oracle
    return oracle.from_plan(plan)


def _oracle_np(V, S, D, L, lab, bounds):
    from oracle import oracle
    return oracle.Oracle.create(V, S, D, L, lab, bounds)


def _gpu_x(gp):
    return gp.get_weights_f64(np.empty(gp.n_cols, np.float64))


def _rel_l2(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


# the stored forms of a plan (fredopt_create_options): index width automatic (16-bit where exact) or int32 everywhere; rows per
# stored block row automatic (fewest bytes) or forced to 1, 2, 4
INDEX_FORMS = [pytest.param({}, id="auto"), pytest.param({"index_width": 32}, id="idx32"),
               pytest.param({"block_rows": 1}, id="rows1"), pytest.param({"block_rows": 2}, id="rows2"),
               pytest.param({"block_rows": 4}, id="rows4"), pytest.param({"block_rows": 2, "index_width": 32}, id="rows2-idx32")]


def _assert_fwd(got, ref, what):
    got = got.astype(np.float64)
    # fp32 output rounding: half an ulp = 6e-8 relative; the bar is 1e-5
    err = np.abs(got - ref)
    bad = err > TOL_SPMV * np.abs(ref)
    assert not bad.any(), f"{what}: max rel err {np.max(err[ref != 0] / np.abs(ref[ref != 0])):.3e}"
    assert np.all(got[ref == 0] == 0)


# ------------------------------------------------------------------------------------------ per pass
def test_forward_all_rows_and_dose_let_config0(fredopt, plan0):
    orc = _oracle(plan0)
    gp = fredopt.from_plan(plan0)
    x = pg.log_uniform_weights(7, plan0.n_cols)
    d_ref, l_ref, t_ref = orc.dose_let(x.astype(np.float64))
    d = np.full(plan0.n_rows, -1, np.float32); l = np.full(plan0.n_rows, -1, np.float32)
    gp.spmv_forward(fredopt.ROWS_ALL, x, d, l)
    _assert_fwd(d, d_ref, "D x")
    _assert_fwd(l, l_ref, "L x")
    # single-matrix passes
    d1 = np.empty_like(d); gp.spmv_forward(fredopt.ROWS_ALL, x, d1, None)
    l1 = np.empty_like(l); gp.spmv_forward(fredopt.ROWS_ALL, x, None, l1)
    assert np.array_equal(d1, d) and np.array_equal(l1, l)
    # dose_let: LETd = l / d, 0 where d = 0 (Eq. 1; reading R15)
    dose = np.empty_like(d); letd = np.empty_like(d)
    gp.dose_let(x, dose, letd)
    assert np.array_equal(dose, d)
    _assert_fwd(letd, t_ref, "LETd")
    # device pointers give the same bits as host pointers; x = NULL uses the plan's x
    gp.set_weights(x)
    dd = torch.empty(plan0.n_rows, dtype=torch.float32, device="cuda"); tt = torch.empty_like(dd)
    gp.dose_let(None, dd, tt)
    torch.cuda.synchronize()
    assert np.array_equal(dd.cpu().numpy(), dose) and np.array_equal(tt.cpu().numpy(), letd)


def test_forward_active_rows_config0(fredopt, plan0):
    orc = _oracle(plan0)
    gp = fredopt.from_plan(plan0)
    x = plan0.x0
    lab = plan0.labels.numpy()
    d_ref, l_ref, _ = orc.dose_let(x.astype(np.float64))
    d = np.empty(plan0.n_rows, np.float32); l = np.empty(plan0.n_rows, np.float32)
    gp.spmv_forward(fredopt.ROWS_ACTIVE, x, d, l)
    _assert_fwd(d, np.where(lab != 0, d_ref, 0.0), "D x (active)")
    _assert_fwd(l, np.where(lab != 0, l_ref, 0.0), "L x (active)")


@pytest.mark.parametrize("copt", INDEX_FORMS)
@pytest.mark.parametrize("rows", ["all", "active"])
def test_transpose_config0(fredopt, plan0, rows, copt):
    orc = _oracle(plan0)
    gp = fredopt.from_plan(plan0, **copt)
    V = plan0.n_rows
    # signed, dense coefficient vectors (lower-bound violations are negative)
    u = (pg.uniform01_array(11, V) - 0.4).astype(np.float32)
    v = (pg.uniform01_array(12, V) - 0.6).astype(np.float32)
    sel = fredopt.ROWS_ALL if rows == "all" else fredopt.ROWS_ACTIVE
    for uu, vv in ((u, v), (u, None), (None, v)):
        ref, ref_abs = orc.transpose(None if uu is None else uu.astype(np.float64),
                                     None if vv is None else vv.astype(np.float64), active_only=(rows == "active"))
        out = np.empty(plan0.n_cols, np.float32)
        gp.spmv_transpose(sel, uu, vv, out)
        err = np.abs(out.astype(np.float64) - ref)
        assert np.all(err <= TOL_SPMV * ref_abs + 1e-300), f"max {np.max(err / np.maximum(ref_abs, 1e-300)):.3e}"
        assert _rel_l2(out.astype(np.float64), ref) <= TOL_SPMV


def test_proximity_config0(fredopt, plan0):
    orc = _oracle(plan0)
    gp = fredopt.from_plan(plan0)
    for x in (plan0.x0, pg.log_uniform_weights(3, plan0.n_cols)):
        p_ref, n_ref = orc.proximity(x.astype(np.float64))
        p, n = gp.proximity(x)
        assert n == n_ref
        assert abs(p - p_ref) <= 1e-12 * abs(p_ref)
    st = gp.stats()
    os_ = orc.stats()
    assert st["n_sets"] == os_["n_sets"] and st["n_zero_norm_sets"] == os_["n_zero_norm_sets"]
    assert abs(st["weight_sum"] - os_["W"]) <= 1e-12 * os_["W"]
    assert st["nnz"] == plan0.nnz and st["n_active_rows"] == int((plan0.labels != 0).sum())


# ------------------------------------------------------------------------------------------ iteration
def _run_pair(fredopt, plan, n_iter, lam, beta0, a, opts=(), gp=None, orc=None, copt=None):
    orc = orc or _oracle(plan)
    gp = gp or fredopt.from_plan(plan, **(copt or {}))
    for k, v in opts:
        orc.set_option(k, v); gp.set_option(k, v)
    orc.set_x(plan.x0); gp.set_weights(plan.x0)
    orc.iterate(n_iter, lam, beta0, a); gp.iterate(n_iter, lam, beta0, a)
    return gp, orc


def _assert_state(gp, orc, tol=TOL_X20):
    xg, xo = _gpu_x(gp), orc.get_x()
    assert _rel_l2(xg, xo) <= tol, f"rel L2 {_rel_l2(xg, xo):.3e}"
    pg_, ng = gp.proximity(None)
    po, no = orc.proximity(None)
    assert ng == no, f"violation count {ng} vs oracle {no}"
    assert abs(pg_ - po) <= 1e-6 * abs(po) + 1e-300
    sg, so = gp.stats(), orc.stats()
    assert sg["k"] == so["k"] and sg["s"] == so["s"] and sg["trials"] == so["trials"]
    if so["last_beta"]:
        assert abs(sg["last_beta"] - so["last_beta"]) <= 1e-15 * so["last_beta"]


@pytest.mark.parametrize("copt", INDEX_FORMS)
@pytest.mark.parametrize("n_iter", [1, 20, 50])
def test_superiorized_iterations_config0(fredopt, plan0, n_iter, copt):
    sp = plan0.spec
    gp, orc = _run_pair(fredopt, plan0, n_iter, sp.lam, sp.beta0, sp.a, copt=copt)
    _assert_state(gp, orc)
    assert (_gpu_x(gp) >= 0).all()


@pytest.mark.parametrize("lam", [0.5, 1.0, 1.9, 2.0])
def test_pure_feasibility_seeking_config0(fredopt, plan0, lam):
    gp, orc = _run_pair(fredopt, plan0, 20, lam, 0.0, 0.5)
    _assert_state(gp, orc)
    assert gp.stats()["s"] == 0


def test_violation_count_identical_every_iteration_config0(fredopt, plan0):
    orc = _oracle(plan0); gp = fredopt.from_plan(plan0)
    orc.set_x(plan0.x0); gp.set_weights(plan0.x0)
    for _ in range(30):
        orc.iterate(1, 1.0, 1.0, 0.99); gp.iterate(1, 1.0, 1.0, 0.99)
        assert gp.proximity(None)[1] == orc.proximity(None)[1]


def test_options_eta_reductions_accept_maxtrials(fredopt, plan0):
    f = fredopt
    for opts in ([(f.OPT_ETA, 0.9)], [(f.OPT_REDUCTIONS, 3)], [(f.OPT_ACCEPT_CHECK, 0)],
                 [(f.OPT_ETA, 0.95), (f.OPT_REDUCTIONS, 2)]):
        gp, orc = _run_pair(fredopt, plan0, 12, 1.3, 1.0, 0.9, opts)
        _assert_state(gp, orc)
    # block-sequential sweep after two reductions (the residual pass of the last reduction writes no u, v there)
    from oracle import oracle as om
    gp = f.from_plan(plan0); orc = _oracle(plan0)
    for o_, m_ in ((gp, f), (orc, om)):
        o_.set_option(m_.OPT_BLOCK_SEQUENTIAL, 1); o_.set_option(m_.OPT_REDUCTIONS, 2)
    gp.set_weights(plan0.x0); orc.set_x(plan0.x0)
    gp.iterate(12, 1.3, 1.0, 0.9); orc.iterate(12, 1.3, 1.0, 0.9)
    _assert_block_state(gp, orc)
    # a cost step far too large: every trial up to the cap is rejected, x is kept, s still advances (R10)
    gp, orc = _run_pair(fredopt, plan0, 2, 1.0, 1.0e6, 0.999, [(f.OPT_MAX_TRIALS, 5)])
    _assert_state(gp, orc)
    assert gp.stats()["s"] == 10


def test_state_two_calls_equal_one_and_graph_equals_launches(fredopt, plan0):
    f = fredopt
    a = f.from_plan(plan0); a.set_weights(plan0.x0); a.iterate(20, 1.0, 1.0, 0.99)
    b = f.from_plan(plan0); b.set_weights(plan0.x0); b.iterate(10, 1.0, 1.0, 0.99); b.iterate(10, 1.0, 1.0, 0.99)
    c = f.from_plan(plan0); c.set_option(f.OPT_USE_GRAPH, 0); c.set_weights(plan0.x0); c.iterate(20, 1.0, 1.0, 0.99)
    d = f.from_plan(plan0); d.set_option(f.OPT_USE_PDL, 0); d.set_weights(plan0.x0); d.iterate(20, 1.0, 1.0, 0.99)
    e = f.from_plan(plan0); e.set_weights(plan0.x0); e.iterate(8, 1.0, 1.0, 0.99); e.set_option(f.OPT_USE_PDL, 0); e.iterate(12, 1.0, 1.0, 0.99)
    xa, xb, xc = _gpu_x(a), _gpu_x(b), _gpu_x(c)
    assert np.array_equal(xa, xb) and np.array_equal(xa, xc)      # no atomics: bitwise reproducible
    assert np.array_equal(xa, _gpu_x(d)) and np.array_equal(xa, _gpu_x(e))     # with and without programmatic dependent launch
    # RESET restarts beta at beta0
    a.set_option(f.OPT_RESET, 1); a.set_weights(plan0.x0); a.iterate(20, 1.0, 1.0, 0.99)
    assert np.array_equal(_gpu_x(a), xa)
    assert a.launch_count() > 0


def test_rejected_trials_multi_beam(fredopt):
    """Three beams: the first iterations reject many step sizes (reading R8); the device-side accept loop must
    consume exactly the trials the oracle's literal re-evaluation consumes."""
    plan = pg.build_plan(pg.config_spec(2, scale=0.25), device="cuda")
    gp, orc = _run_pair(fredopt, plan, 20, 1.0, 1.0, 0.99)
    assert orc.stats()["trials"] > 20
    _assert_state(gp, orc)


# ------------------------------------------------------------------------------------------ small / ragged / degenerate
@pytest.mark.parametrize("rows", [0, 1, 2, 4])
@pytest.mark.parametrize("seed,same", [(1, True), (2, False), (5, False)])
def test_random_small_plans_union_pattern(fredopt, seed, same, rows):
    V, S = 300, 37
    D, L, lab, x0 = pg.random_small_plan(seed, V=V, S=S, n_struct=3, density=0.3, same_pattern=same)
    nan = np.nan
    bounds = np.array([[1.0, 0.5, 0.9, nan, nan, nan, 0.7, nan],
                       [2.0, nan, 0.4, nan, 1.5, 3.0, nan, 1.5],
                       [0.5, 0.1, nan, 0.2, 2.0, nan, 0.3, 1.0]], np.float32)
    orc = _oracle_np(V, S, D, L, lab, bounds)
    gp = fredopt.Plan(V, S, D, L, lab, bounds, block_rows=rows)
    assert gp.stats()["block_rows"] == rows or rows == 0
    x = x0
    d_ref, l_ref, _ = orc.dose_let(x.astype(np.float64))
    d = np.empty(V, np.float32); l = np.empty(V, np.float32)
    gp.spmv_forward(fredopt.ROWS_ALL, x, d, l)
    _assert_fwd(d, d_ref, "D x"); _assert_fwd(l, l_ref, "L x")
    orc.set_x(x0); gp.set_weights(x0)
    orc.iterate(20, 1.5, 0.5, 0.8); gp.iterate(20, 1.5, 0.5, 0.8)
    _assert_state(gp, orc)


@pytest.mark.parametrize("seed", list(range(20, 32)))
def test_random_bound_combinations(fredopt, seed):
    """Random presence / absence of every bound and cost reference per structure, random weights, both AMS forms, ragged
    shapes (V, S not multiples of anything), differing D / L patterns on odd seeds."""
    from oracle import oracle as om
    u = pg.uniform01_array(1000 + seed, 64)
    V, S, ns = 150 + int(u[0] * 400), 5 + int(u[1] * 90), 1 + int(u[2] * 5)
    D, L, lab, x0 = pg.random_small_plan(seed, V=V, S=S, n_struct=ns, density=0.15 + 0.5 * u[3], same_pattern=seed % 2 == 0)
    nan = np.nan
    rows = []
    for s_ in range(ns):
        r = pg.uniform01_array(2000 + seed * 16 + s_, 12)
        lo, hi = 0.2 + 0.6 * r[0], 1.0 + 0.8 * r[1]
        rows.append([0.25 + 2.0 * r[2],
                     lo if r[3] < 0.5 else nan, hi if r[4] < 0.6 else nan,
                     2.0 * lo if r[5] < 0.3 else nan, 3.0 * hi if r[6] < 0.5 else nan,
                     2.0 + 3.0 * r[7] if r[8] < 0.5 else nan,
                     0.5 * (lo + hi) if r[9] < 0.6 else nan, 2.5 * hi if r[10] < 0.5 else nan])
    bounds = np.array(rows, np.float32)
    for block in (0, 1):
        orc = _oracle_np(V, S, D, L, lab, bounds)
        gp = fredopt.Plan(V, S, D, L, lab, bounds, block_rows=(0, 1, 2, 4)[seed % 4])
        gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, block); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, block)
        orc.set_x(x0); gp.set_weights(x0)
        orc.iterate(20, 1.3, 0.8, 0.85); gp.iterate(20, 1.3, 0.8, 0.85)
        if block:
            _assert_block_state(gp, orc)
        else:
            _assert_state(gp, orc)
        gp.destroy()


def test_more_than_65536_spots_uses_32_bit_columns(fredopt):
    """n_cols > 65536: the forward kernels read int32 column indices while the transposes keep 16-bit row indices."""
    V, S, per_row = 500, 70000, 40
    u = pg.uniform01_array(77, V * per_row * 3 + V)
    cols = np.sort((u[:V * per_row].reshape(V, per_row) * (S // per_row)).astype(np.int64) + np.arange(per_row) * (S // per_row), axis=1)
    rp = np.arange(V + 1, dtype=np.int64) * per_row
    ci = cols.reshape(-1).astype(np.int32)
    vd = (0.05 + u[V * per_row:2 * V * per_row]).astype(np.float32)
    vl = (vd * (2.0 + 6.0 * u[2 * V * per_row:3 * V * per_row])).astype(np.float32)
    lab = (np.floor(u[3 * V * per_row:] * 3)).astype(np.int32)
    nan = np.nan
    bounds = np.array([[1.0, 8.0, 11.0, nan, nan, nan, 10.0, nan],
                       [1.0, nan, 9.0, nan, 40.0, 4.5, nan, 35.0]], np.float32)
    assert ci.max() > 65536
    orc = _oracle_np(V, S, (rp, ci, vd), (rp, ci, vl), lab, bounds)
    gp = fredopt.Plan(V, S, (rp, ci, vd), (rp, ci, vl), lab, bounds)
    x0 = (0.2 + 0.5 * pg.uniform01_array(78, S)).astype(np.float32)
    d_ref, l_ref, _ = orc.dose_let(x0.astype(np.float64))
    d = np.empty(V, np.float32); l = np.empty(V, np.float32)
    gp.spmv_forward(fredopt.ROWS_ALL, x0, d, l)
    _assert_fwd(d, d_ref, "D x"); _assert_fwd(l, l_ref, "L x")
    orc.set_x(x0); gp.set_weights(x0)
    orc.iterate(20, 1.0, 1.0, 0.9); gp.iterate(20, 1.0, 1.0, 0.9)
    _assert_state(gp, orc)


def test_degenerate_inputs(fredopt):
    f = fredopt
    nan = np.nan
    b1 = np.array([[1.0, nan, 1.0, nan, nan, nan, nan, nan]], np.float32)
    # all rows empty: nothing participates, x is unchanged, a violated lower bound on an unreachable voxel is counted (R14)
    V, S = 5, 3
    rp = np.zeros(V + 1, np.int64); ci = np.zeros(0, np.int32); vv = np.zeros(0, np.float32)
    lab = np.array([0, 1, 1, 0, 1], np.int32)
    blo = np.array([[1.0, 0.5, nan, nan, nan, nan, nan, nan]], np.float32)
    gp = f.Plan(V, S, (rp, ci, vv), (rp, ci, vv), lab, blo)
    x = np.array([1, 2, 3], np.float32)
    gp.set_weights(x); gp.iterate(3, 1.0, 1.0, 0.5)
    assert np.array_equal(_gpu_x(gp), x.astype(np.float64))
    assert gp.proximity(None) == (0.0, 3)
    orc = _oracle_np(V, S, (rp, ci, vv), (rp, ci, vv), lab, blo)
    orc.set_x(x); orc.iterate(3, 1.0, 1.0, 0.5)
    assert orc.proximity(None) == (0.0, 3)
    # no labelled voxel / no structure
    rp = np.array([0, 2, 2, 3], np.int64); ci = np.array([0, 1, 1], np.int32); vv = np.array([1, 2, 3], np.float32)
    gp = f.Plan(3, 2, (rp, ci, vv), (rp, ci, vv), np.zeros(3, np.int32), np.zeros((0, 8), np.float32))
    gp.set_weights(np.array([1, 1], np.float32)); gp.iterate(2, 1.0, 0.0, 0.5)
    d = np.empty(3, np.float32); gp.spmv_forward(f.ROWS_ALL, None, d, None)
    assert np.array_equal(d, np.array([3, 0, 3], np.float32))
    # one very long row (several 256-entry tiles and a ragged tail) and rows of length 1..9
    S = 3001
    lens = [S, 1, 2, 3, 4, 5, 6, 7, 8, 9, 0, 257, 511]
    rp = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    ci = np.concatenate([np.arange(n, dtype=np.int32) * (S // max(n, 1)) for n in lens]).astype(np.int32)
    vv = (0.1 + pg.uniform01_array(9, int(rp[-1]))).astype(np.float32)
    vl = (vv * (2 + pg.uniform01_array(10, int(rp[-1])))).astype(np.float32)
    lab = np.ones(len(lens), np.int32)
    b = np.array([[1.0, 1.0, 2.0, nan, 30.0, 3.0, 1.5, nan]], np.float32)
    gp = f.Plan(len(lens), S, (rp, ci, vv), (rp, ci, vl), lab, b)
    orc = _oracle_np(len(lens), S, (rp, ci, vv), (rp, ci, vl), lab, b)
    x0 = pg.log_uniform_weights(4, S)
    orc.set_x(x0); gp.set_weights(x0)
    orc.iterate(20, 1.0, 0.3, 0.9); gp.iterate(20, 1.0, 0.3, 0.9)
    _assert_state(gp, orc)


def test_invalid_arguments(fredopt):
    f = fredopt
    nan = np.nan
    rp = np.array([0, 2, 3], np.int64); ci = np.array([0, 1, 1], np.int32); vv = np.array([1, 2, 3], np.float32)
    lab = np.array([1, 0], np.int32)
    b = np.array([[1.0, nan, 1.0, nan, nan, nan, nan, nan]], np.float32)

    def bad(**kw):
        a = dict(rp=rp, ci=ci, vv=vv, lab=lab, b=b)
        a.update(kw)
        with pytest.raises(f.FredoptError) as e:
            f.Plan(2, 2, (a["rp"], a["ci"], a["vv"]), (a["rp"], a["ci"], a["vv"]), a["lab"], a["b"])
        assert e.value.code == f.INVALID_ARG

    bad(rp=np.array([0, 3, 2], np.int64))                      # decreasing row_ptr
    bad(rp=np.array([1, 2, 3], np.int64))                      # row_ptr[0] != 0
    bad(ci=np.array([1, 0, 1], np.int32))                      # unsorted columns
    bad(ci=np.array([0, 0, 1], np.int32))                      # duplicate column
    bad(ci=np.array([0, 2, 1], np.int32))                      # column out of range
    bad(vv=np.array([1, np.inf, 3], np.float32))               # non-finite value
    bad(lab=np.array([2, 0], np.int32))                        # label outside 0..n_struct
    bad(b=np.array([[0.0, nan, 1.0, nan, nan, nan, nan, nan]], np.float32))    # weight <= 0
    bad(b=np.array([[1.0, 2.0, 1.0, nan, nan, nan, nan, nan]], np.float32))    # lo > hi
    gp = f.Plan(2, 2, (rp, ci, vv), (rp, ci, vv), lab, b)
    x = np.array([1, 1], np.float32); gp.set_weights(x)
    for args in ((-1, 1.0, 1.0, 0.5), (1, 0.0, 1.0, 0.5), (1, 2.5, 1.0, 0.5), (1, 1.0, -1.0, 0.5), (1, 1.0, 1.0, 1.0),
                 (1, 1.0, 1.0, 0.0)):
        with pytest.raises(f.FredoptError):
            gp.iterate(*args)
    assert np.array_equal(_gpu_x(gp), x.astype(np.float64))    # state untouched on failure
    with pytest.raises(f.FredoptError):
        gp.set_option(99, 1.0)


# ------------------------------------------------------------------------------------------ options of Fig. 3 / Eq. (2)
@pytest.mark.parametrize("norm,one_sided", [(1, 0), (0, 1), (1, 1)])
def test_options_normalised_gradient_and_one_sided_cost(fredopt, norm, one_sided):
    """R9 / R11 options on a plan with both cost terms; the one-sided accept loop runs its trials on the stored products."""
    from oracle import oracle as om
    V, S = 300, 37
    D, L, lab, x0 = pg.random_small_plan(8, V=V, S=S, n_struct=3, density=0.3)
    nan = np.nan
    bounds = np.array([[1.0, 0.5, 0.9, nan, nan, nan, 0.7, nan],
                       [2.0, nan, 0.4, nan, 1.5, 3.0, nan, 1.0],
                       [0.5, 0.1, nan, 0.2, 2.0, nan, 0.3, 0.8]], np.float32)
    orc = _oracle_np(V, S, D, L, lab, bounds)
    gp = fredopt.Plan(V, S, D, L, lab, bounds)
    for g_, o_, v in ((fredopt.OPT_NORMALIZE_GRAD, om.OPT_NORMALIZE_GRAD, norm), (fredopt.OPT_ONE_SIDED_COST, om.OPT_ONE_SIDED_COST, one_sided)):
        gp.set_option(g_, v); orc.set_option(o_, v)
    orc.set_x(x0); gp.set_weights(x0)
    orc.iterate(20, 1.2, 2.0, 0.7); gp.iterate(20, 1.2, 2.0, 0.7)       # beta0 = 2: the first trials are rejected
    assert orc.stats()["trials"] > 20
    _assert_state(gp, orc)


def test_options_on_three_beam_plan(fredopt):
    from oracle import oracle as om
    plan = pg.build_plan(pg.config_spec(2, scale=0.25), device="cuda")
    gp = fredopt.from_plan(plan, stream=torch.cuda.current_stream().cuda_stream); orc = _oracle(plan)
    gp.set_option(fredopt.OPT_ONE_SIDED_COST, 1); orc.set_option(om.OPT_ONE_SIDED_COST, 1)
    gp.set_weights(plan.x0); orc.set_x(plan.x0)
    gp.iterate(20, 1.0, 1.0, 0.99); orc.iterate(20, 1.0, 1.0, 0.99)
    _assert_state(gp, orc)


# ------------------------------------------------------------------------------------------ evaluation quantities
def _assert_evaluation(gp, orc, n_struct, x):
    x64 = x.astype(np.float64)
    for label in range(1, n_struct + 1):
        for q in (0, 1, 2):
            mn, mean, mx, n = gp.structure_stats(q, label, x)
            omn, omean, omx, on = orc.structure_stats(q, label, x64)
            assert n == on
            assert np.allclose([mn, mean, mx], [omn, omean, omx], rtol=1e-12, atol=1e-300)
            if n == 0 or omx <= 0:
                continue
            for frac in (0.02, 0.3, 0.5, 1.0):
                assert abs(gp.percentile_value(q, label, frac, x) - orc.percentile_value(q, label, frac, x64)) <= 1e-12 * omx
            hist = np.empty(64, np.float32)
            gp.volume_histogram(q, label, 64, omx * 1.05, hist, x)
            ref = orc.volume_histogram(q, label, 64, omx * 1.05, x64)
            assert np.all(np.abs(hist - ref) <= 1.5 / n + 1e-6)      # a value within rounding of a bin edge may move one voxel
            assert hist[0] == 1.0


def test_evaluation_quantities_config0(fredopt, plan0):
    gp = fredopt.from_plan(plan0); orc = _oracle(plan0)
    _assert_evaluation(gp, orc, 2, plan0.x0)
    # and at the plan's own x after some iterations (x = NULL)
    gp.set_weights(plan0.x0); gp.iterate(10, 1.0, 1.0, 0.99)
    orc.set_x(plan0.x0); orc.iterate(10, 1.0, 1.0, 0.99)
    v = gp.percentile_value(0, 2, 0.3)
    assert abs(v - orc.percentile_value(0, 2, 0.3)) <= 1e-12 * max(abs(v), 1e-30)
    with pytest.raises(fredopt.FredoptError):
        gp.percentile_value(0, 3, 0.3)
    with pytest.raises(fredopt.FredoptError):
        gp.percentile_value(3, 1, 0.3)
    with pytest.raises(fredopt.FredoptError):
        gp.percentile_value(0, 1, 0.0)


def test_evaluation_quantities_three_beam_plan(fredopt):
    plan = pg.build_plan(pg.config_spec(2, scale=0.25), device="cuda")
    gp = fredopt.from_plan(plan, stream=torch.cuda.current_stream().cuda_stream); orc = _oracle(plan)
    _assert_evaluation(gp, orc, 4, pg.log_uniform_weights(3, plan.n_cols))


# ------------------------------------------------------------------------------------------ block-sequential AMS (R23)
def _assert_block_state(gp, orc):
    po, no = orc.sweep_stats()
    sg = gp.stats()                      # before _assert_state: fredopt_proximity overwrites these two statistics
    assert sg["n_violated"] == no, f"sets violated when visited: {sg['n_violated']} vs oracle {no}"
    assert abs(sg["prox"] - po) <= 1e-9 * abs(po) + 1e-300
    _assert_state(gp, orc)


@pytest.mark.parametrize("copt", INDEX_FORMS)
@pytest.mark.parametrize("beta0", [0.0, 1.0])
@pytest.mark.parametrize("lam", [1.0, 1.7])
def test_block_sequential_config0(fredopt, plan0, beta0, lam, copt):
    """Fig. 2's loop nest block by block (option BLOCK_SEQUENTIAL), pure and superiorized, 20 iterations."""
    from oracle import oracle as om
    gp = fredopt.from_plan(plan0, **copt); orc = _oracle(plan0)
    gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, 1); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, 1)
    gp.set_weights(plan0.x0); orc.set_x(plan0.x0)
    for n in (1, 19):                                          # one plain launch sequence, then graph replays
        gp.iterate(n, lam, beta0, 0.99); orc.iterate(n, lam, beta0, 0.99)
        _assert_block_state(gp, orc)
    # and back to the simultaneous step on the same plan
    gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, 0); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, 0)
    gp.iterate(3, lam, beta0, 0.99); orc.iterate(3, lam, beta0, 0.99)
    _assert_state(gp, orc)


@pytest.mark.parametrize("seed,same", [(3, True), (4, False)])
def test_block_sequential_random_small_plans(fredopt, seed, same):
    from oracle import oracle as om
    V, S = 300, 37
    D, L, lab, x0 = pg.random_small_plan(seed, V=V, S=S, n_struct=4, density=0.3, same_pattern=same)
    nan = np.nan
    bounds = np.array([[1.0, 0.5, 0.9, nan, nan, nan, 0.7, nan],
                       [2.0, nan, 0.4, nan, 1.5, 3.0, nan, 1.5],
                       [0.5, 0.1, nan, 0.2, 2.0, nan, 0.3, 1.0],
                       [0.25, nan, nan, nan, nan, 2.5, nan, nan]], np.float32)
    orc = _oracle_np(V, S, D, L, lab, bounds)
    gp = fredopt.Plan(V, S, D, L, lab, bounds)
    gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, 1); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, 1)
    gp.set_option(fredopt.OPT_ETA, 0.97); orc.set_option(om.OPT_ETA, 0.97)
    orc.set_x(x0); gp.set_weights(x0)
    orc.iterate(20, 1.5, 0.5, 0.8); gp.iterate(20, 1.5, 0.5, 0.8)
    _assert_block_state(gp, orc)


def test_block_sequential_three_beam_plan(fredopt):
    """A scaled configs[2] plan (three beams, four structures, all three kinds): 20 superiorized block-sequential iterations."""
    from oracle import oracle as om
    plan = pg.build_plan(pg.config_spec(2, scale=0.25), device="cuda")
    gp = fredopt.from_plan(plan, stream=torch.cuda.current_stream().cuda_stream); orc = _oracle(plan)
    gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, 1); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, 1)
    gp.set_weights(plan.x0); orc.set_x(plan.x0)
    gp.iterate(20, 1.0, 1.0, 0.99); orc.iterate(20, 1.0, 1.0, 0.99)
    _assert_block_state(gp, orc)


# ------------------------------------------------------------------------------------------ full-size configurations
def _full_size_parity(fredopt, plan, n_sample_rows, copt=None):
    """20 superiorized iterations in the launch configuration bench.py times (one fredopt_iterate call = graph replay),
    sampled outputs of the full forward pass computed one by one by the oracle, and the full transposed pass."""
    gp = fredopt.from_plan(plan, stream=torch.cuda.current_stream().cuda_stream, **(copt or {}))
    orc = _oracle(plan)
    sp = plan.spec
    orc.set_x(plan.x0); gp.set_weights(plan.x0)
    orc.iterate(20, sp.lam, sp.beta0, sp.a); gp.iterate(20, sp.lam, sp.beta0, sp.a)
    _assert_state(gp, orc)
    # sampled outputs of the full forward pass, computed one by one by the oracle
    x = pg.log_uniform_weights(21, plan.n_cols)
    dose = torch.empty(plan.n_rows, dtype=torch.float32, device="cuda"); letd = torch.empty_like(dose)
    gp.dose_let(torch.from_numpy(x).cuda(), dose, letd)
    torch.cuda.synchronize()
    nz = (plan.row_ptr[1:] > plan.row_ptr[:-1]).nonzero().reshape(-1).cpu().numpy()
    rows = nz[(pg.uniform01_array(22, n_sample_rows) * len(nz)).astype(np.int64)]
    d_ref, _, t_ref = orc.dose_let_rows(rows, x.astype(np.float64))
    _assert_fwd(dose.cpu().numpy()[rows], d_ref, "dose (sampled)")
    _assert_fwd(letd.cpu().numpy()[rows], t_ref, "LETd (sampled)")
    # rows no spot reaches are exactly 0
    empty = (plan.row_ptr[1:] == plan.row_ptr[:-1])
    assert float(dose[empty].abs().max().item() if bool(empty.any()) else 0.0) == 0.0
    # transposed pass over all rows, full size
    V = plan.n_rows
    u = (pg.uniform01_array(31, V) - 0.4).astype(np.float32); v = (pg.uniform01_array(32, V) - 0.6).astype(np.float32)
    ref, ref_abs = orc.transpose(u.astype(np.float64), v.astype(np.float64))
    out = np.empty(plan.n_cols, np.float32)
    gp.spmv_transpose(fredopt.ROWS_ALL, u, v, out)
    assert np.all(np.abs(out - ref) <= TOL_SPMV * ref_abs)
    # and over the labelled rows only, with the D-only and L-only forms
    for uu, vv in ((u, v), (u, None), (None, v)):
        ref, ref_abs = orc.transpose(None if uu is None else uu.astype(np.float64),
                                     None if vv is None else vv.astype(np.float64), active_only=True)
        gp.spmv_transpose(fredopt.ROWS_ACTIVE, uu, vv, out)
        assert np.all(np.abs(out - ref) <= TOL_SPMV * ref_abs)
    # block-sequential form (R23) from the same state, and the evaluation quantities of the PTV and one OAR
    from oracle import oracle as om
    gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, 1); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, 1)
    gp.iterate(5, sp.lam, sp.beta0, sp.a); orc.iterate(5, sp.lam, sp.beta0, sp.a)
    _assert_block_state(gp, orc)
    for label, q in ((1, 0), (2, 1), (2, 2)):
        v, vo = gp.percentile_value(q, label, 0.3), orc.percentile_value(q, label, 0.3)
        assert abs(v - vo) <= 1e-12 * max(abs(vo), 1e-30)
    gp.destroy()


@pytest.mark.parametrize("copt", INDEX_FORMS)
def test_config1_20_iterations_full_size(fredopt, copt):
    """BASELINE.json configs[1] (mid-size phantom, L2-resident working set), both stored index forms."""
    _full_size_parity(fredopt, pg.build_plan(pg.config_spec(1), device="cuda"), 4000, copt)


def test_config2_20_iterations_full_size(fredopt):
    """BASELINE.json configs[2] (three beams: the first iteration rejects ~200 step sizes), at full size."""
    _full_size_parity(fredopt, pg.build_plan(pg.config_spec(2), device="cuda"), 8000)


def test_config1_all_200_iterations(fredopt):
    """BASELINE.json configs[1] over its full iteration count: the violation count is compared every 25 iterations (SURVEY
    sec. 7.5: all-fp32 arithmetic flips it at 3 of 200 iterations here; fp64 vectors must not)."""
    plan = pg.build_plan(pg.config_spec(1), device="cuda")
    gp = fredopt.from_plan(plan, stream=torch.cuda.current_stream().cuda_stream)
    orc = _oracle(plan)
    sp = plan.spec
    orc.set_x(plan.x0); gp.set_weights(plan.x0)
    for _ in range(8):
        orc.iterate(25, sp.lam, sp.beta0, sp.a); gp.iterate(25, sp.lam, sp.beta0, sp.a)
        _assert_state(gp, orc)
    assert gp.stats()["k"] == sp.n_iter == 200


def test_config3_20_iterations_in_bench_configuration(fredopt):
    """BASELINE.json configs[3]: the workload bench.py times (1.15e9 non-zeros per matrix), at full size."""
    plan = pg.build_plan(pg.config_spec(3), device="cuda")
    assert plan.nnz > 1.0e9
    _full_size_parity(fredopt, plan, 20000)


@pytest.mark.skipif(os.environ.get("FREDOPT_LONG") != "1", reason="the full horizons of configs[2] and configs[3] take ~12 min of oracle time: FREDOPT_LONG=1")
@pytest.mark.parametrize("config", [2, 3])
def test_full_size_over_the_full_horizon(fredopt, config):
    """BASELINE.json configs[2] and configs[3] at full size over the 500 iterations they state: x, s, trials and the violation
    count against the oracle every 100 iterations (the record is profiles/r02_parity_full_horizon.md)."""
    plan = pg.build_plan(pg.config_spec(config), device="cuda")
    gp = fredopt.from_plan(plan, stream=torch.cuda.current_stream().cuda_stream); orc = _oracle(plan)
    sp = plan.spec
    assert sp.n_iter == 500
    gp.set_weights(plan.x0); orc.set_x(plan.x0)
    for k in range(5):
        gp.iterate(100, sp.lam, sp.beta0, sp.a); orc.iterate(100, sp.lam, sp.beta0, sp.a)
        xg, xo = _gpu_x(gp), orc.get_x()
        (pgp, ng), (po, no) = gp.proximity(None), orc.proximity(None)
        sg, so = gp.stats(), orc.stats()
        print(f"configs[{config}] after {100 * (k + 1)} iterations: rel L2(x) {_rel_l2(xg, xo):.3e}; violated sets gpu / oracle {ng} / {no}; "
              f"proximity {pgp:.9e} / {po:.9e}; s {sg['s']} / {so['s']}; trials {sg['trials']} / {so['trials']}")
        _assert_state(gp, orc)
    gp.destroy()


# ------------------------------------------------------------------------------------------ horizons, state, limits
def test_500_iterations_three_beam_plan(fredopt):
    """The horizon BASELINE.json configs[2] states (500 iterations) on the scaled three-beam plan, which rejects step sizes:
    s, trials, the violation count and x are compared with the oracle's from-definition accept test every 50 iterations."""
    plan = pg.build_plan(pg.config_spec(2, scale=0.25), device="cuda")
    gp = fredopt.from_plan(plan, stream=torch.cuda.current_stream().cuda_stream); orc = _oracle(plan)
    sp = plan.spec
    gp.set_weights(plan.x0); orc.set_x(plan.x0)
    for _ in range(10):
        gp.iterate(50, sp.lam, sp.beta0, sp.a); orc.iterate(50, sp.lam, sp.beta0, sp.a)
        _assert_state(gp, orc)
    st = gp.stats()
    assert st["k"] == 500 and st["trials"] > 500


def test_step_sizes_below_the_resolution_of_the_cost(fredopt, plan0):
    """a = 0.5: after ~60 trials beta |g|^2 falls below the fp64 resolution of chi^2.  Fig. 3 accepts iff chi^2(x - beta g) <
    chi^2(x) AS EVALUATED, so from then on every trial is rejected and s advances by max_trials per iteration; the closed form
    beta c < |g|^2 alone would accept them all.  Identical s while the decrease is far above the resolution; the same
    per-iteration advance far below it (in the few-ulp zone between, the two summation orders may decide differently)."""
    gp = fredopt.from_plan(plan0); orc = _oracle(plan0)
    gp.set_weights(plan0.x0); orc.set_x(plan0.x0)
    gp.iterate(30, 1.0, 1.0, 0.5); orc.iterate(30, 1.0, 1.0, 0.5)          # beta >= 2^-30: decrease ~1e-9 chi^2
    _assert_state(gp, orc)
    gp.iterate(50, 1.0, 1.0, 0.5); orc.iterate(50, 1.0, 1.0, 0.5)          # through the zone
    sg0, so0 = gp.stats()["s"], orc.stats()["s"]
    gp.iterate(5, 1.0, 1.0, 0.5); orc.iterate(5, 1.0, 1.0, 0.5)
    assert gp.stats()["s"] - sg0 == 5 * 200 and orc.stats()["s"] - so0 == 5 * 200
    xg, xo = _gpu_x(gp), orc.get_x()
    assert _rel_l2(xg, xo) <= TOL_X20
    assert gp.proximity(None)[1] == orc.proximity(None)[1]


def test_step_size_sequence_belongs_to_the_plan(fredopt, plan0):
    """GPU twin of oracle pin 26 (reading R8): AMS calls neither latch nor consume beta0 a^s; another pair needs a RESET."""
    f = fredopt
    gp = f.from_plan(plan0); orc = _oracle(plan0)
    gp.set_weights(plan0.x0); orc.set_x(plan0.x0)
    for n, b0, a in ((0, 0.7, 0.5), (2, 0.0, 0.5), (3, 0.5, 0.9), (2, 0.0, 0.9), (3, 0.5, 0.9)):
        gp.iterate(n, 1.0, b0, a); orc.iterate(n, 1.0, b0, a)
    _assert_state(gp, orc)
    for b0, a in ((0.25, 0.9), (0.5, 0.8)):
        with pytest.raises(f.FredoptError) as e:
            gp.iterate(1, 1.0, b0, a)
        assert e.value.code == f.INVALID_ARG
    from oracle import oracle as om
    gp.set_option(f.OPT_RESET, 1); orc.set_option(om.OPT_RESET, 1)
    gp.iterate(2, 1.0, 0.25, 0.8); orc.iterate(2, 1.0, 0.25, 0.8)
    _assert_state(gp, orc)


def test_negative_weight_on_a_spot_no_labelled_row_touches(fredopt):
    """Reading R6: the clamp runs over EVERY spot, also one that no labelled row reaches (x stays >= 0 at the ABI)."""
    nan = np.nan
    rp = np.array([0, 2, 4, 5], np.int64); ci = np.array([0, 1, 0, 1, 3], np.int32); vv = np.array([1, 2, 3, 1, 5], np.float32)
    lab = np.array([1, 1, 0], np.int32)                       # spot 2 is in no row at all, spot 3 only in an unlabelled row
    b = np.array([[1.0, nan, 1.0, nan, nan, nan, 0.5, nan]], np.float32)
    x0 = np.array([1.0, 1.0, -2.0, -3.0], np.float32)
    for beta0 in (0.0, 0.5):
        for block in (0, 1):
            gp = fredopt.Plan(3, 4, (rp, ci, vv), (rp, ci, vv), lab, b)
            orc = _oracle_np(3, 4, (rp, ci, vv), (rp, ci, vv), lab, b)
            from oracle import oracle as om
            gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, block); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, block)
            gp.set_weights(x0); orc.set_x(x0)
            gp.iterate(1, 1.0, beta0, 0.5); orc.iterate(1, 1.0, beta0, 0.5)
            xg = _gpu_x(gp)
            assert xg[2] == 0.0 and xg[3] == 0.0 and (xg >= 0).all()
            assert _rel_l2(xg, orc.get_x()) <= 1e-14


def test_more_structures_than_the_work_items_can_carry(fredopt):
    """n_struct > 255: FREDOPT_UNSUPPORTED (documented limit), never a wrong result."""
    nan = np.nan
    rp = np.array([0, 1], np.int64); ci = np.array([0], np.int32); vv = np.array([1.0], np.float32)
    b = np.tile(np.array([[1.0, nan, 1.0, nan, nan, nan, nan, nan]], np.float32), (256, 1))
    with pytest.raises(fredopt.FredoptError) as e:
        fredopt.Plan(1, 1, (rp, ci, vv), (rp, ci, vv), np.array([1], np.int32), b)
    assert e.value.code == fredopt.UNSUPPORTED
    gp = fredopt.Plan(1, 1, (rp, ci, vv), (rp, ci, vv), np.array([255], np.int32), b[:255])     # 255 structures are fine
    gp.set_weights(np.array([3.0], np.float32)); gp.iterate(1, 1.0, 0.0, 0.5)
    assert abs(_gpu_x(gp)[0] - 1.0) < 1e-15
    with pytest.raises(fredopt.FredoptError):
        fredopt.Plan(1, 1, (rp, ci, vv), (rp, ci, vv), np.array([1], np.int32), b[:1], index_width=8)


@pytest.mark.parametrize("copt", INDEX_FORMS)
def test_more_than_65536_labelled_rows(fredopt, copt):
    """More labelled rows than one 16-bit block of the transposes holds (several 65536-row blocks per spot run), cheaply: short
    random rows, two structures, both stored index forms."""
    V, S, per_row = 150000, 300, 6
    u = pg.uniform01_array(91, V * per_row * 3 + V)
    cols = np.sort((u[:V * per_row].reshape(V, per_row) * (S // per_row)).astype(np.int64) + np.arange(per_row) * (S // per_row), axis=1)
    rp = np.arange(V + 1, dtype=np.int64) * per_row
    ci = cols.reshape(-1).astype(np.int32)
    vd = (0.05 + u[V * per_row:2 * V * per_row]).astype(np.float32)
    vl = (vd * (2.0 + 6.0 * u[2 * V * per_row:3 * V * per_row])).astype(np.float32)
    lab = (1 + np.floor(u[3 * V * per_row:] * 2)).astype(np.int32)         # every row labelled: 150 000 > 2 x 65 536
    nan = np.nan
    bounds = np.array([[1.0, 0.8, 1.1, nan, nan, nan, 1.0, nan],
                       [1.0, nan, 0.9, nan, 4.0, 4.5, nan, 3.5]], np.float32)
    orc = _oracle_np(V, S, (rp, ci, vd), (rp, ci, vl), lab, bounds)
    gp = fredopt.Plan(V, S, (rp, ci, vd), (rp, ci, vl), lab, bounds, **copt)
    x0 = (0.2 + 0.5 * pg.uniform01_array(92, S)).astype(np.float32)
    uu = (pg.uniform01_array(93, V) - 0.4).astype(np.float32); vv_ = (pg.uniform01_array(94, V) - 0.6).astype(np.float32)
    ref, ref_abs = orc.transpose(uu.astype(np.float64), vv_.astype(np.float64), active_only=True)
    out = np.empty(S, np.float32)
    gp.spmv_transpose(fredopt.ROWS_ACTIVE, uu, vv_, out)
    assert np.all(np.abs(out - ref) <= TOL_SPMV * ref_abs)
    from oracle import oracle as om
    for block in (0, 1):
        gp.set_option(fredopt.OPT_RESET, 1); orc.set_option(om.OPT_RESET, 1)
        gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, block); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, block)
        orc.set_x(x0); gp.set_weights(x0)
        orc.iterate(10, 1.0, 1.0, 0.9); gp.iterate(10, 1.0, 1.0, 0.9)
        if block:
            _assert_block_state(gp, orc)
        else:
            _assert_state(gp, orc)


def test_work_distribution_never_changes_a_result(fredopt, plan0):
    """FREDOPT_OPT_WORK_QUEUE: items dealt statically or from the queue, in storage order or longest first, in either orientation
    -- the same bits in x after 20 superiorized + 5 block-sequential iterations (an item's sum is formed by one warp in a fixed
    order and lands in a place of its own; partial sums are added in a fixed order)."""
    f = fredopt
    ref = None
    for mode in range(16):
        gp = f.from_plan(plan0)
        gp.set_option(f.OPT_WORK_QUEUE, mode)
        gp.set_weights(plan0.x0)
        gp.iterate(20, 1.0, 1.0, 0.99)
        gp.set_option(f.OPT_BLOCK_SEQUENTIAL, 1)
        gp.iterate(5, 1.0, 1.0, 0.99)
        x = _gpu_x(gp)
        st = gp.stats()
        key = (st["k"], st["s"], st["trials"], st["n_violated"], st["prox"])
        if ref is None:
            ref = (x, key)
        assert np.array_equal(x, ref[0]) and key == ref[1], f"mode {mode}"
        gp.destroy()
    with pytest.raises(f.FredoptError):
        gp = f.from_plan(plan0); gp.set_option(f.OPT_WORK_QUEUE, 16)


@pytest.mark.parametrize("copt", INDEX_FORMS)
@pytest.mark.parametrize("beta0", [0.0, 1.0])
def test_skipping_rows_without_a_coefficient_never_changes_a_result(fredopt, plan0, beta0, copt):
    """FREDOPT_OPT_SKIP_SATISFIED: the back-projection streams the values of a (block) row only if the row has a non-zero step
    coefficient (Fig. 2 touches a row only when its test fires).  Every skipped term is an exact zero, so x,
    the counters and the statistics carry the same bits with the option on and off -- superiorized and pure feasibility-seeking
    (the two kernels that write the liveness bytes), every stored form, reductionsN = 2 -- and both match the oracle."""
    f = fredopt
    from oracle import oracle as om
    res = []
    for skip in (1, 0):
        gp = f.from_plan(plan0, **copt)
        gp.set_option(f.OPT_SKIP_SATISFIED, skip)
        gp.set_weights(plan0.x0)
        gp.iterate(30, 1.0, beta0, 0.99)
        gp.set_option(f.OPT_REDUCTIONS, 2)
        gp.iterate(5, 1.7, beta0, 0.99)
        st = gp.stats()
        res.append((_gpu_x(gp), (st["k"], st["s"], st["trials"], st["n_violated"], st["prox"], st["phi"])))
        if skip:
            orc = _oracle(plan0)
            orc.set_x(plan0.x0)
            orc.iterate(30, 1.0, beta0, 0.99)
            orc.set_option(om.OPT_REDUCTIONS, 2)
            orc.iterate(5, 1.7, beta0, 0.99)
            _assert_state(gp, orc)
        gp.destroy()
    assert np.array_equal(res[0][0], res[1][0]) and res[0][1] == res[1][1]


def test_skipping_on_a_plan_where_most_rows_are_satisfied(fredopt):
    """A three-beam plan driven close to feasibility (block-sequential sweeps first): afterwards few rows carry a coefficient, the
    timed byte count of the back-projection (fredopt_get_pass_bytes_timed) falls below the static one, and the simultaneous
    iterations that follow are bit-identical with and without skipping."""
    f = fredopt
    spec = pg.config_spec(2, scale=0.2)
    plan = pg.build_plan(spec, device="cuda")
    xs = []
    for skip in (1, 0):
        gp = f.from_plan(plan)
        gp.set_option(f.OPT_SKIP_SATISFIED, skip)
        gp.set_weights(plan.x0)
        gp.set_option(f.OPT_BLOCK_SEQUENTIAL, 1)
        gp.iterate(150, 1.0, 0.0, 0.99)
        gp.set_option(f.OPT_BLOCK_SEQUENTIAL, 0)
        gp.set_option(f.OPT_TIME_PASSES, 1)
        gp.iterate(10, 1.0, 0.0, 0.99)
        static, timed = gp.pass_bytes(), gp.pass_bytes_timed()
        gp.set_option(f.OPT_TIME_PASSES, 0)
        gp.iterate(10, 1.0, 1.0, 0.99)
        xs.append(_gpu_x(gp))
        st = gp.stats()
        if skip:
            assert timed["transpose_b"] < static["transpose_b"], (timed, static)
            assert timed["forward_x"] == static["forward_x"]
            assert st["n_violated"] < 0.5 * st["n_sets"]
        else:
            assert timed["transpose_b"] == static["transpose_b"]
        gp.destroy()
    assert np.array_equal(xs[0], xs[1])


# ------------------------------------------------------------------------------------------ 16-bit values
def _rounded_to_half(plan):
    """The plan of the matrices rounded to IEEE half by numpy (float32 -> float16 -> float32): what value_bits = 16 stores."""
    import dataclasses
    rd = lambda t: torch.from_numpy(t.cpu().numpy().astype(np.float16).astype(np.float32)).to(t.device)
    return dataclasses.replace(plan, val_D=rd(plan.val_D), val_L=rd(plan.val_L))


@pytest.mark.parametrize("copt", [pytest.param({}, id="auto"), pytest.param({"block_rows": 1}, id="rows1"),
                                  pytest.param({"block_rows": 4, "index_width": 32}, id="rows4-idx32")])
def test_16_bit_values_are_the_plan_of_the_rounded_matrices(fredopt, plan0, copt):
    """fredopt_create_options.value_bits = 16 (SURVEY sec. 8f-2 "16-bit values ... parity to be re-established"): the library
    rounds every value of D and L to the nearest IEEE half and streams 2-byte copies.  Parity is re-established against the
    oracle fed the SAME rounding done independently (numpy's float16 conversion): iterations within the usual bars, and -- since
    half -> float is exact and the kernels add in the same order -- the same bits in x as the fp32-storage plan of the rounded
    matrices; forward, transposed, block-sequential and evaluation calls agree too; the fp32 plan of the ORIGINAL matrices
    differs (the rounding is real); a value beyond the range of a half is refused."""
    f = fredopt
    pr = _rounded_to_half(plan0)
    assert not torch.equal(pr.val_D, plan0.val_D)
    sp = plan0.spec
    gp = f.from_plan(plan0, value_bits=16, **copt)               # the library rounds
    g32 = f.from_plan(pr, **copt)                                # fp32 storage of the rounded matrices
    orc = _oracle(pr)
    assert gp.pass_bytes()["forward_x"] < g32.pass_bytes()["forward_x"]
    for p_ in (gp, g32):
        p_.set_weights(plan0.x0)
        p_.iterate(30, sp.lam, sp.beta0, sp.a)
    orc.set_x(plan0.x0); orc.iterate(30, sp.lam, sp.beta0, sp.a)
    _assert_state(gp, orc)
    assert np.array_equal(_gpu_x(gp), _gpu_x(g32))
    # forward over all rows (fp32 row set of the rounded values) and over the labelled rows (half copies)
    x = pg.log_uniform_weights(7, plan0.n_cols)
    d_ref, l_ref, t_ref = orc.dose_let(x.astype(np.float64))
    dose = np.empty(plan0.n_rows, np.float32); letd = np.empty(plan0.n_rows, np.float32)
    gp.dose_let(x, dose, letd)
    _assert_fwd(dose, d_ref, "dose"); _assert_fwd(letd, t_ref, "LETd")
    d = np.empty(plan0.n_rows, np.float32); l = np.empty(plan0.n_rows, np.float32)
    gp.spmv_forward(f.ROWS_ACTIVE, x, d, l)
    lab = plan0.labels.numpy() > 0
    _assert_fwd(d[lab], d_ref[lab], "D x (labelled)"); _assert_fwd(l[lab], l_ref[lab], "L x (labelled)")
    # transposed over the labelled rows
    V = plan0.n_rows
    u = (pg.uniform01_array(31, V) - 0.4).astype(np.float32); v = (pg.uniform01_array(32, V) - 0.6).astype(np.float32)
    ref, ref_abs = orc.transpose(u.astype(np.float64), v.astype(np.float64), active_only=True)
    out = np.empty(plan0.n_cols, np.float32)
    gp.spmv_transpose(f.ROWS_ACTIVE, u, v, out)
    assert np.all(np.abs(out - ref) <= TOL_SPMV * ref_abs)
    # block-sequential form
    from oracle import oracle as om
    gp.set_option(f.OPT_BLOCK_SEQUENTIAL, 1); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, 1)
    gp.iterate(5, sp.lam, sp.beta0, sp.a); orc.iterate(5, sp.lam, sp.beta0, sp.a)
    _assert_block_state(gp, orc)
    # the rounding is real: the plan of the original matrices goes elsewhere
    g0 = f.from_plan(plan0, **copt)
    g0.set_weights(plan0.x0); g0.iterate(30, sp.lam, sp.beta0, sp.a)
    g32.set_option(f.OPT_RESET, 1); g32.set_weights(plan0.x0); g32.iterate(30, sp.lam, sp.beta0, sp.a)
    assert 1e-7 < _rel_l2(_gpu_x(g0), _gpu_x(g32)) < 1e-2
    for p_ in (gp, g32, g0):
        p_.destroy()
    # out of range
    big = _rounded_to_half(plan0)
    vd = plan0.val_D.clone(); vd[0] = 7.0e4
    import dataclasses
    with pytest.raises(f.FredoptError) as e:
        f.from_plan(dataclasses.replace(plan0, val_D=vd), value_bits=16)
    assert e.value.code == f.INVALID_ARG
    with pytest.raises(f.FredoptError):
        f.from_plan(plan0, value_bits=8)


def test_16_bit_values_three_beam_plan(fredopt):
    """The same on a three-beam plan (rejected step sizes, LETd rows that read both matrices) with 20 + 5 iterations."""
    f = fredopt
    plan = pg.build_plan(pg.config_spec(2, scale=0.2), device="cuda")
    pr = _rounded_to_half(plan)
    sp = plan.spec
    gp = f.from_plan(plan, value_bits=16); orc = _oracle(pr)
    gp.set_weights(plan.x0); orc.set_x(plan.x0)
    gp.iterate(20, sp.lam, sp.beta0, sp.a); orc.iterate(20, sp.lam, sp.beta0, sp.a)
    _assert_state(gp, orc)
    gp.iterate(5, sp.lam, 0.0, sp.a); orc.iterate(5, sp.lam, 0.0, sp.a)
    _assert_state(gp, orc)
    gp.destroy()


# ------------------------------------------------------------------------------------------ per-voxel bounds
def _varying_voxel_bounds(plan, bounds, seed):
    """Per-voxel arrays around the structures' scalars (+-, NaN on ~30 % of the voxels), voxel-indexed float32, for every field."""
    lab = plan.labels.cpu().numpy() if hasattr(plan.labels, "cpu") else np.asarray(plan.labels)
    V = len(lab)
    u = pg.uniform01_array(seed, 8 * V).reshape(8, V)
    out = {}
    for field in range(7):
        col = np.where(lab > 0, bounds[np.maximum(lab, 1) - 1, field + 1], np.nan).astype(np.float64)
        scale = 0.8 + 0.4 * u[field]
        if field in (0, 2):
            scale = 0.7 + 0.25 * u[field]
        if field in (1, 3):
            scale = 1.0 + 0.3 * u[field]
        out[field] = np.where(u[7] < 0.3, np.nan, col * scale).astype(np.float32)
    return out


@pytest.mark.parametrize("copt", [pytest.param({}, id="auto"), pytest.param({"block_rows": 1}, id="rows1"), pytest.param({"block_rows": 4}, id="rows4")])
def test_per_voxel_bounds_config0(fredopt, plan0, copt):
    from oracle import oracle as om
    f = fredopt
    # arrays of the structures' own scalars: the same bits as the scalar plan
    a = f.from_plan(plan0, **copt); b = f.from_plan(plan0, **copt)
    lab = plan0.labels.numpy()
    for field in range(7):
        col = np.where(lab > 0, plan0.bounds[np.maximum(lab, 1) - 1, field + 1], np.nan).astype(np.float32)
        b.set_voxel_bounds(field, col)
    for g in (a, b):
        g.set_weights(plan0.x0); g.iterate(20, 1.0, 1.0, 0.99)
    assert np.array_equal(_gpu_x(a), _gpu_x(b)) and a.stats() == b.stats()
    # genuinely varying bounds, both AMS forms, against the oracle
    vb = _varying_voxel_bounds(plan0, plan0.bounds, 5)
    for block in (0, 1):
        gp = f.from_plan(plan0, **copt); orc = _oracle(plan0)
        for field, arr in vb.items():
            gp.set_voxel_bounds(field, torch.from_numpy(arr).cuda() if field % 2 else arr)     # device and host pointers
            orc.set_voxel_bounds(field, arr)
        assert abs(gp.stats()["weight_sum"] - orc.stats()["W"]) <= 1e-12 * orc.stats()["W"]
        gp.set_option(f.OPT_BLOCK_SEQUENTIAL, block); orc.set_option(om.OPT_BLOCK_SEQUENTIAL, block)
        gp.set_weights(plan0.x0); orc.set_x(plan0.x0)
        gp.iterate(20, 1.0, 1.0, 0.99); orc.iterate(20, 1.0, 1.0, 0.99)
        if block:
            _assert_block_state(gp, orc)
        else:
            _assert_state(gp, orc)
        # the arrays matter: the scalar plan is elsewhere
        assert _rel_l2(_gpu_x(gp), _gpu_x(a)) > 1e-4 or block
    # removing the arrays restores the scalar plan; invalid arrays are refused and change nothing
    for field in range(7):
        gp.set_voxel_bounds(field, None)
    gp.set_option(f.OPT_BLOCK_SEQUENTIAL, 0); gp.set_option(f.OPT_RESET, 1)
    gp.set_weights(plan0.x0); gp.iterate(20, 1.0, 1.0, 0.99)
    assert np.array_equal(_gpu_x(gp), _gpu_x(a))
    with pytest.raises(f.FredoptError) as e:
        gp.set_voxel_bounds(f.VB_DOSE_LO, np.full(plan0.n_rows, 9.0, np.float32))          # above the PTV's dose_hi
    assert e.value.code == f.INVALID_ARG
    with pytest.raises(f.FredoptError):
        gp.set_voxel_bounds(f.VB_DOSE_HI, np.full(plan0.n_rows, np.inf, np.float32))
    with pytest.raises(f.FredoptError):
        gp.set_voxel_bounds(7, np.zeros(plan0.n_rows, np.float32))
    gp.set_option(f.OPT_RESET, 1); gp.set_weights(plan0.x0); gp.iterate(20, 1.0, 1.0, 0.99)
    assert np.array_equal(_gpu_x(gp), _gpu_x(a))


@pytest.mark.parametrize("seed", [3, 4])
def test_per_voxel_bounds_random_plans_one_sided_cost(fredopt, seed):
    """Differing D / L patterns, every field varying per voxel, reductionsN = 2 and the one-sided cost (its accept loop reads
    the per-voxel cDL references from the stored products)."""
    from oracle import oracle as om
    V, S = 300, 37
    D, L, lab, x0 = pg.random_small_plan(seed, V=V, S=S, n_struct=3, density=0.3, same_pattern=False)
    nan = np.nan
    bounds = np.array([[1.0, 0.5, 0.9, nan, nan, nan, 0.7, nan],
                       [2.0, nan, 0.4, nan, 1.5, 3.0, nan, 1.0],
                       [0.5, 0.1, nan, 0.2, 2.0, 2.5, 0.3, 0.8]], np.float32)

    class _P:
        labels = lab
    vb = _varying_voxel_bounds(_P, bounds, 100 + seed)
    for one_sided in (0, 1):
        orc = _oracle_np(V, S, D, L, lab, bounds)
        gp = fredopt.Plan(V, S, D, L, lab, bounds, block_rows=(2, 4)[seed % 2])
        for field, arr in vb.items():
            gp.set_voxel_bounds(field, arr); orc.set_voxel_bounds(field, arr)
        for g_, o_, v in ((fredopt.OPT_ONE_SIDED_COST, om.OPT_ONE_SIDED_COST, one_sided), (fredopt.OPT_REDUCTIONS, om.OPT_REDUCTIONS, 2)):
            gp.set_option(g_, v); orc.set_option(o_, v)
        orc.set_x(x0); gp.set_weights(x0)
        orc.iterate(20, 1.2, 2.0, 0.7); gp.iterate(20, 1.2, 2.0, 0.7)
        _assert_state(gp, orc)


def test_oar_bound_from_the_cdl30_of_the_forward_plan(fredopt):
    """The paper's constraint selection: the cDL value that 30 % of an OAR's volume receives in the forward
    (starting) plan becomes that OAR's upper cDL bound -- here per voxel, through fredopt_percentile_value and
    fredopt_set_voxel_bounds, end to end on the scaled three-beam plan, against the oracle doing the same."""
    from oracle import oracle as om
    plan = pg.build_plan(pg.config_spec(2, scale=0.25), device="cuda")
    gp = fredopt.from_plan(plan, stream=torch.cuda.current_stream().cuda_stream); orc = _oracle(plan)
    lab = plan.labels.cpu().numpy()
    hi_g = np.full(plan.n_rows, np.nan, np.float32); hi_o = hi_g.copy()
    for label in (2, 3):                                        # brainstem-like and chiasm-like OARs carry a cDL slab
        cg = gp.percentile_value(1, label, 0.3, plan.x0)
        co = orc.percentile_value(1, label, 0.3, plan.x0.astype(np.float64))
        assert abs(cg - co) <= 1e-12 * max(abs(co), 1e-30)
        hi_g[lab == label] = np.float32(cg); hi_o[lab == label] = np.float32(co)
    assert np.array_equal(hi_g, hi_o, equal_nan=True) and np.isfinite(hi_g[lab == 2]).all()
    gp.set_voxel_bounds(fredopt.VB_DL_HI, hi_g); orc.set_voxel_bounds(om.VB_DL_HI, hi_o)
    gp.set_voxel_bounds(fredopt.VB_DL_REF, hi_g); orc.set_voxel_bounds(om.VB_DL_REF, hi_o)
    gp.set_weights(plan.x0); orc.set_x(plan.x0)
    gp.iterate(20, 1.0, 1.0, 0.99); orc.iterate(20, 1.0, 1.0, 0.99)
    _assert_state(gp, orc)


def test_checkpoint_and_resume_in_a_new_plan(fredopt, plan0, tmp_path):
    """fredopt_get_state + fredopt_get_weights_f64 written to a file, read into a NEW plan (as another process would): the
    resumed run continues bit for bit as the uninterrupted one, in both AMS forms with eta < 1 and two reductions."""
    f = fredopt
    for block in (0, 1):
        def mk():
            g = f.from_plan(plan0)
            g.set_option(f.OPT_ETA, 0.97); g.set_option(f.OPT_REDUCTIONS, 2); g.set_option(f.OPT_BLOCK_SEQUENTIAL, block)
            return g
        a = mk(); a.set_weights(plan0.x0); a.iterate(4, 1.2, 0.0, 0.9); a.iterate(16, 1.2, 1.0, 0.9)
        b = mk(); b.set_weights(plan0.x0); b.iterate(4, 1.2, 0.0, 0.9); b.iterate(6, 1.2, 1.0, 0.9)
        path = tmp_path / f"ckpt{block}.bin"
        with open(path, "wb") as fh:
            fh.write(bytes(b.get_state())); fh.write(_gpu_x(b).tobytes())
        b.destroy()
        raw = open(path, "rb").read()
        n = C_sizeof_state = len(bytes(f.State()))
        c = mk()
        c.set_weights_f64(np.frombuffer(raw[n:], np.float64).copy())
        c.set_state(f.State.from_buffer_copy(raw[:n]))
        c.iterate(10, 1.2, 1.0, 0.9)
        assert np.array_equal(_gpu_x(c), _gpu_x(a))
        sa, sc = a.stats(), c.stats()
        assert all(sa[k] == sc[k] for k in ("k", "s", "trials", "last_beta", "n_violated", "prox"))
        assert bytes(a.get_state()) == bytes(c.get_state())
        with pytest.raises(f.FredoptError):                      # the latched pair came back with the state
            c.iterate(1, 1.2, 0.5, 0.9)
    bad = f.State(); bad.k = -1
    with pytest.raises(f.FredoptError):
        c.set_state(bad)


def test_iterate_host_is_the_four_calls_in_one(fredopt, plan0):
    """fredopt_iterate_host(x_in, x_out, stats) = set_weights, iterate, get_weights, get_stats made one after the other, bit for
    bit, over steps that pass x through the caller's fp32 array each time (bench.py's end-to-end loop); with NULL arrays it is
    fredopt_iterate on the plan's own x; and three such steps stay on the oracle's trajectory fed the same rounded x."""
    f = fredopt
    sp = plan0.spec
    a, b = f.from_plan(plan0), f.from_plan(plan0)
    xa, xb = plan0.x0.copy(), plan0.x0.copy()
    out_a, out_b = np.empty_like(xa), np.empty_like(xb)
    orc = _oracle(plan0)
    for step in range(3):
        a.set_weights(xa); a.iterate(2, sp.lam, sp.beta0, sp.a); a.get_weights(out_a); sa = a.stats()
        sb = b.iterate_host(2, sp.lam, sp.beta0, sp.a, xb, out_b)
        assert np.array_equal(out_a, out_b)
        assert sa == sb
        orc.set_x(xa.astype(np.float64)); orc.iterate(2, sp.lam, sp.beta0, sp.a)
        assert _rel_l2(out_b.astype(np.float64), orc.get_x()) <= 1e-6            # out is rounded to fp32
        xa, xb = out_a.copy(), out_b.copy()
    # device arrays, and no arrays at all
    import torch
    xd = torch.from_numpy(plan0.x0).cuda(); od = torch.empty_like(xd)
    c = f.from_plan(plan0)
    c.iterate_host(2, sp.lam, sp.beta0, sp.a, xd, od, stats=False)
    d = f.from_plan(plan0); d.set_weights(plan0.x0); d.iterate_host(2, sp.lam, sp.beta0, sp.a)
    assert np.array_equal(_gpu_x(c), _gpu_x(d))
    torch.cuda.synchronize()
    ref = np.empty_like(plan0.x0); d.get_weights(ref)
    assert np.array_equal(od.cpu().numpy(), ref)
    # a refused iteration returns the error of fredopt_iterate
    with pytest.raises(f.FredoptError):
        d.iterate_host(1, 3.0, sp.beta0, sp.a, plan0.x0, out_a)
    for g in (a, b, c, d):
        g.destroy()
