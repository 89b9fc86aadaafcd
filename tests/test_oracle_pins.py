"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

The paper prints no worked numbers for an iteration, so the oracle is pinned by
dense brute force, closed forms, invariants and reductions to textbook/library routines (SURVEY.md
sec. 8c pins 1-12).  Each test names the part of oracle/fredopt_oracle.cpp a plausible mistake in
which would make it fail.
"""
import os

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2509_20012_b200 import plangen as pg

NAN = np.nan
F32 = np.float32


# ----------------------------------------------------------------------------- helpers
def dense_to_csr(M):
    V, _ = M.shape
    rp = np.zeros(V + 1, np.int64)
    ci, vv = [], []
    for i in range(V):
        js = np.nonzero(M[i])[0]
        rp[i + 1] = rp[i] + len(js)
        ci.append(js.astype(np.int32))
        vv.append(M[i, js].astype(F32))
    return rp, np.concatenate(ci) if len(ci) else np.zeros(0, np.int32), \
        np.concatenate(vv) if len(vv) else np.zeros(0, F32)


def csr_to_dense(csr, S):
    rp, ci, vv = csr
    M = np.zeros((len(rp) - 1, S))
    for i in range(len(rp) - 1):
        M[i, ci[rp[i]:rp[i + 1]]] = vv[rp[i]:rp[i + 1]].astype(np.float64)
    return M


def bounds_rows(*rows):
    """rows: dicts with keys of plangen.Bounds."""
    return np.array([pg.Bounds(**r).as_row() for r in rows], dtype=F32)


class DenseReference:
    """Dense restatement of SURVEY.md sec. 8c, written separately from the oracle (numpy mat-vecs)."""

    def __init__(self, Dd, Ld, labels, bounds, vb=None):
        """vb: optional {field index 1..7 of a bounds row: per-voxel float32 array, NaN = the structure's scalar} (PAPER.md:161:
        bounds "defined for each point in the image space"); the structure's scalars decide which sets / cost terms exist."""
        self.D, self.L, self.lab = Dd, Ld, labels
        self.b = np.asarray(bounds, dtype=F32).astype(np.float64)
        self.vb = {k: np.asarray(v, dtype=F32).astype(np.float64) for k, v in (vb or {}).items()}

        def val(i, s, k):
            a = self.vb.get(k)
            return a[i] if a is not None and not np.isnan(a[i]) else self.b[s - 1, k]
        self.val = val
        sets = []   # (row vector a, lo, hi, structure)
        for i, s in enumerate(labels):
            if s == 0:
                continue
            w, dlo, dhi, llo, lhi, tmax, _, _ = self.b[s - 1]
            if not (np.isnan(dlo) and np.isnan(dhi)):
                sets.append((Dd[i], val(i, s, 1), val(i, s, 2), s))
            if not (np.isnan(llo) and np.isnan(lhi)):
                sets.append((Ld[i], val(i, s, 3), val(i, s, 4), s))
            if not np.isnan(tmax):
                sets.append((Ld[i] - val(i, s, 5) * Dd[i], NAN, 0.0, s))
        self.sets = sets
        self.W = sum(self.b[s - 1, 0] for a, lo, hi, s in sets if a @ a > 0)
        self.what = self.b[:, 0] / self.W if self.W > 0 else self.b[:, 0] * 0

    @staticmethod
    def resid(val, lo, hi):
        if not np.isnan(hi) and val > hi:
            return val - hi
        if not np.isnan(lo) and val < lo:
            return val - lo
        return 0.0

    def proximity(self, x):
        p, nv = 0.0, 0
        for a, lo, hi, s in self.sets:
            r = self.resid(a @ x, lo, hi)
            nv += r != 0
            if a @ a > 0:
                p += 0.5 * self.what[s - 1] * r * r / (a @ a)
        return p, nv

    def cost(self, x):
        phi = 0.0
        d, l = self.D @ x, self.L @ x
        for i, s in enumerate(self.lab):
            if s == 0:
                continue
            dref, lref = self.b[s - 1, 6], self.b[s - 1, 7]
            if not np.isnan(dref):
                phi += self.what[s - 1] * (self.val(i, s, 6) - d[i]) ** 2
            if not np.isnan(lref):
                phi += self.what[s - 1] * (self.val(i, s, 7) - l[i]) ** 2
        return phi

    def grad(self, x):
        g = np.zeros_like(x)
        d, l = self.D @ x, self.L @ x
        for i, s in enumerate(self.lab):
            if s == 0:
                continue
            dref, lref = self.b[s - 1, 6], self.b[s - 1, 7]
            if not np.isnan(dref):
                g += 2 * self.what[s - 1] * (d[i] - self.val(i, s, 6)) * self.D[i]
            if not np.isnan(lref):
                g += 2 * self.what[s - 1] * (l[i] - self.val(i, s, 7)) * self.L[i]
        return g

    def iterate(self, x, n, lam, beta0, a, max_trials=200, reductions=1, eta=1.0):
        """Fig. 3 around the simultaneous Fig. 2 step: `while t < reductionsN` holds the
        `while loop` over step sizes; w_k = eta^k w multiplies the projection step."""
        lam, beta0, a = float(F32(lam)), float(F32(beta0)), float(F32(a))
        beta = beta0
        s_count = 0
        eta_k = 1.0
        for _ in range(n):
            if beta0 != 0:
                t = 0
                while t < reductions:
                    phi0, g = self.cost(x), self.grad(x)
                    if not np.any(g != 0):
                        break
                    for _t in range(max_trials):
                        b = beta
                        beta *= a
                        s_count += 1
                        xn = x - b * g
                        if self.cost(xn) < phi0:
                            x = xn
                            break
                    t += 1
            step = np.zeros_like(x)
            for av, lo, hi, s in self.sets:
                n2 = av @ av
                if n2 > 0:
                    step += self.what[s - 1] * self.resid(av @ x, lo, hi) / n2 * av
            x = np.maximum(x - lam * eta_k * step, 0.0)
            eta_k *= eta
        return x, s_count


def make_oracle(Dd, Ld, labels, bounds):
    V, S = Dd.shape
    return orc.Oracle.create(V, S, dense_to_csr(Dd), dense_to_csr(Ld), np.asarray(labels, np.int32), bounds)


def f32mat(M):
    return M.astype(F32).astype(np.float64)


# ----------------------------------------------------------------------------- pin 1: dense brute force
@pytest.mark.parametrize("seed,same", [(1, True), (2, True), (3, False), (4, False)])
def test_pin1_dense_brute_force(seed, same):
    """Whole iteration, CSR traversal, scatter back-projection, union-pattern LETd rows."""
    D, L, labels, x0 = pg.random_small_plan(seed, V=45, S=9, n_struct=3, same_pattern=same)
    S = 9
    Dd, Ld = csr_to_dense(D, S), csr_to_dense(L, S)
    b = bounds_rows(dict(weight=1.0, dose_lo=1.2, dose_hi=1.6, dose_ref=1.4),
                    dict(weight=2.5, dose_hi=0.9, dl_hi=4.0, dl_lo=0.5, letd_max=5.0, dl_ref=3.0),
                    dict(weight=0.5, letd_max=4.0, dose_lo=0.3))
    o = orc.Oracle.create(45, S, D, L, labels, b)
    ref = DenseReference(Dd, Ld, labels, b)
    x0d = x0.astype(np.float64)
    o.set_x(x0)
    assert o.stats()["n_sets"] == len(ref.sets)
    assert np.isclose(o.stats()["W"], ref.W, rtol=1e-14)
    d, l, t = o.dose_let()
    np.testing.assert_allclose(d, Dd @ x0d, rtol=1e-13)
    np.testing.assert_allclose(l, Ld @ x0d, rtol=1e-13)
    p, nv = o.proximity()
    pr, nvr = ref.proximity(x0d)
    assert nv == nvr and np.isclose(p, pr, rtol=1e-12)
    assert np.isclose(o.cost(), ref.cost(x0d), rtol=1e-12)
    np.testing.assert_allclose(o.grad(), ref.grad(x0d), rtol=1e-11, atol=1e-15)
    for lam, beta0 in [(1.0, 0.0), (1.3, 1.0), (0.7, 0.5)]:
        o.set_option(orc.OPT_RESET, 1)
        o.set_x(x0)
        o.iterate(7, lam, beta0, 0.9)
        xr, s_ref = ref.iterate(x0d.copy(), 7, lam, beta0, 0.9)
        np.testing.assert_allclose(o.get_x(), xr, rtol=1e-10, atol=1e-13)
        assert o.stats()["s"] == s_ref
        assert o.proximity()[1] == ref.proximity(xr)[1]


# ----------------------------------------------------------------------------- pin 2: single half-space
@pytest.mark.parametrize("side", ["upper", "lower"])
def test_pin2_single_halfspace_closed_form(side):
    """Projection formula, sign of the lower branch (reading R2), norms: lambda=1 lands ON the boundary,
    is idempotent; general lambda: <a,x+> - b = (1 - lambda)(<a,x> - b)."""
    a = f32mat(np.array([[0.3, 1.1, 0.0, 0.7, 2.0]]))
    x0 = np.array([1.0, 2.0, 3.0, 0.5, 1.5], F32)
    val0 = float(a[0] @ x0.astype(np.float64))
    bnd = F32(val0 - 1.7) if side == "upper" else F32(val0 + 0.9)
    kw = dict(dose_hi=float(bnd)) if side == "upper" else dict(dose_lo=float(bnd))
    o = make_oracle(a, a * 3.0, [1], bounds_rows(dict(weight=3.0, **kw)))
    for lam in (1.0, 0.4, 1.7):
        o.set_x(x0)
        o.iterate(1, lam, 0.0, 0.5)
        x1 = o.get_x()
        assert np.all(x1 > 0)   # clamp inactive in this construction
        lhs = a[0] @ x1 - float(bnd)
        rhs = (1.0 - float(F32(lam))) * (val0 - float(bnd))
        assert abs(lhs - rhs) <= 1e-13 * max(1.0, abs(val0))
        if lam == 1.0:
            assert abs(lhs) < 1e-13
            # the move is along a (orthogonal projection)
            dx = x1 - x0.astype(np.float64)
            assert abs(abs(dx @ a[0]) - np.linalg.norm(dx) * np.linalg.norm(a[0])) < 1e-12
            o.iterate(1, lam, 0.0, 0.5)
            assert np.max(np.abs(o.get_x() - x1)) < 1e-14      # idempotent
            assert o.proximity()[0] < 1e-25


def test_pin2b_cdl_and_letd_halfspace():
    """Same closed form through the cDLET block and the linearised LETd row (a = L - LETmax D)."""
    Dd = f32mat(np.array([[0.5, 0.2, 0.9, 0.4]]))
    Ld = f32mat(np.array([[2.5, 2.2, 1.0, 3.1]]))
    x0 = np.array([1.0, 1.0, 1.0, 1.0], F32)
    # cDL upper
    o = make_oracle(Dd, Ld, [1], bounds_rows(dict(dl_hi=5.0)))
    o.set_x(x0); o.iterate(1, 1.0, 0.0, 0.5)
    assert abs(Ld[0] @ o.get_x() - 5.0) < 1e-13
    # LETd: <L - 3 D, x> <= 0
    o = make_oracle(Dd, Ld, [1], bounds_rows(dict(letd_max=3.0)))
    o.set_x(x0)
    a = Ld[0] - 3.0 * Dd[0]
    assert a @ x0 > 0
    o.iterate(1, 1.0, 0.0, 0.5)
    x1 = o.get_x()
    assert abs(a @ x1) < 1e-13
    d, l, t = o.dose_let()
    assert abs(t[0] - 3.0) < 1e-12          # LETd sits exactly at LETmax after the projection
    assert o.proximity() == (0.0, 0) or o.proximity()[0] < 1e-25


# ----------------------------------------------------------------------------- pin 3: diagonal system
def test_pin3_diagonal_geometric_decay():
    """w^ normalisation (R3) and multi-iteration bookkeeping: D = I, upper bounds, x0 above them:
    residual_i(k) = (1 - lambda/S)^k residual_i(0)."""
    S = 6
    I = np.eye(S)
    o = make_oracle(I, 2 * I, [1] * S, bounds_rows(dict(weight=7.0, dose_hi=1.0)))
    x0 = (2.0 + np.arange(S)).astype(F32)
    lam = 1.5
    o.set_x(x0)
    for k in range(1, 6):
        o.iterate(1, lam, 0.0, 0.5)
        np.testing.assert_allclose(o.get_x() - 1.0, (1 - float(F32(lam)) / S) ** k * (x0 - 1.0), rtol=1e-13)


# ----------------------------------------------------------------------------- pin 4: Cimmino averaging
def test_pin4_two_orthogonal_halfspaces_mean_of_projections():
    Dd = f32mat(np.array([[1.0, 0.0, 0.0], [0.0, 2.0, 0.0]]))
    o = make_oracle(Dd, Dd, [1, 1], bounds_rows(dict(dose_hi=1.0)))
    x0 = np.array([3.0, 4.0, 5.0], F32)
    o.set_x(x0); o.iterate(1, 1.0, 0.0, 0.5)
    p1 = np.array([1.0, 4.0, 5.0]); p2 = np.array([3.0, 0.5, 5.0])
    np.testing.assert_allclose(o.get_x(), 0.5 * (p1 + p2), rtol=1e-14)


def test_pin4b_copies_of_one_halfspace_equal_that_halfspace():
    a = f32mat(np.array([[0.3, 1.1, 0.7]]))
    x0 = np.array([2.0, 2.0, 2.0], F32)
    o1 = make_oracle(a, a, [1], bounds_rows(dict(dose_hi=1.0)))
    oM = make_oracle(np.repeat(a, 5, 0), np.repeat(a, 5, 0), [1] * 5, bounds_rows(dict(dose_hi=1.0)))
    for o in (o1, oM):
        o.set_x(x0); o.iterate(3, 0.8, 0.0, 0.5)
    np.testing.assert_allclose(oM.get_x(), o1.get_x(), rtol=1e-14)
    assert np.isclose(oM.proximity()[0], o1.proximity()[0], rtol=1e-13)


# ----------------------------------------------------------------------------- pin 5: monotone proximity
@pytest.mark.parametrize("lam", [0.5, 1.0, 1.5, 1.9])
def test_pin5_monotone_proximity_config0(plan0, lam):
    """Step direction/scale, clamp, proximity definition: beta0 = 0, lambda in (0,2) => p nonincreasing."""
    o = orc.from_plan(plan0)
    o.set_x(plan0.x0)
    prev = o.proximity()[0]
    for _ in range(25):
        o.iterate(1, lam, 0.0, 0.99)
        cur = o.proximity()[0]
        assert cur <= prev * (1 + 1e-12)
        prev = cur


# ----------------------------------------------------------------------------- pin 6: known feasible point / least squares
def test_pin6_known_feasible_point_converges():
    u = pg.uniform01_array(11, 30 * 6 + 6)
    A = f32mat((u[:180].reshape(30, 6) < 0.6) * (0.2 + u[:180].reshape(30, 6)))
    A[0, 0] = 0.5     # no empty row 0
    xs = 0.5 + u[180:186]
    Lm = f32mat(A * 3.0)
    d, l = A @ xs, Lm @ xs
    labels = np.arange(30) % 2 + 1
    # per-structure scalar bounds that xs satisfies
    b = bounds_rows(dict(dose_lo=float(F32(d[labels == 1].min() * 0.999)), dose_hi=float(F32(d[labels == 1].max() * 1.001))),
                    dict(dose_hi=float(F32(d[labels == 2].max() * 1.001)), dl_hi=float(F32(l[labels == 2].max() * 1.001)),
                         letd_max=3.001))
    o = make_oracle(A, Lm, labels, b)
    assert o.proximity(xs) == (0.0, 0)
    o.set_x((xs * 3 + 1).astype(F32))
    p0, n0 = o.proximity()
    assert n0 > 0
    o.iterate(4000, 1.9, 0.0, 0.5)
    p1, n1 = o.proximity()
    assert p1 < 1e-24 * p0 and n1 < n0    # on the feasible set to rounding (sets met on their boundary keep ulp-level residuals)


def test_pin6b_equalities_reduce_to_weighted_least_squares():
    """lo = hi = b with the clamp inactive: Landweber on min sum_k w^ (a_k x - b_k)^2 / n_k  ->  numpy lstsq."""
    u = pg.uniform01_array(5, 12 * 4 + 12)
    A = f32mat(0.2 + u[:48].reshape(12, 4))
    xs = np.array([1.0, 2.0, 1.5, 0.7])
    # one structure per row so each row has its own (equality) bound; noisy right-hand side
    rhs = (A @ xs + 0.05 * (u[48:60] - 0.5)).astype(F32)
    b = bounds_rows(*[dict(weight=1.0 + (i % 3), dose_lo=float(rhs[i]), dose_hi=float(rhs[i])) for i in range(12)])
    o = make_oracle(A, A, np.arange(12) + 1, b)
    o.set_x(np.ones(4, F32))
    o.iterate(60000, 1.9, 0.0, 0.5)
    w = np.array([1.0 + (i % 3) for i in range(12)])
    sc = np.sqrt(w / (A * A).sum(1))
    xl = np.linalg.lstsq(A * sc[:, None], rhs.astype(np.float64) * sc, rcond=None)[0]
    assert np.all(xl > 0)
    np.testing.assert_allclose(o.get_x(), xl, rtol=1e-8)


# ----------------------------------------------------------------------------- pin 7: cost / gradient / accept loop
def test_pin7_gradient_and_accept_loop(plan0):
    o = orc.from_plan(plan0)
    x = plan0.x0.astype(np.float64) * (1 + 0.3 * (pg.uniform01_array(3, plan0.n_cols) - 0.5))
    g = o.grad(x)
    # central differences of Eq. (2) on a few coordinates (phi is quadratic => exact up to rounding)
    for j in (0, 137, 455, 799):
        e = np.zeros_like(x); e[j] = 1e-3
        fd = (o.cost(x + e) - o.cost(x - e)) / 2e-3
        assert abs(fd - g[j]) <= 1e-8 * max(1.0, abs(g[j]))
    # phi(x - beta g) = phi - beta |g|^2 + beta^2 c  with  c = sum w^ (Dg)^2 (+ cDL terms)
    phi0, gg = o.cost(x), g @ g
    c = (o.cost(x - 1.0 * g) - phi0 + gg)
    for beta in (0.5, 0.1, 2.0):
        assert np.isclose(o.cost(x - beta * g), phi0 - beta * gg + beta * beta * c, rtol=1e-10)
    # every accepted perturbation strictly lowers phi; s grows by the number of trials; sum beta <= beta0/(1-a)
    o.set_x(x)
    s_prev, tot_beta = 0, 0.0
    for _ in range(10):
        xb = o.get_x(); phib = o.cost(xb)
        gb = o.grad(xb)
        o.set_option(orc.OPT_MAX_TRIALS, 200)
        o.iterate(1, 1.0, 1.0, 0.9)
        st = o.stats()
        assert st["s"] > s_prev
        # the accepted beta is beta0 * a^(s-1) by recursion
        beta = 1.0
        for _k in range(st["s"] - 1):
            beta *= float(F32(0.9))
        assert st["last_beta"] == beta
        assert o.cost(xb - beta * gb) < phib
        # the rejected ones did not lower phi
        b2 = 1.0
        for _k in range(s_prev):
            b2 *= float(F32(0.9))
        for _k in range(s_prev, st["s"] - 1):
            assert not (o.cost(xb - b2 * gb) < phib)
            b2 *= float(F32(0.9))
        tot_beta += beta
        s_prev = st["s"]
    assert tot_beta <= 1.0 / (1 - float(F32(0.9)))


# ----------------------------------------------------------------------------- pin 8: control flow / state
def test_pin8_state_and_control_flow(plan0):
    a = orc.from_plan(plan0); b = orc.from_plan(plan0); c = orc.from_plan(plan0)
    for o in (a, b, c):
        o.set_x(plan0.x0)
    a.iterate(20, 1.0, 1.0, 0.99)
    b.iterate(10, 1.0, 1.0, 0.99); b.iterate(10, 1.0, 1.0, 0.99)
    assert np.array_equal(a.get_x(), b.get_x()) and a.stats() == b.stats()
    # beta0 = 0 => SA == AMS bit for bit, whatever a is; s stays 0
    c.iterate(5, 1.0, 0.0, 0.5)
    d = orc.from_plan(plan0); d.set_x(plan0.x0); d.iterate(5, 1.0, 0.0, 0.99)
    assert np.array_equal(c.get_x(), d.get_x()) and c.stats()["s"] == 0
    # accept_check = 0 => unconditional beta0 a^k steps, s == k
    e = orc.from_plan(plan0); e.set_x(plan0.x0); e.set_option(orc.OPT_ACCEPT_CHECK, 0); e.iterate(7, 1.0, 0.3, 0.9)
    assert e.stats()["s"] == 7 and e.stats()["k"] == 7


# ----------------------------------------------------------------------------- pin 9: exact row scaling, permutations
def test_pin9_row_scaling_and_permutation_invariance():
    D, L, labels, x0 = pg.random_small_plan(21, V=36, S=7, n_struct=2)
    S = 7
    Dd, Ld = csr_to_dense(D, S), csr_to_dense(L, S)
    labels = np.where(labels == 0, 0, labels)
    b1 = bounds_rows(dict(dose_lo=1.0, dose_hi=1.5), dict(dose_hi=0.75))
    o1 = make_oracle(Dd, Ld, labels, b1)
    # scale every row of D by 2 (exact in binary) and the dose bounds by 2: iterates bit-identical
    b2 = bounds_rows(dict(dose_lo=2.0, dose_hi=3.0), dict(dose_hi=1.5))
    o2 = make_oracle(2 * Dd, Ld, labels, b2)
    for o in (o1, o2):
        o.set_x(x0); o.iterate(6, 1.2, 0.0, 0.5)
    assert np.array_equal(o1.get_x(), o2.get_x())
    # voxel permutation / spot permutation: same result up to summation order
    pv = np.argsort(pg.uniform01_array(8, 36)); ps = np.argsort(pg.uniform01_array(9, S))
    o3 = make_oracle(Dd[pv][:, ps], Ld[pv][:, ps], labels[pv], b1)
    o3.set_x(x0[ps]); o3.iterate(6, 1.2, 0.0, 0.5)
    np.testing.assert_allclose(o3.get_x(), o1.get_x()[ps], rtol=1e-12, atol=1e-15)


# ----------------------------------------------------------------------------- pin 10: transpose identity
def test_pin10_transpose_identity(plan0):
    o = orc.from_plan(plan0)
    x = pg.uniform01_array(5, plan0.n_cols)
    r = pg.uniform01_array(6, plan0.n_rows) - 0.5
    q = pg.uniform01_array(7, plan0.n_rows) - 0.5
    d, l, _ = o.dose_let(x)
    out, oabs = o.transpose(r, q)
    assert np.isclose(d @ r + l @ q, x @ out, rtol=1e-11)
    assert np.all(oabs >= np.abs(out) - 1e-12)
    lab = plan0.labels.numpy()
    outa, _ = o.transpose(r, None, active_only=True)
    assert np.isclose(d[lab != 0] @ r[lab != 0], x @ outa, rtol=1e-11)


# ----------------------------------------------------------------------------- pin 11: analytic LETd, generator
def test_pin11_analytic_letd_single_spot(plan0):
    """x = e_j => LETd_i = L_ij/D_ij = 2 + 10 exp(-max(R_j - z_i, 0)/5 mm) on every voxel the spot touches;
    uniform x0 => mean PTV dose = 2 Gy.  (Pins dose_let and the generator's depth convention.)"""
    o = orc.from_plan(plan0)
    nx, ny, nz = plan0.spec.grid
    h = plan0.spec.h
    for j in (0, 417, 799):
        x = np.zeros(plan0.n_cols); x[j] = 1.0
        d, l, t = o.dose_let(x)
        rows = np.nonzero(d > 0)[0]
        assert len(rows) > 500
        z = ((rows // (nx * ny)) + 0.5) * h               # beam along +z entering at z = 0
        R = plan0.spot_range[j]
        np.testing.assert_allclose(t[rows], 2 + 10 * np.exp(-np.maximum(R - z, 0) / 5.0), rtol=3e-7)   # fp32 storage
        assert np.all(t[d == 0] == 0)
    d, _, _ = o.dose_let(plan0.x0.astype(np.float64))
    lab = plan0.labels.numpy()
    assert abs(d[lab == 1].mean() - 2.0) < 1e-6


# ----------------------------------------------------------------------------- pin 12: sequential Fig. 2 sweep
def test_pin12_sequential_sweep_reaches_feasible_point_of_same_system():
    u = pg.uniform01_array(31, 24 * 5 + 5)
    A = f32mat(0.1 + u[:120].reshape(24, 5))
    xs = 0.5 + u[120:125]
    d = A @ xs
    labels = np.arange(24) % 2 + 1
    b = bounds_rows(dict(dose_lo=float(F32(d[labels == 1].min() * 0.99)), dose_hi=float(F32(d[labels == 1].max() * 1.01))),
                    dict(dose_hi=float(F32(d[labels == 2].max() * 1.01)), dl_hi=float(F32(2 * d[labels == 2].max() * 1.01))))
    o = make_oracle(A, 2 * A, labels, b)
    o.set_x((xs * 2).astype(F32))
    assert o.proximity()[1] > 0
    for _ in range(300):
        o.sequential_sweep(1.0)
    assert o.proximity()[1] == 0


# ----------------------------------------------------------------------------- external fixture (SURVEY probe)
def test_config0_matches_survey_probe_trajectory(plan0):
    path = os.path.join(os.path.dirname(__file__), "golden", "config0_trajectory.txt")
    gold = {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        gold[k] = float(v)
    o = orc.from_plan(plan0)
    st = o.stats()
    assert st["n_sets"] == gold["n_sets"] and st["n_sets"] - st["n_zero_norm_sets"] == gold["n_participating"]
    assert np.isclose(plan0.x0[0], gold["x0"], rtol=2e-7)
    o.set_x(plan0.x0)
    assert np.isclose(o.cost(), gold["phi0"], rtol=2e-6)
    assert np.isclose(np.linalg.norm(o.grad()), gold["gnorm0"], rtol=2e-6)
    p, nv = o.proximity()
    assert np.isclose(p, gold["prox0"], rtol=2e-6) and nv == gold["viol0"]
    for tag, beta0 in (("sa", 1.0), ("ams", 0.0)):
        o = orc.from_plan(plan0); o.set_x(plan0.x0)
        done = 0
        for n in (1, 10, 20, 50):
            o.iterate(n - done, 1.0, beta0, 0.99); done = n
            p, nv = o.proximity()
            assert np.isclose(p, gold[f"{tag}_prox_{n}"], rtol=2e-6), (tag, n, p)
            assert nv == gold[f"{tag}_viol_{n}"], (tag, n, nv)
        if tag == "sa":
            assert o.stats()["s"] == 50       # single beam: no rejections


# ----------------------------------------------------------------------------- block-sequential AMS (reading R23)
def _dense_block_sweep(Dd, Ld, labels, b, x, lam):
    """Dense restatement of the block-sequential sweep, written separately from the oracle: Fig. 2's loop nest (dose kind
    over the ROIs, then cDLET, then the LETd rows), one averaged simultaneous step per (kind, ROI) block, clamp at the end."""
    b = np.asarray(b, dtype=F32).astype(np.float64)
    x = x.copy()
    nviol = 0
    for kind in range(3):
        for s in range(1, b.shape[0] + 1):
            w, dlo, dhi, llo, lhi, tmax = b[s - 1, :6]
            rows = [i for i, lab in enumerate(labels) if lab == s]
            if kind == 0:
                if np.isnan(dlo) and np.isnan(dhi):
                    continue
                A, lo, hi = Dd[rows], dlo, dhi
            elif kind == 1:
                if np.isnan(llo) and np.isnan(lhi):
                    continue
                A, lo, hi = Ld[rows], llo, lhi
            else:
                if np.isnan(tmax):
                    continue
                A, lo, hi = Ld[rows] - tmax * Dd[rows], NAN, 0.0
            vals = A @ x
            r = np.array([DenseReference.resid(v, lo, hi) for v in vals])
            n2 = np.einsum("ij,ij->i", A, A)
            nviol += int(np.count_nonzero(r))
            part = n2 > 0
            if not part.any():
                continue
            step = (r[part] / n2[part]) @ A[part]
            x = x - lam * min(w, 1.0) / part.sum() * step
    return np.maximum(x, 0.0), nviol


@pytest.mark.parametrize("seed,same", [(11, True), (12, False), (13, True)])
def test_pin13_block_sequential_dense_brute_force(seed, same):
    """CSR traversal, block order (kind-major, then ROI), block averaging, priority factor, clamp, sweep statistics."""
    D, L, labels, x0 = pg.random_small_plan(seed, V=36, S=7, n_struct=3, same_pattern=same)
    bounds = bounds_rows(dict(weight=1.0, dose_lo=0.8, dose_hi=1.1, dose_ref=1.0),
                         dict(weight=0.5, dose_hi=0.6, dl_lo=0.5, dl_hi=2.5, letd_max=3.5, dl_ref=2.0),
                         dict(weight=2.0, dose_hi=0.7, letd_max=4.0))
    Dd, Ld = csr_to_dense(D, 7), csr_to_dense(L, 7)
    o = orc.Oracle.create(36, 7, D, L, labels, bounds)
    o.set_option(orc.OPT_BLOCK_SEQUENTIAL, 1)
    o.set_x(x0)
    x = x0.astype(np.float64)
    for k in range(6):
        o.iterate(1, 1.3, 0.0, 0.5)
        x, nv = _dense_block_sweep(Dd, Ld, labels, bounds, x, float(F32(1.3)))
        assert np.allclose(o.get_x(), x, rtol=1e-12, atol=1e-14)
        assert o.sweep_stats()[1] == nv


def test_pin14_single_block_equals_simultaneous_step():
    """One structure, one kind => the block sweep IS the simultaneous (Cimmino) step of R1/R3: w^ = 1/|P|."""
    D, L, labels, x0 = pg.random_small_plan(21, V=30, S=6, n_struct=1)
    labels = np.where(labels > 0, 1, 0).astype(np.int32)
    bounds = bounds_rows(dict(weight=1.0, dose_lo=0.9, dose_hi=1.0))
    a = orc.Oracle.create(30, 6, D, L, labels, bounds)
    b = orc.Oracle.create(30, 6, D, L, labels, bounds)
    b.set_option(orc.OPT_BLOCK_SEQUENTIAL, 1)
    a.set_x(x0); b.set_x(x0)
    a.iterate(8, 1.5, 0.0, 0.5); b.iterate(8, 1.5, 0.0, 0.5)
    assert np.allclose(a.get_x(), b.get_x(), rtol=1e-13, atol=1e-15)


def test_pin15_one_voxel_blocks_equal_the_sequential_listing():
    """Every structure holds one voxel => a block is one row and the sweep is Fig. 2 read literally (oracle_sequential_sweep)."""
    rng = np.random.default_rng(5)
    V, S = 6, 5
    Dd = f32mat(rng.uniform(0.1, 1.0, (V, S)))
    Ld = f32mat(Dd * rng.uniform(2.0, 6.0, (V, S)))
    labels = np.arange(1, V + 1, dtype=np.int32)
    bounds = bounds_rows(*[dict(weight=1.0, dose_lo=0.5, dose_hi=0.9, dl_hi=2.0, letd_max=3.0) for _ in range(V)])
    a, b = make_oracle(Dd, Ld, labels, bounds), make_oracle(Dd, Ld, labels, bounds)
    x0 = rng.uniform(0.2, 1.0, S).astype(F32)
    a.set_x(x0); b.set_x(x0)
    b.set_option(orc.OPT_BLOCK_SEQUENTIAL, 1)
    for _ in range(5):
        a.sequential_sweep(1.0)
        b.iterate(1, 1.0, 0.0, 0.5)
        assert np.allclose(a.get_x(), b.get_x(), rtol=1e-13, atol=1e-15)


def test_pin16_block_sequential_is_fejer_monotone_and_reaches_feasibility():
    """Sequential relaxed projections (lambda in (0,2)) never move away from a feasible point, and converge to the set."""
    rng = np.random.default_rng(9)
    V, S = 40, 8
    Dd = f32mat(rng.uniform(0.0, 1.0, (V, S)) * (rng.uniform(size=(V, S)) < 0.6))
    Ld = f32mat(Dd * rng.uniform(2.0, 8.0, (V, S)))
    xs = rng.uniform(0.2, 1.0, S)
    labels = (np.arange(V) % 3 + 1).astype(np.int32)
    d, l = Dd @ xs, Ld @ xs
    bounds = bounds_rows(dict(weight=1.0, dose_lo=float(d[labels == 1].min()) * 0.98, dose_hi=float(d[labels == 1].max()) * 1.02),
                         dict(weight=0.7, dose_hi=float(d[labels == 2].max()) * 1.02, dl_hi=float(l[labels == 2].max()) * 1.02),
                         dict(weight=1.0, dl_lo=float(l[labels == 3].min()) * 0.98, dl_hi=float(l[labels == 3].max()) * 1.02,
                              letd_max=float((l / np.maximum(d, 1e-9))[labels == 3].max()) * 1.05))
    o = make_oracle(Dd, Ld, labels, bounds)
    o.set_option(orc.OPT_BLOCK_SEQUENTIAL, 1)
    for lam in (0.6, 1.0, 1.8):
        o.set_option(orc.OPT_RESET, 1)
        o.set_x((xs * rng.uniform(0.3, 2.0, S)).astype(F32))
        dist = np.linalg.norm(o.get_x() - xs)
        p0 = o.proximity(None)[0]
        for _ in range(400):
            o.iterate(1, lam, 0.0, 0.5)
            dn = np.linalg.norm(o.get_x() - xs)
            assert dn <= dist * (1 + 1e-12)
            dist = dn
        p, _ = o.proximity(None)
        assert p0 > 1e-4 and p < 1e-6 * p0                  # asymptotic convergence to the feasible set


# ----------------------------------------------------------------------------- option variants of Fig. 3 / Eq. (2) (R9, R11)
def _small_cost_plan():
    D, L, labels, x0 = pg.random_small_plan(31, V=40, S=8, n_struct=2)
    bounds = bounds_rows(dict(weight=1.0, dose_lo=0.6, dose_hi=1.0, dose_ref=0.8),
                         dict(weight=1.5, dose_hi=0.7, dl_hi=2.0, dl_ref=1.2))
    return D, L, labels, x0, bounds


def test_pin17_one_sided_cost_and_its_gradient():
    """(cDL - cDLref)_+^2: only rows above the reference contribute; gradient vs central differences; cost <= two-sided cost."""
    D, L, labels, x0, _ = _small_cost_plan()
    Dd, Ld = csr_to_dense(D, 8), csr_to_dense(L, 8)
    lref = float(F32(np.median((Ld @ x0.astype(np.float64))[labels == 2])))     # some OAR rows above, some below
    bounds = bounds_rows(dict(weight=1.0, dose_lo=0.6, dose_hi=1.0, dose_ref=0.8),
                         dict(weight=1.5, dose_hi=0.7, dl_hi=2.0, dl_ref=lref))
    ref = DenseReference(Dd, Ld, labels, bounds)
    o = orc.Oracle.create(40, 8, D, L, labels, bounds)
    two = o.cost(x0.astype(np.float64))
    o.set_option(orc.OPT_ONE_SIDED_COST, 1)
    x = x0.astype(np.float64)
    # dense restatement
    d, l = Dd @ x, Ld @ x
    phi = sum(ref.what[0] * (float(F32(0.8)) - d[i]) ** 2 for i in range(40) if labels[i] == 1) + \
        sum(ref.what[1] * max(l[i] - lref, 0.0) ** 2 for i in range(40) if labels[i] == 2)
    assert abs(o.cost(x) - phi) <= 1e-13 * phi and o.cost(x) < two
    assert any(l[i] < lref for i in range(40) if labels[i] == 2) and any(l[i] > lref for i in range(40) if labels[i] == 2)
    g = o.grad(x)
    for j in range(8):
        e = np.zeros(8); e[j] = 1e-6
        fd = (o.cost(x + e) - o.cost(x - e)) / 2e-6
        assert abs(fd - g[j]) <= 1e-6 * max(1.0, abs(g[j]))


def test_pin18_normalised_gradient_step_has_length_beta():
    """R9 option: x' = x - beta g/|g|  =>  |x' - x|_2 = beta for the accepted beta (projection step switched off by a slack plan)."""
    D, L, labels, x0, _ = _small_cost_plan()
    bounds = bounds_rows(dict(weight=1.0, dose_hi=1e6, dose_ref=0.8), dict(weight=1.5, dose_hi=1e6, dl_ref=1.2))
    o = orc.Oracle.create(40, 8, D, L, labels, bounds)
    o.set_option(orc.OPT_NORMALIZE_GRAD, 1)
    o.set_x(x0)
    phi0 = o.cost(None)
    o.iterate(1, 1.0, 0.25, 0.5)                      # nothing is violated: the AMS step is the identity, x stays >= 0
    st = o.stats()
    step = np.linalg.norm(o.get_x() - x0.astype(np.float64))
    assert st["last_beta"] > 0 and abs(step - st["last_beta"]) <= 1e-14
    assert o.cost(None) < phi0 and st["trials"] == st["s"] >= 1


# ----------------------------------------------------------------------------- evaluation quantities
def test_pin19_volume_histogram_percentile_and_table1_statistics():
    """DVH / cDLVH / cDL30 and Table 1's columns on a hand example and against numpy."""
    # hand example: D = identity on 10 voxels of one structure => d_i = x_i = 1..10; "value received by 30% of the volume" = 8
    V = S = 10
    Dd = np.eye(V); Ld = 2.0 * np.eye(V)
    labels = np.ones(V, np.int32)
    bounds = bounds_rows(dict(weight=1.0, dose_hi=100.0))
    o = make_oracle(Dd, Ld, labels, bounds)
    x = np.arange(1.0, 11.0)
    assert o.percentile_value(0, 1, 0.3, x) == 8.0 and o.percentile_value(1, 1, 0.3, x) == 16.0
    assert o.percentile_value(0, 1, 1.0, x) == 1.0 and o.percentile_value(0, 1, 0.05, x) == 10.0
    assert o.structure_stats(0, 1, x) == (1.0, 5.5, 10.0, 10)
    assert o.structure_stats(2, 1, x)[:3] == (2.0, 2.0, 2.0)                       # LETd = l/d = 2 everywhere
    assert np.array_equal(o.volume_histogram(0, 1, 5, 10.0, x), [1.0, 0.9, 0.7, 0.5, 0.3])   # edges 0, 2, 4, 6, 8
    # against numpy on a random plan
    D, L, lab, x0 = pg.random_small_plan(41, V=60, S=9, n_struct=2)
    Dd, Ld = csr_to_dense(D, 9), csr_to_dense(L, 9)
    o = orc.Oracle.create(60, 9, D, L, lab, bounds_rows(dict(weight=1.0, dose_hi=1.0), dict(weight=1.0, dl_hi=1.0)))
    xx = x0.astype(np.float64)
    for s_ in (1, 2):
        d, l = (Dd @ xx)[lab == s_], (Ld @ xx)[lab == s_]
        for q, v in ((0, d), (1, l), (2, np.where(d > 0, l / np.where(d > 0, d, 1.0), 0.0))):
            mn, mean, mx, n = o.structure_stats(q, s_, xx)
            assert n == len(v) and np.allclose([mn, mean, mx], [v.min(), v.mean(), v.max()], rtol=1e-13)
            pv = o.percentile_value(q, s_, 0.3, xx)
            assert np.mean(v >= pv * (1 - 1e-13)) >= 0.3 and np.mean(v > pv * (1 + 1e-13)) < 0.3
            hst = o.volume_histogram(q, s_, 16, float(v.max()) * 1.01, xx)
            assert hst[0] == 1.0 and np.all(np.diff(hst) <= 0) and hst[-1] > 0


# ----------------------------------------------------------------------------- options of Fig. 3: eta, reductionsN, trial cap
@pytest.mark.parametrize("eta", [0.9, 0.5])
def test_pin20_eta_decay_diagonal_closed_form(eta):
    """w_k = eta^k w (Fig. 3; reading R12): on pin 3's diagonal system the residual after k iterations is
    prod_{j<k} (1 - lambda eta^j / S) * residual(0).  Guards `relax = lambda * eta_pow` and `eta_pow *= eta` in
    oracle_iterate (a decay applied cumulatively, one iteration late, or to the wrong factor fails)."""
    S = 6
    I = np.eye(S)
    o = make_oracle(I, 2 * I, [1] * S, bounds_rows(dict(weight=7.0, dose_hi=1.0)))
    o.set_option(orc.OPT_ETA, eta)
    x0 = (2.0 + np.arange(S)).astype(F32)
    r0 = x0.astype(np.float64) - 1.0
    lam = float(F32(1.5))
    o.set_x(x0)
    fac = 1.0
    for k in range(1, 9):
        o.iterate(1, 1.5, 0.0, 0.5)
        fac *= 1.0 - lam * eta ** (k - 1) / S
        np.testing.assert_allclose(o.get_x() - 1.0, fac * r0, rtol=1e-13)
    # RESET restarts the decay at eta^0
    o.set_option(orc.OPT_RESET, 1); o.set_x(x0); o.iterate(1, 1.5, 0.0, 0.5)
    np.testing.assert_allclose(o.get_x() - 1.0, (1.0 - lam / S) * r0, rtol=1e-13)


@pytest.mark.parametrize("reductions", [2, 3])
@pytest.mark.parametrize("seed,same", [(1, True), (3, False)])
def test_pin21_reductions_loop_dense_brute_force(reductions, seed, same):
    """`while t < reductionsN` (Fig. 3): N cost-reducing steps, each with a fresh chi^2 and gradient, before
    one AMS step.  Guards the `for t < reductionsN` loop of oracle_iterate (phi0 / g not refreshed, or the AMS step inside the
    loop, fails); x, s and the violation count are compared with the separate dense restatement, with eta < 1 on top."""
    D, L, labels, x0 = pg.random_small_plan(seed, V=45, S=9, n_struct=3, same_pattern=same)
    Dd, Ld = csr_to_dense(D, 9), csr_to_dense(L, 9)
    b = bounds_rows(dict(weight=1.0, dose_lo=1.2, dose_hi=1.6, dose_ref=1.4),
                    dict(weight=2.5, dose_hi=0.9, dl_hi=4.0, dl_lo=0.5, letd_max=5.0, dl_ref=3.0),
                    dict(weight=0.5, letd_max=4.0, dose_lo=0.3))
    o = orc.Oracle.create(45, 9, D, L, labels, b)
    ref = DenseReference(Dd, Ld, labels, b)
    o.set_option(orc.OPT_REDUCTIONS, reductions); o.set_option(orc.OPT_ETA, 0.95)
    o.set_x(x0)
    o.iterate(7, 1.3, 2.0, 0.8)                      # beta0 = 2: the first trials are rejected
    xr, s_ref = ref.iterate(x0.astype(np.float64), 7, 1.3, 2.0, 0.8, reductions=reductions, eta=0.95)
    np.testing.assert_allclose(o.get_x(), xr, rtol=1e-10, atol=1e-13)
    st = o.stats()
    assert st["s"] == s_ref and st["trials"] == s_ref and s_ref > 7 * reductions
    assert o.proximity()[1] == ref.proximity(xr)[1]
    # one reduction per iteration gives a different trajectory (the loop is not a no-op)
    o1 = orc.Oracle.create(45, 9, D, L, labels, b)
    o1.set_option(orc.OPT_ETA, 0.95); o1.set_x(x0); o1.iterate(7, 1.3, 2.0, 0.8)
    assert np.max(np.abs(o1.get_x() - o.get_x())) > 1e-6


def test_pin22_trial_cap_keeps_x_and_still_advances_s():
    """Reading R10 (Fig. 3's `while loop`, never ends if chi^2 cannot decrease): after `max_trials`
    rejections x is kept and s has still advanced.  beta0 = 1e6 with a = 0.999 rejects every trial, so with a cap of 5 the
    trajectory is that of pure feasibility-seeking bit for bit and s grows by exactly 5 per iteration.  Guards the
    `trial < max_trials` bound and the keep-x fall-through of oracle_iterate."""
    D, L, labels, x0 = pg.random_small_plan(2, V=45, S=9, n_struct=2)
    b = bounds_rows(dict(weight=1.0, dose_lo=1.2, dose_hi=1.6, dose_ref=1.4), dict(weight=2.0, dose_hi=0.9, dl_ref=3.0))
    a = orc.Oracle.create(45, 9, D, L, labels, b)
    c = orc.Oracle.create(45, 9, D, L, labels, b)
    a.set_option(orc.OPT_MAX_TRIALS, 5)
    a.set_x(x0); c.set_x(x0)
    for k in range(1, 5):
        a.iterate(1, 1.1, 1.0e6, 0.999); c.iterate(1, 1.1, 0.0, 0.999)
        assert np.array_equal(a.get_x(), c.get_x())
        st = a.stats()
        assert st["s"] == 5 * k and st["trials"] == 5 * k and st["last_beta"] == 0.0 and st["k"] == k
    # beta_next = beta0 a^(5k) by repeated multiplication
    bn = float(F32(1.0e6))
    for _ in range(20):
        bn *= float(F32(0.999))
    assert a.stats()["beta_next"] == bn


def test_pin23_letd_row_over_entries_in_D_only_and_L_only():
    """The LETd row a = L_i - LETmax D_i over the UNION pattern (north_star; reading R18): independent D / L masks give entries
    in D only (a_j = -LETmax D_ij), in L only (a_j = L_ij) and in both.  Guards all three branches of letd_row_dot (the
    `cd < cl` branch had no test before: a dropped -LETmax D_ij term changes the norm, the residual and the step)."""
    D, L, labels, x0 = pg.random_small_plan(6, V=40, S=10, n_struct=2, density=0.45, same_pattern=False)
    Dd, Ld = csr_to_dense(D, 10), csr_to_dense(L, 10)
    only_d = (Dd != 0) & (Ld == 0) & (labels[:, None] != 0)
    only_l = (Dd == 0) & (Ld != 0) & (labels[:, None] != 0)
    assert only_d.sum() > 20 and only_l.sum() > 20 and ((Dd != 0) & (Ld != 0)).sum() > 20
    b = bounds_rows(dict(weight=1.0, letd_max=1.5), dict(weight=3.0, letd_max=0.7, dose_hi=1.0))
    o = orc.Oracle.create(40, 10, D, L, labels, b)
    ref = DenseReference(Dd, Ld, labels, b)
    # norms of the LETd rows over the union pattern
    _, _, nT = o.norms()
    for i in range(40):
        if labels[i]:
            a = Ld[i] - float(b[labels[i] - 1, 5]) * Dd[i]
            assert abs(nT[i] - a @ a) <= 1e-14 * max(a @ a, 1e-300)
    x = x0.astype(np.float64)
    p, nv = o.proximity(x)
    pr, nvr = ref.proximity(x)
    assert nv == nvr and nv > 5 and abs(p - pr) <= 1e-13 * pr
    o.set_x(x0)
    o.iterate(9, 1.4, 0.0, 0.5)
    xr, _ = ref.iterate(x.copy(), 9, 1.4, 0.0, 0.5)
    np.testing.assert_allclose(o.get_x(), xr, rtol=1e-11, atol=1e-14)
    # block-sequential form over the same rows
    ob = orc.Oracle.create(40, 10, D, L, labels, b)
    ob.set_option(orc.OPT_BLOCK_SEQUENTIAL, 1); ob.set_x(x0)
    xb = x.copy()
    for _ in range(4):
        ob.iterate(1, 1.2, 0.0, 0.5)
        xb, _ = _dense_block_sweep(Dd, Ld, labels, b, xb, float(F32(1.2)))
    np.testing.assert_allclose(ob.get_x(), xb, rtol=1e-11, atol=1e-14)


def test_pin24_dose_let_rows_equals_dose_let(plan0):
    """oracle_dose_let_rows (the checker of the full-size sampled forward parity) returns exactly the listed rows of
    oracle_dose_let (Eq. 1) -- bit for bit, repeated and unordered rows included."""
    o = orc.from_plan(plan0)
    x = pg.log_uniform_weights(5, plan0.n_cols).astype(np.float64)
    d, l, t = o.dose_let(x)
    rows = (pg.uniform01_array(8, 3000) * plan0.n_rows).astype(np.int64)
    rows[:3] = [0, plan0.n_rows - 1, rows[5]]
    dr, lr, tr = o.dose_let_rows(rows, x)
    assert np.array_equal(dr, d[rows]) and np.array_equal(lr, l[rows]) and np.array_equal(tr, t[rows])
    assert np.count_nonzero(dr) > 100
    # and at the oracle's own x (x = NULL)
    o.set_x(plan0.x0)
    d0, l0, t0 = o.dose_let(None)
    dr0, _, tr0 = o.dose_let_rows(rows, None)
    assert np.array_equal(dr0, d0[rows]) and np.array_equal(tr0, t0[rows])


def test_pin25_transpose_abs_scale_is_the_dense_abs_product():
    """oracle_transpose's second output (the scale of the per-element tolerance of the transposed GPU passes, SURVEY sec. 8c
    parity rule) is sum_i |D_ij u_i| + |L_ij v_i| -- no more (a too-large scale would loosen the tolerance), no less."""
    D, L, labels, _ = pg.random_small_plan(9, V=50, S=11, n_struct=2, density=0.35, same_pattern=False)
    Dd, Ld = csr_to_dense(D, 11), csr_to_dense(L, 11)
    o = orc.Oracle.create(50, 11, D, L, labels, bounds_rows(dict(dose_hi=1.0), dict(dl_hi=1.0)))
    u = pg.uniform01_array(12, 50) - 0.5
    v = pg.uniform01_array(13, 50) - 0.4
    for uu, vv in ((u, v), (u, None), (None, v)):
        for act in (False, True):
            m = (labels != 0) if act else np.ones(50, bool)
            out, oabs = o.transpose(uu, vv, active_only=act)
            ref = np.zeros(11); refa = np.zeros(11)
            if uu is not None:
                ref += Dd[m].T @ uu[m]; refa += np.abs(Dd[m]).T @ np.abs(uu[m])
            if vv is not None:
                ref += Ld[m].T @ vv[m]; refa += np.abs(Ld[m]).T @ np.abs(vv[m])
            np.testing.assert_allclose(out, ref, rtol=1e-13, atol=1e-16)
            np.testing.assert_allclose(oabs, refa, rtol=1e-13)


def test_pin26_step_size_sequence_belongs_to_the_plan():
    """Reading R8: beta_s = beta0 a^s is ONE sequence per plan.  beta0, a are latched by the first superiorized call; calls
    with beta0 = 0 in between are pure AMS steps that neither latch nor consume it; another (beta0, a) needs a RESET."""
    D, L, labels, x0 = pg.random_small_plan(2, V=45, S=9, n_struct=2)
    b = bounds_rows(dict(weight=1.0, dose_lo=1.2, dose_hi=1.6, dose_ref=1.4), dict(weight=2.0, dose_hi=0.9, dl_ref=3.0))
    o = orc.Oracle.create(45, 9, D, L, labels, b)
    o.set_x(x0)
    o.iterate(0, 1.0, 0.7, 0.5)                     # n_iter = 0 latches nothing
    o.iterate(2, 1.0, 0.0, 0.5)                     # pure AMS first: nothing latched, s stays 0
    assert o.stats()["s"] == 0 and o.stats()["k"] == 2
    o.iterate(1, 1.0, 0.5, 0.9)                     # first superiorized call latches (0.5, 0.9)
    s1 = o.stats()["s"]
    bn = float(F32(0.5))
    for _ in range(s1):
        bn *= float(F32(0.9))
    assert s1 >= 1 and o.stats()["beta_next"] == bn
    o.iterate(1, 1.0, 0.0, 0.9)                     # AMS step in between: s unchanged
    assert o.stats()["s"] == s1
    with pytest.raises(ValueError):
        o.iterate(1, 1.0, 0.25, 0.9)
    with pytest.raises(ValueError):
        o.iterate(1, 1.0, 0.5, 0.8)
    o.iterate(1, 1.0, 0.5, 0.9)
    assert o.stats()["s"] > s1 and o.stats()["k"] == 5


# ----------------------------------------------------------------------------- per-voxel bounds and references
def _voxel_bound_plan():
    D, L, labels, x0 = pg.random_small_plan(7, V=48, S=9, n_struct=3, same_pattern=False)
    b = bounds_rows(dict(weight=1.0, dose_lo=1.2, dose_hi=1.6, dose_ref=1.4),
                    dict(weight=2.5, dose_hi=0.9, dl_hi=4.0, dl_lo=0.5, letd_max=5.0, dl_ref=3.0),
                    dict(weight=0.5, letd_max=4.0, dose_lo=0.3))
    return D, L, labels, x0, b


def test_pin27_per_voxel_arrays_of_the_structure_scalars_change_nothing():
    """Per-voxel arrays filled with the structures' own scalars (or with NaN = "use the scalar") reproduce the trajectory of the
    scalar plan BIT FOR BIT: the per-voxel path evaluates the same formulas (Eq. (2))."""
    D, L, labels, x0, b = _voxel_bound_plan()
    base = orc.Oracle.create(48, 9, D, L, labels, b)
    full = orc.Oracle.create(48, 9, D, L, labels, b)
    nan_ = orc.Oracle.create(48, 9, D, L, labels, b)
    for field in range(7):
        col = np.where(labels > 0, b[np.maximum(labels, 1) - 1, field + 1], NAN).astype(F32)
        full.set_voxel_bounds(field, col)
        nan_.set_voxel_bounds(field, np.full(48, NAN, F32))
    for o in (base, full, nan_):
        o.set_x(x0); o.iterate(9, 1.3, 0.7, 0.9)
    assert np.array_equal(base.get_x(), full.get_x()) and np.array_equal(base.get_x(), nan_.get_x())
    assert base.stats() == full.stats() == nan_.stats()
    assert base.proximity() == full.proximity() and base.cost() == full.cost()
    # removing an array restores the scalar
    full.set_voxel_bounds(orc.VB_DOSE_HI, np.full(48, 5.0, F32))
    assert full.proximity() != base.proximity()
    full.set_voxel_bounds(orc.VB_DOSE_HI, None)
    assert full.proximity() == base.proximity()


@pytest.mark.parametrize("block", [0, 1])
def test_pin28_per_voxel_bounds_dense_brute_force(block):
    """Bounds and references that genuinely vary from voxel to voxel against the separate dense restatement: dose / cDL slabs,
    the LETd limit (its row L_i - LETmax_i D_i and norm change with the voxel's LETmax_i) and both cost references.  Guards
    voxel_bounds() and every place the oracle reads a bound (a place still reading the structure scalar fails)."""
    D, L, labels, x0, b = _voxel_bound_plan()
    Dd, Ld = csr_to_dense(D, 9), csr_to_dense(L, 9)
    u = pg.uniform01_array(77, 7 * 48).reshape(7, 48)
    vb = {}
    for field in range(7):
        k = field + 1
        col = b[np.maximum(labels, 1) - 1, k].astype(np.float64)
        scale = 0.8 + 0.4 * u[field]                                   # +-20 % around the structure's value ...
        if field in (0, 2):
            scale = 0.7 + 0.25 * u[field]                              # (lower bounds stay below upper bounds)
        if field in (1, 3):
            scale = 1.0 + 0.3 * u[field]
        arr = np.where(u[(field + 3) % 7] < 0.3, NAN, col * scale)     # ... and NaN (= scalar) on ~30 % of the voxels
        vb[k] = arr.astype(F32)
    o = orc.Oracle.create(48, 9, D, L, labels, b)
    for k, arr in vb.items():
        o.set_voxel_bounds(k - 1, arr)
    ref = DenseReference(Dd, Ld, labels, b, vb=vb)
    x = x0.astype(np.float64)
    assert abs(o.stats()["W"] - ref.W) <= 1e-13 * ref.W
    p, nv = o.proximity(x); pr, nvr = ref.proximity(x)
    assert nv == nvr and nv > 5 and abs(p - pr) <= 1e-12 * pr
    assert abs(o.cost(x) - ref.cost(x)) <= 1e-12 * ref.cost(x)
    np.testing.assert_allclose(o.grad(x), ref.grad(x), rtol=1e-11, atol=1e-15)
    # the scalar plan differs (the arrays are not a no-op)
    o0 = orc.Oracle.create(48, 9, D, L, labels, b)
    assert abs(o0.proximity(x)[0] - p) > 1e-3 * p
    if not block:
        o.set_x(x0); o.iterate(7, 1.3, 1.0, 0.9)
        xr, s_ref = ref.iterate(x.copy(), 7, 1.3, 1.0, 0.9)
        np.testing.assert_allclose(o.get_x(), xr, rtol=1e-10, atol=1e-13)
        assert o.stats()["s"] == s_ref and o.proximity()[1] == ref.proximity(xr)[1]
    else:
        # block-sequential sweep against a dense restatement with per-voxel bounds
        o.set_option(orc.OPT_BLOCK_SEQUENTIAL, 1); o.set_x(x0)
        xb = x.copy()
        for _ in range(4):
            o.iterate(1, 1.2, 0.0, 0.5)
            for kind in range(3):
                for s_ in range(1, 4):
                    rows = [i for i in range(48) if labels[i] == s_]
                    if kind == 0 and np.isnan(b[s_ - 1, 1]) and np.isnan(b[s_ - 1, 2]) or kind == 1 and np.isnan(b[s_ - 1, 3]) and np.isnan(b[s_ - 1, 4]) \
                            or kind == 2 and np.isnan(b[s_ - 1, 5]):
                        continue
                    step = np.zeros(9); m = 0
                    for i in rows:
                        if kind == 0:
                            a, lo, hi = Dd[i], ref.val(i, s_, 1), ref.val(i, s_, 2)
                        elif kind == 1:
                            a, lo, hi = Ld[i], ref.val(i, s_, 3), ref.val(i, s_, 4)
                        else:
                            a, lo, hi = Ld[i] - ref.val(i, s_, 5) * Dd[i], NAN, 0.0
                        n2 = a @ a
                        if n2 > 0:
                            m += 1
                            step += DenseReference.resid(a @ xb, lo, hi) / n2 * a
                    if m:
                        xb = xb - float(F32(1.2)) * min(float(b[s_ - 1, 0]), 1.0) / m * step
            xb = np.maximum(xb, 0.0)
        np.testing.assert_allclose(o.get_x(), xb, rtol=1e-11, atol=1e-14)


def test_pin29_per_voxel_letd_limit_lands_on_the_voxels_own_boundary():
    """Single LETd half-space with a per-voxel limit: lambda = 1 lands on <L_i - t_i D_i, x> = 0 for the VOXEL'S t_i (closed
    form), i.e. LETd_i = t_i afterwards; with the structure scalar it would land elsewhere."""
    Dd = f32mat(np.array([[0.5, 0.2, 0.9, 0.4]]))
    Ld = f32mat(np.array([[2.5, 2.2, 1.0, 3.1]]))
    x0 = np.array([1.0, 1.0, 1.0, 1.0], F32)
    o = make_oracle(Dd, Ld, [1], bounds_rows(dict(letd_max=3.0)))
    o.set_voxel_bounds(orc.VB_LETD_MAX, np.array([2.5], F32))
    o.set_x(x0); o.iterate(1, 1.0, 0.0, 0.5)
    d, l, t = o.dose_let()
    assert abs(t[0] - 2.5) < 1e-12
    _, _, nT = o.norms()
    a = Ld[0] - 2.5 * Dd[0]
    assert abs(nT[0] - a @ a) <= 1e-15 * (a @ a)
    # invalid: lo > hi on a voxel, infinite value -> refused, state unchanged
    o2 = make_oracle(Dd, Ld, [1], bounds_rows(dict(dose_lo=1.0, dose_hi=2.0)))
    with pytest.raises(ValueError):
        o2.set_voxel_bounds(orc.VB_DOSE_LO, np.array([2.5], F32))
    with pytest.raises(ValueError):
        o2.set_voxel_bounds(orc.VB_DOSE_HI, np.array([np.inf], F32))
    o2.set_x(x0)
    assert o2.proximity()[1] == 0 or o2.proximity()[1] == 1


# ----------------------------------------------------------------------------- the OpenMP timing build
def test_openmp_timing_build_is_the_same_oracle(plan0):
    """bench.py's all-cores cpu_baseline runs oracle/fredopt_oracle.cpp compiled with -fopenmp.  With one thread it returns the
    plain build's bits; with several, static row chunks and per-thread S-vectors added in thread order change the summation
    order only (1e-13), never a decision (s, trials, violation count)."""
    plain = orc.from_plan(plan0)
    plain.set_x(plan0.x0); plain.iterate(12, 1.0, 1.0, 0.99)
    for nt, tol in ((1, 0.0), (4, 1e-13)):
        assert orc.omp_threads(nt) == nt
        o = orc.from_plan(plan0, omp=True)
        o.set_x(plan0.x0); o.iterate(12, 1.0, 1.0, 0.99)
        err = np.linalg.norm(o.get_x() - plain.get_x()) / np.linalg.norm(plain.get_x())
        assert err <= tol, (nt, err)
        assert o.stats()["s"] == plain.stats()["s"] and o.proximity()[1] == plain.proximity()[1]
        assert abs(o.proximity()[0] - plain.proximity()[0]) <= max(tol, 0.0) * plain.proximity()[0]
        assert abs(o.cost() - plain.cost()) <= max(tol, 0.0) * plain.cost()


def test_state_snapshot_continues_bit_for_bit(plan0):
    """get_state / set_state (+ x) carry everything Fig. 3 keeps between calls: a second oracle resumed from the snapshot
    continues exactly as the first (bench.py times the one-thread oracle from the all-cores oracle's warm state this way)."""
    a = orc.from_plan(plan0); a.set_option(orc.OPT_ETA, 0.97)
    a.set_x(plan0.x0); a.iterate(6, 1.0, 1.0, 0.9)
    b = orc.from_plan(plan0); b.set_option(orc.OPT_ETA, 0.97)
    b.set_x(a.get_x()); b.set_state(a.get_state())
    a.iterate(6, 1.0, 1.0, 0.9); b.iterate(6, 1.0, 1.0, 0.9)
    assert np.array_equal(a.get_x(), b.get_x()) and a.stats() == b.stats()
