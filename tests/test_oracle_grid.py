"""Pins of the CPU oracle's grid-side functions: areas (Eq.8), deposit (Eq.21-23), field
update (Eq.9-11, B8-B11), sort/compaction -- against closed forms, library routines,
brute force and the invariants the paper states."""
import math

import numpy as np
import pytest
import scipy.integrate

import oracle
import inputs


def small_params(nr=24, nth=20, a=0.9, **kw):
    return inputs.grid_params(nr, nth, a, r_out=20.0, **kw)


# ------------------------------------------------------------------ quadrature, areas
def test_gauss_legendre_nodes():
    x, w = oracle.gauss_legendre(10)
    xr, wr = np.polynomial.legendre.leggauss(10)
    o = np.argsort(x)
    assert np.allclose(x[o], xr, atol=1e-15) and np.allclose(w[o], wr, atol=1e-15)


def test_areas_against_scipy_quad_and_closed_form():
    p = small_params(12, 10, 0.95)
    g = oracle.Grid(p)
    A = oracle.areas(p)
    a, dxi, dth, dphi = p["a"], g.dxi, g.dth, p["dphi"]
    sg = lambda r, th: float(inputs.kerr_schild(a, 1.0, r, th)["sqrtg"])
    r_ = lambda i: math.exp(p["xi_in"] + i * dxi)
    for (i, j) in [(0, 0), (3, 4), (11, 10), (5, 9), (-1, 3)]:
        tlo, thi = max((j - .5) * dth, 0), min((j + .5) * dth, math.pi)
        ref = dphi * scipy.integrate.quad(lambda t: sg(r_(i + .5), t), tlo, thi, epsabs=0, epsrel=1e-13)[0]
        assert np.isclose(A["ADr"][g.ij(i, j)], ref, rtol=1e-12)
        ref = dphi * scipy.integrate.quad(lambda r: sg(r, j * dth), r_(i), r_(i + 1), epsabs=0, epsrel=1e-13)[0]
        assert np.isclose(A["ABth"][g.ij(i, j)], ref, rtol=1e-12, atol=1e-16)
        ref = scipy.integrate.dblquad(lambda t, r: sg(r, t), r_(i - .5), r_(i + .5), tlo, thi,
                                      epsabs=0, epsrel=1e-12)[0]
        assert np.isclose(A["ADph"][g.ij(i, j)], ref, rtol=1e-11)
        if j < p["nth"]:
            ref = dphi * scipy.integrate.quad(lambda r: sg(r, (j + .5) * dth), r_(i - .5), r_(i + .5), epsabs=0, epsrel=1e-13)[0]
            assert np.isclose(A["ADth"][g.ij(i, j)], ref, rtol=1e-12)
            ref = dphi * scipy.integrate.quad(lambda t: sg(r_(i), t), j * dth, (j + 1) * dth, epsabs=0, epsrel=1e-13)[0]
            assert np.isclose(A["ABr"][g.ij(i, j)], ref, rtol=1e-12)
            ref = scipy.integrate.dblquad(lambda t, r: sg(r, t), r_(i), r_(i + 1), j * dth, (j + 1) * dth,
                                          epsabs=0, epsrel=1e-12)[0]
            assert np.isclose(A["ABph"][g.ij(i, j)], ref, rtol=1e-11)
    # a = 0 closed form: A^B_r = dphi r^2 sqrt(1+2/r) (cos th_j - cos th_{j+1})
    p0 = small_params(12, 10, 0.0)
    g0, A0 = oracle.Grid(p0), oracle.areas(p0)
    i, j = 4, 3
    r = math.exp(p0["xi_in"] + i * g0.dxi)
    ref = p0["dphi"] * r * r * math.sqrt(1 + 2 / r) * (math.cos(j * g0.dth) - math.cos((j + 1) * g0.dth))
    assert np.isclose(A0["ABr"][g0.ij(i, j)], ref, rtol=1e-13)
    # total volume of the a=0 shell = dphi * int r^2 sqrt(1+2/r) dr * 2
    tot = sum(A0["ABph"][g0.ij(i, j)] for i in range(p0["nr"]) for j in range(p0["nth"]))
    ref = 2 * scipy.integrate.quad(lambda r: r * r * math.sqrt(1 + 2 / r), math.exp(p0["xi_in"]), 20.0, epsabs=0, epsrel=1e-13)[0]
    assert np.isclose(tot, ref, rtol=1e-12)


# ------------------------------------------------------------------ deposit
def random_moves(p, n, seed, maxmove=0.9, axis_crossers=True):
    rng = np.random.default_rng(seed)
    g = oracle.Grid(p)
    x = rng.uniform(0, p["nr"], n)
    y = rng.uniform(0, p["nth"], n)
    if axis_crossers:
        y[: n // 5] = rng.uniform(0, 0.4, n // 5)
        y[n // 5: 2 * n // 5] = p["nth"] - rng.uniform(0, 0.4, n // 5)
    xn = x + rng.uniform(-maxmove, maxmove, n)
    yn = y + rng.uniform(-maxmove, maxmove, n)
    old = dict(x1=p["xi_in"] + x * g.dxi, x2=y * g.dth, x3=rng.uniform(0, 6, n),
               flag=rng.integers(0, 2, n).astype(np.uint32))
    new = dict(x1=p["xi_in"] + xn * g.dxi, x2dep=yn * g.dth, x3=old["x3"] + rng.uniform(-.1, .1, n))
    # reflected new position (what the pusher stores)
    x2 = new["x2dep"].copy()
    x2 = np.where(x2 < 0, -x2, x2)
    x2 = np.where(x2 > np.pi, 2 * np.pi - x2, x2)
    new["x2"] = x2
    new["flag"] = old["flag"].copy()
    w = rng.uniform(0.5, 2.0, n)
    return old, new, w


def test_deposit_continuity_to_roundoff():
    """Eq.(21): d(rho dV)/dt + div(F) = 0 node by node, incl. the axis nodes (fold)."""
    p = small_params()
    g = oracle.Grid(p)
    old, new, w = random_moves(p, 400, 1)
    dt = 0.013
    F = oracle.fold_current(p, oracle.deposit(p, old, new, w, dt))
    rho0 = oracle.rho(p, old, w, divide=False)
    rho1 = oracle.rho(p, new, w, divide=False)
    G = g.G
    Fr, Fth = F[0], F[1]
    # interior nodes i = 1..nr-1 (radial edge nodes exchange charge with the guards), all j = 0..nth
    res = (rho1 - rho0) / dt
    div = np.zeros_like(res)
    div[G:G + p["nth"] + 1, 1:] += Fr[G:G + p["nth"] + 1, 1:] - Fr[G:G + p["nth"] + 1, :-1]
    div[G:G + p["nth"] + 1, :] += Fth[G:G + p["nth"] + 1, :] - Fth[G - 1:G + p["nth"], :]
    tot = (res + div)[G:G + p["nth"] + 1, G + 1:G + p["nr"]]
    scale = np.max(np.abs(rho1)) / dt
    assert np.max(np.abs(tot)) <= 1e-13 * scale, np.max(np.abs(tot)) / scale
    assert np.max(np.abs(res)) > 1e-3 * scale         # non-trivial


def test_deposit_bruteforce_whole_row_prefix_sum():
    """Literal Eq.(21)-(22): W_r, W_th on EVERY node of the (padded) grid, prefix sums along
    whole rows/columns; Eq.(23) on every node.  1..8 particles."""
    p = small_params(10, 8, 0.7)
    g = oracle.Grid(p)
    G, dt = g.G, 0.02
    for n in (1, 2, 5, 8):
        old, new, w = random_moves(p, n, 10 + n)
        F = oracle.deposit(p, old, new, w, dt)
        I = np.arange(-G, p["nr"] + G + 1)[None, :]
        J = np.arange(-G, p["nth"] + G + 1)[:, None]
        S = lambda x, y: np.maximum(0, 1 - np.abs(x - I)) * np.maximum(0, 1 - np.abs(y - J))
        Fr = np.zeros(g.shape); Fth = np.zeros(g.shape); Fph = np.zeros(g.shape)
        for k in range(n):
            Q = (1.0 if old["flag"][k] & 1 else -1.0) * w[k]
            xa, xb = (old["x1"][k] - p["xi_in"]) / g.dxi, (new["x1"][k] - p["xi_in"]) / g.dxi
            ya, yb = old["x2"][k] / g.dth, new["x2dep"][k] / g.dth
            Wr = 0.5 * Q * (S(xb, yb) - S(xa, yb) + S(xb, ya) - S(xa, ya))
            Wth = 0.5 * Q * (S(xb, yb) - S(xb, ya) + S(xa, yb) - S(xa, ya))
            Fr += -np.cumsum(Wr, axis=1) / dt
            Fth += -np.cumsum(Wth, axis=0) / dt
            Fph += Q * (new["x3"][k] - old["x3"][k]) / dt * (S(xb, yb) / 3 + S(xb, ya) / 6 + S(xa, yb) / 6 + S(xa, ya) / 3)
        sc = max(np.max(np.abs(Fr)), np.max(np.abs(Fth)))
        assert np.max(np.abs(F[0] - Fr)) < 1e-13 * sc
        assert np.max(np.abs(F[1] - Fth)) < 1e-13 * sc
        assert np.max(np.abs(F[2] - Fph)) < 1e-13 * np.max(np.abs(Fph))


def test_deposit_moments_and_sign():
    """sum F_ph = sum Q dphi/dt; sum F_r = sum Q (x'-x)/dt in index units: a positive charge
    moving to larger r gives positive J^r (sign convention of Eq.4 / reading G5)."""
    p = small_params()
    g = oracle.Grid(p)
    old, new, w = random_moves(p, 300, 5, axis_crossers=False)
    dt = 0.01
    F = oracle.deposit(p, old, new, w, dt)
    Q = np.where(old["flag"] & 1, 1.0, -1.0) * w
    assert np.isclose(F[2].sum(), np.sum(Q * (new["x3"] - old["x3"])) / dt, rtol=1e-12)
    assert np.isclose(F[0].sum(), np.sum(Q * (new["x1"] - old["x1"]) / g.dxi) / dt, rtol=1e-11)
    assert np.isclose(F[1].sum(), np.sum(Q * (new["x2dep"] - old["x2"]) / g.dth) / dt, rtol=1e-11)


def test_rho_total_charge():
    p = small_params()
    old, _, w = random_moves(p, 200, 7)
    Q = np.where(old["flag"] & 1, 1.0, -1.0) * w
    assert np.isclose(oracle.rho(p, old, w, divide=False).sum(), Q.sum(), rtol=1e-12)


# ------------------------------------------------------------------ field solver
def interior(g, X, m=2):
    return X[g.G + m:g.G + g.nth + 1 - m, g.G + m:g.G + g.nr + 1 - m]


@pytest.mark.parametrize("kind", ["wald", "monopole"])
def test_analytic_solutions_are_discretely_stationary_second_order(kind):
    """Appendix C fields are exact stationary vacuum solutions, so the discrete circulations
    (B8)-(B11) vanish as Delta^2.  Fails O(1) without the 1/2 in E_phi (reading G2) or with a
    wrong sign / index offset anywhere in B8-B11."""
    res = []
    for n in (16, 32, 64):
        p = inputs.grid_params(n, n, 0.9, r_out=20.0, r_in=1.3)
        g = oracle.Grid(p)
        f = inputs.analytic_fields(p, kind)
        Cs = oracle.circulation(p, f)
        # fixed physical sub-domain (1/8 of the range away from every boundary and the axis)
        res.append([np.max(np.abs(interior(g, Cs[c], n // 8))) for c in range(6)])
    res = np.array(res)
    assert np.all(res[2] < 2e-3), res[2]
    for c in range(6):
        if res[0, c] > 1e-9:
            assert res[0, c] / res[1, c] > 2.5 and res[1, c] / res[2, c] > 3.3, (c, res[:, c])


def divB(g, A, f):
    G, nr, nth = g.G, g.nr, g.nth
    Br, Bth = f[3] * A["ABr"], f[4] * A["ABth"]
    # cell (i+1/2, j+1/2), i<nr, j<nth
    return (Br[G:G + nth, G + 1:G + nr + 1] - Br[G:G + nth, G:G + nr]) + \
           (Bth[G + 1:G + nth + 1, G:G + nr] - Bth[G:G + nth, G:G + nr])


def test_divB_preserved_exactly_and_linearity():
    p = small_params(20, 16, 0.95, damp_cells=0)
    g = oracle.Grid(p)
    A = oracle.areas(p)
    rng = np.random.default_rng(2)
    f = [rng.normal(size=g.shape) for _ in range(6)]
    f = oracle.apply_bc(p, f)
    d0 = divB(g, A, f)
    f1 = [x.copy() for x in f]
    oracle.field_step(p, f1, None, 0.01)
    d1 = divB(g, A, f1)
    sc = np.max(np.abs(f[3] * A["ABr"]))
    assert np.max(np.abs(d1 - d0)) < 1e-13 * sc
    # linearity of the whole step in (D,B,J)
    h = [rng.normal(size=g.shape) for _ in range(6)]
    h = oracle.apply_bc(p, h)
    J = [rng.normal(size=g.shape) for _ in range(3)]
    s1 = oracle.field_step(p, [x.copy() for x in f], J, 0.01)
    s2 = oracle.field_step(p, [x.copy() for x in h], None, 0.01)
    s12 = oracle.field_step(p, [x + 2 * y for x, y in zip(f, h)], J, 0.01)
    for c in range(6):
        assert np.allclose(s12[c], s1[c] + 2 * s2[c], atol=1e-11 * np.max(np.abs(s12[c])))


def test_field_step_heun_limit_and_euler():
    """N=0 is forward Euler D^n + dt (C_H - J); N=1 with beta=1/2 is Heun's method
    (reading G3)."""
    p = small_params(16, 12, 0.9)
    g = oracle.Grid(p)
    f0 = inputs.analytic_fields(p, "wald")
    f0[5] = f0[5] + 1e-2 * np.exp(-((np.arange(g.shape[1])[None, :] - 10.0) ** 2 + (np.arange(g.shape[0])[:, None] - 8.0) ** 2) / 8.0)
    f0 = oracle.apply_bc(p, f0)
    rng = np.random.default_rng(4)
    J = [1e-3 * rng.normal(size=g.shape) for _ in range(3)]
    dt = 0.004
    # physical range of component c; D^ph, B^th are imposed (= 0) on the axis rows, skip those
    ph = lambda X, c: X[g.G + (1 if c in (2, 4) else 0):g.G + g.nth + (0 if c in (1, 2, 3, 4, 5) else 1),
                        g.G:g.G + g.nr + (0 if c in (0, 4, 5) else 1)]
    # Euler
    pe = dict(p, field_iters=0)
    fe = oracle.field_step(pe, [x.copy() for x in f0], J, dt)
    C0 = oracle.circulation(p, f0)
    for c in range(6):
        ref = f0[c] + dt * (C0[c] - (J[c] if c < 3 else 0))
        assert np.allclose(ph(fe[c], c), ph(ref, c), atol=1e-14 * np.max(np.abs(ref)) + 1e-18), c
    # Heun
    phn = dict(p, field_iters=1, beta_impl=0.5)
    fh = oracle.field_step(phn, [x.copy() for x in f0], J, dt)
    C1 = oracle.circulation(p, oracle.apply_bc(p, [x.copy() for x in fe]))
    for c in range(6):
        ref = f0[c] + dt * (0.5 * C0[c] + 0.5 * C1[c] - (J[c] if c < 3 else 0))
        assert np.allclose(ph(fh[c], c), ph(ref, c), atol=1e-14 * np.max(np.abs(ref)) + 1e-18), c


def test_field_step_second_order_in_dt():
    p = small_params(16, 12, 0.9, field_iters=7, beta_impl=0.5)
    g = oracle.Grid(p)
    f0 = inputs.analytic_fields(p, "monopole")
    bump = 1e-2 * np.exp(-((np.arange(g.shape[1])[None, :] - 10.0) ** 2 + (np.arange(g.shape[0])[:, None] - 8.0) ** 2) / 8.0)
    f0[5] = f0[5] + bump
    f0 = oracle.apply_bc(p, f0)
    T = 0.08
    def run(n):
        f = [x.copy() for x in f0]
        for _ in range(n):
            oracle.field_step(p, f, None, T / n)
        return f
    f1, f2, f4 = run(4), run(8), run(16)
    e1 = max(np.max(np.abs(interior(g, a - b))) for a, b in zip(f1, f2))
    e2 = max(np.max(np.abs(interior(g, a - b))) for a, b in zip(f2, f4))
    assert 3.2 < e1 / e2 < 4.8, (e1, e2)


def test_gauss_law_preserved_with_deposited_current():
    """div D - rho is unchanged by a step when J comes from the charge-conserving deposit
    (PAPER.md:130, :337), including the axis nodes (Eq.11)."""
    p = small_params(20, 16, 0.9)
    g = oracle.Grid(p)
    A = oracle.areas(p)
    dt = 0.01
    old, new, w = random_moves(p, 300, 9, maxmove=0.45)
    F = oracle.deposit(p, old, new, w, dt)
    J = oracle.finalize_current(p, [x.copy() for x in F], 0)
    f0 = oracle.apply_bc(p, inputs.analytic_fields(p, "monopole"))
    f1 = oracle.field_step(p, [x.copy() for x in f0], J, dt)
    G, nr, nth = g.G, g.nr, g.nth
    def divD(f):
        Dr, Dth = f[0] * A["ADr"], f[1] * A["ADth"]
        d = np.zeros(g.shape)
        d[:, 1:] += Dr[:, 1:] - Dr[:, :-1]
        d[G + 1:G + nth, :] += Dth[G + 1:G + nth, :] - Dth[G:G + nth - 1, :]
        d[G, :] += Dth[G, :]                     # axis theta=0: only the +1/2 face
        d[G + nth, :] += -Dth[G + nth - 1, :]    # axis theta=pi
        return d
    drho = oracle.rho(p, new, w, divide=False) - oracle.rho(p, old, w, divide=False)
    lhs = divD(f1) - divD(f0)
    sel = (slice(G, G + nth + 1), slice(G + 1, G + nr))
    sc = np.max(np.abs(drho))
    assert np.max(np.abs((lhs - drho)[sel])) < 1e-12 * sc
    assert sc > 0


def test_damping_layer_profile():
    p = small_params(20, 8, 0.9, damp_cells=5, damp_coef=0.8, field_iters=0)
    g = oracle.Grid(p)
    f = [np.ones(g.shape) for _ in range(6)]
    bg = [np.full(g.shape, 0.25) for _ in range(6)]
    out = oracle.field_step(p, [x.copy() for x in f], None, 0.0, bg=bg)
    i0 = 15
    for i in (14, 16, 18, 20):
        s = max(0, i - i0) / 5
        lam = 1 - 0.8 * s ** 3
        assert np.isclose(out[2][g.ij(i, 3)], 0.25 + 0.75 * lam, rtol=1e-14)


def test_filter_preserves_sums_and_kernel():
    p = small_params(12, 10, 0.5)
    g = oracle.Grid(p)
    F = [np.zeros(g.shape) for _ in range(3)]
    F[2][g.ij(5, 5)] = 16.0
    ref_area = oracle.areas(p)
    J = oracle.finalize_current(p, [x.copy() for x in F], 1)
    back = J[2] * ref_area["ADph"] * p["dphi"]
    assert np.isclose(back[g.ij(5, 5)], 4.0) and np.isclose(back[g.ij(4, 5)], 2.0)
    assert np.isclose(back[g.ij(4, 4)], 1.0) and np.isclose(back.sum(), 16.0)


# ------------------------------------------------------------------ sort / compaction
def test_sort_and_compact_definitions():
    rng = np.random.default_rng(0)
    n = 5000
    cell = rng.integers(0, 97, n).astype(np.uint32)
    flag = (rng.integers(0, 2, n) | (2 * (rng.uniform(size=n) < 0.1))).astype(np.uint32)
    perm = oracle.sort(cell, flag)
    key = np.where(flag & 2, 0xFFFFFFFF, cell).astype(np.uint64)
    assert np.array_equal(perm, np.argsort(key, kind="stable").astype(np.uint32))
    idx = oracle.compact(flag)
    assert np.array_equal(idx, np.nonzero((flag & 2) == 0)[0].astype(np.uint32))


def test_sort_interleaved_definition():
    """S11b: order by (cell // B, rank within the cell in stable order, cell % B), removed last in
    input order.  Pinned by (i) a hand-built example, (ii) numpy's lexsort of the defining tuple with
    ranks computed independently, (iii) B = 1 reducing to the plain stable sort, (iv) being a
    permutation whose adjacent live entries of equal rank sit in different cells."""
    # (i) cells of particles 0..7; B = 2: block 0 = cells {0,1}, block 1 = cells {2,3}
    cell = np.array([1, 0, 1, 3, 0, 2, 1, 3], dtype=np.uint32)
    flag = np.array([0, 0, 0, 0, 0, 2, 0, 0], dtype=np.uint32)       # particle 5 removed
    # cell 0: particles 1,4 (ranks 0,1); cell 1: 0,2,6 (ranks 0,1,2); cell 3: 3,7 (ranks 0,1)
    # block 0 rank-major: (r0: c0->1, c1->0), (r1: c0->4, c1->2), (r2: c1->6); block 1: 3, 7; tail: 5
    assert list(oracle.sort_interleaved(cell, flag, 4, 2)) == [1, 0, 4, 2, 6, 3, 7, 5]
    rng = np.random.default_rng(1)
    n, ncells = 6000, 137
    cell = rng.integers(0, ncells, n).astype(np.uint32)
    flag = (rng.integers(0, 2, n) | (2 * (rng.uniform(size=n) < 0.1))).astype(np.uint32)
    live = (flag & 2) == 0
    for B in (1, 2, 8, 32):
        perm = oracle.sort_interleaved(cell, flag, ncells, B)
        assert np.array_equal(np.sort(perm), np.arange(n, dtype=np.uint32))
        # (ii) ranks by counting earlier particles of the same cell
        rank = np.zeros(n, dtype=np.int64)
        seen = {}
        for k in range(n):
            if live[k]:
                rank[k] = seen.get(int(cell[k]), 0)
                seen[int(cell[k])] = rank[k] + 1
        c = cell.astype(np.int64)
        idx = np.arange(n)
        order = np.lexsort((idx, np.where(live, c % B, 0), rank, np.where(live, c // B, 1 << 40)))
        assert np.array_equal(perm, order.astype(np.uint32)), B
        if B == 1:      # (iii)
            assert np.array_equal(perm, oracle.sort(cell, flag))
        # (iv) inside a block, neighbours of equal rank are in different cells
        pc, pr = c[perm], rank[perm]
        nl = int(live.sum())
        same = (pc[1:nl] == pc[:nl - 1]) & (pr[1:nl] == pr[:nl - 1])
        assert not same.any()


# ------------------------------------------------------------------ third-order spline shape
def test_spline3_shape_is_the_cubic_bspline():
    """partition of unity, first moment, variance 1/3 (cubic B-spline = 4-fold convolution of the
    unit box: variance 4/12), support |x| < 2, C2 continuity at the knots, known values."""
    with oracle.shape_order(3):
        S = np.vectorize(oracle.shape)
        assert abs(S(0.0) - 2.0 / 3.0) < 1e-16 and abs(S(1.0) - 1.0 / 6.0) < 1e-16
        assert S(2.0) == 0.0 and S(-2.5) == 0.0 and S(1.999) > 0.0
        nodes = np.arange(-4, 5)
        for x in np.random.default_rng(0).uniform(-0.5, 0.5, 50):
            wts = S(x - nodes)
            assert abs(wts.sum() - 1.0) < 1e-15
            assert abs((wts * nodes).sum() - x) < 1e-15
            assert abs((wts * (nodes - x) ** 2).sum() - 1.0 / 3.0) < 1e-15
        h = 1e-5
        for knot in (-1.0, 0.0, 1.0):      # second derivative continuous across the knots
            d2l = (S(knot - 2 * h) - 2 * S(knot - h) + S(knot)) / h ** 2
            d2r = (S(knot) - 2 * S(knot + h) + S(knot + 2 * h)) / h ** 2
            assert abs(d2l - d2r) < 1e-4
    assert oracle.shape(0.25) == 0.75                      # option restored: cloud-in-cell


def test_spline3_deposit_continuity_and_moments():
    """The prefix-sum deposit (Eq.21-22) is charge conserving for any shape: with the cubic
    B-spline in BOTH rho and the fluxes the continuity residual is round-off, incl. axis nodes."""
    p = small_params()
    g = oracle.Grid(p)
    old, new, w = random_moves(p, 400, 4)
    dt = 0.013
    with oracle.shape_order(3):
        F = oracle.fold_current(p, oracle.deposit(p, old, new, w, dt))
        rho0 = oracle.rho(p, old, w, divide=False)
        rho1 = oracle.rho(p, new, w, divide=False)
    G = g.G
    Fr, Fth = F[0], F[1]
    res = (rho1 - rho0) / dt
    div = np.zeros_like(res)
    div[G:G + p["nth"] + 1, 1:] += Fr[G:G + p["nth"] + 1, 1:] - Fr[G:G + p["nth"] + 1, :-1]
    div[G:G + p["nth"] + 1, :] += Fth[G:G + p["nth"] + 1, :] - Fth[G - 1:G + p["nth"], :]
    tot = (res + div)[G:G + p["nth"] + 1, G + 2:G + p["nr"] - 1]       # support 2: nodes 2..nr-2
    scale = np.max(np.abs(rho1)) / dt
    assert np.max(np.abs(tot)) <= 1e-13 * scale, np.max(np.abs(tot)) / scale
    assert np.max(np.abs(res)) > 1e-3 * scale
    # moments (particles that stay clear of the radial edges): sum F_ph = sum Q dphi/dt
    Q = np.where(old["flag"] & 1, 1.0, -1.0) * w
    with oracle.shape_order(3):
        Fraw = oracle.deposit(p, old, new, w, dt)
    assert abs(Fraw[2].sum() - np.sum(Q * (new["x3"] - old["x3"])) / dt) < 1e-10 * np.sum(np.abs(Q)) / dt
    # and the cubic-spline fluxes differ from the cloud-in-cell ones (the option does something)
    F1 = oracle.deposit(p, old, new, w, dt)
    assert np.max(np.abs(F1[0] - Fraw[0])) > 1e-3 * np.max(np.abs(F1[0]))


def test_spline3_gather_reproduces_linear_fields():
    """a cubic B-spline reproduces linear functions exactly: the gather of a field linear in the
    logical coordinates returns the field at the particle (each component on its own lattice)."""
    p = small_params(nr=24, nth=20)
    g = oracle.Grid(p)
    rng = np.random.default_rng(2)
    n = 200
    x = rng.uniform(2.0, p["nr"] - 2.0, n)
    y = rng.uniform(2.5, p["nth"] - 2.5, n)
    x1, x2 = p["xi_in"] + x * g.dxi, y * g.dth
    fields, exact = [], []
    for k, name in enumerate(inputs.FIELD_NAMES):
        sr, sth = inputs.STAGGER[name][:2]
        ii = np.arange(-g.G, p["nr"] + g.G + 1)[None, :] + sr
        jj = np.arange(-g.G, p["nth"] + g.G + 1)[:, None] + sth
        a0, a1, a2 = 0.3 + k, 0.7 - 0.1 * k, -0.2 + 0.05 * k
        fields.append(np.ascontiguousarray(a0 + a1 * ii + a2 * jj + 0.0 * ii * jj))
        exact.append(a0 + a1 * x + a2 * y)
    with oracle.shape_order(3):
        got = np.array([oracle.gather(p, fields, x1[q], x2[q]) for q in range(n)])
    for k in range(6):
        assert np.allclose(got[:, k], exact[k], rtol=0, atol=1e-12), k


# ------------------------------------------------------------------ first-order gather (G11/G12) and filter edges (S10)
def _linear_fields(p, coef):
    """six stored arrays with F(i, j) = a + b (i + s_r) + c (j + s_theta) at every stored index"""
    G, nr, nth = p["ng"], p["nr"], p["nth"]
    jj, ii = np.meshgrid(np.arange(-G, nth + G + 1), np.arange(-G, nr + G + 1), indexing="ij")
    out = []
    for (a, b, c), name in zip(coef, inputs.FIELD_NAMES):
        sr, sth, _ = inputs.STAGGER[name]
        out.append(np.ascontiguousarray(a + b * (ii + sr) + c * (jj + sth), dtype=np.float64))
    return out


def test_cic_gather_exact_on_linear_fields_per_lattice():
    """PAPER.md:228, :297 'first order interpolation': bilinear weights on each component's OWN
    staggered lattice reproduce a field that is linear in the index coordinates exactly.  A wrong
    stagger offset, swapped x/y weights or a dropped corner shows up as an O(1) error."""
    p = small_params(20, 16, 0.9)
    rng = np.random.default_rng(5)
    coef = rng.uniform(-2, 2, (6, 3))
    fields = _linear_fields(p, coef)
    dxi, dth = inputs.spacing(p)
    for _ in range(200):
        fx, fy = rng.uniform(0, p["nr"]), rng.uniform(1.0, p["nth"] - 1.0)   # away from the axis rows
        got = oracle.gather(p, fields, p["xi_in"] + fx * dxi, fy * dth)
        want = coef[:, 0] + coef[:, 1] * fx + coef[:, 2] * fy
        assert np.allclose(got, want, rtol=0, atol=2e-13), (fx, fy, got - want)
    # each component only sees its own array: perturbing one array changes one output
    base = oracle.gather(p, fields, p["xi_in"] + 7.3 * dxi, 5.6 * dth)
    for c in range(6):
        f2 = [f.copy() for f in fields]
        f2[c] += 1.0
        d = oracle.gather(p, f2, p["xi_in"] + 7.3 * dxi, 5.6 * dth) - base
        assert np.allclose(d, np.eye(6)[c], atol=1e-13)


def test_cic_gather_axis_parity():
    """G12: beyond the axis a component continues with its parity under theta -> -theta (r, phi
    components even, theta components odd).  With random stored values the
    interpolant must be mirror symmetric about theta = 0 and theta = pi, odd components must vanish
    on the axis, and inside the first half cell a half-staggered even component must not depend on
    theta."""
    p = small_params(12, 10, 0.7)
    rng = np.random.default_rng(6)
    g = oracle.Grid(p)
    fields = [rng.uniform(-1, 1, g.shape) for _ in range(6)]
    G, nth = p["ng"], p["nth"]
    for name in ("Dph", "Bth"):                     # axis nodes of D^phi, B^theta are zero
        k = inputs.FIELD_NAMES.index(name)
        fields[k][G, :] = 0.0
        fields[k][G + nth, :] = 0.0
    dxi, dth = inputs.spacing(p)
    par = np.array([inputs.STAGGER[n][2] for n in inputs.FIELD_NAMES], dtype=float)
    par[inputs.FIELD_NAMES.index("Dph")] = +1.0
    for _ in range(100):
        x1 = p["xi_in"] + rng.uniform(1, p["nr"] - 1) * dxi
        t = rng.uniform(0.0, 1.9) * dth
        up, dn = oracle.gather(p, fields, x1, t), oracle.gather(p, fields, x1, -t)
        assert np.allclose(dn, par * up, atol=1e-14), (t / dth, dn, up)
        up, dn = oracle.gather(p, fields, x1, math.pi - t), oracle.gather(p, fields, x1, math.pi + t)
        assert np.allclose(dn, par * up, atol=1e-13), (t / dth, dn, up)
    x1 = p["xi_in"] + 4.25 * dxi
    on_axis = oracle.gather(p, fields, x1, 0.0)
    for name in ("Dth", "Bth"):
        assert abs(on_axis[inputs.FIELD_NAMES.index(name)]) < 1e-15
    kBr = inputs.FIELD_NAMES.index("Br")            # half-staggered, even: flat across the axis
    a = oracle.gather(p, fields, x1, 0.1 * dth)[kBr]
    b = oracle.gather(p, fields, x1, 0.4 * dth)[kBr]
    row0 = 0.75 * fields[kBr][g.ij(4, 0)] + 0.25 * fields[kBr][g.ij(5, 0)]
    assert abs(a - b) < 1e-15 and abs(a - row0) < 1e-15


def _filter_numpy(F, p, half_theta, parity):
    """(1,2,1) x (1,2,1) / 16 on the physical rows: theta neighbours beyond the axis by parity,
    radial neighbours beyond the first / last stored node clamped (S10), written with numpy slices."""
    G, nr, nth = p["ng"], p["nr"], p["nth"]
    jhi = nth - 1 if half_theta else nth
    A = F[G:G + jhi + 1, :].copy()                   # rows 0..jhi, all stored columns
    if half_theta:
        lo, hi = parity * A[0], parity * A[jhi]      # row -1/2 mirrors row +1/2
    else:
        lo, hi = parity * A[1], parity * A[jhi - 1]  # row -1 mirrors row +1
    T = np.vstack([lo, A, hi])
    T = (T[:-2] + 2 * T[1:-1] + T[2:]) / 4.0
    R = np.hstack([T[:, :1], T, T[:, -1:]])
    R = (R[:, :-2] + 2 * R[:, 1:-1] + R[:, 2:]) / 4.0
    out = F.copy()
    out[G:G + jhi + 1, :] = R
    return out


def test_filter_pass_matches_numpy_convolution_including_edges():
    """S10 on a random array, every physical row and every stored column (axis rows 0 and n_theta,
    first and last radial guard), one and three passes, against a numpy convolution with parity
    padding: pins the stencil weights, the parity sign per component and the radial clamp."""
    p = small_params(14, 9, 0.6)
    rng = np.random.default_rng(8)
    g = oracle.Grid(p)
    F0 = [rng.uniform(-1, 1, g.shape) for _ in range(3)]
    A = oracle.areas(p)
    area = [A["ADr"], A["ADth"], A["ADph"] * p["dphi"]]
    folded = oracle.fold_current(p, [x.copy() for x in F0])
    for passes in (1, 3):
        J = oracle.finalize_current(p, [x.copy() for x in F0], passes)
        ref = [x.copy() for x in folded]
        for _ in range(passes):
            ref = [_filter_numpy(ref[0], p, False, +1.0), _filter_numpy(ref[1], p, True, -1.0),
                   _filter_numpy(ref[2], p, False, +1.0)]
        for c in range(3):
            ok = area[c] > 0
            assert np.allclose((J[c] * area[c])[ok], ref[c][ok], rtol=1e-13, atol=1e-14), (passes, c)


def test_field_step_threads_bit_identical():
    """The OpenMP loops of the oracle's field step run over grid rows with no reduction: one thread
    and all threads must give the same bits (areas, circulations, a full N = 7 step with damping)."""
    p = small_params(40, 28, 0.9, damp_cells=6, damp_coef=1.0)
    rng = np.random.default_rng(12)
    f0 = inputs.fill_guards(p, inputs.perturb(inputs.analytic_fields(p, "wald"), 1e-2, rng))
    J = [rng.uniform(-1e-3, 1e-3, f0[0].shape) for _ in range(3)]
    dt = inputs.courant_dt(p)
    old = oracle.set_num_threads(1)
    try:
        A1 = oracle.areas(p)
        C1 = oracle.circulation(p, f0)
        F1 = oracle.field_step(p, [f.copy() for f in f0], J, dt, bg=f0)
        oracle.set_num_threads(max(2, old))
        A2 = oracle.areas(p)
        C2 = oracle.circulation(p, f0)
        F2 = oracle.field_step(p, [f.copy() for f in f0], J, dt, bg=f0)
    finally:
        oracle.set_num_threads(old)
    for k in A1:
        assert np.array_equal(A1[k], A2[k]), k
    for a, b in zip(C1 + F1, C2 + F2):
        assert np.array_equal(a, b)


def test_damping_layer_properties():
    """PAPER.md:138 gives no profile (reading G14); whatever the profile, an absorbing layer must
    (1) leave every column inside i <= nr - damp_cells bit-exactly alone, (2) pull the fields towards
    the background, never past it and never away from it (0 <= lambda <= 1), (3) act monotonically
    more strongly outwards, (4) be the identity on a field that equals the background, and (5) vanish
    continuously at its inner edge.  dt = 0 isolates the damping stage of the step."""
    p = small_params(40, 10, 0.9, damp_cells=12, damp_coef=0.7, field_iters=2)
    g = oracle.Grid(p)
    rng = np.random.default_rng(3)
    bg = inputs.fill_guards(p, [rng.uniform(-1, 1, g.shape) for _ in range(6)])
    f = inputs.fill_guards(p, [b + rng.uniform(0.5, 1.5, g.shape) for b in bg])    # f - bg > 0 everywhere
    out = oracle.field_step(p, [x.copy() for x in f], None, 0.0, bg=bg)
    G, nr, nth = p["ng"], p["nr"], p["nth"]
    i0 = nr - p["damp_cells"]
    for c, name in enumerate(inputs.FIELD_NAMES):
        sr, sth, _ = inputs.STAGGER[name]
        jlo, jhi = (1, nth - 1) if name in ("Dph", "Bth") else (0, nth if sth == 0.0 else nth - 1)
        ihi = nr if sr == 0.0 else nr - 1
        rows = slice(G + jlo, G + jhi + 1)
        assert np.array_equal(out[c][rows, G:G + i0 + 1], f[c][rows, G:G + i0 + 1]), name          # (1)
        lam = (out[c][rows, G + i0 + 1:G + ihi + 1] - bg[c][rows, G + i0 + 1:G + ihi + 1]) / \
              (f[c][rows, G + i0 + 1:G + ihi + 1] - bg[c][rows, G + i0 + 1:G + ihi + 1])
        assert np.all(lam >= 0.0) and np.all(lam <= 1.0), name                                     # (2)
        assert np.all(np.diff(lam, axis=1) <= 1e-15), name                                         # (3)
        assert np.all(lam[:, 0] > 0.999) and np.all(lam[:, -1] < 0.5), name                        # (5), strong at the edge
        assert np.allclose(lam, lam[:1, :], atol=1e-14), name                                      # same for every row
    same = oracle.field_step(p, [x.copy() for x in bg], None, 0.0, bg=bg)                          # (4)
    for c, name in enumerate(inputs.FIELD_NAMES):
        sth = inputs.STAGGER[name][1]
        jlo, jhi = (1, nth - 1) if name in ("Dph", "Bth") else (0, nth if sth == 0.0 else nth - 1)
        assert np.array_equal(same[c][G + jlo:G + jhi + 1, G:G + nr], bg[c][G + jlo:G + jhi + 1, G:G + nr]), name
