"""Pins of the CPU oracle's metric, geodesic integrator and Boris push against what the
paper and the mathematics fix (not against the oracle itself, and never against CUDA)."""
import math
import os

import numpy as np
import pytest

import oracle
import inputs

HERE = os.path.dirname(os.path.abspath(__file__))


def table1():
    rows = {}
    for line in open(os.path.join(HERE, "golden", "table1_orbits.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        rows[t[0]] = dict(a=float(t[1]), B0=float(t[2]), ur=float(t[3]), uth=float(t[4]),
                          uph=float(t[5]), r=float(t[6]), th=math.pi / 2 - float(t[7]))
    return rows


# ------------------------------------------------------------------ metric (Appendix A)
@pytest.mark.parametrize("a,M,r,th", [(0.99, 1.0, 1.3, 0.4), (0.5, 1.0, 7.0, 2.5),
                                      (0.0, 1.0, 3.0, 1.0), (0.9, 2.0, 5.0, 0.05)])
def test_metric_inverse_det_and_sqrtg(a, M, r, th):
    m = oracle.metric(a, M, r, th)
    g = np.array([[m["g_rr"], 0, m["g_rph"]], [0, m["g_thth"], 0], [m["g_rph"], 0, m["g_phph"]]])
    gu = np.array([[m["gu_rr"], 0, m["gu_rph"]], [0, m["gu_thth"], 0], [m["gu_rph"], 0, m["gu_phph"]]])
    assert np.allclose(g @ gu, np.eye(3), atol=1e-13)
    assert np.isclose(np.linalg.det(g), m["sqrtg"] ** 2, rtol=1e-13)
    # 4-metric consistency: g_tt = beta^2 - alpha^2 = z - 1, g_tr = beta_r = z   (A2)
    z = 2 * M * r / (r * r + a * a * math.cos(th) ** 2)
    beta_lo_r = m["g_rr"] * m["beta_r"]
    assert np.isclose(beta_lo_r * m["beta_r"] - m["alpha"] ** 2, z - 1.0, rtol=1e-13)
    assert np.isclose(beta_lo_r, z, rtol=1e-13)
    # g_t_phi = beta_phi = gamma_{phi r} beta^r = -a z sin^2     (A2)
    assert np.isclose(m["g_rph"] * m["beta_r"], -a * z * math.sin(th) ** 2, rtol=1e-13, atol=1e-300)


@pytest.mark.parametrize("a,M,r,th", [(0.99, 1.0, 1.3, 0.4), (0.5, 1.0, 7.0, 2.5), (0.9, 2.0, 5.0, 0.3)])
def test_metric_derivatives_finite_difference(a, M, r, th):
    m = oracle.metric(a, M, r, th)
    h = 1e-5
    for q in ("alpha", "beta", "gu_rr", "gu_thth", "gu_phph", "gu_rph"):
        key = "beta_r" if q == "beta" else q
        # 4th-order central differences
        def f(rr, tt):
            return oracle.metric(a, M, rr, tt)[key]
        dr = (-f(r + 2 * h, th) + 8 * f(r + h, th) - 8 * f(r - h, th) + f(r - 2 * h, th)) / (12 * h)
        dth = (-f(r, th + 2 * h) + 8 * f(r, th + h) - 8 * f(r, th - h) + f(r, th - 2 * h)) / (12 * h)
        assert np.isclose(m["dr_" + q], dr, rtol=1e-8, atol=1e-10), q
        assert np.isclose(m["dth_" + q], dth, rtol=1e-8, atol=1e-10), q


def test_metric_matches_independent_form():
    # the input generator writes Appendix A in a different algebraic form (no Sigma, Delta)
    rng = np.random.default_rng(0)
    for _ in range(20):
        a, r, th = rng.uniform(0, 0.999), rng.uniform(1.0, 40.0), rng.uniform(0.01, 3.13)
        m, k = oracle.metric(a, 1.0, r, th), inputs.kerr_schild(a, 1.0, r, th)
        for key in ("alpha", "beta_r", "g_rr", "g_thth", "g_phph", "g_rph", "gu_rr", "gu_thth",
                    "gu_phph", "gu_rph", "sqrtg"):
            assert np.isclose(m[key], float(k[key]), rtol=1e-13), key


# ------------------------------------------------------------------ geodesics
def energy(a, M, y):
    """E = -u_t = alpha^2 u^0 - beta^r u_r (massive)."""
    m = oracle.metric(a, M, y[0], y[1])
    u = y[3:6]
    nrm = m["gu_rr"] * u[0] ** 2 + m["gu_thth"] * u[1] ** 2 + m["gu_phph"] * u[2] ** 2 + 2 * m["gu_rph"] * u[0] * u[2]
    u0 = math.sqrt(1 + nrm) / m["alpha"]
    return m["alpha"] ** 2 * u0 - m["beta_r"] * u[0]


def test_geodesic_uphi_exact_and_energy_second_order():
    o = table1()["(3,3,2)"]
    y0 = np.array([o["r"], o["th"], 0.0, o["ur"], o["uth"], o["uph"]])
    errs = []
    for dt in (0.1, 0.05, 0.025):
        n = int(round(120.0 / dt))
        tr = oracle.geodesic_traj(o["a"], 1.0, 3, y0, dt, n, every=1)
        assert np.all(tr[:, 5] == y0[5])           # U_phi = 0: bit-exact conservation
        E = np.array([energy(o["a"], 1.0, y) for y in tr[:: max(1, n // 400)]])
        errs.append(np.mean(np.abs(E - E[0])))
    # "relative error decreases as dt^2"
    assert 3.3 < errs[0] / errs[1] < 4.7 and 3.3 < errs[1] / errs[2] < 4.7, errs


@pytest.mark.parametrize("name,zwv", [("(2,0,1)", (2, 0, 1)), ("(3,3,1)", (3, 3, 1)),
                                      ("(3,3,2)", (3, 3, 2)), ("(4,3,1)", (4, 3, 1))])
def test_table1_periodic_orbit_taxonomy(name, zwv):
    """Table 1 rows start at apoapsis; over one radial period the azimuth advances by
    2 pi (1 + w + v/z) for a (z,w,v) periodic orbit."""
    o = table1()[name]
    z, w, v = zwv
    y0 = np.array([o["r"], o["th"], 0.0, o["ur"], o["uth"], o["uph"]])
    dt = 0.02
    n = int(600.0 / dt)
    tr = oracle.geodesic_traj(o["a"], 1.0, 3, y0, dt, n, every=1)
    r, ph = tr[:, 0], tr[:, 2]
    assert np.allclose(tr[:, 1], math.pi / 2, atol=1e-12)     # stays equatorial
    # first interior local maximum of r after leaving apoapsis = next apoapsis
    k = np.where((r[1:-1] > r[:-2]) & (r[1:-1] >= r[2:]) & (np.arange(1, n - 1) > 100))[0][0] + 1
    # parabolic refinement of the apoapsis time
    den = r[k - 1] - 2 * r[k] + r[k + 1]
    off = 0.5 * (r[k - 1] - r[k + 1]) / den
    phi_apo = ph[k] + off * 0.5 * (ph[k + 1] - ph[k - 1])
    assert abs(phi_apo / (2 * math.pi) - (1 + w + v / z)) < 2e-3
    assert abs(r[k] - o["r"]) < 2e-3 * o["r"]


@pytest.mark.parametrize("a,rfac", [(0.0, 1.0), (0.9, 1.5), (0.99, 1.5)])
def test_circular_orbit_frequency(a, rfac):
    """Textbook prograde circular equatorial Kerr orbits (Bardeen, Press & Teukolsky 1972):
    Omega = 1/(r^{3/2}+a); r_isco(a=0) = 6 gives Omega = 6^{-3/2} = 0.0680413817."""
    Z1 = 1 + (1 - a * a) ** (1 / 3) * ((1 + a) ** (1 / 3) + (1 - a) ** (1 / 3))
    Z2 = math.sqrt(3 * a * a + Z1 * Z1)
    r_isco = 3 + Z2 - math.sqrt((3 - Z1) * (3 + Z1 + 2 * Z2))
    if a == 0.0:
        assert abs(r_isco - 6.0) < 1e-12
    r = rfac * r_isco
    den = r ** 0.75 * math.sqrt(r ** 1.5 - 3 * math.sqrt(r) + 2 * a)
    E = (r ** 1.5 - 2 * math.sqrt(r) + a) / den
    L = (r * r - 2 * a * math.sqrt(r) + a * a) / den
    Delta = r * r + a * a - 2 * r
    # BL -> KS covariant momentum (from A6): u_r^KS = u_r^BL + (2 r E - a L)/Delta
    y0 = np.array([r, math.pi / 2, 0.0, (2 * r * E - a * L) / Delta, 0.0, L])
    assert abs(energy(a, 1.0, y0) - E) < 1e-12
    Omega = 1.0 / (r ** 1.5 + a)
    T = 2 * math.pi / Omega
    dt = T / 20000
    tr = oracle.geodesic_traj(a, 1.0, 3, y0, dt, 20001, every=1)
    assert np.max(np.abs(tr[:, 0] - r)) < 2e-6 * r
    assert abs((tr[-1, 2] - tr[0, 2]) / (20000 * dt) - Omega) < 1e-7
    if a == 0.0 and rfac == 1.0:
        assert abs(Omega - 0.0680413817) < 1e-9


def test_photon_null_and_energy():
    a = 0.9
    m = oracle.metric(a, 1.0, 6.0, 1.0)
    y0 = np.array([6.0, 1.0, 0.0, 0.3, 1.0, 2.0])
    tr = oracle.geodesic_traj(a, 1.0, 3, y0, 0.01, 2000, every=100, eps=0.0)
    def Eph(y):
        mm = oracle.metric(a, 1.0, y[0], y[1])
        u = y[3:6]
        nrm = mm["gu_rr"] * u[0] ** 2 + mm["gu_thth"] * u[1] ** 2 + mm["gu_phph"] * u[2] ** 2 + 2 * mm["gu_rph"] * u[0] * u[2]
        return mm["alpha"] * math.sqrt(nrm) - mm["beta_r"] * u[0]
    E = np.array([Eph(y) for y in tr])
    assert np.max(np.abs(E - E[0])) < 1e-5 * abs(E[0])


# ------------------------------------------------------------------ Boris (Eq.16-19)
def _cross_lo(m, A, B):
    return m["sqrtg"] * np.cross(A, B)


def _raise(m, u):
    return np.array([m["gu_rr"] * u[0] + m["gu_rph"] * u[2], m["gu_thth"] * u[1],
                     m["gu_rph"] * u[0] + m["gu_phph"] * u[2]])


def _lower(m, v):
    return np.array([m["g_rr"] * v[0] + m["g_rph"] * v[2], m["g_thth"] * v[1],
                     m["g_rph"] * v[0] + m["g_phph"] * v[2]])


def test_boris_norm_residual_and_angle():
    a, r, th = 0.99, 1.7, 0.6
    m = oracle.metric(a, 1.0, r, th)
    rng = np.random.default_rng(3)
    u = rng.normal(size=3) * 3
    B = rng.normal(size=3)
    D = rng.normal(size=3) * 0.3
    dt, sgn = 0.05, -1.0
    # (i) pure magnetic rotation preserves gamma^ij u_i u_j to round-off
    up = oracle.boris(a, 1.0, r, th, u, np.zeros(3), B, sgn, dt)
    n0, n1 = u @ _raise(m, u), up @ _raise(m, up)
    assert abs(n1 - n0) < 1e-13 * n0
    # rotation angle = 2 atan sqrt(t_k t^k)
    u0bar = math.sqrt(1 + n0) / m["alpha"]
    t = sgn * B * dt / (2 * u0bar)
    t2 = t @ _lower(m, t)
    # decompose u^i perpendicular to B^i with the metric inner product
    uu, upu = _raise(m, u), _raise(m, up)
    Bl = _lower(m, B)
    perp = lambda x: x - (x @ Bl) / (B @ Bl) * B
    pa, pb = perp(uu), perp(upu)
    cosang = (pa @ _lower(m, pb)) / math.sqrt((pa @ _lower(m, pa)) * (pb @ _lower(m, pb)))
    assert abs(math.acos(cosang) - 2 * math.atan(math.sqrt(t2))) < 1e-12
    # (ii) Eq.(16) with ubar = (u^- + u^+)/2 and ubar^0 of Eq.(18) is solved exactly
    up = oracle.boris(a, 1.0, r, th, u, D, B, sgn, dt)
    Dl = _lower(m, D)
    um = u + sgn * m["alpha"] * dt / 2 * Dl
    upl = up - sgn * m["alpha"] * dt / 2 * Dl
    ubar = 0.5 * (um + upl)
    u0b = math.sqrt(1 + um @ _raise(m, um)) / m["alpha"]
    rhs = u + sgn * dt * (m["alpha"] * Dl + _cross_lo(m, _raise(m, ubar), B) / u0b)
    assert np.max(np.abs(up - rhs)) < 1e-13 * np.max(np.abs(up))


def test_flat_space_gyration():
    """M = 0, a = 0: special-relativistic gyration in uniform B_z = B0:
    B^r = B0 cos(th), B^th = -B0 sin(th)/r; |u| constant, phase advance per step
    2 atan(q B0 dt / (2 m Gamma)); full push = Boris + straight-line geodesic."""
    B0, dt = 2.0, 0.01
    r, th, ph = 5.0, 1.1, 0.3
    # Cartesian momentum (ux, uy, uz) -> covariant spherical components
    ux, uy, uz = 1.5, -0.7, 0.4
    Gam = math.sqrt(1 + ux * ux + uy * uy + uz * uz)
    def to_cov(r, th, ph, ux, uy, uz):
        er = np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
        et = np.array([math.cos(th) * math.cos(ph), math.cos(th) * math.sin(ph), -math.sin(th)])
        ep = np.array([-math.sin(ph), math.cos(ph), 0.0])
        U = np.array([ux, uy, uz])
        return np.array([U @ er, r * (U @ et), r * math.sin(th) * (U @ ep)]), (er, et, ep)
    u, _ = to_cov(r, th, ph, ux, uy, uz)
    pos = np.array([r * math.sin(th) * math.cos(ph), r * math.sin(th) * math.sin(ph), r * math.cos(th)])
    y = np.array([r, th, ph, *u])
    nsteps = 400
    for _ in range(nsteps):
        B = np.array([B0 * math.cos(y[1]), -B0 * math.sin(y[1]) / y[0], 0.0])
        ub = oracle.boris(0.0, 0.0, y[0], y[1], y[3:6], np.zeros(3), B, +1.0, dt)
        y = oracle.geodesic(0.0, 0.0, 3, np.array([y[0], y[1], y[2], *ub]), dt)
    # back to Cartesian momentum
    r1, th1, ph1 = y[0:3]
    er = np.array([math.sin(th1) * math.cos(ph1), math.sin(th1) * math.sin(ph1), math.cos(th1)])
    et = np.array([math.cos(th1) * math.cos(ph1), math.cos(th1) * math.sin(ph1), -math.sin(th1)])
    ep = np.array([-math.sin(ph1), math.cos(ph1), 0.0])
    U = y[3] * er + y[4] / r1 * et + y[5] / (r1 * math.sin(th1)) * ep
    assert abs(np.linalg.norm(U) - math.sqrt(ux * ux + uy * uy + uz * uz)) < 1e-6
    assert abs(U[2] - uz) < 1e-6                        # u_z unchanged along B
    # positive charge in B_z gyrates clockwise: phase = -n * 2 atan(B0 dt/(2 Gamma)), up to the
    # O(dt^2) splitting error of moving-frame bases
    phase = math.atan2(U[1], U[0]) - math.atan2(uy, ux)
    expect = -nsteps * 2 * math.atan(B0 * dt / (2 * Gam))
    assert abs((phase - expect + math.pi) % (2 * math.pi) - math.pi) < 2e-4
    # z advances uniformly
    assert abs(r1 * math.cos(th1) - (pos[2] + uz / Gam * nsteps * dt)) < 1e-5


# ------------------------------------------------------------------ charged orbit, Eq.(24)
@pytest.mark.parametrize("name", ["RKA3", "RKA8"])
def test_charged_orbit_conserves_eq24(name):
    """Full step (Boris with the analytic Wald field of C14-C19 + geodesic) conserves
    E = -u_0 - (q/m) A_0 (Eq.24) and L = u_phi + (q/m) A_phi, with the
    potentials of (C12), to second order in dt."""
    o = table1()[name]
    a, B0, qm = o["a"], o["B0"], +1.0

    def A_t(r, th):
        c2 = math.cos(th) ** 2
        return B0 * (a * r * (1 + c2) / (r * r + a * a * c2) - a)

    def A_ph(r, th):
        c2 = math.cos(th) ** 2
        return B0 * 0.5 * math.sin(th) ** 2 * (r * r + a * a - 2 * a * a * r * (1 + c2) / (r * r + a * a * c2))

    def half_boris(y, dt):
        D = [float(v) for v in inputs.analytic_DB(a, 1.0, B0, y[0], y[1], "wald")]
        ub = oracle.boris(a, 1.0, y[0], y[1], y[3:6], D[0:3], D[3:6], qm, 0.5 * dt)
        return np.array([y[0], y[1], y[2], *ub])

    def run(dt, T):
        y = np.array([o["r"], o["th"], 0.0, o["ur"], o["uth"], o["uph"]])
        E0 = energy(a, 1.0, y) - qm * A_t(y[0], y[1])
        L0 = y[5] + qm * A_ph(y[0], y[1])
        dE = dL = 0.0
        for _ in range(int(round(T / dt))):
            # Strang sequence of PAPER.md:155: half Boris, full geodesic, half Boris at the new
            # position (the production loop bundles adjacent halves into one full Boris, :204)
            y = half_boris(y, dt)
            y = oracle.geodesic(a, 1.0, 3, y, dt)
            y = half_boris(y, dt)
            dE = max(dE, abs(energy(a, 1.0, y) - qm * A_t(y[0], y[1]) - E0))
            dL = max(dL, abs(y[5] + qm * A_ph(y[0], y[1]) - L0))
        return dE / abs(E0), dL / abs(L0)

    e1, l1 = run(0.02, 20.0)
    e2, l2 = run(0.01, 20.0)
    assert e1 < 2e-3 and l1 < 2e-3
    assert 2.8 < e1 / e2 < 5.5 and 2.8 < l1 / l2 < 5.5, (e1, e2, l1, l2)


# ------------------------------------------------------------------ photon species
def test_photon_species_push_ignores_fields_and_moves_at_light_speed():
    """flag bit2 = photon: no Lorentz force (identical result in any field), eps = 0 in u^0.
    Flat space (M = 0): a photon follows a straight line at unit speed whatever |u| is
    (closed form), and its energy |u| is conserved; pins eps = 0 (a massive particle with the
    same u would move at |u|/sqrt(1+u^2) < 1)."""
    import inputs
    p = inputs.grid_params(32, 32, 0.0, r_out=40.0, r_in=2.0, M=0.0)
    strong = [np.full(inputs.grid_shape(p), 3.0) for _ in range(6)]
    zero = [np.zeros(inputs.grid_shape(p)) for _ in range(6)]
    n = 64
    rng = np.random.default_rng(5)
    r0 = rng.uniform(5.0, 20.0, n)
    th0 = rng.uniform(0.5, 2.6, n)
    # local orthonormal direction (e_r, e_theta, e_phi), |u| = p0
    d = rng.normal(size=(n, 3)); d /= np.linalg.norm(d, axis=1)[:, None]
    p0 = rng.uniform(0.05, 50.0, n)
    ptc = dict(x1=np.log(r0), x2=th0.copy(), x3=np.zeros(n), u1=p0 * d[:, 0], u2=p0 * d[:, 1] * r0,
               u3=p0 * d[:, 2] * r0 * np.sin(th0), w=np.ones(n),
               flag=np.full(n, 4, np.uint32), cell=inputs.cells_of(p, np.log(r0), th0))
    dt, steps = 0.01, 100
    cur_a, cur_b = dict(ptc), dict(ptc)
    for _ in range(steps):
        na, nb = oracle.push(p, strong, cur_a, dt), oracle.push(p, zero, cur_b, dt)
        for k in ("x1", "x2", "x3", "u1", "u2", "u3"):
            assert np.array_equal(na[k], nb[k]), k                      # fields are not seen
        cur_a = {**cur_a, **{k: na[k] for k in ("x1", "x2", "x3", "u1", "u2", "u3", "flag", "cell")}}
        cur_b = {**cur_b, **{k: nb[k] for k in ("x1", "x2", "x3", "u1", "u2", "u3", "flag", "cell")}}
    def cart(x1, x2, x3):
        r = np.exp(x1)
        return np.stack([r * np.sin(x2) * np.cos(x3), r * np.sin(x2) * np.sin(x3), r * np.cos(x2)], 1)
    X0, X1 = cart(ptc["x1"], ptc["x2"], ptc["x3"]), cart(cur_a["x1"], cur_a["x2"], cur_a["x3"])
    er = np.stack([np.sin(th0), np.zeros(n), np.cos(th0)], 1)
    et = np.stack([np.cos(th0), np.zeros(n), -np.sin(th0)], 1)
    ep = np.stack([np.zeros(n), np.ones(n), np.zeros(n)], 1)
    dirc = d[:, :1] * er + d[:, 1:2] * et + d[:, 2:3] * ep
    T = dt * steps
    assert np.max(np.linalg.norm(X1 - (X0 + T * dirc), axis=1)) < 2e-4      # straight line, speed 1 (O(dt^2))
    r1, t1 = np.exp(cur_a["x1"]), cur_a["x2"]
    pmag = np.sqrt(cur_a["u1"] ** 2 + (cur_a["u2"] / r1) ** 2 + (cur_a["u3"] / (r1 * np.sin(t1))) ** 2)
    assert np.max(np.abs(pmag / p0 - 1.0)) < 1e-5
    # the same states as MASSIVE particles are slower: eps matters
    mass = dict(ptc); mass["flag"] = np.zeros(n, np.uint32)
    nm = oracle.push(p, zero, mass, dt)
    v_m = np.linalg.norm(cart(nm["x1"], nm["x2"], nm["x3"]) - X0, axis=1) / dt
    assert np.all(v_m < 1.0) and np.allclose(v_m, p0 / np.sqrt(1 + p0 ** 2), rtol=1e-3)


def test_photons_carry_no_current_and_no_charge():
    import inputs
    p = inputs.grid_params(24, 20, 0.9)
    ptc = inputs.make_particles(p, 400, 3, "logical", ("loguniform", 0.1, 10.0))
    fields = inputs.analytic_fields(p, "monopole")
    dt = inputs.courant_dt(p)
    ph = np.arange(400) % 3 == 0
    mixed = dict(ptc); mixed["flag"] = (ptc["flag"] | np.where(ph, 4, 0)).astype(np.uint32)
    new = oracle.push(p, fields, mixed, dt)
    F = oracle.deposit(p, mixed, new, mixed["w"], dt)
    sub = {k: np.ascontiguousarray(v[~ph]) for k, v in mixed.items()}
    nsub = {k: np.ascontiguousarray(v[~ph]) for k, v in new.items()}
    Fs = oracle.deposit(p, sub, nsub, sub["w"], dt)
    for a, b in zip(F, Fs):
        assert np.allclose(a, b, rtol=0, atol=1e-13 * max(1.0, np.max(np.abs(b))))
    assert np.allclose(oracle.rho(p, mixed, mixed["w"]), oracle.rho(p, sub, sub["w"]), rtol=0, atol=1e-14)


# ------------------------------------------------------------------ pair production (Eq.26)
def test_philox_known_answers():
    here = os.path.dirname(os.path.abspath(__file__))
    rows = [l.split() for l in open(os.path.join(here, "golden", "philox4x32_10.txt")) if l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == v[6:10]
    u = np.array([oracle.uniform(7, 3, k) for k in range(20000)])
    assert 0.0 <= u.min() and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.01 and abs(u.var() - 1.0 / 12.0) < 0.005
    assert oracle.uniform(7, 3, 5) != oracle.uniform(7, 4, 5) != oracle.uniform(8, 3, 5)


def _fido_norm(a, M, x1, x2, u1, u2, u3):
    out = np.zeros(len(x1))
    for k in range(len(x1)):
        m = oracle.metric(a, M, math.exp(x1[k]), x2[k])
        out[k] = (m["gu_rr"] * u1[k] ** 2 + m["gu_thth"] * u2[k] ** 2 + m["gu_phph"] * u3[k] ** 2
                  + 2 * m["gu_rph"] * u1[k] * u3[k])
    return out


def test_pair_production_conserves_fido_momentum_and_energy():
    """emission: photon + recoiling lepton carry the lepton's covariant momentum, the photon's FIDO
    energy is eps_ph and only leptons with Gamma >= gamma_thr emit; conversion: a fraction
    p_convert of the photons (Eq.26), the two leptons share the photon's FIDO energy, all momenta
    parallel; children appended in parent order with position, cell and weight of the parent."""
    import inputs
    p = inputs.grid_params(32, 32, 0.9)
    n = 6000
    ptc = inputs.make_particles(p, n, 9, "logical", ("loguniform", 1.0, 1e3))
    ph = np.arange(n) % 2 == 1
    ptc["flag"] = (ptc["flag"] | np.where(ph, 4, 0)).astype(np.uint32)
    ptc["flag"][::50] |= 2                                    # some removed: untouched
    ptc["w"] = np.random.default_rng(1).uniform(0.5, 2.0, n)
    gthr, eph, pc = 100.0, 4.0, 0.3
    out, ov = oracle.pair_production(p, ptc, 2 * n, gthr, eph, pc, seed=11, step=2)
    assert not ov
    m = len(out["x1"])
    a, M = p["a"], p["M"]
    N0 = _fido_norm(a, M, ptc["x1"], ptc["x2"], ptc["u1"], ptc["u2"], ptc["u3"])
    live = (ptc["flag"] & 2) == 0
    lep, pho = live & ~ph, live & ph
    emit = lep & (np.sqrt(1 + N0) >= gthr) & (np.sqrt(N0) > eph)
    assert 0 < emit.sum() < lep.sum()
    changed = np.flatnonzero((out["u1"][:n] != ptc["u1"]) | (out["flag"][:n] != ptc["flag"]))
    conv = np.zeros(n, bool); conv[changed] = True; conv &= pho
    assert np.array_equal(np.flatnonzero(emit | conv), changed)       # nobody else was touched
    assert m == n + len(changed)
    # conversion decision = the stated uniform numbers, and the fraction is p_convert
    U = np.array([oracle.uniform(11, 2, int(k)) for k in np.flatnonzero(pho)])
    assert np.array_equal(np.flatnonzero(pho)[(U < pc) & (0.5 * np.sqrt(N0[pho]) > 1.0)], np.flatnonzero(conv))
    assert abs(conv.sum() / pho.sum() - pc) < 4 * math.sqrt(pc * (1 - pc) / pho.sum())
    # children in parent order, inheriting position, cell, weight
    par = changed
    for k in ("x1", "x2", "x3", "w", "cell"):
        assert np.array_equal(out[k][n:], ptc[k][par]), k
    U0 = np.stack([ptc["u1"], ptc["u2"], ptc["u3"]], 1)
    Up = np.stack([out["u1"][:n], out["u2"][:n], out["u3"][:n]], 1)[par]
    Uc = np.stack([out["u1"][n:], out["u2"][n:], out["u3"][n:]], 1)
    Nc = _fido_norm(a, M, out["x1"][n:], out["x2"][n:], Uc[:, 0], Uc[:, 1], Uc[:, 2])
    Np = _fido_norm(a, M, ptc["x1"][par], ptc["x2"][par], Up[:, 0], Up[:, 1], Up[:, 2])
    e = emit[par]
    # emission: momentum conserved, photon energy eps_ph, flags
    assert np.allclose(Up[e] + Uc[e], U0[par][e], rtol=1e-13, atol=0)
    assert np.allclose(np.sqrt(Nc[e]), eph, rtol=1e-12)
    assert np.all(out["flag"][n:][e] == 4) and np.array_equal(out["flag"][:n][par][e], ptc["flag"][par][e])
    # conversion: electron in the photon's slot, positron appended, each Gamma = E/2, parallel to the photon
    c = ~e
    E = np.sqrt(N0[par][c])
    assert np.all(out["flag"][:n][par][c] == 0) and np.all(out["flag"][n:][c] == 1)
    assert np.allclose(np.sqrt(1 + Np[c]), 0.5 * E, rtol=1e-12) and np.allclose(np.sqrt(1 + Nc[c]), 0.5 * E, rtol=1e-12)
    assert np.array_equal(Up[c], Uc[c])
    cosang = np.sum(Up[c] * U0[par][c], 1) / (np.linalg.norm(Up[c], axis=1) * np.linalg.norm(U0[par][c], axis=1))
    assert np.allclose(cosang, 1.0, rtol=1e-12)
    # capacity overflow is reported and nothing is written past it
    out2, ov2 = oracle.pair_production(p, ptc, n + 5, gthr, eph, pc, seed=11, step=2)
    assert ov2 and len(out2["x1"]) == n + 5
    for k in out2:
        assert np.array_equal(out2[k][n:], out[k][n:n + 5]), k
    # P5: the events whose child found no room did not happen -- those parents are untouched (same
    # momentum, same species), so no charge or momentum disappears; the first five events are the
    # ones of the unbounded run
    kept, dropped = par[:5], par[5:]
    for k in ("u1", "u2", "u3", "flag"):
        assert np.array_equal(out2[k][:n][dropped], ptc[k][dropped]), k
        assert np.array_equal(out2[k][:n][kept], out[k][:n][kept]), k


# ------------------------------------------------------------------ Vay pusher in the FIDO frame
def _triad_up(m, Vhat):
    """orthonormal FIDO components -> contravariant V^i (inverse of the oracle's own map, written
    from the triad e_(1) = sqrt(g^rr)(d_r - g_rph/g_phph d_ph), e_(2) = d_th/sqrt(g_thth), e_(3) = d_ph/sqrt(g_phph))."""
    sgrr, sth, sph = math.sqrt(m["gu_rr"]), math.sqrt(m["g_thth"]), math.sqrt(m["g_phph"])
    k = m["g_rph"] / m["g_phph"]
    return np.array([sgrr * Vhat[0], Vhat[1] / sth, -sgrr * k * Vhat[0] + Vhat[2] / sph])


def _hat_of_cov(m, u):
    sgrr, sth, sph = math.sqrt(m["gu_rr"]), math.sqrt(m["g_thth"]), math.sqrt(m["g_phph"])
    return np.array([sgrr * (u[0] - m["g_rph"] / m["g_phph"] * u[2]), u[1] / sth, u[2] / sph])


def _cov_of_hat(m, uh):
    sgrr, sth, sph = math.sqrt(m["gu_rr"]), math.sqrt(m["g_thth"]), math.sqrt(m["g_phph"])
    return np.array([uh[0] / sgrr + uh[2] * m["g_rph"] / sph, sth * uh[1], sph * uh[2]])


def test_vay_holds_the_ExB_drift_exactly_and_boris_does_not():
    """Vay (2008): a particle moving with the E x B drift velocity feels no net force and must stay
    at that velocity for ANY time step; the Boris update only does to O(dt^2).  Fields and momentum
    are set up in the orthonormal FIDO frame at a point of the a = 0.9 Kerr metric."""
    a, M, r, th = 0.9, 1.0, 3.0, 1.0
    m = oracle.metric(a, M, r, th)
    assert abs(m["sqrtg"] * math.sqrt(m["gu_rr"]) / (math.sqrt(m["g_thth"]) * math.sqrt(m["g_phph"])) - 1.0) < 1e-13
    Ehat, Bhat = np.array([0.0, 0.6, 0.0]), np.array([0.0, 0.0, 1.0])
    vd = np.cross(Ehat, Bhat) / Bhat.dot(Bhat)                        # (0.6, 0, 0)
    G = 1.0 / math.sqrt(1.0 - vd.dot(vd))
    uh0 = G * vd
    D, B = _triad_up(m, Ehat), _triad_up(m, Bhat)
    u0 = _cov_of_hat(m, uh0)
    for dt in (0.01, 1.0, 30.0):
        u = u0.copy()
        for _ in range(50):
            u = oracle.vay(a, M, r, th, u, D, B, +1.0, dt)
        assert np.max(np.abs(_hat_of_cov(m, u) - uh0)) < 1e-12, dt
    ub = oracle.boris(a, M, r, th, u0, D, B, +1.0, 1.0)
    assert np.max(np.abs(_hat_of_cov(m, ub) - uh0)) > 1e-3            # Boris leaves the drift at large dt


def test_vay_pure_B_conserves_energy_and_matches_boris_to_second_order():
    a, M, r, th = 0.7, 1.0, 2.5, 0.8
    m = oracle.metric(a, M, r, th)
    rng = np.random.default_rng(3)
    u = rng.normal(size=3) * np.array([1.0, 2.0, 2.0])
    B = rng.normal(size=3)
    nrm = lambda w: (m["gu_rr"] * w[0] ** 2 + m["gu_thth"] * w[1] ** 2 + m["gu_phph"] * w[2] ** 2
                     + 2 * m["gu_rph"] * w[0] * w[2])
    v = u.copy()
    for _ in range(100):
        v = oracle.vay(a, M, r, th, v, np.zeros(3), B, -1.0, 0.3)
    assert abs(nrm(v) / nrm(u) - 1.0) < 1e-13                          # |u| exact in a pure magnetic field
    # with E != 0 the two pushers are both second order: their difference falls as dt^3 per step
    D = rng.normal(size=3) * 0.3
    d = []
    for dt in (0.04, 0.02, 0.01):
        d.append(np.max(np.abs(oracle.vay(a, M, r, th, u, D, B, 1.0, dt) - oracle.boris(a, M, r, th, u, D, B, 1.0, dt))))
    assert 6.0 < d[0] / d[1] < 10.0 and 6.0 < d[1] / d[2] < 10.0, d


def test_push_with_vay_option_uses_vay():
    import inputs
    p = inputs.grid_params(24, 20, 0.9)
    fields = inputs.analytic_fields(p, "wald")
    ptc = inputs.make_particles(p, 50, 3, "logical", ("loguniform", 0.1, 10.0))
    dt = inputs.courant_dt(p)
    with oracle.pusher(1):
        nv = oracle.push(p, fields, ptc, dt)
    nb = oracle.push(p, fields, ptc, dt)
    assert np.max(np.abs(nv["u1"] - nb["u1"])) > 0 and np.allclose(nv["u1"], nb["u1"], rtol=1e-3, atol=1e-6)
    # one particle by hand: gather -> vay -> geodesic
    k = 7
    D6 = oracle.gather(p, fields, ptc["x1"][k], ptc["x2"][k])
    sgn = 1.0 if ptc["flag"][k] & 1 else -1.0
    r, th = math.exp(ptc["x1"][k]), ptc["x2"][k]
    ub = oracle.vay(p["a"], p["M"], r, th, [ptc["u1"][k], ptc["u2"][k], ptc["u3"][k]], D6[:3], D6[3:], sgn, dt)
    yn = oracle.geodesic(p["a"], p["M"], 3, np.array([r, th, ptc["x3"][k], *ub]), dt)
    assert abs(math.log(yn[0]) - nv["x1"][k]) < 1e-15 and abs(yn[3] - nv["u1"][k]) < 1e-15


# ------------------------------------------------------------------ S4.5-S4.7: reflection, removal flag, new cell
def test_push_reflection_removal_and_cell_on_hand_built_particles():
    """PAPER.md:136 ('correct reflection'), :138 (removal at the radial boundaries).  With D = B = 0
    the Boris step is the identity, so orc_push = geodesic step (pinned above) + the post-processing
    under test.  Hand-built particles: one crosses theta = 0, one crosses theta = pi, one ends below
    xi_in, one at / beyond xi_out, one stays inside.  Expected: theta -> -theta (2 pi - theta) with
    u_theta flipped and x2dep the un-reflected angle; flag bit 1 and cell 0xFFFFFFFF exactly for the
    two leavers; cell = floor(theta / dtheta) * nr + floor((xi - xi_in) / dxi) for the others."""
    import inputs
    p = inputs.grid_params(32, 24, 0.9, r_out=20.0)
    a, M = p["a"], 1.0
    g = oracle.Grid(p)
    dxi, dth = inputs.spacing(p)
    fields = [np.zeros(g.shape) for _ in range(6)]
    dt = 0.02
    r_in, r_out = math.exp(p["xi_in"]), math.exp(p["xi_out"])
    rows = [  # r, theta, phi, u_r, u_theta, u_phi
        (5.0, 2e-3, 0.3, 0.0, -8.0, 0.0),             # crosses theta = 0 (u_theta < 0; no u_phi: no centrifugal wall)
        (6.0, math.pi - 2e-3, 1.0, 0.2, 9.0, 0.0),    # crosses theta = pi
        (r_in * 1.004, 1.1, 0.0, -30.0, 0.1, 0.2),    # falls below r_in
        (r_out * 0.9995, 2.0, 0.0, 40.0, 0.0, 0.1),   # leaves through r_out
        (7.0, 1.3, 2.0, 0.5, -0.7, 1.5),              # stays inside
    ]
    y = np.array(rows)
    y[:, 0] = np.exp(np.log(y[:, 0]))               # the state stores xi = ln r: start from r = exp(xi)
    ptc = {"x1": np.log(y[:, 0]), "x2": y[:, 1].copy(), "x3": y[:, 2].copy(), "u1": y[:, 3].copy(),
           "u2": y[:, 4].copy(), "u3": y[:, 5].copy(), "flag": np.array([0, 1, 0, 1, 0], dtype=np.uint32)}
    out = oracle.push(p, fields, ptc, dt)
    geo = np.array([oracle.geodesic(a, M, 3, yy, dt) for yy in y])
    th_new = geo[:, 1]
    assert th_new[0] < 0 and th_new[1] > math.pi                   # the cases are what they claim to be
    assert math.log(geo[2, 0]) < p["xi_in"] and math.log(geo[3, 0]) >= p["xi_out"]
    # un-reflected angle for the deposit, mirrored angle and flipped u_theta in the state
    assert np.array_equal(out["x2dep"], th_new)
    assert out["x2"][0] == -th_new[0] and out["u2"][0] == -geo[0, 4]
    assert out["x2"][1] == 2 * math.pi - th_new[1] and out["u2"][1] == -geo[1, 4]
    for k in (2, 3, 4):
        assert out["x2"][k] == th_new[k] and out["u2"][k] == geo[k, 4]
    assert np.all((out["x2"] >= 0) & (out["x2"] <= math.pi))
    assert np.array_equal(out["x1"], np.log(geo[:, 0])) and np.array_equal(out["x3"], geo[:, 2])
    assert np.array_equal(out["u1"], geo[:, 3]) and np.array_equal(out["u3"], geo[:, 5])
    # removal flag (bit 1) and cell
    assert list(out["flag"]) == [0, 1, 0 | 2, 1 | 2, 0]
    assert out["cell"][2] == 0xFFFFFFFF and out["cell"][3] == 0xFFFFFFFF
    for k in (0, 1, 4):
        ic = int(math.floor((out["x1"][k] - p["xi_in"]) / dxi))
        jc = int(math.floor(out["x2"][k] / dth))
        assert 0 <= ic < p["nr"] and 0 <= jc < p["nth"]
        assert out["cell"][k] == jc * p["nr"] + ic
    assert out["cell"][0] // p["nr"] == 0 and out["cell"][1] // p["nr"] == p["nth"] - 1   # rows next to the axes
    # a particle already flagged removed is passed through untouched
    ptc2 = {k: v.copy() for k, v in ptc.items()}
    ptc2["flag"][4] |= 2
    out2 = oracle.push(p, fields, ptc2, dt)
    for k in ("x1", "x2", "x3", "u1", "u2", "u3"):
        assert out2[k][4] == ptc[k][4]
    assert out2["flag"][4] == 2 and out2["cell"][4] == 0xFFFFFFFF


# ------------------------------------------------------------------ Boyer-Lindquist / FIDO diagnostics ((A6), (A7))
def test_ks_to_bl_diagnostics():
    """orc_ks_to_bl: (1) the transformed four-momentum (u_t, u_r^BL, u_theta, u_phi) is normalised with
    the TEXTBOOK Boyer-Lindquist inverse metric, g^{mu nu} u_mu u_nu = -eps, for massive particles and
    photons, inside and outside the ergosphere; (2) (A7) differentiates to (A6): d(phi_KS - phi_BL)/dr =
    a / Delta; (3) a particle at rest in the FIDO frame has Gamma = 1; (4) E_inf is the quantity the
    geodesic integrator conserves (same number along an orbit to the integrator's accuracy)."""
    rng = np.random.default_rng(9)
    for a in (0.0, 0.5, 0.998):
        rh = 1.0 + math.sqrt(1.0 - a * a)
        for _ in range(40):
            r, th = rng.uniform(1.05 * rh, 20.0), rng.uniform(0.2, math.pi - 0.2)
            u = rng.normal(size=3) * rng.choice([0.1, 3.0, 50.0])
            for eps in (1.0, 0.0):
                E, Gam, urb, phb = oracle.ks_to_bl(a, 1.0, math.log(r), th, 0.7, u, eps)
                s2, rho2, Delta = math.sin(th) ** 2, r * r + a * a * math.cos(th) ** 2, r * r - 2 * r + a * a
                gtt = -((r * r + a * a) ** 2 - a * a * Delta * s2) / (rho2 * Delta)
                gtp = -2.0 * a * r / (rho2 * Delta)
                grr, gthth = Delta / rho2, 1.0 / rho2
                gpp = (Delta - a * a * s2) / (rho2 * Delta * s2)
                ut = -E
                norm = gtt * ut * ut + 2 * gtp * ut * u[2] + grr * urb * urb + gthth * u[1] ** 2 + gpp * u[2] ** 2
                scale = abs(gtt * ut * ut) + grr * urb * urb + gthth * u[1] ** 2 + abs(gpp) * u[2] ** 2 + 1.0
                assert abs(norm + eps) <= 1e-12 * scale, (a, r, th, eps, norm)
                assert Gam >= 1.0 - 1e-15 if eps == 1.0 else Gam > 0.0
        if a > 0:
            r, h = 3.7, 1e-5
            d = lambda rr: 0.7 - oracle.ks_to_bl(a, 1.0, math.log(rr), 1.0, 0.7, np.zeros(3))[3]   # phi_KS - phi_BL
            Delta = r * r - 2 * r + a * a
            assert abs((d(r + h) - d(r - h)) / (2 * h) - a / Delta) < 1e-8
        assert abs(oracle.ks_to_bl(a, 1.0, math.log(4.0), 1.1, 0.0, np.zeros(3))[1] - 1.0) < 1e-15
    # (4) along a Table-1-like bound orbit
    a = 0.9
    y0 = np.array([6.0, math.pi / 2, 0.0, 0.05, 0.3, 3.2])
    traj = oracle.geodesic_traj(a, 1.0, 3, y0, 1e-2, 4000, every=400)
    Es = [oracle.ks_to_bl(a, 1.0, math.log(y[0]), y[1], y[2], y[3:6])[0] for y in traj]
    assert max(Es) - min(Es) < 1e-6 * abs(Es[0])
