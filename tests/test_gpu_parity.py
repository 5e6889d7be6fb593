"""Parity of the CUDA path (through the C ABI of libgrpic.so) against the CPU oracle on the
same seeded inputs.  Tolerances are BASELINE.json's: integer outputs bit-exact; x,u <= 1e-12
relative after one step; J and fields <= 1e-11 relative; continuity residual <= 1e-13 max|rho|."""
import math
import os

import numpy as np
import pytest

import inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def G():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2503_04558_b200 import grpic
    return grpic


@pytest.fixture(scope="module")
def O():
    import oracle
    return oracle


# ------------------------------------------------------------------ helpers
def ptc_err(ref, got, keys):
    """G20 norm: per particle max_k |d_k| / max(1, max_k |ref_k|)."""
    d = np.max(np.abs(np.stack([got[k] - ref[k] for k in keys])), axis=0)
    s = np.maximum(1.0, np.max(np.abs(np.stack([ref[k] for k in keys])), axis=0))
    return d / s


def edge_ambiguous(p, ref, ulps=8):
    """particles whose oracle xi' / theta' lies within a few ulp of a cell or boundary edge:
    CUDA and glibc log/sincos may differ by an ulp there (reported, expected empty)."""
    dxi, dth = inputs.spacing(p)
    fx = (ref["x1"] - p["xi_in"]) / dxi
    fy = ref["x2"] / dth
    tol = ulps * np.finfo(np.float64).eps
    ax = np.abs(fx - np.round(fx)) <= tol * np.maximum(1.0, np.abs(fx)) * p["nr"]
    ay = np.abs(fy - np.round(fy)) <= tol * np.maximum(1.0, np.abs(fy)) * p["nth"]
    return ax | ay


def grid_err(ref, got):
    return np.max(np.abs(got - ref)) / max(np.max(np.abs(ref)), 1e-300)


def gpu_push_deposit(G, p, fields, ptc, dt, ctx=None):
    ctx = ctx or G.Context(p, len(ptc["x1"]))
    f_t = [ctx.to_device(f) for f in fields]
    P = G.Particles.from_numpy(ptc)
    F_t = ctx.zeros(3)
    ctx.status.zero_()
    ctx.push_deposit(P, f_t, F_t, dt)
    torch.cuda.synchronize()
    return ctx, P, F_t


def oracle_push_deposit(O, p, fields, ptc, dt):
    new = O.push(p, fields, ptc, dt)
    F = O.deposit(p, ptc, new, ptc["w"], dt)
    return new, F


AXIS_BAND = 1e-3      # sin(theta) below which the comparison uses the conditioning rule
PARITY_LOG = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out", "parity_stats.jsonl")


def check_push(p, ptc, ref, got, O=None, fields=None, dt=None, tol=1e-12, max_over=0, label=""):
    """DESIGN.md section 7 "comparison rule for x, u".  G20 norm per particle.
    * Every particle with sin(theta) >= AXIS_BAND before and after the step: x, u <= 1e-12, no exception.
    * Inside the band the geodesic force ~ u_phi^2 cos/sin^3 amplifies one ulp of the input by up to
      1/sin^3: there the bound is max(1e-12, 10 x the oracle's OWN response to a 4-ulp change of the
      input position), and at most `max_over` particles of the case may exceed 1e-12 at all (set per
      call site to <= 2x the count measured on B200, printed and logged to gpurun_out/parity_stats.jsonl:
      0 everywhere except BASELINE config 1, whose 1e5 particles are uniform in theta down to 1e-9).
    * cell / flag bit-exact outside the edge-ambiguous set (G20)."""
    import json
    amb = edge_ambiguous(p, ref)
    ex = ptc_err(ref, got, ("x1", "x2", "x3"))
    eu = ptc_err(ref, got, ("u1", "u2", "u3"))
    err = np.maximum(ex, eu)
    near_axis = (np.sin(ptc["x2"]) < AXIS_BAND) | (np.sin(np.clip(ref["x2"], 0.0, math.pi)) < AXIS_BAND)
    tolk = np.full(len(err), tol)
    sens = np.zeros(len(err))
    if O is not None and near_axis.any():
        eps = 4 * np.finfo(np.float64).eps
        pert = dict(ptc)
        pert["x1"] = ptc["x1"] * (1.0 + eps)
        pert["x2"] = ptc["x2"] * (1.0 + eps)
        refp = O.push(p, fields, pert, dt)
        sens = np.maximum(ptc_err(ref, refp, ("x1", "x2", "x3")), ptc_err(ref, refp, ("u1", "u2", "u3")))
        tolk = np.where(near_axis, np.maximum(tol, 10.0 * sens), tol)
    over = err > tol
    stats = {"case": label or os.environ.get("PYTEST_CURRENT_TEST", "").split(" ")[0], "n": int(len(err)),
             "n_near_axis": int(near_axis.sum()), "n_over_1e-12": int(over.sum()),
             "worst_err": float(err.max()) if len(err) else 0.0,
             "worst_err_outside_band": float(err[~near_axis].max()) if (~near_axis).any() else 0.0,
             "worst_err_over_sens": float((err[over] / np.maximum(sens[over], 1e-300)).max()) if over.any() else 0.0,
             "max_sin_theta_of_over": float(np.sin(ptc["x2"][over]).max()) if over.any() else 0.0,
             "edge_ambiguous": int(amb.sum())}
    print("parity", json.dumps(stats))
    try:
        os.makedirs(os.path.dirname(PARITY_LOG), exist_ok=True)
        with open(PARITY_LOG, "a") as fh:
            fh.write(json.dumps(stats) + "\n")
    except OSError:
        pass
    assert not (over & ~near_axis).any(), ("outside the axis band", stats)
    assert int(over.sum()) <= max_over, stats
    assert np.all(err <= tolk), stats
    ok = ~amb
    assert np.array_equal(ref["cell"][ok], got["cell"][ok])
    assert np.array_equal(ref["flag"][ok], got["flag"][ok])
    return int(amb.sum())


def small_case(k, nr, nth, n):
    return inputs.config(k, nr=nr, nth=nth, n=n)


# ------------------------------------------------------------------ tests
def test_areas_match_oracle(G, O):
    p = inputs.grid_params(40, 36, 0.95, r_out=30.0)
    ctx = G.Context(p)
    A = [ctx.to_host(t) for t in ctx.get_areas()]
    ref = O.areas(p)
    for a, name in zip(A, ("ADr", "ADth", "ADph", "ABr", "ABth", "ABph")):
        assert np.allclose(a, ref[name], rtol=1e-12, atol=1e-13 * np.max(ref[name])), name


@pytest.mark.parametrize("k,nr,nth,n", [(1, 64, 48, 20011), (2, 96, 64, 30000), (3, 80, 72, 25013)])
def test_push_deposit_one_step(G, O, k, nr, nth, n):
    cfg = small_case(k, nr, nth, n)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    ref, Fref = oracle_push_deposit(O, p, fields, ptc, dt)
    ctx, P, F_t = gpu_push_deposit(G, p, fields, ptc, dt)
    got = P.to_numpy()
    namb = check_push(p, ptc, ref, got, O, fields, dt)
    assert namb <= 2
    assert np.array_equal(got["w"], ptc["w"])
    for c in range(3):
        assert grid_err(Fref[c], ctx.to_host(F_t[c])) <= 1e-11, c
    assert int(ctx.status.item()) & ~1 == 0
    # some particles do leave / cross the axis in these cases (otherwise the test is vacuous)
    if k == 3:
        assert (ref["flag"] & 2).sum() > 0


def test_axis_crossers_and_leavers(G, O):
    """particles placed within a fraction of a cell of the axis and of both radial
    boundaries, moving outwards: reflection, removal flags, ghost/guard deposits."""
    p = inputs.grid_params(48, 40, 0.9, r_out=25.0)
    dt = inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "monopole")
    ptc = inputs.make_particles(p, 4000, 11, "logical", ("loguniform", 1.0, 50.0))
    dxi, dth = inputs.spacing(p)
    n = len(ptc["x1"])
    rng = np.random.default_rng(5)
    q = n // 4
    for lo, sgn in ((0, -1.0), (q, +1.0)):      # fast, nearly polar motion close to the hole
        sl = slice(lo, lo + q)
        ptc["x1"][sl] = p["xi_in"] + rng.uniform(0.5, 12.0, q) * dxi
        off = rng.uniform(1e-3, 0.08, q) * dth
        ptc["x2"][sl] = off if sgn < 0 else np.pi - off
        ptc["u1"][sl] = rng.normal(size=q)
        ptc["u2"][sl] = sgn * rng.uniform(30.0, 300.0, q)
        ptc["u3"][sl] = rng.normal(size=q) * 1e-3
    ptc["x1"][2 * q:3 * q] = p["xi_in"] + rng.uniform(1e-3, 0.2, q) * dxi
    ptc["u1"][2 * q:3 * q] = -np.abs(ptc["u1"][2 * q:3 * q]) - 3.0
    ptc["x1"][3 * q:] = p["xi_out"] - rng.uniform(1e-3, 0.2, n - 3 * q) * dxi
    ptc["u1"][3 * q:] = np.abs(ptc["u1"][3 * q:]) + 30.0
    ptc["cell"] = inputs.cells_of(p, ptc["x1"], ptc["x2"])
    ref, Fref = oracle_push_deposit(O, p, fields, ptc, dt)
    assert (ref["x2dep"] < 0).sum() > 50 and (ref["x2dep"] > np.pi).sum() > 50
    assert (ref["flag"] & 2).sum() > 100
    ctx, P, F_t = gpu_push_deposit(G, p, fields, ptc, dt)
    check_push(p, ptc, ref, P.to_numpy(), O, fields, dt)
    for c in range(3):
        assert grid_err(Fref[c], ctx.to_host(F_t[c])) <= 1e-11, c
    # a second step must leave the removed particles untouched and deposit nothing for them
    ptc2 = {k: ref[k] for k in ("x1", "x2", "x3", "u1", "u2", "u3", "cell", "flag")}
    ptc2["w"] = ptc["w"]
    ref2, Fref2 = oracle_push_deposit(O, p, fields, ptc2, dt)
    ctx2, P2, F2 = gpu_push_deposit(G, p, fields, ptc2, dt, ctx)
    got2 = P2.to_numpy()
    rem = (ptc2["flag"] & 2) != 0
    for key in ("x1", "x2", "x3", "u1", "u2", "u3"):
        assert np.array_equal(got2[key][rem], ptc2[key][rem])
    for c in range(3):
        assert grid_err(Fref2[c], ctx.to_host(F2[c])) <= 1e-11, c


@pytest.mark.parametrize("n,frac", [(0, 0.0), (31, 0.3), (5000, 0.0), (70001, 0.25), (4096, 1.0)])
def test_push_deposit_compact_equals_compact_then_push(G, O, n, frac):
    """grpic_push_deposit_compact == oracle compact -> oracle push+deposit: survivor order and
    count bit-exact, x,u <= 1e-12, fluxes <= 1e-11, tail marked removed, input untouched."""
    p = inputs.grid_params(64, 48, 0.99)
    dt = inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "wald")
    ptc = inputs.make_particles(p, max(n, 1), 21, "crowded", ("loguniform", 0.1, 1e3))
    ptc = {k: v[:n].copy() for k, v in ptc.items()}
    rng = np.random.default_rng(n + 1)
    dead = rng.uniform(size=n) < frac
    ptc["flag"] = (ptc["flag"] | np.where(dead, 2, 0)).astype(np.uint32)
    keep = O.compact(ptc["flag"]) if n else np.zeros(0, np.int64)
    assert len(keep) == int((~dead).sum())
    sub = {k: np.ascontiguousarray(v[keep]) for k, v in ptc.items()}
    ctx = G.Context(p, max(n, 1))
    f_t = [ctx.to_device(f) for f in fields]
    src, dst = G.Particles.from_numpy(ptc), G.Particles(n)
    for t in dst.t.values():
        t.fill_(7)
    F_t = ctx.zeros(3)
    n_alive = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    ctx.push_deposit_compact(src, dst, f_t, F_t, dt, n_alive)
    torch.cuda.synchronize()
    m = int(n_alive.item())
    assert m == len(keep)
    back = src.to_numpy()
    for k in ptc:
        assert np.array_equal(back[k], ptc[k]), k            # input not modified
    got = dst.to_numpy()
    if n:
        assert np.all(got["flag"][m:] & 2) and np.all(got["cell"][m:] == 0xFFFFFFFF)
    if m == 0:
        assert all(float(F.abs().max()) == 0.0 for F in F_t)
        return
    ref, Fref = oracle_push_deposit(O, p, fields, sub, dt)
    head = {k: v[:m] for k, v in got.items()}
    check_push(p, sub, ref, head, O, fields, dt)
    assert np.array_equal(head["w"], sub["w"])
    for c in range(3):
        assert grid_err(Fref[c], ctx.to_host(F_t[c])) <= 1e-11, c


@pytest.mark.parametrize("n,chunk", [(9000, 2048), (3000, 0), (0, 64)])
def test_step_host_matches_oracle_step(G, O, n, chunk):
    """grpic_step_host (host buffers, chunked + overlapped copies) == oracle compact -> push ->
    deposit -> finalize -> field step."""
    p = inputs.grid_params(48, 40, 0.99, field_iters=3)
    dt = inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "wald")
    ptc = inputs.make_particles(p, max(n, 1), 33, "r2", ("loguniform", 0.1, 1e2))
    ptc = {k: v[:n].copy() for k, v in ptc.items()}
    rng = np.random.default_rng(7)
    ptc["flag"] = (ptc["flag"] | np.where(rng.uniform(size=n) < 0.1, 2, 0)).astype(np.uint32)
    ptc["w"] = rng.uniform(0.5, 1.5, n) * 1e-3
    keep = O.compact(ptc["flag"]) if n else np.zeros(0, np.int64)
    sub = {k: np.ascontiguousarray(v[keep]) for k, v in ptc.items()}
    ctx = G.Context(p, max(n, 1))
    f_t = [ctx.to_device(f) for f in fields]
    host = {k: torch.from_numpy(v.copy() if v.dtype != np.uint32 else v.view(np.int32).copy()).pin_memory()
            for k, v in ptc.items()}
    host["n"] = n
    hJ = [torch.zeros((ctx.rows, ctx.pitch), dtype=torch.float64).pin_memory() for _ in range(3)]
    m = ctx.step_host(host, f_t, dt, host_J=hJ, chunk=chunk)
    assert m == len(keep) and host["n"] == m
    if m:
        ref, Fref = oracle_push_deposit(O, p, fields, sub, dt)
        got = {k: host[k][:m].numpy() for k in ("x1", "x2", "x3", "u1", "u2", "u3", "w")}
        got.update({k: host[k][:m].numpy().view(np.uint32) for k in ("cell", "flag")})
        check_push(p, sub, ref, got, O, fields, dt)
        assert np.array_equal(got["w"], sub["w"])
    else:
        Fref = [np.zeros_like(fields[0]) for _ in range(3)]
    Jref = O.finalize_current(p, Fref, 0)
    fref = O.field_step(p, [f.copy() for f in fields], Jref, dt)
    for c in range(3):
        assert grid_err(Jref[c], ctx.to_host(hJ[c].cuda())) <= 1e-11 or np.max(np.abs(Jref[c])) == 0.0, c
    for c in range(6):
        assert grid_err(fref[c], ctx.to_host(f_t[c])) <= 1e-11, c


def test_photon_species_parity(G, O):
    """mixed e-/e+/photon input (flag bit2 = photon): photons follow null
    geodesics, ignore the fields and deposit nothing; same tolerances as the charged species."""
    p = inputs.grid_params(64, 48, 0.99)
    dt = inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "wald")
    ptc = inputs.make_particles(p, 30000, 17, "crowded", ("loguniform", 0.1, 1e3))
    ph = (np.arange(30000) % 3) == 0
    ptc["flag"] = (ptc["flag"] | np.where(ph, 4, 0)).astype(np.uint32)
    ref, Fref = oracle_push_deposit(O, p, fields, ptc, dt)
    ctx, P, F_t = gpu_push_deposit(G, p, fields, ptc, dt)
    got = P.to_numpy()
    check_push(p, ptc, ref, got, O, fields, dt)
    assert np.array_equal(got["flag"] & 4, ptc["flag"] & 4)
    for c in range(3):
        assert grid_err(Fref[c], ctx.to_host(F_t[c])) <= 1e-11, c
    rho = ctx.zeros()
    ctx.deposit_rho(P, rho)
    alive = dict(ref); alive["w"] = ptc["w"]
    assert grid_err(O.rho(p, alive, ptc["w"]), ctx.to_host(rho)) <= 1e-11


@pytest.mark.parametrize("n,cap,step", [(20000, 40000, 3), (777, 800, 0), (0, 16, 1), (300007, 450000, 2), (300007, 330000, 5)])
def test_pair_production_parity(G, O, n, cap, step):
    """grpic_pair_production vs the oracle (Eq.26): who emits / converts, the
    new particle count and the append ORDER bit-exact (same Philox numbers on both sides),
    momenta <= 1e-12; capacity overflow reported."""
    p = inputs.grid_params(64, 48, 0.99)
    ptc = inputs.make_particles(p, max(n, 1), 29, "crowded", ("loguniform", 1.0, 1e4))
    ptc = {k: v[:n].copy() for k, v in ptc.items()}
    ph = np.arange(n) % 2 == 1
    ptc["flag"] = (ptc["flag"] | np.where(ph, 4, 0)).astype(np.uint32)
    ptc["flag"][::37] |= 2
    ptc["w"] = np.random.default_rng(2).uniform(0.5, 2.0, n)
    gthr, eph, pc, seed = 100.0, 4.0, 0.35, 0x1234567890ABCDEF
    ref, ov = O.pair_production(p, ptc, cap, gthr, eph, pc, seed, step)
    ctx = G.Context(p, cap)
    P = G.Particles(cap)
    for t in P.t.values():
        t.zero_()
    for k in ptc:
        src = ptc[k] if ptc[k].dtype != np.uint32 else ptc[k].view(np.int32)
        P.t[k][:n].copy_(torch.from_numpy(src))
    n_new = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    ctx.status.zero_()
    ctx.pair_production(P, n, n_new, gthr, eph, pc, seed, step)
    torch.cuda.synchronize()
    m = int(n_new.item())
    assert m == len(ref["x1"])
    assert bool(int(ctx.status.item()) & 8) == ov
    if n:
        assert m > n                                       # something was created
    got = P.to_numpy(m)
    for k in ("x1", "x2", "x3", "w", "cell", "flag"):
        assert np.array_equal(got[k], ref[k]), k
    for k in ("u1", "u2", "u3"):
        err = np.abs(got[k] - ref[k]) / np.maximum(1.0, np.abs(ref[k]))
        assert err.max(initial=0.0) <= 1e-12, (k, err.max())


def test_far_moves_take_the_general_window(G, O):
    """dt three times the Courant-limited step: fast particles move more than one cell, leave the
    3x3 window and must take the exact general-window deposit (GRPIC_STATUS_FAR_MOVE is set);
    fluxes still match the oracle, which deposits on whatever window the move spans."""
    p = inputs.grid_params(64, 64, 0.9, r_out=30.0)
    dt = 6.0 * inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "monopole")
    ptc = inputs.make_particles(p, 20000, 13, "logical", ("loguniform", 5.0, 100.0))
    dxi, dth = inputs.spacing(p)
    inner = (ptc["x1"] > p["xi_in"] + 8 * dxi) & (ptc["x1"] < p["xi_out"] - 8 * dxi) & \
            (ptc["x2"] > 8 * dth) & (ptc["x2"] < np.pi - 8 * dth)
    ptc = {k: np.ascontiguousarray(v[inner]) for k, v in ptc.items()}
    ref, Fref = oracle_push_deposit(O, p, fields, ptc, dt)
    far = (np.abs(np.floor((ref["x1"] - p["xi_in"]) / dxi) - np.floor((ptc["x1"] - p["xi_in"]) / dxi)) > 1) | \
          (np.abs(np.floor(ref["x2dep"] / dth) - np.floor(ptc["x2"] / dth)) > 1)
    assert far.sum() > 100
    ctx, P, F_t = gpu_push_deposit(G, p, fields, ptc, dt)
    st = int(ctx.status.item())
    assert st & 1 and not (st & ~1)
    check_push(p, ptc, ref, P.to_numpy(), O, fields, dt)
    for c in range(3):
        assert grid_err(Fref[c], ctx.to_host(F_t[c])) <= 1e-11, c


@pytest.mark.parametrize("nr,nth,n", [(48, 40, 20000), (320, 256, 300007)])
def test_spline3_push_deposit_parity(G, O, nr, nth, n):
    """third-order (cubic B-spline) shape option: gather, push and deposit vs the
    oracle run with the same option; includes axis crossers, leavers and photons.  The second size
    spans many CTAs and a ragged tail."""
    p = inputs.grid_params(nr, nth, 0.99, ng=3)
    dt = inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "wald")
    ptc = inputs.make_particles(p, n, 23, "crowded", ("loguniform", 0.1, 1e3))
    ptc["flag"] = (ptc["flag"] | np.where(np.arange(n) % 7 == 0, 4, 0)).astype(np.uint32)
    with O.shape_order(3):
        ref, Fref = oracle_push_deposit(O, p, fields, ptc, dt)
    ref1, Fref1 = oracle_push_deposit(O, p, fields, ptc, dt)
    assert np.max(np.abs(Fref[0] - Fref1[0])) > 1e-3 * np.max(np.abs(Fref1[0]))     # the option matters
    ctx = G.Context(p, len(ptc["x1"]))
    f_t = [ctx.to_device(f) for f in fields]
    P = G.Particles.from_numpy(ptc)
    F_t = ctx.zeros(3)
    ctx.status.zero_()
    ctx.push_deposit_spline3(P, f_t, F_t, dt)
    torch.cuda.synchronize()
    assert int(ctx.status.item()) == 0
    with O.shape_order(3):
        check_push(p, ptc, ref, P.to_numpy(), O, fields, dt)
    for c in range(3):
        assert grid_err(Fref[c], ctx.to_host(F_t[c])) <= 1e-11, c
    ctx2 = G.Context(inputs.grid_params(48, 40, 0.99), 16)                         # ng = 2: refused
    with pytest.raises(G.GrpicError):
        ctx2.push_deposit_spline3(G.Particles.from_numpy({k: v[:16].copy() for k, v in ptc.items()}),
                                  [ctx2.to_device(f) for f in inputs.analytic_fields(inputs.grid_params(48, 40, 0.99), "wald")],
                                  ctx2.zeros(3), dt)


def test_gpu_geodesic_orbit_invariants(G, O):
    """Physics on the GPU path itself (Table 1 orbit (3,3,2), a = 0.995, zero
    fields): u_phi is conserved bit for bit (U_phi = 0) and the error of the energy at infinity
    E = alpha^2 u^0 - beta^r u_r falls as dt^2 over 120 r_g/c of the zoom-whirl orbit."""
    vals = None
    here = os.path.dirname(os.path.abspath(__file__))
    for line in open(os.path.join(here, "golden", "table1_orbits.txt")):
        if line.startswith("(3,3,2)"):
            vals = [float(v) for v in line.split()[1:]]
    a, _, ur, uth, uph, r0, off = vals
    p = inputs.grid_params(32, 32, a, r_out=20.0)
    zero = [np.zeros(inputs.grid_shape(p)) for _ in range(6)]
    ctx = G.Context(p, 4)
    f_t = [ctx.to_device(f) for f in zero]

    def E_of(x1, x2, u1, u2, u3):
        m = O.metric(a, 1.0, math.exp(x1), x2)
        nrm = m["gu_rr"] * u1 ** 2 + m["gu_thth"] * u2 ** 2 + m["gu_phph"] * u3 ** 2 + 2 * m["gu_rph"] * u1 * u3
        return m["alpha"] * math.sqrt(1.0 + nrm) - m["beta_r"] * u1

    errs = []
    for dt in (0.1, 0.05, 0.025):
        one = dict(x1=np.array([math.log(r0)]), x2=np.array([math.pi / 2 - off]), x3=np.zeros(1),
                   u1=np.array([ur]), u2=np.array([uth]), u3=np.array([uph]), w=np.zeros(1),
                   flag=np.zeros(1, np.uint32))
        one["cell"] = inputs.cells_of(p, one["x1"], one["x2"])
        P = G.Particles.from_numpy(one)
        F_t = ctx.zeros(3)
        E0 = E_of(one["x1"][0], one["x2"][0], ur, uth, uph)
        dE, n = [], int(round(120.0 / dt))
        for s in range(n):
            ctx.push_deposit(P, f_t, F_t, dt)
            if s % max(1, n // 300) == 0:
                q = P.to_numpy()
                assert q["u3"][0] == uph and not (q["flag"][0] & 2)
                dE.append(abs(E_of(q["x1"][0], q["x2"][0], q["u1"][0], q["u2"][0], q["u3"][0]) - E0))
        errs.append(float(np.mean(dE)))
    assert errs[2] < 2e-4 * abs(E0)
    assert 3.3 < errs[0] / errs[1] < 4.7 and 3.3 < errs[1] / errs[2] < 4.7, errs


def test_gpu_field_step_preserves_divB(G, O):
    """Invariant on the GPU path itself: the discrete div B (fluxes B^r A^B_r,
    B^th A^B_th through the faces of every cell, areas from the library) does not change in a
    field step, over 5 steps of random fields with the damping layer off, on a grid that spans
    several CTA chunks and the TMA interior path."""
    p = inputs.grid_params(200, 150, 0.95)
    ctx = G.Context(p, 16)
    rng = np.random.default_rng(4)
    shape = inputs.grid_shape(p)
    f = [rng.normal(size=shape) for _ in range(6)]
    f_t = [ctx.to_device(x) for x in f]
    ctx.fill_guards(f_t)
    A = [ctx.to_host(a) for a in ctx.get_areas()]
    Gd, nr, nth = p["ng"], p["nr"], p["nth"]

    def div(ft):
        Br, Bth = ctx.to_host(ft[3]) * A[3], ctx.to_host(ft[4]) * A[4]
        return (Br[Gd:Gd + nth, Gd + 1:Gd + nr + 1] - Br[Gd:Gd + nth, Gd:Gd + nr]) + \
               (Bth[Gd + 1:Gd + nth + 1, Gd:Gd + nr] - Bth[Gd:Gd + nth, Gd:Gd + nr])

    d0 = div(f_t)
    sc = np.max(np.abs(ctx.to_host(f_t[3]) * A[3]))
    dt = inputs.courant_dt(p)
    for _ in range(5):
        ctx.field_step(f_t, None, dt)
    torch.cuda.synchronize()
    d1 = div(f_t)
    assert np.max(np.abs(ctx.to_host(f_t[3]) - f[3][:, :])) > 1e-6        # the fields did change
    assert np.max(np.abs(d1 - d0)) < 1e-12 * sc, np.max(np.abs(d1 - d0)) / sc


def test_gpu_coupled_loop_preserves_gauss_law(G, O):
    """Invariant of the coupled GPU path: with the charge-conserving deposit
    feeding the field step, div D - rho does not drift.  100 coupled steps (fused push+deposit+
    removal, finalize, field step) of 20000 particles on a 64 x 64 grid; the change of
    [div(D A) - rho dV] on interior nodes (incl. the axis nodes, Eq.11) stays at round-off of the
    accumulated charge motion."""
    p = inputs.grid_params(64, 64, 0.9, r_out=30.0)
    dt = inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "monopole")
    ptc = inputs.make_particles(p, 20000, 31, "logical", ("loguniform", 0.1, 5.0))
    ptc["w"][:] = 1e-3
    n = len(ptc["x1"])
    ctx = G.Context(p, n)
    f_t = [ctx.to_device(f) for f in fields]
    ctx.fill_guards(f_t)
    A = [ctx.to_host(a) for a in ctx.get_areas()]
    Gd, nr, nth = p["ng"], p["nr"], p["nth"]

    def gauss(ft, P):
        Dr, Dth = ctx.to_host(ft[0]) * A[0], ctx.to_host(ft[1]) * A[1]
        d = np.zeros_like(Dr)
        d[:, 1:] += Dr[:, 1:] - Dr[:, :-1]
        d[Gd + 1:Gd + nth, :] += Dth[Gd + 1:Gd + nth, :] - Dth[Gd:Gd + nth - 1, :]
        d[Gd, :] += Dth[Gd, :]
        d[Gd + nth, :] += -Dth[Gd + nth - 1, :]
        rho = ctx.zeros()
        ctx.deposit_rho(P, rho, divide=False)
        return d - ctx.to_host(rho), ctx.to_host(rho)

    cur, alt = G.Particles.from_numpy(ptc), G.Particles(n)
    n_alive = torch.zeros(1, dtype=torch.int64, device="cuda")
    g0, rho0 = gauss(f_t, cur)
    moved = 0.0
    for step in range(100):
        F_t = ctx.zeros(3)
        ctx.push_deposit_compact(cur, alt, f_t, F_t, dt, n_alive)
        cur, alt = alt, cur
        if step == 0:
            moved = max(float(F.abs().max()) for F in F_t) * dt
        ctx.finalize_current(F_t, 0)
        ctx.field_step(f_t, F_t, dt)
    torch.cuda.synchronize()
    assert int(ctx.status.item()) == 0
    g1, rho1 = gauss(f_t, cur)
    # interior nodes only: nodes next to the radial edges exchange charge with the guards (leavers)
    sel = (slice(Gd, Gd + nth + 1), slice(Gd + 2, Gd + nr - 1))
    sc = np.max(np.abs(rho0))
    assert moved > 0 and np.max(np.abs(rho1 - rho0)[sel]) > 1e-2 * sc          # charge really moved
    assert np.max(np.abs((g1 - g0)[sel])) < 1e-11 * sc, np.max(np.abs((g1 - g0)[sel])) / sc


@pytest.mark.parametrize("order,pusher,nr,nth,n", [(1, 0, 48, 40, 20000), (1, 1, 48, 40, 20000), (3, 1, 48, 40, 20000),
                                                   (1, 1, 320, 256, 300007), (3, 1, 320, 256, 300007)])
def test_push_deposit_variants_parity(G, O, order, pusher, nr, nth, n):
    """grpic_push_deposit_variant vs the oracle with the same options: shape order 1 / 3
     and pusher Boris / Vay in the FIDO frame.  (1, 0) must also
    agree with the tuned default kernel's result through the oracle.  The larger size spans many
    CTAs and a ragged tail."""
    p = inputs.grid_params(nr, nth, 0.99, ng=3)
    dt = inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "wald")
    ptc = inputs.make_particles(p, n, 41, "crowded", ("loguniform", 0.1, 1e3))
    with O.shape_order(order), O.pusher(pusher):
        ref, Fref = oracle_push_deposit(O, p, fields, ptc, dt)
    ctx = G.Context(p, len(ptc["x1"]))
    f_t = [ctx.to_device(f) for f in fields]
    P = G.Particles.from_numpy(ptc)
    F_t = ctx.zeros(3)
    ctx.status.zero_()
    ctx.push_deposit_variant(P, f_t, F_t, dt, shape_order=order, pusher=pusher)
    torch.cuda.synchronize()
    assert int(ctx.status.item()) == 0
    with O.shape_order(order), O.pusher(pusher):
        check_push(p, ptc, ref, P.to_numpy(), O, fields, dt)
    for c in range(3):
        assert grid_err(Fref[c], ctx.to_host(F_t[c])) <= 1e-11, c
    if pusher == 1:     # the option matters: Vay and Boris momenta differ at O(dt^3) per step
        refb = O.push(p, fields, ptc, dt)
        assert np.max(np.abs(refb["u1"] - ref["u1"])) > 0


def test_cic_vay_tuned_and_general_kernels_agree(G, O):
    """grpic_push_deposit_variant(1, 1) runs the tuned kernel (bulk-TMA tiles, 16-byte aligned particle
    arrays) and falls back to the general kernel for arrays off that grid: both against the oracle with
    the Vay option, and against each other."""
    p = inputs.grid_params(96, 80, 0.99, ng=3)
    dt = inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "wald")
    n = 50001
    ptc = inputs.make_particles(p, n, 43, "crowded", ("loguniform", 0.1, 1e3))
    with O.pusher(1):
        ref, Fref = oracle_push_deposit(O, p, fields, ptc, dt)
    ctx = G.Context(p, n)
    f_t = [ctx.to_device(f) for f in fields]
    got = []
    for shift in (0, 1):
        P = G.Particles(n + shift)
        if shift:          # views that start one element into their allocations: 8 / 4 bytes off the 16-byte grid
            P.t = {k: v[1:] for k, v in P.t.items()}
            P.n = n
        P.upload(ptc)
        assert (P.t["x1"].data_ptr() % 16 != 0) == bool(shift)
        F_t = ctx.zeros(3)
        ctx.status.zero_()
        ctx.push_deposit_variant(P, f_t, F_t, dt, shape_order=1, pusher=1)
        torch.cuda.synchronize()
        assert int(ctx.status.item()) == 0
        out = P.to_numpy()
        with O.pusher(1):
            check_push(p, ptc, ref, out, O, fields, dt)
        for c in range(3):
            assert grid_err(Fref[c], ctx.to_host(F_t[c])) <= 1e-11, c
        got.append(out)
    for k in ("x1", "x2", "x3", "u1", "u2", "u3"):
        assert np.max(np.abs(got[0][k] - got[1][k]) / (np.abs(got[1][k]) + 1e-300)) < 1e-11, k
    assert np.array_equal(got[0]["cell"], got[1]["cell"]) and np.array_equal(got[0]["flag"], got[1]["flag"])


def test_vacuum_wald_relaxation(G, O):
    """Section 3.2 of the paper (Fig.6): the a = 0 Wald field (Eq.25) placed in an
    a = 0.998 Kerr metric evolves, through damped oscillations, to a steady state with H_phi -> 0
    and with magnetic flux expelled from the horizon; "the field solver ... is well-behaved over a
    long time".  128 x 128 grid, ~8800 vacuum field steps (t = 90 r_g/c), damping layer towards the
    initial field.  H_phi is observed through the circulations C_H^r, C_H^theta it generates."""
    a, N = 0.998, 128
    p = inputs.grid_params(N, N, a, r_out=60.0, damp_cells=N // 8, damp_coef=1.0)
    dt = inputs.courant_dt(p)
    f0 = inputs.analytic_fields(p, "wald0")
    ctx = G.Context(p, 16)
    f_t = [ctx.to_device(f) for f in f0]
    bg = [ctx.to_device(f) for f in f0]
    ctx.fill_guards(f_t)
    A = [ctx.to_host(x) for x in ctx.get_areas()]
    Gd = p["ng"]
    dxi, _ = inputs.spacing(p)
    rn = np.exp(p["xi_in"] + np.arange(-Gd, N + Gd + 1) * dxi)
    rh = 1.0 + math.sqrt(1.0 - a * a)
    ih = int(np.argmin(np.abs(rn - rh)))
    sel = (rn > rh) & (rn < 10.0)

    def diag():
        C = ctx.circulation(f_t)
        ch = [float(np.max(np.abs(ctx.to_host(C[c])[Gd:Gd + N, :][:, sel]))) for c in range(2)]
        Br = ctx.to_host(f_t[3])
        return ch, float(np.sum(np.abs(Br[Gd:Gd + N // 2, ih] * A[3][Gd:Gd + N // 2, ih])))

    (chr0, cht0), flux0 = diag()
    for _ in range(int(90.0 / dt)):
        ctx.field_step(f_t, None, dt, bg)
    torch.cuda.synchronize()
    assert all(bool(torch.isfinite(x).all()) for x in f_t)
    (chr1, cht1), flux1 = diag()
    assert chr1 < chr0 / 30.0 and cht1 < cht0 / 30.0, (chr0, chr1, cht0, cht1)     # H_phi -> 0
    assert flux1 < flux0 / 1.8, (flux0, flux1)                                       # flux expelled from the horizon


def test_continuity_residual_gpu(G, O):
    """Charge conservation of the CUDA path itself: (rho1 - rho0) dV/dt + div F = 0 node by
    node to <= 1e-13 max|rho dV|/dt, using the library's own rho deposit."""
    cfg = small_case(2, 64, 64, 50000)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    # config 2's pairs are co-located with equal weights (rho = 0 exactly): use random weights
    ptc["w"] = np.random.default_rng(8).uniform(0.5, 1.5, len(ptc["x1"]))
    ctx = G.Context(p, len(ptc["x1"]))
    f_t = [ctx.to_device(f) for f in fields]
    P = G.Particles.from_numpy(ptc)
    rho0, rho1 = ctx.zeros(), ctx.zeros()
    ctx.deposit_rho(P, rho0, divide=False)
    F_t = ctx.zeros(3)
    ctx.push_deposit(P, f_t, F_t, dt)
    ctx.deposit_rho(P, rho1, divide=False)
    # fold the fluxes exactly as finalize does, but keep them as fluxes: use the oracle-free
    # route -- finalize divides by areas, so multiply back with the library's own areas.
    A = ctx.get_areas()
    J = [t.clone() for t in F_t]
    ctx.finalize_current(J, 0)
    torch.cuda.synchronize()
    Fr = ctx.to_host(J[0] * A[0])
    Fth = ctx.to_host(J[1] * A[1])
    r0, r1 = ctx.to_host(rho0), ctx.to_host(rho1)
    # oracle rho agrees (parity of deposit_rho)
    assert grid_err(O.rho(p, ptc, ptc["w"], divide=False), r0) <= 1e-12
    Gd, nr, nth = p["ng"], p["nr"], p["nth"]
    res = (r1 - r0) / dt
    div = np.zeros_like(res)
    div[:, 1:] += Fr[:, 1:] - Fr[:, :-1]
    div[1:, :] += Fth[1:, :] - Fth[:-1, :]
    tot = (res + div)[Gd:Gd + nth + 1, Gd + 1:Gd + nr]
    # particles that left through a radial boundary no longer contribute to rho1 but their
    # last move was deposited (reading G15): restrict to nodes they cannot touch
    scale = np.max(np.abs(r1)) / dt
    inner = tot[:, 2:-2]
    assert np.max(np.abs(inner)) <= 1e-13 * scale, np.max(np.abs(inner)) / scale


@pytest.mark.parametrize("nr,nth,ng", [(37, 29, 2), (130, 67, 3), (260, 131, 2)])
def test_fill_guards_bit_exact(G, O, nr, nth, ng):
    """grpic_fill_guards (axis values, radial guards, theta ghost rows: one launch whose threads compose
    the three rules) on arrays whose every entry, guards included, is random: bit for bit the oracle's
    boundary pass (copies and sign flips only), corners of guard columns x ghost rows included."""
    p = inputs.grid_params(nr, nth, 0.9, ng=ng)
    rng = np.random.default_rng(nr + ng)
    f = [rng.standard_normal(inputs.grid_shape(p)) for _ in range(6)]
    ref = O.apply_bc(p, [x.copy() for x in f])
    ctx = G.Context(p)
    f_t = [ctx.to_device(x) for x in f]
    ctx.fill_guards(f_t)
    torch.cuda.synchronize()
    for c in range(6):
        got = ctx.to_host(f_t[c])
        assert np.array_equal(got, ref[c]), (c, np.argwhere(got != ref[c])[:5])


@pytest.mark.parametrize("kind,damp,ng", [("wald", 0, 2), ("monopole", 9, 2), ("wald", 0, 3), ("monopole", 5, 4)])
def test_field_step_parity(G, O, kind, damp, ng):
    """Three field steps (predictor + N correctors, axis values, radial guards, ghost rows, damping
    layer) element by element against the oracle, guard nodes included; ng = 3 is the layout of the
    cubic-spline runs, ng = 4 exercises the guard loops beyond it."""
    p = inputs.grid_params(90, 70, 0.9, r_out=30.0, damp_cells=damp, damp_coef=0.7, ng=ng)
    dt = inputs.courant_dt(p)
    rng = np.random.default_rng(3)
    bg = inputs.analytic_fields(p, kind)
    f = [b.copy() for b in bg]
    f[5] = f[5] + inputs.gaussian_packet_Bph(p, amp=1e-2, width=2.0, r0=8.0)
    f = inputs.fill_guards(p, inputs.perturb(f, 1e-3, rng))
    J = inputs.random_current(p, rng)
    ctx = G.Context(p)
    f_t = [ctx.to_device(x) for x in f]
    J_t = [ctx.to_device(x) for x in J]
    bg_t = [ctx.to_device(x) for x in bg]
    fo = [x.copy() for x in f]
    # circulations of the initial state
    Cg = [ctx.to_host(t) for t in ctx.circulation(f_t)]
    Cr = O.circulation(p, O.apply_bc(p, [x.copy() for x in f]))
    for c in range(6):
        assert grid_err(Cr[c], Cg[c]) <= 1e-11, ("C", c)
    for step in range(3):
        O.field_step(p, fo, J, dt, bg=bg if damp else None)
        ctx.field_step(f_t, J_t, dt, background=bg_t if damp else None)
    torch.cuda.synchronize()
    for c in range(6):
        assert grid_err(fo[c], ctx.to_host(f_t[c])) <= 1e-11, c


def test_field_step_vacuum_euler_and_heun(G, O):
    for N, beta in ((0, 0.53), (1, 0.5)):
        p = inputs.grid_params(33, 29, 0.99, r_out=15.0, field_iters=N, beta_impl=beta)
        f = inputs.analytic_fields(p, "wald")
        ctx = G.Context(p)
        f_t = [ctx.to_device(x) for x in f]
        fo = [x.copy() for x in f]
        O.field_step(p, fo, None, 0.01)
        ctx.field_step(f_t, None, 0.01)
        for c in range(6):
            assert grid_err(fo[c], ctx.to_host(f_t[c])) <= 1e-11, (N, c)


@pytest.mark.parametrize("passes", [0, 3])
def test_finalize_current_parity(G, O, passes):
    cfg = small_case(1, 56, 44, 30000)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    ref, Fref = oracle_push_deposit(O, p, fields, ptc, dt)
    Jref = O.finalize_current(p, [x.copy() for x in Fref], passes)
    ctx, P, F_t = gpu_push_deposit(G, p, fields, ptc, dt)
    ctx.finalize_current(F_t, passes)
    torch.cuda.synchronize()
    for c in range(3):
        assert grid_err(Jref[c], ctx.to_host(F_t[c])) <= 1e-11, c


@pytest.mark.parametrize("n", [0, 1, 31, 2048, 2049, 70001])
def test_sort_and_compact_bit_exact(G, O, n):
    p = inputs.grid_params(64, 64, 0.9)
    ctx = G.Context(p, max(n, 1))
    rng = np.random.default_rng(n)
    ptc = inputs.make_particles(p, max(n, 2), 7, "crowded", ("loguniform", 0.1, 10.0))
    ptc = {k: v[:n].copy() for k, v in ptc.items()}
    ptc["flag"] = (ptc["flag"] | (2 * (rng.uniform(size=n) < 0.15))).astype(np.uint32)
    ptc["w"] = rng.uniform(0.5, 1.5, n)
    src = G.Particles.from_numpy(ptc) if n else G.Particles(0)
    dst = G.Particles(n)
    perm = torch.zeros(max(n, 1), dtype=torch.int32, device="cuda")
    ctx.sort(src, dst, perm)
    torch.cuda.synchronize()
    if n:
        pref = O.sort(ptc["cell"], ptc["flag"])
        assert np.array_equal(perm[:n].cpu().numpy().view(np.uint32), pref)
        got = dst.to_numpy()
        for k in ptc:
            assert np.array_equal(got[k], ptc[k][pref]), k
    dst2 = G.Particles(n)
    na = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    ctx.compact(src, dst2, na)
    torch.cuda.synchronize()
    idx = O.compact(ptc["flag"]) if n else np.zeros(0, dtype=np.uint32)
    assert int(na.item()) == len(idx)
    if n:
        got = dst2.to_numpy(len(idx))
        for k in ptc:
            assert np.array_equal(got[k], ptc[k][idx]), k
        tail = dst2.to_numpy()
        assert np.all(tail["flag"][len(idx):] & 2)


@pytest.mark.parametrize("n,B", [(0, 8), (1, 8), (33, 8), (2049, 1), (70001, 2), (70001, 8), (70001, 32), (300000, 8)])
def test_sort_interleaved_bit_exact(G, O, n, B):
    """grpic_sort_interleaved against the oracle's definition (S11b): permutation and reordered
    SoA bit-exact; crowded positions (many particles per cell), empty cells, removed particles."""
    p = inputs.grid_params(64, 48, 0.9)
    ctx = G.Context(p, max(n, 1))
    rng = np.random.default_rng(n + B)
    ptc = inputs.make_particles(p, max(n, 2), 11, "crowded", ("loguniform", 0.1, 10.0))
    ptc = {k: v[:n].copy() for k, v in ptc.items()}
    ptc["flag"] = (ptc["flag"] | (2 * (rng.uniform(size=n) < 0.1))).astype(np.uint32)
    src = G.Particles.from_numpy(ptc) if n else G.Particles(0)
    dst = G.Particles(n)
    perm = torch.zeros(max(n, 1), dtype=torch.int32, device="cuda")
    ctx.sort_interleaved(src, dst, B, perm)
    torch.cuda.synchronize()
    if n:
        pref = O.sort_interleaved(ptc["cell"], ptc["flag"], p["nr"] * p["nth"], B)
        assert np.array_equal(perm[:n].cpu().numpy().view(np.uint32), pref)
        got = dst.to_numpy()
        for k in ptc:
            assert np.array_equal(got[k], ptc[k][pref]), k


@pytest.mark.parametrize("n,frac", [(4096, 0.0), (4096, 1.0), (5, 1.0), (4100, 0.5)])
def test_sort_interleaved_degenerate_removal(G, O, n, frac):
    """No particle removed, every particle removed, half of them: both sorts against the oracle
    (the list of cell starts is closed by the position of the first removed particle and by n)."""
    p = inputs.grid_params(32, 32, 0.9)
    ctx = G.Context(p, n)
    rng = np.random.default_rng(n)
    ptc = inputs.make_particles(p, n, 13, "logical", ("loguniform", 0.1, 10.0))
    ptc["flag"] = (ptc["flag"] | (2 * (rng.uniform(size=n) < frac))).astype(np.uint32)
    src = G.Particles.from_numpy(ptc)
    for B in (0, 8):
        dst = G.Particles(n)
        perm = torch.zeros(n, dtype=torch.int32, device="cuda")
        if B:
            ctx.sort_interleaved(src, dst, B, perm)
            pref = O.sort_interleaved(ptc["cell"], ptc["flag"], p["nr"] * p["nth"], B)
        else:
            ctx.sort(src, dst, perm)
            pref = O.sort(ptc["cell"], ptc["flag"])
        torch.cuda.synchronize()
        assert np.array_equal(perm.cpu().numpy().view(np.uint32), pref)
        got = dst.to_numpy()
        for k in ptc:
            assert np.array_equal(got[k], ptc[k][pref]), k


def test_config1_ten_coupled_steps(G, O):
    """BASELINE.json config 1 at full size: 128x128, 1e5 particles, 10 x (push+deposit,
    finalize, field step N=7)."""
    cfg = inputs.config(1)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    ctx = G.Context(p, len(ptc["x1"]))
    f_t = [ctx.to_device(f) for f in fields]
    P = G.Particles.from_numpy(ptc)
    fo = [f.copy() for f in fields]
    cur = dict(ptc)
    # a second oracle trajectory from 4-ulp perturbed positions measures each particle's own
    # sensitivity over the 10 steps (ill-conditioned near-axis particles, see check_push)
    eps = 4 * np.finfo(np.float64).eps
    cur2 = dict(ptc, x1=ptc["x1"] * (1 + eps), x2=ptc["x2"] * (1 + eps))
    for step in range(10):
        new, F = oracle_push_deposit(O, p, fo, cur, dt)
        new2 = O.push(p, fo, cur2, dt)
        fields_before = [f.copy() for f in fo] if step == 0 else None
        J = O.finalize_current(p, F, 0)
        O.field_step(p, fo, J, dt)
        cur = {k: new[k] for k in ("x1", "x2", "x3", "u1", "u2", "u3", "cell", "flag")}
        cur["w"] = ptc["w"]
        cur2 = {k: new2[k] for k in ("x1", "x2", "x3", "u1", "u2", "u3", "cell", "flag")}
        cur2["w"] = ptc["w"]
        F_t = ctx.zeros(3)
        ctx.push_deposit(P, f_t, F_t, dt)
        ctx.finalize_current(F_t, 0)
        ctx.field_step(f_t, F_t, dt)
        if step == 0:
            torch.cuda.synchronize()
            check_push(p, ptc, new, P.to_numpy(), O, fields_before, dt, max_over=10)   # measured on B200: 5 of 1e5, all with sin(theta) < 3.6e-4
            for c in range(3):
                assert grid_err(J[c], ctx.to_host(F_t[c])) <= 1e-11
            for c in range(6):
                assert grid_err(fo[c], ctx.to_host(f_t[c])) <= 1e-11
    torch.cuda.synchronize()
    got = P.to_numpy()
    same = (got["flag"] == cur["flag"]) & (cur2["flag"] == cur["flag"])
    assert same.mean() > 0.9999
    sens = np.maximum(ptc_err(cur, cur2, ("x1", "x2", "x3")), ptc_err(cur, cur2, ("u1", "u2", "u3")))
    tolk = np.maximum(1e-10, 100.0 * sens)
    assert (np.maximum(ptc_err(cur, got, ("x1", "x2", "x3")), ptc_err(cur, got, ("u1", "u2", "u3")))[same]
            > 1e-10).mean() < 1e-3
    ex = ptc_err(cur, got, ("x1", "x2", "x3"))
    eu = ptc_err(cur, got, ("u1", "u2", "u3"))
    assert np.all(ex[same] <= tolk[same]) and np.all(eu[same] <= tolk[same]), \
        (ex[same].max(), eu[same].max())
    for c in range(6):
        assert grid_err(fo[c], ctx.to_host(f_t[c])) <= 1e-10, c


def test_config5_coupled_loop_reduced(G, O):
    """BASELINE.json config 5 recipe at reduced size (96^2, 40000 particles): 6 x (sort every 2
    steps, fused push+deposit+removal, 3 binomial filter passes, field step N=7).  After every
    step the particle ORDER and the integer state are compared bit for bit with the oracle loop
    (stable sort, stable compaction), the float state at 1e-12 .. 1e-10 as the steps accumulate."""
    cfg = inputs.config(5, nr=96, nth=96, n=40000)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    ptc["w"][:] = 1e-6
    n = len(ptc["x1"])
    ctx = G.Context(p, n)
    f_t = [ctx.to_device(f) for f in fields]
    A, B = G.Particles.from_numpy(ptc), G.Particles(n)
    n_alive = torch.zeros(1, dtype=torch.int64, device="cuda")
    fo = [f.copy() for f in fields]
    cur = dict(ptc)
    keys = ("x1", "x2", "x3", "u1", "u2", "u3", "cell", "flag")
    for step in range(6):
        if step % 2 == 0:
            perm = O.sort(cur["cell"], cur["flag"])
            cur = {k: np.ascontiguousarray(v[perm]) for k, v in cur.items()}
            ctx.sort(A, B)
            A, B = B, A
        keep = O.compact(cur["flag"])
        cur = {k: np.ascontiguousarray(v[keep]) for k, v in cur.items()}
        new, F = oracle_push_deposit(O, p, fo, cur, dt)
        J = O.finalize_current(p, F, 3)
        O.field_step(p, fo, J, dt)
        w = cur["w"]
        cur = {k: new[k] for k in keys}
        cur["w"] = w
        F_t = ctx.zeros(3)
        ctx.push_deposit_compact(A, B, f_t, F_t, dt, n_alive)
        A, B = B, A
        ctx.finalize_current(F_t, 3)
        ctx.field_step(f_t, F_t, dt)
        torch.cuda.synchronize()
        m = int(n_alive.item())
        assert m == len(keep), (step, m, len(keep))
        got = A.to_numpy(m)
        tol = 1e-12 * 10 ** min(step, 2)
        ex, eu = ptc_err(cur, got, ("x1", "x2", "x3")), ptc_err(cur, got, ("u1", "u2", "u3"))
        assert (np.maximum(ex, eu) > tol).mean() < 1e-3, (step, (np.maximum(ex, eu) > tol).mean())
        assert np.array_equal(got["flag"], cur["flag"]) and np.array_equal(got["cell"], cur["cell"]), step
        for c in range(3):
            assert grid_err(J[c], ctx.to_host(F_t[c])) <= 1e-10, (step, c)
        for c in range(6):
            assert grid_err(fo[c], ctx.to_host(f_t[c])) <= 1e-10, (step, c)


def test_config2_full_size_sampled(G, O):
    """BASELINE.json config 2 at full size (1024^2, 2e7 particles) in the launch
    configuration bench.py times: sort, then one push+deposit step.  The oracle pushes a
    sample of particles one by one (particles are independent); the deposit is checked by
    properties that hold at any size (moments of the fluxes, continuity residual)."""
    cfg = inputs.config(2)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    n = len(ptc["x1"])
    ctx = G.Context(p, n)
    f_t = [ctx.to_device(f) for f in fields]
    A, B = G.Particles.from_numpy(ptc), G.Particles(n)
    perm_t = torch.zeros(n, dtype=torch.int32, device="cuda")
    ctx.sort(A, B, perm_t)
    torch.cuda.synchronize()
    perm = perm_t.cpu().numpy().view(np.uint32)
    key = ptc["cell"].astype(np.int64)
    assert np.all(np.diff(key[perm]) >= 0)
    # stability + permutation: equal keys keep index order
    same = np.diff(key[perm]) == 0
    assert np.all(np.diff(perm.astype(np.int64))[same] > 0)
    assert np.array_equal(np.sort(perm), np.arange(n, dtype=np.uint32))
    rho0, rho1 = ctx.zeros(), ctx.zeros()
    ctx.deposit_rho(B, rho0, divide=False)
    F_t = ctx.zeros(3)
    ctx.push_deposit(B, f_t, F_t, dt)
    ctx.deposit_rho(B, rho1, divide=False)
    torch.cuda.synchronize()
    got = B.to_numpy()
    rng = np.random.default_rng(0)
    sample = rng.choice(n, 20000, replace=False)
    src = perm[sample]
    sub = {k: np.ascontiguousarray(v[src]) for k, v in ptc.items()}
    ref = O.push(p, fields, sub, dt)
    gsub = {k: got[k][sample] for k in got}
    check_push(p, sub, ref, gsub, O, fields, dt)
    # moments: sum F_ph = sum Q dphi/dt over all particles
    Q = np.where(ptc["flag"][perm] & 1, 1.0, -1.0) * ptc["w"][perm]
    dphi = got["x3"] - ptc["x3"][perm]
    Fph = ctx.to_host(F_t[2])
    assert abs(Fph.sum() - np.sum(Q * dphi) / dt) <= 1e-9 * np.sum(np.abs(Q * dphi)) / dt
    # continuity on interior nodes
    Aar = ctx.get_areas()
    J = [t.clone() for t in F_t]
    ctx.finalize_current(J, 0)
    Fr, Fth = ctx.to_host(J[0] * Aar[0]), ctx.to_host(J[1] * Aar[1])
    r0, r1 = ctx.to_host(rho0), ctx.to_host(rho1)
    Gd, nr, nth = p["ng"], p["nr"], p["nth"]
    res = (r1 - r0) / dt
    div = np.zeros_like(res)
    div[:, 1:] += Fr[:, 1:] - Fr[:, :-1]
    div[1:, :] += Fth[1:, :] - Fth[:-1, :]
    tot = (res + div)[Gd:Gd + nth + 1, Gd + 3:Gd + nr - 2]
    scale = np.max(np.abs(r1)) / dt
    assert np.max(np.abs(tot)) <= 1e-13 * scale, np.max(np.abs(tot)) / scale


@pytest.mark.gpu
def test_config3_full_size_bench_path(G, O):
    """BASELINE.json config 3 at full size (2048^2, 1e8 particles) in the launch configuration
    bench.py times: cell sort, then two fused push+deposit+compaction steps (the second one
    squeezes out what the first removed).  Sort permutation vs the oracle's stable sort on the
    whole set; a sample of particles pushed one by one by the oracle through both steps;
    survivor counts and order bit-exact; flux moments at full size."""
    cfg = inputs.config(3)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    n = len(ptc["x1"])
    ctx = G.Context(p, n)
    f_t = [ctx.to_device(f) for f in fields]
    A, B = G.Particles.from_numpy(ptc), G.Particles(n)
    perm_t = torch.zeros(n, dtype=torch.int32, device="cuda")
    ctx.sort(A, B, perm_t)
    torch.cuda.synchronize()
    perm = perm_t.cpu().numpy().view(np.uint32)
    del perm_t
    assert np.array_equal(perm, O.sort(ptc["cell"], ptc["flag"]))       # bit-exact at 1e8
    n1 = torch.zeros(1, dtype=torch.int64, device="cuda")
    n2 = torch.zeros(1, dtype=torch.int64, device="cuda")
    F1, F2 = ctx.zeros(3), ctx.zeros(3)
    ctx.status.zero_()
    ctx.push_deposit_compact(B, A, f_t, F1, dt, n1)                      # step 1: B -> A
    torch.cuda.synchronize()
    got1 = A.to_numpy()
    assert int(n1.item()) == n and int(ctx.status.item()) == 0
    ctx.push_deposit_compact(A, B, f_t, F2, dt, n2)                      # step 2: A -> B
    torch.cuda.synchronize()
    got2 = B.to_numpy()
    alive1 = (got1["flag"] & 2) == 0
    m2 = int(n2.item())
    assert m2 == int(alive1.sum()) and m2 < n                            # some particles did leave
    assert np.all(got2["flag"][m2:] & 2)
    # oracle on a sample (particles are independent): positions in the sorted order
    rng = np.random.default_rng(3)
    sample = np.sort(rng.choice(n, 200_000, replace=False))
    lost = np.flatnonzero(~alive1)
    sample = np.union1d(sample, lost[:5000])                             # include leavers
    src = perm[sample]
    sub = {k: np.ascontiguousarray(v[src]) for k, v in ptc.items()}
    ref1 = O.push(p, fields, sub, dt)
    check_push(p, sub, ref1, {k: got1[k][sample] for k in got1}, O, fields, dt)
    # step 2: survivors of the sample, at their compacted positions
    pos2 = np.cumsum(alive1)[sample] - 1
    keep = alive1[sample]
    sub2 = {k: np.ascontiguousarray(got1[k][sample][keep]) for k in ("x1", "x2", "x3", "u1", "u2", "u3", "cell", "flag")}
    # inputs of the oracle's second step are the ORACLE's own first-step outputs where they agree
    # bit for bit in the integer fields; the float state is taken from the oracle
    for k in ("x1", "x2", "x3", "u1", "u2", "u3"):
        sub2[k] = np.ascontiguousarray(ref1[k][keep])
    sub2["w"] = np.ascontiguousarray(sub["w"][keep])
    ref2 = O.push(p, fields, sub2, dt)
    g2 = {k: got2[k][pos2[keep]] for k in got2}
    # the GPU's second step started from its own first-step state (<= 1e-12 from the oracle's):
    # compare at 1e-11 (one more step of the same conditioning)
    check_push(p, sub2, ref2, g2, O, fields, dt, tol=1e-11)
    # flux moments of step 1 over all particles (properties that hold at any size)
    Q = np.where(ptc["flag"][perm] & 1, 1.0, -1.0) * ptc["w"][perm]
    dphi = got1["x3"] - ptc["x3"][perm]
    Fph = ctx.to_host(F1[2])
    assert abs(Fph.sum() - np.sum(Q * dphi) / dt) <= 1e-9 * np.sum(np.abs(Q * dphi)) / dt


# ------------------------------------------------------------------ full-size cases added in round 2
@pytest.mark.parametrize("N", [2048, 4096])
def test_field_step_full_size_parity(G, O, N):
    """One full grpic_field_step (predictor + 7 correctors, axis / guard conditions, damping over the
    outer 10 % of the radial cells, prescribed random J) at the sizes bench.py runs: 2048^2 (configs[2],
    [4]) and BASELINE.json configs[3]'s 4096^2, in the launch shape of those sizes (32-row chunks,
    several waves of CTAs, TMA row rings), element by element against the oracle: <= 1e-11 of the
    array's max.  The second field step is compared at 2048^2 too (the
    first one's output, guards included, is the second one's input)."""
    cfg = inputs.config(4, nr=N, nth=N)
    p, dt = cfg["params"], cfg["dt"]
    ctx = G.Context(p, 16)
    f_t = [ctx.to_device(x) for x in cfg["fields"]]
    bg_t = [ctx.to_device(x) for x in cfg["bg"]]
    J_t = [ctx.to_device(x) for x in cfg["J"]]
    ctx.fill_guards(f_t)
    fo = [x.copy() for x in cfg["fields"]]
    steps = 2 if N == 2048 else 1
    for s in range(steps):
        ctx.field_step(f_t, J_t, dt, bg_t)
        O.field_step(p, fo, cfg["J"], dt, bg=cfg["bg"])
        torch.cuda.synchronize()
        for c in range(6):
            got = ctx.to_host(f_t[c])
            assert np.all(np.isfinite(got))
            assert grid_err(fo[c], got) <= 1e-11, (N, s, c, grid_err(fo[c], got))


def test_field_step_arrays_off_the_16_byte_grid(G):
    """Field and current arrays that start 8 bytes off a 16-byte boundary (a caller's view) cannot be
    fetched by bulk copies: grpic_field_step takes its load path for them and gives bit-identical
    results to the aligned call."""
    cfg = inputs.config(4, nr=256, nth=192)
    p, dt = cfg["params"], cfg["dt"]
    ctx = G.Context(p, 16)
    def shifted(t):
        buf = torch.zeros(t.numel() + 1, dtype=torch.float64, device="cuda")
        v = buf[1:].view(t.shape)
        v.copy_(t)
        assert v.data_ptr() % 16 == 8
        return v
    f_a = [ctx.to_device(x) for x in cfg["fields"]]
    J_a = [ctx.to_device(x) for x in cfg["J"]]
    bg = [ctx.to_device(x) for x in cfg["bg"]]
    ctx.fill_guards(f_a)
    f_b = [shifted(t) for t in f_a]
    J_b = [shifted(t) for t in J_a]
    for _ in range(2):
        ctx.field_step(f_a, J_a, dt, bg)
        ctx.field_step(f_b, J_b, dt, bg)
    torch.cuda.synchronize()
    for c in range(6):
        assert torch.equal(f_a[c], f_b[c]), c


def test_config3_full_size_interleaved_lazy_path(G, O):
    """The path bench.py times by default since round 2, at BASELINE.json config 3's full size (2048^2,
    1e8 particles): grpic_sort_interleaved (block of 8 cells) -- permutation bit-exact against the
    oracle's definition S11b on all 1e8 particles -- then two IN-PLACE pushes with lazy removal: the
    removed counters equal the number of flags set, flagged particles are skipped by the second
    push (state untouched), a sample is pushed one by one by the oracle through both steps."""
    cfg = inputs.config(3)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    n = len(ptc["x1"])
    ctx = G.Context(p, n)
    f_t = [ctx.to_device(f) for f in fields]
    A, B = G.Particles.from_numpy(ptc), G.Particles(n)
    perm_t = torch.zeros(n, dtype=torch.int32, device="cuda")
    ctx.sort_interleaved(A, B, 8, perm_t)
    torch.cuda.synchronize()
    perm = perm_t.cpu().numpy().view(np.uint32)
    del perm_t, A
    assert np.array_equal(perm, O.sort_interleaved(ptc["cell"], ptc["flag"], p["nr"] * p["nth"], 8))
    removed = torch.zeros(2, dtype=torch.int64, device="cuda")
    F1, F2 = ctx.zeros(3), ctx.zeros(3)
    ctx.status.zero_()
    ctx.set_removed_counter(removed[0:1])
    ctx.push_deposit(B, f_t, F1, dt)
    torch.cuda.synchronize()
    got1 = B.to_numpy()
    ctx.set_removed_counter(removed[1:2])
    ctx.push_deposit(B, f_t, F2, dt)
    ctx.set_removed_counter(None)
    torch.cuda.synchronize()
    got2 = B.to_numpy()
    assert int(ctx.status.item()) == 0
    gone1 = (got1["flag"] & 2) != 0
    gone2 = (got2["flag"] & 2) != 0
    r = removed.cpu().numpy()
    assert int(r[0]) == int(gone1.sum()) > 0 and int(r[0] + r[1]) == int(gone2.sum())
    for k in ("x1", "x2", "x3", "u1", "u2", "u3"):          # lazily removed particles are not touched again
        assert np.array_equal(got2[k][gone1], got1[k][gone1]), k
    rng = np.random.default_rng(4)
    sample = np.union1d(np.sort(rng.choice(n, 200_000, replace=False)), np.flatnonzero(gone1)[:5000])
    src = perm[sample]
    sub = {k: np.ascontiguousarray(v[src]) for k, v in ptc.items()}
    ref1 = O.push(p, fields, sub, dt)
    check_push(p, sub, ref1, {k: got1[k][sample] for k in got1}, O, fields, dt, label="c3 lazy step 1")
    sub2 = {k: np.ascontiguousarray(ref1[k]) for k in ("x1", "x2", "x3", "u1", "u2", "u3", "cell", "flag")}
    sub2["w"] = sub["w"]
    ref2 = O.push(p, fields, sub2, dt)
    check_push(p, sub2, ref2, {k: got2[k][sample] for k in got2}, O, fields, dt, tol=1e-11,
               label="c3 lazy step 2")
    Q = np.where(ptc["flag"][perm] & 1, 1.0, -1.0) * ptc["w"][perm]
    dphi = got1["x3"] - ptc["x3"][perm]
    Fph = ctx.to_host(F1[2])
    assert abs(Fph.sum() - np.sum(Q * dphi) / dt) <= 1e-9 * np.sum(np.abs(Q * dphi)) / dt


def test_config2_multi_step_loop_reduced(G, O):
    """BASELINE.json config 2's recipe ("100 steps, sort every 20 steps", fields frozen) at reduced size
    (128^2, 60000 particles = 30000 pairs), 45 steps with a cell sort at steps 0, 20 and 40, both sort
    orders: particle ORDER, cells and flags bit-exact against the oracle loop after every sort; the
    float state within the accumulated-conditioning bound of section 7 at the end."""
    cfg = inputs.config(2, nr=128, nth=128, n=30000)
    p, dt, fields, ptc0 = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    n = len(ptc0["x1"])
    ncells = p["nr"] * p["nth"]
    for order in ("stable", "interleaved"):
        ctx = G.Context(p, n)
        f_t = [ctx.to_device(f) for f in fields]
        A, B = G.Particles.from_numpy(ptc0), G.Particles(n)
        cur = {k: v.copy() for k, v in ptc0.items()}
        eps = 4 * np.finfo(np.float64).eps
        cur2 = dict(cur, x1=cur["x1"] * (1 + eps), x2=cur["x2"] * (1 + eps))
        F_t = ctx.zeros(3)
        for step in range(45):
            if step % 20 == 0:
                perm = O.sort(cur["cell"], cur["flag"]) if order == "stable" else \
                    O.sort_interleaved(cur["cell"], cur["flag"], ncells, 8)
                cur = {k: np.ascontiguousarray(v[perm]) for k, v in cur.items()}
                cur2 = {k: np.ascontiguousarray(v[perm]) for k, v in cur2.items()}
                if order == "stable":
                    ctx.sort(A, B)
                else:
                    ctx.sort_interleaved(A, B, 8)
                A, B = B, A
                torch.cuda.synchronize()
                got = A.to_numpy()
                same = got["flag"] == cur["flag"]
                # the order is decided by integer keys: identical as long as the cells agree
                assert np.array_equal(got["cell"], cur["cell"]) and same.all(), (order, step)
                assert np.array_equal(got["w"], cur["w"])
            new = O.push(p, fields, cur, dt)
            new2 = O.push(p, fields, cur2, dt)
            for k in ("x1", "x2", "x3", "u1", "u2", "u3", "cell", "flag"):
                cur[k], cur2[k] = new[k], new2[k]
            ctx.push_deposit(A, f_t, F_t, dt)
        torch.cuda.synchronize()
        got = A.to_numpy()
        ok = (got["flag"] == cur["flag"]) & (cur2["flag"] == cur["flag"])
        assert ok.mean() > 0.9999
        sens = np.maximum(ptc_err(cur, cur2, ("x1", "x2", "x3")), ptc_err(cur, cur2, ("u1", "u2", "u3")))
        err = np.maximum(ptc_err(cur, got, ("x1", "x2", "x3")), ptc_err(cur, got, ("u1", "u2", "u3")))
        print("parity c2 loop", order, "worst", err[ok].max(), "over 1e-10:", int((err[ok] > 1e-10).sum()))
        assert np.all(err[ok] <= np.maximum(1e-10, 100.0 * sens[ok]))
        assert (err[ok] > 1e-10).mean() < 1e-3


def test_config5_full_size(G, O):
    """BASELINE.json configs[4] at full size: 2048^2 grid, 2e8 particles (density ~ r^-2, thermal
    momenta), one step of the coupled loop in bench.py's launch configuration: stable cell sort
    (permutation bit-exact on all 2e8 keys), fused push + deposit + removal, 3 binomial filter passes +
    normalisation.  A sample of 2e5 particles is pushed one by one by the oracle; J is compared on a
    band of theta rows that the oracle deposits from exactly the particles that can reach it (a move
    is shorter than one cell, the filter reaches 3 rows further): <= 1e-11 of the band's max."""
    cfg = inputs.config(5)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    ptc["w"][:] = 1e-6
    n = len(ptc["x1"])
    assert n == 200_000_000
    ctx = G.Context(p, n)
    f_t = [ctx.to_device(f) for f in fields]
    A, B = G.Particles.from_numpy(ptc), G.Particles(n)
    perm_t = torch.zeros(n, dtype=torch.int32, device="cuda")
    ctx.sort(A, B, perm_t)
    torch.cuda.synchronize()
    perm = perm_t.cpu().numpy().view(np.uint32)
    del perm_t
    assert np.array_equal(perm, O.sort(ptc["cell"], ptc["flag"]))
    n1 = torch.zeros(1, dtype=torch.int64, device="cuda")
    F = ctx.zeros(3)
    ctx.status.zero_()
    ctx.push_deposit_compact(B, A, f_t, F, dt, n1)
    ctx.finalize_current(F, 3)
    torch.cuda.synchronize()
    assert int(n1.item()) == n and int(ctx.status.item()) == 0
    got = A.to_numpy()
    rng = np.random.default_rng(5)
    sample = np.sort(rng.choice(n, 200_000, replace=False))
    src = perm[sample]
    sub = {k: np.ascontiguousarray(v[src]) for k, v in ptc.items()}
    ref = O.push(p, fields, sub, dt)
    check_push(p, sub, ref, {k: got[k][sample] for k in got}, O, fields, dt, label="c5 full size")
    # J on a band of rows: every particle whose old or new theta row lies within the band +- 6 rows
    dth = math.pi / p["nth"]
    j0, j1 = 1000, 1024
    jo = np.floor(ptc["x2"] / dth).astype(np.int64)
    jn = np.floor(got["x2"] / dth).astype(np.int64)           # sorted order
    inv_sel = ((jn >= j0 - 8) & (jn <= j1 + 8))
    sel_sorted = np.flatnonzero(inv_sel | ((jo[perm] >= j0 - 8) & (jo[perm] <= j1 + 8)))
    srcb = perm[sel_sorted]
    subb = {k: np.ascontiguousarray(v[srcb]) for k, v in ptc.items()}
    refb = O.push(p, fields, subb, dt)
    Jb = O.finalize_current(p, O.deposit(p, subb, refb, subb["w"], dt), 3)
    Gd = p["ng"]
    for c in range(3):
        gotJ = ctx.to_host(F[c])[Gd + j0:Gd + j1 + 1, :]
        refJ = Jb[c][Gd + j0:Gd + j1 + 1, :]
        e = np.max(np.abs(gotJ - refJ)) / np.max(np.abs(refJ))
        assert e <= 1e-11, (c, e)


def test_step_host_flux_exchange_hook(G, O):
    """grpic_set_flux_exchange: the multi-GPU hook of grpic_step_host is called exactly once per step,
    between the deposit and the finalisation, with the context's contiguous 3-array flux block.  One GPU
    stands in for N identical ranks: a hook that triples the block (the sum over three equal ranks) must
    give exactly the oracle's J for three copies of the particle set, and the fields that follow."""
    p = inputs.grid_params(40, 32, 0.9, field_iters=2)
    dt = inputs.courant_dt(p)
    fields = inputs.analytic_fields(p, "wald")
    n = 5000
    ptc = inputs.make_particles(p, n, 5, "r2", ("loguniform", 0.1, 10.0))
    ptc["w"][:] = 1e-3
    ctx = G.Context(p, n)
    f_t = [ctx.to_device(f) for f in fields]
    host = {k: torch.from_numpy(v.copy() if v.dtype != np.uint32 else v.view(np.int32).copy()).pin_memory()
            for k, v in ptc.items()}
    host["n"] = n
    hJ = [torch.zeros((ctx.rows, ctx.pitch), dtype=torch.float64).pin_memory() for _ in range(3)]
    calls = []

    def hook(block):
        calls.append(tuple(block.shape))
        block.mul_(3.0)
    ctx.set_flux_exchange(hook)
    ctx.step_host(host, f_t, dt, host_J=hJ)
    ctx.set_flux_exchange(None)
    assert calls == [(3, ctx.rows, ctx.pitch)]
    ref, Fref = oracle_push_deposit(O, p, fields, ptc, dt)
    Jref = O.finalize_current(p, [3.0 * F for F in Fref], 0)
    fref = O.field_step(p, [f.copy() for f in fields], Jref, dt)
    for c in range(3):
        assert grid_err(Jref[c], ctx.to_host(hJ[c].cuda())) <= 1e-11, c
    for c in range(6):
        assert grid_err(fref[c], ctx.to_host(f_t[c])) <= 1e-11, c
    ctx.step_host(host, f_t, dt, host_J=hJ)            # hook removed: not called again
    assert len(calls) == 1


def test_bench_two_ranks_if_two_gpus():
    """bench.py --gpus 2 on a box with at least two devices: two NCCL ranks, n_gpus = 2 on the line."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (the pool's boxes expose one)")
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "3",
                          "--particles", "2000000", "--grid", "512", "--no-cpu-baseline", "--e2e-steps", "1"],
                         capture_output=True, text=True, timeout=900, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert d["n_gpus"] == 2 and d["value"] > 0 and "allreduce" in d["phases_ms"]


def test_ks_to_bl_parity(G, O):
    """grpic_ks_to_bl against the oracle's (A6)/(A7) transform, particle by particle (photons, removed
    particles, near-horizon and near-axis positions included): <= 1e-12 relative."""
    p = inputs.grid_params(64, 48, 0.95)
    n = 20000
    ptc = inputs.make_particles(p, n, 21, "crowded", ("loguniform", 0.1, 1e4))
    rng = np.random.default_rng(2)
    ptc["flag"] = (ptc["flag"] | np.where(rng.uniform(size=n) < 0.2, 4, 0) | np.where(rng.uniform(size=n) < 0.05, 2, 0)).astype(np.uint32)
    ctx = G.Context(p, n)
    P = G.Particles.from_numpy(ptc)
    got = [t.cpu().numpy() for t in ctx.ks_to_bl(P)]
    live = (ptc["flag"] & 2) == 0
    for k in range(n):
        if not live[k]:
            assert all(np.isnan(g[k]) for g in got)
            continue
        if k % 7:
            continue
        ref = O.ks_to_bl(p["a"], 1.0, ptc["x1"][k], ptc["x2"][k], ptc["x3"][k],
                         [ptc["u1"][k], ptc["u2"][k], ptc["u3"][k]], 0.0 if ptc["flag"][k] & 4 else 1.0)
        for c in range(4):
            assert abs(got[c][k] - ref[c]) <= 1e-12 * max(1.0, abs(ref[c])), (k, c, got[c][k], ref[c])


def _h_phi(p, f):
    """H_phi at (i+1/2, j+1/2) from stored D, B by (B9), written with numpy and the
    input module's metric (independent of the oracle and of the CUDA path)."""
    G, nr, nth = p["ng"], p["nr"], p["nth"]
    a, M = p["a"], p["M"]
    def at(name):
        r, th = inputs.positions(p, name)
        return inputs.kerr_schild(a, M, r, th)
    mB, mR, mT = at("Bph"), at("Br"), at("Dth")
    Dth, Br, Bph = f[1], f[3], f[5]
    cB = (mB["alpha"] * mB["g_phph"]) * np.ones_like(Bph)
    tR = (mR["alpha"] * mR["g_rph"]) * Br
    tT = (mT["sqrtg"] * mT["beta_r"]) * Dth
    H = cB * Bph
    H[:, :-1] += 0.5 * (tR[:, :-1] + tR[:, 1:]) - 0.5 * (tT[:, :-1] + tT[:, 1:])
    return H[G:G + nth, G:G + nr]


def test_vacuum_wald_relaxation_quantitative(G, O):
    """Section 3.2 (Fig.6) at 512^2: the a = 0 Wald potential A_phi = (B0/2) gamma_phiphi
    (Eq.25, reading G6) in an a = 0.998 Kerr metric, flux-initialised (B^r A^B_r = dphi Delta_theta A_phi,
    B^theta A^B_theta = -dphi Delta_r A_phi: discrete div B = 0 to round-off) with D^phi from Eq.(6) at
    E_i = 0 and D^r = D^theta = 0 (reading W1: "D^phi is nonzero and needs to be solved using Equation
    (6)"; a toroidal D is divergence-free, so the vacuum run carries no spurious charge).  After
    t = 90 r_g/c the paper reports H_phi -> 0, the magnetic flux expelled from the horizon and agreement
    with the spinning Wald solution (C14-C19).  Asserted here (values measured on B200 in the comments)."""
    a, N = 0.998, 512
    p = inputs.grid_params(N, N, a, r_out=60.0, damp_cells=N // 8, damp_coef=1.0)
    dt = inputs.courant_dt(p)
    ctx = G.Context(p, 16)
    Gd = p["ng"]
    A = [ctx.to_host(x) for x in ctx.get_areas()]             # A^D_r, A^D_th, A^D_ph, A^B_r, A^B_th, A^B_ph
    dxi, dth = inputs.spacing(p)
    ii = np.arange(-Gd, N + Gd + 1)
    jj = np.arange(-Gd, N + Gd + 1)
    rn, thn = np.exp(p["xi_in"] + ii * dxi)[None, :], (jj * dth)[:, None]
    Aphi = 0.5 * inputs.kerr_schild(a, 1.0, rn, thn)["g_phph"]           # B0 = 1, at nodes (i, j)
    f0 = inputs.analytic_fields(p, "wald0")
    Br, Bth = np.zeros_like(f0[3]), np.zeros_like(f0[4])
    with np.errstate(divide="ignore", invalid="ignore"):
        Br[:-1, :] = p["dphi"] * (Aphi[1:, :] - Aphi[:-1, :]) / A[3][:-1, :]
        Bth[:, :-1] = -p["dphi"] * (Aphi[:, 1:] - Aphi[:, :-1]) / A[4][:, :-1]
    Br, Bth = np.where(np.isfinite(Br), Br, 0.0), np.where(np.isfinite(Bth), Bth, 0.0)
    f0 = inputs.fill_guards(p, [np.zeros_like(Br), np.zeros_like(Br), f0[2], Br, Bth, np.zeros_like(Br)])
    f_t = [ctx.to_device(f) for f in f0]
    bg = [ctx.to_device(f) for f in f0]
    ctx.fill_guards(f_t)
    rh = 1.0 + math.sqrt(1.0 - a * a)
    r_c = np.exp(p["xi_in"] + (np.arange(N) + 0.5) * dxi)
    sel = (r_c > 1.02 * rh) & (r_c < 10.0)
    ih = int(np.argmin(np.abs(np.exp(p["xi_in"] + np.arange(N + 1) * dxi) - rh)))

    def state():
        f = [ctx.to_host(x) for x in f_t]
        H = _h_phi(p, f)
        flux = float(np.sum(np.abs(f[3][Gd:Gd + N // 2, Gd + ih] * A[3][Gd:Gd + N // 2, Gd + ih])))
        return f, float(np.max(np.abs(H[:, sel]))), flux

    # discrete div B of the initial state: sum of the face fluxes of every primal cell
    FB_r = f0[3] * A[3]
    FB_t = f0[4] * A[4]
    div = (FB_r[Gd:Gd + N, Gd + 1:Gd + N + 1] - FB_r[Gd:Gd + N, Gd:Gd + N]) + (FB_t[Gd + 1:Gd + N + 1, Gd:Gd + N] - FB_t[Gd:Gd + N, Gd:Gd + N])
    assert np.max(np.abs(div)) <= 1e-12 * np.max(np.abs(FB_r))
    _, h0, flux0 = state()
    for _ in range(int(90.0 / dt)):
        ctx.field_step(f_t, None, dt, bg)
    torch.cuda.synchronize()
    f1, h1, flux1 = state()
    assert all(np.all(np.isfinite(x)) for x in f1)
    wald = inputs.analytic_fields(p, "wald")
    reg = (np.exp(p["xi_in"] + np.arange(N + 1) * dxi) > 1.2 * rh) & (np.exp(p["xi_in"] + np.arange(N + 1) * dxi) < 15.0)
    rows = slice(Gd + 8, Gd + N - 8)
    errs = []
    for c in (3, 4):        # B^r, B^theta against the spinning Wald field, relative to the largest value in the region
        x, w = f1[c][rows, Gd:Gd + N + 1][:, reg], wald[c][rows, Gd:Gd + N + 1][:, reg]
        x0 = f0[c][rows, Gd:Gd + N + 1][:, reg]
        errs.append((float(np.max(np.abs(x - w)) / np.max(np.abs(w))), float(np.max(np.abs(x0 - w)) / np.max(np.abs(w)))))
    fw = float(np.sum(np.abs(wald[3][Gd:Gd + N // 2, Gd + ih] * A[3][Gd:Gd + N // 2, Gd + ih])))
    print("wald relaxation: max|H_phi| %.3e -> %.3e; horizon flux %.4f -> %.4f (spinning Wald %.4f); "
          "B^r, B^theta vs Wald (final, initial): %s" % (h0, h1, flux0, flux1, fw, errs))
    # measured on B200: max|H_phi|/B0 1.444 -> 0.0165; horizon flux 12.566 -> 0.7445 (spinning Wald: 0.7907);
    # B^r, B^theta within 0.17 % / 0.81 % of the spinning Wald field (initially 72 % / 64 % away)
    assert h1 < h0 / 50.0
    assert abs(flux1 - fw) < 0.1 * fw and flux1 < 0.1 * flux0
    assert errs[0][0] < 5e-3 and errs[1][0] < 2e-2


def test_clock_probe_and_removed_counter(G, O):
    """grpic_set_clock_probe: a push launch reports start / end SM cycle counter and nanosecond timer
    (plausible clock, positive duration); grpic_set_removed_counter: += the number of particles the
    launch flagged removed, equal to the oracle's count, for the in-place and the compacting push."""
    cfg = small_case(3, 80, 72, 40000)
    p, dt, fields, ptc = cfg["params"], cfg["dt"], cfg["fields"], cfg["particles"]
    ref = O.push(p, fields, ptc, dt)
    n_gone = int(((ref["flag"] & 2) != 0).sum())
    assert n_gone > 0
    ctx = G.Context(p, len(ptc["x1"]))
    f_t = [ctx.to_device(f) for f in fields]
    words = torch.zeros(4, dtype=torch.int64, device="cuda")
    cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
    P = G.Particles.from_numpy(ptc)
    ctx.set_clock_probe(words)
    ctx.set_removed_counter(cnt[0:1])
    ctx.push_deposit(P, f_t, ctx.zeros(3), dt)
    torch.cuda.synchronize()
    w = words.cpu().numpy()
    assert w[3] > w[1] and w[2] > w[0]
    mhz = 1e3 * float(w[2] - w[0]) / float(w[3] - w[1])
    assert 300.0 < mhz < 3000.0, mhz
    A, B = G.Particles.from_numpy(ptc), G.Particles(len(ptc["x1"]))
    na = torch.zeros(1, dtype=torch.int64, device="cuda")
    ctx.set_removed_counter(cnt[1:2])
    ctx.push_deposit_compact(A, B, f_t, ctx.zeros(3), dt, na)
    ctx.set_removed_counter(None)
    ctx.set_clock_probe(None)
    ctx.push_deposit(G.Particles.from_numpy(ptc), f_t, ctx.zeros(3), dt)       # no counter: nothing added
    torch.cuda.synchronize()
    assert cnt.cpu().tolist() == [n_gone, n_gone]
