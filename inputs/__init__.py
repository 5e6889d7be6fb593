"""Seeded synthetic inputs for the GRPIC hot path (numpy only).

This module is the ONE piece shared by the CUDA path's tests/bench and the CPU oracle's
tests: it only *produces inputs* (grid parameters, analytic initial fields of Appendix C,
particle positions/momenta drawn from numpy's PCG64) and holds none of the method's
push / deposit / field-update arithmetic.  It imports neither `oracle` nor the CUDA
binding.  The recipes follow SURVEY.md section 8(d) / DESIGN.md "Input recipe"; the paper
measures on no public dataset, its workloads are its own Wald / monopole setups
 and these inputs stand in for them.

Grid arrays are in the *logical layout*: float64 [nth+1+2G, nr+1+2G], r fastest,
logical index (i, j) at [j+G, i+G]; staggering as in Fig.1 / Appendix B of the paper:
  D^r, B^th : (i+1/2, j)    D^th, B^r : (i, j+1/2)    D^ph : (i, j)    B^ph : (i+1/2, j+1/2)
"""
import math

import numpy as np

FIELD_NAMES = ("Dr", "Dth", "Dph", "Br", "Bth", "Bph")
# (stagger in r, stagger in theta, parity under theta -> -theta)
STAGGER = {"Dr": (0.5, 0.0, +1), "Dth": (0.0, 0.5, -1), "Dph": (0.0, 0.0, +1),
           "Br": (0.0, 0.5, +1), "Bth": (0.5, 0.0, -1), "Bph": (0.5, 0.5, +1)}


# --------------------------------------------------------------------------- geometry
def kerr_schild(a, M, r, th):
    """Appendix A quantities needed to build initial conditions."""
    s, c = np.sin(th), np.cos(th)
    rho2 = r * r + a * a * c * c
    z = 2.0 * M * r / rho2
    out = dict(rho2=rho2, z=z, alpha=1.0 / np.sqrt(1.0 + z), beta_r=z / (1.0 + z),
               g_rr=1.0 + z, g_thth=rho2, g_rph=-a * s * s * (1.0 + z),
               g_phph=s * s * (rho2 + a * a * s * s * (1.0 + z)),
               gu_rr=(r * r + a * a) / rho2 - z / (1.0 + z), gu_thth=1.0 / rho2,
               gu_rph=a / rho2, sqrtg=rho2 * s * np.sqrt(1.0 + z))
    with np.errstate(divide="ignore"):
        out["gu_phph"] = 1.0 / (rho2 * s * s)
    return out


def grid_params(nr, nth, a, r_out=50.0, r_in=None, M=1.0, ng=2, **kw):
    """Grid law of BASELINE.json: log-spaced r from 0.9 r_horizon to r_out, uniform theta."""
    if r_in is None:
        r_in = 0.9 * (M + math.sqrt(M * M - a * a))
    p = dict(a=float(a), M=float(M), nr=int(nr), nth=int(nth), ng=int(ng),
             xi_in=math.log(r_in), xi_out=math.log(r_out), dphi=2.0 * math.pi,
             geo_iters=3, field_iters=7, beta_impl=0.53, damp_cells=0, damp_coef=0.0)
    p.update(kw)
    return p


def grid_shape(p):
    return (p["nth"] + 1 + 2 * p["ng"], p["nr"] + 1 + 2 * p["ng"])


def spacing(p):
    return (p["xi_out"] - p["xi_in"]) / p["nr"], math.pi / p["nth"]


def courant_dt(p, factor=0.5):
    """Reading G16: dt_CFL = min over cell centres of
    [((alpha sqrt(g^rr) + beta^r)/(r dxi))^2 + (alpha sqrt(g^thth)/dth)^2]^(-1/2)."""
    dxi, dth = spacing(p)
    r = np.exp(p["xi_in"] + (np.arange(p["nr"]) + 0.5) * dxi)[None, :]
    th = ((np.arange(p["nth"]) + 0.5) * dth)[:, None]
    m = kerr_schild(p["a"], p["M"], r, th)
    vr = (m["alpha"] * np.sqrt(m["gu_rr"]) + m["beta_r"]) / (r * dxi)
    vt = m["alpha"] * np.sqrt(m["gu_thth"]) / dth
    return factor * float(np.min(1.0 / np.sqrt(vr * vr + vt * vt)))


def positions(p, name):
    """(r, theta) meshes of the stored lattice of component `name`, full padded shape."""
    G = p["ng"]
    dxi, dth = spacing(p)
    sr, sth, _ = STAGGER[name]
    i = np.arange(-G, p["nr"] + G + 1) + sr
    j = np.arange(-G, p["nth"] + G + 1) + sth
    return np.exp(p["xi_in"] + i * dxi)[None, :], (j * dth)[:, None]


# --------------------------------------------------------------------------- fields
def _wald(a, M, B0, r, th):
    """Appendix C (C14)-(C19), PAPER.md:534-544 (M = 1 in the paper's formulas)."""
    s, c = np.sin(th), np.cos(th)
    rho2 = r * r + a * a * c * c
    Delta = r * r + a * a - 2.0 * r
    sg = kerr_schild(a, M, r, th)["sqrtg"]
    with np.errstate(divide="ignore", invalid="ignore"):
        Br = B0 / sg * (Delta + 2.0 * r * (r ** 4 - a ** 4) / rho2 ** 2) * s * c
        Bth = -B0 / sg * (r + a * a * (1.0 + c * c) * (2.0 * r * r - rho2) / rho2 ** 2) * s * s
        Bph = -B0 / sg * (2.0 * a * r * (a * a - r * r) / rho2 ** 2 - a) * s * c
    Er = B0 * a * (1.0 + c * c) * (a * a * c * c - r * r) / rho2 ** 2
    Eth = B0 * 2.0 * a * r * (a * a - r * r) / rho2 ** 2 * s * c
    return Br, Bth, Bph, Er, Eth, np.zeros_like(Er)


def _monopole(a, M, B0, r, th):
    """Appendix C (C21)-(C26)."""
    s, c = np.sin(th), np.cos(th)
    rho2 = r * r + a * a * c * c
    sg = kerr_schild(a, M, r, th)["sqrtg"]
    with np.errstate(divide="ignore", invalid="ignore"):
        Br = B0 / sg * (a * a + r * r) * (r * r - a * a * c * c) * s / rho2 ** 2
        Bth = -B0 / sg * 2.0 * a * a * r * s * s * c / rho2 ** 2
        Bph = B0 / sg * a * (r * r - a * a * c * c) * s / rho2 ** 2
    Er = -B0 * 2.0 * a * r * c / rho2 ** 2
    Eth = -B0 * a * (r * r - a * a * c * c) * s / rho2 ** 2
    return Br, Bth, Bph, Er, Eth, np.zeros_like(Er)


def _wald_nonrotating(a, M, B0, r, th):
    """Eq.(25), PAPER.md:315-317 (reading G6): the a = 0 Wald potential A_phi = (B0/2) gamma_phiphi
    placed in the spinning metric: B^r = d_theta A_phi / sqrt(gamma), B^theta = -d_r A_phi / sqrt(gamma),
    B^phi = 0, E_i = 0 (initial state of the vacuum relaxation test, Section 3.2)."""
    s, c = np.sin(th), np.cos(th)
    rho2 = r * r + a * a * c * c
    F = rho2 + a * a * s * s + 2.0 * M * r * a * a * s * s / rho2          # gamma_phiphi = s^2 F
    dFr = 2.0 * r + 2.0 * M * a * a * s * s * (rho2 - 2.0 * r * r) / rho2 ** 2
    dFt = 4.0 * M * r * a * a * s * c * (r * r + a * a) / rho2 ** 2
    sg = kerr_schild(a, M, r, th)["sqrtg"]
    with np.errstate(divide="ignore", invalid="ignore"):
        Br = 0.5 * B0 * (2.0 * s * c * F + s * s * dFt) / sg
        Bth = -0.5 * B0 * s * s * dFr / sg
    z = np.zeros_like(Br)
    return Br, Bth, z, z, z, z


def analytic_DB(a, M, B0, r, th, kind):
    """Contravariant D^i, B^i at points (r, th) from the analytic E_i, B^i through Eq.(6)
    (PAPER.md:84): alpha D_i = E_i - e_ijk beta^j B^k, D^i = gamma^ij D_j."""
    r, th = np.broadcast_arrays(np.asarray(r, dtype=np.float64), np.asarray(th, dtype=np.float64))
    fn = {"wald": _wald, "monopole": _monopole, "wald0": _wald_nonrotating}[kind]
    Br, Bth, Bph, Er, Eth, Eph = fn(a, M, B0, r, th)
    m = kerr_schild(a, M, r, th)
    e_r = Er
    e_th = Eth + m["sqrtg"] * m["beta_r"] * Bph
    e_ph = Eph - m["sqrtg"] * m["beta_r"] * Bth
    with np.errstate(divide="ignore", invalid="ignore"):
        Dr = (m["gu_rr"] * e_r + m["gu_rph"] * e_ph) / m["alpha"]
        Dth = m["gu_thth"] * e_th / m["alpha"]
        Dph = (m["gu_rph"] * e_r + m["gu_phph"] * e_ph) / m["alpha"]
    return Dr, Dth, Dph, Br, Bth, Bph


def fill_guards(p, fields):
    """Make stored guard values consistent: axis-node D^ph = B^th = 0, radial guards =
    copy of the last physical value, theta ghost rows by parity."""
    G, nr, nth = p["ng"], p["nr"], p["nth"]
    out = []
    for name, F in zip(FIELD_NAMES, fields):
        F = F.copy()
        sr, sth, par = STAGGER[name]
        ihi = nr if sr == 0.0 else nr - 1
        jhi = nth if sth == 0.0 else nth - 1
        if name in ("Dph", "Bth"):
            F[G, :] = 0.0
            F[G + nth, :] = 0.0
        F[:, :G] = F[:, G:G + 1]
        F[:, G + ihi + 1:] = F[:, G + ihi:G + ihi + 1]
        for g in range(1, G + 1):
            if sth == 0.0:
                F[G - g, :] = par * F[G + g, :]
                F[G + nth + g, :] = par * F[G + nth - g, :]
            else:
                F[G - g, :] = par * F[G + g - 1, :]
                F[G + nth - 1 + g, :] = par * F[G + nth - g, :]
        if sth != 0.0:   # last stored row of a half-staggered component: mirror of row nth-1-G
            F[G + nth + G, :] = par * F[nth - 1, :]
        out.append(F)
    return out


def analytic_fields(p, kind, B0=1.0):
    """Six stored arrays sampled pointwise from the analytic solution `kind` in
    {"wald", "monopole"} at each component's own staggered position."""
    fields = []
    for k, name in enumerate(FIELD_NAMES):
        r, th = positions(p, name)
        F = analytic_DB(p["a"], p["M"], B0, r, th, kind)[k]
        F = np.where(np.isfinite(F), F, 0.0)
        fields.append(np.ascontiguousarray(np.broadcast_to(F, grid_shape(p)).astype(np.float64)))
    return fill_guards(p, fields)


def split_monopole_fields(p, B0=1.0):
    """Config 1 field: B^r = B0 sin(theta)/sqrt(gamma), everything else zero."""
    fields = [np.zeros(grid_shape(p)) for _ in range(6)]
    r, th = positions(p, "Br")
    sg = kerr_schild(p["a"], p["M"], r, th)["sqrtg"]
    with np.errstate(divide="ignore", invalid="ignore"):
        Br = B0 * np.sin(th) / sg
    fields[3] = np.ascontiguousarray(np.where(np.isfinite(Br), Br, 0.0) * np.ones(grid_shape(p)))
    return fill_guards(p, fields)


def perturb(fields, rel, rng):
    """each stored value x (1 + rel * U(-1,1))   (config 2)"""
    return [F * (1.0 + rel * rng.uniform(-1.0, 1.0, size=F.shape)) for F in fields]


def gaussian_packet_Bph(p, amp=1e-2, width=2.0, r0=10.0):
    """Config 4 perturbation: dB^ph = amp exp(-d^2/(2 width^2))/sqrt(g_phph),
    d^2 = r^2 + r0^2 - 2 r r0 sin(theta)."""
    r, th = positions(p, "Bph")
    d2 = r * r + r0 * r0 - 2.0 * r * r0 * np.sin(th)
    gpp = kerr_schild(p["a"], p["M"], r, th)["g_phph"]
    with np.errstate(divide="ignore", invalid="ignore"):
        dB = amp * np.exp(-d2 / (2.0 * width * width)) / np.sqrt(gpp)
    return np.where(np.isfinite(dB), dB, 0.0)


def random_current(p, rng, amp=1e-3):
    """Config 4: prescribed J^i iid U(-amp, amp) per stored value (constant in time)."""
    return [rng.uniform(-amp, amp, size=grid_shape(p)) for _ in range(3)]


# --------------------------------------------------------------------------- particles
def _isotropic(n, rng):
    mu = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2.0 * np.pi, n)
    st = np.sqrt(1.0 - mu * mu)
    return st * np.cos(ph), st * np.sin(ph), mu


def _maxwell_juttner_u(n, theta, rng):
    """|u| with f(u) du ~ u^2 exp(-sqrt(1+u^2)/theta) du by tabulated inverse CDF."""
    umax = 40.0 * theta + 12.0 * math.sqrt(theta) + 1.0
    u = np.linspace(0.0, umax, 200001)
    f = u * u * np.exp(-(np.sqrt(1.0 + u * u) - 1.0) / theta)
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (f[1:] + f[:-1]) * np.diff(u))])
    cdf /= cdf[-1]
    return np.interp(rng.uniform(0.0, 1.0, n), cdf, u)


def momenta(p, r, th, umag, rng):
    """Isotropic in the local orthonormal Kerr-Schild FIDO triad with magnitude umag,
    converted to covariant components: u_r = u1/sqrt(g^rr) + u3 g_rph/sqrt(g_phph),
    u_th = sqrt(g_thth) u2, u_ph = sqrt(g_phph) u3, so that g^ij u_i u_j = |u|^2."""
    n1, n2, n3 = _isotropic(len(r), rng)
    m = kerr_schild(p["a"], p["M"], r, th)
    sq = np.sqrt(m["g_phph"])
    u1 = umag * n1 / np.sqrt(m["gu_rr"]) + umag * n3 * m["g_rph"] / sq
    u2 = np.sqrt(m["g_thth"]) * umag * n2
    u3 = sq * umag * n3
    return u1, u2, u3


def cells_of(p, x1, x2):
    dxi, dth = spacing(p)
    i = np.clip(np.floor((x1 - p["xi_in"]) / dxi).astype(np.int64), 0, p["nr"] - 1)
    j = np.clip(np.floor(x2 / dth).astype(np.int64), 0, p["nth"] - 1)
    return (j * p["nr"] + i).astype(np.uint32)


def make_particles(p, n, seed, position="logical", momentum=("loguniform", 0.1, 10.0),
                   pairs=False):
    """Seeded particle set.
    position: "logical"  - (xi, theta) iid uniform on the logical domain       (config 1)
              "r2"       - r uniform in [r_in, r_out], cos(theta) uniform (n ~ r^-2) (configs 2, 5)
              "crowded"  - 70% xi uniform in [xi_in, ln 3], 30% r uniform in [3, r_out] (config 3)
    momentum: ("loguniform", lo, hi) | ("mj", Theta) | ("mj_tail", Theta, frac, g1, g2)
    pairs:    n is the number of PARTICLES; if True, e-/e+ are co-located pairwise.
    Returns dict of x1 (= ln r), x2, x3, u1, u2, u3, w (f64), flag, cell (u32)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    npos = n // 2 if pairs else n
    r_in, r_out = math.exp(p["xi_in"]), math.exp(p["xi_out"])
    eps = 1e-9
    if position == "logical":
        x1 = rng.uniform(p["xi_in"], p["xi_out"], npos)
        x2 = rng.uniform(0.0, np.pi, npos)
    elif position == "r2":
        x1 = np.log(rng.uniform(r_in, r_out, npos))
        x2 = np.arccos(rng.uniform(-1.0, 1.0, npos))
    elif position == "crowded":
        near = rng.uniform(0.0, 1.0, npos) < 0.7
        xi_a = rng.uniform(p["xi_in"], math.log(3.0), npos)
        xi_b = np.log(rng.uniform(3.0, r_out, npos))
        x1 = np.where(near, xi_a, xi_b)
        x2 = np.arccos(rng.uniform(-1.0, 1.0, npos))
    else:
        raise ValueError(position)
    x1 = np.clip(x1, p["xi_in"] + eps, p["xi_out"] - eps)
    x2 = np.clip(x2, eps, np.pi - eps)
    if pairs:
        x1, x2 = np.repeat(x1, 2), np.repeat(x2, 2)
    n = len(x1)
    x3 = rng.uniform(0.0, 2.0 * np.pi, n)
    kind = momentum[0]
    if kind == "loguniform":
        umag = np.exp(rng.uniform(math.log(momentum[1]), math.log(momentum[2]), n))
    elif kind == "mj":
        umag = _maxwell_juttner_u(n, momentum[1], rng)
    elif kind == "mj_tail":
        _, theta, frac, g1, g2 = momentum
        umag = _maxwell_juttner_u(n, theta, rng)
        tail = rng.uniform(0.0, 1.0, n) < frac
        X = rng.uniform(0.0, 1.0, n)
        gam = 1.0 / (1.0 / g1 - X * (1.0 / g1 - 1.0 / g2))   # dN/dgamma ~ gamma^-2
        umag = np.where(tail, np.sqrt(gam * gam - 1.0), umag)
    else:
        raise ValueError(kind)
    u1, u2, u3 = momenta(p, np.exp(x1), x2, umag, rng)
    flag = (np.arange(n) % 2).astype(np.uint32)          # alternate e-, e+
    ptc = dict(x1=x1, x2=x2, x3=x3, u1=u1, u2=u2, u3=u3, w=np.ones(n),
               flag=flag, cell=cells_of(p, x1, x2))
    return {k: np.ascontiguousarray(v) for k, v in ptc.items()}


# --------------------------------------------------------------------------- configs
def config(k, scale=1.0, nr=None, nth=None, n=None, ng=2):
    """The five BASELINE.json configs (k = 1..5); `nr`, `nth`, `n` override the size for
    reduced-size parity tests (the recipe is otherwise unchanged); `ng` = guard nodes (3 for the
    cubic-spline shape).
    Returns dict(params, dt, fields, particles, J, bg, meta)."""
    out = dict(J=None, bg=None, particles=None)
    if k == 1:
        p = grid_params(nr or 128, nth or 128, 0.99, ng=ng)
        out.update(params=p, dt=courant_dt(p), fields=split_monopole_fields(p),
                   particles=make_particles(p, n or 100_000, 0, "logical", ("loguniform", 0.1, 10.0)),
                   meta=dict(steps=10, sort_every=0, filter_passes=0, field=True))
    elif k == 2:
        p = grid_params(nr or 1024, nth or 1024, 0.99, ng=ng)
        rng = np.random.Generator(np.random.PCG64(1001))
        out.update(params=p, dt=courant_dt(p),
                   fields=fill_guards(p, perturb(analytic_fields(p, "wald"), 1e-3, rng)),
                   particles=make_particles(p, n or 20_000_000, 1, "r2",
                                            ("mj_tail", 1.0, 0.1, 10.0, 1e4), pairs=True),
                   meta=dict(steps=100, sort_every=20, filter_passes=0, field=False))
    elif k == 3:
        p = grid_params(nr or 2048, nth or 2048, 0.99, ng=ng)
        rng = np.random.Generator(np.random.PCG64(1002))
        out.update(params=p, dt=courant_dt(p),
                   fields=fill_guards(p, perturb(analytic_fields(p, "wald"), 1e-3, rng)),
                   particles=make_particles(p, n or 100_000_000, 2, "crowded",
                                            ("loguniform", 0.1, 1e5)),
                   meta=dict(steps=50, sort_every=0, compact_every=1, filter_passes=0, field=False))
    elif k == 4:
        p = grid_params(nr or 4096, nth or 4096, 0.9, ng=ng)
        p["damp_cells"] = p["nr"] // 10
        p["damp_coef"] = 1.0
        rng = np.random.Generator(np.random.PCG64(3))
        bg = analytic_fields(p, "monopole")
        f = [b.copy() for b in bg]
        f[5] = f[5] + gaussian_packet_Bph(p)
        out.update(params=p, dt=courant_dt(p), fields=fill_guards(p, f), bg=bg,
                   J=random_current(p, rng),
                   meta=dict(steps=1000, sort_every=0, filter_passes=0, field=True))
    elif k == 5:
        p = grid_params(nr or 2048, nth or 2048, 0.99, ng=ng)
        out.update(params=p, dt=courant_dt(p), fields=analytic_fields(p, "monopole"),
                   particles=make_particles(p, n or 200_000_000, 4, "r2", ("mj", 0.1)),
                   meta=dict(steps=200, sort_every=10, filter_passes=3, field=True))
    else:
        raise ValueError(k)
    return out
