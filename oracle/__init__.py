"""ctypes binding of the CPU oracle (oracle/grpic_oracle.cpp).

TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports
paper_2503_04558_b200 and the product never imports it.

All grid arrays are numpy float64 of shape [nth+1+2G, nr+1+2G] (the oracle's own
unpitched layout, see the header of grpic_oracle.cpp); `Grid.ij(i, j)` maps a logical
index to the array index.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "grpic_oracle.cpp")
_LIB = os.path.join(_HERE, "libgrpic_oracle.so")


def build(force=False):
    """Compile the oracle with g++ (-O2, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
             "-o", _LIB, _SRC])
    return _LIB


class Params(C.Structure):
    _fields_ = [("a", C.c_double), ("M", C.c_double), ("nr", C.c_int32), ("nth", C.c_int32),
                ("ng", C.c_int32), ("xi_in", C.c_double), ("xi_out", C.c_double),
                ("dphi", C.c_double), ("geo_iters", C.c_int32), ("field_iters", C.c_int32),
                ("beta_impl", C.c_double), ("damp_cells", C.c_int32), ("damp_coef", C.c_double)]


def make_params(d):
    """dict (as produced by the input generators) -> Params"""
    return Params(a=d["a"], M=d.get("M", 1.0), nr=d["nr"], nth=d["nth"], ng=d.get("ng", 2),
                  xi_in=d["xi_in"], xi_out=d["xi_out"], dphi=d.get("dphi", 2 * np.pi),
                  geo_iters=d.get("geo_iters", 3), field_iters=d.get("field_iters", 7),
                  beta_impl=d.get("beta_impl", 0.53), damp_cells=d.get("damp_cells", 0),
                  damp_coef=d.get("damp_coef", 0.0))


_lib = None
_dp = C.POINTER(C.c_double)
_up = C.POINTER(C.c_uint32)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_compact.restype = C.c_int64
        _lib.orc_pair_production.restype = C.c_int64
        _lib.orc_uniform.restype = C.c_double
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _d(a):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(_dp)


def _u(a):
    assert a.dtype == np.uint32 and a.flags.c_contiguous
    return a.ctypes.data_as(_up)


METRIC_NAMES = ["alpha", "beta_r", "g_rr", "g_thth", "g_phph", "g_rph", "gu_rr", "gu_thth",
                "gu_phph", "gu_rph", "sqrtg", "dr_alpha", "dth_alpha", "dr_beta", "dth_beta",
                "dr_gu_rr", "dth_gu_rr", "dr_gu_thth", "dth_gu_thth", "dr_gu_phph",
                "dth_gu_phph", "dr_gu_rph", "dth_gu_rph"]


def metric(a, M, r, th):
    out = np.zeros(23)
    lib().orc_metric(C.c_double(a), C.c_double(M), C.c_double(r), C.c_double(th), _d(out))
    return dict(zip(METRIC_NAMES, out))


def gauss_legendre(n):
    x, w = np.zeros(n), np.zeros(n)
    lib().orc_gauss_legendre(C.c_int(n), _d(x), _d(w))
    return x, w


class Grid:
    def __init__(self, p):
        self.p = p if isinstance(p, Params) else make_params(p)
        self.nr, self.nth, self.G = self.p.nr, self.p.nth, self.p.ng
        self.shape = (self.nth + 1 + 2 * self.G, self.nr + 1 + 2 * self.G)
        self.dxi = (self.p.xi_out - self.p.xi_in) / self.nr
        self.dth = np.pi / self.nth

    def ij(self, i, j):
        return (j + self.G, i + self.G)

    def zeros(self, n=1):
        return [np.zeros(self.shape) for _ in range(n)] if n > 1 else np.zeros(self.shape)


def areas(p):
    g = Grid(p)
    A = g.zeros(6)
    lib().orc_areas(C.byref(g.p), *[_d(x) for x in A])
    return dict(zip(["ADr", "ADth", "ADph", "ABr", "ABth", "ABph"], A))


def gather(p, fields, x1, x2):
    g = Grid(p)
    out = np.zeros(6)
    lib().orc_gather(C.byref(g.p), *[_d(f) for f in fields], C.c_double(x1), C.c_double(x2), _d(out))
    return out


def boris(a, M, r, th, u, D, B, sgn, dt):
    u, D, B = (np.ascontiguousarray(v, dtype=np.float64) for v in (u, D, B))
    out = np.zeros(3)
    lib().orc_boris(C.c_double(a), C.c_double(M), C.c_double(r), C.c_double(th), _d(u), _d(D),
                    _d(B), C.c_double(sgn), C.c_double(dt), _d(out))
    return out


def vay(a, M, r, th, u, D, B, sgn, dt):
    u, D, B = (np.ascontiguousarray(v, dtype=np.float64) for v in (u, D, B))
    out = np.zeros(3)
    lib().orc_vay(C.c_double(a), C.c_double(M), C.c_double(r), C.c_double(th), _d(u), _d(D),
                  _d(B), C.c_double(sgn), C.c_double(dt), _d(out))
    return out


class pusher:
    """context manager: `with oracle.pusher(1): ...` makes push() use the Vay update."""

    def __init__(self, which):
        self.which = which

    def __enter__(self):
        self.old = lib().orc_set_pusher(C.c_int(self.which))
        return self

    def __exit__(self, *a):
        lib().orc_set_pusher(C.c_int(self.old))


def geodesic_rhs(a, M, y, eps=1.0):
    y = np.ascontiguousarray(y, dtype=np.float64)
    f = np.zeros(6)
    lib().orc_geodesic_rhs(C.c_double(a), C.c_double(M), _d(y), C.c_double(eps), _d(f))
    return f


def geodesic(a, M, K, y, dt, eps=1.0):
    y = np.ascontiguousarray(y, dtype=np.float64)
    yn = np.zeros(6)
    lib().orc_geodesic(C.c_double(a), C.c_double(M), C.c_int(K), _d(y), C.c_double(dt),
                       C.c_double(eps), _d(yn))
    return yn


def geodesic_traj(a, M, K, y0, dt, nsteps, every=1, eps=1.0):
    y0 = np.ascontiguousarray(y0, dtype=np.float64)
    nrec = (nsteps + every - 1) // every
    traj = np.zeros((nrec, 6))
    lib().orc_geodesic_traj(C.c_double(a), C.c_double(M), C.c_int(K), _d(y0), C.c_double(dt),
                            C.c_double(eps), C.c_int64(nsteps), C.c_int64(every), _d(traj))
    return traj


def push(p, fields, ptc, dt):
    """ptc: dict of x1,x2,x3,u1,u2,u3 (f64), flag (u32).  Returns dict with the new state
    plus x2dep (un-reflected theta), cell, flag."""
    g = Grid(p)
    n = len(ptc["x1"])
    out = {k: np.zeros(n) for k in ("x1", "x2", "x3", "u1", "u2", "u3", "x2dep")}
    out["cell"] = np.zeros(n, dtype=np.uint32)
    out["flag"] = np.zeros(n, dtype=np.uint32)
    lib().orc_push(C.byref(g.p), *[_d(f) for f in fields], C.c_int64(n),
                   *[_d(ptc[k]) for k in ("x1", "x2", "x3", "u1", "u2", "u3")], _u(ptc["flag"]),
                   C.c_double(dt), *[_d(out[k]) for k in ("x1", "x2", "x3", "u1", "u2", "u3", "x2dep")],
                   _u(out["cell"]), _u(out["flag"]))
    return out


def deposit(p, old, new, w, dt, F=None):
    """Accumulate fluxes (F_r, F_th, F_ph) of the move old -> new (new['x2dep'] un-reflected)."""
    g = Grid(p)
    if F is None:
        F = g.zeros(3)
    n = len(old["x1"])
    lib().orc_deposit(C.byref(g.p), C.c_int64(n), _d(old["x1"]), _d(old["x2"]), _d(old["x3"]),
                      _d(new["x1"]), _d(new["x2dep"]), _d(new["x3"]), _d(w), _u(old["flag"]),
                      C.c_double(dt), *[_d(f) for f in F])
    return F


def finalize_current(p, F, filter_passes=0):
    g = Grid(p)
    lib().orc_finalize_current(C.byref(g.p), *[_d(f) for f in F], C.c_int(filter_passes))
    return F


def fold_current(p, F):
    g = Grid(p)
    lib().orc_fold_current(C.byref(g.p), *[_d(f) for f in F])
    return F


def rho(p, ptc, w, divide=True):
    g = Grid(p)
    out = g.zeros()
    lib().orc_rho(C.byref(g.p), C.c_int64(len(w)), _d(ptc["x1"]), _d(ptc["x2"]), _d(w),
                  _u(ptc["flag"]), C.c_int(1 if divide else 0), _d(out))
    return out


def apply_bc(p, fields):
    g = Grid(p)
    lib().orc_apply_bc(C.byref(g.p), *[_d(f) for f in fields])
    return fields


def circulation(p, fields):
    g = Grid(p)
    Cs = g.zeros(6)
    lib().orc_circulation(C.byref(g.p), *[_d(f) for f in fields], *[_d(c) for c in Cs])
    return Cs


def field_step(p, fields, J, dt, bg=None):
    """In-place update of fields (list of 6 arrays).  J: list of 3 arrays or None."""
    g = Grid(p)
    null = C.cast(None, _dp)
    Jp = [_d(j) for j in J] if J is not None else [null] * 3
    if bg is not None:
        arr = (_dp * 6)(*[_d(b) for b in bg])
        bgp = C.cast(arr, C.POINTER(_dp))
    else:
        bgp = C.cast(None, C.POINTER(_dp))
    lib().orc_field_step(C.byref(g.p), *[_d(f) for f in fields], *Jp, bgp, C.c_double(dt))
    return fields


def sort(cell, flag):
    n = len(cell)
    perm = np.zeros(n, dtype=np.uint32)
    lib().orc_sort(C.c_int64(n), _u(cell), _u(flag), _u(perm))
    return perm


def sort_interleaved(cell, flag, ncells, block_cells):
    n = len(cell)
    perm = np.zeros(n, dtype=np.uint32)
    lib().orc_sort_interleaved(C.c_int64(n), _u(cell), _u(flag), C.c_uint32(ncells), C.c_uint32(block_cells),
                               _u(perm))
    return perm


def compact(flag):
    n = len(flag)
    idx = np.zeros(n, dtype=np.uint32)
    c = lib().orc_compact(C.c_int64(n), _u(flag), _u(idx))
    return idx[:c].copy()


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def uniform(seed, step, index):
    return float(lib().orc_uniform(C.c_uint64(seed), C.c_uint32(step), C.c_uint64(index)))


def pair_production(p, ptc, capacity, gamma_thr, eps_ph, p_convert, seed, step):
    """one pass of the simplified pair production; returns (new particle
    dict of the new length, overflow flag).  Input dict is not modified."""
    n = len(ptc["x1"])
    out = {}
    for k, v in ptc.items():
        a = np.zeros(capacity, dtype=v.dtype)
        a[:n] = v
        out[k] = a
    ov = C.c_int32(0)
    m = lib().orc_pair_production(C.byref(make_params(p)), C.c_int64(n), C.c_int64(capacity),
                                  _d(out["x1"]), _d(out["x2"]), _d(out["x3"]), _d(out["u1"]), _d(out["u2"]),
                                  _d(out["u3"]), _d(out["w"]), _u(out["cell"]), _u(out["flag"]),
                                  C.c_double(gamma_thr), C.c_double(eps_ph), C.c_double(p_convert),
                                  C.c_uint64(seed), C.c_uint32(step), C.byref(ov))
    return {k: v[:m].copy() for k, v in out.items()}, bool(ov.value)


class shape_order:
    """context manager: `with oracle.shape_order(3): ...` runs gather, deposit and rho with the cubic
    B-spline shape ("third order spline ... through a configuration option")."""

    def __init__(self, order):
        self.order = order

    def __enter__(self):
        self.old = lib().orc_set_shape_order(C.c_int(self.order))
        return self

    def __exit__(self, *a):
        lib().orc_set_shape_order(C.c_int(self.old))


def shape(x):
    lib().orc_shape.restype = C.c_double
    return float(lib().orc_shape(C.c_double(x)))


def ks_to_bl(a, M, x1, th, ph, u, eps=1.0):
    """(E_inf, Gamma_FIDO, u_r^BL, phi_BL) of one Kerr-Schild particle state"""
    u = np.ascontiguousarray(u, dtype=np.float64)
    out = np.zeros(4)
    lib().orc_ks_to_bl(C.c_double(a), C.c_double(M), C.c_double(x1), C.c_double(th), C.c_double(ph), _d(u),
                       C.c_double(eps), _d(out))
    return out


def set_num_threads(n):
    """OpenMP threads of the oracle's parallel loops; returns the previous setting."""
    lib().orc_set_num_threads.restype = C.c_int
    return int(lib().orc_set_num_threads(C.c_int(int(n))))


def num_threads():
    return lib().orc_num_threads()
