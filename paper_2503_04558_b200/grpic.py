"""Thin ctypes binding of libgrpic.so (include/grpic.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library; PyTorch is used here
for device memory and streams only.  There is no CPU fallback: if the library is not built
or no CUDA device is present the calls raise.
"""
import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

_dp = C.POINTER(C.c_double)
_up = C.POINTER(C.c_uint32)


class GrpicError(RuntimeError):
    pass


class Params(C.Structure):
    _fields_ = [("a", C.c_double), ("M", C.c_double), ("nr", C.c_int32), ("nth", C.c_int32),
                ("ng", C.c_int32), ("xi_in", C.c_double), ("xi_out", C.c_double),
                ("dphi", C.c_double), ("geo_iters", C.c_int32), ("field_iters", C.c_int32),
                ("beta_impl", C.c_double), ("damp_cells", C.c_int32), ("damp_coef", C.c_double)]


class ParticlesC(C.Structure):
    _fields_ = [(k, _dp) for k in ("x1", "x2", "x3", "u1", "u2", "u3", "w")] + \
               [("cell", _up), ("flag", _up), ("n", C.c_int64)]


class PairParamsC(C.Structure):
    _fields_ = [("gamma_thr", C.c_double), ("eps_ph", C.c_double), ("p_convert", C.c_double),
                ("seed", C.c_uint64), ("step", C.c_uint32)]


class FieldsC(C.Structure):
    _fields_ = [(k, _dp) for k in ("Dr", "Dth", "Dph", "Br", "Bth", "Bph")]


class CurrentC(C.Structure):
    _fields_ = [(k, _dp) for k in ("Fr", "Fth", "Fph")]


EXPORTS = ["grpic_create", "grpic_destroy", "grpic_grid_layout", "grpic_get_areas",
           "grpic_workspace_bytes", "grpic_set_workspace", "grpic_set_removed_counter", "grpic_set_flux_exchange", "grpic_push_deposit",
           "grpic_push_deposit_compact", "grpic_step_host", "grpic_pair_production", "grpic_push_deposit_spline3", "grpic_push_deposit_variant",
           "grpic_finalize_current", "grpic_field_step", "grpic_fill_guards",
           "grpic_circulation", "grpic_ks_to_bl", "grpic_sort", "grpic_sort_interleaved", "grpic_compact", "grpic_compact_static", "grpic_deposit_rho",
           "grpic_measure_fp64_peak", "grpic_measure_fp64_peak_clocked", "grpic_set_clock_probe", "grpic_kernel_launches", "grpic_strerror"]

_lib = None


def library_path():
    return _build.LIB


def load(build_if_missing=True):
    """dlopen libgrpic.so (building it in-tree with nvcc first if it is missing/stale)."""
    global _lib
    if _lib is None:
        if build_if_missing:
            _build.build()
        if not os.path.exists(_build.LIB):
            raise GrpicError("libgrpic.so is not built: run `python -m paper_2503_04558_b200.build`")
        lib = C.CDLL(_build.LIB)
        for name in EXPORTS:
            getattr(lib, name)          # raises AttributeError if a declared symbol is missing
        lib.grpic_workspace_bytes.restype = C.c_size_t
        lib.grpic_workspace_bytes.argtypes = [C.c_void_p, C.c_int64]
        lib.grpic_strerror.restype = C.c_char_p
        lib.grpic_kernel_launches.restype = C.c_int64
        lib.grpic_create.argtypes = [C.POINTER(Params), C.POINTER(C.c_void_p)]
        _lib = lib
    return _lib


def _check(rc):
    if rc != 0:
        raise GrpicError("grpic error %d: %s" % (rc, load().grpic_strerror(rc).decode()))


def _ptr(t, ctype=_dp):
    return C.cast(C.c_void_p(t.data_ptr()), ctype)


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


PTC_F64 = ("x1", "x2", "x3", "u1", "u2", "u3", "w")
PTC_U32 = ("cell", "flag")


class Particles:
    """SoA particle store on the device (torch tensors; uint32 stored as int32 bit patterns)."""

    def __init__(self, n, device="cuda"):
        self.n = int(n)
        self.t = {k: torch.empty(self.n, dtype=torch.float64, device=device) for k in PTC_F64}
        self.t.update({k: torch.empty(self.n, dtype=torch.int32, device=device) for k in PTC_U32})

    @classmethod
    def from_numpy(cls, d, device="cuda"):
        p = cls(len(d["x1"]), device)
        p.upload(d)
        return p

    def upload(self, d, non_blocking=False):
        for k in PTC_F64:
            self.t[k].copy_(torch.from_numpy(d[k]) if isinstance(d[k], np.ndarray) else d[k],
                            non_blocking=non_blocking)
        for k in PTC_U32:
            src = torch.from_numpy(d[k].view(np.int32)) if isinstance(d[k], np.ndarray) else d[k]
            self.t[k].copy_(src, non_blocking=non_blocking)

    def to_numpy(self, n=None):
        n = self.n if n is None else n
        out = {k: self.t[k][:n].cpu().numpy() for k in PTC_F64}
        out.update({k: self.t[k][:n].cpu().numpy().view(np.uint32) for k in PTC_U32})
        return out

    def struct(self):
        s = ParticlesC()
        for k in PTC_F64:
            setattr(s, k, _ptr(self.t[k]))
        for k in PTC_U32:
            setattr(s, k, _ptr(self.t[k], _up))
        s.n = self.n
        return s


class Context:
    """grpic_ctx + the device arrays' layout helpers."""

    def __init__(self, params, n_particles=0):
        if not torch.cuda.is_available():
            raise GrpicError("no CUDA device: libgrpic has no CPU fallback")
        lib = load()
        self.params = dict(params)
        d = self.params
        self.p = Params(a=d["a"], M=d.get("M", 1.0), nr=d["nr"], nth=d["nth"], ng=d.get("ng", 2),
                        xi_in=d["xi_in"], xi_out=d["xi_out"], dphi=d.get("dphi", 2 * np.pi),
                        geo_iters=d.get("geo_iters", 3), field_iters=d.get("field_iters", 7),
                        beta_impl=d.get("beta_impl", 0.53), damp_cells=d.get("damp_cells", 0),
                        damp_coef=d.get("damp_coef", 0.0))
        self.h = C.c_void_p()
        _check(lib.grpic_create(C.byref(self.p), C.byref(self.h)))
        pitch, rows, i0, j0 = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32()
        _check(lib.grpic_grid_layout(self.h, C.byref(pitch), C.byref(rows), C.byref(i0), C.byref(j0)))
        self.pitch, self.rows, self.i0, self.j0 = pitch.value, rows.value, i0.value, j0.value
        self.ng, self.nr, self.nth = self.p.ng, self.p.nr, self.p.nth
        self.ws = None
        self.status = torch.zeros(1, dtype=torch.int32, device="cuda")
        self.reserve(n_particles)

    def reserve(self, n_particles):
        nbytes = load().grpic_workspace_bytes(self.h, int(n_particles))
        if self.ws is None or self.ws.numel() < nbytes:
            self.ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
            off = (-self.ws.data_ptr()) % 256
            _check(load().grpic_set_workspace(self.h, C.c_void_p(self.ws.data_ptr() + off),
                                              C.c_size_t(nbytes)))

    def set_removed_counter(self, counter):
        """counter: uint64/int64 device tensor of one element (or None): every push adds the number of
        particles it flags removed."""
        self._removed = counter          # keep the tensor alive while the library holds its pointer
        ptr = C.c_void_p(counter.data_ptr()) if counter is not None else None
        _check(load().grpic_set_removed_counter(self.h, ptr))

    def set_flux_exchange(self, fn):
        """fn(flux_block) or None.  flux_block: torch view [3, rows, pitch] of the context's own flux
        arrays inside grpic_step_host; fn must sum it over the ranks in stream order (e.g.
        torch.distributed.all_reduce on the current stream)."""
        if fn is None:
            self._fx_cb = None
            _check(load().grpic_set_flux_exchange(self.h, None, None))
            return
        rows, pitch = self.rows, self.pitch

        class _Dev:                                   # raw device pointer -> torch tensor, no copy
            def __init__(self, ptr, n):
                self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (ptr, False), "version": 2}

        def cb(user, ptr, n, stream):
            try:
                t = torch.as_tensor(_Dev(ptr, int(n)), device="cuda").view(3, rows, pitch)
                fn(t)
                return 0
            except Exception:                          # never let an exception cross the C boundary
                return 1
        proto = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p)
        self._fx_cb = proto(cb)                        # keep the thunk alive
        _check(load().grpic_set_flux_exchange(self.h, self._fx_cb, None))

    def close(self):
        if self.h:
            load().grpic_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- grid arrays: logical numpy [nth+1+2G, nr+1+2G]  <->  pitched device tensor ----
    def zeros(self, n=1):
        z = [torch.zeros(self.rows, self.pitch, dtype=torch.float64, device="cuda") for _ in range(n)]
        return z if n > 1 else z[0]

    def zeros_block(self, n):
        """n grid arrays in ONE contiguous allocation [n, rows, pitch] (block[k] is array k): the
        three flux arrays of a multi-GPU run are summed over ranks with a single all-reduce."""
        return torch.zeros(n, self.rows, self.pitch, dtype=torch.float64, device="cuda")

    def to_device(self, arr):
        t = torch.zeros(self.rows, self.pitch, dtype=torch.float64, device="cuda")
        G = self.ng
        t[self.j0 - G:self.j0 - G + arr.shape[0], self.i0 - G:self.i0 - G + arr.shape[1]] = \
            torch.from_numpy(np.ascontiguousarray(arr)).cuda()
        return t

    def to_host(self, t):
        G = self.ng
        return t[self.j0 - G:self.j0 + self.nth + G + 1, self.i0 - G:self.i0 + self.nr + G + 1] \
            .contiguous().cpu().numpy()

    @staticmethod
    def _fields(f):
        s = FieldsC()
        for k, t in zip(("Dr", "Dth", "Dph", "Br", "Bth", "Bph"), f):
            setattr(s, k, _ptr(t))
        return s

    @staticmethod
    def _current(J):
        s = CurrentC()
        for k, t in zip(("Fr", "Fth", "Fph"), J):
            setattr(s, k, _ptr(t))
        return s

    # ---- the C-ABI calls (same names as include/grpic.h, without the prefix) ----
    def get_areas(self):
        out = self.zeros(6)
        arr = (_dp * 6)(*[_ptr(t) for t in out])
        _check(load().grpic_get_areas(self.h, arr, _stream()))
        return out

    def push_deposit(self, ptc, fields, flux, dt):
        ps, fs, js = ptc.struct(), self._fields(fields), self._current(flux)
        _check(load().grpic_push_deposit(self.h, C.byref(ps), C.byref(fs), C.byref(js),
                                         C.c_double(dt), _ptr(self.status, _up), _stream()))

    def push_deposit_spline3(self, ptc, fields, flux, dt):
        ps, fs, js = ptc.struct(), self._fields(fields), self._current(flux)
        _check(load().grpic_push_deposit_spline3(self.h, C.byref(ps), C.byref(fs), C.byref(js),
                                                 C.c_double(dt), _ptr(self.status, _up), _stream()))

    def push_deposit_variant(self, ptc, fields, flux, dt, shape_order=1, pusher=0):
        ps, fs, js = ptc.struct(), self._fields(fields), self._current(flux)
        _check(load().grpic_push_deposit_variant(self.h, C.byref(ps), C.byref(fs), C.byref(js), C.c_double(dt),
                                                 C.c_int32(shape_order), C.c_int32(pusher),
                                                 _ptr(self.status, _up), _stream()))

    def push_deposit_compact(self, src, dst, fields, flux, dt, n_alive):
        """compact(src -> dst) fused with push_deposit(dst); n_alive: int64 device tensor (1)."""
        self.reserve(src.n)
        a, b, fs, js = src.struct(), dst.struct(), self._fields(fields), self._current(flux)
        _check(load().grpic_push_deposit_compact(
            self.h, C.byref(a), C.byref(b), C.byref(fs), C.byref(js), C.c_double(dt),
            C.cast(C.c_void_p(n_alive.data_ptr()), C.POINTER(C.c_int64)), _ptr(self.status, _up), _stream()))
        dst.n = src.n

    def step_host(self, host, fields, dt, host_J=None, background=None, filter_passes=0, chunk=0):
        """grpic_step_host: `host` = dict of (pinned) CPU torch tensors x1..u3, w, cell, flag and
        "n" (int); updated in place, returns the survivor count."""
        self.reserve(min(int(host["n"]), chunk or (4 << 20)))
        ps = ParticlesC()
        for k in PTC_F64:
            setattr(ps, k, _ptr(host[k]))
        for k in PTC_U32:
            setattr(ps, k, _ptr(host[k], _up))
        ps.n = int(host["n"])
        fs = self._fields(fields)
        bp = C.byref(self._fields(background)) if background is not None else None
        jp = C.byref(self._current(host_J)) if host_J is not None else None
        st = C.c_uint32(0)
        _check(load().grpic_step_host(self.h, C.byref(ps), C.byref(fs), bp, jp, C.c_double(dt),
                                      C.c_int32(filter_passes), C.c_int64(chunk), C.byref(st), _stream()))
        host["n"] = int(ps.n)
        self.last_host_status = st.value
        return int(ps.n)

    def pair_production(self, ptc, n, n_new, gamma_thr, eps_ph, p_convert, seed, step):
        """grpic_pair_production on the first n entries of `ptc` (capacity = ptc.n);
        n_new: int64 device tensor (1)."""
        self.reserve(ptc.n)
        ps = ptc.struct()
        ps.n = int(n)
        pp = PairParamsC(gamma_thr=gamma_thr, eps_ph=eps_ph, p_convert=p_convert, seed=seed, step=step)
        _check(load().grpic_pair_production(
            self.h, C.byref(ps), C.c_int64(ptc.n), C.byref(pp),
            C.cast(C.c_void_p(n_new.data_ptr()), C.POINTER(C.c_int64)), _ptr(self.status, _up), _stream()))

    def finalize_current(self, flux, filter_passes=0):
        js = self._current(flux)
        _check(load().grpic_finalize_current(self.h, C.byref(js), C.c_int32(filter_passes), _stream()))

    def field_step(self, fields, J, dt, background=None):
        fs = self._fields(fields)
        jp = C.byref(self._current(J)) if J is not None else None
        bp = C.byref(self._fields(background)) if background is not None else None
        _check(load().grpic_field_step(self.h, C.byref(fs), jp, bp, C.c_double(dt), _stream()))

    def fill_guards(self, fields):
        fs = self._fields(fields)
        _check(load().grpic_fill_guards(self.h, C.byref(fs), _stream()))

    def circulation(self, fields):
        out = self.zeros(6)
        fs = self._fields(fields)
        arr = (_dp * 6)(*[_ptr(t) for t in out])
        _check(load().grpic_circulation(self.h, C.byref(fs), arr, _stream()))
        return out

    def sort(self, src, dst, perm=None):
        self.reserve(src.n)
        a, b = src.struct(), dst.struct()
        pp = _ptr(perm, _up) if perm is not None else None
        _check(load().grpic_sort(self.h, C.byref(a), C.byref(b), pp, _stream()))
        dst.n = src.n

    def sort_interleaved(self, src, dst, block_cells=8, perm=None):
        self.reserve(src.n)
        a, b = src.struct(), dst.struct()
        pp = _ptr(perm, _up) if perm is not None else None
        _check(load().grpic_sort_interleaved(self.h, C.byref(a), C.byref(b), pp, C.c_int32(block_cells), _stream()))
        dst.n = src.n

    def compact(self, src, dst, n_alive):
        """n_alive: int64 device tensor of one element (written asynchronously)."""
        self.reserve(src.n)
        a, b = src.struct(), dst.struct()
        _check(load().grpic_compact(self.h, C.byref(a), C.byref(b),
                                    C.cast(C.c_void_p(n_alive.data_ptr()), C.POINTER(C.c_int64)), _stream()))
        dst.n = src.n

    COMPACT_STATIC_MAX_PARTICLES = 1 << 26

    def compact_static(self, src, dst, n_alive):
        """grpic_compact without a workspace or any allocation (scratch in a static device array of the
        library; at most COMPACT_STATIC_MAX_PARTICLES particles; calls must not overlap on the GPU)."""
        a, b = src.struct(), dst.struct()
        _check(load().grpic_compact_static(self.h, C.byref(a), C.byref(b),
                                           C.cast(C.c_void_p(n_alive.data_ptr()), C.POINTER(C.c_int64)), _stream()))
        dst.n = src.n

    def ks_to_bl(self, ptc):
        """(E_inf, gamma_fido, ur_bl, phi_bl): four float64 device tensors of length ptc.n"""
        out = [torch.empty(max(ptc.n, 1), dtype=torch.float64, device="cuda") for _ in range(4)]
        ps = ptc.struct()
        _check(load().grpic_ks_to_bl(self.h, C.byref(ps), *[_ptr(t) for t in out], _stream()))
        return [t[:ptc.n] for t in out]

    def set_clock_probe(self, words):
        """words: int64 device tensor of 4 elements (or None), see grpic_set_clock_probe"""
        self._clk = words
        _check(load().grpic_set_clock_probe(self.h, C.c_void_p(words.data_ptr()) if words is not None else None))

    def measure_fp64_peak_clocked(self):
        """(FP64 instructions per second, SM clock in MHz during the probe)"""
        v, c = C.c_double(0.0), C.c_double(0.0)
        _check(load().grpic_measure_fp64_peak_clocked(self.h, C.byref(v), C.byref(c)))
        return v.value, c.value

    def measure_fp64_peak(self):
        """measured FP64 pipe rate of this device, FP64 instructions (lane-ops) per second"""
        v = C.c_double(0.0)
        _check(load().grpic_measure_fp64_peak(self.h, C.byref(v)))
        return v.value

    @staticmethod
    def kernel_launches():
        return int(load().grpic_kernel_launches())

    def deposit_rho(self, ptc, rho, divide=True):
        ps = ptc.struct()
        _check(load().grpic_deposit_rho(self.h, C.byref(ps), _ptr(rho), C.c_int32(1 if divide else 0), _stream()))
