"""ctypes loader for the CPU oracle (oracle/dnsref.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It never imports the CUDA package and the CUDA
package never imports it.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dnsref.c")
_LIB = os.path.join(_HERE, "libdnsref.so")


class Params(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("nu", C.c_double), ("alpha_c", C.c_double), ("dt", C.c_double),
                ("body", C.c_double * 3), ("n_piter", C.c_int32), ("flags", C.c_uint32)]


class Source(C.Structure):
    _fields_ = [("lo", C.c_int32 * 3), ("size", C.c_int32 * 3), ("B", C.c_double * 3),
                ("u_set", C.c_double * 3), ("c_set", C.c_double), ("tau_f", C.c_double),
                ("comps", C.c_uint32)]


def build(force=False):
    """gcc -O2, no fast-math, no FMA contraction; OpenMP only over outer loops."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.dnsref_create.argtypes = [C.POINTER(Params), C.c_void_p, C.POINTER(Source), C.c_int32,
                                    C.POINTER(C.c_void_p)]
        L.dnsref_destroy.argtypes = [C.c_void_p]
        L.dnsref_set_fields.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        L.dnsref_get_fields.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        L.dnsref_step.argtypes = [C.c_void_p, C.c_int]
        L.dnsref_poisson.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.dnsref_rhs.argtypes = [C.c_void_p] + [C.c_void_p] * 8
        L.dnsref_rhs.restype = None
        L.dnsref_div.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.dnsref_div.restype = None
        L.dnsref_poisson_rhs.argtypes = [C.c_void_p] + [C.c_void_p] * 3
        L.dnsref_poisson_rhs.restype = None
        L.dnsref_particles_step.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        L.dnsref_particles_attach.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        L.dnsref_courant.argtypes = [C.c_void_p]
        L.dnsref_courant.restype = C.c_double
        L.dnsref_set_dt.argtypes = [C.c_void_p, C.c_double]
        L.dnsref_scalar_stats.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_double)]
        L.dnsref_filter.argtypes = [C.c_void_p] + [C.c_void_p] * 2
        L.dnsref_filter.restype = None
        L.dnsref_project.argtypes = [C.c_void_p] + [C.c_void_p] * 7
        L.dnsref_project.restype = None
        L.dnsref_fft1d.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_int]
        L.dnsref_fft1d.restype = None
        L.dnsref_dft1d.argtypes = [C.c_int] + [C.c_void_p] * 4 + [C.c_int]
        L.dnsref_dft1d.restype = None
        L.dnsref_fft3.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int]
        L.dnsref_fft3.restype = None
        L.dnsref_eig.argtypes = [C.POINTER(Params), C.c_int, C.c_int, C.c_int]
        L.dnsref_eig.restype = C.c_double
        L.dnsref_source_table.argtypes = [C.c_int, C.c_double, C.c_int, C.c_int, C.c_double, C.c_void_p]
        L.dnsref_source_table.restype = None
        L.dnsref_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def make_params(shape, d, nu, alpha_c, dt, body=(0.0, 0.0, 0.0), n_piter=1, flags=0):
    """shape = (nz, ny, nx) numpy shape; d = (dx, dy, dz)."""
    nz, ny, nx = shape
    P = Params()
    P.nx, P.ny, P.nz = nx, ny, nz
    P.dx, P.dy, P.dz = d
    P.nu, P.alpha_c, P.dt = nu, alpha_c, dt
    P.body[:] = body
    P.n_piter, P.flags = n_piter, flags
    return P


def make_sources(sources):
    """sources: list of dicts(lo, size, B, u_set, c_set, tau_f, comps)."""
    arr = (Source * max(1, len(sources)))()
    for s, d in zip(arr, sources):
        s.lo[:] = d["lo"]
        s.size[:] = d["size"]
        s.B[:] = d.get("B", (0.0, 0.0, 0.0))
        s.u_set[:] = d.get("u_set", (0.0, 0.0, 0.0))
        s.c_set = d.get("c_set", 0.0)
        s.tau_f = d["tau_f"]
        s.comps = d.get("comps", 0xF)
    return arr


class Oracle:
    """Handle on one oracle problem.  Arrays are numpy float64 of shape (nz, ny, nx)."""

    def __init__(self, shape, d, nu, alpha_c, dt, mask=None, sources=(), body=(0.0, 0.0, 0.0), n_piter=1,
                 flags=0):
        self.shape = tuple(int(s) for s in shape)
        self.P = make_params(self.shape, d, nu, alpha_c, dt, body, n_piter, flags)
        self._mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
        if self._mask is not None:
            assert self._mask.shape == self.shape
        self._src = make_sources(list(sources))
        self._h = C.c_void_p()
        rc = lib().dnsref_create(C.byref(self.P), _ptr(self._mask), self._src, len(sources), C.byref(self._h))
        if rc != 0:
            raise ValueError(f"dnsref_create failed: {rc}")

    def close(self):
        if self._h:
            lib().dnsref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _new(self):
        return np.empty(self.shape, dtype=np.float64)

    def set_fields(self, u, v, w, c, p=None):
        a = [_f64(x) for x in (u, v, w, c)]
        pp = None if p is None else _f64(p)
        rc = lib().dnsref_set_fields(self._h, *[_ptr(x) for x in a], _ptr(pp))
        assert rc == 0

    def fields(self):
        out = [self._new() for _ in range(5)]
        rc = lib().dnsref_get_fields(self._h, *[_ptr(x) for x in out])
        assert rc == 0
        return dict(zip("uvwcp", out))

    def step(self, n=1):
        rc = lib().dnsref_step(self._h, int(n))
        assert rc == 0

    def poisson(self, rhs):
        rhs = _f64(rhs)
        p = self._new()
        rc = lib().dnsref_poisson(self._h, _ptr(rhs), _ptr(p))
        assert rc == 0
        return p

    def rhs(self, u, v, w, c):
        a = [_f64(x) for x in (u, v, w, c)]
        F = [self._new() for _ in range(4)]
        lib().dnsref_rhs(self._h, *[_ptr(x) for x in a], *[_ptr(x) for x in F])
        return F

    def div(self, u, v, w):
        a = [_f64(x) for x in (u, v, w)]
        d = self._new()
        lib().dnsref_div(self._h, *[_ptr(x) for x in a], _ptr(d))
        return d

    def poisson_rhs(self, d, p):
        d, p = _f64(d), _f64(p)
        r = self._new()
        lib().dnsref_poisson_rhs(self._h, _ptr(d), _ptr(p), _ptr(r))
        return r

    def particles_step(self, state, rho_f, g):
        """One particle step (eqs. 10-13) in the current velocity field; state: float64 (8, n) rows x y z u v w d rho_p,
        updated in place."""
        assert state.dtype == np.float64 and state.ndim == 2 and state.shape[0] == 8 and state.flags.c_contiguous
        gg = (C.c_double * 3)(*[float(x) for x in g])
        rc = lib().dnsref_particles_step(self._h, state.shape[1], _ptr(state), float(rho_f), gg)
        if rc:
            raise ValueError("dnsref_particles_step")

    def particles_attach(self, state, rho_f=1.2, g=(0.0, 0.0, 0.0)):
        """Advance these particles at the end of every step (state is kept and updated in place); None detaches."""
        gg = (C.c_double * 3)(*[float(x) for x in g])
        if state is None:
            rc = lib().dnsref_particles_attach(self._h, 0, None, 1.0, gg)
        else:
            assert state.dtype == np.float64 and state.ndim == 2 and state.shape[0] == 8 and state.flags.c_contiguous
            rc = lib().dnsref_particles_attach(self._h, state.shape[1], _ptr(state), float(rho_f), gg)
        self._particles = state
        if rc:
            raise ValueError("dnsref_particles_attach")

    def courant(self):
        """dt * max_cells(|u|/dx + |v|/dy + |w|/dz) of the current state (reading R24)."""
        return float(lib().dnsref_courant(self._h))

    def set_dt(self, dt):
        rc = lib().dnsref_set_dt(self._h, float(dt))
        if rc:
            raise ValueError("dnsref_set_dt")
        self.P.dt = float(dt)

    def scalar_stats(self, lo, size):
        """(mean, std, count) of c over the fluid cells of the index box lo (x,y,z), size (x,y,z) (reading R25)."""
        a = (C.c_int32 * 3)(*[int(x) for x in lo])
        b = (C.c_int32 * 3)(*[int(x) for x in size])
        out = (C.c_double * 3)()
        rc = lib().dnsref_scalar_stats(self._h, a, b, out)
        if rc:
            raise ValueError("dnsref_scalar_stats")
        return out[0], out[1], int(out[2])

    def filter(self, f):
        """eq. 6 on one field (masked by the select)."""
        f = _f64(f)
        out = self._new()
        lib().dnsref_filter(self._h, _ptr(f), _ptr(out))
        return out

    def project(self, us, vs, ws, p):
        a = [_f64(x) for x in (us, vs, ws, p)]
        out = [self._new() for _ in range(3)]
        lib().dnsref_project(self._h, *[_ptr(x) for x in a], *[_ptr(x) for x in out])
        return out

    def eig(self, kx, ky, kz):
        return lib().dnsref_eig(C.byref(self.P), int(kx), int(ky), int(kz))


def fft1d(re, im, sign):
    re, im = _f64(re).copy(), _f64(im).copy()
    lib().dnsref_fft1d(len(re), _ptr(re), _ptr(im), int(sign))
    return re, im


def dft1d(re, im, sign):
    re, im = _f64(re), _f64(im)
    ore, oim = np.empty_like(re), np.empty_like(im)
    lib().dnsref_dft1d(len(re), _ptr(re), _ptr(im), _ptr(ore), _ptr(oim), int(sign))
    return ore, oim


def fft3(re, im, sign):
    re, im = _f64(re).copy(), _f64(im).copy()
    nz, ny, nx = re.shape
    lib().dnsref_fft3(nx, ny, nz, _ptr(re), _ptr(im), int(sign))
    return re, im


def source_table(n, d, lo, size, B):
    out = np.empty(n, dtype=np.float64)
    lib().dnsref_source_table(int(n), float(d), int(lo), int(size), float(B), _ptr(out))
    return out


def num_threads():
    return lib().dnsref_num_threads()
