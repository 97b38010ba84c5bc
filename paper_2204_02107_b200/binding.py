"""Thin Python binding over the C ABI of libdnslab.so (include/dnslab.h).

Argument marshalling only: every step of the hot path runs in the library's CUDA kernels.
PyTorch provides the device workspace and the stream, nothing else.  There is no CPU
fallback: if the library is missing or no sm_100 GPU is present the calls raise.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdnslab.so")

SYMBOLS = ["dnslab_workspace_bytes", "dnslab_create", "dnslab_set_fields", "dnslab_step", "dnslab_poisson",
           "dnslab_rfft3", "dnslab_irfft3", "dnslab_fields", "dnslab_get_fields", "dnslab_launch_count", "dnslab_profile", "dnslab_profile_read",
           "dnslab_courant", "dnslab_set_dt", "dnslab_scalar_stats", "dnslab_scalar_stats_static", "dnslab_particles_attach", "dnslab_destroy", "dnslab_strerror"]
KERNEL_CLASSES = ["rk_stage", "div", "fft_x", "fft_y", "fft_z_solve", "project", "eq9_sparse", "filter", "reduce", "particles",
                  "fft_xy", "fft_yz_solve"]


class Params(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("nu", C.c_double), ("alpha_c", C.c_double), ("dt", C.c_double),
                ("body", C.c_double * 3), ("n_piter", C.c_int32), ("flags", C.c_uint32)]


class Source(C.Structure):
    _fields_ = [("lo", C.c_int32 * 3), ("size", C.c_int32 * 3), ("B", C.c_double * 3),
                ("u_set", C.c_double * 3), ("c_set", C.c_double), ("tau_f", C.c_double),
                ("comps", C.c_uint32)]


class DnslabError(RuntimeError):
    pass


_lib = None


def lib():
    """Load libdnslab.so (built in-tree by paper_2204_02107_b200/build.py).  Fails loudly."""
    global _lib
    if _lib is None:
        _lib = load(LIB_PATH)
    return _lib


def load(path):
    """A library at `path` with the C ABI of include/dnslab.h, argument types declared (lib() loads the product;
    the GPU tests also load the test-only no-TMA build through this)."""
    if not os.path.exists(path):
        raise DnslabError(f"{path} not built: run `python -m paper_2204_02107_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(path)
    L.dnslab_workspace_bytes.argtypes = [C.POINTER(Params)]
    L.dnslab_workspace_bytes.restype = C.c_size_t
    L.dnslab_create.argtypes = [C.POINTER(Params), C.c_void_p, C.POINTER(Source), C.c_int32, C.c_void_p,
                                C.c_void_p, C.POINTER(C.c_void_p)]
    L.dnslab_set_fields.argtypes = [C.c_void_p] + [C.c_void_p] * 5
    L.dnslab_step.argtypes = [C.c_void_p, C.c_int32]
    L.dnslab_poisson.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.dnslab_rfft3.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.dnslab_irfft3.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.dnslab_fields.argtypes = [C.c_void_p] + [C.POINTER(C.c_void_p)] * 5
    L.dnslab_get_fields.argtypes = [C.c_void_p] + [C.c_void_p] * 5
    L.dnslab_launch_count.argtypes = [C.c_void_p]
    L.dnslab_launch_count.restype = C.c_int64
    L.dnslab_profile.argtypes = [C.c_void_p, C.c_int]
    L.dnslab_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    L.dnslab_courant.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
    L.dnslab_set_dt.argtypes = [C.c_void_p, C.c_double]
    L.dnslab_scalar_stats.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_double)]
    L.dnslab_scalar_stats_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_int32),
                                             C.POINTER(C.c_int32), C.c_void_p, C.c_void_p]
    L.dnslab_particles_attach.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_double, C.POINTER(C.c_double)]
    L.dnslab_destroy.argtypes = [C.c_void_p]
    L.dnslab_strerror.argtypes = [C.c_int]
    L.dnslab_strerror.restype = C.c_char_p
    return L


def _check(rc, what):
    if rc != 0:
        raise DnslabError(f"{what} failed: {lib().dnslab_strerror(rc).decode()} ({rc})")


def make_params(shape, d, nu, alpha_c, dt, body=(0.0, 0.0, 0.0), n_piter=1, flags=0):
    nz, ny, nx = (int(s) for s in shape)
    P = Params()
    P.nx, P.ny, P.nz = nx, ny, nz
    P.dx, P.dy, P.dz = (float(x) for x in d)
    P.nu, P.alpha_c, P.dt = float(nu), float(alpha_c), float(dt)
    P.body[:] = [float(b) for b in body]
    P.n_piter, P.flags = int(n_piter), int(flags)
    return P


def make_sources(sources):
    arr = (Source * max(1, len(sources)))()
    for s, d in zip(arr, sources):
        s.lo[:] = [int(x) for x in d["lo"]]
        s.size[:] = [int(x) for x in d["size"]]
        s.B[:] = d.get("B", (0.0, 0.0, 0.0))
        s.u_set[:] = d.get("u_set", (0.0, 0.0, 0.0))
        s.c_set = d.get("c_set", 0.0)
        s.tau_f = d["tau_f"]
        s.comps = d.get("comps", 0xF)
    return arr


def workspace_bytes(params):
    return int(lib().dnslab_workspace_bytes(C.byref(params)))


def _addr(x, dtype="float64"):
    """Address of a contiguous torch tensor (device or host) or numpy array of the given dtype, or None.
    The library reads raw bytes: a wrong dtype would be an out-of-bounds read, so it is refused here."""
    if x is None:
        return None
    if str(x.dtype).split(".")[-1] != dtype:
        raise DnslabError(f"expected a {dtype} buffer, got {x.dtype}")
    if hasattr(x, "data_ptr"):
        if not x.is_contiguous():
            raise DnslabError("buffer must be contiguous")
        return x.data_ptr()
    if not x.flags["C_CONTIGUOUS"]:
        raise DnslabError("buffer must be contiguous")
    return x.ctypes.data


STATIC_MAX_ROWS = 65536  # DNSLAB_STATIC_MAX_ROWS


def scalar_stats_static(c, mask, lo, size, out, stream=None):
    """dnslab_scalar_stats_static: (mean, std, count) of c over the fluid cells of the index box lo, size (x,y,z),
    for callers that cannot allocate device memory (a monitor handed borrowed pointers while the HBM is fully
    committed; code that must not stall the device with a cudaMalloc).  Allocates nothing: c (float64 CUDA,
    (nz, ny, nx)), mask (uint8 CUDA, non-zero = fluid, or None) and out (float64 CUDA, 3 elements) all come from
    the caller; the scratch is a 1 MiB array inside the library, shared by every call on the device, so calls
    must not overlap on the GPU.  Asynchronous on `stream` (a torch stream; None = the default stream).  Boxes
    with size[1]*size[2] > STATIC_MAX_ROWS raise ("... more rows ... than the static scratch array holds")."""
    nz, ny, nx = (int(s) for s in c.shape)
    if not (c.is_cuda and out.is_cuda and out.numel() >= 3 and (mask is None or (mask.is_cuda and tuple(mask.shape) == tuple(c.shape)))):
        raise DnslabError("c, mask and out must be CUDA tensors; mask shaped like c; out with 3 elements")
    a = (C.c_int32 * 3)(*[int(x) for x in lo])
    b = (C.c_int32 * 3)(*[int(x) for x in size])
    _check(lib().dnslab_scalar_stats_static(_addr(c), _addr(mask, "uint8"), nx, ny, nz, a, b,
                                            stream.cuda_stream if stream is not None else None, _addr(out)),
           "dnslab_scalar_stats_static")
    return out


class Solver:
    """dnslab_create / set_fields / step / poisson / fields / get_fields / destroy.

    Arrays are (nz, ny, nx), x fastest.  `mask` (uint8, 1 = fluid) and the inputs of set_fields /
    outputs of get_fields may be host (numpy or torch CPU) or device (torch CUDA) buffers.
    """

    def __init__(self, shape, d, nu, alpha_c, dt, mask=None, sources=(), body=(0.0, 0.0, 0.0), n_piter=1, flags=0,
                 device="cuda:0", stream=None):
        import torch  # device memory and streams only
        if not torch.cuda.is_available():
            raise DnslabError("no CUDA device: the DNSLAB path has no CPU fallback")
        self._torch = torch
        self.shape = tuple(int(s) for s in shape)
        self.device = torch.device(device)
        self.params = make_params(self.shape, d, nu, alpha_c, dt, body, n_piter, flags)
        nbytes = workspace_bytes(self.params)
        if nbytes == 0:
            raise DnslabError("invalid parameters (dnslab_workspace_bytes returned 0)")
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        self._src = make_sources(list(sources))
        self._h = C.c_void_p()
        if mask is not None and hasattr(mask, "dtype") and not hasattr(mask, "data_ptr"):
            import numpy as np
            mask = np.ascontiguousarray(mask, dtype=np.uint8)
        self._mask = mask
        _check(lib().dnslab_create(C.byref(self.params), _addr(mask, "uint8"), self._src, len(sources), self._ws_ptr,
                                   self.stream.cuda_stream, C.byref(self._h)), "dnslab_create")

    # -- C ABI calls ---------------------------------------------------------------------
    def set_fields(self, u, v, w, c, p=None):
        self._keep = (u, v, w, c, p)  # keep host buffers alive until the async copies ran
        _check(lib().dnslab_set_fields(self._h, _addr(u), _addr(v), _addr(w), _addr(c), _addr(p)), "dnslab_set_fields")

    def step(self, n=1):
        _check(lib().dnslab_step(self._h, int(n)), "dnslab_step")

    def poisson(self, rhs, out=None):
        torch = self._torch
        assert rhs.is_cuda and rhs.dtype == torch.float64 and rhs.is_contiguous()
        if out is None:
            out = torch.empty_like(rhs)
        _check(lib().dnslab_poisson(self._h, rhs.data_ptr(), out.data_ptr()), "dnslab_poisson")
        return out

    def rfft3(self, x):
        """dnslab_rfft3: x float64 CUDA (nz, ny, nx) -> complex128 CUDA (nz, ny, nx/2 + 1), unnormalised."""
        torch = self._torch
        assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous() and tuple(x.shape) == self.shape
        out = torch.empty(self.shape[:2] + (self.shape[2] // 2 + 1,), dtype=torch.complex128, device=x.device)
        _check(lib().dnslab_rfft3(self._h, x.data_ptr(), out.data_ptr()), "dnslab_rfft3")
        return out

    def irfft3(self, X):
        """dnslab_irfft3: complex128 CUDA (nz, ny, nx/2 + 1) -> float64 CUDA (nz, ny, nx), includes 1/N."""
        torch = self._torch
        assert X.is_cuda and X.dtype == torch.complex128 and X.is_contiguous()
        assert tuple(X.shape) == self.shape[:2] + (self.shape[2] // 2 + 1,)
        out = torch.empty(self.shape, dtype=torch.float64, device=X.device)
        _check(lib().dnslab_irfft3(self._h, X.data_ptr(), out.data_ptr()), "dnslab_irfft3")
        return out

    def field_ptrs(self):
        ptrs = [C.c_void_p() for _ in range(5)]
        _check(lib().dnslab_fields(self._h, *[C.byref(p) for p in ptrs]), "dnslab_fields")
        return dict(zip("uvwcp", (p.value for p in ptrs)))

    def get_fields(self, u=None, v=None, w=None, c=None, p=None):
        _check(lib().dnslab_get_fields(self._h, _addr(u), _addr(v), _addr(w), _addr(c), _addr(p)), "dnslab_get_fields")

    def launch_count(self):
        return int(lib().dnslab_launch_count(self._h))

    def particles_attach(self, state, rho_f=1.2, g=(0.0, 0.0, 0.0)):
        """dnslab_particles_attach: state is a contiguous float64 CUDA tensor of shape (8, n) (rows x y z u v w d rho_p),
        advanced in place at the end of every step; None detaches.  The caller keeps the tensor alive."""
        gg = (C.c_double * 3)(*[float(x) for x in g])
        if state is None:
            _check(lib().dnslab_particles_attach(self._h, 0, None, 1.0, gg), "dnslab_particles_attach")
        else:
            assert state.is_cuda and state.is_contiguous() and state.dim() == 2 and state.shape[0] == 8
            _check(lib().dnslab_particles_attach(self._h, int(state.shape[1]), state.data_ptr(), float(rho_f), gg),
                   "dnslab_particles_attach")
        self._particles = state

    def courant(self):
        """dnslab_courant: dt * max_cells(|u|/dx + |v|/dy + |w|/dz); synchronises."""
        out = C.c_double(0.0)
        _check(lib().dnslab_courant(self._h, C.byref(out)), "dnslab_courant")
        return out.value

    def set_dt(self, dt):
        _check(lib().dnslab_set_dt(self._h, float(dt)), "dnslab_set_dt")

    def scalar_stats(self, lo, size):
        """dnslab_scalar_stats: (mean, std, count) of c over the fluid cells of the index box lo, size (x,y,z)."""
        a = (C.c_int32 * 3)(*[int(x) for x in lo])
        b = (C.c_int32 * 3)(*[int(x) for x in size])
        out = (C.c_double * 3)()
        _check(lib().dnslab_scalar_stats(self._h, a, b, out), "dnslab_scalar_stats")
        return out[0], out[1], int(out[2])

    def profile(self, enable):
        _check(lib().dnslab_profile(self._h, int(bool(enable))), "dnslab_profile")

    def profile_read(self):
        """{class: (total ms, launches)} since profile(True)."""
        n = len(KERNEL_CLASSES)
        ms, cnt = (C.c_double * n)(), (C.c_int64 * n)()
        _check(lib().dnslab_profile_read(self._h, ms, cnt), "dnslab_profile_read")
        return {k: (ms[i], int(cnt[i])) for i, k in enumerate(KERNEL_CLASSES)}

    # -- conveniences (marshalling only) ---------------------------------------------------
    def fields(self):
        """Device copies of u,v,w,c,p as torch tensors."""
        torch = self._torch
        out = {k: torch.empty(self.shape, dtype=torch.float64, device=self.device) for k in "uvwcp"}
        with torch.cuda.stream(self.stream):
            self.get_fields(**out)
        return out

    def fields_numpy(self):
        f = self.fields()
        self.stream.synchronize()
        return {k: t.cpu().numpy() for k, t in f.items()}

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        if getattr(self, "_h", None):
            self.stream.synchronize()
            lib().dnslab_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def solver_for_case(case, n_piter=None, flags=0, **kw):
    """Solver for a dict from paper_2204_02107_b200.cases, fields loaded from its host arrays."""
    s = Solver(case["shape"], case["d"], case["nu"], case["alpha_c"], case["dt"], mask=case["mask"],
               sources=case["sources"], body=case["body"], n_piter=n_piter or case["n_piter"], flags=flags, **kw)
    s.set_fields(case["u"], case["v"], case["w"], case["c"])
    s.synchronize()
    return s
