"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle (tests, bench, smoke) and
therefore holds none of the method's arithmetic: it only draws geometry, masks and
initial fields with numpy.random.default_rng(seed).  The paper's room layouts live
in figures that are not available (Table 3), so
these generators take the shapes, sizes and value ranges of those workloads and
stand in for them.

A case is a dict:
  shape (nz, ny, nx), d (dx, dy, dz), nu, alpha_c, dt, body, n_piter,
  mask (uint8 (nz,ny,nx), 1 = fluid) or None, sources (list of dicts),
  u, v, w, c (float64 (nz,ny,nx)), steps, name
Arrays are x-fastest: element [k, j, i].
"""
import math

import numpy as np


def _walls(mask, axes=(0, 1, 2), thick=2):
    for ax in axes:
        sl = [slice(None)] * 3
        sl[ax] = slice(0, thick)
        mask[tuple(sl)] = 0
        sl[ax] = slice(mask.shape[ax] - thick, None)
        mask[tuple(sl)] = 0


def _boxes(mask, rng, n, lo_side, hi_side, clearance=4):
    nz, ny, nx = mask.shape
    out = []
    for _ in range(n):
        sx, sy, sz = (int(rng.integers(lo_side, hi_side + 1)) for _ in range(3))
        sx, sy, sz = min(sx, nx - 2 * clearance - 1), min(sy, ny - 2 * clearance - 1), min(sz, nz - 2 * clearance - 1)
        ox = int(rng.integers(clearance, nx - clearance - sx + 1))
        oy = int(rng.integers(clearance, ny - clearance - sy + 1))
        oz = int(rng.integers(clearance, nz - clearance - sz + 1))
        mask[oz:oz + sz, oy:oy + sy, ox:ox + sx] = 0
        out.append(((ox, oy, oz), (sx, sy, sz)))
    return out


def _duct(mask, axis, lo2, size2, thick=2):
    """Open a hole through the wall slab that straddles the periodic seam of `axis`
    (numpy axis order: 0 = z, 1 = y, 2 = x).  lo2/size2 are (lo, size) on the two other
    axes in x,y,z order with the duct axis removed.  Returns the source box (lo, size) in
    x,y,z order: it fills the hole (2*thick cells long, wrapping)."""
    n = mask.shape[axis]
    dims = mask.shape[::-1]  # nx, ny, nz
    a_xyz = 2 - axis
    lo = [0, 0, 0]
    size = [0, 0, 0]
    others = [a for a in range(3) if a != a_xyz]
    for a, l, s in zip(others, lo2, size2):
        lo[a], size[a] = int(l), int(s)
    lo[a_xyz], size[a_xyz] = n - thick, 2 * thick
    idx = [None] * 3  # in x,y,z
    for a in range(3):
        idx[a] = np.arange(lo[a], lo[a] + size[a]) % dims[a]
    mask[np.ix_(idx[2], idx[1], idx[0])] = 1
    return tuple(lo), tuple(size)


def _binary_S(shape, lo, size):
    nz, ny, nx = shape
    S = np.zeros(shape, dtype=np.float64)
    ix = np.arange(lo[0], lo[0] + size[0]) % nx
    iy = np.arange(lo[1], lo[1] + size[1]) % ny
    iz = np.arange(lo[2], lo[2] + size[2]) % nz
    S[np.ix_(iz, iy, ix)] = 1.0
    return S


def _room_fields(mask, sources, rng, sigma=1e-3):
    shape = mask.shape
    b = mask.astype(np.float64)
    u = b * (sigma * rng.standard_normal(shape))
    v = b * (sigma * rng.standard_normal(shape))
    w = b * (sigma * rng.standard_normal(shape))
    S = np.zeros(shape)
    for s in sources:
        S = np.maximum(S, _binary_S(shape, s["lo"], s["size"]))
    c = b * (1.0 - S)
    return u, v, w, c


def taylor_green(n=32, nu=0.01, cfl=0.3, steps=10):
    """Config 1: 32^3 periodic Taylor-Green vortex on [0,2pi)^3, Re = 100, no mask."""
    d = 2.0 * math.pi / n
    x = np.arange(n) * d
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    u = np.sin(X) * np.cos(Y) * np.cos(Z)
    v = -np.cos(X) * np.sin(Y) * np.cos(Z)
    w = np.zeros_like(u)
    c = np.cos(X) + 0.0 * Y
    return dict(name=f"tgv{n}", shape=(n, n, n), d=(d, d, d), nu=nu, alpha_c=nu, dt=cfl * d / 1.0,
                body=(0.0, 0.0, 0.0), n_piter=1, mask=None, sources=[], u=u, v=v, w=w, c=c, steps=steps)


def duct_room(nx=128, ny=64, nz=64, seed=1002, n_piter=4, steps=100):
    """Config 2: duct-like room, walls 2 thick on six faces, 4 seeded boxes of 4..16 cells,
    8x8 inlet through the x-seam wall slab (it is the outlet on its far side), 0.1 m/s."""
    rng = np.random.default_rng(seed)
    h = 1.0 / 16.0 * (128.0 / nx)
    U = 0.1
    dt = 0.25 * h / U
    mask = np.ones((nz, ny, nx), dtype=np.uint8)
    _walls(mask)
    f = nx / 128.0
    _boxes(mask, rng, 4, max(2, round(4 * f)), max(3, round(16 * f)), clearance=4)
    dsz = max(2, round(8 * f))
    lo, size = _duct(mask, 2, ((ny - dsz) // 2, (nz - dsz) // 2), (dsz, dsz))
    sources = [dict(lo=lo, size=size, B=(0.0, 0.0, 0.0), u_set=(U, 0.0, 0.0), c_set=0.0, tau_f=2.0 * dt, comps=0xF)]
    u, v, w, c = _room_fields(mask, sources, rng)
    return dict(name=f"duct{nx}x{ny}x{nz}", shape=(nz, ny, nx), d=(h, h, h), nu=1.6e-5, alpha_c=1.6e-5, dt=dt,
                body=(0.0, 0.0, 0.0), n_piter=n_piter, mask=mask, sources=sources, u=u, v=v, w=w, c=c, steps=steps)


def _spectral_field(rng, n, k0):
    """Real random-phase field with E(k) ~ k^4 exp(-2 (k/k0)^2): FFT of unit white noise times
    sqrt(E(k) / (4 pi k^2))."""
    k1 = np.fft.fftfreq(n, 1.0 / n)
    kz, ky, kx = np.meshgrid(k1, k1, k1[: n // 2 + 1], indexing="ij")
    kk = np.sqrt(kx * kx + ky * ky + kz * kz)
    amp = np.zeros_like(kk)
    nzk = kk > 0
    E = kk[nzk] ** 4 * np.exp(-2.0 * (kk[nzk] / k0) ** 2)
    amp[nzk] = np.sqrt(E / (4.0 * math.pi * kk[nzk] ** 2))
    return np.fft.rfftn(rng.standard_normal((n, n, n)), axes=(0, 1, 2)) * amp, (kx, ky, kz)


def periodic_turbulence(n=256, seed=1003, nu=0.01, k0=4.0, cfl=0.3, steps=100):
    """Config 3: n^3 periodic box, random-phase velocity made solenoidal with respect to the
    central-difference wavevector sin(k_a h)/h, u' = 1; scalar from the same spectrum."""
    rng = np.random.default_rng(seed)
    h = 2.0 * math.pi / n
    uh, (kx, ky, kz) = _spectral_field(rng, n, k0)
    vh, _ = _spectral_field(rng, n, k0)
    wh, _ = _spectral_field(rng, n, k0)
    ch, _ = _spectral_field(rng, n, k0)
    mx, my, mz = np.sin(kx * h) / h, np.sin(ky * h) / h, np.sin(kz * h) / h
    m2 = mx * mx + my * my + mz * mz
    ok = m2 > 1e-20
    dot = np.where(ok, (mx * uh + my * vh + mz * wh) / np.where(ok, m2, 1.0), 0.0)
    uh, vh, wh = uh - dot * mx, vh - dot * my, wh - dot * mz
    u, v, w, c = (np.fft.irfftn(a, s=(n, n, n), axes=(0, 1, 2)) for a in (uh, vh, wh, ch))
    up = math.sqrt((np.mean(u * u) + np.mean(v * v) + np.mean(w * w)) / 3.0)
    u, v, w = u / up, v / up, w / up
    c = (c - c.mean()) / c.std()
    umax = max(np.abs(u).max(), np.abs(v).max(), np.abs(w).max())
    return dict(name=f"turb{n}", shape=(n, n, n), d=(h, h, h), nu=nu, alpha_c=nu, dt=cfl * h / umax,
                body=(0.0, 0.0, 0.0), n_piter=1, mask=None, sources=[],
                u=np.ascontiguousarray(u), v=np.ascontiguousarray(v), w=np.ascontiguousarray(w),
                c=np.ascontiguousarray(c), steps=steps)


def room(nx=512, ny=256, nz=128, seed=1004, n_piter=4, steps=1000):
    """Config 4: box room, walls 2 thick, one 32x16 (x by y) ceiling duct through the z-seam slab
    at 1 m/s downwards, 10 seeded boxes with sides 8..40 cells."""
    rng = np.random.default_rng(seed)
    f = nx / 512.0
    h = 1.0 / 64.0 / f
    U = 1.0
    dt = 0.25 * h / U
    mask = np.ones((nz, ny, nx), dtype=np.uint8)
    _walls(mask)
    _boxes(mask, rng, 10, max(2, round(8 * f)), max(3, round(40 * f)), clearance=4)
    dx_, dy_ = max(2, round(32 * f)), max(2, round(16 * f))
    ox = int(rng.integers(4, nx - 4 - dx_ + 1))
    oy = int(rng.integers(4, ny - 4 - dy_ + 1))
    lo, size = _duct(mask, 0, (ox, oy), (dx_, dy_))
    sources = [dict(lo=lo, size=size, B=(0.0, 0.0, 0.0), u_set=(0.0, 0.0, -U), c_set=0.0, tau_f=2.0 * dt, comps=0xF)]
    u, v, w, c = _room_fields(mask, sources, rng)
    return dict(name=f"room{nx}x{ny}x{nz}", shape=(nz, ny, nx), d=(h, h, h), nu=1.6e-5, alpha_c=1.6e-5, dt=dt,
                body=(0.0, 0.0, 0.0), n_piter=n_piter, mask=mask, sources=sources, u=u, v=v, w=w, c=c, steps=steps)


def three_rooms(nx=1024, ny=512, nz=256, seed=1005, n_piter=4, steps=200, fields=True):
    """Config 5: three rooms split by 2-thick partition walls normal to x, each with a 40x80 (y by z)
    doorway from the floor; two 64x64 ducts through the x-seam slab at 0.1 and 1 m/s; 30 boxes."""
    rng = np.random.default_rng(seed)
    f = nx / 1024.0
    h = 1.0 / 128.0 / f
    dt = 0.25 * h / 1.0
    mask = np.ones((nz, ny, nx), dtype=np.uint8)
    _walls(mask)
    _boxes(mask, rng, 30, max(2, round(8 * f)), max(3, round(40 * f)), clearance=4)
    dw, dh = max(2, round(40 * f)), max(2, round(80 * f))
    for ip in (nx // 3 - 1, 2 * nx // 3):
        mask[:, :, ip:ip + 2] = 0
        oy = int(rng.integers(4, ny - 4 - dw + 1))
        mask[2:2 + dh, oy:oy + dw, ip:ip + 2] = 1
    ds = max(2, round(64 * f))
    oy1 = int(rng.integers(4, ny // 2 - ds - 4 + 1))
    oy2 = int(rng.integers(ny // 2 + 4, ny - 4 - ds + 1))
    oz1 = int(rng.integers(4, nz - 4 - ds + 1))
    oz2 = int(rng.integers(4, nz - 4 - ds + 1))
    sources = []
    for (oy, oz, U) in ((oy1, oz1, 0.1), (oy2, oz2, 1.0)):
        lo, size = _duct(mask, 2, (oy, oz), (ds, ds))
        sources.append(dict(lo=lo, size=size, B=(0.0, 0.0, 0.0), u_set=(U, 0.0, 0.0), c_set=0.0, tau_f=2.0 * dt,
                            comps=0xF))
    case = dict(name=f"rooms{nx}x{ny}x{nz}", shape=(nz, ny, nx), d=(h, h, h), nu=1.6e-5, alpha_c=1.6e-5, dt=dt,
                body=(0.0, 0.0, 0.0), n_piter=n_piter, mask=mask, sources=sources, steps=steps)
    if fields:
        case["u"], case["v"], case["w"], case["c"] = _room_fields(mask, sources, rng)
    return case


def config(i, shrink=1):
    """BASELINE.json configs[i-1]; shrink divides every grid dimension (for quick tests)."""
    s = int(shrink)
    if i == 1:
        return taylor_green(32 // s)
    if i == 2:
        return duct_room(128 // s, 64 // s, 64 // s)
    if i == 3:
        return periodic_turbulence(256 // s)
    if i == 4:
        return room(512 // s, 256 // s, 128 // s)
    if i == 5:
        return three_rooms(1024 // s, 512 // s, 256 // s)
    raise ValueError(i)
