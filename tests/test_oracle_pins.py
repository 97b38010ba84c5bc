"""Pins for the CPU oracle (oracle/dnsref.c): each part is checked against something
other than itself -- a library routine, a dense matrix built here from index
arithmetic, a closed form, an exact amplification factor or an invariant.
Numbering follows SURVEY.md section 8(c) (P1..P14).  CPU only.
"""
import math
import os

import numpy as np
import pytest

from oracle import dnsref
from paper_2204_02107_b200 import cases

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def rng(seed):
    return np.random.default_rng(seed)


def mk(shape, d=(1.0, 1.0, 1.0), nu=0.0, alpha_c=0.0, dt=1.0, **kw):
    return dnsref.Oracle(shape, d, nu, alpha_c, dt, **kw)


# ---------------------------------------------------------------- FFT (P0)
@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 64, 12, 24])
def test_fft1d_matches_definition_and_library(n):
    r = rng(n)
    re, im = r.standard_normal(n), r.standard_normal(n)
    for sign in (-1, +1):
        fr, fi = dnsref.fft1d(re, im, sign)
        dr, di = dnsref.dft1d(re, im, sign)
        lib = np.fft.fft(re + 1j * im) if sign < 0 else np.fft.ifft(re + 1j * im) * n
        assert np.allclose(fr + 1j * fi, lib, rtol=0, atol=1e-12 * n)
        assert np.allclose(dr + 1j * di, lib, rtol=0, atol=1e-12 * n)


def test_fft1d_impulse_and_single_mode():
    n = 32
    re = np.zeros(n); im = np.zeros(n); re[3] = 1.0
    fr, fi = dnsref.fft1d(re, im, -1)
    k = np.arange(n)
    assert np.allclose(fr, np.cos(2 * np.pi * 3 * k / n), atol=1e-14)
    assert np.allclose(fi, -np.sin(2 * np.pi * 3 * k / n), atol=1e-14)  # forward sign is exp(-i...)


def test_fft3_matches_library_nonsquare():
    r = rng(7)
    shape = (8, 4, 16)  # nz, ny, nx
    a = r.standard_normal(shape) + 1j * r.standard_normal(shape)
    fr, fi = dnsref.fft3(a.real, a.imag, -1)
    assert np.allclose(fr + 1j * fi, np.fft.fftn(a), atol=1e-11)
    br, bi = dnsref.fft3(fr, fi, +1)
    assert np.allclose((br + 1j * bi) / a.size, a, atol=1e-13)


# ---------------------------------------------------------------- dense operator (P1, P2)
def _d1(n, h):
    """Central first-difference circulant matrix, built from index arithmetic."""
    D = np.zeros((n, n))
    for i in range(n):
        D[i, (i + 1) % n] += 1.0 / (2 * h)
        D[i, (i - 1) % n] -= 1.0 / (2 * h)
    return D


def _dense_ops(shape, d):
    nz, ny, nx = shape
    Ix, Iy, Iz = np.eye(nx), np.eye(ny), np.eye(nz)
    Dx = np.kron(Iz, np.kron(Iy, _d1(nx, d[0])))
    Dy = np.kron(Iz, np.kron(_d1(ny, d[1]), Ix))
    Dz = np.kron(_d1(nz, d[2]), np.kron(Iy, Ix))
    return Dx, Dy, Dz


def test_P1_dense_operator_spectrum_and_null_space():
    shape, d = (8, 8, 8), (0.5, 0.7, 1.1)
    Dx, Dy, Dz = _dense_ops(shape, d)
    L = Dx @ Dx + Dy @ Dy + Dz @ Dz
    assert np.allclose(L, L.T, atol=1e-14)
    ev = np.sort(np.linalg.eigvalsh(L))
    o = mk(shape, d)
    lam = np.sort([o.eig(kx, ky, kz) for kz in range(8) for ky in range(8) for kx in range(8)])
    assert np.allclose(ev, lam, atol=1e-12)
    assert int(np.sum(np.abs(ev) < 1e-10)) == 8


def test_P2_bruteforce_dense_poisson():
    shape, d = (8, 8, 8), (0.5, 0.7, 1.1)
    Dx, Dy, Dz = _dense_ops(shape, d)
    L = Dx @ Dx + Dy @ Dy + Dz @ Dz
    w, V = np.linalg.eigh(L)
    Nn = V[:, np.abs(w) < 1e-10]          # orthonormal null-space basis (8 vectors)
    assert Nn.shape[1] == 8
    r = rng(11).standard_normal(512)
    r_perp = r - Nn @ (Nn.T @ r)
    p_dense = np.linalg.solve(L + Nn @ Nn.T, r_perp)   # Gaussian elimination, unique solution _|_ null
    o = mk(shape, d)
    p = o.poisson(r.reshape(shape)).ravel()            # the oracle zeroes the null modes of r itself
    assert np.abs(p - p_dense).max() <= 1e-12 * np.abs(p_dense).max()
    assert np.abs(Nn.T @ p).max() < 1e-13              # result carries no null-space component


def test_P3_manufactured_single_modes():
    shape, d = (16, 8, 32), (0.3, 0.45, 0.2)
    nz, ny, nx = shape
    o = mk(shape, d)
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    for (kx, ky, kz, ph) in [(1, 0, 0, 0.3), (0, 1, 0, 0.1), (0, 0, 1, 1.0), (3, 2, 5, 0.7), (8, 2, 4, 0.2),
                             (15, 3, 7, 0.5), (31, 7, 15, 0.4), (16, 1, 0, 0.9)]:
        p = np.cos(2 * np.pi * kx * i / nx + ph) * np.cos(2 * np.pi * ky * j / ny + 2 * ph) * \
            np.cos(2 * np.pi * kz * k / nz - ph)
        lam = -(math.sin(2 * math.pi * kx / nx) ** 2 / d[0] ** 2 + math.sin(2 * math.pi * ky / ny) ** 2 / d[1] ** 2 +
                math.sin(2 * math.pi * kz / nz) ** 2 / d[2] ** 2)
        assert abs(o.eig(kx, ky, kz) - lam) < 1e-13 * abs(lam)
        got = o.poisson(lam * p)
        assert np.abs(got - p).max() < 1e-13, (kx, ky, kz)


def test_P4_projection_gives_roundoff_divergence():
    shape, d = (24, 16, 32), (0.11, 0.17, 0.13)
    r = rng(4)
    us, vs, ws = (r.standard_normal(shape) for _ in range(3))
    o = mk(shape, d)
    dv = o.div(us, vs, ws)
    # independent check of the divergence itself (np.roll form of the central difference)
    ref = (np.roll(us, -1, 2) - np.roll(us, 1, 2)) / (2 * d[0]) + (np.roll(vs, -1, 1) - np.roll(vs, 1, 1)) / (2 * d[1]) \
        + (np.roll(ws, -1, 0) - np.roll(ws, 1, 0)) / (2 * d[2])
    assert np.abs(dv - ref).max() < 1e-12
    p = o.poisson(dv)
    u, v, w = o.project(us, vs, ws, p)
    assert np.abs(o.div(u, v, w)).max() <= 1e-12 * np.abs(dv).max()
    # gradient sign/axis: for p = sin(2 pi i/nx) only u changes, by -cos()*sin(2pi/nx)/dx
    nz, ny, nx = shape
    i = np.arange(nx)
    p1 = np.broadcast_to(np.sin(2 * np.pi * i / nx), shape).copy()
    u1, v1, w1 = o.project(us, vs, ws, p1)
    assert np.array_equal(v1, vs) and np.array_equal(w1, ws)
    assert np.allclose(us - u1, np.broadcast_to(np.cos(2 * np.pi * i / nx) * math.sin(2 * math.pi / nx) / d[0], shape),
                       atol=1e-13)


# ---------------------------------------------------------------- convection identities (P5, P6)
def _solenoidal(shape, d, seed):
    """Discretely solenoidal random field built here with numpy FFTs (independent of the oracle)."""
    r = rng(seed)
    nz, ny, nx = shape
    f = [np.fft.fftn(r.standard_normal(shape)) for _ in range(3)]
    mx = np.sin(2 * np.pi * np.fft.fftfreq(nx))[None, None, :] / d[0]
    my = np.sin(2 * np.pi * np.fft.fftfreq(ny))[None, :, None] / d[1]
    mz = np.sin(2 * np.pi * np.fft.fftfreq(nz))[:, None, None] / d[2]
    m2 = mx * mx + my * my + mz * mz
    ok = m2 > 1e-14
    dot = np.where(ok, (mx * f[0] + my * f[1] + mz * f[2]) / np.where(ok, m2, 1.0), 0.0)
    return [np.fft.ifftn(f[0] - dot * mx).real, np.fft.ifftn(f[1] - dot * my).real, np.fft.ifftn(f[2] - dot * mz).real]


def test_P5_skew_symmetric_energy_identities():
    shape, d = (12, 16, 20), (0.1, 0.13, 0.09)
    r = rng(5)
    u, v, w, c = (r.standard_normal(shape) for _ in range(4))
    o = mk(shape, d, nu=0.0, alpha_c=0.0)
    Fu, Fv, Fw, Fc = o.rhs(u, v, w, c)
    scale = np.abs(u * Fu).sum() + np.abs(v * Fv).sum() + np.abs(w * Fw).sum()
    assert abs((u * Fu + v * Fv + w * Fw).sum()) < 1e-13 * scale       # kinetic energy conserved for ANY u
    assert abs((c * Fc).sum()) < 1e-13 * np.abs(c * Fc).sum()          # scalar variance conserved
    assert abs(Fu.sum()) > 1e-3 * np.abs(Fu).sum() * 1e-3             # momentum NOT conserved if div u != 0


def test_P6_momentum_conserved_for_solenoidal_field():
    shape, d = (12, 16, 20), (0.1, 0.13, 0.09)
    u, v, w = _solenoidal(shape, d, 6)
    c = rng(66).standard_normal(shape)
    o = mk(shape, d, nu=0.3, alpha_c=0.2)
    assert np.abs(o.div(u, v, w)).max() < 1e-11
    F = o.rhs(u, v, w, c)
    for f in F:
        assert abs(f.sum()) < 1e-11 * np.abs(f).sum()


def test_rhs_constant_advection_of_linear_product():
    """Sign and axis pin of each convective term: u = (U,V,W) constant, c = one cosine per axis.
    F_c = -(U d_x c + V d_y c + W d_z c) with the central-difference symbol sin(theta)/D."""
    shape, d = (8, 16, 32), (0.2, 0.3, 0.5)
    nz, ny, nx = shape
    U, V, W = 0.7, -0.4, 1.3
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    o = mk(shape, d)
    one = np.ones(shape)
    for ax, (n, idx, vel, h) in enumerate([(nx, i, U, d[0]), (ny, j, V, d[1]), (nz, k, W, d[2])]):
        th = 2 * np.pi * 3 / n
        c = np.sin(th * idx)
        Fc = o.rhs(U * one, V * one, W * one, c)[3]
        assert np.allclose(Fc, -vel * np.cos(th * idx) * math.sin(th) / h, atol=1e-13), ax


# ---------------------------------------------------------------- exact linear solutions (P7, P8)
def _G(z):
    return 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24


def test_P7_shear_flow_exact_rk4_amplification():
    shape, d = (16, 8, 4), (0.4, 0.25, 0.2)
    nz, ny, nx = shape
    nu, ac, dt = 0.05, 0.03, 0.11
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    ty, tz = 2 * np.pi * 2 / ny, 2 * np.pi * 3 / nz
    mode = np.cos(ty * j + 0.3) * np.cos(tz * k - 0.2)
    zero = np.zeros(shape)
    o = mk(shape, d, nu=nu, alpha_c=ac, dt=dt)
    o.set_fields(1.7 * mode, zero, zero, -0.6 * mode)
    nsteps = 3
    o.step(nsteps)
    f = o.fields()
    sym = (2 * math.cos(ty) - 2) / d[1] ** 2 + (2 * math.cos(tz) - 2) / d[2] ** 2
    assert np.abs(f["u"] - 1.7 * mode * _G(nu * dt * sym) ** nsteps).max() < 1e-14
    assert np.abs(f["c"] + 0.6 * mode * _G(ac * dt * sym) ** nsteps).max() < 1e-14
    assert np.abs(f["v"]).max() == 0 and np.abs(f["w"]).max() == 0 and np.abs(f["p"]).max() < 1e-15


def test_P8_uniform_advection_exact_rk4_amplification():
    shape, d = (8, 16, 32), (0.2, 0.3, 0.5)
    nz, ny, nx = shape
    U, V, W = 0.7, -0.4, 1.3
    ac, dt = 0.02, 0.05
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    tx, ty, tz = 2 * np.pi * 3 / nx, 2 * np.pi * 1 / ny, 2 * np.pi * 2 / nz
    phase = tx * i + ty * j + tz * k
    one = np.ones(shape)
    o = mk(shape, d, nu=0.01, alpha_c=ac, dt=dt)
    o.set_fields(U * one, V * one, W * one, np.cos(phase))
    o.step(2)
    f = o.fields()
    z = dt * (-1j * (U * math.sin(tx) / d[0] + V * math.sin(ty) / d[1] + W * math.sin(tz) / d[2])
              + ac * ((2 * math.cos(tx) - 2) / d[0] ** 2 + (2 * math.cos(ty) - 2) / d[1] ** 2 +
                      (2 * math.cos(tz) - 2) / d[2] ** 2))
    expect = (np.exp(1j * phase) * _G(z) ** 2).real
    assert np.abs(f["c"] - expect).max() < 1e-14
    assert np.abs(f["u"] - U).max() < 1e-14 and np.abs(f["v"] - V).max() < 1e-14 and np.abs(f["w"] - W).max() < 1e-14


# ---------------------------------------------------------------- paper's channel case (P9)
def test_P9_poiseuille_fixed_point_with_mask_and_body_force():
    """U(y) = (-b_x/2nu) y^2 + (b_x D/2nu) y is recovered in the masked channel.
    Discretely it is an exact fixed point (the 3-point Laplacian is exact on a parabola)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "poiseuille.txt")) if not l.startswith("#")]
    U = np.array([float(r[1]) for r in rows])
    bx, nu, ny, dy, wall = 1.0e-3, 0.05, 32, 0.25, 2
    shape = (4, ny, 8)
    mask = np.ones(shape, dtype=np.uint8)
    mask[:, :wall, :] = 0
    mask[:, ny - wall:, :] = 0
    u0 = np.broadcast_to(U[None, :, None], shape).copy()
    zero = np.zeros(shape)
    o = mk(shape, (0.3, dy, 0.4), nu=nu, alpha_c=nu, dt=0.2, mask=mask, body=(bx, 0.0, 0.0), n_piter=4)
    o.set_fields(u0, zero, zero, mask.astype(float))
    o.step(5)
    f = o.fields()
    assert np.abs(f["u"] - u0).max() < 1e-13 * U.max()
    assert np.abs(f["v"]).max() < 1e-15 and np.abs(f["w"]).max() < 1e-15 and np.abs(f["p"]).max() < 1e-15
    assert np.abs(f["c"] - mask).max() < 1e-14          # dc/dn = 0 at the walls keeps c = 1 in the fluid
    # bulk velocity of the paper's closed form, continuous: b_x D^2 / (12 nu); the sampled mean is within O(dy^2)
    D = (ny - wall - (wall - 1)) * dy
    assert abs(U[wall - 1:ny - wall + 1].sum() * dy / D - bx * D * D / (12 * nu)) < 2e-3 * bx * D * D / (12 * nu)


# ---------------------------------------------------------------- nonlinear closed forms (P10-P12)
def _tgv2d(n, nu, dt, steps, flags=0):
    h = 2 * math.pi / n
    x = np.arange(n) * h
    X, Y = np.meshgrid(x, x, indexing="xy")   # arrays [j, i]
    u2, v2 = np.sin(X) * np.cos(Y), -np.cos(X) * np.sin(Y)
    shape = (4, n, n)
    u = np.broadcast_to(u2, shape).copy()
    v = np.broadcast_to(v2, shape).copy()
    o = mk(shape, (h, h, h), nu=nu, alpha_c=nu, dt=dt, flags=flags)
    o.set_fields(u, v, np.zeros(shape), np.zeros(shape))
    o.step(steps)
    f = o.fields()
    lam2 = 2 * (2 * math.cos(h) - 2) / h ** 2
    return f, u, v, lam2


def test_P11_taylor_green_2d_first_order_in_dt():
    """2-D Taylor-Green is an exact NS solution; with one projection per step the scheme
    is first order in dt: the error halves with dt (ratio 2 +- 0.1)."""
    n, nu, T = 32, 0.01, 0.3 * (2 * math.pi / 32) * 8
    errs = []
    for steps in (8, 16, 32):
        f, u, v, lam2 = _tgv2d(n, nu, T / steps, steps)
        errs.append(np.abs(f["u"] - u * math.exp(nu * lam2 * T)).max())
    assert 1.9 < errs[0] / errs[1] < 2.1 and 1.9 < errs[1] / errs[2] < 2.1
    assert errs[0] < 5e-2


def test_P11b_per_stage_projection_is_rk4_exact():
    """NEXT-2 variant (flags bit1): projecting every stage makes 2-D Taylor-Green decay by RK4's G(z)."""
    n, nu = 32, 0.01
    dt = 0.3 * 2 * math.pi / n
    f, u, v, lam2 = _tgv2d(n, nu, dt, 4, flags=2)
    g = _G(nu * lam2 * dt) ** 4
    assert np.abs(f["u"] - u * g).max() < 1e-13 and np.abs(f["v"] - v * g).max() < 1e-13


def test_P10_linear_limit_of_full_step():
    case = cases.taylor_green(16)
    eps = 1e-6
    o = mk(case["shape"], case["d"], nu=case["nu"], alpha_c=case["nu"], dt=case["dt"])
    o.set_fields(eps * case["u"], eps * case["v"], eps * case["w"], case["c"])
    o.step(4)
    h = case["d"][0]
    lam3 = 3 * (2 * math.cos(h) - 2) / h ** 2
    g = _G(case["nu"] * lam3 * case["dt"]) ** 4
    f = o.fields()
    assert np.abs(f["u"] - eps * case["u"] * g).max() < 1e-5 * eps


def test_P12_config1_taylor_green_energy_decay():
    gold = np.array([[float(x) for x in l.split()] for l in open(os.path.join(GOLD, "tgv32_energy.txt"))
                     if not l.startswith("#")])
    case = cases.config(1)
    o = mk(case["shape"], case["d"], nu=case["nu"], alpha_c=case["alpha_c"], dt=case["dt"], n_piter=1)
    o.set_fields(case["u"], case["v"], case["w"], case["c"])
    assert np.abs(o.div(case["u"], case["v"], case["w"])).max() < 1e-14   # initial field discretely solenoidal
    E0 = sum((case[k] ** 2).sum() for k in "uvw")
    done = 0
    for step, e_proto, e_lin in gold:
        o.step(int(step) - done)
        done = int(step)
        f = o.fields()
        E = sum((f[k] ** 2).sum() for k in "uvw") / E0
        assert abs(E - e_proto) < 5e-8, (step, E)        # the digits SURVEY.md prints
        assert abs(E / e_lin - 1) < 0.02                  # "analytic viscous decay", 2 % (splitting + transfer)
        assert np.abs(o.div(f["u"], f["v"], f["w"])).max() < 1e-13
    h = case["d"][0]
    lam3 = 3 * (2 * math.cos(h) - 2) / h ** 2
    assert abs(math.exp(2 * case["nu"] * lam3 * 10 * case["dt"]) - gold[-1, 2]) < 1e-5


# ---------------------------------------------------------------- mask and eq. 9 (P13)
def _masked_lap_dense_free(p, beta, d):
    """sum_a delta_a[ beta delta_a p ] (eq. 7's operator) written with np.roll."""
    out = np.zeros_like(p)
    for ax, h in ((2, d[0]), (1, d[1]), (0, d[2])):
        g = beta * (np.roll(p, -1, ax) - np.roll(p, 1, ax)) / (2 * h)
        out += (np.roll(g, -1, ax) - np.roll(g, 1, ax)) / (2 * h)
    return out


def test_eq9_fixed_point_is_the_masked_operator():
    """If p satisfies eq. 7, sum_a delta_a[beta delta_a p] = d, then eq. 9's right-hand side equals
    sum_a delta_a delta_a p and one solve returns p (up to its null-space part)."""
    case = cases.duct_room(32, 16, 16)
    shape, d, beta = case["shape"], case["d"], case["mask"].astype(float)
    o = mk(shape, d, mask=case["mask"])
    p = rng(9).standard_normal(shape)
    p = o.poisson(_masked_lap_dense_free(p, np.ones(shape), d))     # strip the null-space component
    dd = _masked_lap_dense_free(p, beta, d)
    r = o.poisson_rhs(dd, p)
    assert np.abs(r - _masked_lap_dense_free(p, np.ones(shape), d)).max() < 1e-10 * np.abs(r).max()
    assert np.abs(o.poisson(r) - p).max() < 1e-11 * np.abs(p).max()
    # with beta == 1 the bracket vanishes identically
    o1 = mk(shape, d)
    assert np.array_equal(o1.poisson_rhs(dd, p), dd)


def test_P13_masked_step_invariants():
    case = cases.duct_room(32, 16, 16, steps=5)
    beta = case["mask"].astype(float)

    def run(n_piter, steps, cold=False):
        o = mk(case["shape"], case["d"], nu=case["nu"], alpha_c=case["alpha_c"], dt=case["dt"], mask=case["mask"],
               sources=case["sources"], n_piter=n_piter)
        o.set_fields(case["u"], case["v"], case["w"], case["c"])
        o.step(steps)
        return o, o.fields()

    resid = []
    for P in (1, 2, 4, 8, 40):
        o, f = run(P, 1)
        solid = case["mask"] == 0
        for k in "uvwc":
            assert np.all(f[k][solid] == 0.0) and not np.any(np.signbit(f[k][solid]))   # bit-exact +0.0
        resid.append(np.abs(o.div(f["u"], f["v"], f["w"]) * beta).max())
    assert all(resid[i + 1] <= resid[i] * (1 + 1e-12) for i in range(len(resid) - 1)), resid
    assert resid[-1] < 0.5 * resid[0]
    o, f = run(4, 5)
    assert all(np.isfinite(f[k]).all() for k in "uvwcp")
    # the source drives the duct towards u_set
    s = case["sources"][0]
    assert f["u"][s["lo"][2] + 1, s["lo"][1] + 1, 0] > 0.5 * s["u_set"][0]


def test_source_table_eq5():
    """eq. 5: S = 1 at the centre, 1/2 at |x-xc| = W/2, -> 0 far away, symmetric,
    periodic; binary box for B <= 0."""
    n, d = 64, 0.25
    t = dnsref.source_table(n, d, lo=20, size=9, B=4.0)       # centre at cell 24, W/2 = 4.5 cells
    assert t[24] == 1.0
    assert np.allclose(t[24 - 10:24], t[25:24 + 11][::-1])
    x = abs(np.arange(n) - 24.0) * d
    W2 = 4.5 * d
    with np.errstate(divide="ignore"):
        ref = 0.5 * (1 - np.tanh(4.0 * (x / W2 - W2 / x)))
    assert np.allclose(t, ref, atol=1e-15)
    assert t[60] < 1e-12 and np.all((t >= 0) & (t <= 1))
    half = dnsref.source_table(n, d, lo=20, size=8, B=4.0)     # W/2 = 4 cells: cell 23.5 +- 4 not on grid
    assert abs(dnsref.source_table(64, 1.0, 10, 4, 3.0)[13] - 0.5 * (1 - math.tanh(3.0 * (1.5 / 2 - 2 / 1.5)))) < 1e-15
    b = dnsref.source_table(16, 1.0, lo=14, size=4, B=0.0)
    assert list(np.nonzero(b)[0]) == [0, 1, 14, 15]
    w = dnsref.source_table(16, 1.0, lo=14, size=5, B=2.0)     # wraps across the seam: centre at cell 0
    assert w[0] == 1.0 and np.allclose(w[1:8], w[15:8:-1])
    assert half.max() <= 1.0


# ---------------------------------------------------------------- source relaxation term of eqs. 2-3 (P18)
# S (phi_set - phi)/tau_f, PAPER.md:49-52 (eqs. 2-3); readings R8-R10.  Closed forms only: nothing
# below calls the oracle to make its own expectation.
def _src(lo, size, u_set=(0.0, 0.0, 0.0), c_set=0.0, tau_f=1.0, comps=0xF, B=(0.0, 0.0, 0.0)):
    return dict(lo=lo, size=size, B=B, u_set=u_set, c_set=c_set, tau_f=tau_f, comps=comps)


def _box_indicator(shape, lo, size):
    """1 inside the index box lo..lo+size-1 (x,y,z order, wrapping), written from index arithmetic."""
    nz, ny, nx = shape
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return (((i - lo[0]) % nx < size[0]) & ((j - lo[1]) % ny < size[1]) & ((k - lo[2]) % nz < size[2])).astype(float)


@pytest.mark.parametrize("comps", range(16))
def test_P18_source_zero_field_binary_box_every_component_mask(comps):
    """Zero fields, binary box (B <= 0): F_phi = phi_set/tau_f inside the box for the enabled components (bit m of
    `comps` <-> m-th of u,v,w,c), exactly 0 everywhere else and for the disabled ones."""
    shape, tau = (8, 12, 16), 0.37
    sets = (0.9, -1.7, 2.3, 0.6)
    lo, size = (13, 3, 6), (6, 4, 5)          # wraps through the x seam and the z seam
    o = mk(shape, (0.5, 0.25, 0.2), nu=0.3, alpha_c=0.2, sources=[_src(lo, size, sets[:3], sets[3], tau, comps)])
    z = np.zeros(shape)
    F = o.rhs(z, z, z, z)
    inside = _box_indicator(shape, lo, size)
    assert inside.sum() == 6 * 4 * 5
    for m in range(4):
        expect = inside * (sets[m] / tau) if comps & (1 << m) else z
        assert np.array_equal(F[m], expect), (comps, m)


def test_P18_source_relaxation_exact_rk4_decay_towards_the_set_value():
    """S == 1 over the whole periodic box, uniform fields, no mask: convection, diffusion and the divergence vanish
    identically, so each component obeys d(phi)/dt = (phi_set - phi)/tau_f and RK4 gives
    phi_n = phi_set + (phi_0 - phi_set) G(-dt/tau_f)^n with the polynomial G of P7/P8."""
    shape, dt, tau, n = (8, 8, 16), 0.05, 0.13, 5
    sets, init = (0.8, -0.3, 0.45, 2.0), (0.1, 0.2, -0.15, 0.5)
    o = mk(shape, (0.1, 0.2, 0.15), nu=0.0, alpha_c=0.0, dt=dt,
           sources=[_src((3, 1, 5), (16, 8, 8), sets[:3], sets[3], tau)])
    one = np.ones(shape)
    o.set_fields(*(v * one for v in init))
    o.step(n)
    f = o.fields()
    g = _G(-dt / tau).real ** n
    for m, key in enumerate("uvwc"):
        expect = sets[m] + (init[m] - sets[m]) * g
        assert np.abs(f[key] - expect).max() < 1e-14, key
    assert np.abs(f["p"]).max() < 1e-14
    # a different tau_f per source, one source per component: each decays at its own rate
    taus = (0.07, 0.11, 0.2, 0.31)
    o = mk(shape, (0.1, 0.2, 0.15), dt=dt, sources=[_src((0, 0, 0), (16, 8, 8), sets[:3], sets[3], taus[m], 1 << m)
                                                    for m in range(4)])
    o.set_fields(*(v * one for v in init))
    o.step(n)
    f = o.fields()
    for m, key in enumerate("uvwc"):
        expect = sets[m] + (init[m] - sets[m]) * _G(-dt / taus[m]).real ** n
        assert np.abs(f[key] - expect).max() < 1e-14, key


def test_P18_overlapping_sources_add():
    """Two boxes that overlap: F = sum_s S_s (set_s - phi)/tau_s (reading R8), here with a uniform non-zero field."""
    shape = (8, 8, 16)
    a = _src((2, 1, 1), (8, 5, 4), (1.0, 0.5, -0.25), 0.7, 0.2)
    b = _src((6, 3, 2), (6, 4, 5), (-2.0, 0.125, 0.75), 0.1, 0.5, comps=0b1011)   # b does not force w
    o = mk(shape, (1.0, 1.0, 1.0), sources=[a, b])
    phi = (0.3, -0.2, 0.1, 0.4)
    one = np.ones(shape)
    F = o.rhs(*(v * one for v in phi))
    Ia, Ib = _box_indicator(shape, a["lo"], a["size"]), _box_indicator(shape, b["lo"], b["size"])
    assert (Ia * Ib).sum() == 4 * 3 * 3                     # they do overlap
    seta, setb = a["u_set"] + (a["c_set"],), b["u_set"] + (b["c_set"],)
    for m in range(4):
        eb = Ib * (setb[m] - phi[m]) / b["tau_f"] if b["comps"] & (1 << m) else 0.0
        expect = Ia * (seta[m] - phi[m]) / a["tau_f"] + eb
        assert np.abs(F[m] - expect).max() < 1e-15, m


def test_P18_smooth_source_enters_to_the_first_power():
    """B > 0 (eq. 5): F = S_x S_y S_z phi_set/tau_f with each factor the tanh window written out here
    -- the first power of S, and the product of the three one-dimensional factors."""
    shape, d = (16, 16, 32), (0.25, 0.5, 0.125)
    lo, size, B = (10, 4, 5), (9, 5, 7), (4.0, 2.5, 3.0)
    tau, cset = 0.4, 1.5

    def window(n, h, l, s, b):
        xc, w2 = (l + 0.5 * (s - 1)) * h, 0.5 * s * h
        r = np.abs(np.arange(n) * h - xc)
        r = np.minimum(r, n * h - r)                       # minimum image
        with np.errstate(divide="ignore"):
            return 0.5 * (1.0 - np.tanh(b * (r / w2 - w2 / r)))

    sx, sy, sz = (window(shape[2 - a], d[a], lo[a], size[a], B[a]) for a in range(3))
    S = sz[:, None, None] * sy[None, :, None] * sx[None, None, :]
    assert S.max() == 1.0 and ((S > 0.1) & (S < 0.9)).sum() > 50          # really smooth: S and S^2 differ
    o = mk(shape, d, sources=[_src(lo, size, (0.0, 0.0, -1.0), cset, tau, comps=0b1100, B=B)])
    z = np.zeros(shape)
    F = o.rhs(z, z, z, z)
    assert np.abs(F[3] - S * cset / tau).max() < 1e-15 and np.abs(F[2] + S / tau).max() < 1e-15
    assert not F[0].any() and not F[1].any()
    assert np.abs(F[3] - S * S * cset / tau).max() > 0.1              # what a squared window would give


def test_P18_set_fields_selects_plus_zero_in_solid_cells():
    """PAPER.md:58 as a select (reading R7): whatever the caller passes in solid cells -- here large values, negative
    values and a NaN -- is stored as +0.0; fluid cells and the whole of p are stored untouched."""
    r = rng(21)
    shape = (6, 8, 10)
    mask = (r.random(shape) < 0.6).astype(np.uint8)
    o = mk(shape, mask=mask)
    fld = [r.standard_normal(shape) * 1e3 - 5.0 for _ in range(5)]
    solid = mask == 0
    fld[0][solid] = -7.0
    fld[3][tuple(np.argwhere(solid)[0])] = np.nan
    o.set_fields(*fld[:4], p=fld[4])
    f = o.fields()
    for m, key in enumerate("uvwc"):
        assert np.all(f[key][solid] == 0.0) and not np.any(np.signbit(f[key][solid])), key
        assert np.array_equal(f[key][~solid], fld[m][~solid]), key
    assert np.array_equal(f["p"], fld[4])


# ---------------------------------------------------------------- symmetries (P14)
def _run_case(case, steps, n_piter=None):
    o = mk(case["shape"], case["d"], nu=case["nu"], alpha_c=case["alpha_c"], dt=case["dt"], mask=case["mask"],
           sources=case["sources"], body=case["body"], n_piter=n_piter or case["n_piter"])
    o.set_fields(case["u"], case["v"], case["w"], case["c"])
    o.step(steps)
    return o.fields()


def test_P14_shift_symmetry():
    case = cases.duct_room(32, 16, 16)
    f0 = _run_case(case, 2)
    sh = (3, 5, 7)  # z, y, x
    c2 = dict(case)
    for k in "uvwc":
        c2[k] = np.roll(case[k], sh, (0, 1, 2))
    c2["mask"] = np.roll(case["mask"], sh, (0, 1, 2))
    nz, ny, nx = case["shape"]
    c2["sources"] = [dict(s, lo=((s["lo"][0] + sh[2]) % nx, (s["lo"][1] + sh[1]) % ny, (s["lo"][2] + sh[0]) % nz))
                     for s in case["sources"]]
    f1 = _run_case(c2, 2)
    for k in "uvwcp":
        ref = np.roll(f0[k], sh, (0, 1, 2))
        assert np.abs(f1[k] - ref).max() <= 1e-12 * max(np.abs(ref).max(), 1e-300), k


def test_P14_axis_permutation_symmetry():
    """Swap x and z everywhere (fields, components, spacings, mask, sources): outputs swap too."""
    case = cases.duct_room(32, 16, 8)
    case["d"] = (0.05, 0.07, 0.06)
    f0 = _run_case(case, 2)
    T = lambda a: np.ascontiguousarray(a.transpose(2, 1, 0))
    c2 = dict(case)
    c2["shape"] = case["shape"][::-1]
    c2["d"] = case["d"][::-1]
    c2["u"], c2["v"], c2["w"], c2["c"] = T(case["w"]), T(case["v"]), T(case["u"]), T(case["c"])
    c2["mask"] = T(case["mask"])
    c2["sources"] = [dict(s, lo=s["lo"][::-1], size=s["size"][::-1], u_set=s["u_set"][::-1]) for s in case["sources"]]
    f1 = _run_case(c2, 2)
    for a, b in (("u", "w"), ("v", "v"), ("w", "u"), ("c", "c"), ("p", "p")):
        ref = T(f0[b])
        assert np.abs(f1[a] - ref).max() <= 1e-12 * max(np.abs(ref).max(), 1e-300), a


def test_momentum_drift_bound_full_step():
    """P6, full step: stages are unprojected, so mean velocity drifts slightly -- bound, not equality."""
    case = cases.periodic_turbulence(32, steps=1)
    f = _run_case(case, 1)
    for k in "uvw":
        assert 0 < abs(f[k].mean() - case[k].mean()) < 1e-4      # 32^3, k0 = 4: ~2e-5 u' per step


# ---------------------------------------------------------------- eq. 6 filter (P15, NEXT-1)
def test_P15_filter_mode_amplification_closed_form():
    """A Fourier mode is multiplied by G = 1 - (64/pi^6) sum_a sin^6(theta_a/2): the symbol of the central
    7-point sixth-derivative stencil times gamma_a = Delta_a^6/pi^6 (eq. 6); Delta cancels, so
    unequal spacings give the same factor.  Constant fields pass unchanged; a one-axis Nyquist mode is
    damped by 1 - 64/pi^6 (not zeroed: reading R23)."""
    shape = (16, 8, 32)
    nz, ny, nx = shape
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    for d in [(0.1, 0.1, 0.1), (0.05, 0.2, 0.13)]:
        o = mk(shape, d)
        for (kx, ky, kz, ph) in [(0, 0, 0, 0.3), (1, 0, 0, 0.0), (3, 2, 5, 0.7), (nx // 2, 0, 0, 0.0), (nx // 2, ny // 2, nz // 2, 0.0),
                                 (nx // 4, ny // 4, 1, 1.1)]:
            th = (2 * np.pi * kx / nx, 2 * np.pi * ky / ny, 2 * np.pi * kz / nz)
            f = np.cos(th[0] * i + th[1] * j + th[2] * k + ph)
            G = 1.0 - 64.0 / np.pi ** 6 * sum(np.sin(t / 2) ** 6 for t in th)
            assert np.abs(o.filter(f) - G * f).max() <= 2e-14, (d, kx, ky, kz)
    assert abs((1.0 - 64.0 / np.pi ** 6) - 0.93343) < 1e-5


def test_P15_filter_stencil_is_cubed_second_difference_and_masked_by_select():
    """The 7-point weights (1,-6,15,-20,15,-6,1) are the second difference applied three times (binomial
    identity), built here from np.roll; solid cells come out as +0.0 exactly, fluid cells see the solid
    zeros like any other value."""
    rng = np.random.default_rng(15)
    shape = (8, 16, 8)
    f = rng.standard_normal(shape)
    mask = (rng.random(shape) > 0.2).astype(np.uint8)
    d2 = lambda a, ax: np.roll(a, 1, ax) - 2 * a + np.roll(a, -1, ax)
    ref = f + sum(d2(d2(d2(f, ax), ax), ax) for ax in range(3)) / np.pi ** 6
    got = mk(shape, (0.1, 0.2, 0.3)).filter(f)
    assert np.abs(got - ref).max() <= 1e-14
    fm = np.where(mask != 0, f, 0.0)
    refm = fm + sum(d2(d2(d2(fm, ax), ax), ax) for ax in range(3)) / np.pi ** 6
    gotm = mk(shape, (0.1, 0.2, 0.3), mask=mask).filter(fm)
    solid = mask == 0
    assert np.all(gotm[solid] == 0.0) and not np.any(np.signbit(gotm[solid]))
    assert np.abs(gotm - refm)[~solid].max() <= 1e-14


def test_P15_filtered_step_is_step_then_filter_and_stays_solenoidal():
    """flags bit 0: the step ends with eq. 6 on u, v, w, c (p untouched).  With beta == 1 the filter
    commutes with the central differences, so the divergence stays at round-off."""
    case = cases.periodic_turbulence(16, steps=1)
    kw = dict(nu=case["nu"], alpha_c=case["alpha_c"], dt=case["dt"], n_piter=1)
    a = mk(case["shape"], case["d"], **kw)
    b = mk(case["shape"], case["d"], flags=1, **kw)
    for o in (a, b):
        o.set_fields(case["u"], case["v"], case["w"], case["c"])
        o.step(1)
    fa, fb = a.fields(), b.fields()
    for k in "uvwc":
        assert np.abs(fb[k] - a.filter(fa[k])).max() <= 1e-15 * max(1.0, np.abs(fa[k]).max())
    assert np.array_equal(fa["p"], fb["p"])
    div = a.div(fb["u"], fb["v"], fb["w"])
    assert np.abs(div).max() <= 1e-12 * np.abs(fb["u"]).max() / min(case["d"])
    # a second step runs from the filtered state (the filter output is the state)
    b.step(1)
    assert np.isfinite(b.fields()["u"]).all()


# ---------------------------------------------------------------- reductions (P16, NEXT-3)
def test_P16_courant_number_closed_forms():
    """Co = dt max(|u|/dx + |v|/dy + |w|/dz): exact for a uniform field, picks out a single spike wherever it
    sits (incl. the last cell), scales with dt, ignores the sign."""
    shape, d = (8, 16, 32), (0.1, 0.2, 0.25)
    o = mk(shape, d, dt=0.5)
    one = np.ones(shape)
    o.set_fields(0.3 * one, -0.4 * one, 0.5 * one, 0 * one)
    assert o.courant() == 0.5 * (0.3 / 0.1 + 0.4 / 0.2 + 0.5 / 0.25)
    for pos in [(0, 0, 0), (7, 15, 31), (3, 9, 17)]:
        u = 0.3 * one
        u[pos] = -2.0
        o.set_fields(u, -0.4 * one, 0.5 * one, 0 * one)
        assert o.courant() == 0.5 * (2.0 / 0.1 + 0.4 / 0.2 + 0.5 / 0.25)
    o.set_dt(0.25)
    assert o.courant() == 0.25 * (2.0 / 0.1 + 0.4 / 0.2 + 0.5 / 0.25)
    # the step uses the new dt: shear-flow decay factor of P7 with dt = 0.25
    with pytest.raises(ValueError):
        o.set_dt(0.0)


def test_P16_set_dt_changes_the_step():
    """Two steps of dt/2 set through set_dt equal two steps of an oracle created with dt/2, and differ from dt."""
    case = cases.taylor_green(16)
    kw = dict(nu=case["nu"], alpha_c=case["alpha_c"], n_piter=1)
    a = mk(case["shape"], case["d"], dt=case["dt"], **kw)
    b = mk(case["shape"], case["d"], dt=case["dt"] / 2, **kw)
    for o in (a, b):
        o.set_fields(case["u"], case["v"], case["w"], case["c"])
    a.set_dt(case["dt"] / 2)
    a.step(2)
    b.step(2)
    assert all(np.array_equal(a.fields()[k], b.fields()[k]) for k in "uvwcp")


def test_P16_scalar_stats_closed_form_library_and_mask():
    """Mean/std of c over the fluid cells of a wrapping box: a full-box cosine mode has mean 0 and std 1/sqrt 2;
    numpy's own mean/std (pairwise sums, a different routine) agree on a random field with a random mask and a
    box that wraps through the periodic seam; solid cells are left out; an all-solid box gives (0, 0, 0)."""
    shape = (8, 16, 32)
    nz, ny, nx = shape
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    o = mk(shape)
    z = np.zeros(shape)
    o.set_fields(z, z, z, 3.0 + np.cos(2 * np.pi * 3 * i / nx + 0.4))
    m, s, n = o.scalar_stats((0, 0, 0), (nx, ny, nz))
    assert n == nx * ny * nz and abs(m - 3.0) < 1e-13 and abs(s - math.sqrt(0.5)) < 1e-13   # plain index-order sums of 4096 terms
    r = np.random.default_rng(16)
    c = r.standard_normal(shape)
    mask = (r.random(shape) > 0.3).astype(np.uint8)
    o = mk(shape, mask=mask)
    o.set_fields(z, z, z, c)
    lo, size = (28, 10, 6), (9, 11, 5)          # wraps in x, y and z
    sel = np.zeros(shape, bool)
    sel[np.ix_([(lo[2] + a) % nz for a in range(size[2])], [(lo[1] + a) % ny for a in range(size[1])],
               [(lo[0] + a) % nx for a in range(size[0])])] = True
    sel &= mask != 0
    m, s, n = o.scalar_stats(lo, size)
    assert n == sel.sum() and abs(m - c[sel].mean()) < 1e-14 and abs(s - c[sel].std()) < 1e-14
    solid = mk(shape, mask=np.zeros(shape, np.uint8))
    solid.set_fields(z, z, z, c)
    assert solid.scalar_stats((0, 0, 0), (4, 4, 4)) == (0.0, 0.0, 0)


# ---------------------------------------------------------------- Lagrangian particles (P17, NEXT-4)
def _particles(rows):
    return np.ascontiguousarray(np.array(rows, dtype=np.float64).T)          # (8, n): x y z u v w d rho_p


def test_P17_sedimentation_times_printed_in_the_paper():
    """Quiescent air: the settling velocity reached by the implicit Euler steps gives tau_s = h/v for h = 1.5 m of
    36/9/1 min for d = 5/10/30 um (tests/golden/sedimentation.txt) at the paper's rounding; the
    steady state satisfies eq. 10 with du_p/dt = 0:  (C_d/tau_p)(0 - w) + g = 0."""
    rows = [l.split() for l in open(os.path.join(GOLD, "sedimentation.txt")) if l.strip() and not l.startswith("#")]
    nu, rho_f, rho_p, g = 1.6e-5, 1.2, 1000.0, -9.81
    o = mk((8, 8, 8), (0.25, 0.25, 0.25), nu=nu, dt=0.05)            # dt >> tau_p: implicit Euler stays stable
    z = np.zeros((8, 8, 8))
    o.set_fields(z, z, z, z)
    st = _particles([[1.0, 1.0, 1.0, 0.0, 0.0, 0.0, float(d) * 1e-6, rho_p] for d, _ in rows])
    for _ in range(40):
        o.particles_step(st, rho_f, (0.0, 0.0, g))
    for q, (d, minutes) in enumerate(rows):
        d_m, w = float(d) * 1e-6, st[5, q]
        tau_p = rho_p * d_m ** 2 / (18 * rho_f * nu)
        cd = 1 + (abs(w) * d_m / nu) ** (2.0 / 3.0) / 6
        assert abs(cd / tau_p * (0.0 - w) + g) <= 1e-9 * abs(g)                     # fixed point of eq. 10
        tau_s_min = 1.5 / abs(w) / 60.0
        assert abs(tau_s_min - float(minutes)) <= 0.06 * float(minutes) + 0.05, (d, tau_s_min)
        assert st[3, q] == 0.0 and st[4, q] == 0.0


def test_P17_implicit_euler_is_bounded_and_unconditionally_stable():
    """From rest in still air |w| stays within [0, g tau_p] (C_d >= 1) and settles on the fixed point of eq. 10 for
    dt from 0.01 tau_p to 1e4 tau_p (C_d is lagged, reading R27, so the approach may overshoot the fixed point a
    little, but never the Stokes velocity)."""
    nu, rho_f, rho_p, d = 1.6e-5, 1.2, 1000.0, 30e-6
    tau_p = rho_p * d * d / (18 * rho_f * nu)
    for fac, nsteps in ((0.01, 3000), (1.0, 60), (1e4, 30)):
        o = mk((8, 8, 8), (1.0, 1.0, 1.0), nu=nu, dt=fac * tau_p)
        z = np.zeros((8, 8, 8))
        o.set_fields(z, z, z, z)
        st = _particles([[4.0, 4.0, 4.0, 0, 0, 0, d, rho_p]])
        for _ in range(nsteps):
            o.particles_step(st, rho_f, (0, 0, -9.81))
            assert 0.0 <= -st[5, 0] <= 9.81 * tau_p
        w = st[5, 0]
        cd = 1 + (abs(w) * d / nu) ** (2.0 / 3.0) / 6
        assert abs(cd / tau_p * (0.0 - w) - 9.81) <= 1e-6 * 9.81, fac


def test_P17_trilinear_interpolation_at_nodes_midpoints_and_across_the_seam():
    """A very light particle (dt C_d/tau_p ~ 1e12) takes the interpolated fluid velocity in one step: node value at a
    node, two-point mean at an edge midpoint (also across the periodic seam), eight-point mean at a cell centre;
    the position moves by dt u_p and wraps into [0, L)."""
    rng_ = np.random.default_rng(17)
    shape, d = (8, 8, 8), (0.5, 0.25, 0.2)
    u, v, w = (rng_.standard_normal(shape) for _ in range(3))
    o = mk(shape, d, nu=1.0, dt=1e-3)
    o.set_fields(u, v, w, np.zeros(shape))
    pts = [((3, 2, 1), [(3, 2, 1)]), ((3.5, 2, 1), [(3, 2, 1), (4, 2, 1)]), ((7.5, 0, 0), [(7, 0, 0), (0, 0, 0)]),
           ((2, 7.5, 3), [(2, 7, 3), (2, 0, 3)]), ((1, 1, 7.5), [(1, 1, 7), (1, 1, 0)]),
           ((1.5, 2.5, 3.5), [(a, b, c) for a in (1, 2) for b in (2, 3) for c in (3, 4)])]
    st = _particles([[p[0] * d[0], p[1] * d[1], p[2] * d[2], 0, 0, 0, 1e-9, 1.0] for p, _ in pts])
    x0 = st[:3].copy()
    o.particles_step(st, 1.0, (0, 0, 0))
    L = np.array([8 * d[0], 8 * d[1], 8 * d[2]])
    for q, (_, cells) in enumerate(pts):
        for comp, f in enumerate((u, v, w)):
            want = np.mean([f[c[2], c[1], c[0]] for c in cells])
            assert abs(st[3 + comp, q] - want) <= 1e-11 * max(1.0, abs(want)), (q, comp)
        xn = (x0[:, q] + 1e-3 * st[3:6, q]) % L
        assert np.abs(st[:3, q] - xn).max() <= 1e-14 and np.all(st[:3, q] >= 0) and np.all(st[:3, q] < L)


def test_P17_attached_particles_follow_the_stepped_field():
    """attach: the particle step runs after each fluid step with the NEW field -- equal to stepping by hand."""
    case = cases.taylor_green(16)
    kw = dict(nu=case["nu"], alpha_c=case["alpha_c"], dt=case["dt"], n_piter=1)
    a, b = mk(case["shape"], case["d"], **kw), mk(case["shape"], case["d"], **kw)
    for o in (a, b):
        o.set_fields(case["u"], case["v"], case["w"], case["c"])
    st_a = _particles([[1.0, 2.0, 3.0, 0, 0, 0, 1e-3, 1000.0], [5.0, 0.1, 6.2, 0.1, 0, 0, 2e-3, 500.0]])
    st_b = st_a.copy()
    a.particles_attach(st_a, 1.2, (0, 0, -9.81))
    a.step(3)
    for _ in range(3):
        b.step(1)
        b.particles_step(st_b, 1.2, (0, 0, -9.81))
    assert np.array_equal(st_a, st_b) and not np.array_equal(st_a[:3], _particles([[1.0, 2.0, 3.0, 0, 0, 0, 1e-3, 1000.0]])[:3])


# ---------------------------------------------------------------- pins added in round 3 ("What's weak" 1)
def _model_step(o, Q, p, dt, P, flags):
    """SURVEY.md 8(c)'s pseudo-code of one step written out here from the oracle's separately pinned operators
    (rhs: P5-P9/P18, div and project: P4, poisson_rhs: the eq. 9 fixed-point pin, poisson: P1-P3).  PAPER.md:43 (RK4,
    projection once per step), PAPER.md:104 (eq. 9 restarts "from the previous available value of pressure": p is
    state), R29 (flags bit 1: each stage projection iterates on a COPY of p^n and leaves p^n untouched)."""
    a, b = (0.5, 0.5, 1.0), (1.0 / 6.0, 1.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0)
    Qc, Qs = [q.copy() for q in Q], [q.copy() for q in Q]
    for s in range(4):
        F = o.rhs(*Qs)
        for m in range(4):
            Qc[m] = Qc[m] + (b[s] * dt) * F[m]
            if s < 3:
                Qs[m] = Q[m] + (a[s] * dt) * F[m]
        if s < 3 and flags & 2:
            ps = p.copy()
            d = o.div(Qs[0], Qs[1], Qs[2])
            for _ in range(P):
                ps = o.poisson(o.poisson_rhs(d, ps))
            Qs[0], Qs[1], Qs[2] = o.project(Qs[0], Qs[1], Qs[2], ps)
    d = o.div(Qc[0], Qc[1], Qc[2])
    for _ in range(P):
        p = o.poisson(o.poisson_rhs(d, p))
    u, v, w = o.project(Qc[0], Qc[1], Qc[2], p)
    return [u, v, w, Qc[3]], p


@pytest.mark.parametrize("flags", [0, 2])
def test_P19_step_orchestration_two_steps_warm_started_pressure(flags):
    """dnsref_step over TWO steps of a masked duct with sources and P = 3 equals the model above: the pressure the
    first step ends with is where the second step's eq. 9 iterations start (a cold start p = 0 in every step, or stage
    projections that iterate on p itself instead of a copy, change step 2 / the final p and turn this red)."""
    case = cases.duct_room(32, 16, 16, steps=2)
    P = 3
    kw = dict(nu=case["nu"], alpha_c=case["alpha_c"], dt=case["dt"], mask=case["mask"], sources=case["sources"],
              body=case["body"], n_piter=P)
    o = mk(case["shape"], case["d"], flags=flags, **kw)
    ops = mk(case["shape"], case["d"], **kw)                    # operators only; never stepped
    o.set_fields(case["u"], case["v"], case["w"], case["c"])
    ops.set_fields(case["u"], case["v"], case["w"], case["c"])
    f0 = ops.fields()                                           # masked initial data
    Q, p = [f0[k] for k in "uvwc"], np.zeros(case["shape"])
    for step in (1, 2):
        o.step(1)
        Q, p = _model_step(ops, Q, p, case["dt"], P, flags)
        f = o.fields()
        for k, m in zip("uvwcp", Q + [p]):
            assert np.abs(f[k] - m).max() <= 1e-15 * max(np.abs(m).max(), 1e-300), (step, k)
    assert np.abs(p).max() > 0
    # the model run cold (p = 0 at the start of step 2) is a different answer: the pin can tell the two apart
    o1 = mk(case["shape"], case["d"], flags=flags, **kw)
    o1.set_fields(case["u"], case["v"], case["w"], case["c"])
    o1.step(1)
    f1 = o1.fields()
    Qcold, pcold = _model_step(ops, [f1[k] for k in "uvwc"], np.zeros(case["shape"]), case["dt"], P, flags)
    assert np.abs(pcold - p).max() > 1e-6 * np.abs(p).max()


def test_P19_warm_start_leaves_a_smaller_masked_residual_than_a_cold_start():
    """SURVEY.md 8(c) S14 / PAPER.md:104: with the same number of eq. 9 iterations, a step that starts from the previous
    pressure ends with a smaller divergence in the fluid than one that starts from zero (the survey's probe found a
    factor ~10 after 100 steps; after 10 steps of this small duct the factor is already > 1.5)."""
    case = cases.duct_room(32, 16, 16, steps=10)
    beta = case["mask"].astype(float)
    kw = dict(nu=case["nu"], alpha_c=case["alpha_c"], dt=case["dt"], mask=case["mask"], sources=case["sources"],
              body=case["body"], n_piter=4)
    o = mk(case["shape"], case["d"], **kw)
    o.set_fields(case["u"], case["v"], case["w"], case["c"])
    o.step(9)
    f9 = o.fields()
    o.step(1)
    fw = o.fields()
    warm = np.abs(o.div(fw["u"], fw["v"], fw["w"]) * beta).max()
    oc = mk(case["shape"], case["d"], **kw)                                    # same state, pressure forgotten
    oc.set_fields(f9["u"], f9["v"], f9["w"], f9["c"])
    oc.step(1)
    fc = oc.fields()
    cold = np.abs(oc.div(fc["u"], fc["v"], fc["w"]) * beta).max()
    assert warm > 0 and cold > 1.5 * warm, (warm, cold)


def test_P20_scalar_wall_flux_vanishes_on_every_axis():
    """eq. 4, dc/dn = 0 at the immersed boundary: in a closed room with walls on all six faces and an
    obstacle, c = 1 in the fluid (0 in the solid) and no flow, the scalar right-hand side is exactly zero in every
    cell -- each face towards a solid cell carries no diffusive flux, on the x, y and z faces alike.  A compact second
    difference on any axis would see the jump from 1 to 0 at that axis' walls."""
    shape = (12, 10, 16)
    mask = np.zeros(shape, dtype=np.uint8)
    mask[2:-2, 2:-2, 2:-2] = 1
    mask[5:8, 4:6, 6:11] = 0                                                    # an obstacle with faces on all axes
    o = mk(shape, (0.3, 0.2, 0.25), nu=0.01, alpha_c=0.7, dt=0.1, mask=mask)
    z = np.zeros(shape)
    F = o.rhs(z, z, z, mask.astype(float))
    assert np.all(F[3] == 0.0)
    # and each axis on its own: a slab of solid normal to that axis only
    for ax in range(3):
        m = np.ones(shape, dtype=np.uint8)
        sl = [slice(None)] * 3
        sl[ax] = slice(0, 2)
        m[tuple(sl)] = 0
        oa = mk(shape, (0.3, 0.2, 0.25), alpha_c=0.7, mask=m)
        assert np.all(oa.rhs(z, z, z, m.astype(float))[3] == 0.0), ax
        # whereas a c that varies along the wall-normal axis inside the fluid does diffuse (the term is not switched off)
        ramp = np.arange(shape[ax], dtype=float).reshape([-1 if a == ax else 1 for a in range(3)]) ** 2 * np.ones(shape) * m
        assert np.abs(oa.rhs(z, z, z, ramp)[3]).max() > 0.1, ax


@pytest.mark.parametrize("wall_axis", ["x", "z"])
def test_P20_poiseuille_fixed_point_with_the_walls_turned(wall_axis):
    """P9 with the channel turned: walls normal to x (flow along y) and normal to z (flow along x).  The
    printed parabola (tests/golden/poiseuille.txt) stays an exact fixed point and c = 1 stays 1 in the fluid, which pins
    the wall treatment of eqs. 2-4 on the two axes P9 does not reach."""
    rows = [l.split() for l in open(os.path.join(GOLD, "poiseuille.txt")) if not l.startswith("#")]
    U = np.array([float(r[1]) for r in rows])
    b, nu, n, h, wall = 1.0e-3, 0.05, 32, 0.25, 2
    if wall_axis == "x":
        shape, d, body, flow = (4, 8, n), (h, 0.3, 0.4), (0.0, b, 0.0), "v"
        prof = U[None, None, :]
        solid = (slice(None), slice(None))
        wsl = lambda s: (slice(None), slice(None), s)
    else:
        shape, d, body, flow = (n, 4, 8), (0.3, 0.4, h), (b, 0.0, 0.0), "u"
        prof = U[:, None, None]
        wsl = lambda s: (s, slice(None), slice(None))
    mask = np.ones(shape, dtype=np.uint8)
    mask[wsl(slice(0, wall))] = 0
    mask[wsl(slice(n - wall, n))] = 0
    f0 = np.broadcast_to(prof, shape).copy()
    zero = np.zeros(shape)
    o = mk(shape, d, nu=nu, alpha_c=nu, dt=0.2, mask=mask, body=body, n_piter=4)
    init = dict(u=zero, v=zero, w=zero)
    init[flow] = f0
    o.set_fields(init["u"], init["v"], init["w"], mask.astype(float))
    o.step(5)
    f = o.fields()
    assert np.abs(f[flow] - f0).max() < 1e-13 * U.max()
    for k in "uvw":
        if k != flow:
            assert np.abs(f[k]).max() < 1e-15
    assert np.abs(f["p"]).max() < 1e-15
    assert np.abs(f["c"] - mask).max() < 1e-14


def test_P21_heavy_particle_position_is_the_sum_of_its_new_velocities():
    """eq. 10 by implicit Euler, reading R27: x_p' = x_p + dt u_p' with the NEW particle velocity.
    A heavy droplet (dt = tau_p / 100) released at rest in a uniform, slow stream (Re_p ~ 6e-6, so C_d = 1 to 6e-5)
    has u_n = U (1 - r^n), r = 1 / (1 + dt/tau_p), hence x_n - x_0 = dt U (n - r (1 - r^n) / (1 - r)).  After 50 steps
    the particle has 39 % of the fluid speed; advancing x with the fluid velocity instead would have moved it 3.7 times
    as far, with the old particle velocity 4 % less far."""
    nu, rho_f, rho_p, dp, U = 1.6e-5, 1.2, 1000.0, 1.0e-4, 1.0e-6
    tau_p = rho_p * dp * dp / (18 * rho_f * nu)
    dt, n = tau_p / 100, 50
    shape = (8, 8, 8)
    o = mk(shape, (0.5, 0.5, 0.5), nu=nu, dt=dt)
    z = np.zeros(shape)
    o.set_fields(np.full(shape, U), z, z, z)
    st = _particles([[0.0, 1.3, 2.1, 0.0, 0.0, 0.0, dp, rho_p]])
    for _ in range(n):
        o.particles_step(st, rho_f, (0.0, 0.0, 0.0))
    r = 1.0 / (1.0 + dt / tau_p)
    un = U * (1 - r ** n)
    xn = dt * U * (n - r * (1 - r ** n) / (1 - r))
    assert 0.38 < un / U < 0.40
    assert abs(st[3, 0] - un) <= 1e-4 * un
    assert abs(st[0, 0] - xn) <= 1e-4 * xn, (st[0, 0], xn, dt * U * n)
    assert st[1, 0] == 1.3 and st[2, 0] == 2.1 and st[4, 0] == 0.0 and st[5, 0] == 0.0
