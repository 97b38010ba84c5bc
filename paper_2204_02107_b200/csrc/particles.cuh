// particles.cuh -- NEXT-4: Lagrangian particles, eqs. 10-13, one implicit Euler step of size dt
// in the velocity field of the finished fluid step ("SolveDrops.m" after the fluid solve):
//     tau_p = rho_p d^2 / (18 rho_f nu),  Re_p = |u_f - u_p| d / nu,  C_d = 1 + Re_p^(2/3)/6,
//     u_p' = (u_p + dt (k u_f + g)) / (1 + dt k),  k = C_d / tau_p  (C_d from the old velocities, R27),
//     x_p' = x_p + dt u_p', wrapped into [0, L);  u_f = trilinear interpolation of the collocated velocity with
//     cell centres at x_i = i Delta, periodic (R26).
// One thread per particle: 24 gathered doubles, ~100 flops -- bound by the gather latency, not by bandwidth.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dnspart {

struct PartArgs {
    const double *u, *v, *w;
    double *state; // 8 arrays of n doubles: x y z u v w d rho_p
    long long n;
    int nx, ny, nz;
    double dx, dy, dz, dt, nu, rho_f, g[3];
};

__global__ void __launch_bounds__(128) k_particles(const PartArgs a)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= a.n) return;
    const long long n = a.n;
    double *s = a.state;
    const double x = s[q], y = s[n + q], z = s[2 * n + q];
    const double pu = s[3 * n + q], pv = s[4 * n + q], pw = s[5 * n + q], d = s[6 * n + q], rho = s[7 * n + q];
    const int nx = a.nx, ny = a.ny, nz = a.nz;
    const double gx = x / a.dx, gy = y / a.dy, gz = z / a.dz;
    const double fx = floor(gx), fy = floor(gy), fz = floor(gz);
    const double ax = gx - fx, ay = gy - fy, az = gz - fz;
    const int i0 = (int)fx & (nx - 1), j0 = (int)fy & (ny - 1), k0 = (int)fz & (nz - 1); // extents are powers of two
    const int i1 = (i0 + 1) & (nx - 1), j1 = (j0 + 1) & (ny - 1), k1 = (k0 + 1) & (nz - 1);
    const size_t r00 = (size_t)nx * ((size_t)j0 + (size_t)ny * k0), r10 = (size_t)nx * ((size_t)j1 + (size_t)ny * k0);
    const size_t r01 = (size_t)nx * ((size_t)j0 + (size_t)ny * k1), r11 = (size_t)nx * ((size_t)j1 + (size_t)ny * k1);
    auto interp = [&](const double *__restrict__ f) {
        const double c00 = __ldg(f + r00 + i0) * (1.0 - ax) + __ldg(f + r00 + i1) * ax;
        const double c10 = __ldg(f + r10 + i0) * (1.0 - ax) + __ldg(f + r10 + i1) * ax;
        const double c01 = __ldg(f + r01 + i0) * (1.0 - ax) + __ldg(f + r01 + i1) * ax;
        const double c11 = __ldg(f + r11 + i0) * (1.0 - ax) + __ldg(f + r11 + i1) * ax;
        const double c0 = c00 * (1.0 - ay) + c10 * ay, c1 = c01 * (1.0 - ay) + c11 * ay;
        return c0 * (1.0 - az) + c1 * az;
    };
    const double uf = interp(a.u), vf = interp(a.v), wf = interp(a.w);
    const double tau = rho * d * d / (18.0 * a.rho_f * a.nu);
    const double rel = sqrt((uf - pu) * (uf - pu) + (vf - pv) * (vf - pv) + (wf - pw) * (wf - pw));
    const double rep = rel * d / a.nu;
    const double cd = 1.0 + cbrt(rep * rep) / 6.0;
    const double k = cd / tau, dt = a.dt;
    const double un = (pu + dt * (k * uf + a.g[0])) / (1.0 + dt * k);
    const double vn = (pv + dt * (k * vf + a.g[1])) / (1.0 + dt * k);
    const double wn = (pw + dt * (k * wf + a.g[2])) / (1.0 + dt * k);
    const double len[3] = {nx * a.dx, ny * a.dy, nz * a.dz};
    double xn[3] = {x + dt * un, y + dt * vn, z + dt * wn};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        xn[c] = xn[c] - floor(xn[c] / len[c]) * len[c];
        if (!(xn[c] < len[c])) xn[c] = 0.0; // rounding at the upper edge
    }
    s[q] = xn[0];
    s[n + q] = xn[1];
    s[2 * n + q] = xn[2];
    s[3 * n + q] = un;
    s[4 * n + q] = vn;
    s[5 * n + q] = wn;
}

} // namespace dnspart
