// stencil.cuh -- finite-difference kernels of the DNSLABIB step (eqs. 2-4, 7-8):
// fused RHS + Runge-Kutta stage update, divergence, pressure-gradient projection, mask set-up.
// fp64, x fastest, all axes periodic with power-of-two extents (wrap = bit mask).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dnsst {

#define DNS_MAX_SRC 16

// face byte: bit0 beta(cell), bit1 beta(x+1), bit2 beta(x-1), bit3 beta(y+1), bit4 beta(y-1),
// bit5 beta(z+1), bit6 beta(z-1)
__global__ void k_face_mask(const uint8_t *__restrict__ beta, uint8_t *__restrict__ face, int nx, int ny, int nz)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= nx) return;
    auto B = [&](int ii, int jj, int kk) -> unsigned {
        return beta[(size_t)(ii & (nx - 1)) + (size_t)nx * ((size_t)(jj & (ny - 1)) + (size_t)ny * (kk & (nz - 1)))] != 0;
    };
    unsigned f = B(i, j, k) | (B(i + 1, j, k) << 1) | (B(i - 1, j, k) << 2) | (B(i, j + 1, k) << 3) | (B(i, j - 1, k) << 4) |
                 (B(i, j, k + 1) << 5) | (B(i, j, k - 1) << 6);
    face[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * k)] = (uint8_t)f;
}

// q = beta ? q : +0.0 on up to four fields (set_fields, select not multiply)
__global__ void k_mask_select(double *q0, double *q1, double *q2, double *q3, const uint8_t *__restrict__ face, size_t n)
{
    const size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= n) return;
    if (!(face[o] & 1)) {
        q0[o] = 0.0;
        q1[o] = 0.0;
        q2[o] = 0.0;
        q3[o] = 0.0;
    }
}

struct SourceDev {
    double set[4]; // u_set, v_set, w_set, c_set
    double rtau;   // 1/tau_f
    uint32_t comps;
    int off; // offset of this source's sx|sy|sz tables (nx+ny+nz doubles) in stab
};

struct RKArgs {
    const double *qs[4]; // stage field (stencil input)
    const double *qn[4]; // Q^n
    const double *qc[4]; // running combination Qc, read (stages 2-4); with ELIM at stage 4: Q2
    const double *q3[4]; // ELIM, stage 4 only: Q3
    double *qo[4];       // next stage field, written (stages 1-3)
    double *qco[4];      // Qc written (accumulate form); with ELIM at stage 4: Q* (aliases Q2)
    const uint8_t *face; // null: no solid cells
    int nx, ny, nz;
    double r2x, r2y, r2z;    // 1/(2 D_a)
    double rxx, ryy, rzz;    // 1/D_a^2
    double nu, ac;           // viscosity, scalar diffusivity
    double body[3];
    double ca, cb;           // a_s dt, b_s dt
    int nsrc;
    const double *stab;
    SourceDev src[DNS_MAX_SRC];
};

// One RK stage (a1-a3 of DESIGN.md): F = beta ? RHS(Qs) : +0.0 fused with the stage update.
// One thread per cell; a block is a small 3-D brick so that x, y and z neighbours are shared
// through L1 (DRAM traffic stays at the compulsory bytes, see profiles/).
//
// ELIM = false, the accumulate form of the oracle:   Qc (+)= b_s dt F ;  Qs' = Qn + a_s dt F.
// ELIM = true, Qc eliminated algebraically (12 fewer field passes per step):
//     stages 1-3:  Qs' = Qn + a_s dt F
//     stage 4:     Q*  = (-Qn + Q2 + 2 Q3 + Q4)/3 + (dt/6) F4
//   which equals Qn + dt/6 (F1 + 2 F2 + 2 F3 + F4) because Q2 = Qn + dt/2 F1, Q3 = Qn + dt/2 F2,
//   Q4 = Qn + dt F3 (classical RK4).  Q* overwrites Q2 in place.
template <int STAGE, bool ELIM, bool MASKED, bool SOURCES> __global__ void __launch_bounds__(256, 3) k_rk(const RKArgs a)
{
    const int nx = a.nx, ny = a.ny, nz = a.nz;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z * blockDim.z + threadIdx.z;
    const int ip = (i + 1) & (nx - 1), im = (i - 1) & (nx - 1);
    const size_t plane = (size_t)nx * ny;
    const size_t pk = plane * k, rowc = (size_t)nx * j;
    const size_t o = pk + rowc + i;
    const size_t oyp = pk + (size_t)nx * ((j + 1) & (ny - 1)) + i, oym = pk + (size_t)nx * ((j - 1) & (ny - 1)) + i;
    const size_t ozp = plane * ((k + 1) & (nz - 1)) + rowc + i, ozm = plane * ((k - 1) & (nz - 1)) + rowc + i;
    unsigned f = 0x7f;
    if (MASKED) f = a.face[o];
    double f0[4], xp[4], xm[4], yp[4], ym[4], fp[4], fm[4], qn[4], qc[4], q3[4];
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        f0[m] = __ldg(&a.qs[m][o]);
        xp[m] = __ldg(&a.qs[m][pk + rowc + ip]);
        xm[m] = __ldg(&a.qs[m][pk + rowc + im]);
        yp[m] = __ldg(&a.qs[m][oyp]);
        ym[m] = __ldg(&a.qs[m][oym]);
        fp[m] = __ldg(&a.qs[m][ozp]);
        fm[m] = __ldg(&a.qs[m][ozm]);
        qn[m] = f0[m];
        if (STAGE >= 2 && (STAGE <= 3 || ELIM)) qn[m] = __ldg(&a.qn[m][o]);
        qc[m] = qn[m];
        if (STAGE >= 2 && !ELIM) qc[m] = a.qc[m][o]; // plain loads: updated in place
        if (STAGE == 4 && ELIM) {
            qc[m] = a.qc[m][o]; // Q2, overwritten below by Q*
            q3[m] = __ldg(&a.q3[m][o]);
        }
    }
    double F[4];
    if (!MASKED || (f & 1)) {
        const double u = f0[0], v = f0[1], w = f0[2];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const double c0 = f0[m];
            double conv = 0.0;
            conv += (xp[0] * xp[m] - xm[0] * xm[m]) * a.r2x + u * (xp[m] - xm[m]) * a.r2x;
            conv += (yp[1] * yp[m] - ym[1] * ym[m]) * a.r2y + v * (yp[m] - ym[m]) * a.r2y;
            conv += (fp[2] * fp[m] - fm[2] * fm[m]) * a.r2z + w * (fp[m] - fm[m]) * a.r2z;
            double diff;
            if (m < 3 || !MASKED) {
                diff = (m < 3 ? a.nu : a.ac) * ((xp[m] - 2.0 * c0 + xm[m]) * a.rxx + (yp[m] - 2.0 * c0 + ym[m]) * a.ryy +
                                                (fp[m] - 2.0 * c0 + fm[m]) * a.rzz);
            } else {
                // eq. 4: no flux through solid faces (beta+- = beta * beta[+-1])
                const double dxp = (f & 2) ? (xp[m] - c0) : 0.0, dxm = (f & 4) ? (c0 - xm[m]) : 0.0;
                const double dyp = (f & 8) ? (yp[m] - c0) : 0.0, dym = (f & 16) ? (c0 - ym[m]) : 0.0;
                const double dzp = (f & 32) ? (fp[m] - c0) : 0.0, dzm = (f & 64) ? (c0 - fm[m]) : 0.0;
                diff = a.ac * ((dxp - dxm) * a.rxx + (dyp - dym) * a.ryy + (dzp - dzm) * a.rzz);
            }
            double val = -0.5 * conv + diff;
            if (m < 3) val += a.body[m];
            F[m] = val;
        }
        if (SOURCES) {
            for (int s = 0; s < a.nsrc; ++s) {
                const double *t = a.stab + a.src[s].off;
                const double sy = __ldg(&t[nx + j]), sz = __ldg(&t[nx + ny + k]);
                if (sy == 0.0 || sz == 0.0) continue;
                const double Sv = __ldg(&t[i]) * sy * sz;
                if (Sv == 0.0) continue;
                const uint32_t comps = a.src[s].comps;
#pragma unroll
                for (int m = 0; m < 4; ++m)
                    if (comps & (1u << m)) F[m] += Sv * (a.src[s].set[m] - f0[m]) * a.src[s].rtau;
            }
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            if (ELIM) {
                if (STAGE < 4) a.qo[m][o] = qn[m] + a.ca * F[m];
                else a.qco[m][o] = (qc[m] - qn[m] + 2.0 * q3[m] + f0[m]) * (1.0 / 3.0) + a.cb * F[m];
            } else {
                a.qco[m][o] = qc[m] + a.cb * F[m];
                if (STAGE < 4) a.qo[m][o] = qn[m] + a.ca * F[m];
            }
        }
    } else {
        // solid cell: every field it holds is +0.0 and stays +0.0 (select)
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            if (!ELIM || STAGE == 4) a.qco[m][o] = 0.0;
            if (STAGE < 4) a.qo[m][o] = 0.0;
        }
    }
}

// a4: d = sum_a delta_a u_a (eq. 7 right-hand side)
__global__ void __launch_bounds__(256) k_div(const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
                                             double *__restrict__ d, int nx, int ny, int nz, double r2x, double r2y, double r2z)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    const size_t plane = (size_t)nx * ny;
    const size_t o = plane * k + (size_t)nx * j + i;
    const size_t row = plane * k + (size_t)nx * j;
    d[o] = (__ldg(&u[row + ((i + 1) & (nx - 1))]) - __ldg(&u[row + ((i - 1) & (nx - 1))])) * r2x +
           (__ldg(&v[plane * k + (size_t)nx * ((j + 1) & (ny - 1)) + i]) - __ldg(&v[plane * k + (size_t)nx * ((j - 1) & (ny - 1)) + i])) * r2y +
           (__ldg(&w[plane * ((k + 1) & (nz - 1)) + (size_t)nx * j + i]) - __ldg(&w[plane * ((k - 1) & (nz - 1)) + (size_t)nx * j + i])) * r2z;
}

// a6: u_a = beta ? u*_a - delta_a p : +0.0, in place (eq. 8)
template <bool MASKED>
__global__ void __launch_bounds__(256) k_project(double *__restrict__ u, double *__restrict__ v, double *__restrict__ w, const double *__restrict__ p,
                                                 const uint8_t *__restrict__ face, int nx, int ny, int nz, double r2x, double r2y, double r2z)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    const size_t plane = (size_t)nx * ny;
    const size_t row = plane * k + (size_t)nx * j;
    const size_t o = row + i;
    if (MASKED) {
        if (!(face[o] & 1)) {
            u[o] = 0.0;
            v[o] = 0.0;
            w[o] = 0.0;
            return;
        }
    }
    const double gx = (__ldg(&p[row + ((i + 1) & (nx - 1))]) - __ldg(&p[row + ((i - 1) & (nx - 1))])) * r2x;
    const double gy = (__ldg(&p[plane * k + (size_t)nx * ((j + 1) & (ny - 1)) + i]) - __ldg(&p[plane * k + (size_t)nx * ((j - 1) & (ny - 1)) + i])) * r2y;
    const double gz = (__ldg(&p[plane * ((k + 1) & (nz - 1)) + (size_t)nx * j + i]) - __ldg(&p[plane * ((k - 1) & (nz - 1)) + (size_t)nx * j + i])) * r2z;
    u[o] = u[o] - gx;
    v[o] = v[o] - gy;
    w[o] = w[o] - gz;
}

} // namespace dnsst
