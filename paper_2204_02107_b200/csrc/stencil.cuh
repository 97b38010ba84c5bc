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
    const double *qc[4]; // running combination, read (stages 2-4)
    double *qo[4];       // next stage field, written (stages 1-3)
    double *qco[4];      // running combination, written
    const uint8_t *face; // null: no solid cells
    int nx, ny, nz, zchunk;
    double r2x, r2y, r2z;    // 1/(2 D_a)
    double rxx, ryy, rzz;    // 1/D_a^2
    double nu, ac;           // viscosity, scalar diffusivity
    double body[3];
    double ca, cb;           // a_s dt, b_s dt
    int nsrc;
    const double *stab;
    SourceDev src[DNS_MAX_SRC];
};

// One RK stage (a1-a3 of DESIGN.md): F = beta ? RHS(Qs) : 0; Qc(+)= b_s dt F; Qs' = Qn + a_s dt F.
// Block = 32 x by 8 y cells (narrower in x on tiny grids); each thread marches zchunk planes in z keeping the k-1, k, k+1
// values of the four fields in registers; x and y neighbours come through L1.
//   STAGE 1: Qs == Qn, Qc is written fresh (= Qn + b dt F).   STAGE 4: no next stage field.
template <int STAGE, bool MASKED, bool SOURCES> __global__ void __launch_bounds__(256) k_rk_stage(const RKArgs a)
{
    const int nx = a.nx, ny = a.ny, nz = a.nz;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k0 = blockIdx.z * a.zchunk;
    const int ip = (i + 1) & (nx - 1), im = (i - 1) & (nx - 1);
    const int jp = (j + 1) & (ny - 1), jm = (j - 1) & (ny - 1);
    const size_t plane = (size_t)nx * ny;
    const size_t rowc = (size_t)nx * j, rowp = (size_t)nx * jp, rowm = (size_t)nx * jm;

    double fm[4], f0[4], fp[4];
    {
        const size_t om = plane * ((k0 - 1) & (nz - 1)) + rowc + i;
        const size_t oc = plane * k0 + rowc + i;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            fm[m] = __ldg(&a.qs[m][om]);
            f0[m] = __ldg(&a.qs[m][oc]);
        }
    }
    for (int kk = 0; kk < a.zchunk; ++kk) {
        const int k = k0 + kk;
        const size_t pk = plane * k;
        const size_t pkp = plane * ((k + 1) & (nz - 1));
        const size_t o = pk + rowc + i;
        double xp[4], xm[4], yp[4], ym[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            fp[m] = __ldg(&a.qs[m][pkp + rowc + i]);
            xp[m] = __ldg(&a.qs[m][pk + rowc + ip]);
            xm[m] = __ldg(&a.qs[m][pk + rowc + im]);
            yp[m] = __ldg(&a.qs[m][pk + rowp + i]);
            ym[m] = __ldg(&a.qs[m][pk + rowm + i]);
        }
        unsigned f = 0x7f;
        if (MASKED) f = a.face[o];
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
        } else {
#pragma unroll
            for (int m = 0; m < 4; ++m) F[m] = 0.0;
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            double qn = f0[m];
            if (STAGE == 2 || STAGE == 3) qn = __ldg(&a.qn[m][o]);
            const double qc = (STAGE == 1) ? qn : a.qc[m][o]; // plain load: Qc is updated in place
            a.qco[m][o] = qc + a.cb * F[m];
            if (STAGE < 4) a.qo[m][o] = qn + a.ca * F[m];
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            fm[m] = f0[m];
            f0[m] = fp[m];
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
