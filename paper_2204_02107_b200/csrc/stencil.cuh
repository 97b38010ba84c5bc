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
    int kc;                  // k_rk_march: planes per block
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

// ---------------------------------------------------------------------------------------------
// k_rk_march: the same stage (a1-a3) for grids with nx >= 64, marching along z.
//
// A block owns a 64 x 8 (x by y) column of cells and walks kc planes of it.  Each thread owns two
// x-adjacent cells (one double2 per field).  The stage field's plane k+2 is in flight (cp.async,
// LDGSTS) into one of three shared-memory plane tiles (4 fields x 10 rows x 64+2 cells, halo included,
// periodic wrap applied to the source address) while plane k is being computed: x/y neighbours come
// from the tile of plane k, the z+1 neighbour from the tile of plane k+1, the z-1 neighbour and the
// centre are carried in registers.  So every stage-field value is fetched from L2/HBM once per block
// (plus the one-cell halo), the bytes in flight live in shared memory rather than in registers, and
// the other operands (Qn, Q2, Q3) and the result are streamed as 16-byte accesses.
// One __syncthreads per plane.  Arithmetic and select semantics are those of k_rk above.
constexpr int RKM_TX = 64, RKM_TY = 8, RKM_SW = 68, RKM_ROWS = RKM_TY + 2, RKM_NBUF = 3;
constexpr int RKM_SMEM = RKM_NBUF * 4 * RKM_ROWS * RKM_SW * (int)sizeof(double);

__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async8(void *dst_smem, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

// RHS of one cell for field m given its seven-point neighbourhood and the advecting velocities.
template <bool MASKED_C>
__device__ __forceinline__ double rk_rhs_cell(const RKArgs &a, int m, unsigned f, double c0, double xp, double xm, double yp, double ym,
                                              double zp, double zm, double u, double v, double w, double uxp, double uxm, double vyp,
                                              double vym, double wzp, double wzm)
{
    double conv = ((uxp * xp - uxm * xm) + u * (xp - xm)) * a.r2x;
    conv += ((vyp * yp - vym * ym) + v * (yp - ym)) * a.r2y;
    conv += ((wzp * zp - wzm * zm) + w * (zp - zm)) * a.r2z;
    double diff;
    if (!MASKED_C) {
        diff = (m < 3 ? a.nu : a.ac) * ((xp - 2.0 * c0 + xm) * a.rxx + (yp - 2.0 * c0 + ym) * a.ryy + (zp - 2.0 * c0 + zm) * a.rzz);
    } else {
        // eq. 4: no flux through solid faces (beta+- = beta * beta[+-1])
        const double dxp = (f & 2) ? (xp - c0) : 0.0, dxm = (f & 4) ? (c0 - xm) : 0.0;
        const double dyp = (f & 8) ? (yp - c0) : 0.0, dym = (f & 16) ? (c0 - ym) : 0.0;
        const double dzp = (f & 32) ? (zp - c0) : 0.0, dzm = (f & 64) ? (c0 - zm) : 0.0;
        diff = a.ac * ((dxp - dxm) * a.rxx + (dyp - dym) * a.ryy + (dzp - dzm) * a.rzz);
    }
    double val = -0.5 * conv + diff;
    if (m < 3) val += a.body[m];
    return val;
}

template <int STAGE, bool ELIM, bool MASKED, bool SOURCES> __global__ void __launch_bounds__(256, 2) k_rk_march(const RKArgs a)
{
    constexpr int TX = RKM_TX, SW = RKM_SW, ROWS = RKM_ROWS, PLANE = 4 * RKM_ROWS * RKM_SW;
    extern __shared__ double2 rkm_smem2[];
    double *sm = reinterpret_cast<double *>(rkm_smem2);
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * 32 + tx;
    const int nx = a.nx, ny = a.ny, nz = a.nz, kc = a.kc;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * RKM_TY, k0 = blockIdx.z * kc;
    const int i = x0 + 2 * tx, j = y0 + ty;
    const size_t plane = (size_t)nx * ny;
    const size_t orow = (size_t)nx * j + i;

    // this thread's share of one plane tile: per field 10 rows x 32 double2 (interior + y halo) and 20 x-halo values
    const int r_a = tid >> 5, q_a = tid & 31;                 // copy A: rows 0..7
    const size_t src_a = (size_t)nx * ((y0 - 1 + r_a) & (ny - 1)) + x0 + 2 * q_a;
    const int dst_a = r_a * SW + 2 + 2 * q_a;
    const bool has_b = tid < 64;                              // copy B: rows 8..9
    const size_t src_b = (size_t)nx * ((y0 + 7 + r_a) & (ny - 1)) + x0 + 2 * q_a;
    const int dst_b = (8 + r_a) * SW + 2 + 2 * q_a;
    const bool has_h = tid >= 64 && tid < 64 + 4 * ROWS * 2;  // x halo: 80 values
    const int hh = tid - 64, h_m = hh / (ROWS * 2), h_r = (hh % (ROWS * 2)) >> 1, h_s = hh & 1;
    const size_t src_h = (size_t)nx * ((y0 - 1 + h_r) & (ny - 1)) + (h_s ? ((x0 + TX) & (nx - 1)) : ((x0 - 1) & (nx - 1)));
    const int dst_h = (h_m * ROWS + h_r) * SW + (h_s ? 2 + TX : 1);
    auto issue_plane = [&](int kk, int buf) {
        const size_t pk = plane * (size_t)(kk & (nz - 1));
        double *sb = sm + buf * PLANE;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            cp_async16(sb + m * ROWS * SW + dst_a, a.qs[m] + pk + src_a);
            if (has_b) cp_async16(sb + m * ROWS * SW + dst_b, a.qs[m] + pk + src_b);
        }
        if (has_h) cp_async8(sb + dst_h, a.qs[h_m] + pk + src_h);
        cp_async_commit();
    };

    issue_plane(k0, 0);
    issue_plane(k0 + 1, 1);
    double2 zm[4], cur[4];
    {
        const size_t pkm = plane * (size_t)((k0 - 1) & (nz - 1));
#pragma unroll
        for (int m = 0; m < 4; ++m) zm[m] = __ldg(reinterpret_cast<const double2 *>(a.qs[m] + pkm + orow));
    }
    const int own = (ty + 1) * SW + 2 + 2 * tx; // this thread's pair inside a field's tile

    for (int t = 0; t < kc; ++t) {
        const int k = k0 + t;
        const size_t o = plane * (size_t)k + orow;
        // operands that do not go through shared memory: issue their loads before waiting
        double2 qn[4], q2[4], q3[4];
        unsigned fA = 0x7f, fB = 0x7f;
        if (MASKED) {
            const uchar2 fv = *reinterpret_cast<const uchar2 *>(a.face + o);
            fA = fv.x;
            fB = fv.y;
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            if (STAGE >= 2) qn[m] = __ldg(reinterpret_cast<const double2 *>(a.qn[m] + o));
            if (STAGE >= 2 && !ELIM) q2[m] = *reinterpret_cast<const double2 *>(a.qc[m] + o); // Qc, updated in place
            if (STAGE == 4 && ELIM) {
                q2[m] = *reinterpret_cast<const double2 *>(a.qc[m] + o); // Q2, overwritten below by Q*
                q3[m] = __ldg(reinterpret_cast<const double2 *>(a.q3[m] + o));
            }
        }
        cp_async_wait_all();
        __syncthreads(); // plane k+1 visible to all; every thread is done with the tile of plane k-1
        if (t + 2 <= kc) issue_plane(k + 2, (t + 2) % RKM_NBUF);
        const double *sC = sm + (t % RKM_NBUF) * PLANE, *sN = sm + ((t + 1) % RKM_NBUF) * PLANE;
        if (t == 0) {
#pragma unroll
            for (int m = 0; m < 4; ++m) cur[m] = *reinterpret_cast<const double2 *>(sC + m * ROWS * SW + own);
        }
        double2 zp[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) zp[m] = *reinterpret_cast<const double2 *>(sN + m * ROWS * SW + own);
        if (STAGE == 1) {
#pragma unroll
            for (int m = 0; m < 4; ++m) qn[m] = cur[m];
        }
        const double2 vym = *reinterpret_cast<const double2 *>(sC + 1 * ROWS * SW + own - SW);
        const double2 vyp = *reinterpret_cast<const double2 *>(sC + 1 * ROWS * SW + own + SW);
        const double uxmA = sC[own - 1], uxpB = sC[own + 2];
        double2 F[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const double *sf = sC + m * ROWS * SW + own;
            const double2 ym = *reinterpret_cast<const double2 *>(sf - SW), yp = *reinterpret_cast<const double2 *>(sf + SW);
            const double xmA = sf[-1], xpB = sf[2];
            if (m < 3 || !MASKED) {
                F[m].x = rk_rhs_cell<false>(a, m, fA, cur[m].x, cur[m].y, xmA, yp.x, ym.x, zp[m].x, zm[m].x, cur[0].x, cur[1].x, cur[2].x,
                                            cur[0].y, uxmA, vyp.x, vym.x, zp[2].x, zm[2].x);
                F[m].y = rk_rhs_cell<false>(a, m, fB, cur[m].y, xpB, cur[m].x, yp.y, ym.y, zp[m].y, zm[m].y, cur[0].y, cur[1].y, cur[2].y,
                                            uxpB, cur[0].x, vyp.y, vym.y, zp[2].y, zm[2].y);
            } else {
                F[m].x = rk_rhs_cell<true>(a, m, fA, cur[m].x, cur[m].y, xmA, yp.x, ym.x, zp[m].x, zm[m].x, cur[0].x, cur[1].x, cur[2].x,
                                           cur[0].y, uxmA, vyp.x, vym.x, zp[2].x, zm[2].x);
                F[m].y = rk_rhs_cell<true>(a, m, fB, cur[m].y, xpB, cur[m].x, yp.y, ym.y, zp[m].y, zm[m].y, cur[0].y, cur[1].y, cur[2].y,
                                           uxpB, cur[0].x, vyp.y, vym.y, zp[2].y, zm[2].y);
            }
        }
        if (SOURCES) {
            for (int s = 0; s < a.nsrc; ++s) {
                const double *tb = a.stab + a.src[s].off;
                const double sz = __ldg(&tb[nx + ny + k]), sy = __ldg(&tb[nx + j]);
                if (sy == 0.0 || sz == 0.0) continue;
                const double2 sx = __ldg(reinterpret_cast<const double2 *>(tb + i));
                const double SA = sx.x * sy * sz, SB = sx.y * sy * sz;
                const uint32_t comps = a.src[s].comps;
#pragma unroll
                for (int m = 0; m < 4; ++m)
                    if (comps & (1u << m)) {
                        if (SA != 0.0) F[m].x += SA * (a.src[s].set[m] - cur[m].x) * a.src[s].rtau;
                        if (SB != 0.0) F[m].y += SB * (a.src[s].set[m] - cur[m].y) * a.src[s].rtau;
                    }
            }
        }
        const bool flA = !MASKED || (fA & 1), flB = !MASKED || (fB & 1);
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            // solid cell: every field it holds is +0.0 and stays +0.0 (select)
            if (ELIM) {
                double2 r;
                if (STAGE < 4) {
                    r.x = flA ? qn[m].x + a.ca * F[m].x : 0.0;
                    r.y = flB ? qn[m].y + a.ca * F[m].y : 0.0;
                    *reinterpret_cast<double2 *>(a.qo[m] + o) = r;
                } else {
                    r.x = flA ? (q2[m].x - qn[m].x + 2.0 * q3[m].x + cur[m].x) * (1.0 / 3.0) + a.cb * F[m].x : 0.0;
                    r.y = flB ? (q2[m].y - qn[m].y + 2.0 * q3[m].y + cur[m].y) * (1.0 / 3.0) + a.cb * F[m].y : 0.0;
                    *reinterpret_cast<double2 *>(a.qco[m] + o) = r;
                }
            } else {
                double2 c, r;
                const double2 qcv = STAGE >= 2 ? q2[m] : qn[m];
                c.x = flA ? qcv.x + a.cb * F[m].x : 0.0;
                c.y = flB ? qcv.y + a.cb * F[m].y : 0.0;
                *reinterpret_cast<double2 *>(a.qco[m] + o) = c;
                if (STAGE < 4) {
                    r.x = flA ? qn[m].x + a.ca * F[m].x : 0.0;
                    r.y = flB ? qn[m].y + a.ca * F[m].y : 0.0;
                    *reinterpret_cast<double2 *>(a.qo[m] + o) = r;
                }
            }
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            zm[m] = cur[m];
            cur[m] = zp[m];
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

// a5, right-hand side of eq. 9: r = d + sum_a delta_a[(1-beta) delta_a p], evaluated only
// where the bracket can be non-zero.  (1-beta) is 0 in the fluid, so those are the cells with at least
// one solid face neighbour; `list` holds their linear indices in ascending order (built at create).
// The first iteration of a step saves d at those cells (`save`), later ones restore it from there, and
// r overwrites d in place: everywhere else r == d already, so the forward x pass reads one plain array.
// face: bit0 beta(cell), bit1/2 beta(x+1/x-1), bit3/4 beta(y+1/y-1), bit5/6 beta(z+1/z-1).
__global__ void __launch_bounds__(256) k_eq9_sparse(double *__restrict__ d, const double *__restrict__ p, const uint8_t *__restrict__ face,
                                                    const uint32_t *__restrict__ list, double *__restrict__ save, int nlist, int first,
                                                    int nx, int ny, int nz, int lgx, int lgy, double r2x, double r2y, double r2z)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= nlist) return;
    const uint32_t o = list[n];
    const int i = o & (nx - 1), j = (o >> lgx) & (ny - 1), k = o >> (lgx + lgy);
    const unsigned f = face[o];
    double dv;
    if (first) {
        dv = d[o];
        save[n] = dv;
    } else {
        dv = save[n];
    }
    const size_t row = (size_t)nx * ((size_t)j + (size_t)ny * k);
    const double pc = __ldg(&p[o]);
    double gxp = 0.0, gxm = 0.0, gyp = 0.0, gym = 0.0, gzp = 0.0, gzm = 0.0;
    if (!(f & 2)) gxp = (__ldg(&p[row + ((i + 2) & (nx - 1))]) - pc) * r2x;
    if (!(f & 4)) gxm = (pc - __ldg(&p[row + ((i - 2) & (nx - 1))])) * r2x;
    if (!(f & 8)) gyp = (__ldg(&p[(size_t)nx * ((size_t)((j + 2) & (ny - 1)) + (size_t)ny * k) + i]) - pc) * r2y;
    if (!(f & 16)) gym = (pc - __ldg(&p[(size_t)nx * ((size_t)((j - 2) & (ny - 1)) + (size_t)ny * k) + i])) * r2y;
    if (!(f & 32)) gzp = (__ldg(&p[(size_t)nx * ((size_t)j + (size_t)ny * ((k + 2) & (nz - 1))) + i]) - pc) * r2z;
    if (!(f & 64)) gzm = (pc - __ldg(&p[(size_t)nx * ((size_t)j + (size_t)ny * ((k - 2) & (nz - 1))) + i])) * r2z;
    d[o] = dv + ((gxp - gxm) * r2x + (gyp - gym) * r2y + (gzp - gzm) * r2z);
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
