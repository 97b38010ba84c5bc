// stencil.cuh -- finite-difference kernels of the DNSLABIB step (eqs. 2-4, 7-8):
// fused RHS + Runge-Kutta stage update, divergence, pressure-gradient projection, mask set-up.
// fp64, x fastest, all axes periodic with power-of-two extents (wrap = bit mask).
#pragma once
#include <cuda.h> // CUtensorMap (type only: the encoder is fetched through cudaGetDriverEntryPoint, nothing links libcuda)
#include <cuda_runtime.h>
#include <stdint.h>

#include "tma.cuh"

namespace dnsst {

using namespace dnstma;

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

// coefficients of the factored right-hand side of k_rk_march (host-computed, read from the constant bank)
struct RhsCoef {
    double hx, hy, hz;    // -1/(4 Delta_a)
    double dvx, dvy, dvz; // nu / Delta_a^2
    double dcx, dcy, dcz; // alpha_c / Delta_a^2
    double dv0, dc0;      // -2 sum_a of the above
};

struct RKArgs {
    const double *qs[4]; // stage field (stencil input)
    const double *qn[4]; // Q^n
    const double *qc[4]; // running combination Qc, read (stages 2-4); with ELIM at stage 4: S = Q2 - Qn + 2 Q3
    double *qo[4];       // next stage field, written (stages 1-3)
    double *qco[4];      // Qc written (accumulate form); with ELIM: S at stage 2, Q* at stage 4 (in place of S)
    const uint8_t *face; // null: no solid cells
    int nx, ny, nz;
    double r2x, r2y, r2z;    // 1/(2 D_a)
    double rxx, ryy, rzz;    // 1/D_a^2
    double nu, ac;           // viscosity, scalar diffusivity
    double body[3];
    double ca, cb;           // a_s dt, b_s dt
    int nsrc;
    int kc;                  // k_rk_march: planes per block
    int rev;                 // k_rk_march: walk the y tiles and z chunks from the far end (start on what the kernel before left in L2)
    int use_tma;             // k_rk_march: tensor maps of the stage field are valid (interior blocks load their tiles by TMA)
    const double *stab;
    RhsCoef kf;
    SourceDev src[DNS_MAX_SRC];
};

// One RK stage (a1-a3 of DESIGN.md): F = beta ? RHS(Qs) : +0.0 fused with the stage update.
// One thread per cell; a block is a small 3-D brick so that x, y and z neighbours are shared
// through L1 (DRAM traffic stays at the compulsory bytes, see profiles/).
//
// ELIM = false, the accumulate form of the oracle:   Qc (+)= b_s dt F ;  Qs' = Qn + a_s dt F.
// ELIM = true, Qc eliminated algebraically (48 instead of 65 field passes per step):
//     stages 1-3:  Qs' = Qn + a_s dt F;   stage 2 also writes  S = Q2 - Qn + 2 Q3  (it holds all three)
//     stage 4:     Q*  = (S + Q4)/3 + (dt/6) F4,  in place of S
//   which equals Qn + dt/6 (F1 + 2 F2 + 2 F3 + F4) because Q2 = Qn + dt/2 F1, Q3 = Qn + dt/2 F2,
//   Q4 = Qn + dt F3 (classical RK4).  Stage 4 then reads two fields sets, not four.
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
    double f0[4], xp[4], xm[4], yp[4], ym[4], fp[4], fm[4], qn[4], qc[4];
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
        if (STAGE >= 2 && (STAGE <= 3 || !ELIM)) qn[m] = __ldg(&a.qn[m][o]);
        qc[m] = qn[m];
        if (STAGE >= 2 && !ELIM) qc[m] = a.qc[m][o]; // plain loads: updated in place
        if (STAGE == 4 && ELIM) qc[m] = a.qc[m][o]; // S, overwritten below by Q*
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
                if (STAGE < 4) {
                    const double r = qn[m] + a.ca * F[m];
                    a.qo[m][o] = r;
                    if (STAGE == 2) a.qco[m][o] = (f0[m] - qn[m]) + 2.0 * r;
                } else {
                    a.qco[m][o] = (qc[m] + f0[m]) * (1.0 / 3.0) + a.cb * F[m];
                }
            } else {
                a.qco[m][o] = qc[m] + a.cb * F[m];
                if (STAGE < 4) a.qo[m][o] = qn[m] + a.ca * F[m];
            }
        }
    } else {
        // solid cell: every field it holds is +0.0 and stays +0.0 (select)
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            if (!ELIM || STAGE == 4 || STAGE == 2) a.qco[m][o] = 0.0;
            if (STAGE < 4) a.qo[m][o] = 0.0;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// k_rk_march: the same stage (a1-a3) for grids with nx >= 64, marching along z.
//
// A block owns a 64 x 8 (x by y) column of cells and walks kc planes of it.  Each thread owns two
// x-adjacent cells (one double2 per field).  The stage field's planes k+2 and k+3 are in flight (cp.async,
// LDGSTS) into two of four shared-memory plane tiles (4 fields x 10 rows x 64+2 cells, halo included,
// periodic wrap applied to the source address) while plane k is being computed: x/y neighbours come
// from the tile of plane k, the z+1 neighbour from the tile of plane k+1, the z-1 neighbour and the
// centre are carried in registers.  So every stage-field value is fetched from L2/HBM once per block
// (plus the one-cell halo), the bytes in flight live in shared memory rather than in registers, and
// the other operands (Qn, Q2, Q3) and the result are streamed as 16-byte accesses.
// One __syncthreads per plane.  Arithmetic and select semantics are those of k_rk above.
constexpr int RKM_TX = 64, RKM_TY = 8, RKM_SW = 68, RKM_ROWS = RKM_TY + 2, RKM_NBUF = 4; // 5 tiles (three planes in flight) measured slower: 1.31 vs 1.10 ms per step
constexpr int RKM_FS = 688;                                      // doubles per field tile: 10 x 68 = 680, padded to a multiple of 128 bytes (TMA destination)
constexpr int RKM_TILE_BYTES = RKM_ROWS * RKM_SW * (int)sizeof(double); // what one TMA box writes
constexpr int RKM_SMEM = RKM_NBUF * 4 * RKM_FS * (int)sizeof(double);

// The four tensor maps of a stage field (one per component): rank 3 (x, y, z), fp64, box 68 x 10 x 1.
struct RKMaps {
    CUtensorMap m[4];
};

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
__device__ __forceinline__ void cp_async_wait_one() { asm volatile("cp.async.wait_group 1;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait_n() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <bool B> struct BoolTag { static constexpr bool value = B; };

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

template <int STAGE, bool ELIM, bool MASKED, bool SOURCES>
__global__ void __launch_bounds__(256, 2) k_rk_march(const RKArgs a, const __grid_constant__ RKMaps maps)
{
    constexpr int TX = RKM_TX, SW = RKM_SW, ROWS = RKM_ROWS, FS = RKM_FS, PLANE = 4 * RKM_FS;
    extern __shared__ __align__(128) double2 rkm_smem2[];
    __shared__ __align__(8) uint64_t mbar[RKM_NBUF];
    double *sm = reinterpret_cast<double *>(rkm_smem2);
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * 32 + tx;
    const int nx = a.nx, ny = a.ny, nz = a.nz, kc = a.kc;
    const int by = a.rev ? gridDim.y - 1 - blockIdx.y : blockIdx.y, bz = a.rev ? gridDim.z - 1 - blockIdx.z : blockIdx.z;
    const int x0 = blockIdx.x * TX, y0 = by * RKM_TY, k0 = bz * kc;
    const int i = x0 + 2 * tx, j = y0 + ty;
    // element offsets are 32-bit (a field has at most 2^31 cells): one IMAD.WIDE per access instead of 64-bit chains
    const unsigned plane = (unsigned)nx * (unsigned)ny;
    const unsigned orow = (unsigned)nx * j + i;

    // this thread's share of one plane tile: per field 10 rows x 32 double2 (interior + y halo) and 20 x-halo values
    const int r_a = tid >> 5, q_a = tid & 31;                 // copy A: rows 0..7
    const unsigned src_a = (unsigned)nx * ((y0 - 1 + r_a) & (ny - 1)) + x0 + 2 * q_a;
    const int dst_a = r_a * SW + 2 + 2 * q_a;
    const bool has_b = tid < 64;                              // copy B: rows 8..9
    const unsigned src_b = (unsigned)nx * ((y0 + 7 + r_a) & (ny - 1)) + x0 + 2 * q_a;
    const int dst_b = (8 + r_a) * SW + 2 + 2 * q_a;
    const bool has_h = tid >= 64 && tid < 64 + 4 * ROWS * 2;  // x halo: 80 values
    const int hh = tid - 64, h_m = hh / (ROWS * 2), h_r = (hh % (ROWS * 2)) >> 1, h_s = hh & 1;
    const unsigned src_h = (unsigned)nx * ((y0 - 1 + h_r) & (ny - 1)) + (h_s ? ((x0 + TX) & (nx - 1)) : ((x0 - 1) & (nx - 1)));
    const int dst_h = h_m * FS + h_r * SW + (h_s ? 2 + TX : 1);
    const double *qs_h = has_h ? a.qs[h_m & 3] : a.qs[0];
    // Interior blocks (the 68 x 10 box x0-2 .. x0+65, y0-1 .. y0+8 lies inside the grid: 70 % of the blocks of a
    // 512 x 256 plane) fetch a plane tile with four TMA box loads issued by one thread, counted in bytes on the tile's
    // mbarrier; blocks at the periodic seams, where a box would be zero-filled instead of wrapped, copy their tiles
    // with per-thread cp.async whose source addresses wrap.  Same tile layout for both.
    const bool tma = a.use_tma && blockIdx.x >= 1 && blockIdx.x + 2 <= gridDim.x && by >= 1 && by + 2 <= (int)gridDim.y;
    if (tma && tid == 0) {
#pragma unroll
        for (int b = 0; b < RKM_NBUF; ++b) mbar_init(&mbar[b], 1);
        mbar_fence_init();
    }
    if (tma) __syncthreads();
    auto issue_plane = [&](int kk, int buf) {
        double *sb = sm + buf * PLANE;
        if (tma) {
            if (tid == 0) {
                mbar_arrive_expect_tx(&mbar[buf], 4 * RKM_TILE_BYTES);
#pragma unroll
                for (int m = 0; m < 4; ++m) tma_load_3d(sb + m * FS, &maps.m[m], &mbar[buf], x0 - 2, y0 - 1, kk & (nz - 1));
            }
        } else {
            const unsigned pk = plane * (unsigned)(kk & (nz - 1));
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                cp_async16(sb + m * FS + dst_a, a.qs[m] + (pk + src_a));
                if (has_b) cp_async16(sb + m * FS + dst_b, a.qs[m] + (pk + src_b));
            }
            if (has_h) cp_async8(sb + dst_h, qs_h + (pk + src_h));
        }
        cp_async_commit();
    };

#pragma unroll
    for (int n = 0; n <= RKM_NBUF - 2; ++n) issue_plane(k0 + n, n);
    // z-carried values of this thread's column: z-1, centre, z+1 (rotated by copy at the end of every plane)
    double2 zm[4], cur[4], zp[4];
    {
        const unsigned pkm = plane * (unsigned)((k0 - 1) & (nz - 1)) + orow;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            zm[m] = __ldg(reinterpret_cast<const double2 *>(a.qs[m] + pkm));
            cur[m] = zp[m] = make_double2(0.0, 0.0);
        }
    }
    const int own = (ty + 1) * SW + 2 + 2 * tx; // this thread's pair inside a field's tile
    unsigned fraw_next = 0x7f7f;
    if (MASKED) fraw_next = *reinterpret_cast<const unsigned short *>(a.face + (plane * (unsigned)k0 + orow));
    // sources whose x and y factors are non-zero at this thread's cells (their z factor is checked per plane)
    unsigned smask = 0;
    if (SOURCES) {
        for (int s = 0; s < a.nsrc; ++s) {
            const double *tb = a.stab + a.src[s].off;
            const double2 sx = __ldg(reinterpret_cast<const double2 *>(tb + i));
            if ((sx.x != 0.0 || sx.y != 0.0) && __ldg(&tb[nx + j]) != 0.0) smask |= 1u << s;
        }
    }
    const RhsCoef &kf = a.kf;

    for (int t = 0; t < kc; ++t) {
        const int k = k0 + t;
        const unsigned o = plane * (unsigned)k + orow;
        // operands that do not go through shared memory: issue their loads before waiting
        double2 qn[4], q2[4];
        // face bytes: fetched one plane ahead and left packed until here, so the load is never waited for
        const unsigned fraw = fraw_next;
        if (MASKED && t + 1 < kc) fraw_next = *reinterpret_cast<const unsigned short *>(a.face + (o + plane));
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            if (STAGE >= 2 && (STAGE <= 3 || !ELIM)) qn[m] = __ldg(reinterpret_cast<const double2 *>(a.qn[m] + o));
            if (STAGE >= 2 && !ELIM) q2[m] = *reinterpret_cast<const double2 *>(a.qc[m] + o); // Qc, updated in place
            if (STAGE == 4 && ELIM) q2[m] = *reinterpret_cast<const double2 *>(a.qc[m] + o);  // S, overwritten below by Q*
        }
        cp_async_wait_n<RKM_NBUF - 3>();
        if (tma) { // the tile of plane k+1 (and of plane k at the first step) has landed: tile n of the block is use n/4 of its mbarrier
            if (t == 0) mbar_wait(&mbar[0], 0);
            mbar_wait(&mbar[(t + 1) % RKM_NBUF], ((t + 1) / RKM_NBUF) & 1);
        }
        __syncthreads(); // plane k+1 visible to all; every thread is done with the tile of plane k-1
        if (t + RKM_NBUF - 1 <= kc) issue_plane(k + RKM_NBUF - 1, (t + RKM_NBUF - 1) % RKM_NBUF);
        else cp_async_commit();
        const double *sC = sm + (t % RKM_NBUF) * PLANE, *sN = sm + ((t + 1) % RKM_NBUF) * PLANE;
        if (t == 0) {
#pragma unroll
            for (int m = 0; m < 4; ++m) cur[m] = *reinterpret_cast<const double2 *>(sC + m * FS + own);
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) zp[m] = *reinterpret_cast<const double2 *>(sN + m * FS + own);
        if (STAGE == 1) {
#pragma unroll
            for (int m = 0; m < 4; ++m) qn[m] = cur[m];
        }
        // factored form of the right-hand side: per cell six coefficients shared by the four fields
        //   A+-_a = -(u_a(+-a) + u_a)/(4 Delta_a), then F = sum_a [q(+a)(A+_a + D_a) + q(-a)(D_a - A-_a)] - 2 sum_a D_a q0 + b
        double axp[2], axm[2], ayp[2], aym[2], azp[2], azm[2];
        {
            const double2 vym = *reinterpret_cast<const double2 *>(sC + 1 * FS + own - SW);
            const double2 vyp = *reinterpret_cast<const double2 *>(sC + 1 * FS + own + SW);
            const double uxmA = sC[own - 1], uxpB = sC[own + 2];
            axp[0] = (cur[0].y + cur[0].x) * kf.hx; axm[0] = (uxmA + cur[0].x) * kf.hx;
            axp[1] = (uxpB + cur[0].y) * kf.hx;     axm[1] = axp[0];
            ayp[0] = (vyp.x + cur[1].x) * kf.hy; aym[0] = (vym.x + cur[1].x) * kf.hy;
            ayp[1] = (vyp.y + cur[1].y) * kf.hy; aym[1] = (vym.y + cur[1].y) * kf.hy;
            azp[0] = (zp[2].x + cur[2].x) * kf.hz; azm[0] = (zm[2].x + cur[2].x) * kf.hz;
            azp[1] = (zp[2].y + cur[2].y) * kf.hz; azm[1] = (zm[2].y + cur[2].y) * kf.hz;
        }
        // The rest of the plane in two versions chosen per warp (no divergence): WALL = some cell of this warp's row
        // has a solid cell in its seven-point neighbourhood.  Nine warps in ten of a room see none and run without a
        // single select (the face-weighted diffusion of eq. 4 and the beta ? x : +0.0 of PAPER.md:58 cost 20 selects per
        // cell); both versions give the same bits for an all-fluid neighbourhood.
        auto finish = [&](auto wall_tag) {
            constexpr bool WALL = decltype(wall_tag)::value;
            const unsigned fA = fraw & 0xffu, fB = fraw >> 8;
            double2 F[4];
            {
                // scalar first: its diffusive coefficients carry the face bits of eq. 4
                const double *sf = sC + 3 * FS + own;
                const double2 ym = *reinterpret_cast<const double2 *>(sf - SW), yp = *reinterpret_cast<const double2 *>(sf + SW);
                const double xpv[2] = {cur[3].y, sf[2]}, xmv[2] = {sf[-1], cur[3].x};
                const double ypv[2] = {yp.x, yp.y}, ymv[2] = {ym.x, ym.y}, zpv[2] = {zp[3].x, zp[3].y}, zmv[2] = {zm[3].x, zm[3].y};
                const double c0v[2] = {cur[3].x, cur[3].y};
                const unsigned fv[2] = {fA, fB};
                double out[2];
#pragma unroll
                for (int l = 0; l < 2; ++l) {
                    double v;
                    if (!WALL) {
                        v = kf.dc0 * c0v[l];
                        v = fma(xpv[l], axp[l] + kf.dcx, v);
                        v = fma(xmv[l], kf.dcx - axm[l], v);
                        v = fma(ypv[l], ayp[l] + kf.dcy, v);
                        v = fma(ymv[l], kf.dcy - aym[l], v);
                        v = fma(zpv[l], azp[l] + kf.dcz, v);
                        v = fma(zmv[l], kf.dcz - azm[l], v);
                    } else {
                        const unsigned fl = fv[l];
                        const double exp_ = (fl & 2) ? kf.dcx : 0.0, exm = (fl & 4) ? kf.dcx : 0.0;
                        const double eyp = (fl & 8) ? kf.dcy : 0.0, eym = (fl & 16) ? kf.dcy : 0.0;
                        const double ezp = (fl & 32) ? kf.dcz : 0.0, ezm = (fl & 64) ? kf.dcz : 0.0;
                        v = -(((exp_ + exm) + (eyp + eym)) + (ezp + ezm)) * c0v[l];
                        v = fma(xpv[l], axp[l] + exp_, v);
                        v = fma(xmv[l], exm - axm[l], v);
                        v = fma(ypv[l], ayp[l] + eyp, v);
                        v = fma(ymv[l], eym - aym[l], v);
                        v = fma(zpv[l], azp[l] + ezp, v);
                        v = fma(zmv[l], ezm - azm[l], v);
                    }
                    out[l] = v;
                }
                F[3] = make_double2(out[0], out[1]);
            }
            double bxp[2], bxm[2], byp[2], bym[2], bzp[2], bzm[2];
#pragma unroll
            for (int l = 0; l < 2; ++l) {
                bxp[l] = axp[l] + kf.dvx; bxm[l] = kf.dvx - axm[l];
                byp[l] = ayp[l] + kf.dvy; bym[l] = kf.dvy - aym[l];
                bzp[l] = azp[l] + kf.dvz; bzm[l] = kf.dvz - azm[l];
            }
#pragma unroll
            for (int m = 0; m < 3; ++m) {
                const double *sf = sC + m * FS + own;
                const double2 ym = *reinterpret_cast<const double2 *>(sf - SW), yp = *reinterpret_cast<const double2 *>(sf + SW);
                const double xmA = sf[-1], xpB = sf[2];
                double vx = fma(kf.dv0, cur[m].x, a.body[m]), vy = fma(kf.dv0, cur[m].y, a.body[m]);
                vx = fma(cur[m].y, bxp[0], vx); vy = fma(xpB, bxp[1], vy);
                vx = fma(xmA, bxm[0], vx);      vy = fma(cur[m].x, bxm[1], vy);
                vx = fma(yp.x, byp[0], vx);     vy = fma(yp.y, byp[1], vy);
                vx = fma(ym.x, bym[0], vx);     vy = fma(ym.y, bym[1], vy);
                vx = fma(zp[m].x, bzp[0], vx);  vy = fma(zp[m].y, bzp[1], vy);
                vx = fma(zm[m].x, bzm[0], vx);  vy = fma(zm[m].y, bzm[1], vy);
                F[m] = make_double2(vx, vy);
            }
            if (SOURCES) {
                for (unsigned sm_ = smask; sm_; sm_ &= sm_ - 1) {
                    const int s = __ffs(sm_) - 1;
                    const double *tb = a.stab + a.src[s].off;
                    const double sz = __ldg(&tb[nx + ny + k]), sy = __ldg(&tb[nx + j]);
                    if (sz == 0.0) continue;
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
            const bool flA = !WALL || (fA & 1), flB = !WALL || (fB & 1);
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                // solid cell: every field it holds is +0.0 and stays +0.0 (select)
                if (ELIM) {
                    double2 r;
                    if (STAGE < 4) {
                        r.x = flA ? qn[m].x + a.ca * F[m].x : 0.0;
                        r.y = flB ? qn[m].y + a.ca * F[m].y : 0.0;
                        *reinterpret_cast<double2 *>(a.qo[m] + o) = r;
                        if (STAGE == 2) { // S = Q2 - Qn + 2 Q3 (all +0.0 in solid cells)
                            double2 sv;
                            sv.x = flA ? (cur[m].x - qn[m].x) + 2.0 * r.x : 0.0;
                            sv.y = flB ? (cur[m].y - qn[m].y) + 2.0 * r.y : 0.0;
                            *reinterpret_cast<double2 *>(a.qco[m] + o) = sv;
                        }
                    } else {
                        r.x = flA ? (q2[m].x + cur[m].x) * (1.0 / 3.0) + a.cb * F[m].x : 0.0;
                        r.y = flB ? (q2[m].y + cur[m].y) * (1.0 / 3.0) + a.cb * F[m].y : 0.0;
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
        };
        if (MASKED && __any_sync(0xffffffffu, fraw != 0x7f7fu)) finish(BoolTag<true>{});
        else finish(BoolTag<false>{});
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
// one solid face neighbour; `rec` holds one 64-bit record per such cell in ascending index order (built at
// create): bits 0-31 the linear index, bits 32-38 the face byte, so that one coalesced load tells a thread
// both where its cell is and which of the six p neighbours it needs -- every other load of the kernel can then
// be issued at once (it was a chain of three dependent loads: index, face byte, neighbours).
// The first iteration of a step saves d at those cells (`save`), later ones restore it from there, and
// r overwrites d in place: everywhere else r == d already, so the forward x pass reads one plain array.
// face: bit0 beta(cell), bit1/2 beta(x+1/x-1), bit3/4 beta(y+1/y-1), bit5/6 beta(z+1/z-1).
// The kernel is a chain of two memory latencies (record, then d / p and its neighbours) and nothing else, so the grid is
// one wave of blocks that stride through the list and each thread asks for its NEXT record before it works on the current
// one: the two latencies overlap (measured on 512x256x128, 1.5 M records: see DESIGN.md section 6).
template <bool FIRST>
__global__ void __launch_bounds__(256) k_eq9_sparse(double *__restrict__ d, const double *__restrict__ p, const unsigned long long *__restrict__ rec,
                                                    double *__restrict__ save, int nlist, int nx, int ny, int nz, int lgx, int lgy,
                                                    double r2x, double r2y, double r2z)
{
    // neighbour offsets two cells away, periodic: extents are powers of two and the whole array has fewer than 2^32
    // elements, so each axis is a bit field of the linear index and the wrap is a masked add
    const uint32_t mx_ = (uint32_t)nx - 1u, my_ = ((uint32_t)ny - 1u) << lgx, mz_ = ((uint32_t)nz - 1u) << (lgx + lgy);
    const uint32_t sx = 2u, sy = 2u << lgx, sz = 2u << (lgx + lgy);
    const int stride = gridDim.x * 256;
    int n = blockIdx.x * 256 + threadIdx.x;
    unsigned long long rc = n < nlist ? __ldg(&rec[n]) : 0ull;
    for (; n < nlist; n += stride) {
        const unsigned long long cur = rc;
        if (n + stride < nlist) rc = __ldg(&rec[n + stride]);
        const uint32_t oo = (uint32_t)cur;
        const unsigned ff = (unsigned)(cur >> 32);
        const double dv = FIRST ? d[oo] : save[n];
        const double pc = __ldg(&p[oo]);
        double pn[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        if (!(ff & 2)) pn[0] = __ldg(&p[(oo & ~mx_) | ((oo + sx) & mx_)]);
        if (!(ff & 4)) pn[1] = __ldg(&p[(oo & ~mx_) | ((oo - sx) & mx_)]);
        if (!(ff & 8)) pn[2] = __ldg(&p[(oo & ~my_) | ((oo + sy) & my_)]);
        if (!(ff & 16)) pn[3] = __ldg(&p[(oo & ~my_) | ((oo - sy) & my_)]);
        if (!(ff & 32)) pn[4] = __ldg(&p[(oo & ~mz_) | ((oo + sz) & mz_)]);
        if (!(ff & 64)) pn[5] = __ldg(&p[(oo & ~mz_) | ((oo - sz) & mz_)]);
        if (FIRST) save[n] = dv;
        double gxp = 0.0, gxm = 0.0, gyp = 0.0, gym = 0.0, gzp = 0.0, gzm = 0.0;
        if (!(ff & 2)) gxp = (pn[0] - pc) * r2x;
        if (!(ff & 4)) gxm = (pc - pn[1]) * r2x;
        if (!(ff & 8)) gyp = (pn[2] - pc) * r2y;
        if (!(ff & 16)) gym = (pc - pn[3]) * r2y;
        if (!(ff & 32)) gzp = (pn[4] - pc) * r2z;
        if (!(ff & 64)) gzm = (pc - pn[5]) * r2z;
        d[oo] = dv + ((gxp - gxm) * r2x + (gyp - gym) * r2y + (gzp - gzm) * r2z);
    }
}

// NEXT-1, eq. 6: out = beta ? f + sum_a gamma_a d6_a f : +0.0 with gamma_a = Delta_a^6/pi^6 and
// d6_a the central 7-point stencil (1,-6,15,-20,15,-6,1)/Delta_a^6 (reading R23), on u, v, w, c.
// One thread per (x, y) column of one field, marching kc planes: the seven z values ride in registers,
// the x and y neighbours come through L1 (a block touches a 38 x 14 patch of each plane).
// blockIdx.z enumerates (z chunk, field).
struct FilterArgs {
    const double *in[4];
    double *out[4];
    const uint8_t *face; // null: no solid cells
    int nx, ny, nz, kc;
    double g;            // 1/pi^6
};

template <bool MASKED> __global__ void __launch_bounds__(256) k_filter(const FilterArgs a)
{
    const int nx = a.nx, ny = a.ny, nz = a.nz;
    const int m = blockIdx.z & 3, k0 = (blockIdx.z >> 2) * a.kc;
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    const double *__restrict__ f = a.in[m];
    double *__restrict__ o = a.out[m];
    const size_t plane = (size_t)nx * ny;
    const size_t col = (size_t)nx * j + i, row = (size_t)nx * j;
    size_t xo[6], yo[6];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        xo[d] = row + ((i - 3 + d) & (nx - 1));
        xo[3 + d] = row + ((i + 1 + d) & (nx - 1));
        yo[d] = (size_t)nx * ((j - 3 + d) & (ny - 1)) + i;
        yo[3 + d] = (size_t)nx * ((j + 1 + d) & (ny - 1)) + i;
    }
    double z[7]; // z[3] is the centre
#pragma unroll
    for (int d = 0; d < 6; ++d) z[d + 1] = __ldg(f + plane * (size_t)((k0 - 3 + d) & (nz - 1)) + col);
    for (int t = 0; t < a.kc; ++t) {
        const int k = k0 + t;
        const size_t pk = plane * (size_t)k;
#pragma unroll
        for (int d = 0; d < 6; ++d) z[d] = z[d + 1];
        z[6] = __ldg(f + plane * (size_t)((k + 3) & (nz - 1)) + col);
        bool fluid = true;
        if (MASKED) fluid = (a.face[pk + col] & 1) != 0;
        const double f0 = z[3];
        const double sx = __ldg(f + pk + xo[0]) - 6.0 * __ldg(f + pk + xo[1]) + 15.0 * __ldg(f + pk + xo[2]) - 20.0 * f0 +
                          15.0 * __ldg(f + pk + xo[3]) - 6.0 * __ldg(f + pk + xo[4]) + __ldg(f + pk + xo[5]);
        const double sy = __ldg(f + pk + yo[0]) - 6.0 * __ldg(f + pk + yo[1]) + 15.0 * __ldg(f + pk + yo[2]) - 20.0 * f0 +
                          15.0 * __ldg(f + pk + yo[3]) - 6.0 * __ldg(f + pk + yo[4]) + __ldg(f + pk + yo[5]);
        const double sz = z[0] - 6.0 * z[1] + 15.0 * z[2] - 20.0 * f0 + 15.0 * z[4] - 6.0 * z[5] + z[6];
        o[pk + col] = fluid ? f0 + a.g * ((sx + sy) + sz) : 0.0;
    }
}

// k_filter_march: eq. 6 for grids with nx >= 64, ny >= 8.  A block owns a 64 x 8 (x by y) column of ONE field
// and walks kc planes; each thread owns two x-adjacent cells.  Plane tiles (14 rows x 72 doubles: three-cell
// halo in y, four in x so that every pair is 16-byte aligned) arrive by cp.async, two planes in flight; the
// x and y neighbours of plane k come from its tile, the z+3 value from the tile of plane k+3, the other six
// z values ride in registers.  Every value is fetched from L2/HBM once per block (plus halo).
constexpr int FM_TX = 64, FM_TY = 8, FM_W = FM_TX + 8, FM_ROWS = FM_TY + 6, FM_NBUF = 6;
constexpr int FM_TILE = FM_ROWS * FM_W;
constexpr int FM_SMEM = FM_NBUF * FM_TILE * (int)sizeof(double);
constexpr int FM_CHUNKS = FM_ROWS * (FM_W / 2);

template <bool MASKED> __global__ void __launch_bounds__(256) k_filter_march(const FilterArgs a)
{
    extern __shared__ double2 fm_smem2[];
    double *sm = reinterpret_cast<double *>(fm_smem2);
    const int nx = a.nx, ny = a.ny, nz = a.nz, kc = a.kc;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * 32 + tx;
    const int m = blockIdx.z & 3, k0 = (blockIdx.z >> 2) * kc;
    const int x0 = blockIdx.x * FM_TX, y0 = blockIdx.y * FM_TY;
    const double *__restrict__ f = a.in[m];
    double *__restrict__ o = a.out[m];
    const size_t plane = (size_t)nx * ny;
    const size_t col = (size_t)nx * (y0 + ty) + x0 + 2 * tx;
    const int own = (ty + 3) * FM_W + 4 + 2 * tx;

    // this thread's chunks of one plane tile
    const int c1 = tid + 256;
    const int r0 = tid / (FM_W / 2), q0 = tid - r0 * (FM_W / 2), r1 = c1 / (FM_W / 2), q1 = c1 - r1 * (FM_W / 2);
    const bool has1 = c1 < FM_CHUNKS;
    const unsigned s0 = (unsigned)nx * ((y0 - 3 + r0) & (ny - 1)) + ((x0 - 4 + 2 * q0) & (nx - 1));
    const unsigned s1 = (unsigned)nx * ((y0 - 3 + r1) & (ny - 1)) + ((x0 - 4 + 2 * q1) & (nx - 1));
    const int d0 = r0 * FM_W + 2 * q0, d1 = r1 * FM_W + 2 * q1;
    auto issue = [&](int n, int buf) { // plane k0+n into tile `buf` (= n % 6)
        const double *src = f + plane * (size_t)((k0 + n) & (nz - 1));
        double *dst = sm + buf * FM_TILE;
        cp_async16(dst + d0, src + s0);
        if (has1) cp_async16(dst + d1, src + s1);
    };
#pragma unroll
    for (int n = 0; n < 5; ++n) {
        issue(n, n);
        cp_async_commit();
    }
    double2 z[7]; // z[3] is the centre plane
#pragma unroll
    for (int d = 0; d < 3; ++d) z[d + 1] = __ldg(reinterpret_cast<const double2 *>(f + plane * (size_t)((k0 - 3 + d) & (nz - 1)) + col));
    asm volatile("cp.async.wait_group 2;\n" ::: "memory");
    __syncthreads();
#pragma unroll
    for (int d = 0; d < 3; ++d) z[d + 4] = *reinterpret_cast<const double2 *>(sm + d * FM_TILE + own);

    // tile indices t % 6, (t + 3) % 6, (t + 5) % 6 as running counters (a modulo by 6 per use cost ~15 instructions each);
    // the face bytes of plane t + 1 are fetched while plane t is computed
    int bc = 0, b3 = 3, b5 = 5;
    size_t pk = plane * (size_t)k0 + col;
    unsigned fnext = 0x0101;
    if (MASKED) fnext = *reinterpret_cast<const unsigned short *>(a.face + pk);
    for (int t = 0; t < kc; ++t, pk += plane) {
        const unsigned fcur = fnext;
        if (MASKED && t + 1 < kc) fnext = *reinterpret_cast<const unsigned short *>(a.face + pk + plane);
        cp_async_wait_one();
        __syncthreads(); // tile t+3 visible; every thread is done with tile t-1
        if (t + 5 <= kc + 2) issue(t + 5, b5);
        cp_async_commit();
#pragma unroll
        for (int d = 0; d < 6; ++d) z[d] = z[d + 1];
        z[6] = *reinterpret_cast<const double2 *>(sm + b3 * FM_TILE + own);
        const double *sc = sm + bc * FM_TILE + own;
        bc = bc == FM_NBUF - 1 ? 0 : bc + 1;
        b3 = b3 == FM_NBUF - 1 ? 0 : b3 + 1;
        b5 = b5 == FM_NBUF - 1 ? 0 : b5 + 1;
        const double2 xa = *reinterpret_cast<const double2 *>(sc - 4), xb = *reinterpret_cast<const double2 *>(sc - 2);
        const double2 xc = *reinterpret_cast<const double2 *>(sc + 2), xd = *reinterpret_cast<const double2 *>(sc + 4);
        const double2 c = z[3];
        // cell A = c.x: x-3..x+3 = xa.y xb.x xb.y | c.y xc.x xc.y;   cell B = c.y: xb.x xb.y c.x | xc.x xc.y xd.x
        const double sxA = xa.y - 6.0 * xb.x + 15.0 * xb.y - 20.0 * c.x + 15.0 * c.y - 6.0 * xc.x + xc.y;
        const double sxB = xb.x - 6.0 * xb.y + 15.0 * c.x - 20.0 * c.y + 15.0 * xc.x - 6.0 * xc.y + xd.x;
        const double2 y0v = *reinterpret_cast<const double2 *>(sc - 3 * FM_W), y1v = *reinterpret_cast<const double2 *>(sc - 2 * FM_W);
        const double2 y2v = *reinterpret_cast<const double2 *>(sc - FM_W), y4v = *reinterpret_cast<const double2 *>(sc + FM_W);
        const double2 y5v = *reinterpret_cast<const double2 *>(sc + 2 * FM_W), y6v = *reinterpret_cast<const double2 *>(sc + 3 * FM_W);
        const double syA = y0v.x - 6.0 * y1v.x + 15.0 * y2v.x - 20.0 * c.x + 15.0 * y4v.x - 6.0 * y5v.x + y6v.x;
        const double syB = y0v.y - 6.0 * y1v.y + 15.0 * y2v.y - 20.0 * c.y + 15.0 * y4v.y - 6.0 * y5v.y + y6v.y;
        const double szA = z[0].x - 6.0 * z[1].x + 15.0 * z[2].x - 20.0 * c.x + 15.0 * z[4].x - 6.0 * z[5].x + z[6].x;
        const double szB = z[0].y - 6.0 * z[1].y + 15.0 * z[2].y - 20.0 * c.y + 15.0 * z[4].y - 6.0 * z[5].y + z[6].y;
        double2 r;
        r.x = (!MASKED || (fcur & 1)) ? c.x + a.g * ((sxA + syA) + szA) : 0.0;
        r.y = (!MASKED || (fcur & 0x100)) ? c.y + a.g * ((sxB + syB) + szB) : 0.0;
        *reinterpret_cast<double2 *>(o + pk) = r;
    }
}

// a4 and a6 with two x-adjacent cells per thread (16-byte accesses, twice the bytes in flight per thread); nx >= 64.
// blockDim = (32, 8): a block covers 64 x 8 cells of one plane.
__global__ void __launch_bounds__(256) k_div2(const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
                                              double *__restrict__ d, int nx, int ny, int nz, double r2x, double r2y, double r2z, int rev)
{
    const int i = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
    const int j = (rev ? gridDim.y - 1 - blockIdx.y : blockIdx.y) * blockDim.y + threadIdx.y, k = rev ? gridDim.z - 1 - blockIdx.z : blockIdx.z;
    const size_t plane = (size_t)nx * ny, pk = plane * k, row = pk + (size_t)nx * j;
    const double2 vp = __ldg(reinterpret_cast<const double2 *>(v + pk + (size_t)nx * ((j + 1) & (ny - 1)) + i));
    const double2 vm = __ldg(reinterpret_cast<const double2 *>(v + pk + (size_t)nx * ((j - 1) & (ny - 1)) + i));
    const double2 wp = __ldg(reinterpret_cast<const double2 *>(w + plane * ((k + 1) & (nz - 1)) + (size_t)nx * j + i));
    const double2 wm = __ldg(reinterpret_cast<const double2 *>(w + plane * ((k - 1) & (nz - 1)) + (size_t)nx * j + i));
    const double2 uc = __ldg(reinterpret_cast<const double2 *>(u + row + i));
    const double um = __ldg(u + row + ((i - 1) & (nx - 1))), up = __ldg(u + row + ((i + 2) & (nx - 1)));
    double2 r;
    r.x = (uc.y - um) * r2x + (vp.x - vm.x) * r2y + (wp.x - wm.x) * r2z;
    r.y = (up - uc.x) * r2x + (vp.y - vm.y) * r2y + (wp.y - wm.y) * r2z;
    *reinterpret_cast<double2 *>(d + row + i) = r;
}

template <bool MASKED>
__global__ void __launch_bounds__(256) k_project2(double *__restrict__ u, double *__restrict__ v, double *__restrict__ w, const double *__restrict__ p,
                                                  const uint8_t *__restrict__ face, int nx, int ny, int nz, double r2x, double r2y, double r2z, int rev)
{
    const int i = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
    const int j = (rev ? gridDim.y - 1 - blockIdx.y : blockIdx.y) * blockDim.y + threadIdx.y, k = rev ? gridDim.z - 1 - blockIdx.z : blockIdx.z;
    const size_t plane = (size_t)nx * ny, pk = plane * k, row = pk + (size_t)nx * j, o = row + i;
    unsigned f = 0x0101;
    if (MASKED) f = *reinterpret_cast<const unsigned short *>(face + o);
    const double2 pyp = __ldg(reinterpret_cast<const double2 *>(p + pk + (size_t)nx * ((j + 1) & (ny - 1)) + i));
    const double2 pym = __ldg(reinterpret_cast<const double2 *>(p + pk + (size_t)nx * ((j - 1) & (ny - 1)) + i));
    const double2 pzp = __ldg(reinterpret_cast<const double2 *>(p + plane * ((k + 1) & (nz - 1)) + (size_t)nx * j + i));
    const double2 pzm = __ldg(reinterpret_cast<const double2 *>(p + plane * ((k - 1) & (nz - 1)) + (size_t)nx * j + i));
    const double2 pc = __ldg(reinterpret_cast<const double2 *>(p + o));
    const double pm = __ldg(p + row + ((i - 1) & (nx - 1))), pp = __ldg(p + row + ((i + 2) & (nx - 1)));
    double2 uu = *reinterpret_cast<const double2 *>(u + o), vv = *reinterpret_cast<const double2 *>(v + o), ww = *reinterpret_cast<const double2 *>(w + o);
    const bool fa = (f & 1) != 0, fb = (f & 0x100) != 0;
    uu.x = fa ? uu.x - (pc.y - pm) * r2x : 0.0;
    uu.y = fb ? uu.y - (pp - pc.x) * r2x : 0.0;
    vv.x = fa ? vv.x - (pyp.x - pym.x) * r2y : 0.0;
    vv.y = fb ? vv.y - (pyp.y - pym.y) * r2y : 0.0;
    ww.x = fa ? ww.x - (pzp.x - pzm.x) * r2z : 0.0;
    ww.y = fb ? ww.y - (pzp.y - pzm.y) * r2z : 0.0;
    *reinterpret_cast<double2 *>(u + o) = uu;
    *reinterpret_cast<double2 *>(v + o) = vv;
    *reinterpret_cast<double2 *>(w + o) = ww;
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
