// reduce.cuh -- NEXT-3: the two global reductions of the paper's main loop ("AdjustDt.m",
// PAPER.md:265-269 mean and standard deviation of the CO2 field): Courant number, and mean / standard
// deviation of the scalar over the fluid cells of an index box.  Both are one streaming read of the
// fields; partial results are combined in a fixed order, so the results are reproducible run to run.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dnsred {

// max over all cells of |u|/dx + |v|/dy + |w|/dz (reading R24), bit-identical to a plain loop of that
// expression.  Three correctly rounded fp64 divisions per cell would make this a compute-bound kernel (132 us on
// 512x256x128 against 62 us for its one read of u, v, w), so every cell is first rated with reciprocal multiplies
// (|u| rx + |v| ry + |w| rz, within 1e-15 relative of the exact expression: all terms are non-negative), and the
// exact expression with its divisions is evaluated only where that rating comes within 1e-14 of the largest rating
// the WARP has seen so far -- which always includes the cell of the true maximum, and happens O(log n) times per warp
// (a per-thread threshold would make some lane of the warp take the slow path at almost every step).
// The bit pattern of a non-negative double orders like an unsigned integer, which makes the final maximum an integer
// atomicMax.  A NaN rate never compares greater and is skipped, as in `if (r > best) best = r`.
__global__ void __launch_bounds__(256) k_courant(const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
                                                 size_t n, double dx, double dy, double dz, unsigned long long *__restrict__ out)
{
    const double rx = 1.0 / dx, ry = 1.0 / dy, rz = 1.0 / dz;
    double best = 0.0, rated = 0.0; // exact maximum of this thread's cells so far; largest rating this warp knows of
    // the largest rating any warp of the block has seen (bit pattern: non-negative doubles order like integers).  Any rating
    // seen anywhere is a valid threshold -- its cell was evaluated exactly when it set its warp's record -- and a shared
    // one rises faster: with per-warp records only, a quarter of the trips took the slow path on a noisy field.
    __shared__ unsigned long long s_rated;
    if (threadIdx.x == 0) s_rated = 0ull;
    __syncthreads();
    auto rate = [&](double uu, double vv, double ww) { return fma(fabs(ww), rz, fma(fabs(vv), ry, fabs(uu) * rx)); };
    auto exact = [&](double uu, double vv, double ww) {
        const double r = fabs(uu) / dx + fabs(vv) / dy + fabs(ww) / dz;
        if (r > best) best = r;
    };
    const size_t n2 = n / 2, stride = (size_t)gridDim.x * blockDim.x;
    const double2 *u2 = reinterpret_cast<const double2 *>(u), *v2 = reinterpret_cast<const double2 *>(v), *w2 = reinterpret_cast<const double2 *>(w);
    // whole warps enter or leave the loop together: the bound is rounded up to a multiple of 32 and lanes past the end idle
    const size_t first = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    // two strides per trip: six 16-byte loads in flight per thread (with three, at the 24 warps per SM the exact path's
    // registers allow, the kernel ran at 4.3 TB/s)
    for (size_t o = first; o - (threadIdx.x & 31) < n2; o += 2 * stride) {
        double2 a[2], b[2], c[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const size_t oh = o + h * stride;
            a[h] = b[h] = c[h] = make_double2(0.0, 0.0);
            if (oh < n2) {
                a[h] = __ldg(u2 + oh);
                b[h] = __ldg(v2 + oh);
                c[h] = __ldg(w2 + oh);
            }
        }
        rated = fmax(rated, __longlong_as_double((long long)*(volatile unsigned long long *)&s_rated));
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const double q0 = rate(a[h].x, b[h].x, c[h].x), q1 = rate(a[h].y, b[h].y, c[h].y);
            const double thr = rated * (1.0 - 1e-14);
            const bool t0 = q0 >= thr, t1 = q1 >= thr;
            if (__any_sync(0xffffffffu, t0 || t1)) {
                if (t0) exact(a[h].x, b[h].x, c[h].x);
                if (t1) exact(a[h].y, b[h].y, c[h].y);
                double m = fmax(rated, fmax(q0, q1)); // fmax ignores a NaN rating
#pragma unroll
                for (int s = 16; s > 0; s >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, s));
                rated = m;
                if ((threadIdx.x & 31) == 0) atomicMax(&s_rated, (unsigned long long)__double_as_longlong(m));
            }
        }
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) exact(u[n - 1], v[n - 1], w[n - 1]);
    unsigned long long b = (unsigned long long)__double_as_longlong(best);
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        const unsigned long long t = __shfl_xor_sync(0xffffffffu, b, s);
        b = t > b ? t : b;
    }
    if ((threadIdx.x & 31) == 0 && b != 0ull) atomicMax(out, b);
}

struct BoxArgs {
    const double *c;
    const uint8_t *face; // null: every cell is fluid
    int nx, ny, nz;
    int lo[3], size[3];  // index box, wraps modulo N
    size_t count;        // size[0]*size[1]*size[2]
};

// sum over the block's threads, valid in thread 0 (fixed order: lanes by shuffle tree, then warps 0..7)
__device__ __forceinline__ double block_sum(double v, double *sh)
{
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) v += __shfl_down_sync(0xffffffffu, v, s);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int wv = 0; wv < (int)(blockDim.x >> 5); ++wv) t += sh[wv];
    __syncthreads();
    return t;
}

// PASS 0: partial sums of c and fluid-cell counts;  PASS 1: partial sums of (c - mean)^2, mean = res[0].
// The box is walked by rows (j, k): block b takes rows b*rpb .. (b+1)*rpb-1, its warps take them in turn, the lanes
// stride along x -- no division per cell, coalesced 256-byte reads.  part[b], part[G + b].
template <int PASS>
__global__ void __launch_bounds__(256) k_box_partial(const BoxArgs a, unsigned rows, unsigned rpb, const double *__restrict__ res,
                                                     double *__restrict__ part)
{
    __shared__ double sh[8];
    const double mean = PASS == 1 ? res[0] : 0.0;
    const unsigned beg = blockIdx.x * rpb, end = beg + rpb < rows ? beg + rpb : rows;
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    double s = 0.0, cnt = 0.0;
    for (unsigned row = beg + wv; row < end; row += 8) {
        const unsigned k = row / (unsigned)a.size[1], j = row - k * (unsigned)a.size[1];
        const size_t rowo = (size_t)a.nx * ((size_t)((a.lo[1] + j) & (a.ny - 1)) + (size_t)a.ny * ((a.lo[2] + k) & (a.nz - 1)));
        const double *cr = a.c + rowo;
        const uint8_t *fr = a.face != nullptr ? a.face + rowo : nullptr;
        // a row segment that starts on an even cell, has an even length and does not wrap is walked two cells per lane
        // (16-byte loads: 3.3 -> 5 TB/s on a whole 512x256x128 box); the order of a lane's additions is fixed either way
        if (((a.lo[0] | a.size[0]) & 1) == 0 && a.lo[0] + a.size[0] <= a.nx) {
            const double2 *cr2 = reinterpret_cast<const double2 *>(cr + a.lo[0]);
            const uchar2 *fr2 = fr != nullptr ? reinterpret_cast<const uchar2 *>(fr + a.lo[0]) : nullptr;
#pragma unroll 4
            for (int i = lane; i < a.size[0] / 2; i += 32) {
                const double2 cv = __ldg(cr2 + i);
                uchar2 f = make_uchar2(1, 1);
                if (fr2 != nullptr) f = fr2[i];
                const bool f0 = f.x & 1, f1 = f.y & 1;
                if (PASS == 0) {
                    s += f0 ? cv.x : 0.0;
                    s += f1 ? cv.y : 0.0;
                    cnt += (f0 ? 1.0 : 0.0) + (f1 ? 1.0 : 0.0);
                } else {
                    const double d0 = cv.x - mean, d1 = cv.y - mean;
                    s += f0 ? d0 * d0 : 0.0;
                    s += f1 ? d1 * d1 : 0.0;
                }
            }
            continue;
        }
        // four independent loads in flight per lane; solid cells add +0.0 (the sums keep their order)
#pragma unroll 4
        for (int i = lane; i < a.size[0]; i += 32) {
            const int x = (a.lo[0] + i) & (a.nx - 1);
            const bool fluid = fr == nullptr || (fr[x] & 1);
            const double cv = __ldg(cr + x);
            if (PASS == 0) {
                s += fluid ? cv : 0.0;
                cnt += fluid ? 1.0 : 0.0;
            } else {
                const double dv = cv - mean;
                s += fluid ? dv * dv : 0.0;
            }
        }
    }
    const double ts = block_sum(s, sh);
    const double tc = PASS == 0 ? block_sum(cnt, sh) : 0.0;
    if (threadIdx.x == 0) {
        part[blockIdx.x] = ts;
        if (PASS == 0) part[gridDim.x + blockIdx.x] = tc;
    }
}

// One block: combines the G partials in index order.  PASS 0: res[0] = mean, res[2] = count;
// PASS 1: res[1] = sqrt(sum / count) (population standard deviation, reading R25).  Empty box: zeros.
template <int PASS> __global__ void __launch_bounds__(256) k_box_final(const double *__restrict__ part, int G, double *__restrict__ res)
{
    __shared__ double sh[8];
    double s = 0.0, cnt = 0.0;
    for (int b = threadIdx.x; b < G; b += blockDim.x) {
        s += part[b];
        if (PASS == 0) cnt += part[G + b];
    }
    const double ts = block_sum(s, sh);
    const double tc = PASS == 0 ? block_sum(cnt, sh) : 0.0;
    if (threadIdx.x == 0) {
        if (PASS == 0) {
            res[2] = tc;
            res[0] = tc > 0.0 ? ts / tc : 0.0;
            res[1] = 0.0;
        } else {
            res[1] = res[2] > 0.0 ? sqrt(ts / res[2]) : 0.0;
        }
    }
}

// Variant of k_box_partial for dnslab_scalar_stats_static (the entry point whose scratch is the library's static
// device array): ONE partial per row (j, k) of the box instead of one per block -- part[row] holds the row's sum,
// part[rows + row] its fluid-cell count (PASS 0) -- so the number of scratch slots follows from the box alone and the
// result does not depend on how many SMs the device has.  One warp per row, lanes stride along x, lane sums folded by
// a shuffle tree (fixed order).  Every slot k_box_final<PASS>(part, rows, res) reads is written here first, whatever
// an earlier call left behind.  a.face is the CALLER's mask here: any non-zero byte is a fluid cell (k_box_partial
// reads the solver's face bytes, bit 0).
template <int PASS>
__global__ void __launch_bounds__(256) k_box_rows(const BoxArgs a, unsigned rows, const double *__restrict__ res, double *__restrict__ part)
{
    const unsigned row = blockIdx.x * 8u + (threadIdx.x >> 5);
    if (row >= rows) return; // whole warps leave together
    const int lane = threadIdx.x & 31;
    const double mean = PASS == 1 ? res[0] : 0.0;
    const unsigned k = row / (unsigned)a.size[1], j = row - k * (unsigned)a.size[1];
    const size_t rowo = (size_t)a.nx * ((size_t)((a.lo[1] + j) & (a.ny - 1)) + (size_t)a.ny * ((a.lo[2] + k) & (a.nz - 1)));
    const double *cr = a.c + rowo;
    const uint8_t *fr = a.face != nullptr ? a.face + rowo : nullptr;
    double s = 0.0, cnt = 0.0;
    // 16-byte loads where the segment is even, does not wrap and the caller's buffers are aligned for them
    if (((a.lo[0] | a.size[0]) & 1) == 0 && a.lo[0] + a.size[0] <= a.nx && ((uintptr_t)a.c & 15) == 0 && ((uintptr_t)a.face & 1) == 0) {
        const double2 *cr2 = reinterpret_cast<const double2 *>(cr + a.lo[0]);
        const uchar2 *fr2 = fr != nullptr ? reinterpret_cast<const uchar2 *>(fr + a.lo[0]) : nullptr;
#pragma unroll 4
        for (int i = lane; i < a.size[0] / 2; i += 32) {
            const double2 cv = __ldg(cr2 + i);
            uchar2 f = make_uchar2(1, 1);
            if (fr2 != nullptr) f = fr2[i];
            const bool f0 = f.x != 0, f1 = f.y != 0;
            if (PASS == 0) {
                s += f0 ? cv.x : 0.0;
                s += f1 ? cv.y : 0.0;
                cnt += (f0 ? 1.0 : 0.0) + (f1 ? 1.0 : 0.0);
            } else {
                const double d0 = cv.x - mean, d1 = cv.y - mean;
                s += f0 ? d0 * d0 : 0.0;
                s += f1 ? d1 * d1 : 0.0;
            }
        }
    } else {
#pragma unroll 4
        for (int i = lane; i < a.size[0]; i += 32) {
            const int x = (a.lo[0] + i) & (a.nx - 1);
            const bool fluid = fr == nullptr || fr[x] != 0;
            const double cv = __ldg(cr + x);
            if (PASS == 0) {
                s += fluid ? cv : 0.0;
                cnt += fluid ? 1.0 : 0.0;
            } else {
                const double dv = cv - mean;
                s += fluid ? dv * dv : 0.0;
            }
        }
    }
#pragma unroll
    for (int sh = 16; sh > 0; sh >>= 1) {
        s += __shfl_down_sync(0xffffffffu, s, sh);
        if (PASS == 0) cnt += __shfl_down_sync(0xffffffffu, cnt, sh);
    }
    if (lane == 0) {
        part[row] = s;
        if (PASS == 0) part[rows + row] = cnt;
    }
}

} // namespace dnsred
