// reduce.cuh -- NEXT-3: the two global reductions of the paper's main loop ("AdjustDt.m",
// PAPER.md:265-269 mean and standard deviation of the CO2 field): Courant number, and mean / standard
// deviation of the scalar over the fluid cells of an index box.  Both are one streaming read of the
// fields; partial results are combined in a fixed order, so the results are reproducible run to run.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dnsred {

// max over all cells of |u|/dx + |v|/dy + |w|/dz (reading R24).  Divisions and the order of the
// sum are those of the definition, so the value is bit-identical to a plain loop; the bit pattern of a
// non-negative double orders like an unsigned integer, which makes the maximum an integer atomicMax.
// A NaN rate never compares greater and is skipped, as in `if (r > best) best = r`.
__global__ void __launch_bounds__(256) k_courant(const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
                                                 size_t n, double dx, double dy, double dz, unsigned long long *__restrict__ out)
{
    double best = 0.0;
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        const double r = fabs(u[o]) / dx + fabs(v[o]) / dy + fabs(w[o]) / dz;
        if (r > best) best = r;
    }
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
// Block b handles box cells b*chunk .. (b+1)*chunk-1 (x fastest inside the box); part[b], part[G + b].
template <int PASS>
__global__ void __launch_bounds__(256) k_box_partial(const BoxArgs a, size_t chunk, const double *__restrict__ res, double *__restrict__ part)
{
    __shared__ double sh[8];
    const double mean = PASS == 1 ? res[0] : 0.0;
    const size_t beg = (size_t)blockIdx.x * chunk, end = beg + chunk < a.count ? beg + chunk : a.count;
    double s = 0.0, cnt = 0.0;
    for (size_t n = beg + threadIdx.x; n < end; n += blockDim.x) {
        const int i = (int)(n % a.size[0]), j = (int)((n / a.size[0]) % a.size[1]), k = (int)(n / ((size_t)a.size[0] * a.size[1]));
        const size_t o = (size_t)((a.lo[0] + i) & (a.nx - 1)) +
                         (size_t)a.nx * ((size_t)((a.lo[1] + j) & (a.ny - 1)) + (size_t)a.ny * ((a.lo[2] + k) & (a.nz - 1)));
        if (a.face != nullptr && !(a.face[o] & 1)) continue;
        const double cv = a.c[o];
        if (PASS == 0) {
            s += cv;
            cnt += 1.0;
        } else {
            const double dv = cv - mean;
            s += dv * dv;
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

} // namespace dnsred
