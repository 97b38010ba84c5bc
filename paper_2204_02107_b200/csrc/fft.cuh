// fft.cuh -- hand-written fp64 complex FFT passes for the pressure Poisson solve (eq. 9).
//
// The solve works on the real nx*ny*nz array reinterpreted as (nx/2)*ny*nz complex numbers
// (even cell -> re, odd cell -> im).  The operator sum_a delta_a delta_a only couples cells two
// apart, so even and odd x-sublattices are independent real problems and one complex-to-complex
// transform of half length in x solves both.
//
// Every pass is a Stockham autosort FFT held in registers (E elements per thread, radix-8/4/2
// butterflies) with shared-memory exchanges between radix stages.  Thread `tid` of a line always
// owns elements tid + e*T (T = L/E), both on entry and on exit, so the first stage reads global
// memory directly and the last stage writes it directly; the fused z pass keeps the spectrum in
// registers between the forward and the inverse transform.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "tma.cuh"

namespace dnsfft {

typedef double2 c2;

__device__ __forceinline__ c2 cadd(c2 a, c2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ c2 csub(c2 a, c2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ c2 cmul(c2 a, c2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// multiply by -i (forward quarter turn) or +i (inverse)
template <int DIR> __device__ __forceinline__ c2 rot90(c2 a)
{
    return DIR < 0 ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x);
}
// multiply by the table twiddle w = exp(-2 pi i t/L) (forward) or its conjugate (inverse)
template <int DIR> __device__ __forceinline__ c2 twmul(c2 a, c2 w)
{
    return DIR < 0 ? make_double2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x)
                   : make_double2(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y);
}

template <int DIR> __device__ __forceinline__ void dft2(c2 &a, c2 &b)
{
    c2 t = a;
    a = cadd(t, b);
    b = csub(t, b);
}

template <int DIR> __device__ __forceinline__ void dft4(c2 &a0, c2 &a1, c2 &a2, c2 &a3)
{
    c2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = rot90<DIR>(csub(a1, a3));
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    a1 = cadd(t1, t3);
    a3 = csub(t1, t3);
}

template <int DIR> __device__ __forceinline__ void dft8(c2 (&v)[8])
{
    const double h = 0.70710678118654752440;
    // even and odd 4-point transforms
    dft4<DIR>(v[0], v[2], v[4], v[6]);
    dft4<DIR>(v[1], v[3], v[5], v[7]);
    // odd outputs times w8^k, k = 1,2,3:  forward w8 = (1 - i)/sqrt2
    c2 o1 = DIR < 0 ? make_double2((v[3].x + v[3].y) * h, (v[3].y - v[3].x) * h)
                    : make_double2((v[3].x - v[3].y) * h, (v[3].y + v[3].x) * h);
    c2 o2 = rot90<DIR>(v[5]);
    c2 o3 = DIR < 0 ? make_double2((v[7].y - v[7].x) * h, -(v[7].x + v[7].y) * h)
                    : make_double2(-(v[7].x + v[7].y) * h, (v[7].x - v[7].y) * h);
    c2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
    v[0] = cadd(e0, o0);
    v[4] = csub(e0, o0);
    v[1] = cadd(e1, o1);
    v[5] = csub(e1, o1);
    v[2] = cadd(e2, o2);
    v[6] = csub(e2, o2);
    v[3] = cadd(e3, o3);
    v[7] = csub(e3, o3);
}

// 16-point transform as 4 x 4: y[b][c] = sum_a v[4a+b] w4^(ac), times w16^(bc), then X[c+4d] = sum_b y[b][c] w4^(bd).
template <int DIR> __device__ __forceinline__ c2 mul_w16(c2 a, int p) // a * w16^p, w16 = exp(-+2 pi i/16), p compile-time after unrolling
{
    const double c1 = 0.92387953251128675613, s1 = 0.38268343236508977173, h = 0.70710678118654752440;
    double wr, wi; // forward twiddle (cos, -sin)
    switch (p) {
    case 0: return a;
    case 1: wr = c1; wi = -s1; break;
    case 2: wr = h; wi = -h; break;
    case 3: wr = s1; wi = -c1; break;
    case 4: return rot90<DIR>(a);
    case 6: wr = -h; wi = -h; break;
    default: wr = -c1; wi = s1; break; // 9
    }
    return DIR < 0 ? make_double2(a.x * wr - a.y * wi, a.x * wi + a.y * wr) : make_double2(a.x * wr + a.y * wi, a.y * wr - a.x * wi);
}

template <int DIR> __device__ __forceinline__ void dft16(c2 (&v)[16])
{
#pragma unroll
    for (int b = 0; b < 4; ++b) dft4<DIR>(v[b], v[4 + b], v[8 + b], v[12 + b]); // v[4c+b] = y[b][c]
#pragma unroll
    for (int b = 1; b < 4; ++b)
#pragma unroll
        for (int c = 1; c < 4; ++c) v[4 * c + b] = mul_w16<DIR>(v[4 * c + b], b * c);
#pragma unroll
    for (int c = 0; c < 4; ++c) dft4<DIR>(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]); // v[4c+d] = X[c+4d]
    // transpose the 4 x 4 index so that v[k] = X[k]
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int d = c + 1; d < 4; ++d) {
            const c2 t = v[4 * c + d];
            v[4 * c + d] = v[4 * d + c];
            v[4 * d + c] = t;
        }
}

// One Stockham stage of radix R on the E register elements of thread `tid` (element e <-> index
// tid + e*T).  Ns = product of the radices of the earlier stages.  On exit slot q + r*(E/R) holds
// output r of butterfly jj = tid + q*T, whose natural position is oidx = expand(jj) + r*Ns.
template <int L, int E, int R, int NS, int DIR, bool TWPOW, bool TWSMEM = false> __device__ __forceinline__ void stage(c2 (&x)[E], int tid, const c2 *__restrict__ tw)
{
    constexpr int T = L / E;
    constexpr int Q = E / R;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        c2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = x[q + r * Q];
        if constexpr (NS > 1) {
            const int jm = (tid + q * T) & (NS - 1);
            const int kb = jm * (L / (NS * R));
            if constexpr (TWPOW && R > 2) {
                // one table look-up per butterfly, the other twiddles as its powers (product depth <= 3):
                // lanes of a warp hold different jm in the x pass, so each look-up is a gather
                c2 w[R];
                w[1] = __ldg(&tw[kb]);
                w[2] = cmul(w[1], w[1]);
                w[3] = cmul(w[2], w[1]);
                if constexpr (R >= 8) {
                    w[4] = cmul(w[2], w[2]);
                    w[5] = cmul(w[4], w[1]);
                    w[6] = cmul(w[4], w[2]);
                    w[7] = cmul(w[4], w[3]);
                }
                if constexpr (R == 16) {
                    w[8] = cmul(w[4], w[4]);
#pragma unroll
                    for (int r = 9; r < 16; ++r) w[r] = cmul(w[8], w[r - 8]);
                }
#pragma unroll
                for (int r = 1; r < R; ++r) v[r] = twmul<DIR>(v[r], w[r]);
            } else {
#pragma unroll
                for (int r = 1; r < R; ++r) v[r] = twmul<DIR>(v[r], TWSMEM ? tw[kb * r] : __ldg(&tw[kb * r]));
            }
        }
        if constexpr (R == 16) {
            dft16<DIR>(v);
        } else if constexpr (R == 8) {
            dft8<DIR>(v);
        } else if constexpr (R == 4) {
            dft4<DIR>(v[0], v[1], v[2], v[3]);
        } else if constexpr (R == 2) {
            dft2<DIR>(v[0], v[1]);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) x[q + r * Q] = v[r];
    }
}

// a view may declare `static constexpr bool TWSMEM = true`: the twiddle table passed to fft_line then lives in shared
// memory and is read with plain loads, one look-up per twiddle (lanes that share a butterfly index broadcast)
template <class SM, class = void> struct tw_in_smem { static constexpr bool value = false; };
template <class SM> struct tw_in_smem<SM, decltype((void)SM::TWSMEM)> { static constexpr bool value = SM::TWSMEM; };

template <int L, int E, int NS> struct NextRadix {
    static constexpr int rem = L / NS;
    static constexpr int cap = E >= 16 ? 16 : (E >= 8 ? 8 : E);
    static constexpr int value = rem >= cap ? cap : rem;
};

// Full transform of one line held as x[e] <-> element tid + e*T, exchanging through `sm`
// (SM::at(n) gives a reference to the shared slot of logical element n of this thread's line).
// All threads that share the view must call this together (sm.sync() is a barrier among them).
// `before_exchange` runs once, after the first radix stage and before anything is written to the exchange area (a caller
// whose exchange area is still being read by someone else waits there).
struct NoHook {
    __device__ __forceinline__ void operator()() const {}
};
template <int L, int E, int DIR, int NS, class SM, class HOOK = NoHook>
__device__ __forceinline__ void fft_line(c2 (&x)[E], int tid, const c2 *__restrict__ tw, SM &sm, HOOK before_exchange = HOOK())
{
    constexpr int T = L / E;
    constexpr int R = NextRadix<L, E, NS>::value;
    constexpr int Q = E / R;
    stage<L, E, R, NS, DIR, SM::TWPOW, tw_in_smem<SM>::value>(x, tid, tw);
    before_exchange();
    if constexpr (NS * R < L) {
#pragma unroll
        for (int q = 0; q < Q; ++q) {
            const int jj = tid + q * T;
            const int jm = jj & (NS - 1);
            const int j0 = (jj - jm) * R + jm;
#pragma unroll
            for (int r = 0; r < R; ++r) sm.at(j0 + r * NS) = x[q + r * Q];
        }
        sm.sync();
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = sm.at(tid + e * T);
        sm.sync();
        fft_line<L, E, DIR, NS * R, SM>(x, tid, tw, sm);
    }
}

// shared-memory views -------------------------------------------------------------------
// contiguous line with one pad element per 8 (x pass: threads of a warp walk along the line)
// The T threads of a line are T consecutive threads: inside one warp for T <= 32 (__syncwarp), else a
// named barrier per line (id 1 + line-in-block, at most 15 lines per block then).
// PSH: one pad element per 2^PSH.  A thread writes runs of R consecutive elements after a radix-R stage, so the lanes
// of a quarter-warp are R elements apart: with R = 16 the pad must come every 16 (stride 17 = 1 mod 8 sixteen-byte
// units, conflict-free); every 8 leaves a two-way conflict there (measured: 23 % of the wavefronts of k_fft_xy).
template <int T, int PSH = 3> struct SmLine {
    static constexpr bool TWPOW = true;
    c2 *base;
    int bar;
    __device__ __forceinline__ c2 &at(int n) { return base[n + (n >> PSH)]; }
    __device__ __forceinline__ void sync()
    {
        if constexpr (T <= 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(T) : "memory");
    }
};
// column of a tile whose fastest index is the XT-wide x offset (y and z passes)
// TWP: twiddles of a butterfly as powers of one look-up (else one look-up each; lanes share them here)
template <int XT, bool TWP = true> struct SmCol {
    static constexpr bool TWPOW = TWP;
    c2 *base; // already offset by tx
    __device__ __forceinline__ c2 &at(int n) { return base[n * XT]; }
    __device__ __forceinline__ void sync() { __syncthreads(); }
};

template <int L> struct ElemsPerThread { static constexpr int value = L >= 8 ? 8 : L; };
// the fused z pass holds 16 elements per thread: one exchange per transform for L <= 256 (radix 16 x 16)
template <int L> struct ElemsPerThreadZ { static constexpr int value = L >= 16 ? 16 : L; };

// ---------------------------------------------------------------------------------------
// Right-hand side of eq. 9 at one cell: r = d + sum_a delta_a[(1-beta) delta_a p].
// face: bit0 beta(cell), bit1/2 beta(x+1/x-1), bit3/4 beta(y+1/y-1), bit5/6 beta(z+1/z-1).
// (1-beta) is 0 in the fluid, so the bracket needs p only next to solid cells.
struct PoissonRhsArgs {
    const double *d;
    const double *p;
    const uint8_t *face; // null: beta == 1 everywhere
    int nx, ny, nz;
    double r2x, r2y, r2z; // 1/(2 D_a)
};

__device__ __forceinline__ double eq9_rhs(const PoissonRhsArgs &a, double dv, int i, int j, int k, unsigned f)
{
    if ((f & 0x7e) == 0x7e) return dv; // all six neighbours fluid: bracket is exactly 0
    const int nx = a.nx, ny = a.ny, nz = a.nz;
    const size_t row = (size_t)nx * ((size_t)j + (size_t)ny * k);
    const double *p = a.p;
    const double pc = __ldg(&p[row + i]);
    double gxp = 0.0, gxm = 0.0, gyp = 0.0, gym = 0.0, gzp = 0.0, gzm = 0.0;
    if (!(f & 2)) gxp = (__ldg(&p[row + ((i + 2) & (nx - 1))]) - pc) * a.r2x;
    if (!(f & 4)) gxm = (pc - __ldg(&p[row + ((i - 2) & (nx - 1))])) * a.r2x;
    if (!(f & 8)) gyp = (__ldg(&p[(size_t)nx * ((size_t)((j + 2) & (ny - 1)) + (size_t)ny * k) + i]) - pc) * a.r2y;
    if (!(f & 16)) gym = (pc - __ldg(&p[(size_t)nx * ((size_t)((j - 2) & (ny - 1)) + (size_t)ny * k) + i])) * a.r2y;
    if (!(f & 32)) gzp = (__ldg(&p[(size_t)nx * ((size_t)j + (size_t)ny * ((k + 2) & (nz - 1))) + i]) - pc) * a.r2z;
    if (!(f & 64)) gzm = (pc - __ldg(&p[(size_t)nx * ((size_t)j + (size_t)ny * ((k - 2) & (nz - 1))) + i])) * a.r2z;
    return dv + ((gxp - gxm) * a.r2x + (gyp - gym) * a.r2y + (gzp - gzm) * a.r2z);
}

// ---------------------------------------------------------------------------------------
// The fused z pass is persistent: a block walks tiles blockIdx.x, blockIdx.x + gridDim.x, ... and keeps the
// NEXT tile in flight (cp.async, 16 bytes per complex element, into the other of two shared-memory
// buffers) while it transforms the current one.  Every thread copies exactly the elements it will hold
// in registers, so reading them back needs only cp.async.wait_group; the buffer then serves as the
// exchange area of the radix stages (one __syncthreads first: other threads' slots are overwritten).
__device__ __forceinline__ void cp_async_c2(c2 *dst_smem, const c2 *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_1() { asm volatile("cp.async.wait_group 1;\n" ::: "memory"); }
// Ask L2 for `bytes` (multiple of 16) starting at the 16-byte aligned global address p; no register, no wait.
// The two-pass kernels hold one tile per SM in shared memory, so a block cannot stage its successor's tile on chip;
// it asks for it in L2 instead, while it computes (the blocks of a grid are handed out in index order).
__device__ __forceinline__ void prefetch_l2(const void *p, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(p), "r"(bytes) : "memory");
}
// x pass: lines of L = nx/2 complex numbers, contiguous.  NL lines per block, one line per T consecutive
// threads, so the exchanges of a line never leave its warp (or its named barrier).
//   FWD with PROLOGUE: in = d (real array viewed as complex), r = eq9_rhs(...) computed on load.
//   out-of-place or in-place (a line is read completely before it is written).
template <int L, int DIR, bool PROLOGUE>
__global__ void __launch_bounds__(256) k_fft_x(const c2 *__restrict__ in, c2 *__restrict__ out, const c2 *__restrict__ tw, int nlines_per_block,
                                               int rev, PoissonRhsArgs ra)
{
    constexpr int E = ElemsPerThreadZ<L>::value;
    constexpr int T = L / E;
    extern __shared__ double2 smem[];
    const int lt = threadIdx.x / T; // line within block
    const int tid = threadIdx.x - lt * T;
    // rev: walk the lines from the far end, so that a pass starts on what the pass before it left in L2
    const size_t line = (size_t)(rev ? gridDim.x - 1 - blockIdx.x : blockIdx.x) * nlines_per_block + lt;
    const c2 *src = in + line * L;
    c2 x[E];
#pragma unroll
    for (int e = 0; e < E; ++e) x[e] = src[tid + e * T];
    if (PROLOGUE) {
        if (ra.face != nullptr) {
            const int j = (int)(line % ra.ny), k = (int)(line / ra.ny);
            const uint8_t *frow = ra.face + line * (size_t)(2 * L);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int m = tid + e * T;
                const uchar2 f = *reinterpret_cast<const uchar2 *>(frow + 2 * m);
                x[e].x = eq9_rhs(ra, x[e].x, 2 * m, j, k, f.x);
                x[e].y = eq9_rhs(ra, x[e].y, 2 * m + 1, j, k, f.y);
            }
        }
    }
    SmLine<T> sm{smem + lt * (L + L / 8), 1 + lt};
    fft_line<L, E, DIR, 1, SmLine<T>>(x, tid, tw, sm);
    c2 *dst = out + line * L;
#pragma unroll
    for (int e = 0; e < E; ++e) dst[tid + e * T] = x[e];
}

// y or z pass, in place: XT adjacent x (complex) by L elements along the axis; element n of
// column tx is at base + n*stride + tx.  blockIdx.x enumerates (x tile, other index).
template <int L, int XT, int DIR>
__global__ void __launch_bounds__(XT *(L / ElemsPerThreadZ<L>::value) < 32 ? 32 : XT *(L / ElemsPerThreadZ<L>::value))
    k_fft_col(c2 *__restrict__ data, const c2 *__restrict__ tw, int mx, size_t stride, size_t other_stride, int rev)
{
    constexpr int E = ElemsPerThreadZ<L>::value;
    constexpr int T = L / E;
    extern __shared__ double2 smem[];
    const int tx = threadIdx.x % XT;
    const int tid = threadIdx.x / XT;
    const int xtiles = mx / XT;
    const unsigned bid = rev ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
    const int xt = bid % xtiles;
    const size_t other = bid / xtiles;
    c2 *base = data + other * other_stride + (size_t)xt * XT + tx;
    c2 x[E];
#pragma unroll
    for (int e = 0; e < E; ++e) x[e] = base[(size_t)(tid + e * T) * stride];
    SmCol<XT> sm{smem + tx};
    fft_line<L, E, DIR, 1, SmCol<XT>>(x, tid, tw, sm);
#pragma unroll
    for (int e = 0; e < E; ++e) base[(size_t)(tid + e * T) * stride] = x[e];
}

// 1/a for finite, normal a != 0: hardware seed (rcp.approx, 20 bits) and two Newton steps -- about an ulp, no special
// cases, a third of the instructions of a correctly rounded reciprocal.  lambda is bounded away from 0 and from
// overflow on every non-null mode; null modes are replaced by 0 by the caller.
__device__ __forceinline__ double rcp_newton(double a)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
    r = fma(r, fma(-a, r, 1.0), r);
    r = fma(r, fma(-a, r, 1.0), r);
    return r;
}

// Fused middle pass along z: forward transform, division by the modified-wavenumber eigenvalue
//   lambda(m,ky,kz) = -(ex[m] + ey[ky] + ez[kz]),  e_a[k] = (sin(2 pi k/N_a)/D_a)^2,
// null modes (m = 0, 2ky = 0 mod ny, 2kz = 0 mod nz) set to 0, scaling by 1/N, inverse transform.
// The tile index enumerates (x tile, ky).
template <int L, int XT>
__global__ void __launch_bounds__(XT *(L / ElemsPerThreadZ<L>::value) < 32 ? 32 : XT *(L / ElemsPerThreadZ<L>::value))
    k_fft_z_solve(c2 *__restrict__ data, const c2 *__restrict__ tw, int mx, int ny, const double *__restrict__ ex,
                  const double *__restrict__ ey, const double *__restrict__ ez, double inv_n, int ntiles, int rev)
{
    constexpr int E = ElemsPerThreadZ<L>::value;
    constexpr int T = L / E;
    extern __shared__ double2 smem[];
    const int tx = threadIdx.x % XT;
    const int tid = threadIdx.x / XT;
    const int xtiles = mx / XT;
    const size_t stride = (size_t)mx * ny;
    auto issue = [&](int t_, int b) {
        const int tile = rev ? ntiles - 1 - t_ : t_;
        const c2 *src = data + (size_t)(tile / xtiles) * mx + (tile % xtiles) * XT + tx;
        c2 *dst = smem + b * (XT * L) + tx;
#pragma unroll
        for (int e = 0; e < E; ++e) cp_async_c2(&dst[(tid + e * T) * XT], &src[(size_t)(tid + e * T) * stride]);
    };
    double ezr[E]; // 1/N scaling folded in later; ez depends only on this thread's kz
#pragma unroll
    for (int e = 0; e < E; ++e) ezr[e] = __ldg(&ez[tid + e * T]);
    int lt_ = blockIdx.x, b = 0; // logical tile; the physical one counts from the far end when rev
    if (lt_ < ntiles) issue(lt_, 0);
    cp_async_commit();
    for (; lt_ < ntiles; lt_ += gridDim.x, b ^= 1) {
        if (lt_ + (int)gridDim.x < ntiles) issue(lt_ + gridDim.x, b ^ 1);
        cp_async_commit();
        cp_async_wait_1();
        const int tile = rev ? ntiles - 1 - lt_ : lt_;
        const int ky = tile / xtiles, m = (tile % xtiles) * XT + tx;
        SmCol<XT> sm{smem + b * (XT * L) + tx};
        c2 x[E];
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = sm.at(tid + e * T);
        __syncthreads();
        fft_line<L, E, -1, 1, SmCol<XT>>(x, tid, tw, sm);
        const double exy = __ldg(&ex[m]) + __ldg(&ey[ky]);
        const bool null_xy = (m == 0) && (((2 * ky) & (ny - 1)) == 0);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int kz = tid + e * T;
            const double lam = -(exy + ezr[e]);
            const bool null = null_xy && (((2 * kz) & (L - 1)) == 0);
            const double s = inv_n * rcp_newton(lam);
            x[e].x = null ? 0.0 : x[e].x * s;
            x[e].y = null ? 0.0 : x[e].y * s;
        }
        __syncthreads();
        fft_line<L, E, +1, 1, SmCol<XT>>(x, tid, tw, sm);
        c2 *base = data + (size_t)ky * mx + m;
#pragma unroll
        for (int e = 0; e < E; ++e) base[(size_t)(tid + e * T) * stride] = x[e];
    }
}

// ---------------------------------------------------------------------------------------
// Two-pass transform (3 HBM round trips per solve instead of 5).  The y transform is split by Cooley-Tukey,
// y = y0 + NY0 y1, ky = ky1 + NY1 ky0 (NY0 NY1 = ny):
//     Y[ky1 + NY1 ky0] = sum_y0 w_NY0^(y0 ky0) { w_ny^(y0 ky1) [ sum_y1 f[y0 + NY0 y1] w_NY1^(y1 ky1) ] } .
// k_fft_xy does x and the inner sum (over y1) plus the twiddle on a tile of NY1 whole rows y0 + NY0 y1 (each row is
// LX contiguous complex numbers) and leaves ky1 where y1 was; k_fft_yz_solve does the outer sum (over y0: NY0
// adjacent rows), z, the division by lambda(kx, ky1 + NY1 ky0, kz), and the way back.  Frequencies stay in this
// digit-reversed place between the passes; nothing is reordered in memory.  Inverse: the same steps backwards.
//
// k_fft_xy: one block per (y0, z); LX NY1 / 16 threads, 16 elements each; the tile lives in shared memory
// (row stride LX + LX/16) between the row phase (x transform, T = LX/16 consecutive threads per row, exchanges
// inside the row's warp) and the column phase (length-NY1 transform, lanes of a warp on adjacent columns).
template <int RS> struct SmTileCol {
    static constexpr bool TWPOW = true;
    c2 *base; // already offset to this thread's column
    __device__ __forceinline__ c2 &at(int n) { return base[n * RS]; }
    __device__ __forceinline__ void sync() { __syncthreads(); }
};

template <int LX, int NY1, int DIR>
__global__ void __launch_bounds__(LX *NY1 / 16, (LX * NY1 / 16 <= 256 ? 2 : 1)) // three blocks per SM at 80 registers: 58 instead of 52 us
    k_fft_xy(const c2 *__restrict__ in, c2 *__restrict__ out, const c2 *__restrict__ twx, const c2 *__restrict__ twy1, const c2 *__restrict__ twy,
             int ny, int rev, int ahead)
{
    constexpr int E = 16, TX = LX / E, RS = LX + LX / 16, T2 = NY1 / E;
    static_assert(LX >= 64 && NY1 >= 16, "tile too small for 16 elements per thread");
    extern __shared__ double2 smem[];
    const int ny0 = ny / NY1;
    const unsigned bid = rev ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
    const int y0 = bid % ny0;
    const size_t z = bid / ny0;
    const size_t tile0 = (z * ny + y0) * LX, rstride = (size_t)ny0 * LX; // row r of the tile starts at tile0 + r rstride
    const int t = threadIdx.x;
    const int r = t / TX, tid = t - r * TX;      // row phase
    const int tid2 = t / LX, kx = t - tid2 * LX; // column phase
    SmLine<TX, 4> sl{smem + r * RS, 1 + r};
    SmTileCol<RS> sc{smem + kx + (kx >> 4)};
    c2 x[E];
    // One block per tile (a persistent block walking several tiles measured slower here: 58 against 52 us per pass on
    // 512x256x128).  While it computes, the block asks L2 for the tile of the block `ahead` places behind it in launch
    // order -- the one that will take over an SM about when this one retires -- one row per thread.
    auto prefetch_next = [&]() {
        const unsigned nb = blockIdx.x + ahead;
        if (ahead > 0 && nb < gridDim.x && t < NY1) {
            const unsigned nbid = rev ? gridDim.x - 1 - nb : nb;
            prefetch_l2(in + ((size_t)(nbid / ny0) * ny + nbid % ny0) * LX + t * rstride, LX * sizeof(c2));
        }
    };
    if (DIR < 0) {
        const c2 *row = in + tile0 + r * rstride;
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = row[tid + e * TX];
        prefetch_next();
        fft_line<LX, E, -1, 1, SmLine<TX, 4>>(x, tid, twx, sl);
#pragma unroll
        for (int e = 0; e < E; ++e) sl.at(tid + e * TX) = x[e];
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = sc.at(tid2 + e * T2);
        if (T2 > 1) __syncthreads(); // the exchanges of the column transform overwrite what its other threads read
        fft_line<NY1, E, -1, 1, SmTileCol<RS>>(x, tid2, twy1, sc);
        c2 *dst = out + tile0 + kx;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int ky1 = tid2 + e * T2;
            dst[ky1 * rstride] = twmul<-1>(x[e], __ldg(&twy[(y0 * ky1) & (ny - 1)]));
        }
    } else {
        const c2 *src = in + tile0 + kx;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int ky1 = tid2 + e * T2;
            x[e] = twmul<+1>(src[ky1 * rstride], __ldg(&twy[(y0 * ky1) & (ny - 1)]));
        }
        prefetch_next();
        fft_line<NY1, E, +1, 1, SmTileCol<RS>>(x, tid2, twy1, sc);
#pragma unroll
        for (int e = 0; e < E; ++e) sc.at(tid2 + e * T2) = x[e];
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = sl.at(tid + e * TX);
        sl.sync();
        fft_line<LX, E, +1, 1, SmLine<TX, 4>>(x, tid, twx, sl);
        c2 *row = out + tile0 + r * rstride;
#pragma unroll
        for (int e = 0; e < E; ++e) row[tid + e * TX] = x[e];
    }
}

// k_fft_yz_solve: the middle pass.  A tile is the NY0 LZ XT values (kx, y0, z) of the rows ky1 NY0 + y0 for XT adjacent kx
// (XT = 2 on 512x256x128: 4096 points, 64 KB); the complex array is a rank-3 tensor (2 mx doubles, ny, nz) and one TMA box
// (2 XT, NY0, LZ) is the whole tile, landing dense as [z][y0][xl] and leaving the same way: no load or store instruction
// touches global memory and no register waits on one, so 32-byte runs cost the LSU nothing.  A dense tile is
// conflict-free for threads that hold a z line (lanes on adjacent (xl, y0)), so z is transformed FIRST, straight out of
// the landing buffer; the tile is then exchanged through a padded layout [z][y0][xl] (+XT per z) to threads that hold all
// NY0 values of 16/NY0 planes: y0 transform, multiplication by inv_n / lambda, and everything backwards.
// The block is persistent and works as two groups of NT threads.  Each group transforms its own tile stream (tiles
// n = 0, 1, 2, ... of the block alternate between the groups) in its own work buffer; one landing buffer is shared: as soon
// as a group has taken its tile out of it into registers, the box of the OTHER group's next tile is requested, so a load
// is always in flight while both groups compute, and the store of a finished tile drains while its group works on the
// first radix stage of the next one.  Group-wide named barriers only; one mbarrier per group for its loads.
template <int N, int DIR> __device__ __forceinline__ void dft_small(c2 *v)
{
    if constexpr (N == 2) {
        dft2<DIR>(v[0], v[1]);
    } else if constexpr (N == 4) {
        dft4<DIR>(v[0], v[1], v[2], v[3]);
    } else if constexpr (N == 8) {
        dft8<DIR>(*reinterpret_cast<c2(*)[8]>(v));
    } else {
        dft16<DIR>(*reinterpret_cast<c2(*)[16]>(v));
    }
}

// Plane stride of the padded layout, in complex numbers: NY0 XT plus XT when XT < 8, so that the quarter-warps of both
// layouts hit 32 different banks -- unless the padded buffers would not fit the SM (long z, few rows: the pad is then
// half of a plane), where the y0 phase lives with two-way conflicts instead.
template <int NY0, int LZ, int XT> struct YzLayout {
    static constexpr int DROW = NY0 * XT;
    static constexpr int padded = DROW + (NY0 > 1 && XT < 8 ? XT : 0); // NY0 == 1: the padded layout is not used
    static constexpr size_t bytes_with(int zrow) { return ((size_t)LZ * DROW + 2 * (size_t)((LZ * zrow + 7) / 8 * 8) + LZ) * sizeof(c2) + LZ * sizeof(double); }
    static constexpr int ZROW = bytes_with(padded) <= 227 * 1024 ? padded : DROW;
    static constexpr int WBUF = (LZ * ZROW + 7) / 8 * 8; // work buffer of a group, in complex numbers (a multiple of 128 bytes)
    static constexpr size_t SMEM = bytes_with(ZROW);     // landing buffer, two work buffers, z twiddles, z eigenvalue parts
};

template <int STRIDE> struct SmStrideBar {
    static constexpr bool TWPOW = false, TWSMEM = true; // all lanes of a warp share a z butterfly: table look-ups broadcast
    c2 *base;
    int bar, nthreads;
    __device__ __forceinline__ c2 &at(int n) { return base[n * STRIDE]; }
    __device__ __forceinline__ void sync() { asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(nthreads) : "memory"); }
};

template <int NY0, int LZ, int XT>
__global__ void __launch_bounds__(2 * XT * NY0 * LZ / 16, 1)
    k_fft_yz_solve(const __grid_constant__ CUtensorMap map, const c2 *__restrict__ twz, int mx, int ny, const double *__restrict__ ex,
                       const double *__restrict__ ey, const double *__restrict__ ez, double inv_n, int rev, int ntiles)
{
    using namespace dnstma;
    constexpr int E = 16, G = E / NY0, ZQ = LZ / G, T = LZ / E, NT = XT * NY0 * LZ / E;
    constexpr int DROW = NY0 * XT, ZROW = YzLayout<NY0, LZ, XT>::ZROW, WBUF = YzLayout<NY0, LZ, XT>::WBUF, ZB = LZ > 256 ? 256 : LZ;
    static_assert(NY0 >= 1 && NY0 <= 16 && LZ >= 32, "unsupported split");
    extern __shared__ __align__(128) double2 smem[];
    __shared__ __align__(8) uint64_t full[2];
    c2 *land = smem;                                    // dense landing buffer [z][y0][xl]
    c2 *stw = smem + LZ * DROW + 2 * WBUF;              // z twiddles
    double *sez = reinterpret_cast<double *>(stw + LZ); // z eigenvalue parts
    const int ny1 = ny / NY0, xtiles = mx / XT;
    const int grp = threadIdx.x / NT, t = threadIdx.x - grp * NT;
    c2 *work = smem + LZ * DROW + grp * WBUF;
    const int xl = t % XT, rest = t / XT;
    const int y0 = rest % NY0, tid = rest / NY0, zq = rest;
    auto tile_of = [&](int n) { // the block's n-th tile, or -1
        const long q = (long)blockIdx.x + (long)n * gridDim.x;
        return q < ntiles ? (int)(rev ? ntiles - 1 - q : q) : -1;
    };
    auto request = [&](int n) { // thread-level: ask for the box of the block's n-th tile (if any) into the landing buffer
        const int tl = tile_of(n);
        if (tl < 0) return;
        uint64_t *bar = &full[n & 1];
        mbar_arrive_expect_tx(bar, (unsigned)(LZ * DROW * sizeof(c2)));
#pragma unroll
        for (int z0 = 0; z0 < LZ; z0 += ZB) tma_load_3d(land + z0 * DROW, &map, bar, 2 * (tl % xtiles) * XT, (tl / xtiles) * NY0, z0);
    };
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        mbar_fence_init();
        request(0);
    }
    for (int q = threadIdx.x; q < LZ; q += 2 * NT) {
        sez[q] = ez[q];
        stw[q] = twz[q];
    }
    __syncthreads();
    SmStrideBar<DROW> sl{land + y0 * XT + xl, 1 + grp, NT};
    SmStrideBar<DROW> sd{work + y0 * XT + xl, 1 + grp, NT};
    for (int n = grp; tile_of(n) >= 0; n += 2) {
        const int tl = tile_of(n), xt = tl % xtiles, ky1 = tl / xtiles;
        mbar_wait(&full[grp], (n >> 1) & 1);
        c2 x[E];
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = sl.at(tid + e * T);
        sd.sync(); // the landing buffer is consumed
        if (t == 0) request(n + 1);
        fft_line<LZ, E, -1, 1, SmStrideBar<DROW>>(x, tid, stw, sd, [&]() {
            if (t == 0) tma_store_wait_read(); // the store of this group's previous tile has read the work buffer
            sd.sync();
        });
        if constexpr (NY0 > 1) {
#pragma unroll
            for (int e = 0; e < E; ++e) work[(tid + e * T) * ZROW + y0 * XT + xl] = x[e];
            sd.sync();
#pragma unroll
            for (int g = 0; g < G; ++g)
#pragma unroll
                for (int q = 0; q < NY0; ++q) x[g * NY0 + q] = work[(zq + g * ZQ) * ZROW + q * XT + xl];
#pragma unroll
            for (int g = 0; g < G; ++g) dft_small<NY0, -1>(x + g * NY0);
            {
                const int m = xt * XT + xl;
                const double exm = __ldg(&ex[m]);
#pragma unroll
                for (int g = 0; g < G; ++g) {
                    const int kz = zq + g * ZQ;
                    const double exz = exm + sez[kz];
                    const bool null_xz = (m == 0) && (((2 * kz) & (LZ - 1)) == 0);
#pragma unroll
                    for (int q = 0; q < NY0; ++q) {
                        const int ky = ky1 + ny1 * q;
                        const double lam = -(exz + __ldg(&ey[ky]));
                        const bool null = null_xz && (((2 * ky) & (ny - 1)) == 0);
                        const double sc = inv_n * rcp_newton(lam);
                        x[g * NY0 + q].x = null ? 0.0 : x[g * NY0 + q].x * sc;
                        x[g * NY0 + q].y = null ? 0.0 : x[g * NY0 + q].y * sc;
                    }
                }
            }
#pragma unroll
            for (int g = 0; g < G; ++g) dft_small<NY0, +1>(x + g * NY0);
#pragma unroll
            for (int g = 0; g < G; ++g)
#pragma unroll
                for (int q = 0; q < NY0; ++q) work[(zq + g * ZQ) * ZROW + q * XT + xl] = x[g * NY0 + q];
            sd.sync();
#pragma unroll
            for (int e = 0; e < E; ++e) x[e] = work[(tid + e * T) * ZROW + y0 * XT + xl];
            sd.sync();
        } else {
            // no split of y (ny0 == 1, and the z pass of the five single-axis passes): the spectrum is complete in the z layout
            const int m = xt * XT + xl;
            const double exy = __ldg(&ex[m]) + __ldg(&ey[ky1]);
            const bool null_xy = (m == 0) && (((2 * ky1) & (ny - 1)) == 0);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int kz = tid + e * T;
                const double lam = -(exy + sez[kz]);
                const bool null = null_xy && (((2 * kz) & (LZ - 1)) == 0);
                const double sc = inv_n * rcp_newton(lam);
                x[e].x = null ? 0.0 : x[e].x * sc;
                x[e].y = null ? 0.0 : x[e].y * sc;
            }
        }
        fft_line<LZ, E, +1, 1, SmStrideBar<DROW>>(x, tid, stw, sd);
#pragma unroll
        for (int e = 0; e < E; ++e) sd.at(tid + e * T) = x[e];
        fence_proxy_async();
        sd.sync();
        if (t == 0) {
#pragma unroll
            for (int z0 = 0; z0 < LZ; z0 += ZB) tma_store_3d(&map, work + z0 * DROW, 2 * xt * XT, ky1 * NY0, z0);
            tma_store_commit();
        }
    }
    if (t == 0) tma_store_wait_read();
}


// ---------------------------------------------------------------------------------------
// Real-to-complex entry points (dnslab_rfft3 / dnslab_irfft3): the transform itself, apart from the solve.
// The packed array z[i'] = x[2i'] + i x[2i'+1] (M = nx/2 complex numbers per row) has the transform Z = E + iO,
// E and O the transforms of the even and odd real sub-sequences; with Hermitian symmetry of both,
//   E[m] = (Z[m] + conj Z[-m])/2,  O[m] = (Z[m] - conj Z[-m])/(2i)   (-m: all three indices negated, modulo M, ny, nz)
// and the real-to-complex result is X[m] = E[m] + exp(-2 pi i m/nx) O[m] for m = 0..M (M+1 numbers per row).
// inverse = false: Z (M per row) -> X (M+1 per row).  inverse = true: X -> scale * Z, ready for the inverse passes.
__global__ void __launch_bounds__(256) k_r2c_tangle(const c2 *__restrict__ in, c2 *__restrict__ out, int M, int ny, int nz, int inverse,
                                                    double scale)
{
    const int mcount = inverse ? M : M + 1;
    const size_t total = (size_t)mcount * ny * nz, q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= total) return;
    const int m = (int)(q % mcount), ky = (int)((q / mcount) % ny), kz = (int)(q / ((size_t)mcount * ny));
    const int nky = (ny - ky) & (ny - 1), nkz = (nz - kz) & (nz - 1);
    double sn, cs;
    sincospi(-(double)m / (double)M, &sn, &cs); // w = exp(-i pi m/M) = exp(-2 pi i m/nx)
    if (!inverse) {
        const c2 a = in[(size_t)(m & (M - 1)) + (size_t)M * (ky + (size_t)ny * kz)];
        c2 b = in[(size_t)((M - m) & (M - 1)) + (size_t)M * (nky + (size_t)ny * nkz)];
        b.y = -b.y;
        const c2 E = make_double2(0.5 * (a.x + b.x), 0.5 * (a.y + b.y));
        const c2 O = make_double2(0.5 * (a.y - b.y), -0.5 * (a.x - b.x)); // (a - b)/(2i)
        out[q] = make_double2(E.x + (cs * O.x - sn * O.y), E.y + (cs * O.y + sn * O.x));
    } else {
        const int R = M + 1;
        const c2 a = in[(size_t)m + (size_t)R * (ky + (size_t)ny * kz)];
        c2 b = in[(size_t)(M - m) + (size_t)R * (nky + (size_t)ny * nkz)];
        b.y = -b.y;
        const c2 E = make_double2(0.5 * (a.x + b.x), 0.5 * (a.y + b.y));
        const c2 D = make_double2(0.5 * (a.x - b.x), 0.5 * (a.y - b.y));
        const c2 O = make_double2(D.x * cs + D.y * sn, D.y * cs - D.x * sn); // D conj(w), conj(w) = cs - i sn
        out[q] = make_double2(scale * (E.x - O.y), scale * (E.y + O.x));     // scale (E + i O)
    }
}

} // namespace dnsfft
