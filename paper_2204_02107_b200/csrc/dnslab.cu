// dnslab.cu -- host side of libdnslab.so (C ABI in include/dnslab.h): workspace carving, table
// set-up, launch sequence of one DNSLABIB time step.  No device allocation, no host sync in step.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/dnslab.h"
#include "fft.cuh"
#include "particles.cuh"
#include "reduce.cuh"
#include "stencil.cuh"

using dnsfft::c2;

namespace {

constexpr size_t ALIGN = 256;
// Tile traversal direction, one bit per kernel (set: walk from the far end, i.e. start on what the kernel before left
// in the 126 MB L2).  Measured sweeps on 512x256x128: the y passes gain from walking against the x passes
// (41.7 instead of 45 us each); of the stencil kernels only the divergence gains (83 instead of 88 us).
constexpr int FFT_REV = 10; // bits: x fwd, y fwd, z, y inv, x inv
constexpr int ST_REV = 16;  // bits: RK stages 1-4, divergence, projection
inline size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }
inline bool pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

bool valid_params(const dnslab_params_t *P)
{
    if (!P) return false;
    if (!pow2(P->nx) || !pow2(P->ny) || !pow2(P->nz)) return false;
    if (P->nx < 8 || P->nx > 2048 || P->ny < 8 || P->ny > 1024 || P->nz < 8 || P->nz > 1024) return false;
    if (!(P->dx > 0) || !(P->dy > 0) || !(P->dz > 0) || !(P->dt > 0)) return false;
    if (!(P->nu >= 0) || !(P->alpha_c >= 0) || P->n_piter < 1) return false;
    if (P->flags & ~3u) return false;
    return true;
}

struct Layout {
    size_t field_bytes, off_fields, nfields, off_face, off_tw[3], off_twy1, off_eig, off_stab, off_blist, off_bsave, bcap, total;
};

// 19 fields: Q(4) A(4) B(4) Qc(4) p d W (+1 scratch pressure with per-stage projection)
Layout make_layout(const dnslab_params_t *P)
{
    Layout L;
    const size_t n = (size_t)P->nx * P->ny * P->nz;
    L.field_bytes = align_up(n * sizeof(double));
    L.nfields = 19 + ((P->flags & 2u) ? 1 : 0);
    size_t off = 0;
    L.off_fields = off;
    off += L.nfields * L.field_bytes;
    L.off_face = off;
    off += align_up(n);
    const int len[3] = {P->nx / 2, P->ny, P->nz};
    for (int a = 0; a < 3; ++a) {
        L.off_tw[a] = off;
        off += align_up((size_t)len[a] * sizeof(c2));
    }
    L.off_twy1 = off; // twiddles of the inner y transform of the two-pass solve (at most 128 entries)
    off += align_up(128 * sizeof(c2));
    L.off_eig = off;
    off += align_up((size_t)(P->nx / 2 + P->ny + P->nz) * sizeof(double));
    L.off_stab = off;
    off += align_up((size_t)DNSLAB_MAX_SOURCES * (P->nx + P->ny + P->nz) * sizeof(double));
    // eq. 9 boundary list (cells with a solid face neighbour) and the compact copy of d there; masks whose
    // list would be longer than N/2 use the dense prologue of the forward x pass instead
    L.bcap = n / 2;
    L.off_blist = off;
    off += align_up(L.bcap * sizeof(uint64_t));
    L.off_bsave = off;
    off += align_up(L.bcap * sizeof(double));
    L.total = off;
    return L;
}

// eq. 5 one-dimensional factor; reading R10
void source_profile(int n, double d, int lo, int size, double B, double *out)
{
    for (int i = 0; i < n; ++i) {
        if (!(B > 0.0)) {
            const int rel = (((i - lo) % n) + n) % n;
            out[i] = rel < size ? 1.0 : 0.0;
            continue;
        }
        const double len = n * d, centre = (lo + 0.5 * (size - 1)) * d, halfw = 0.5 * size * d;
        double r = std::fmod(std::fabs(i * d - centre), len);
        if (r > 0.5 * len) r = len - r;
        out[i] = (r == 0.0) ? 1.0 : 0.5 * (1.0 - std::tanh(B * (r / halfw - halfw / r)));
    }
}

} // namespace

struct ProfRec {
    int cls;
    cudaEvent_t e0, e1;
};

struct dnslab {
    dnslab_params_t P;
    size_t n;
    cudaStream_t stream;
    char *ws;
    Layout L;
    double *Q[4], *A[4], *Bf[4], *Qc[4], *p, *d, *W, *ps;
    uint8_t *face; // null when the mask has no solid cell
    unsigned long long *blist; // eq. 9 boundary records (index | face << 32); null: dense prologue in the forward x pass
    double *bsave;
    int nb;
    c2 *tw[3];
    c2 *twy1;  // exp(-2 pi i t/NY1), the inner y transform of the two-pass solve
    int f_ny1; // two-pass solve (k_fft_xy + k_fft_yz_solve): rows per xy tile, 0 = five single-axis passes instead
    double *eig[3];
    double *stab;
    int nsrc;
    dnsst::SourceDev src[DNSLAB_MAX_SOURCES];
    int64_t launches;
    dim3 rk_block;
    int nsm;   // SM count of the device
    bool prepare; // set while dnslab_create walks the launchers once: they configure their kernel and do not launch
    unsigned zgrid; // grid of the persistent fused middle pass (occupancy query done once, at create)
    int xy_ahead; // two-pass solve, xy passes: how many blocks ahead a block prefetches into L2 (blocks resident on the chip)
    int rk_kc; // > 0: z-marching RK kernel with this many planes per block; 0: brick kernel (small grids)
    bool tma_ok; // tensor maps of the 16 RK field buffers are built (k_rk_march loads interior tiles by TMA)
    CUtensorMap tmap[16];
    void *tma_encode; // cuTensorMapEncodeTiled, fetched through cudaGetDriverEntryPoint at create (null: no TMA anywhere)
    bool wmap_ok;     // the tensor map of the transform array W is built (the middle pass of the two-pass solve moves its tiles by TMA)
    CUtensorMap wmap;
    bool wmapz_ok;    // the same for the fused z pass without a split of y (box 2 XT x 1 x nz)
    CUtensorMap wmapz;
    long long np;      // NEXT-4: attached particles (0: none); state is the caller's device array
    double *pstate, prho_f, pgrav[3];
    // optional per-launch timing (dnslab_profile): events bracketing every kernel, by class
    bool prof_on;
    std::vector<ProfRec> *prof;
    double prof_ms[DNSLAB_NCLASS];
    int64_t prof_n[DNSLAB_NCLASS];
};

namespace {

#define CK(call)                                   \
    do {                                           \
        cudaError_t e_ = (call);                   \
        if (e_ != cudaSuccess) return DNSLAB_ECUDA; \
    } while (0)

// Accumulate finished event pairs into the per-class totals (synchronises the stream).
int prof_drain(dnslab *h)
{
    if (!h->prof || h->prof->empty()) return DNSLAB_OK;
    CK(cudaStreamSynchronize(h->stream));
    for (ProfRec &r : *h->prof) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, r.e0, r.e1));
        h->prof_ms[r.cls] += ms;
        h->prof_n[r.cls] += 1;
        cudaEventDestroy(r.e0);
        cudaEventDestroy(r.e1);
    }
    h->prof->clear();
    return DNSLAB_OK;
}

// Brackets one kernel launch with events when profiling is on.
struct ProfScope {
    dnslab *h;
    ProfRec r;
    bool on;
    ProfScope(dnslab *h_, int cls) : h(h_), on(h_->prof_on)
    {
        if (!on) return;
        r.cls = cls;
        cudaEventCreate(&r.e0);
        cudaEventCreate(&r.e1);
        cudaEventRecord(r.e0, h->stream);
    }
    ~ProfScope()
    {
        if (!on) return;
        cudaEventRecord(r.e1, h->stream);
        h->prof->push_back(r);
        if (h->prof->size() >= 8192) prof_drain(h);
    }
};

inline int check_launch(dnslab *h)
{
    h->launches++;
    return cudaPeekAtLastError() == cudaSuccess ? DNSLAB_OK : DNSLAB_ECUDA;
}

dim3 tile_block(const dnslab *h)
{
    const int bx = h->P.nx < 32 ? h->P.nx : 32;
    int by = 256 / bx;
    if (by > h->P.ny) by = h->P.ny;
    return dim3(bx, by, 1);
}

// One rank-3 fp64 tensor map (x fastest) through the driver entry point fetched at create; false when it is unavailable.
bool encode_map3(dnslab *h, CUtensorMap *map, void *base, const cuuint64_t (&gdim)[3], const cuuint32_t (&box)[3],
                 CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_128B)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    if (!h->tma_encode) return false;
    const cuuint64_t gstr[2] = {gdim[0] * sizeof(double), gdim[0] * gdim[1] * sizeof(double)};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    return ((encode_fn)h->tma_encode)(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                      CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// ---- RK stage ---------------------------------------------------------------------------
// qs: stage field (stencil input); qo: next stage field; elim: Qc eliminated
template <int STAGE, bool ELIM> int launch_rk(dnslab *h, double *const *qs, double *const *qo, double *const *q2)
{
    static const double ca[4] = {0.5, 0.5, 1.0, 0.0};
    static const double cb[4] = {1.0 / 6.0, 1.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0};
    dnsst::RKArgs a;
    std::memset(&a, 0, sizeof(a));
    for (int m = 0; m < 4; ++m) {
        a.qs[m] = qs[m];
        a.qn[m] = h->Q[m];
        a.qc[m] = ELIM ? (q2 ? q2[m] : nullptr) : h->Qc[m];
        a.qo[m] = qo ? qo[m] : nullptr;
        a.qco[m] = ELIM ? (q2 ? q2[m] : nullptr) : h->Qc[m];
    }
    a.face = h->face;
    a.nx = h->P.nx; a.ny = h->P.ny; a.nz = h->P.nz;
    a.r2x = 1.0 / (2.0 * h->P.dx); a.r2y = 1.0 / (2.0 * h->P.dy); a.r2z = 1.0 / (2.0 * h->P.dz);
    a.rxx = 1.0 / (h->P.dx * h->P.dx); a.ryy = 1.0 / (h->P.dy * h->P.dy); a.rzz = 1.0 / (h->P.dz * h->P.dz);
    a.nu = h->P.nu; a.ac = h->P.alpha_c;
    for (int m = 0; m < 3; ++m) a.body[m] = h->P.body[m];
    a.kf.hx = -0.5 * a.r2x; a.kf.hy = -0.5 * a.r2y; a.kf.hz = -0.5 * a.r2z;
    a.kf.dvx = a.nu * a.rxx; a.kf.dvy = a.nu * a.ryy; a.kf.dvz = a.nu * a.rzz;
    a.kf.dcx = a.ac * a.rxx; a.kf.dcy = a.ac * a.ryy; a.kf.dcz = a.ac * a.rzz;
    a.kf.dv0 = -2.0 * (a.kf.dvx + a.kf.dvy + a.kf.dvz);
    a.kf.dc0 = -2.0 * (a.kf.dcx + a.kf.dcy + a.kf.dcz);
    a.ca = ca[STAGE - 1] * h->P.dt;
    a.cb = cb[STAGE - 1] * h->P.dt;
    a.nsrc = h->nsrc;
    a.stab = h->stab;
    for (int s = 0; s < h->nsrc; ++s) a.src[s] = h->src[s];
    const bool masked = h->face != nullptr, sources = h->nsrc > 0;
    if (h->rk_kc > 0) {
        // z-marching kernel: 64 x 8 columns, kc planes per block
        a.kc = h->rk_kc;
        a.rev = (ST_REV >> (STAGE - 1)) & 1;
        const dim3 blk(32, dnsst::RKM_TY, 1);
        const dim3 grd(h->P.nx / dnsst::RKM_TX, h->P.ny / dnsst::RKM_TY, h->P.nz / h->rk_kc);
        const size_t smem = dnsst::RKM_SMEM;
        // tensor maps of the stage field's four buffers (any of the 16 RK field buffers can hold it: Q rotates)
        dnsst::RKMaps maps;
        a.use_tma = h->tma_ok ? 1 : 0;
        for (int m = 0; m < 4; ++m) {
            const size_t idx = ((const char *)qs[m] - (h->ws + h->L.off_fields)) / h->L.field_bytes;
            if (idx >= 16) a.use_tma = 0;
            maps.m[m] = h->tmap[idx < 16 ? idx : 0];
        }
#define DNS_LAUNCH_MARCH(M, S)                                                                                          \
    do {                                                                                                                \
        auto kern = dnsst::k_rk_march<STAGE, ELIM, M, S>;                                                               \
        if (h->prepare) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess ? DNSLAB_OK : DNSLAB_ECUDA; \
        ProfScope ps(h, DNSLAB_K_RK);                                                                                   \
        kern<<<grd, blk, smem, h->stream>>>(a, maps);                                                                   \
    } while (0)
        if (masked && sources) DNS_LAUNCH_MARCH(true, true);
        else if (masked) DNS_LAUNCH_MARCH(true, false);
        else if (sources) DNS_LAUNCH_MARCH(false, true);
        else DNS_LAUNCH_MARCH(false, false);
#undef DNS_LAUNCH_MARCH
        return check_launch(h);
    }
    if (h->prepare) return DNSLAB_OK;
    ProfScope ps(h, DNSLAB_K_RK);
    const dim3 blk = h->rk_block;
    const dim3 grd(h->P.nx / blk.x, h->P.ny / blk.y, h->P.nz / blk.z);
    if (masked && sources) dnsst::k_rk<STAGE, ELIM, true, true><<<grd, blk, 0, h->stream>>>(a);
    else if (masked) dnsst::k_rk<STAGE, ELIM, true, false><<<grd, blk, 0, h->stream>>>(a);
    else if (sources) dnsst::k_rk<STAGE, ELIM, false, true><<<grd, blk, 0, h->stream>>>(a);
    else dnsst::k_rk<STAGE, ELIM, false, false><<<grd, blk, 0, h->stream>>>(a);
    return check_launch(h);
}

// ---- FFT passes -------------------------------------------------------------------------
template <int L> constexpr int col_xt() { return L >= 1024 ? 4 : (L >= 256 ? 8 : 16); }

// grid of a persistent pass: every SM filled with as many blocks as fit, never more blocks than tiles
template <typename K> int persistent_grid(dnslab *h, K kernel, int threads, size_t smem, size_t ntiles, unsigned *grid)
{
    if (smem > 48 * 1024) CK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem));
    if (per_sm < 1) return DNSLAB_ECUDA;
    size_t g = (size_t)per_sm * h->nsm;
    if (g > ntiles) g = ntiles;
    // equal shares: the smallest grid that still needs the same number of tiles per block
    const size_t per_block = (ntiles + g - 1) / g;
    g = (ntiles + per_block - 1) / per_block;
    *grid = (unsigned)g;
    return DNSLAB_OK;
}

template <int L, int DIR, bool PRO> int launch_fft_x_L(dnslab *h, const c2 *in, c2 *out, const dnsfft::PoissonRhsArgs &ra)
{
    constexpr int E = dnsfft::ElemsPerThreadZ<L>::value;
    constexpr int T = L / E;
    const size_t nlines = (size_t)h->P.ny * h->P.nz;
    size_t nl = 128 / T;
    if (nl > nlines) nl = nlines;
    const size_t smem = nl * (L + L / 8) * sizeof(c2); // <= 18 KB: no opt-in needed
    if (h->prepare) return DNSLAB_OK;
    ProfScope ps(h, DNSLAB_K_FFT_X);
    dnsfft::k_fft_x<L, DIR, PRO><<<(unsigned)(nlines / nl), (unsigned)(nl * T), smem, h->stream>>>(in, out, h->tw[0], (int)nl, (FFT_REV >> (DIR < 0 ? 0 : 4)) & 1, ra);
    return check_launch(h);
}

template <int DIR, bool PRO> int launch_fft_x(dnslab *h, const c2 *in, c2 *out, const dnsfft::PoissonRhsArgs &ra)
{
    switch (h->P.nx / 2) {
    case 4: return launch_fft_x_L<4, DIR, PRO>(h, in, out, ra);
    case 8: return launch_fft_x_L<8, DIR, PRO>(h, in, out, ra);
    case 16: return launch_fft_x_L<16, DIR, PRO>(h, in, out, ra);
    case 32: return launch_fft_x_L<32, DIR, PRO>(h, in, out, ra);
    case 64: return launch_fft_x_L<64, DIR, PRO>(h, in, out, ra);
    case 128: return launch_fft_x_L<128, DIR, PRO>(h, in, out, ra);
    case 256: return launch_fft_x_L<256, DIR, PRO>(h, in, out, ra);
    case 512: return launch_fft_x_L<512, DIR, PRO>(h, in, out, ra);
    case 1024: return launch_fft_x_L<1024, DIR, PRO>(h, in, out, ra);
    }
    return DNSLAB_EINVAL;
}

// y pass: axis 1; z pass (unfused, used only by tests of the transform itself): axis 2
template <int L, int XT, int DIR> int launch_fft_col_LX(dnslab *h, c2 *data, int axis)
{
    constexpr int T = L / dnsfft::ElemsPerThreadZ<L>::value;
    const int mx = h->P.nx / 2;
    const size_t stride = axis == 1 ? (size_t)mx : (size_t)mx * h->P.ny;
    const size_t other_stride = axis == 1 ? (size_t)mx * h->P.ny : (size_t)mx;
    const int nother = axis == 1 ? h->P.nz : h->P.ny;
    const size_t smem = (size_t)XT * L * sizeof(c2);
    auto kern = dnsfft::k_fft_col<L, XT, DIR>;
    if (h->prepare) {
        if (smem > 48 * 1024) CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        return DNSLAB_OK;
    }
    ProfScope ps(h, DNSLAB_K_FFT_Y);
    kern<<<(unsigned)((mx / XT) * nother), XT * T, smem, h->stream>>>(data, h->tw[axis], mx, stride, other_stride, (FFT_REV >> (DIR < 0 ? 1 : 3)) & 1);
    return check_launch(h);
}

template <int L, int DIR> int launch_fft_col_L(dnslab *h, c2 *data, int axis)
{
    constexpr int XT = col_xt<L>();
    if (h->P.nx / 2 >= XT) return launch_fft_col_LX<L, XT, DIR>(h, data, axis);
    return launch_fft_col_LX<L, 4, DIR>(h, data, axis);
}

template <int DIR> int launch_fft_col(dnslab *h, c2 *data, int axis)
{
    switch (axis == 1 ? h->P.ny : h->P.nz) {
    case 8: return launch_fft_col_L<8, DIR>(h, data, axis);
    case 16: return launch_fft_col_L<16, DIR>(h, data, axis);
    case 32: return launch_fft_col_L<32, DIR>(h, data, axis);
    case 64: return launch_fft_col_L<64, DIR>(h, data, axis);
    case 128: return launch_fft_col_L<128, DIR>(h, data, axis);
    case 256: return launch_fft_col_L<256, DIR>(h, data, axis);
    case 512: return launch_fft_col_L<512, DIR>(h, data, axis);
    case 1024: return launch_fft_col_L<1024, DIR>(h, data, axis);
    }
    return DNSLAB_EINVAL;
}

template <int L, int XT> int launch_fft_z_solve_LX(dnslab *h, c2 *data)
{
    constexpr int T = L / dnsfft::ElemsPerThreadZ<L>::value;
    constexpr int NT = XT * T < 32 ? 32 : XT * T;
    const int mx = h->P.nx / 2;
    const size_t smem = 2 * (size_t)XT * L * sizeof(c2);
    const size_t ntiles = (size_t)(mx / XT) * h->P.ny;
    auto kern = dnsfft::k_fft_z_solve<L, XT>;
    if (h->prepare) return persistent_grid(h, kern, NT, smem, ntiles, &h->zgrid);
    ProfScope ps(h, DNSLAB_K_FFT_Z);
    const double inv_n = 2.0 / (double)h->n; // the packed transform has n/2 complex points
    kern<<<h->zgrid, XT * T, smem, h->stream>>>(data, h->tw[2], mx, h->P.ny, h->eig[0], h->eig[1], h->eig[2], inv_n, (int)ntiles, (FFT_REV >> 2) & 1);
    return check_launch(h);
}

// The fused z pass by TMA: k_fft_yz_solve without a split of y (NY0 = 1) -- persistent two-group blocks, tiles of 4096 points
// (XT = 4096 / nz adjacent kx, at most 16) in and out as boxes of W's second tensor map.
template <int L> int launch_fft_z_solve_tma(dnslab *h, c2 *data, bool *done)
{
    constexpr int XT = 4096 / L > 16 ? 16 : 4096 / L, NT = XT * L / 16, ZB = L > 256 ? 256 : L;
    const int mx = h->P.nx / 2;
    *done = false;
    if (mx < XT || data != reinterpret_cast<c2 *>(h->W)) return DNSLAB_OK;
    const size_t smem = dnsfft::YzLayout<1, L, XT>::SMEM;
    auto kern = dnsfft::k_fft_yz_solve<1, L, XT>;
    if (h->prepare) {
        const cuuint64_t gdim[3] = {(cuuint64_t)(2 * mx), (cuuint64_t)h->P.ny, (cuuint64_t)h->P.nz};
        const cuuint32_t box[3] = {(cuuint32_t)(2 * XT), 1u, (cuuint32_t)ZB};
        h->wmapz_ok = encode_map3(h, &h->wmapz, (void *)data, gdim, box);
        if (h->wmapz_ok) CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        *done = h->wmapz_ok;
        return DNSLAB_OK;
    }
    if (!h->wmapz_ok) return DNSLAB_OK;
    *done = true;
    const size_t ntiles = (size_t)(mx / XT) * h->P.ny;
    size_t g = (size_t)h->nsm < ntiles ? (size_t)h->nsm : ntiles;
    const size_t per_block = (ntiles + g - 1) / g;
    g = (ntiles + per_block - 1) / per_block;
    ProfScope ps(h, DNSLAB_K_FFT_Z);
    kern<<<(unsigned)g, 2 * NT, smem, h->stream>>>(h->wmapz, h->tw[2], mx, h->P.ny, h->eig[0], h->eig[1], h->eig[2], 2.0 / (double)h->n,
                                                  (FFT_REV >> 2) & 1, (int)ntiles);
    return check_launch(h);
}

template <int L> int launch_fft_z_solve_L(dnslab *h, c2 *data)
{
    // The TMA route runs one block per SM with XT <= 16 columns per tile: at nz = 32 and 64 its tiles are only 512 and 1024
    // points and it loses to the cp.async kernel, which fills every SM (measured, 30 solves each, us per z pass, TMA / cp.async:
    // 2048x1024x32 476 / 200; 2048x1024x64 612 / 415; 1024x512x64 163 / 110; 2048x512x128 476 / 502; 1024x1024x128 477 / 490;
    // 1024x512x256 429 / 605; no difference on small grids).  So: TMA from nz = 128 up.
    if constexpr (L >= 128) {
        bool done = false;
        const int rc = launch_fft_z_solve_tma<L>(h, data, &done);
        if (rc || (done && !h->prepare)) return rc;
    }
    constexpr int XT = col_xt<L>();
    if (h->P.nx / 2 >= XT) return launch_fft_z_solve_LX<L, XT>(h, data);
    return launch_fft_z_solve_LX<L, 4>(h, data);
}

int launch_fft_z_solve(dnslab *h, c2 *data)
{
    switch (h->P.nz) {
    case 8: return launch_fft_z_solve_L<8>(h, data);
    case 16: return launch_fft_z_solve_L<16>(h, data);
    case 32: return launch_fft_z_solve_L<32>(h, data);
    case 64: return launch_fft_z_solve_L<64>(h, data);
    case 128: return launch_fft_z_solve_L<128>(h, data);
    case 256: return launch_fft_z_solve_L<256>(h, data);
    case 512: return launch_fft_z_solve_L<512>(h, data);
    case 1024: return launch_fft_z_solve_L<1024>(h, data);
    }
    return DNSLAB_EINVAL;
}

// ---- two-pass solve: k_fft_xy (x and the high digit of y) and k_fft_yz_solve (low digit of y, z, division) --------
// A tile of the xy pass is 4096 complex numbers (NY1 = 4096 / (nx/2) whole rows, at least 16; 70 KB of shared memory with
// padding, two blocks per SM); the fused middle pass takes NY0 = ny / NY1 rows by all of z for XT adjacent kx, 4096 numbers
// again, with runs of at least XT = 2 complex numbers (its tiles move by TMA, so short runs cost no LSU instructions).
// Shapes outside these limits (and masks that need the dense eq. 9 prologue) use the five single-axis passes.
// Measured on 512x256x128: xy tiles of 8192 points, one block per SM: 76 instead of 51 us per pass;
// middle pass with ordinary loads and stores: 99 us (8192 points, XT = 4) / 117 us (4096 points, XT = 2); by TMA: 113 us
// (8192 points, one block per SM), 80 us (4096 points, two blocks per SM), 76 us (4096 points, persistent two-group blocks).
constexpr int XY_TILE = 4096, YZ_TILE = 4096, YZ_XTMIN = 2;
constexpr int xy_rows(int mx) { return XY_TILE / mx < 16 ? 16 : XY_TILE / mx; } // rows of an xy tile: at least 16 (one radix-16 column butterfly)

int fused_ny1(const dnslab_params_t *P)
{
    const int mx = P->nx / 2;
    if (mx < 64 || mx > 512) return 0;
    const int ny1 = xy_rows(mx);
    if (P->ny < ny1) return 0;
    const int ny0 = P->ny / ny1;
    if (ny0 == 1) return ny1; // the middle pass is then the plain fused z pass
    if (ny0 > 16 || P->nz < 32 || ny0 * P->nz * YZ_XTMIN > YZ_TILE) return 0;
    return ny1;
}

template <int LX, int DIR> int launch_fft_xy_L(dnslab *h, const c2 *in, c2 *out)
{
    constexpr int NY1 = xy_rows(LX), NT = LX * NY1 / 16;
    const size_t smem = (size_t)NY1 * (LX + LX / 16) * sizeof(c2);
    auto kern = dnsfft::k_fft_xy<LX, NY1, DIR>;
    if (h->prepare) {
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int per_sm = 0;
        CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem));
        h->xy_ahead = per_sm * h->nsm; // the block that takes over an SM when this one retires
        return DNSLAB_OK;
    }
    ProfScope ps(h, DNSLAB_K_FFT_XY);
    kern<<<(unsigned)((h->P.ny / NY1) * h->P.nz), NT, smem, h->stream>>>(in, out, h->tw[0], h->twy1, h->tw[1], h->P.ny, DIR < 0 ? 0 : 1, h->xy_ahead);
    return check_launch(h);
}

template <int DIR> int launch_fft_xy(dnslab *h, const c2 *in, c2 *out)
{
    switch (h->P.nx / 2) {
    case 64: return launch_fft_xy_L<64, DIR>(h, in, out);
    case 128: return launch_fft_xy_L<128, DIR>(h, in, out);
    case 256: return launch_fft_xy_L<256, DIR>(h, in, out);
    case 512: return launch_fft_xy_L<512, DIR>(h, in, out);
    }
    return DNSLAB_EINVAL;
}

// Middle pass (k_fft_yz_solve): persistent blocks of two groups, tiles of YZ_TILE points moved by TMA -- one landing buffer,
// two work buffers and the z tables in shared memory (207 KB on 512x256x128).
template <int NY0, int LZ> int launch_fft_yz_solve_NL(dnslab *h, c2 *data)
{
    constexpr int XT = (YZ_TILE / (NY0 * LZ)) > 16 ? 16 : YZ_TILE / (NY0 * LZ);
    static_assert(XT >= YZ_XTMIN, "tile too large");
    constexpr int NT = XT * NY0 * LZ / 16, ZB = LZ > 256 ? 256 : LZ;
    const int mx = h->P.nx / 2;
    const size_t smem = dnsfft::YzLayout<NY0, LZ, XT>::SMEM;
    static_assert(dnsfft::YzLayout<NY0, LZ, XT>::SMEM <= 227 * 1024, "middle-pass buffers exceed the shared memory of an SM");
    auto kern = dnsfft::k_fft_yz_solve<NY0, LZ, XT>;
    if (h->prepare) {
        // the transform array as a rank-3 tensor of doubles (2 mx, ny, nz); one box is a tile (at most 256 planes per box)
        const cuuint64_t gdim[3] = {(cuuint64_t)(2 * mx), (cuuint64_t)h->P.ny, (cuuint64_t)h->P.nz};
        const cuuint32_t box[3] = {(cuuint32_t)(2 * XT), (cuuint32_t)NY0, (cuuint32_t)ZB};
        h->wmap_ok = encode_map3(h, &h->wmap, (void *)data, gdim, box);
        if (h->wmap_ok) CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        return DNSLAB_OK;
    }
    const size_t ntiles = (size_t)(mx / XT) * (h->P.ny / NY0);
    size_t g = (size_t)h->nsm < ntiles ? (size_t)h->nsm : ntiles;
    const size_t per_block = (ntiles + g - 1) / g; // equal shares: the smallest grid that needs the same number of tiles per block
    g = (ntiles + per_block - 1) / per_block;
    ProfScope ps(h, DNSLAB_K_FFT_YZ);
    kern<<<(unsigned)g, 2 * NT, smem, h->stream>>>(h->wmap, h->tw[2], mx, h->P.ny, h->eig[0], h->eig[1], h->eig[2], 2.0 / (double)h->n, 1, (int)ntiles);
    return check_launch(h);
}

template <int NY0> int launch_fft_yz_solve_N(dnslab *h, c2 *data)
{
    switch (h->P.nz) {
    case 32: return launch_fft_yz_solve_NL<NY0, 32>(h, data);
    case 64: return launch_fft_yz_solve_NL<NY0, 64>(h, data);
    case 128: return launch_fft_yz_solve_NL<NY0, 128>(h, data);
    case 256: if constexpr (NY0 <= 8) return launch_fft_yz_solve_NL<NY0, 256>(h, data); break;
    case 512: if constexpr (NY0 <= 4) return launch_fft_yz_solve_NL<NY0, 512>(h, data); break;
    case 1024: if constexpr (NY0 <= 2) return launch_fft_yz_solve_NL<NY0, 1024>(h, data); break;
    }
    return DNSLAB_EINVAL;
}

int launch_fft_yz_solve(dnslab *h, c2 *data)
{
    switch (h->P.ny / h->f_ny1) {
    case 1: return launch_fft_z_solve(h, data);
    case 2: return launch_fft_yz_solve_N<2>(h, data);
    case 4: return launch_fft_yz_solve_N<4>(h, data);
    case 8: return launch_fft_yz_solve_N<8>(h, data);
    case 16: return launch_fft_yz_solve_N<16>(h, data);
    }
    return DNSLAB_EINVAL;
}

// One solve p = F^-1[F[r]/lambda]; r = eq. 9 right-hand side built from (d, pold, face) on the fly
// when `prologue`, else r = d as given.  pout may alias d or pold (it is written by the last pass).
int poisson_solve(dnslab *h, const double *d, const double *pold, double *pout, bool prologue)
{
    dnsfft::PoissonRhsArgs ra;
    prologue = prologue && h->face && !h->blist;
    ra.d = d; ra.p = pold; ra.face = (prologue ? h->face : nullptr);
    ra.nx = h->P.nx; ra.ny = h->P.ny; ra.nz = h->P.nz;
    ra.r2x = 1.0 / (2.0 * h->P.dx); ra.r2y = 1.0 / (2.0 * h->P.dy); ra.r2z = 1.0 / (2.0 * h->P.dz);
    c2 *W = reinterpret_cast<c2 *>(h->W);
    int rc;
    if (!prologue && h->f_ny1 > 0) {
        if ((rc = launch_fft_xy<-1>(h, reinterpret_cast<const c2 *>(d), W))) return rc;
        if ((rc = launch_fft_yz_solve(h, W))) return rc;
        return launch_fft_xy<+1>(h, W, reinterpret_cast<c2 *>(pout));
    }
    if (prologue) rc = launch_fft_x<-1, true>(h, reinterpret_cast<const c2 *>(d), W, ra);
    else rc = launch_fft_x<-1, false>(h, reinterpret_cast<const c2 *>(d), W, ra);
    if (rc) return rc;
    if ((rc = launch_fft_col<-1>(h, W, 1))) return rc;
    if ((rc = launch_fft_z_solve(h, W))) return rc;
    if ((rc = launch_fft_col<+1>(h, W, 1))) return rc;
    return launch_fft_x<+1, false>(h, W, reinterpret_cast<c2 *>(pout), ra);
}

int launch_div(dnslab *h, double *const *q)
{
    ProfScope ps(h, DNSLAB_K_DIV);
    if (h->P.nx >= 64 && h->P.ny >= 8) {
        const dim3 blk2(32, 8, 1), grd2(h->P.nx / 64, h->P.ny / 8, h->P.nz);
        dnsst::k_div2<<<grd2, blk2, 0, h->stream>>>(q[0], q[1], q[2], h->d, h->P.nx, h->P.ny, h->P.nz, 1.0 / (2.0 * h->P.dx),
                                                    1.0 / (2.0 * h->P.dy), 1.0 / (2.0 * h->P.dz), (ST_REV >> 4) & 1);
        return check_launch(h);
    }
    const dim3 blk = tile_block(h);
    const dim3 grd(h->P.nx / blk.x, h->P.ny / blk.y, h->P.nz);
    dnsst::k_div<<<grd, blk, 0, h->stream>>>(q[0], q[1], q[2], h->d, h->P.nx, h->P.ny, h->P.nz, 1.0 / (2.0 * h->P.dx),
                                              1.0 / (2.0 * h->P.dy), 1.0 / (2.0 * h->P.dz));
    return check_launch(h);
}

int launch_project(dnslab *h, double *const *q, const double *p)
{
    const dim3 blk = tile_block(h);
    const dim3 grd(h->P.nx / blk.x, h->P.ny / blk.y, h->P.nz);
    const double r2x = 1.0 / (2.0 * h->P.dx), r2y = 1.0 / (2.0 * h->P.dy), r2z = 1.0 / (2.0 * h->P.dz);
    ProfScope ps(h, DNSLAB_K_PROJECT);
    if (h->P.nx >= 64 && h->P.ny >= 8) {
        const dim3 blk2(32, 8, 1), grd2(h->P.nx / 64, h->P.ny / 8, h->P.nz);
        if (h->face) dnsst::k_project2<true><<<grd2, blk2, 0, h->stream>>>(q[0], q[1], q[2], p, h->face, h->P.nx, h->P.ny, h->P.nz, r2x, r2y, r2z, (ST_REV >> 5) & 1);
        else dnsst::k_project2<false><<<grd2, blk2, 0, h->stream>>>(q[0], q[1], q[2], p, nullptr, h->P.nx, h->P.ny, h->P.nz, r2x, r2y, r2z, (ST_REV >> 5) & 1);
        return check_launch(h);
    }
    if (h->face) dnsst::k_project<true><<<grd, blk, 0, h->stream>>>(q[0], q[1], q[2], p, h->face, h->P.nx, h->P.ny, h->P.nz, r2x, r2y, r2z);
    else dnsst::k_project<false><<<grd, blk, 0, h->stream>>>(q[0], q[1], q[2], p, nullptr, h->P.nx, h->P.ny, h->P.nz, r2x, r2y, r2z);
    return check_launch(h);
}

int launch_eq9_sparse(dnslab *h, const double *p, bool first)
{
    int lgx = 0, lgy = 0;
    while ((1 << lgx) < h->P.nx) ++lgx;
    while ((1 << lgy) < h->P.ny) ++lgy;
    ProfScope ps(h, DNSLAB_K_EQ9);
    // one wave: 8 blocks of 256 threads per SM, never more blocks than the list needs
    unsigned grid = (unsigned)((h->nb + 255) / 256);
    if (grid > 8u * (unsigned)h->nsm) grid = 8u * (unsigned)h->nsm;
    const double r2x = 1.0 / (2.0 * h->P.dx), r2y = 1.0 / (2.0 * h->P.dy), r2z = 1.0 / (2.0 * h->P.dz);
    if (first) dnsst::k_eq9_sparse<true><<<grid, 256, 0, h->stream>>>(h->d, p, h->blist, h->bsave, h->nb, h->P.nx, h->P.ny, h->P.nz, lgx, lgy, r2x, r2y, r2z);
    else dnsst::k_eq9_sparse<false><<<grid, 256, 0, h->stream>>>(h->d, p, h->blist, h->bsave, h->nb, h->P.nx, h->P.ny, h->P.nz, lgx, lgy, r2x, r2y, r2z);
    return check_launch(h);
}

// NEXT-1: eq. 6 filter of the four fields, in -> out (different buffers)
int launch_filter(dnslab *h, double *const *in, double *const *out)
{
    dnsst::FilterArgs a;
    for (int m = 0; m < 4; ++m) {
        a.in[m] = in[m];
        a.out[m] = out[m];
    }
    a.face = h->face;
    a.nx = h->P.nx; a.ny = h->P.ny; a.nz = h->P.nz;
    const double pi = 3.14159265358979323846;
    a.g = 1.0 / (pi * pi * pi * pi * pi * pi);
    if (h->prepare) { // the only kernels here that need the shared-memory opt-in
        CK(cudaFuncSetAttribute(dnsst::k_filter_march<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dnsst::FM_SMEM));
        CK(cudaFuncSetAttribute(dnsst::k_filter_march<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dnsst::FM_SMEM));
        return DNSLAB_OK;
    }
    ProfScope ps(h, DNSLAB_K_FILTER);
    if (h->P.nx >= dnsst::FM_TX && h->P.ny >= dnsst::FM_TY) {
        // z-marching kernel: 64 x 8 columns of one field; >= 3 waves of 4 blocks per SM, at least 8 planes per block
        // (512x256x128: 64 planes per block 286 us, 32: 296 us, 16: 302 us, 8: 326 us, 128 -- 1.7 waves: 306 us)
        const long tiles = 4L * (h->P.nx / dnsst::FM_TX) * (h->P.ny / dnsst::FM_TY);
        int kc = h->P.nz;
        while (kc > 8 && tiles * (h->P.nz / kc) < 12L * h->nsm) kc /= 2;
        a.kc = kc;
        const dim3 blk(32, dnsst::FM_TY, 1);
        const dim3 grd(h->P.nx / dnsst::FM_TX, h->P.ny / dnsst::FM_TY, 4 * (h->P.nz / kc));
        const size_t smem = dnsst::FM_SMEM;
        if (h->face) dnsst::k_filter_march<true><<<grd, blk, smem, h->stream>>>(a);
        else dnsst::k_filter_march<false><<<grd, blk, smem, h->stream>>>(a);
        return check_launch(h);
    }
    const dim3 blk(h->P.nx < 32 ? h->P.nx : 32, h->P.ny < 8 ? h->P.ny : 8, 1);
    // enough blocks for >= 4 waves of 8 blocks per SM, at least 8 planes per block
    const long tiles = 4L * (h->P.nx / blk.x) * (h->P.ny / blk.y);
    int kc = h->P.nz;
    while (kc > 8 && tiles * (h->P.nz / kc) < 32L * h->nsm) kc /= 2;
    a.kc = kc;
    const dim3 grd(h->P.nx / blk.x, h->P.ny / blk.y, 4 * (h->P.nz / kc));
    if (h->face) dnsst::k_filter<true><<<grd, blk, 0, h->stream>>>(a);
    else dnsst::k_filter<false><<<grd, blk, 0, h->stream>>>(a);
    return check_launch(h);
}

// NEXT-4: one implicit Euler step of the attached particles in the field h->Q
int launch_particles(dnslab *h)
{
    dnspart::PartArgs a;
    a.u = h->Q[0]; a.v = h->Q[1]; a.w = h->Q[2];
    a.state = h->pstate;
    a.n = h->np;
    a.nx = h->P.nx; a.ny = h->P.ny; a.nz = h->P.nz;
    a.dx = h->P.dx; a.dy = h->P.dy; a.dz = h->P.dz;
    a.dt = h->P.dt; a.nu = h->P.nu; a.rho_f = h->prho_f;
    for (int c = 0; c < 3; ++c) a.g[c] = h->pgrav[c];
    ProfScope ps(h, DNSLAB_K_PARTICLES);
    dnspart::k_particles<<<(unsigned)((h->np + 127) / 128), 128, 0, h->stream>>>(a);
    return check_launch(h);
}

// divergence, n_piter iterations of eq. 9 warm-started from p, correction (in place on q)
int pressure_stage(dnslab *h, double *const *q, double *p)
{
    int rc;
    if ((rc = launch_div(h, q))) return rc;
    for (int it = 0; it < h->P.n_piter; ++it) {
        if (h->blist && h->nb > 0 && (rc = launch_eq9_sparse(h, p, it == 0))) return rc;
        if ((rc = poisson_solve(h, h->d, p, p, true))) return rc;
    }
    return launch_project(h, q, p);
}

// called once from dnslab_create with h->prepare set: nothing is launched
int prepare_kernels(dnslab *h)
{
    int rc;
    if (h->P.flags & 2u) {
        if ((rc = launch_rk<1, false>(h, h->Q, h->A, nullptr))) return rc;
        if ((rc = launch_rk<2, false>(h, h->A, h->Bf, nullptr))) return rc;
        if ((rc = launch_rk<3, false>(h, h->Bf, h->A, nullptr))) return rc;
        if ((rc = launch_rk<4, false>(h, h->A, nullptr, nullptr))) return rc;
    } else {
        if ((rc = launch_rk<1, true>(h, h->Q, h->A, nullptr))) return rc;
        if ((rc = launch_rk<2, true>(h, h->A, h->Bf, h->Qc))) return rc;
        if ((rc = launch_rk<3, true>(h, h->Bf, h->A, nullptr))) return rc;
        if ((rc = launch_rk<4, true>(h, h->A, nullptr, h->Qc))) return rc;
    }
    if ((rc = poisson_solve(h, h->d, h->p, h->p, true))) return rc;
    if ((rc = poisson_solve(h, h->d, h->p, h->p, false))) return rc; // dnslab_poisson: never the dense prologue
    // without a tensor map for W (no driver entry point) the solve takes the five single-axis passes, which need none
    if (h->f_ny1 > 0 && h->P.ny / h->f_ny1 > 1 && !h->wmap_ok) h->f_ny1 = 0;
    {
        // dnslab_rfft3 / dnslab_irfft3 always take the single-axis passes, along z too
        const int keep = h->f_ny1;
        h->f_ny1 = 0;
        rc = poisson_solve(h, h->d, h->p, h->p, false);
        h->f_ny1 = keep;
        if (rc) return rc;
        c2 *W = reinterpret_cast<c2 *>(h->W);
        if ((rc = launch_fft_col<-1>(h, W, 2))) return rc;
        if ((rc = launch_fft_col<+1>(h, W, 2))) return rc;
    }
    if ((h->P.flags & 1u) && (rc = launch_filter(h, h->Qc, h->A))) return rc;
    return DNSLAB_OK;
}

} // namespace

extern "C" {

const char *dnslab_strerror(int code)
{
    switch (code) {
    case DNSLAB_OK: return "ok";
    case DNSLAB_EINVAL: return "invalid argument";
    case DNSLAB_ENOMEM: return "workspace too small";
    case DNSLAB_ECUDA: return "CUDA error";
    case DNSLAB_EARCH: return "no sm_100 device";
    case DNSLAB_ELIMIT: return "box has more rows (size[1]*size[2]) than the static scratch array holds";
    }
    return "unknown error";
}

size_t dnslab_workspace_bytes(const dnslab_params_t *params)
{
    if (!valid_params(params)) return 0;
    return make_layout(params).total;
}

int dnslab_create(const dnslab_params_t *params, const uint8_t *mask, const dnslab_source_t *src, int32_t nsrc, void *workspace,
                  void *cuda_stream, dnslab_t **out)
{
    if (!valid_params(params) || !workspace || !out || nsrc < 0 || nsrc > DNSLAB_MAX_SOURCES || (nsrc > 0 && !src)) return DNSLAB_EINVAL;
    if ((uintptr_t)workspace % ALIGN) return DNSLAB_EINVAL;
    for (int s = 0; s < nsrc; ++s) {
        if (!(src[s].tau_f > 0)) return DNSLAB_EINVAL;
        const int nn[3] = {params->nx, params->ny, params->nz};
        for (int a = 0; a < 3; ++a)
            if (src[s].size[a] < 1 || src[s].size[a] > nn[a]) return DNSLAB_EINVAL; // eq. 5 divides by the half width
    }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return DNSLAB_EARCH;
    if (prop.major != 10) return DNSLAB_EARCH;

    dnslab *h = new (std::nothrow) dnslab;
    if (!h) return DNSLAB_ENOMEM;
    std::memset(h, 0, sizeof(*h));
    h->P = *params;
    h->n = (size_t)params->nx * params->ny * params->nz;
    h->stream = (cudaStream_t)cuda_stream;
    h->nsm = prop.multiProcessorCount;
    h->ws = (char *)workspace;
    h->L = make_layout(params);
    const Layout &L = h->L;
    auto fld = [&](int idx) { return (double *)(h->ws + L.off_fields + (size_t)idx * L.field_bytes); };
    for (int m = 0; m < 4; ++m) {
        h->Q[m] = fld(m);
        h->A[m] = fld(4 + m);
        h->Bf[m] = fld(8 + m);
        h->Qc[m] = fld(12 + m);
    }
    h->p = fld(16);
    h->d = fld(17);
    h->W = fld(18);
    h->ps = (params->flags & 2u) ? fld(19) : nullptr;
    {
        // 64 x 2 x 2 brick (256 threads); narrower in x on tiny grids
        unsigned bx = params->nx < 64 ? params->nx : 64, by = 2, bz = 2;
        while (bx * by * bz < 256 && by < (unsigned)params->ny && by <= bz) by *= 2;
        while (bx * by * bz < 256 && bz < (unsigned)params->nz) bz *= 2;
        h->rk_block = dim3(bx, by, bz);
        // marching kernel for nx >= 64: 16 planes per block (the best of 8...128 on 512x256x128, and on 1024x512x256, where
        // 128 planes per block -- 2048 blocks either way -- measured 2.41 instead of 2.15 ms per stage), 8 when that leaves
        // fewer than 6 waves of 2 blocks per SM
        h->rk_kc = 0;
        if (params->nx >= dnsst::RKM_TX) {
            const long tiles = (long)(params->nx / dnsst::RKM_TX) * (params->ny / dnsst::RKM_TY);
            int kc = params->nz < 16 ? params->nz : 16;
            while (kc > 8 && tiles * (params->nz / kc) < 6L * 2 * prop.multiProcessorCount) kc /= 2;
            h->rk_kc = kc;
        }
    }

    // TMA descriptors for k_rk_march's plane tiles: rank 3 (x, y, z), fp64, box 68 x 10 x 1, out-of-bounds = zero (only
    // interior blocks use them).  The encoder is a driver entry point fetched at run time; without it (or for the brick
    // kernel of small grids) every block copies its tiles with cp.async.
    h->tma_ok = false;
    h->wmap_ok = false;
    h->wmapz_ok = false;
    h->tma_encode = nullptr;
#ifndef DNSLAB_TEST_NO_TMA // test-only build (libdnslab_notma.so): the encoder stays null, so every fallback below is the path taken
    {
        void *fp = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qres) == cudaSuccess && fp != nullptr &&
            qres == cudaDriverEntryPointSuccess)
            h->tma_encode = fp;
        (void)cudaGetLastError();
    }
#endif
    if (h->rk_kc > 0) {
        const cuuint64_t gdim[3] = {(cuuint64_t)params->nx, (cuuint64_t)params->ny, (cuuint64_t)params->nz};
        const cuuint32_t box[3] = {(cuuint32_t)dnsst::RKM_SW, (cuuint32_t)dnsst::RKM_ROWS, 1u};
        bool ok = true;
        for (int b = 0; b < 16 && ok; ++b) ok = encode_map3(h, &h->tmap[b], (void *)fld(b), gdim, box);
        h->tma_ok = ok;
    }

    auto fail = [&](int rc) { delete h; return rc; };
#define CKF(call) do { if ((call) != cudaSuccess) return fail(DNSLAB_ECUDA); } while (0)
    CKF(cudaMemsetAsync(h->ws + L.off_fields, 0, L.nfields * L.field_bytes, h->stream));

    // mask -> face bytes; dropped entirely when there is no solid cell
    h->face = nullptr;
    if (mask) {
        uint8_t *face = (uint8_t *)(h->ws + L.off_face);
        uint8_t *tmp = (uint8_t *)h->W; // W is scratch here
        CKF(cudaMemcpyAsync(tmp, mask, h->n, cudaMemcpyDefault, h->stream));
        dim3 blk(params->nx < 128 ? params->nx : 128);
        dim3 grd(params->nx / blk.x, params->ny, params->nz);
        dnsst::k_face_mask<<<grd, blk, 0, h->stream>>>(tmp, face, params->nx, params->ny, params->nz);
        h->launches++;
        CKF(cudaPeekAtLastError());
        std::vector<uint8_t> hm(h->n);
        CKF(cudaMemcpyAsync(hm.data(), tmp, h->n, cudaMemcpyDeviceToHost, h->stream));
        CKF(cudaStreamSynchronize(h->stream));
        bool any_solid = false;
        for (size_t o = 0; o < h->n; ++o)
            if (!hm[o]) { any_solid = true; break; }
        if (any_solid) h->face = face;
        CKF(cudaMemsetAsync(h->W, 0, L.field_bytes, h->stream));
        if (any_solid) {
            // cells with at least one solid face neighbour, ascending index order
            const int nx = params->nx, ny = params->ny, nz = params->nz;
            std::vector<unsigned long long> bl;
            bool fits = true;
            for (int k = 0; k < nz && fits; ++k) {
                const size_t kp = (size_t)((k + 1) & (nz - 1)), km = (size_t)((k - 1) & (nz - 1));
                for (int j = 0; j < ny && fits; ++j) {
                    const size_t jp = (size_t)((j + 1) & (ny - 1)), jm = (size_t)((j - 1) & (ny - 1));
                    const uint8_t *r0 = hm.data() + (size_t)nx * (j + (size_t)ny * k);
                    const uint8_t *ryp = hm.data() + (size_t)nx * (jp + (size_t)ny * k), *rym = hm.data() + (size_t)nx * (jm + (size_t)ny * k);
                    const uint8_t *rzp = hm.data() + (size_t)nx * (j + (size_t)ny * kp), *rzm = hm.data() + (size_t)nx * (j + (size_t)ny * km);
                    for (int i = 0; i < nx; ++i) {
                        const unsigned f = (r0[i] != 0) | ((r0[(i + 1) & (nx - 1)] != 0) << 1) | ((r0[(i - 1) & (nx - 1)] != 0) << 2) |
                                           ((ryp[i] != 0) << 3) | ((rym[i] != 0) << 4) | ((rzp[i] != 0) << 5) | ((rzm[i] != 0) << 6);
                        if ((f & 0x7e) == 0x7e) continue; // all six neighbours fluid: the bracket is exactly 0
                        if (bl.size() >= L.bcap) { fits = false; break; }
                        bl.push_back((unsigned long long)((size_t)i + (size_t)nx * (j + (size_t)ny * k)) | ((unsigned long long)f << 32));
                    }
                }
            }
            if (fits) {
                h->blist = (unsigned long long *)(h->ws + L.off_blist);
                h->bsave = (double *)(h->ws + L.off_bsave);
                h->nb = (int)bl.size();
                if (h->nb) CKF(cudaMemcpyAsync(h->blist, bl.data(), bl.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice, h->stream));
                CKF(cudaStreamSynchronize(h->stream));
            }
        }
    }

    // twiddles exp(-2 pi i t/L) per axis and eigenvalue parts (sin(2 pi k/N_a)/D_a)^2
    {
        const int len[3] = {params->nx / 2, params->ny, params->nz};
        const int full[3] = {params->nx, params->ny, params->nz};
        const double dd[3] = {params->dx, params->dy, params->dz};
        size_t eoff = 0;
        for (int a = 0; a < 3; ++a) {
            std::vector<c2> tw(len[a]);
            for (int t = 0; t < len[a]; ++t) {
                // exact octant reduction keeps the table symmetric and accurate to 0.5 ulp of libm
                const long double ang = -2.0L * 3.141592653589793238462643383279502884L * (long double)t / (long double)len[a];
                tw[t].x = (double)cosl(ang);
                tw[t].y = (double)sinl(ang);
            }
            h->tw[a] = (c2 *)(h->ws + L.off_tw[a]);
            CKF(cudaMemcpyAsync(h->tw[a], tw.data(), tw.size() * sizeof(c2), cudaMemcpyHostToDevice, h->stream));
            std::vector<double> e(len[a]);
            for (int k = 0; k < len[a]; ++k) {
                const double s = std::sin(2.0 * M_PI * (double)k / (double)full[a]) / dd[a];
                e[k] = s * s;
            }
            h->eig[a] = (double *)(h->ws + L.off_eig) + eoff;
            eoff += len[a];
            CKF(cudaMemcpyAsync(h->eig[a], e.data(), e.size() * sizeof(double), cudaMemcpyHostToDevice, h->stream));
            CKF(cudaStreamSynchronize(h->stream));
        }
    }

    h->f_ny1 = fused_ny1(params);
    h->twy1 = (c2 *)(h->ws + L.off_twy1);
    if (h->f_ny1 > 0) {
        std::vector<c2> tw(h->f_ny1);
        for (int t = 0; t < h->f_ny1; ++t) {
            const long double ang = -2.0L * 3.141592653589793238462643383279502884L * (long double)t / (long double)h->f_ny1;
            tw[t].x = (double)cosl(ang);
            tw[t].y = (double)sinl(ang);
        }
        CKF(cudaMemcpyAsync(h->twy1, tw.data(), tw.size() * sizeof(c2), cudaMemcpyHostToDevice, h->stream));
        CKF(cudaStreamSynchronize(h->stream));
    }

    // sources: one-dimensional factor tables of eq. 5
    h->nsrc = nsrc;
    h->stab = (double *)(h->ws + L.off_stab);
    if (nsrc > 0) {
        const int per = params->nx + params->ny + params->nz;
        std::vector<double> tab((size_t)nsrc * per);
        for (int s = 0; s < nsrc; ++s) {
            double *t = tab.data() + (size_t)s * per;
            source_profile(params->nx, params->dx, src[s].lo[0], src[s].size[0], src[s].B[0], t);
            source_profile(params->ny, params->dy, src[s].lo[1], src[s].size[1], src[s].B[1], t + params->nx);
            source_profile(params->nz, params->dz, src[s].lo[2], src[s].size[2], src[s].B[2], t + params->nx + params->ny);
            dnsst::SourceDev &S = h->src[s];
            for (int m = 0; m < 3; ++m) S.set[m] = src[s].u_set[m];
            S.set[3] = src[s].c_set;
            S.rtau = 1.0 / src[s].tau_f;
            S.comps = src[s].comps & 0xF;
            S.off = s * per;
        }
        CKF(cudaMemcpyAsync(h->stab, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice, h->stream));
        CKF(cudaStreamSynchronize(h->stream));
    }
    CKF(cudaStreamSynchronize(h->stream));
#undef CKF
    // one dry walk over the launchers: each configures the kernel instantiation it will use (shared-memory
    // opt-in, persistent grid size) and launches nothing, so that no launch path calls cudaFuncSetAttribute
    h->prepare = true;
    int prc = prepare_kernels(h);
    h->prepare = false;
    if (prc) return fail(prc);
    *out = h;
    return DNSLAB_OK;
}

int dnslab_set_fields(dnslab_t *h, const double *u, const double *v, const double *w, const double *c, const double *p)
{
    if (!h || !u || !v || !w || !c) return DNSLAB_EINVAL;
    const double *in[4] = {u, v, w, c};
    const size_t bytes = h->n * sizeof(double);
    for (int m = 0; m < 4; ++m) CK(cudaMemcpyAsync(h->Q[m], in[m], bytes, cudaMemcpyDefault, h->stream));
    if (p) CK(cudaMemcpyAsync(h->p, p, bytes, cudaMemcpyDefault, h->stream));
    else CK(cudaMemsetAsync(h->p, 0, bytes, h->stream));
    if (h->face) {
        dnsst::k_mask_select<<<(unsigned)((h->n + 255) / 256), 256, 0, h->stream>>>(h->Q[0], h->Q[1], h->Q[2], h->Q[3], h->face, h->n);
        return check_launch(h);
    }
    return DNSLAB_OK;
}

int dnslab_step(dnslab_t *h, int32_t nsteps)
{
    if (!h || nsteps < 0) return DNSLAB_EINVAL;
    const bool stage_proj = (h->P.flags & 2u) != 0, filter = (h->P.flags & 1u) != 0;
    const size_t bytes = h->n * sizeof(double);
    int rc;
    for (int it = 0; it < nsteps; ++it) {
        if (!stage_proj) {
            // Qc eliminated: A = Q2, Bf = Q3, Qc = S = Q2 - Qn + 2 Q3 (written by stage 2), A = Q4, Q* in place of S
            if ((rc = launch_rk<1, true>(h, h->Q, h->A, nullptr))) return rc;
            if ((rc = launch_rk<2, true>(h, h->A, h->Bf, h->Qc))) return rc;
            if ((rc = launch_rk<3, true>(h, h->Bf, h->A, nullptr))) return rc;
            if ((rc = launch_rk<4, true>(h, h->A, nullptr, h->Qc))) return rc;
            // Q* is in Qc; A is free for the filter
            double **fin = h->Qc;
            if ((rc = pressure_stage(h, fin, h->p))) return rc;
            if (filter) {
                if ((rc = launch_filter(h, fin, h->A))) return rc;
                fin = h->A;
            }
            for (int m = 0; m < 4; ++m) {
                double *t = h->Q[m];
                h->Q[m] = fin[m];
                fin[m] = t;
            }
            if (h->np > 0 && (rc = launch_particles(h))) return rc;
            continue;
        }
        // NEXT-2 variant: every stage field is projected, so the accumulate form is needed
        if ((rc = launch_rk<1, false>(h, h->Q, h->A, nullptr))) return rc;
        CK(cudaMemcpyAsync(h->ps, h->p, bytes, cudaMemcpyDeviceToDevice, h->stream));
        if ((rc = pressure_stage(h, h->A, h->ps))) return rc;
        if ((rc = launch_rk<2, false>(h, h->A, h->Bf, nullptr))) return rc;
        CK(cudaMemcpyAsync(h->ps, h->p, bytes, cudaMemcpyDeviceToDevice, h->stream));
        if ((rc = pressure_stage(h, h->Bf, h->ps))) return rc;
        if ((rc = launch_rk<3, false>(h, h->Bf, h->A, nullptr))) return rc;
        CK(cudaMemcpyAsync(h->ps, h->p, bytes, cudaMemcpyDeviceToDevice, h->stream));
        if ((rc = pressure_stage(h, h->A, h->ps))) return rc;
        if ((rc = launch_rk<4, false>(h, h->A, nullptr, nullptr))) return rc;
        if ((rc = pressure_stage(h, h->Qc, h->p))) return rc;
        double **fin = h->Qc;
        if (filter) {
            if ((rc = launch_filter(h, h->Qc, h->A))) return rc;
            fin = h->A;
        }
        for (int m = 0; m < 4; ++m) {
            double *t = h->Q[m];
            h->Q[m] = fin[m];
            fin[m] = t;
        }
        if (h->np > 0 && (rc = launch_particles(h))) return rc;
    }
    return DNSLAB_OK;
}

int dnslab_poisson(dnslab_t *h, const double *rhs, double *p)
{
    if (!h || !rhs || !p) return DNSLAB_EINVAL;
    if (((uintptr_t)rhs | (uintptr_t)p) & 15) return DNSLAB_EINVAL; // every pass moves 16-byte pairs
    return poisson_solve(h, rhs, nullptr, p, false);
}

// true if [a, a + na) and [b, b + nb) share a byte
static bool ranges_overlap(const void *a, size_t na, const void *b, size_t nb)
{
    const uintptr_t a0 = (uintptr_t)a, b0 = (uintptr_t)b;
    return a0 < b0 + nb && b0 < a0 + na;
}

int dnslab_rfft3(dnslab_t *h, const double *in, double *out)
{
    if (!h || !in || !out) return DNSLAB_EINVAL;
    if (((uintptr_t)in | (uintptr_t)out) & 15) return DNSLAB_EINVAL;
    if (ranges_overlap(in, h->n * sizeof(double), out, (size_t)(h->P.nx / 2 + 1) * h->P.ny * h->P.nz * sizeof(c2))) return DNSLAB_EINVAL;
    const int M = h->P.nx / 2;
    dnsfft::PoissonRhsArgs ra{};
    c2 *W = reinterpret_cast<c2 *>(h->W);
    int rc;
    if ((rc = launch_fft_x<-1, false>(h, reinterpret_cast<const c2 *>(in), W, ra))) return rc;
    if ((rc = launch_fft_col<-1>(h, W, 1))) return rc;
    if ((rc = launch_fft_col<-1>(h, W, 2))) return rc;
    const size_t total = (size_t)(M + 1) * h->P.ny * h->P.nz;
    dnsfft::k_r2c_tangle<<<(unsigned)((total + 255) / 256), 256, 0, h->stream>>>(W, reinterpret_cast<c2 *>(out), M, h->P.ny, h->P.nz, 0, 1.0);
    return check_launch(h);
}

int dnslab_irfft3(dnslab_t *h, const double *in, double *out)
{
    if (!h || !in || !out) return DNSLAB_EINVAL;
    if (((uintptr_t)in | (uintptr_t)out) & 15) return DNSLAB_EINVAL;
    if (ranges_overlap(in, (size_t)(h->P.nx / 2 + 1) * h->P.ny * h->P.nz * sizeof(c2), out, h->n * sizeof(double))) return DNSLAB_EINVAL;
    const int M = h->P.nx / 2;
    dnsfft::PoissonRhsArgs ra{};
    c2 *W = reinterpret_cast<c2 *>(h->W);
    const size_t total = (size_t)M * h->P.ny * h->P.nz;
    dnsfft::k_r2c_tangle<<<(unsigned)((total + 255) / 256), 256, 0, h->stream>>>(reinterpret_cast<const c2 *>(in), W, M, h->P.ny, h->P.nz, 1,
                                                                                  1.0 / (double)total);
    int rc;
    if ((rc = check_launch(h))) return rc;
    if ((rc = launch_fft_col<+1>(h, W, 2))) return rc;
    if ((rc = launch_fft_col<+1>(h, W, 1))) return rc;
    return launch_fft_x<+1, false>(h, W, reinterpret_cast<c2 *>(out), ra);
}

int dnslab_fields(dnslab_t *h, const double **u, const double **v, const double **w, const double **c, const double **p)
{
    if (!h) return DNSLAB_EINVAL;
    if (u) *u = h->Q[0];
    if (v) *v = h->Q[1];
    if (w) *w = h->Q[2];
    if (c) *c = h->Q[3];
    if (p) *p = h->p;
    return DNSLAB_OK;
}

int dnslab_get_fields(dnslab_t *h, double *u, double *v, double *w, double *c, double *p)
{
    if (!h) return DNSLAB_EINVAL;
    double *out[5] = {u, v, w, c, p};
    const double *in[5] = {h->Q[0], h->Q[1], h->Q[2], h->Q[3], h->p};
    for (int m = 0; m < 5; ++m)
        if (out[m]) CK(cudaMemcpyAsync(out[m], in[m], h->n * sizeof(double), cudaMemcpyDefault, h->stream));
    return DNSLAB_OK;
}

int64_t dnslab_launch_count(const dnslab_t *h) { return h ? h->launches : -1; }

int dnslab_profile(dnslab_t *h, int enable)
{
    if (!h) return DNSLAB_EINVAL;
    if (int rc = prof_drain(h)) return rc;
    if (enable && !h->prof) h->prof = new (std::nothrow) std::vector<ProfRec>();
    if (enable && !h->prof) return DNSLAB_ENOMEM;
    if (enable) {
        for (int c = 0; c < DNSLAB_NCLASS; ++c) {
            h->prof_ms[c] = 0.0;
            h->prof_n[c] = 0;
        }
    }
    h->prof_on = enable != 0;
    return DNSLAB_OK;
}

int dnslab_profile_read(dnslab_t *h, double *ms, int64_t *launches)
{
    if (!h || !ms || !launches) return DNSLAB_EINVAL;
    if (int rc = prof_drain(h)) return rc;
    for (int c = 0; c < DNSLAB_NCLASS; ++c) {
        ms[c] = h->prof_ms[c];
        launches[c] = h->prof_n[c];
    }
    return DNSLAB_OK;
}

int dnslab_particles_attach(dnslab_t *h, int64_t n, double *state, double rho_f, const double g[3])
{
    if (!h || n < 0) return DNSLAB_EINVAL;
    if (n > 0 && (!state || !g || !(rho_f > 0) || !(h->P.nu > 0))) return DNSLAB_EINVAL;
    h->np = n;
    h->pstate = n > 0 ? state : nullptr;
    if (n > 0) {
        h->prho_f = rho_f;
        for (int c = 0; c < 3; ++c) h->pgrav[c] = g[c];
    }
    return DNSLAB_OK;
}

int dnslab_courant(dnslab_t *h, double *co)
{
    if (!h || !co) return DNSLAB_EINVAL;
    unsigned long long *res = reinterpret_cast<unsigned long long *>(h->W); // W is scratch outside a solve
    CK(cudaMemsetAsync(res, 0, sizeof(*res), h->stream));
    {
        ProfScope ps(h, DNSLAB_K_REDUCE);
        size_t g = (h->n + 255) / 256;
        if (g > (size_t)4 * h->nsm) g = (size_t)4 * h->nsm; // few, long-running blocks: the shared threshold settles early
        dnsred::k_courant<<<(unsigned)g, 256, 0, h->stream>>>(h->Q[0], h->Q[1], h->Q[2], h->n, h->P.dx, h->P.dy, h->P.dz, res);
        if (int rc = check_launch(h)) return rc;
    }
    double rate = 0.0;
    CK(cudaMemcpyAsync(&rate, res, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    *co = rate * h->P.dt;
    return DNSLAB_OK;
}

int dnslab_set_dt(dnslab_t *h, double dt)
{
    if (!h || !(dt > 0)) return DNSLAB_EINVAL;
    h->P.dt = dt;
    return DNSLAB_OK;
}

int dnslab_scalar_stats(dnslab_t *h, const int32_t lo[3], const int32_t size[3], double out[3])
{
    if (!h || !lo || !size || !out) return DNSLAB_EINVAL;
    const int nn[3] = {h->P.nx, h->P.ny, h->P.nz};
    dnsred::BoxArgs a;
    a.c = h->Q[3];
    a.face = h->face;
    a.nx = nn[0]; a.ny = nn[1]; a.nz = nn[2];
    a.count = 1;
    for (int d = 0; d < 3; ++d) {
        if (size[d] < 1 || size[d] > nn[d]) return DNSLAB_EINVAL;
        a.lo[d] = ((lo[d] % nn[d]) + nn[d]) % nn[d];
        a.size[d] = size[d];
        a.count *= (size_t)size[d];
    }
    // W (scratch outside a solve): res[0..3], then 2 G partials; a block takes whole rows of the box
    double *res = h->W, *part = h->W + 8;
    const unsigned rows = (unsigned)size[1] * (unsigned)size[2];
    unsigned G = (unsigned)(16 * h->nsm);
    if (G > rows) G = rows;
    if (2 * (size_t)G + 8 > h->n) G = (unsigned)((h->n - 8) / 2);
    const unsigned rpb = (rows + G - 1) / G;
    G = (rows + rpb - 1) / rpb;
    {
        ProfScope ps(h, DNSLAB_K_REDUCE);
        dnsred::k_box_partial<0><<<G, 256, 0, h->stream>>>(a, rows, rpb, res, part);
        if (int rc = check_launch(h)) return rc;
    }
    dnsred::k_box_final<0><<<1, 256, 0, h->stream>>>(part, (int)G, res);
    if (int rc = check_launch(h)) return rc;
    {
        ProfScope ps(h, DNSLAB_K_REDUCE);
        dnsred::k_box_partial<1><<<G, 256, 0, h->stream>>>(a, rows, rpb, res, part);
        if (int rc = check_launch(h)) return rc;
    }
    dnsred::k_box_final<1><<<1, 256, 0, h->stream>>>(part, (int)G, res);
    if (int rc = check_launch(h)) return rc;
    CK(cudaMemcpyAsync(out, res, 3 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return DNSLAB_OK;
}

int dnslab_destroy(dnslab_t *h)
{
    if (!h) return DNSLAB_EINVAL;
    prof_drain(h);
    delete h->prof;
    delete h;
    return DNSLAB_OK;
}

} // extern "C"

// ---- dnslab_scalar_stats_static: the one entry point that needs no device memory from anybody ---------------------------
// Its scratch (one sum and one count per row of the box) lives in this array, which is part of the library's image: every
// GPU that loads libdnslab.so carries these 1 MiB from the moment the module is loaded until the process exits, used or
// not.  In HOST code the name g_static_scratch is only a handle for the symbol, not a device address -- handing it to a
// kernel would fault, or quietly scribble over host memory on systems where the GPU can reach it -- so the host asks
// the runtime for the address once per device (static_scratch below) and passes that to the kernels.
static __device__ __align__(256) double g_static_scratch[2 * DNSLAB_STATIC_MAX_ROWS];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
double *g_static_ptr[STATIC_MAX_DEVICES]; // device address of g_static_scratch on each device; null until its first call

// Address of the static scratch array on the CURRENT device; looked up (and the device checked) on the first call
// made with that device current, remembered afterwards.
int static_scratch(double **ptr)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return DNSLAB_EARCH;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return DNSLAB_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (g_static_ptr[dev] == nullptr) {
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) return DNSLAB_EARCH;
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || p == nullptr) return DNSLAB_ECUDA;
        g_static_ptr[dev] = static_cast<double *>(p);
    }
    *ptr = g_static_ptr[dev];
    return DNSLAB_OK;
}
} // namespace

extern "C" int dnslab_scalar_stats_static(const double *c, const uint8_t *mask, int32_t nx, int32_t ny, int32_t nz, const int32_t lo[3],
                                          const int32_t size[3], void *cuda_stream, double *out)
{
    if (!c || !lo || !size || !out) return DNSLAB_EINVAL;
    if (!pow2(nx) || !pow2(ny) || !pow2(nz) || nx < 8 || nx > 2048 || ny < 8 || ny > 1024 || nz < 8 || nz > 1024) return DNSLAB_EINVAL;
    const int nn[3] = {nx, ny, nz};
    dnsred::BoxArgs a;
    a.c = c;
    a.face = mask;
    a.nx = nx; a.ny = ny; a.nz = nz;
    a.count = 1;
    for (int d = 0; d < 3; ++d) {
        if (size[d] < 1 || size[d] > nn[d]) return DNSLAB_EINVAL;
        a.lo[d] = ((lo[d] % nn[d]) + nn[d]) % nn[d];
        a.size[d] = size[d];
        a.count *= (size_t)size[d];
    }
    const size_t rows = (size_t)size[1] * (size_t)size[2];
    if (rows > (size_t)DNSLAB_STATIC_MAX_ROWS) return DNSLAB_ELIMIT;
    double *part = nullptr;
    if (int rc = static_scratch(&part)) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned R = (unsigned)rows, G = (R + 7u) / 8u;
    // nothing in `part` has to start at zero: each pass writes slots 0..R-1 (and R..2R-1) before k_box_final reads exactly those
    dnsred::k_box_rows<0><<<G, 256, 0, st>>>(a, R, out, part);
    dnsred::k_box_final<0><<<1, 256, 0, st>>>(part, (int)R, out);
    dnsred::k_box_rows<1><<<G, 256, 0, st>>>(a, R, out, part);
    dnsred::k_box_final<1><<<1, 256, 0, st>>>(part, (int)R, out);
    return cudaPeekAtLastError() == cudaSuccess ? DNSLAB_OK : DNSLAB_ECUDA;
}
