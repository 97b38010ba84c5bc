/*
 * oracle/dnsref.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle of the DNSLABIB Navier-Stokes time step
 * (arxiv 2204.02107), written from the paper's text only.  It shares no code,
 * header, table generator or helper with the CUDA path under
 * paper_2204_02107_b200/csrc/, and neither imports the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call it.
 *
 * Citations are PAPER.md:<line> (+ section / equation).  Readings of silent or
 * ambiguous passages are numbered R1.. in DESIGN.md ("Readings of the paper").
 *
 * Layout: fp64 arrays, x fastest: idx = i + nx*(j + ny*k), all axes periodic
 * ("the present solver is periodic").
 *
 * Every function below is pinned by tests/test_oracle_pins.py to something
 * other than itself (dense operators, brute-force solves, closed forms,
 * exact amplification factors, invariants).  No function is "parity unpinned".
 *
 * The loops are ordinary index-order loops; the only concession to run time
 * is "#pragma omp parallel for" over the outermost (k) loop of independent
 * iterations -- no blocking, fusion or reordering of the arithmetic.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define DNSREF_OK 0
#define DNSREF_EINVAL (-1)
#define DNSREF_ENOMEM (-2)

typedef struct {
    int32_t nx, ny, nz;
    double dx, dy, dz;
    double nu, alpha_c, dt;
    double body[3];
    int32_t n_piter; /* eq. 9 iterations, PAPER.md:104 (paper: 4) */
    uint32_t flags;  /* bit0: eq. 6 filter at the end of each step (NEXT-1); bit1: project every RK stage */
} dnsref_params_t;

typedef struct {
    int32_t lo[3], size[3]; /* index box, wraps modulo N */
    double B[3];            /* eq. 5 smoothness per axis; <=0: binary box */
    double u_set[3], c_set, tau_f;
    uint32_t comps; /* bit0..3: force u,v,w,c */
} dnsref_source_t;

typedef struct {
    dnsref_params_t P;
    int64_t n;
    uint8_t *beta;
    int nsrc;
    dnsref_source_t *src;
    double **sx, **sy, **sz; /* eq. 5 one-dimensional factors, per source */
    double *q[4];            /* u, v, w, c  (state Q^n) */
    double *p;               /* pressure (state: warm start of eq. 9) */
    double *qs[4], *qc[4], *f[4], *d, *r, *re, *im;
    /* NEXT-4: Lagrangian particles attached by the caller (state lives in the caller's array) */
    int64_t np;
    double *part; /* 8 arrays of np doubles: x, y, z, u, v, w, d, rho_p */
    double rho_f, grav[3];
} dnsref_t;

int dnsref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static inline int wrap(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }
static inline int wrapm(int i, int n) { return ((i % n) + n) % n; } /* any offset, any n >= 1 */
#define IDX(i, j, k) ((int64_t)(i) + (int64_t)nx * ((int64_t)(j) + (int64_t)ny * (int64_t)(k)))

/* ------------------------------------------------------------------------
 * eq. 5: one factor of the tanh window,
 *   S_a(x) = 1/2 (1 - tanh(B [ |x-xc|/(W/2) - (W/2)/|x-xc| ])).
 * Reading R10: cell centres x_i = i*d; the box covers cells lo..lo+size-1,
 * xc = (lo + (size-1)/2) d, W = size*d; |x-xc| by minimum image (periodic);
 * at x = xc the bracket -> -inf, tanh -> -1, S = 1.  B <= 0: binary, S = 1
 * inside the index box and 0 outside.
 * ---------------------------------------------------------------------- */
void dnsref_source_table(int n, double d, int lo, int size, double B, double *out)
{
    for (int i = 0; i < n; ++i) {
        if (B <= 0.0) {
            int rel = ((i - lo) % n + n) % n;
            out[i] = rel < size ? 1.0 : 0.0;
        } else {
            double L = n * d;
            double xc = (lo + 0.5 * (size - 1)) * d;
            double W2 = 0.5 * size * d;
            double r = fabs(i * d - xc);
            r = fmod(r, L);
            if (r > 0.5 * L) r = L - r;
            if (r == 0.0)
                out[i] = 1.0;
            else
                out[i] = 0.5 * (1.0 - tanh(B * (r / W2 - W2 / r)));
        }
    }
}

/* ------------------------------------------------------------------------
 * a1: right-hand side F(Q) of eqs. 2-3, one RK stage.
 *   convection: skew-symmetric 2nd-order central form (reading R3/R4)
 *       C(phi) = 1/2 sum_a [ delta_a(u_a phi) + u_a delta_a phi ]
 *   diffusion: nu * sum_a delta2_a phi  (u,v,w);  for c the face-weighted form
 *       alpha_c sum_a [ b+ (c[+a]-c) - b- (c-c[-a]) ]/D_a^2,  b+- = beta*beta[+-a]
 *       which realises dc/dn = 0 on solid faces (eq. 4; reading R5)
 *   body force b, source relaxation S (phi_set - phi)/tau_f
 *   output masked by select: beta ? F : +0.0  (reading R7)
 * ---------------------------------------------------------------------- */
void dnsref_rhs(const dnsref_t *h, const double *u, const double *v, const double *w, const double *c,
                double *Fu, double *Fv, double *Fw, double *Fc)
{
    const int nx = h->P.nx, ny = h->P.ny, nz = h->P.nz;
    const double dx = h->P.dx, dy = h->P.dy, dz = h->P.dz;
    const double nu = h->P.nu, ac = h->P.alpha_c;
    const double *q[4] = {u, v, w, c};
    double *F[4] = {Fu, Fv, Fw, Fc};
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                int64_t o = IDX(i, j, k);
                if (!h->beta[o]) {
                    for (int m = 0; m < 4; ++m) F[m][o] = 0.0;
                    continue;
                }
                int64_t xp = IDX(wrap(i + 1, nx), j, k), xm = IDX(wrap(i - 1, nx), j, k);
                int64_t yp = IDX(i, wrap(j + 1, ny), k), ym = IDX(i, wrap(j - 1, ny), k);
                int64_t zp = IDX(i, j, wrap(k + 1, nz)), zm = IDX(i, j, wrap(k - 1, nz));
                for (int m = 0; m < 4; ++m) {
                    const double *f = q[m];
                    double conv = 0.0;
                    conv += (u[xp] * f[xp] - u[xm] * f[xm]) / (2.0 * dx) + u[o] * (f[xp] - f[xm]) / (2.0 * dx);
                    conv += (v[yp] * f[yp] - v[ym] * f[ym]) / (2.0 * dy) + v[o] * (f[yp] - f[ym]) / (2.0 * dy);
                    conv += (w[zp] * f[zp] - w[zm] * f[zm]) / (2.0 * dz) + w[o] * (f[zp] - f[zm]) / (2.0 * dz);
                    double diff;
                    if (m < 3) {
                        diff = nu * ((f[xp] - 2.0 * f[o] + f[xm]) / (dx * dx) + (f[yp] - 2.0 * f[o] + f[ym]) / (dy * dy) +
                                     (f[zp] - 2.0 * f[o] + f[zm]) / (dz * dz));
                    } else {
                        const uint8_t *b = h->beta;
                        double bxp = b[o] * b[xp], bxm = b[o] * b[xm];
                        double byp = b[o] * b[yp], bym = b[o] * b[ym];
                        double bzp = b[o] * b[zp], bzm = b[o] * b[zm];
                        diff = ac * ((bxp * (f[xp] - f[o]) - bxm * (f[o] - f[xm])) / (dx * dx) +
                                     (byp * (f[yp] - f[o]) - bym * (f[o] - f[ym])) / (dy * dy) +
                                     (bzp * (f[zp] - f[o]) - bzm * (f[o] - f[zm])) / (dz * dz));
                    }
                    double val = -0.5 * conv + diff;
                    if (m < 3) val += h->P.body[m];
                    for (int s = 0; s < h->nsrc; ++s) {
                        const dnsref_source_t *S = &h->src[s];
                        if (!(S->comps & (1u << m))) continue;
                        double Sv = h->sx[s][i] * h->sy[s][j] * h->sz[s][k];
                        if (Sv == 0.0) continue;
                        double set = m < 3 ? S->u_set[m] : S->c_set;
                        val += Sv * (set - f[o]) / S->tau_f;
                    }
                    F[m][o] = val;
                }
            }
}

/* a4: divergence by central differences (eq. 7; reading R11) */
void dnsref_div(const dnsref_t *h, const double *u, const double *v, const double *w, double *d)
{
    const int nx = h->P.nx, ny = h->P.ny, nz = h->P.nz;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                d[IDX(i, j, k)] = (u[IDX(wrap(i + 1, nx), j, k)] - u[IDX(wrap(i - 1, nx), j, k)]) / (2.0 * h->P.dx) +
                                  (v[IDX(i, wrap(j + 1, ny), k)] - v[IDX(i, wrap(j - 1, ny), k)]) / (2.0 * h->P.dy) +
                                  (w[IDX(i, j, wrap(k + 1, nz))] - w[IDX(i, j, wrap(k - 1, nz))]) / (2.0 * h->P.dz);
            }
}

/* ------------------------------------------------------------------------
 * One-dimensional DFTs.  sign = -1 forward, +1 inverse; unnormalised.
 * dft1d: the definition, O(n^2).  fft1d: textbook iterative radix-2
 * decimation in time (bit reversal, then log2 n butterfly levels), every
 * twiddle computed directly from cos/sin of its own angle.
 * ---------------------------------------------------------------------- */
void dnsref_dft1d(int n, const double *re, const double *im, double *ore, double *oim, int sign)
{
    for (int k = 0; k < n; ++k) {
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < n; ++j) {
            int64_t jk = ((int64_t)j * k) % n;
            double a = sign * 2.0 * M_PI * (double)jk / n;
            double cr = cos(a), ci = sin(a);
            sr += re[j] * cr - im[j] * ci;
            si += re[j] * ci + im[j] * cr;
        }
        ore[k] = sr;
        oim[k] = si;
    }
}

void dnsref_fft1d(int n, double *re, double *im, int sign)
{
    if (n & (n - 1)) { /* not a power of two: fall back on the definition */
        double *t = (double *)malloc(sizeof(double) * 2 * n);
        dnsref_dft1d(n, re, im, t, t + n, sign);
        memcpy(re, t, sizeof(double) * n);
        memcpy(im, t + n, sizeof(double) * n);
        free(t);
        return;
    }
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double t = re[i]; re[i] = re[j]; re[j] = t;
            t = im[i]; im[i] = im[j]; im[j] = t;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1;
        for (int j = 0; j < half; ++j) { /* twiddle j of this level, then its butterfly in every block of the level */
            double a = sign * 2.0 * M_PI * (double)j / len;
            double wr = cos(a), wi = sin(a);
            for (int s = 0; s < n; s += len) {
                double xr = re[s + j + half] * wr - im[s + j + half] * wi;
                double xi = re[s + j + half] * wi + im[s + j + half] * wr;
                re[s + j + half] = re[s + j] - xr;
                im[s + j + half] = im[s + j] - xi;
                re[s + j] += xr;
                im[s + j] += xi;
            }
        }
    }
}

/* 3-D DFT: apply the 1-D transform along x, then y, then z. Unnormalised. */
void dnsref_fft3(int nx, int ny, int nz, double *re, double *im, int sign)
{
#pragma omp parallel
    {
        int nmax = nx > ny ? nx : ny;
        if (nz > nmax) nmax = nz;
        double *lr = (double *)malloc(sizeof(double) * 2 * nmax), *li = lr + nmax;
#pragma omp for schedule(static)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                dnsref_fft1d(nx, re + IDX(0, j, k), im + IDX(0, j, k), sign);
#pragma omp for schedule(static)
        for (int k = 0; k < nz; ++k)
            for (int i = 0; i < nx; ++i) {
                for (int j = 0; j < ny; ++j) { lr[j] = re[IDX(i, j, k)]; li[j] = im[IDX(i, j, k)]; }
                dnsref_fft1d(ny, lr, li, sign);
                for (int j = 0; j < ny; ++j) { re[IDX(i, j, k)] = lr[j]; im[IDX(i, j, k)] = li[j]; }
            }
#pragma omp for schedule(static)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                for (int k = 0; k < nz; ++k) { lr[k] = re[IDX(i, j, k)]; li[k] = im[IDX(i, j, k)]; }
                dnsref_fft1d(nz, lr, li, sign);
                for (int k = 0; k < nz; ++k) { re[IDX(i, j, k)] = lr[k]; im[IDX(i, j, k)] = li[k]; }
            }
        free(lr);
    }
}

/* Eigenvalue of sum_a delta_a delta_a on mode (kx,ky,kz): the "discrete
 * modified wavenumber" (north_star; reading R12):
 *   lambda = - sum_a sin^2(2 pi k_a / N_a) / D_a^2 */
double dnsref_eig(const dnsref_params_t *P, int kx, int ky, int kz)
{
    double sx = sin(2.0 * M_PI * kx / P->nx) / P->dx;
    double sy = sin(2.0 * M_PI * ky / P->ny) / P->dy;
    double sz = sin(2.0 * M_PI * kz / P->nz) / P->dz;
    return -(sx * sx + sy * sy + sz * sz);
}

/* a5 (one solve): p = F^-1[ F[r] / lambda ]; the modes with 2 k_a = 0 (mod N_a)
 * for all a -- the null space of the operator -- are set to 0 (reading R13). */
int dnsref_poisson_solve(dnsref_t *h, const double *r, double *p)
{
    const int nx = h->P.nx, ny = h->P.ny, nz = h->P.nz;
    const int64_t n = h->n;
    double *re = h->re, *im = h->im;
#pragma omp parallel for schedule(static)
    for (int64_t o = 0; o < n; ++o) { re[o] = r[o]; im[o] = 0.0; }
    dnsref_fft3(nx, ny, nz, re, im, -1);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                int64_t o = IDX(i, j, k);
                int null = ((2 * i) % nx == 0) && ((2 * j) % ny == 0) && ((2 * k) % nz == 0);
                if (null) {
                    re[o] = 0.0; im[o] = 0.0;
                } else {
                    double lam = dnsref_eig(&h->P, i, j, k);
                    re[o] /= lam; im[o] /= lam;
                }
            }
    dnsref_fft3(nx, ny, nz, re, im, +1);
#pragma omp parallel for schedule(static)
    for (int64_t o = 0; o < n; ++o) p[o] = re[o] / (double)n;
    return DNSREF_OK;
}

/* Right-hand side of eq. 9 (reading R14):
 *   r = d + sum_a delta_a[ (1-beta) delta_a p ] , central differences. */
void dnsref_poisson_rhs(const dnsref_t *h, const double *d, const double *p, double *r)
{
    const int nx = h->P.nx, ny = h->P.ny, nz = h->P.nz;
    const uint8_t *b = h->beta;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                int ip = wrap(i + 1, nx), im = wrap(i - 1, nx), ipp = wrap(i + 2, nx), imm = wrap(i - 2, nx);
                int jp = wrap(j + 1, ny), jm = wrap(j - 1, ny), jpp = wrap(j + 2, ny), jmm = wrap(j - 2, ny);
                int kp = wrap(k + 1, nz), km = wrap(k - 1, nz), kpp = wrap(k + 2, nz), kmm = wrap(k - 2, nz);
                /* g_a = (1-beta) delta_a p at the +1 and -1 neighbours along a */
                double gxp = (1.0 - b[IDX(ip, j, k)]) * (p[IDX(ipp, j, k)] - p[IDX(i, j, k)]) / (2.0 * h->P.dx);
                double gxm = (1.0 - b[IDX(im, j, k)]) * (p[IDX(i, j, k)] - p[IDX(imm, j, k)]) / (2.0 * h->P.dx);
                double gyp = (1.0 - b[IDX(i, jp, k)]) * (p[IDX(i, jpp, k)] - p[IDX(i, j, k)]) / (2.0 * h->P.dy);
                double gym = (1.0 - b[IDX(i, jm, k)]) * (p[IDX(i, j, k)] - p[IDX(i, jmm, k)]) / (2.0 * h->P.dy);
                double gzp = (1.0 - b[IDX(i, j, kp)]) * (p[IDX(i, j, kpp)] - p[IDX(i, j, k)]) / (2.0 * h->P.dz);
                double gzm = (1.0 - b[IDX(i, j, km)]) * (p[IDX(i, j, k)] - p[IDX(i, j, kmm)]) / (2.0 * h->P.dz);
                r[IDX(i, j, k)] = d[IDX(i, j, k)] + ((gxp - gxm) / (2.0 * h->P.dx) + (gyp - gym) / (2.0 * h->P.dy) +
                                                     (gzp - gzm) / (2.0 * h->P.dz));
            }
}

/* a6: u = beta ? u* - delta_a p : +0.0 (eq. 8) */
void dnsref_project(const dnsref_t *h, const double *us, const double *vs, const double *ws, const double *p,
                    double *u, double *v, double *w)
{
    const int nx = h->P.nx, ny = h->P.ny, nz = h->P.nz;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                int64_t o = IDX(i, j, k);
                if (!h->beta[o]) { u[o] = 0.0; v[o] = 0.0; w[o] = 0.0; continue; }
                u[o] = us[o] - (p[IDX(wrap(i + 1, nx), j, k)] - p[IDX(wrap(i - 1, nx), j, k)]) / (2.0 * h->P.dx);
                v[o] = vs[o] - (p[IDX(i, wrap(j + 1, ny), k)] - p[IDX(i, wrap(j - 1, ny), k)]) / (2.0 * h->P.dy);
                w[o] = ws[o] - (p[IDX(i, j, wrap(k + 1, nz))] - p[IDX(i, j, wrap(k - 1, nz))]) / (2.0 * h->P.dz);
            }
}

/* NEXT-1, eq. 6: explicit filter applied "at the end of each timestep" to u, v, w, c:
 *     out = beta ? in + sum_a gamma_a d6_a(in) : +0.0,     gamma_a = Delta_a^6 / pi^6  (as printed),
 * with d6_a the 2nd-order central 7-point stencil of the sixth derivative along axis a,
 *     d6_a f = (f[-3] - 6 f[-2] + 15 f[-1] - 20 f[0] + 15 f[+1] - 6 f[+2] + f[+3]) / Delta_a^6,
 * periodic (reading R23 in DESIGN.md: the paper does not say how the derivative is taken; "2nd order
 * central" is its stated discretisation).  Delta_a^6 cancels: the weight of each stencil
 * sum is 1/pi^6.  The stencil reads solid cells (which hold +0.0) like any other cell; the result is
 * masked by the select of PAPER.md:58.  A Fourier mode with angles theta_a is multiplied by
 *     G = 1 - (64/pi^6) sum_a sin^6(theta_a/2)                                      (pin P15).
 * in and out must not alias. */
void dnsref_filter(const dnsref_t *h, const double *in, double *out)
{
    const int nx = h->P.nx, ny = h->P.ny, nz = h->P.nz;
    const double pi = 3.14159265358979323846;
    const double g = 1.0 / (pi * pi * pi * pi * pi * pi);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const int64_t o = IDX(i, j, k);
                if (!h->beta[o]) { out[o] = 0.0; continue; }
                const double f0 = in[o];
                const double sx = in[IDX(wrapm(i - 3, nx), j, k)] - 6.0 * in[IDX(wrapm(i - 2, nx), j, k)] +
                                  15.0 * in[IDX(wrapm(i - 1, nx), j, k)] - 20.0 * f0 + 15.0 * in[IDX(wrapm(i + 1, nx), j, k)] -
                                  6.0 * in[IDX(wrapm(i + 2, nx), j, k)] + in[IDX(wrapm(i + 3, nx), j, k)];
                const double sy = in[IDX(i, wrapm(j - 3, ny), k)] - 6.0 * in[IDX(i, wrapm(j - 2, ny), k)] +
                                  15.0 * in[IDX(i, wrapm(j - 1, ny), k)] - 20.0 * f0 + 15.0 * in[IDX(i, wrapm(j + 1, ny), k)] -
                                  6.0 * in[IDX(i, wrapm(j + 2, ny), k)] + in[IDX(i, wrapm(j + 3, ny), k)];
                const double sz = in[IDX(i, j, wrapm(k - 3, nz))] - 6.0 * in[IDX(i, j, wrapm(k - 2, nz))] +
                                  15.0 * in[IDX(i, j, wrapm(k - 1, nz))] - 20.0 * f0 + 15.0 * in[IDX(i, j, wrapm(k + 1, nz))] -
                                  6.0 * in[IDX(i, j, wrapm(k + 2, nz))] + in[IDX(i, j, wrapm(k + 3, nz))];
                out[o] = f0 + g * ((sx + sy) + sz);
            }
}

/* The pressure stage: divergence, n_piter iterations of eq. 9 warm-started
 * from p, then the correction.  us.. and u.. may alias. */
static void pressure_stage(dnsref_t *h, double *us, double *vs, double *ws, double *p)
{
    dnsref_div(h, us, vs, ws, h->d);
    for (int it = 0; it < h->P.n_piter; ++it) {
        dnsref_poisson_rhs(h, h->d, p, h->r);
        dnsref_poisson_solve(h, h->r, p);
    }
    dnsref_project(h, us, vs, ws, p, us, vs, ws);
}

int dnsref_particles_step(const dnsref_t *h, int64_t n, double *state, double rho_f, const double g[3]);

/* ------------------------------------------------------------------------
 * One full time step (PAPER.md:43 RK4 + projection once per step):
 *   Qc = Qn; Qs = Qn
 *   for s = 1..4: F = RHS(Qs); Qc += b_s dt F; if s<4: Qs = Qn + a_s dt F
 *   d = div(Qc); p <- eq. 9 x n_piter; u = beta ? Qc.u - grad p : 0; c = Qc.c
 * Classical RK4: a = (1/2,1/2,1), b = (1/6,1/3,1/3,1/6) (reading R1).
 * flags bit1 (NEXT-2): each stage field Qs (s = 2..4) is projected too.
 * flags bit0 (NEXT-1): u, v, w, c are filtered (eq. 6) after the projection.
 * ---------------------------------------------------------------------- */
int dnsref_step(dnsref_t *h, int nsteps)
{
    static const double a[3] = {0.5, 0.5, 1.0};
    static const double b[4] = {1.0 / 6.0, 1.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0};
    if (!h || nsteps < 0) return DNSREF_EINVAL;
    const int64_t n = h->n;
    const double dt = h->P.dt;
    for (int it = 0; it < nsteps; ++it) {
        for (int m = 0; m < 4; ++m) {
            memcpy(h->qc[m], h->q[m], sizeof(double) * n);
            memcpy(h->qs[m], h->q[m], sizeof(double) * n);
        }
        for (int s = 0; s < 4; ++s) {
            dnsref_rhs(h, h->qs[0], h->qs[1], h->qs[2], h->qs[3], h->f[0], h->f[1], h->f[2], h->f[3]);
            for (int m = 0; m < 4; ++m) {
#pragma omp parallel for schedule(static)
                for (int64_t o = 0; o < n; ++o) {
                    h->qc[m][o] = h->qc[m][o] + (b[s] * dt) * h->f[m][o];
                    if (s < 3) h->qs[m][o] = h->q[m][o] + (a[s] * dt) * h->f[m][o];
                }
            }
            if (s < 3 && (h->P.flags & 2u)) {
                /* NEXT-2 variant: project the stage velocity, using a scratch pressure */
                double *ps = (double *)malloc(sizeof(double) * n);
                if (!ps) return DNSREF_ENOMEM;
                memcpy(ps, h->p, sizeof(double) * n);
                pressure_stage(h, h->qs[0], h->qs[1], h->qs[2], ps);
                free(ps);
            }
        }
        pressure_stage(h, h->qc[0], h->qc[1], h->qc[2], h->p);
        for (int m = 0; m < 4; ++m) {
            if (h->P.flags & 1u) dnsref_filter(h, h->qc[m], h->q[m]); /* eq. 6, end of step (NEXT-1) */
            else memcpy(h->q[m], h->qc[m], sizeof(double) * n);
        }
        if (h->np > 0) dnsref_particles_step(h, h->np, h->part, h->rho_f, h->grav); /* NEXT-4, after the fluid step */
    }
    return DNSREF_OK;
}

/* ------------------------------------------------------------------------
 * NEXT-4: Lagrangian particles, eqs. 10-13, advanced by one fluid time step dt with
 * the velocity field given (the paper's "SolveDrops.m" runs after the fluid step):
 *     tau_p = rho_p d^2 / (18 rho_f nu)                                   (eq. 11; d enters as in Stokes' law)
 *     Re_p  = |u_f - u_p| d / nu,   C_d = 1 + Re_p^(2/3) / 6              (eqs. 12, 13)
 *     du_p/dt = (C_d / tau_p)(u_f - u_p) + g                              (eq. 10)
 * "solved using the implicit Euler method".  Readings (R26-R28): u_f is the
 * trilinear interpolation of the collocated velocity (cell centres at x_i = i Delta, periodic); C_d is
 * evaluated with the velocities at the old time level, the drag term is implicit in u_p:
 *     u_p' = (u_p + dt (k u_f + g)) / (1 + dt k),  k = C_d / tau_p;       x_p' = x_p + dt u_p'  (wrapped into [0, L)).
 * state: 8 arrays of n doubles, x y z u v w d rho_p.  Solid cells hold u = 0 and take part in the
 * interpolation like any other cell; there is no deposition model in the paper.
 * ---------------------------------------------------------------------- */
static double interp3(const dnsref_t *h, const double *f, double x, double y, double z)
{
    const int nx = h->P.nx, ny = h->P.ny, nz = h->P.nz;
    const double gx = x / h->P.dx, gy = y / h->P.dy, gz = z / h->P.dz;
    const double fx = floor(gx), fy = floor(gy), fz = floor(gz);
    const double ax = gx - fx, ay = gy - fy, az = gz - fz;
    const int i0 = wrapm((int)fx, nx), j0 = wrapm((int)fy, ny), k0 = wrapm((int)fz, nz);
    const int i1 = wrapm(i0 + 1, nx), j1 = wrapm(j0 + 1, ny), k1 = wrapm(k0 + 1, nz);
    const double c00 = f[IDX(i0, j0, k0)] * (1.0 - ax) + f[IDX(i1, j0, k0)] * ax;
    const double c10 = f[IDX(i0, j1, k0)] * (1.0 - ax) + f[IDX(i1, j1, k0)] * ax;
    const double c01 = f[IDX(i0, j0, k1)] * (1.0 - ax) + f[IDX(i1, j0, k1)] * ax;
    const double c11 = f[IDX(i0, j1, k1)] * (1.0 - ax) + f[IDX(i1, j1, k1)] * ax;
    const double c0 = c00 * (1.0 - ay) + c10 * ay, c1 = c01 * (1.0 - ay) + c11 * ay;
    return c0 * (1.0 - az) + c1 * az;
}

int dnsref_particles_step(const dnsref_t *h, int64_t n, double *state, double rho_f, const double g[3])
{
    if (!h || n < 0 || (n > 0 && !state) || !g || !(rho_f > 0) || !(h->P.nu > 0)) return DNSREF_EINVAL;
    double *px = state, *py = state + n, *pz = state + 2 * n, *pu = state + 3 * n, *pv = state + 4 * n, *pw = state + 5 * n;
    const double *pd = state + 6 * n, *pr = state + 7 * n;
    const double dt = h->P.dt, nu = h->P.nu;
    const double len[3] = {h->P.nx * h->P.dx, h->P.ny * h->P.dy, h->P.nz * h->P.dz};
    for (int64_t q = 0; q < n; ++q) {
        const double uf = interp3(h, h->q[0], px[q], py[q], pz[q]);
        const double vf = interp3(h, h->q[1], px[q], py[q], pz[q]);
        const double wf = interp3(h, h->q[2], px[q], py[q], pz[q]);
        const double tau = pr[q] * pd[q] * pd[q] / (18.0 * rho_f * nu);
        const double rel = sqrt((uf - pu[q]) * (uf - pu[q]) + (vf - pv[q]) * (vf - pv[q]) + (wf - pw[q]) * (wf - pw[q]));
        const double rep = rel * pd[q] / nu;
        const double cd = 1.0 + cbrt(rep * rep) / 6.0;
        const double k = cd / tau;
        pu[q] = (pu[q] + dt * (k * uf + g[0])) / (1.0 + dt * k);
        pv[q] = (pv[q] + dt * (k * vf + g[1])) / (1.0 + dt * k);
        pw[q] = (pw[q] + dt * (k * wf + g[2])) / (1.0 + dt * k);
        double xn[3] = {px[q] + dt * pu[q], py[q] + dt * pv[q], pz[q] + dt * pw[q]};
        for (int a = 0; a < 3; ++a) {
            xn[a] = xn[a] - floor(xn[a] / len[a]) * len[a];
            if (!(xn[a] < len[a])) xn[a] = 0.0; /* rounding at the upper edge */
        }
        px[q] = xn[0]; py[q] = xn[1]; pz[q] = xn[2];
    }
    return DNSREF_OK;
}

/* Particles to be advanced at the end of every dnsref_step (n = 0 detaches); the array stays the caller's. */
int dnsref_particles_attach(dnsref_t *h, int64_t n, double *state, double rho_f, const double g[3])
{
    if (!h || n < 0) return DNSREF_EINVAL;
    if (n > 0 && (!state || !g || !(rho_f > 0) || !(h->P.nu > 0))) return DNSREF_EINVAL;
    h->np = n;
    h->part = n > 0 ? state : NULL;
    if (n > 0) { h->rho_f = rho_f; h->grav[0] = g[0]; h->grav[1] = g[1]; h->grav[2] = g[2]; }
    return DNSREF_OK;
}

/* ------------------------------------------------------------------------
 * NEXT-3: the two global reductions the paper's main loop uses.
 *
 * Courant number of the current state ("the user also specifies the maximum Courant number, as
 * the implementation utilizes dynamic time stepping (in AdjustDt.m)"); the formula is not printed -- reading R24:
 *     Co = dt * max over all cells of ( |u|/dx + |v|/dy + |w|/dz ).
 * The caller turns it into the next dt (dt_new = Co_max / (Co/dt)) and sets it with dnsref_set_dt.
 * ---------------------------------------------------------------------- */
double dnsref_courant(const dnsref_t *h)
{
    double best = 0.0;
    for (int64_t o = 0; o < h->n; ++o) {
        const double r = fabs(h->q[0][o]) / h->P.dx + fabs(h->q[1][o]) / h->P.dy + fabs(h->q[2][o]) / h->P.dz;
        if (r > best) best = r;
    }
    return best * h->P.dt;
}

int dnsref_set_dt(dnsref_t *h, double dt)
{
    if (!h || !(dt > 0)) return DNSREF_EINVAL;
    h->P.dt = dt;
    return DNSREF_OK;
}

/* Mean and standard deviation of the scalar over the fluid cells of an index box that wraps modulo N
 * ("the mean CO2 content as a function of simulation time ... The standard deviation is
 * plotted as well") -- reading R25: population standard deviation sqrt(sum (c - mean)^2 / count) over the
 * cells with beta = 1 inside the box; two passes, plain index-order sums.  out[0] = mean, out[1] = std,
 * out[2] = count.  A box without fluid cells gives 0, 0, 0. */
int dnsref_scalar_stats(const dnsref_t *h, const int32_t lo[3], const int32_t size[3], double out[3])
{
    if (!h || !lo || !size || !out) return DNSREF_EINVAL;
    const int nx = h->P.nx, ny = h->P.ny, nz = h->P.nz;
    if (size[0] < 1 || size[1] < 1 || size[2] < 1 || size[0] > nx || size[1] > ny || size[2] > nz) return DNSREF_EINVAL;
    double sum = 0.0;
    int64_t cnt = 0;
    for (int k = 0; k < size[2]; ++k)
        for (int j = 0; j < size[1]; ++j)
            for (int i = 0; i < size[0]; ++i) {
                const int64_t o = IDX(wrapm(lo[0] + i, nx), wrapm(lo[1] + j, ny), wrapm(lo[2] + k, nz));
                if (!h->beta[o]) continue;
                sum += h->q[3][o];
                ++cnt;
            }
    out[0] = out[1] = 0.0;
    out[2] = (double)cnt;
    if (cnt == 0) return DNSREF_OK;
    const double mean = sum / (double)cnt;
    double ss = 0.0;
    for (int k = 0; k < size[2]; ++k)
        for (int j = 0; j < size[1]; ++j)
            for (int i = 0; i < size[0]; ++i) {
                const int64_t o = IDX(wrapm(lo[0] + i, nx), wrapm(lo[1] + j, ny), wrapm(lo[2] + k, nz));
                if (!h->beta[o]) continue;
                const double dv = h->q[3][o] - mean;
                ss += dv * dv;
            }
    out[0] = mean;
    out[1] = sqrt(ss / (double)cnt);
    return DNSREF_OK;
}

/* ------------------------------------------------------------------------ */
static int valid_params(const dnsref_params_t *P)
{
    if (!P) return 0;
    if (P->nx < 1 || P->ny < 1 || P->nz < 1) return 0;
    if (!(P->dx > 0) || !(P->dy > 0) || !(P->dz > 0) || !(P->dt > 0)) return 0;
    if (P->nu < 0 || P->alpha_c < 0 || P->n_piter < 1) return 0;
    return 1;
}

int dnsref_destroy(dnsref_t *h)
{
    if (!h) return DNSREF_EINVAL;
    free(h->beta);
    for (int s = 0; s < h->nsrc; ++s) { free(h->sx[s]); free(h->sy[s]); free(h->sz[s]); }
    free(h->sx); free(h->sy); free(h->sz); free(h->src);
    for (int m = 0; m < 4; ++m) { free(h->q[m]); free(h->qs[m]); free(h->qc[m]); free(h->f[m]); }
    free(h->p); free(h->d); free(h->r); free(h->re); free(h->im);
    free(h);
    return DNSREF_OK;
}

int dnsref_create(const dnsref_params_t *P, const uint8_t *mask, const dnsref_source_t *src, int32_t nsrc,
                  dnsref_t **out)
{
    if (!valid_params(P) || !out || nsrc < 0 || (nsrc > 0 && !src)) return DNSREF_EINVAL;
    for (int s = 0; s < nsrc; ++s)
        if (!(src[s].tau_f > 0)) return DNSREF_EINVAL;
    dnsref_t *h = (dnsref_t *)calloc(1, sizeof(dnsref_t));
    if (!h) return DNSREF_ENOMEM;
    h->P = *P;
    h->n = (int64_t)P->nx * P->ny * P->nz;
    const int64_t n = h->n;
    h->beta = (uint8_t *)malloc(n);
    for (int64_t o = 0; o < n; ++o) h->beta[o] = mask ? (mask[o] != 0) : 1;
    h->nsrc = nsrc;
    h->src = (dnsref_source_t *)malloc(sizeof(dnsref_source_t) * (nsrc ? nsrc : 1));
    h->sx = (double **)calloc(nsrc ? nsrc : 1, sizeof(double *));
    h->sy = (double **)calloc(nsrc ? nsrc : 1, sizeof(double *));
    h->sz = (double **)calloc(nsrc ? nsrc : 1, sizeof(double *));
    for (int s = 0; s < nsrc; ++s) {
        h->src[s] = src[s];
        h->sx[s] = (double *)malloc(sizeof(double) * P->nx);
        h->sy[s] = (double *)malloc(sizeof(double) * P->ny);
        h->sz[s] = (double *)malloc(sizeof(double) * P->nz);
        dnsref_source_table(P->nx, P->dx, src[s].lo[0], src[s].size[0], src[s].B[0], h->sx[s]);
        dnsref_source_table(P->ny, P->dy, src[s].lo[1], src[s].size[1], src[s].B[1], h->sy[s]);
        dnsref_source_table(P->nz, P->dz, src[s].lo[2], src[s].size[2], src[s].B[2], h->sz[s]);
    }
    for (int m = 0; m < 4; ++m) {
        h->q[m] = (double *)calloc(n, sizeof(double));
        h->qs[m] = (double *)calloc(n, sizeof(double));
        h->qc[m] = (double *)calloc(n, sizeof(double));
        h->f[m] = (double *)calloc(n, sizeof(double));
    }
    h->p = (double *)calloc(n, sizeof(double));
    h->d = (double *)calloc(n, sizeof(double));
    h->r = (double *)calloc(n, sizeof(double));
    h->re = (double *)calloc(n, sizeof(double));
    h->im = (double *)calloc(n, sizeof(double));
    if (!h->beta || !h->p || !h->d || !h->r || !h->re || !h->im || !h->f[3]) { dnsref_destroy(h); return DNSREF_ENOMEM; }
    *out = h;
    return DNSREF_OK;
}

/* copies in; u,v,w,c masked by select (reading R7); p nullable -> 0, not masked */
int dnsref_set_fields(dnsref_t *h, const double *u, const double *v, const double *w, const double *c, const double *p)
{
    if (!h || !u || !v || !w || !c) return DNSREF_EINVAL;
    const double *in[4] = {u, v, w, c};
    for (int m = 0; m < 4; ++m)
        for (int64_t o = 0; o < h->n; ++o) h->q[m][o] = h->beta[o] ? in[m][o] : 0.0;
    for (int64_t o = 0; o < h->n; ++o) h->p[o] = p ? p[o] : 0.0;
    return DNSREF_OK;
}

/* copies out (any pointer may be NULL) */
int dnsref_get_fields(const dnsref_t *h, double *u, double *v, double *w, double *c, double *p)
{
    if (!h) return DNSREF_EINVAL;
    double *out[4] = {u, v, w, c};
    for (int m = 0; m < 4; ++m)
        if (out[m]) memcpy(out[m], h->q[m], sizeof(double) * h->n);
    if (p) memcpy(p, h->p, sizeof(double) * h->n);
    return DNSREF_OK;
}

/* one solve with the beta-term off: p = Delta^-1 rhs (host pointers) */
int dnsref_poisson(dnsref_t *h, const double *rhs, double *p)
{
    if (!h || !rhs || !p) return DNSREF_EINVAL;
    return dnsref_poisson_solve(h, rhs, p);
}
