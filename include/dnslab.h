/*
 * dnslab.h -- C ABI of libdnslab.so: the DNSLABIB incompressible Navier-Stokes time step
 * (arxiv 2204.02107; citations are PAPER.md:<line>) on one NVIDIA B200 (sm_100a), fp64.
 *
 * The library owns no device memory: the caller hands it one device workspace and a CUDA
 * stream (in this repo both come from PyTorch).  Every call is asynchronous on that stream
 * unless stated otherwise.  All functions return 0 (DNSLAB_OK) or a negative error code;
 * nothing throws across this boundary.  dnslab_strerror() gives text for a code.
 *
 * Grid and layout.  nx*ny*nz cells, all axes periodic, spacings dx,dy,dz.
 * A field is nx*ny*nz doubles, x fastest: element (i,j,k) is at i + nx*(j + ny*k)
 * (a contiguous torch/numpy array of shape (nz,ny,nx)).  nx,ny,nz must be powers of two with
 * 8 <= nx <= 2048 and 8 <= ny,nz <= 1024 (the Poisson solve is a radix FFT).  The mask beta is one byte per cell,
 * same layout, non-zero = fluid, 0 = solid.
 *
 * What one step computes (PAPER.md:43 and eqs. 1-4, 7-9; DESIGN.md lists every reading):
 *   Qc = Q^n, Qs = Q^n                    Q = (u,v,w,c)
 *   for s = 1..4 (classical RK4, a=(1/2,1/2,1), b=(1/6,1/3,1/3,1/6)):
 *       F = beta ? RHS(Qs) : +0.0         eqs. 2-3: skew-symmetric central convection,
 *                                         central diffusion (beta-weighted faces for c, eq. 4),
 *                                         body force b, source relaxation S (phi_set - phi)/tau_f
 *       Qc += b_s dt F ;  Qs = Q^n + a_s dt F   (s < 4)
 *   d = sum_a delta_a Qc.u_a                                     (eq. 7 right-hand side)
 *   repeat n_piter times (eq. 9; p starts from the previous step's p):
 *       r = d + sum_a delta_a[(1-beta) delta_a p] ;  p = F^-1[ F[r] / lambda ]
 *       lambda = -sum_a sin^2(2 pi k_a/N_a)/D_a^2 ; the 8 null modes (2 k_a = 0 mod N_a) := 0
 *   u_a^{n+1} = beta ? Qc.u_a - delta_a p : +0.0 ;  c^{n+1} = Qc.c        (eq. 8)
 * delta_a is the periodic central difference (f[+1]-f[-1])/(2 D_a).
 */
#ifndef DNSLAB_H
#define DNSLAB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DNSLAB_OK 0
#define DNSLAB_EINVAL (-1) /* null pointer, bad dims/spacings/dt/nu/n_piter/tau_f, misaligned workspace */
#define DNSLAB_ENOMEM (-2) /* workspace smaller than dnslab_workspace_bytes()                         */
#define DNSLAB_ECUDA (-3)  /* a CUDA call or kernel launch failed (sticky error)                      */
#define DNSLAB_EARCH (-4)  /* no device, or the current device is not compute capability 10.x         */
#define DNSLAB_ELIMIT (-5) /* dnslab_scalar_stats_static: the box has more than DNSLAB_STATIC_MAX_ROWS rows     */

#define DNSLAB_MAX_SOURCES 16

typedef struct dnslab dnslab_t; /* opaque handle; host memory owned by the library */

typedef struct {
    int32_t nx, ny, nz;    /* grid, powers of two: nx in [8,2048], ny,nz in [8,1024]                 */
    double dx, dy, dz;     /* spacings > 0                                                           */
    double nu;             /* kinematic viscosity >= 0 (eq. 2)                                       */
    double alpha_c;        /* scalar diffusivity >= 0 (eq. 3)                                        */
    double dt;             /* fixed time step > 0                                                    */
    double body[3];        /* body force b (eq. 2)                                      */
    int32_t n_piter;       /* eq. 9 iterations >= 1; the paper hard-codes 4           */
    uint32_t flags;        /* bit0: eq. 6 filter on u,v,w,c at the end of every step (PAPER.md:84-88,
                              central 7-point stencil, gamma = Delta^6/pi^6 as printed: a one-axis Nyquist
                              mode is damped by 0.933 per step, not zeroed -- DESIGN.md reading R23);
                              bit1: project every RK stage (what PAPER.md:43 says the authors dropped for
                              speed).  Any other bit set: DNSLAB_EINVAL                                  */
} dnslab_params_t;

/* One inflow/outflow forcing region S(x,y,z) of eqs. 2-3. */
typedef struct {
    int32_t lo[3], size[3]; /* index box in x,y,z: cells lo..lo+size-1, wrapping modulo N            */
    double B[3];            /* eq. 5 smoothness per axis; B <= 0: binary S = 1 inside the box.
                               B > 0: S_a = (1 - tanh(B[r/(W/2) - (W/2)/r]))/2, r = |x - xc| by
                               minimum image, xc = (lo + (size-1)/2) D, W = size D, S_a(xc) = 1      */
    double u_set[3], c_set; /* target values                                                          */
    double tau_f;           /* relaxation time > 0                                                    */
    uint32_t comps;         /* bit0..3: force u, v, w, c                                              */
} dnslab_source_t;

/* Bytes of device workspace dnslab_create needs for these params; 0 if the params are invalid. */
size_t dnslab_workspace_bytes(const dnslab_params_t *params);

/*
 * Create a solver.  mask: nx*ny*nz bytes (host or device pointer; NULL = all fluid), copied.
 * src: nsrc (<= DNSLAB_MAX_SOURCES) host structs, copied; each needs tau_f > 0 and 1 <= size[a] <= N_a
 * (else DNSLAB_EINVAL).  workspace: DEVICE memory, caller-owned,
 * at least dnslab_workspace_bytes() bytes, 256-byte aligned; it must outlive the handle.
 * cuda_stream: a cudaStream_t (NULL = default stream); every later call runs on it.
 * All fields start at 0 (p = 0 is the first warm start).  Synchronous.
 */
int dnslab_create(const dnslab_params_t *params, const uint8_t *mask, const dnslab_source_t *src, int32_t nsrc,
                  void *workspace, void *cuda_stream, dnslab_t **out);

/* Copy fields in (host or device pointers, nx*ny*nz doubles each).  u,v,w,c are stored as
 * beta ? x : +0.0; p may be NULL (-> 0) and is not masked. */
int dnslab_set_fields(dnslab_t *h, const double *u, const double *v, const double *w, const double *c,
                      const double *p);

/* Advance n >= 0 full time steps.  Asynchronous; no host synchronisation inside. */
int dnslab_step(dnslab_t *h, int32_t n);

/* One Poisson solve with the beta term off: p = F^-1[F[rhs]/lambda], null modes 0 (eq. 9 with
 * beta = 1).  rhs and p are DEVICE pointers to nx*ny*nz doubles, 16-byte aligned (else DNSLAB_EINVAL); they may
 * alias.  Does not touch the solver's own pressure. */
int dnslab_poisson(dnslab_t *h, const double *rhs, double *p);

/* The transform of the solve on its own (testing aid: north_star names a real-to-complex transform; the solve itself
 * never forms this spectrum -- it transforms the packed array and divides by the even eigenvalue table).
 * dnslab_rfft3: in = nx*ny*nz doubles (DEVICE); out = (nx/2+1)*ny*nz complex numbers (re, im interleaved, DEVICE),
 *   out[m + (nx/2+1)*(ky + ny*kz)] = sum_{i,j,k} in[i + nx*(j + ny*k)] exp(-2 pi i (m i/nx + ky j/ny + kz k/nz)),
 *   unnormalised, m = 0..nx/2.  Computed with the single-axis passes of the solve (x, y, z) plus one untangling kernel.
 * dnslab_irfft3: the inverse (in = such a half spectrum, Hermitian; out = nx*ny*nz doubles), includes the 1/N.
 * in and out must be 16-byte aligned and must not overlap (either: DNSLAB_EINVAL).  Both use the solver's work array: do not call between dnslab_step launches on
 * another stream.  PAPER.md:43 ("fft"), eq. 9 PAPER.md:102. */
int dnslab_rfft3(dnslab_t *h, const double *in, double *out);
int dnslab_irfft3(dnslab_t *h, const double *in, double *out);

/* Borrowed DEVICE pointers to the current u,v,w,c,p (any out-pointer may be NULL).  No copy.
 * Valid until the next dnslab_step / dnslab_set_fields / dnslab_destroy (buffers rotate). */
int dnslab_fields(dnslab_t *h, const double **u, const double **v, const double **w, const double **c,
                  const double **p);

/* Copy the current fields out to host or device buffers (any may be NULL).  Asynchronous on the
 * stream for device and pinned-host destinations; synchronise the stream before reading. */
int dnslab_get_fields(dnslab_t *h, double *u, double *v, double *w, double *c, double *p);

/* ---- Measurement aids: NOT part of the method ---------------------------------------------------------------
 * dnslab_launch_count, dnslab_profile, dnslab_profile_read and the DNSLAB_K_* classes exist for bench.py and the
 * tests (launch accounting, per-kernel device times).  Nothing the paper defines depends on them; a user of the
 * solver never needs to call them, and the class list follows this implementation's kernels, not the paper. */
/* Number of kernels the library has launched on this handle since create (for bench accounting). */
int64_t dnslab_launch_count(const dnslab_t *h);

/* Per-kernel timing (measurement aid; off by default).  While enabled every kernel launch is
 * bracketed by CUDA events on the solver's stream and accounted to one of these classes.
 * dnslab_profile(h, 1) clears the totals and starts; dnslab_profile(h, 0) stops.
 * dnslab_profile_read synchronises the stream and writes, per class, the summed device time in
 * milliseconds and the number of launches into two host arrays of DNSLAB_NCLASS entries. */
#define DNSLAB_K_RK 0      /* fused RHS + Runge-Kutta stage kernel (4 per step)            */
#define DNSLAB_K_DIV 1     /* divergence                                                   */
#define DNSLAB_K_FFT_X 2   /* x-axis FFT passes (forward with the eq. 9 prologue, inverse) */
#define DNSLAB_K_FFT_Y 3   /* y-axis FFT passes                                            */
#define DNSLAB_K_FFT_Z 4   /* fused z forward + eigenvalue division + z inverse pass       */
#define DNSLAB_K_PROJECT 5 /* pressure-gradient projection                                 */
#define DNSLAB_K_EQ9 6     /* eq. 9 right-hand side at the cells next to solid cells       */
#define DNSLAB_K_FILTER 7  /* eq. 6 filter (flags bit 0)                                    */
#define DNSLAB_K_REDUCE 8  /* Courant-number and scalar mean/std reductions (NEXT-3)         */
#define DNSLAB_K_PARTICLES 9 /* Lagrangian particle step (NEXT-4)                             */
#define DNSLAB_K_FFT_XY 10   /* two-pass solve: x and the high digit of y in one pass (forward, inverse) */
#define DNSLAB_K_FFT_YZ 11   /* two-pass solve: low digit of y, z forward, division, and back             */
#define DNSLAB_NCLASS 12
int dnslab_profile(dnslab_t *h, int enable);
int dnslab_profile_read(dnslab_t *h, double *ms, int64_t *launches);

/* ---- NEXT-3: the reductions of the paper's main loop --------------------------------------------------
 * dnslab_courant: Co = dt * max over all cells of (|u|/dx + |v|/dy + |w|/dz) of the current state -- the
 * quantity the paper's dynamic time stepping limits ("AdjustDt.m"; formula not printed, DESIGN.md
 * reading R24).  *co is HOST memory; the call synchronises the stream.  Bit-identical to a plain loop.
 * dnslab_set_dt: the time step used by the following dnslab_step calls (dt > 0, else DNSLAB_EINVAL); the
 * caller's control law is dt_new = Co_max * dt / Co.
 * dnslab_scalar_stats: mean, population standard deviation and count of the scalar c over the FLUID cells of the
 * index box lo[0..2] (x,y,z), size[0..2] (1 <= size[a] <= N_a; the box wraps modulo N) -- the "mean CO2
 * content" and its standard deviation monitored in PAPER.md:265-269 (reading R25).  out[0..2] is HOST memory
 * (mean, std, count); a box without fluid cells gives zeros.  Synchronises the stream.  Partial sums are combined
 * in a fixed order (reproducible), which is not the order of a plain loop: agreement to ~1e-13 relative. */
int dnslab_courant(dnslab_t *h, double *co);
int dnslab_set_dt(dnslab_t *h, double dt);
int dnslab_scalar_stats(dnslab_t *h, const int32_t lo[3], const int32_t size[3], double out[3]);

/* ---- The same statistic for callers that cannot give the library any device memory -----------------------------
 * Everything else in this header runs out of a device workspace that the caller had to allocate for dnslab_create.
 * Some callers have no way to do that, and must not trigger a cudaMalloc either:
 *   - a monitor or co-processing plug-in that is handed borrowed field pointers (dnslab_fields) by a solver whose
 *     owner has already given the whole HBM to its fields or to a framework's caching pool (config 5 of this repo
 *     is such a "full-HBM working set"): a second workspace or a cudaMalloc simply fails with out-of-memory;
 *   - code on a path where allocation is forbidden or too costly: cudaMalloc / cudaFree synchronise the whole
 *     device and stall every stream of a running simulation, and they are illegal while a stream is being captured;
 *   - hosts that account for every device byte up front (fixed memory budgets, MPS / MIG slices with a hard limit).
 * dnslab_scalar_stats_static computes what dnslab_scalar_stats computes -- mean, population standard deviation and
 * count of c over the fluid cells of an index box (reading R25) -- without a handle and
 * without allocating: it calls no cudaMalloc, cudaFree or any routine that allocates.  Its scratch (one partial sum
 * and one count per row of the box) is a fixed array inside the library's device image: 2 * DNSLAB_STATIC_MAX_ROWS
 * doubles = 1 MiB, which every GPU that loads libdnslab.so holds until the process exits, whether this call is ever
 * made or not.
 *   c     DEVICE, nx*ny*nz doubles, x fastest (the layout at the top of this file); read only.
 *   mask  DEVICE, nx*ny*nz bytes, non-zero = fluid; NULL = every cell is fluid; read only.
 *   nx, ny, nz  powers of two within the limits given at dnslab_params_t; anything else: DNSLAB_EINVAL.
 *   lo, size    HOST, the index box as in dnslab_scalar_stats (1 <= size[a] <= N_a, wraps modulo N).
 *   cuda_stream a cudaStream_t (NULL = default stream); the call is ASYNCHRONOUS on it, no host synchronisation.
 *   out   DEVICE, 3 doubles, caller-owned: mean, std, count (zeros for a box without fluid cells); also read by the
 *         call itself between its passes, so nothing else may write it until the call has finished on the stream.
 * Limit: size[1]*size[2] <= DNSLAB_STATIC_MAX_ROWS (65 536 rows: a full 256 x 256 cross-section, any length in x).
 * A taller box returns DNSLAB_ELIMIT ("box has more rows ... than the static scratch array holds") and launches
 * nothing; split it into slabs, or use dnslab_scalar_stats.
 * First call on a device: the library looks up the device address of its array (cudaGetSymbolAddress) with that
 * device current and remembers it; this one-time set-up is not a stream operation, so make the first call on each
 * device before any stream capture begins.  The calling thread's current device must be the one c, mask and out
 * live on.
 * Sharing: all calls in the process use the same array on a device, and it keeps whatever the last call left in it.
 * Nothing in it needs to start at zero (each pass writes every slot it later reads), but two calls that overlap on
 * the GPU -- different streams, or different threads, without an ordering between them -- race on it and both
 * results are garbage.  Calls on one stream are safe back to back.
 * Summation order: one partial per row, rows combined in index order -- fixed, and independent of the GPU's SM count;
 * not the order of dnslab_scalar_stats or of a plain loop (agreement ~1e-13 relative). */
#define DNSLAB_STATIC_MAX_ROWS 65536
int dnslab_scalar_stats_static(const double *c, const uint8_t *mask, int32_t nx, int32_t ny, int32_t nz,
                               const int32_t lo[3], const int32_t size[3], void *cuda_stream, double *out);

/* ---- NEXT-4: Lagrangian particles, eqs. 10-13 ------------------------------------------
 * dnslab_particles_attach: from now on every time step of dnslab_step ends with one implicit Euler step of size
 * dt of the n particles in `state`, in the velocity field just computed (the paper's "SolveDrops.m" after the
 * fluid solve).  state is DEVICE memory owned by the caller, 8 arrays of n doubles one after the
 * other: x, y, z (positions in [0, N_a Delta_a), cell centres at i Delta), u, v, w (particle velocity),
 * d (diameter as it enters eq. 11), rho_p; the first six are updated in place.  rho_f > 0 is the fluid density of
 * eq. 11, g[3] the gravitational acceleration of eq. 10 (host pointer, copied).  u_f is the trilinear interpolation
 * of u, v, w (R26), C_d is taken from the old velocities (R27), positions wrap periodically (R28).
 * n = 0 detaches.  DNSLAB_EINVAL for n < 0, a null state with n > 0, rho_f <= 0, or nu = 0 (eq. 11 divides by it). */
int dnslab_particles_attach(dnslab_t *h, int64_t n, double *state, double rho_f, const double g[3]);

int dnslab_destroy(dnslab_t *h);

const char *dnslab_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* DNSLAB_H */
