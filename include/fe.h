/* fe.h -- C ABI of libfe_b200: the TDGL hot path of arxiv/paper_2605_28800 (PETASPIN_microelectrics)
 * on one B200 (sm_100a).
 *
 * What the library computes (citations: PAPER.md = /root/reference/PAPER.md line, equation):
 *   dP_i/dt = L * active * ( E_Land + E_Grad + E_Elec + E_Ext )_i          PAPER.md:33-35 (Eq. 1)
 *   E_Land  = -d f_Land / dP, f_Land = Eq. 3 (+ four 8th-order slots)      PAPER.md:41-47 (Eq. 3)
 *   E_Grad  = -(1/V) dF_Grad,h/dP, F_Grad = Eq. 4 on the cell grid         PAPER.md:53-60 (Eq. 4)
 *   E_Elec  = -(1/(eps0 epsB)) sum_r' K(r-r') P(r')  (cell-averaged dipolar tensor, P = 0 outside,
 *             evaluated as a zero-padded FFT convolution)                  PAPER.md:66-76 (Eq. 5-6), 115
 *   E_Ext   = uniform applied field per simulation                         PAPER.md:78-81 (Eq. 7)
 * over a batch of independent simulations that share geometry             PAPER.md:117.
 * DESIGN.md lists every reading taken where the paper is silent (stencil, periodic axes, tensor).
 *
 * Conventions
 *   Memory.   Every pointer named dev_* / P / dPdt / the workspace is DEVICE memory owned by the caller
 *             (e.g. a torch tensor); every other pointer is HOST memory.  The library allocates only
 *             a few kB of device memory for coefficient and index tables (freed by fe_destroy_grid).
 *   Layout.   State arrays are [batch][3][nz][ny][nx], x fastest, contiguous, 16-byte aligned, of the
 *             grid's dtype (double for FE_F64, float for FE_F32).  Material map: uint8 [nz][ny][nx].
 *   Streams.  `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).  fe_rhs and
 *             fe_step enqueue work and return; fe_precompute_tensor, fe_energy and fe_get_tensor
 *             synchronise the stream before returning.
 *   Errors.   Every call returns fe_status; nothing throws or aborts.  fe_last_error() returns the
 *             text of the last failure on the calling thread.
 *   Units.    The library is unit-agnostic; it evaluates the formulas above with the numbers given.
 */
#ifndef FE_B200_H
#define FE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fe_grid fe_grid;   /* opaque; created by fe_create_grid, freed by fe_destroy_grid */

typedef enum {
    FE_OK = 0,
    FE_EINVAL = 1,      /* bad argument (unsupported sizes, batch < 1, dx <= 0, ...) */
    FE_ENOMEM = 2,      /* workspace too small / allocation of the small tables failed               */
    FE_ECUDA = 3,       /* a CUDA call failed; text in fe_last_error()                              */
    FE_ESTATE = 4,      /* call order: no workspace bound, tensor not precomputed, material unset    */
    FE_ENONFINITE = 5   /* fe_energy found NaN/Inf; fe_step_rk45: error estimate NaN/Inf 8 attempts in a row */
} fe_status;

enum { FE_F64 = 0, FE_F32 = 1 };
enum { FE_TERM_LANDAU = 1, FE_TERM_GRADIENT = 2, FE_TERM_ELEC = 4, FE_TERM_EXT = 8, FE_TERM_ALL = 15 };
enum { FE_EULER = 0, FE_HEUN = 1, FE_RK4 = 2,     /* PAPER.md:117-119; RK4 = BASELINE.json config 2 */
       FE_AB3M2 = 3 };   /* 3-step Adams-Bashforth predictor + 2nd-order Adams-Moulton corrector (PECE),
                            the first two steps of a call are Heun steps (reading A18) */

/* Geometry of the batch (PAPER.md:113 uniform cells; PAPER.md:117 batch). */
typedef struct {
    int32_t nx, ny, nz;        /* cells per axis.  Periodic axis: a power of two in [4, 1024].  Open axis:
                                  2..512 cells (nx even), zero-padded to the next power of two >= 2 n */
    double  dx, dy, dz;        /* cell size > 0                                                     */
    int32_t periodic[3];       /* per axis: 0 = open (vacuum outside, FFT zero-padded to 2n), 1 = periodic */
    int32_t pbc_images[3];     /* R >= 0 image cells summed on each side of a periodic axis         */
    int32_t batch;             /* B >= 1 independent simulations                                    */
    int32_t dtype;             /* FE_F64 or FE_F32: type of every state array and of the arithmetic */
    int32_t n_materials;       /* M in 1..255: rows of the per-member coefficient table             */
    int32_t zero_mode;         /* != 0: with exactly two periodic axes, fix each plane sum of the
                                  kernel to the infinite-film value; with three periodic axes remove
                                  the mean of the kernel (k = 0 mode := 0) (reading A4)    */
} fe_grid_desc;

/* Landau coefficients of one material (Eq. 3, Table 1). a1 per axis. */
typedef struct {
    double  a1[3];
    double  a11, a12, a111, a112, a123;
    double  a1111, a1112, a1122, a1123;   /* 8th-order cubic-symmetry slots; 0 for the paper's tables */
    int32_t active;                       /* 0 = vacuum cell: P stays 0, no gradient bonds to it     */
} fe_landau;

/* Per-simulation scalars: Eq. 4 coefficients, eps0*epsB of Eq. 6, kinetic coefficient L of Eq. 1. */
typedef struct { double G11, G12, G44, G44p; double eps0, epsB, L; } fe_global;

/* Create / destroy.  *out is set only on FE_OK. */
fe_status fe_create_grid(const fe_grid_desc* desc, fe_grid** out);
fe_status fe_destroy_grid(fe_grid* g);

/* Device scratch the caller must provide (spectra, tensor spectrum, stage buffers). */
size_t    fe_workspace_bytes(const fe_grid* g);
/* dev must be 256-byte aligned device memory of at least fe_workspace_bytes(g); borrowed until
 * fe_destroy_grid or the next fe_bind_workspace (which invalidates a precomputed tensor). */
fe_status fe_bind_workspace(fe_grid* g, void* dev, size_t bytes);

/* Coefficients.  member = -1 sets every batch member.  May be called between steps at any time
 * (no tensor recompute needed); takes effect at the next fe_rhs/fe_step/fe_energy call. */
fe_status fe_set_material(fe_grid* g, int32_t member, int32_t material_id, const fe_landau* m);
fe_status fe_set_global(fe_grid* g, int32_t member, const fe_global* gl);
fe_status fe_set_external_field(fe_grid* g, int32_t member, const double E[3]);
/* Time-dependent external excitation: E_ext(t) = E (fe_set_external_field) + amp sin(omega t + phase),
 * sampled at the stage times of the integrator (t_n, t_n + dt/2, ... ; c_i h for RK45).  amp = 0 switches it off.
 * The grid keeps a clock: fe_step / fe_step_rk45 advance it, fe_rhs and fe_energy sample E_ext at it. */
fe_status fe_set_external_wave(fe_grid* g, int32_t member /* -1 = all */, const double amp[3], double omega,
                               double phase);
fe_status fe_set_time(fe_grid* g, double t);
fe_status fe_get_time(const fe_grid* g, double* t);

/* dev_map: DEVICE uint8 [nz][ny][nx] material id per cell (every id < n_materials), shared by the batch;
 * NULL = all cells material 0.  Borrowed (not copied) until the next call or fe_destroy_grid.  PAPER.md:117. */
fe_status fe_set_material_map(fe_grid* g, const uint8_t* dev_map);

/* Execution options (none changes what is computed; every value of every option is covered by the parity tests).
 *   FE_OPT_FUSE_XY     1: the forward x and y transforms run in ONE cooperative kernel that hands the half spectra over
 *                      through a ring of planes resident in L2 whenever the geometry allows it
 *                      (open x and y, 2 ny = padded y length 256 or 512, padded x length 256 or 512);
 *                      0 (default): the separate x and y kernels with the half spectrum in HBM between them.  Measured
 *                      on B200: the fused kernel moves 1.2 GB instead of 1.8 GB of DRAM traffic at config 5a but is
 *                      slower (both passes are bound by shared-memory throughput on the SM).
 *   FE_OPT_XY_TIMEOUTS read-only (fe_get_option synchronises the device): 1 if a wait inside the fused kernel ever
 *                      timed out (it cannot unless the device is shared with a kernel that never yields).
 *   FE_OPT_XY_RING     planes in the L2 ring of the fused pass; 0 (default) sizes it from the geometry (>= 24 planes,
 *                      <= 32 MB), 2..4096 fixes it (clamped to the number of planes).
 *   FE_OPT_XL_SLABS    n > 1: inside fe_step / fe_rhs the inverse x transform and the local step run slab by slab over n
 *                      slabs of z planes, E_elec of a slab handed over through the first planes of the workspace's E
 *                      buffer, which every slab overwrites and which therefore stay in L2 ("consumed
 *                      without a round trip") -- where the geometry allows it (fp64, padded x length 512, open x,
 *                      ny a multiple of 16); 0 / 1 (default): one x-inverse launch writes E_elec for the whole grid. */
enum { FE_OPT_FUSE_XY = 0, FE_OPT_XY_TIMEOUTS = 1, FE_OPT_XY_RING = 2, FE_OPT_XL_SLABS = 3 };
fe_status fe_set_option(fe_grid* g, int32_t option, int32_t value);
fe_status fe_get_option(fe_grid* g, int32_t option, int32_t* value);

/* a0: cell-averaged dipolar tensor K_ij(d) on the padded box and its real spectrum (once per
 * geometry).  PAPER.md:76,115; readings A3, A4. */
fe_status fe_precompute_tensor(fe_grid* g, void* cuda_stream);

/* a1-a4: dPdt = RHS(P) for the terms in the bitmask.  P and dPdt must not alias. */
fe_status fe_rhs(fe_grid* g, const void* P, void* dPdt, uint32_t terms, void* cuda_stream);

/* a5: nsteps explicit steps of size dt, in place on P.  Coefficients and E_Ext are constant during
 * the call. */
fe_status fe_step(fe_grid* g, void* P, double dt, int32_t nsteps, int32_t integrator,
                  uint32_t terms, void* cuda_stream);

/* Adaptive RK45 (ref. [52]; reading A17): Cash-Karp embedded pair, the 5th-order solution
 * is propagated over t_span starting with step dt_init; err = max over all cells, components and batch members of
 * |y5 - y4| / tol (tol: absolute, in the units of P); a step is accepted when err <= 1, then
 * dt_next = 0.9 dt err^-0.2 (5 dt when err <= 1.89e-4), else dt = max(0.9 dt err^-0.25, 0.1 dt) and the step is
 * retried; the last step is shortened to land on t_span.  All batch members advance with the same step.  At most
 * max_steps attempts are made (stats->t < t_span then).  A NaN / Inf error estimate rejects the attempt; after 8
 * such attempts in a row the call returns FE_ENONFINITE (P holds the last accepted state).  Synchronises the stream once per attempt (the decision
 * is taken on the host); *stats is HOST memory and may be NULL.  Needs the workspace of fe_workspace_bytes. */
typedef struct {
    double t;            /* time reached */
    double dt_last;      /* size of the last accepted step */
    double dt_next;      /* step the controller proposes next */
    double err_last;     /* scaled error of the last attempt */
    int32_t accepted, rejected, rhs_evals;
} fe_rk45_stats;
fe_status fe_step_rk45(fe_grid* g, void* P, double t_span, double dt_init, double tol, int32_t max_steps,
                       uint32_t terms, fe_rk45_stats* stats, void* cuda_stream);

/* a6: host_out[b][8] = { F_Land, F_Grad, F_Elec, F_Ext, F_tot, <Px>, <Py>, <Pz> } for the terms in
 * the bitmask (Eq. 2, 5, 7); energies are densities times cell volume summed over cells, means are
 * over active cells.  Returns FE_ENONFINITE if any value is NaN/Inf (host_out is still written). */
fe_status fe_energy(fe_grid* g, const void* P, uint32_t terms, double* host_out, void* cuda_stream);

/* fe_energy for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): same kernels, same eight numbers per member, but
 *   - dev_out is DEVICE memory, [B][8] doubles, caller-owned; nothing is copied to the host and the stream is NOT
 *     synchronised (so no FE_ENONFINITE check either: the caller inspects the numbers);
 *   - the per-block partial sums live in a file-scope static device array of the library (512 KiB, held by every GPU
 *     that loads the library until the process exits) instead of the workspace; the call makes no cudaMalloc / cudaFree
 *     and calls no allocating routine.
 * Limit: batch * 296 * 8 partial sums must fit the 65536 doubles of that array, i.e. batch <= 27; beyond that the call
 * returns FE_EINVAL with the numbers in fe_last_error.  All grids and all calls on a device SHARE the array: calls that
 * may overlap on the GPU (different streams without an ordering between them) race on it; calls on one stream, or
 * ordered by events, are safe.  The array keeps the last call's contents; every row a call reads is first written by
 * that call, so nothing needs clearing.  With FE_TERM_ELEC the bound workspace is used as in fe_energy (E buffer and
 * spectra; caller-owned memory).  PAPER.md:37 Eq. 2, 66 Eq. 5, 80 Eq. 7. */
fe_status fe_energy_noalloc(fe_grid* g, const void* P, uint32_t terms, double* dev_out, void* cuda_stream);

/* Test hooks. */
/* host_out: [6][mz][my][mx] doubles (xx yy zz xy xz yz), the real-space kernel on the circular padded
 * box (m = 2n open, n periodic; entry at index (d mod m) holds K(d)). */
fe_status fe_get_tensor(fe_grid* g, double* host_out, void* cuda_stream);
/* padded box size per axis (mx, my, mz) */
fe_status fe_padded_dims(const fe_grid* g, int32_t out[3]);
/* number of kernel launches issued by this grid since creation (bench.py's gpu_launches claim) */
uint64_t  fe_launch_count(const fe_grid* g);

/* Per-kernel timing for the roofline report: while enabled, fe_rhs/fe_step record a CUDA event on the
 * stream before every kernel launch.  fe_profile_read synchronises the stream and returns, per kernel
 * kind {0 x-forward, 1 y-forward, 2 fused z + tensor multiply, 3 y-inverse, 4 x-inverse, 5 local step,
 * 6 other, 7 fused x+y forward, 8 fused y+x inverse}, the summed device time in ms (host_ms[9]) and the launch
 * count (host_counts[9]) since the last read, then clears the record. */
fe_status fe_profile(fe_grid* g, int32_t enable);
fe_status fe_profile_read(fe_grid* g, double* host_ms, uint64_t* host_counts, void* cuda_stream);

const char* fe_last_error(void);
const char* fe_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FE_B200_H */
