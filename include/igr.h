/* igr.h -- C ABI of libigr.so: one SSP-RK3 time step of the 3D compressible Euler equations with
 * information geometric regularisation (IGR) on one NVIDIA B200 (sm_100a).
 *
 * Source of every operation: arXiv 2505.07392 as extracted in PAPER.md (cited "L<line>"), read as
 * recorded in DESIGN.md ("Readings", A1-A18).  The library is hand-written CUDA; there is no CPU
 * fallback: every call fails with IGR_ERR_CUDA if no usable device is present.
 *
 * The method (section 4.1; Algorithm 1):
 *   state q = (rho, m_x, m_y, m_z, E) on a uniform Cartesian grid of nx*ny*nz cells of size dx;
 *   entropic pressure Sigma from   Sigma/rho - alpha div(grad(Sigma)/rho) = alpha (tr((grad u)^2) + (tr grad u)^2)
 *   (eq. 9) by n_jacobi warm-started Jacobi sweeps of the 6-point stencil (L130, L138);
 *   fluxes with p + Sigma (eqs. 6-8), 5th-order linear reconstruction of the conserved
 *   variables and Sigma, Lax-Friedrichs flux (L132, Alg. 1); SSP-RK3 in time (L138).
 *
 * Conventions
 *   - All functions return 0 (IGR_OK) or a negative igr_status; nothing throws or aborts.
 *   - Field layout at the boundary: interior cells only, x fastest: q[c][k][j][i] with c = 0..4,
 *     i.e. index ((c*nz + k)*ny + j)*nx + i; always fp32, also in reduced-storage mode.
 *   - Every `q`/`f` pointer may be a HOST or a DEVICE pointer (resolved with
 *     cudaPointerGetAttributes); it is borrowed for the duration of the call only.
 *   - The solver owns its device buffers (or carves them from igr_options.workspace); `bc` and the
 *     patch arrays are copied at creation.
 *   - igr_step and the per-kernel entry points are asynchronous on the solver's stream; CUDA errors
 *     and non-finite states surface at the next synchronising call (igr_max_wavespeed,
 *     igr_get_*, igr_sync).
 */
#ifndef IGR_H
#define IGR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    IGR_OK = 0,
    IGR_ERR_ARG = -1,        /* null pointer, non-positive size, gamma <= 1, order not in {3,5}, ... */
    IGR_ERR_BC = -2,         /* periodic on only one face of an axis, unknown face code            */
    IGR_ERR_ALLOC = -3,      /* device allocation failed or workspace too small                    */
    IGR_ERR_CUDA = -4,       /* no device, launch or copy failure (see igr_last_error)             */
    IGR_ERR_NONFINITE = -5   /* the state contains NaN/Inf (reported, never repaired: reading A10) */
} igr_status;

/* boundary codes per face (the paper gives no boundary conditions; BASELINE.json names these three;
 * DESIGN.md reading A8).  Order of faces: x-, x+, y-, y+, z-, z+. */
#define IGR_BC_PERIODIC 0    /* wrap modulo n; must be set on both faces of the axis               */
#define IGR_BC_EXTRAP   1    /* zeroth-order extrapolation (clamp to the nearest interior cell)    */
#define IGR_BC_INFLOW   2    /* fixed-state circular patches, extrapolation outside them           */
#define IGR_BC_EXTERNAL 3    /* face shared with a neighbouring sub-domain (DESIGN.md */
                             /* reading A20): ghosts beyond it are never written by the solver, the  */
                             /* caller fills them (igr_pull_halo); sweeps clamp at it                */

/* storage precision of q and Sigma in device memory; arithmetic is always fp32 */
#define IGR_STORE_F32  0
#define IGR_STORE_F16  1
#define IGR_STORE_BF16 2
/* fp64 MODE: fp64 storage AND fp64 arithmetic, for a like-for-like column beside the paper's
 * FP64 grind times (Table 1).  One thread per cell, one launch per row and per Jacobi sweep, IEEE
 * division and square root (parity with the fp64 oracle <= 1e-12).  `fused` and `variant` are ignored; one fluid,
 * no viscosity, no slabs; igr_get_padded / igr_get_source / igr_set_source / igr_get_rhs are not available.  The
 * fp32 calls convert at the boundary; igr_set_state_f64 / igr_get_state_f64 / igr_get_sigma_f64 move fp64 arrays. */
#define IGR_STORE_F64  3

#define IGR_VARIANT_TILED  0
#define IGR_VARIANT_SIMPLE 1

/* A circular inflow patch on a face.  (c0, c1) and radius are in CELL units on the face plane, the
 * transverse axes taken in the order x < y < z.  A ghost cell whose transverse centre (i+1/2, j+1/2)
 * lies at distance r from the centre gets, in all three ghost layers,
 *     q_ghost = q_clamp + w(r) (q_fixed - q_clamp),
 *     w = 1 for r <= radius, 0 otherwise                                   if edge == 0,
 *     w = (1 - tanh((r - radius)/edge))/2, and exactly 0 for r >= radius + 4 edge   if edge > 0,
 * q_fixed = (rho, rho u, rho v, rho w, p/(gamma-1) + rho |u|^2/2), q_clamp = nearest interior cell.
 * Where several patches overlap the one with the largest w wins. */
typedef struct {
    double c0, c1, radius, edge;
    double rho, u, v, w, p;
    double a1, rho2;              /* two fluids only (igr_options.n_fluids = 2): volume fraction of fluid 1 and   */
                                  /* density of fluid 2 in the patch; `rho` is then the density of fluid 1:      */
                                  /* q_fixed = (a1 rho, (1 - a1) rho2, rho_m u, rho_m v, rho_m w, E, a1)         */
} igr_patch;

typedef struct {
    int32_t face[6];              /* IGR_BC_* per face                                            */
    int32_t n_patches[6];         /* used where face[f] == IGR_BC_INFLOW                          */
    const igr_patch *patches[6];  /* host arrays, copied by igr_create                            */
} igr_bc;

typedef struct {
    int32_t storage;       /* IGR_STORE_*                                                         */
    int32_t fused;         /* 1 (what igr_create uses): RK update and stage-3 wave speed fused into */
                           /*    the RHS kernel (one more state buffer, no r array at rest)        */
                           /* 0: one kernel per row of the hot path (source, Jacobi, RHS, update)  */
    int32_t variant;       /* IGR_VARIANT_TILED (default): TMA-staged tiled kernels: the product;  */
                           /* IGR_VARIANT_SIMPLE: TEST-ONLY one-thread-per-cell kernels, one launch */
                           /*    per Jacobi sweep -- the first correct path, kept as a cross-check  */
                           /*    of the tiled kernels against the oracle; never timed, not tuned    */
    int32_t n_fluids;      /* 0 or 1: one ideal gas (the hot path).  2: the TWO-FLUID variant (SURVEY 8(f)  */
                           /*    NEXT-3; Alg. 1; reading A21): the      */
                           /*    five-equation model of two ideal gases (gamma of igr_create_ex and gamma2), */
                           /*    state [7][nz][ny][nx] = (a1 rho1, a2 rho2, rho u, rho v, rho w, E, a1),     */
                           /*    p = (E - rho |u|^2/2)/Gamma, Gamma = a1/(gamma-1) + (1-a1)/(gamma2-1);     */
                           /*    fp32 storage, order 5, fused tiled kernels only (else IGR_ERR_ARG); no      */
                           /*    viscosity, no slabs.  Every call that takes or returns "the state" then     */
                           /*    moves 7 fields, igr_get_padded takes c = 0..7 (7 = Sigma)                   */
    void   *stream;        /* cudaStream_t to run on (NULL: the legacy default stream)             */
    void   *workspace;     /* optional caller-owned DEVICE memory (e.g. a torch tensor), 256-B     */
    size_t  workspace_bytes; /* aligned, at least igr_workspace_bytes(); NULL: library allocates  */
    double  gamma2;        /* n_fluids = 2: ideal-gas exponent of fluid 2 (> 1)                    */
} igr_options;

typedef struct igr_solver igr_solver;

/* Device bytes a solver of this size needs (for igr_options.workspace).  A fused tiled solver keeps no RHS
 * array r[5] at rest (18 fields); it allocates one with cudaMalloc the first time igr_rhs, igr_rk_update,
 * igr_get_rhs or a viscous step needs it (IGR_ERR_ALLOC if that fails). */
size_t igr_workspace_bytes(int nx, int ny, int nz, const igr_options *opt);

/* Create a solver (igr_create: fp32 storage, fused = 1, tiled kernels, default stream, library-owned memory).
 * dx: uniform spacing in all directions; gamma > 1: ideal-gas exponent (eq. 4);
 * alpha >= 0: IGR strength, shock width ~ sqrt(alpha) (L130; the configs use 10 dx^2);
 * order: 5 (L132) or 3; n_jacobi >= 0 sweeps per RHS evaluation (L130 "<~ 10"; configs: 5).
 * Errors: IGR_ERR_ARG (also: a padded field of more than 2^32 - 1 elements, the kernels index cells with
 * 32-bit offsets), IGR_ERR_BC, IGR_ERR_ALLOC, IGR_ERR_CUDA.  *out is NULL on failure. */
int igr_create(int nx, int ny, int nz, double dx, double gamma, double alpha, int order,
               int n_jacobi, const igr_bc *bc, igr_solver **out);
int igr_create_ex(int nx, int ny, int nz, double dx, double gamma, double alpha, int order,
                  int n_jacobi, const igr_bc *bc, const igr_options *opt, igr_solver **out);
void igr_destroy(igr_solver *s);

/* Copy a state in (rounding to the storage format) and reset Sigma = 0 ("Sigma = 0 at t = 0").
 * q (here and in every other call that takes a field): host or device pointer, BORROWED FOR THE DURATION OF
 * THE CALL ONLY: when the call returns a host buffer has been read completely (the library waits for its last
 * host-to-device copy) and may be reused or freed; device buffers are read in stream order. */
int igr_set_state(igr_solver *s, const float *q);
/* Copy the current state out; synchronises.  IGR_ERR_NONFINITE is NOT raised here. */
int igr_get_state(igr_solver *s, float *q);
/* The same for the planes [k0, k0 + nk) only, q: [5][nk][ny][nx] (host or device).  For grids whose whole
 * fp32 state does not fit beside the solver (180 GB: 1280^3 in fp32, 1536^3 with 2-byte storage), and
 * for slab-wise I/O.  igr_set_state_planes does NOT reset Sigma (igr_set_state does) and is refused in
 * the middle of a step; IGR_ERR_ARG for a range outside [0, nz). */
int igr_set_state_planes(igr_solver *s, int k0, int nk, const float *q);
int igr_get_state_planes(igr_solver *s, int k0, int nk, float *q);
/* fp64 arrays (IGR_STORE_F64 only, else IGR_ERR_ARG): same layouts, host or device pointers */
int igr_set_state_f64(igr_solver *s, const double *q);
int igr_get_state_f64(igr_solver *s, double *q);
int igr_get_sigma_f64(igr_solver *s, double *f);
/* Sigma is part of a restart because of the warm start (L130, L138).  f: [nz][ny][nx]. */
int igr_set_sigma(igr_solver *s, const float *f);
int igr_get_sigma(igr_solver *s, float *f);

/* max over cells of max(|u|,|v|,|w|) + sqrt(gamma p / rho): the CFL wave speed (reading A9);
 * the caller chooses dt = CFL dx / *out.  Blocking.  IGR_ERR_NONFINITE if the state holds NaN/Inf
 * or the result is not finite (negative pressure or density). */
int igr_max_wavespeed(igr_solver *s, double *out);

/* One SSP-RK3 step (L138, ref. 17): three RHS evaluations, each = halo/BC, source, n_jacobi
 * warm-started sweeps, fused reconstruction + LF flux + divergence, then the stage update. */
int igr_step(igr_solver *s, double dt);

/* Block until the stream is idle; returns a pending CUDA error if any. */
int igr_sync(igr_solver *s);
const char *igr_last_error(const igr_solver *s);

/* ---- the rows of the hot path as separate calls, for parity tests and
 * profiling.  They act on the solver's CURRENT stage buffer (the state after igr_set_state).   */
int igr_halo_bc(igr_solver *s);        /* a1: ghost layers of q (periodic / extrapolation / inflow) */
int igr_sigma_source(igr_solver *s);   /* a2: b = alpha (tr((grad u)^2) + (tr grad u)^2), 2nd-order */
                                       /*     central differences of u = m/rho (L127, L132)         */
int igr_jacobi(igr_solver *s);         /* a3: n_jacobi sweeps from the stored Sigma + Sigma ghosts  */
int igr_rhs(igr_solver *s);            /* a4: r = -div F^ (reconstruction, LF flux; L132, L183-L210)*/
int igr_rk_update(igr_solver *s, int stage, double dt); /* a5: stage 1..3 of SSP-RK3 (unfused)     */
int igr_get_source(igr_solver *s, float *f);            /* b,   [nz][ny][nx]                        */
int igr_set_source(igr_solver *s, const float *f);      /* test hook: drive igr_jacobi with a given b */
int igr_get_rhs(igr_solver *s, float *r);               /* r,   [5][nz][ny][nx]                     */
/* padded copy (3 ghost layers each side) of component c = 0..4 of q, or Sigma for c = 5:
 * f: [nz+6][ny+6][nx+6] */
int igr_get_padded(igr_solver *s, int c, float *f);

/* ---- NEXT-1: Newtonian viscous stress of eqs. (2), (3), (5):
 * tau_ab = mu (du_a/dx_b + du_b/dx_a) + (zeta - 2 mu/3) delta_ab div u, second-order velocity gradients
 * (L132) reconstructed at the faces (Alg. 1), -tau and -u.tau added to the momentum and energy
 * fluxes.  mu = zeta = 0 (default) is the inviscid path.  With viscosity on, the source row also stores
 * the six components of tau (six fp32 fields, allocated by this call with cudaMalloc: IGR_ERR_ALLOC if
 * that fails), igr_rhs adds the viscous part to r, and igr_step (fused) lets the viscous kernel carry
 * the stage update.  Both arguments must be >= 0 (IGR_ERR_ARG). */
int igr_set_viscosity(igr_solver *s, double mu, double zeta);

/* ---- NEXT-2: z-slab domain decomposition, one halo exchange per RK stage (the
 * paper scales by rectilinear decomposition with GPU-direct neighbour exchange, PAPER.md L258, L297-L311;
 * DESIGN.md section 9, reading A20).  A rank's solver works on its owned planes extended by 8 overlap
 * planes towards every neighbour; those z faces are IGR_BC_EXTERNAL.  One stage on the extended slab is
 * exact on the owned planes (5 sweeps + 3 stencil planes = 8); after every stage the overlap and ghost
 * planes (11 per side, q and Sigma) are overwritten with the neighbour's owned planes.  z is the slowest
 * axis: a plane range of one field is ONE contiguous chunk, moved by cudaMemcpyAsync device-to-device
 * (the copy engines over NVLink when the neighbour is another GPU whose allocation was opened with
 * igr_ipc_open).  Ordering across ranks is the caller's (a barrier after the stage and after the pull:
 * paper_2505_07392_b200/dist.py); the plan comes from paper_2505_07392_b200/slab.py. */
typedef struct {
    unsigned char ipc_handle[64]; /* cudaIpcMemHandle_t of the allocation (valid iff owns_memory)          */
    uint64_t base;                /* address of that allocation in the OWNING process                      */
    uint64_t q_offset[3][5];      /* bytes from base: state buffer b, field c (padded arrays)              */
    uint64_t sig_offset[2];       /* bytes from base: the two Sigma buffers                                */
    uint64_t plane_bytes;         /* one padded z-plane of one field                                       */
    int32_t nz, storage;          /* local interior planes; IGR_STORE_*                                    */
    int32_t cur, sig_cur;         /* buffers holding the current state / Sigma at the time of the call     */
    int32_t owns_memory;          /* 1: the library allocated (cudaMalloc) -> the handle can be opened     */
    int32_t reserved;
} igr_export;

/* one stage (1, 2, 3 in that order) of igr_step: halo, source, sweeps, RHS, update */
int igr_stage(igr_solver *s, int stage, double dt);
int igr_export_fields(igr_solver *s, igr_export *out);
/* open / close a neighbour's allocation in this process (other process, same node).  *peer_base is the
 * address HERE of peer->base THERE.  IGR_ERR_CUDA if the driver refuses (no peer access, same process). */
int igr_ipc_open(const igr_export *peer, void **peer_base);
int igr_ipc_close(void *peer_base);
/* register (peer != NULL) or drop (peer == NULL) the neighbour on side 0 (z-) / 1 (z+): my planes
 * [dst_plane, dst_plane + count) take its planes [src_plane, src_plane + count), interior-relative
 * indices (my ghost planes are -3..-1 and nz..nz+2; the source must be interior planes of the peer).
 * peer_base: its allocation as addressable here (igr_ipc_open, or peer->base inside one process).
 * IGR_ERR_BC if that face is not IGR_BC_EXTERNAL, IGR_ERR_ARG on a shape / range mismatch. */
int igr_set_neighbor(igr_solver *s, int side, const igr_export *peer, const void *peer_base,
                     int dst_plane, int src_plane, int count);
/* enqueue the copies of q (5 fields of the current buffer) and Sigma from every registered neighbour
 * on the solver's stream; drops the cached wave speed if a plane that entered it is overwritten */
int igr_pull_halo(igr_solver *s);
/* Stream-ordered ordering of the exchange between processes (no device synchronisation, no GPU idle time while
 * the hosts talk): every solver owns two INTERPROCESS events, which = 0 "my stage is complete" and which = 1
 * "my pulls are complete".  igr_event_handle returns the 64-byte CUDA IPC handle of one of them (created on
 * first use; the bytes can be shipped to another rank), igr_event_open maps a neighbour's event into this
 * process, igr_event_record records one of mine on my stream, igr_event_wait makes MY stream wait for a
 * neighbour's event (cudaStreamWaitEvent: it captures the neighbour's most recent record, so the hosts must
 * have agreed -- a host-only handshake, dist.py -- that the record was enqueued).  A pull then waits only for
 * the two neighbours' stage, and the next stage's kernels only for the neighbours' pulls. */
int igr_event_handle(igr_solver *s, int which, unsigned char handle[64]);
int igr_event_open(const unsigned char handle[64], void **event);
int igr_event_close(void *event);
int igr_event_record(igr_solver *s, int which);
int igr_event_wait(igr_solver *s, void *event);
/* planes [k0, k1) (0 <= k0 < k1 <= nz) that enter igr_max_wavespeed and the fused stage-3 reduction;
 * default all.  A slab restricts it to its owned planes: the overlap planes are only exact right after a
 * pull, and the max over ranks of the owned maxima is the global maximum. */
int igr_set_wave_range(igr_solver *s, int k0, int k1);

/* ---- measurement hooks (bench.py).  Rows: 0 halo_bc, 1 sigma_source, 2 jacobi (sweeps + Sigma
 * ghosts), 3 rhs, 4 rk_update, 5 max_wavespeed (standalone reduction). */
int igr_kernel_launches(igr_solver *s, long long *out);  /* kernels launched since igr_create     */
int igr_profile(igr_solver *s, int enable);    /* start (1) / stop (0) per-row CUDA-event timing   */
                                               /* on the solver's stream; clears earlier records   */
int igr_profile_read(igr_solver *s, double ms[6], long long count[6]); /* summed ms, calls per row */

/* ---- the CFL wave speed without any allocation (igr_noalloc.cu).
 * For callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it.  The same quantity as igr_max_wavespeed -- max over cells of max(|u|,|v|,|w|) + sqrt(gamma p / rho), Alg. 1
 * L212-L215, readings A5/A9, same per-cell arithmetic -- but it needs no solver and calls no cudaMalloc, cudaFree or
 * allocating library routine: the block partials of the reduction live in a file-scope device array of 512 KB that
 * every GPU which loads the library holds until the process exits.
 *   q       DEVICE pointer, fp32, the unpadded conserved fields [5][nz][ny][nx] (rho, mx, my, mz, E); borrowed,
 *           read only.
 *   out     DEVICE pointer to two floats, written by the call's last kernel: out[0] = the wave speed (the
 *           maximum over the cells that gave a finite value), out[1] = 1 if any cell gave a non-finite value
 *           (NaN/Inf, negative pressure or density: reported, not repaired, reading A10), else 0.
 *   stream  a cudaStream_t (NULL: the default stream).  Two kernels are enqueued on it; the call does not wait
 *           (the caller synchronises before reading `out` on the host) and is capturable after one warm call.
 *   errbuf  optional host buffer of errbuf_len bytes for the message of a failure (may be NULL).
 * Limit: nx * ny * nz <= IGR_NOALLOC_MAX_CELLS (2^30 = 1024^3; one slot of the array per 16384 cells); a larger
 * state, a non-positive size, gamma <= 1 or a null pointer returns IGR_ERR_ARG and launches nothing.  The first
 * call on a device (with that device current) resolves the array's device address (cudaGetSymbolAddress; checked).
 * EVERY call on a device shares the array, which keeps the last call's contents: nothing in it must start at zero
 * (each call overwrites every slot it reads), but two calls that overlap on the GPU -- different streams, or host
 * threads on different streams -- RACE on it.  Order them on one stream or with events. */
#define IGR_NOALLOC_MAX_CELLS (1LL << 30)
int igr_max_wavespeed_noalloc(const float *q, int nx, int ny, int nz, double gamma, float *out, void *stream,
                              char *errbuf, size_t errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* IGR_H */
