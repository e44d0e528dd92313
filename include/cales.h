/* cales.h -- C ABI of the B200-native (sm_100a, fp64 CUDA) hot path of CaLES (arXiv 2411.09364).
 *
 * One low-storage RK3 step of the incompressible staggered-grid finite-difference LES of the paper
 * (Alg. 1; Alg. 2) on ONE GPU.  Every step of the
 * path runs in hand-written CUDA kernels inside libcales.so; there is no CPU fallback and no cuFFT.
 *
 * Conventions:
 *  - Axis convention of the solver: x streamwise (always periodic), y spanwise (periodic
 *    or walls), z wall-normal (periodic or walls; the only direction that may be non-uniform; the
 *    Thomas direction).  The paper's text calls this direction y: paper-y == our z, paper L_22 == L_zz.
 *  - Arrays hold interior values only, fp64, C order [k][j][i], x fastest: idx = i + nx*(j + ny*k).
 *    u sits on the +x face of cell (i,j,k), v on the +y face, w on the +z face; p, phi, nu_t at cell
 *    centres.  In a wall-bounded direction the last face entry (w[nz-1], v[.][ny-1][.]) is the wall
 *    itself and is kept at 0 by the library.
 *  - Pointers marked DEVICE must be device pointers valid on `device`; HOST pointers are host memory.
 *  - Ownership: the caller owns every buffer, including the workspace blob (size from
 *    cales_workspace_bytes) that the library carves into its fields, work arrays and tables.  The
 *    library never allocates device memory.  The workspace and the stream must outlive the solver.
 *  - Every entry point runs on the device given at cales_create whatever the caller's current device is, and leaves the caller's
 *    current device as it found it.
 *  - All work is enqueued on the caller's CUDA stream (`cuda_stream`, a cudaStream_t; NULL = the
 *    legacy default stream).  cales_step / cales_poisson_solve / cales_eddy_viscosity / cales_wall_stress
 *    are asynchronous; cales_create, cales_set_field / cales_get_field with host pointers and
 *    cales_diagnostics synchronise the stream.
 *  - Errors: every function returning int returns CALES_OK (0) or one of the codes below, never throws,
 *    never aborts; cales_last_error() gives a thread-local message.  Argument errors are detected at
 *    cales_create (nothing can fail for argument reasons at step time).
 */
#ifndef CALES_H
#define CALES_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct cales_solver cales_solver; /* opaque */

enum { CALES_OK = 0, CALES_EINVAL = 1, CALES_EUNSUPPORTED = 2, CALES_ENOMEM = 3, CALES_ECUDA = 4, CALES_ENUMERIC = 5 };
enum { CALES_BC_PERIODIC = 0, CALES_BC_WALL = 1 };  /* per direction y, z (both sides share the type); a wall is
                                                      no-slip unless wall_model=1, which turns the z-walls into
                                                      modelled-stress walls */
enum { CALES_SGS_NONE = 0, CALES_SGS_SMAG = 1, CALES_SGS_DSMAG = 2 };
enum { CALES_Z_UNIFORM = 0, CALES_Z_TANH = 1, CALES_Z_USER = 2 };
enum { CALES_U = 0, CALES_V = 1, CALES_W = 2, CALES_P = 3, CALES_NUT = 4 }; /* field ids */

/* Everything the paper's statement of the problem needs. */
typedef struct {
  int nx, ny, nz;            /* cells; nx, ny even and of the form 2^a 3^b; nz >= 4 */
  double lx, ly, lz;         /* box */
  int zstretch;              /* CALES_Z_*; TANH: zf[k] = lz/2 (1 + tanh(a(2k/nz-1))/tanh a), a = zstretch_factor */
  double zstretch_factor;
  const double* zf_user;     /* HOST, nz+1 faces, read during cales_create only (CALES_Z_USER) */
  int bc_y, bc_z;            /* CALES_BC_* */
  double nu;                 /* molecular viscosity */
  int sgs_model;             /* CALES_SGS_*: Eq. 4 / Eq. 5-9 */
  double cs;                 /* Smagorinsky constant of Eq. 4 */
  int van_driest;            /* D = 1 - exp(-z+/A+) */
  double aplus;              /* <= 0 -> 25 */
  int dsm_avg_xy_plane;      /* 1: <> over x-y planes, c_s(k); 0: over x lines, c_s(j,k) (Eq. 6) */
  int dsm_clip_total;        /* 0: c_s = max(c_s, 0); 1: nu_t = max(nu_t, -nu) */
  double dsm_alpha2d;        /* filter-width ratio of the x-y test filter; <= 0 -> 4^(1/3) */
  int wall_model;            /* log-law wall model on the z walls (Eq. 10) */
  double kappa, B;           /* <= 0 kappa -> 0.41; B as given (5.2 in the paper) */
  double h_wm;               /* height of the wall-modelled layer, the same at every modelled wall (z and y): linear interpolation
                                between the two bracketing centres; <= 0 -> first off-wall cell centre; must lie
                                below lz/2 (and ly/2 with wall_model_y) */
  double wm_tol;             /* relative tolerance on tau_w; <= 0 -> 1e-4 */
  int wm_maxit;              /* <= 0 -> 50 */
  int implicit_z;            /* Crank-Nicolson in z, Eq. 20-22 */
  int const_flow_rate;       /* uniform forcing that keeps the bulk velocity at u_bulk */
  double u_bulk;
  void* workspace;           /* DEVICE, 256-byte aligned, >= cales_workspace_bytes(params) */
  size_t workspace_bytes;
  void* cuda_stream;         /* cudaStream_t of the caller */
  int device;                /* CUDA device ordinal the workspace lives on */
  int wall_model_y;          /* log-law wall model on the y walls too (duct WMLES); needs bc_y = wall */
  int dsm_filter3d;          /* dynamic model: 1 = 3-D box test filter (x, y, z; identity in z and alpha = 4^(1/3) in the first
                                off-wall layer, alpha = 2 elsewhere); 0 = x-y filter */
  int implicit_xyz;          /* Crank-Nicolson in all three directions, Eq. 17-19: three modified Helmholtz solves
                                per substep with the eigen-expansion solver.  Needs periodic y (the transforms want
                                homogeneous conditions); the wall model stays available on the z walls; excludes
                                implicit_z */
} cales_params;

typedef struct {
  double max_div;            /* max |div u| over cells */
  double u_bulk;             /* dzf-weighted volume mean of u */
  double kinetic_energy;     /* volume mean of (uc^2+vc^2+wc^2)/2 at cell centres */
  double forcing;            /* equivalent body force of the last substep's bulk correction */
  int wm_max_iters;          /* max Newton iterations of the last wall-model evaluation */
  int nan_count;             /* non-finite entries in u, v, w, p */
  double ms_rhs, ms_implicit, ms_solver, ms_correction, ms_sgs, ms_wall; /* device ms of the last step, by
                                phase, only when cales_set_timing(s, 1) was called before it; else 0 */
} cales_diag;

/* Fill *p with the defaults (everything off/zero, kappa 0.41, B 5.2, A+ 25, cs 0.17, averaging over planes). */
void cales_default_params(cales_params* p);

/* Bytes of workspace a solver with these parameters needs (0 on invalid parameters; see cales_last_error). */
size_t cales_workspace_bytes(const cales_params* p);

/* Create a solver.  Validates the parameters (CALES_EINVAL: bad sizes / null pointers / workspace too small;
 * CALES_EUNSUPPORTED: sizes that do not factor into 2 and 3, odd nx or ny, periodic z with stretching, wall model
 * without z walls, van Driest without z walls / with y walls / with the wall model, implicit_xyz with y walls or together
 * with implicit_z),
 * builds the grid and the transform tables on the host, uploads them into the workspace, zeroes all fields.
 * Synchronises the stream. */
int cales_create(const cales_params* p, cales_solver** out);

/* The positional form named by the problem statement: grid, box, z-stretching, BCs, nu, sgs_model, wall_model,
 * implicit_z; every other parameter takes its default.  The workspace is still the caller's. */
int cales_create_basic(int nx, int ny, int nz, double lx, double ly, double lz, int zstretch, double zstretch_factor,
                       int bc_y, int bc_z, double nu, int sgs_model, int wall_model, int implicit_z,
                       void* workspace, size_t workspace_bytes, void* cuda_stream, int device, cales_solver** out);

int cales_destroy(cales_solver* s);

/* Copy a whole field (nz*ny*nx doubles) into / out of the solver state.  on_device != 0: DEVICE pointer,
 * asynchronous on the stream; 0: HOST pointer, the call synchronises.  Setting a velocity component marks the
 * closures (wall stress, nu_t) stale: they are recomputed at the start of the next cales_step (Alg. 1 l.1-2). */
int cales_set_field(cales_solver* s, int field, const double* src, int src_on_device);
int cales_get_field(cales_solver* s, int field, double* dst, int dst_on_device);

/* One full RK3 step = 3 substeps of Alg. 1 with the coefficients of PAPER.md:100:
 * u* from Eq. 11 (or Eq. 20-21), bulk forcing, Poisson Eq. 12, correction Eq. 13, pressure Eq. 14 / 22,
 * wall stress Eq. 10, nu_t Eq. 4 / Eq. 5-9.  Asynchronous for every dt: dt and the scalars derived from it (and the Crank-Nicolson
 * tables of Eq. 21) are kept in device memory, so a change of dt costs two tiny kernels and neither a synchronisation nor a new
 * CUDA graph.  dt > 0. */
int cales_step(cales_solver* s, double dt);

/* The same with the time step chosen on the device: dt = cfl / max over cells of (|u_c|/dx + |v_c|/dy + |w_c|/dzf) of the current
 * velocity ("maximum allowable value ... multiplied by a safety factor of 0.95"; formula: DESIGN.md reading S18).
 * Asynchronous, no host synchronisation; cales_last_dt reads the value back. */
int cales_step_adaptive(cales_solver* s, double cfl);

/* dt of the last step: HOST output; synchronises the stream if that dt was computed on the device. */
int cales_last_dt(cales_solver* s, double* dt_host);

/* Solve L_h phi = rhs with the solver's boundary conditions (Eq. 12; eigenfunction expansion,
 * PAPER.md:126): real FFT along x, real FFT or DCT-II along y, (cyclic) Thomas along z.  The component of rhs
 * incompatible with the singular operator is discarded; phi has zero dzf-weighted mean.  rhs_dev, phi_dev:
 * DEVICE, nz*ny*nx, may alias.  Asynchronous. */
int cales_poisson_solve(cales_solver* s, const double* rhs_dev, double* phi_dev);

/* nu_t (Eq. 4 or Eq. 5-9) of a velocity field.  u, v, w: DEVICE fields, or all NULL = the solver's own velocity;
 * nut: DEVICE output, nz*ny*nx (NULL = the solver's own nu_t).  External fields must hold 0 on the wall faces
 * (v[.][ny-1][.] with y walls, w[nz-1] with z walls), as the solver's own fields always do.  External fields need an external
 * nut (CALES_EINVAL otherwise).  The evaluation shares the solver's scratch: cales_get_cs afterwards returns the coefficient of
 * THIS evaluation, and the wall-model ghosts / van Driest wall shear of an external field use the wall stresses of the solver's
 * own velocity as they stand.  Asynchronous. */
int cales_eddy_viscosity(cales_solver* s, const double* u, const double* v, const double* w, double* nut);

/* Wall stresses of the log-law wall model from the solver's velocity (Eq. 10):
 * tau_dev DEVICE [wall(0 bottom,1 top)][comp(0: tau_xz at u points, 1: tau_yz at v points)][ny][nx]
 * (NULL = only refresh the internal planes).  Asynchronous. */
int cales_wall_stress(cales_solver* s, double* tau_dev);

/* The same for the y walls (wall_model_y): tau_dev DEVICE [wall(0: j = 0 side, 1: j = ny-1 side)][comp(0: tau_xy at u points,
 * 1: tau_zy at w points)][nz][nx] (NULL = only refresh the internal planes).  Asynchronous. */
int cales_wall_stress_y(cales_solver* s, double* tau_dev);

/* Make the solver's velocity discretely solenoidal by one projection with gamma*dt = 1 (Eq. 12-13). */
int cales_project(cales_solver* s);

/* Adaptive time step (a fixed fraction of the stability limit; reading S18):
 * *dt_host = cfl / max over cells of (|u_c|/dx + |v_c|/dy + |w_c|/dzf), velocities averaged to the cell centres.
 * HOST output; synchronises the stream. */
int cales_cfl_dt(cales_solver* s, double cfl, double* dt_host);

/* Allocation-free variant of the CFL reduction, for callers that cannot allocate (CUDA graph capture, serving loops): the same
 * reduction as cales_cfl_dt (reading S18), its scratch in a file-scope device array of
 * CALES_STATIC_SCRATCH_BYTES that every GPU loading the library holds until exit, not in the workspace.  No cudaMalloc, cudaFree
 * or allocating library call, no host synchronisation.  u, v, w: DEVICE fields nz*ny*nx, or all NULL = the solver's own velocity;
 * dt_dev: DEVICE output, one double = cfl / max rate (0 for a field at rest).  The grid may have at most
 * CALES_STATIC_SCRATCH_BLOCKS blocks of 32 x 8 points per plane (ceil(nx/32) * ceil(ny/8) * nz), CALES_EINVAL with a message
 * otherwise.  All calls on a device share the array (solvers and streams alike): calls that overlap on the GPU race; it keeps the
 * last call's contents and no slot needs clearing (every slot a call reads it has written first).  Asynchronous on the solver's
 * stream. */
#define CALES_STATIC_SCRATCH_BLOCKS (1 << 20)
#define CALES_STATIC_SCRATCH_BYTES (8 * (CALES_STATIC_SCRATCH_BLOCKS + 1024))
int cales_cfl_dt_static(cales_solver* s, const double* u, const double* v, const double* w, double cfl, double* dt_dev);

/* On-line statistics: x-y plane means per k of the centre-averaged u, v, w, uu, vv, ww, uw and of nu_t.
 * out_dev: DEVICE, [8][nz].  Asynchronous. */
int cales_plane_stats(cales_solver* s, double* out_dev);

/* Time-accumulated statistics ("mean quantities"; C_f and Re_tau of Tables 3-5).  cales_stats_accumulate adds
 * weight x (the plane means of cales_plane_stats, the wall-shear means) of the current state to device accumulators (asynchronous;
 * weight > 0, e.g. dt); cales_stats_reset zeroes them.  cales_stats_get (synchronises; HOST outputs, any may be NULL) returns the
 * weighted time averages: prof [8][nz]; wall [8] = mean wall shear stress on the z walls ((tau_xz, tau_yz) bottom, then top) and on
 * the y walls ((tau_xy, tau_zy) at j = 0, then j = ny-1; dzf-weighted), 0 in periodic directions, positive when the wall retards a
 * flow in the positive direction; modelled walls report the wall-model stress, no-slip walls nu x the one-sided difference to the
 * mirror ghost; derived [4] = tau_w (mean of the streamwise components over the walls), u_tau = sqrt(tau_w),
 * Re_tau = u_tau (lz/2) / nu, C_f = 2 tau_w / u_b^2 with u_b the dzf-weighted mean of the averaged <u> profile; *weight = total. */
int cales_stats_reset(cales_solver* s);
int cales_stats_accumulate(cales_solver* s, double weight);
int cales_stats_get(cales_solver* s, double* prof_host, double* wall_host, double* derived_host, double* weight_host);

/* Dynamic coefficient of the last eddy-viscosity evaluation: cs_dev DEVICE, nz (plane averaging) or nz*ny. */
int cales_get_cs(cales_solver* s, double* cs_dev);

/* Batched 1-D transforms of the Poisson solver applied to a whole field, for tests (DEVICE, in place):
 * dir 0: x, dir 1: y (FFT or DCT-II by bc_y); inverse != 0: the inverse transform (normalised). */
int cales_transform(cales_solver* s, double* field_dev, int dir, int inverse);

/* Tiled shared-memory transpose of every k-plane: dst[k][i][j] = src[k][j][i] (DEVICE, out of place). */
int cales_transpose_xy(cales_solver* s, const double* src_dev, double* dst_dev);

/* Per-kernel device timing of cales_step: when on, a CUDA event is recorded on the stream after every kernel
 * launch of a step (off by default; costs one event record per launch). */
int cales_set_timing(cales_solver* s, int on);

/* Number of kernel ids known to cales_kernel_time. */
int cales_kernel_count(void);

/* Device time of kernel `kid` (0 <= kid < cales_kernel_count()) summed over its launches in the LAST cales_step
 * that ran with timing on: *name = static string, *ms_total = milliseconds, *launches = launch count (any of
 * the three may be NULL).  Synchronises the stream. */
int cales_kernel_time(cales_solver* s, int kid, const char** name, double* ms_total, int* launches);

/* cales_step replays its three substeps as one CUDA graph (captured once: dt lives in device memory; on by default, bypassed while
 * timing is on).  on = 0 returns to plain stream launches. */
int cales_set_graph(cales_solver* s, int on);

/* Measured fp64 FMA throughput of the device in TFLOP/s (an FMA counts 2): a register-resident DFMA loop on the solver's stream,
 * best of three timed launches -- the roofline denominator bench.py uses for the one kernel bound by the plain fp64 ALUs.
 * HOST output; synchronises. */
int cales_fp64_peak(cales_solver* s, double* tflops_host);

/* Kernel-selection knobs, for tests and A/B timing only (results do not depend on them beyond round-off; the defaults are the
 * measured best): "rhs_tile_min_points" (grids with fewer points run the momentum kernel one thread per point instead of the
 * staged z-march; default 200000), "smag_tile_min_points" (the same for the static model; default 4000000),
 * "dsm_col_rows" (output rows per CTA of the column march of the dynamic model; 0 (default): chosen from the grid),
 * "lazy_nut" (dynamic model -- 1 (default): the |S| -> nu_t pass is skipped, the momentum kernel forms c_s Delta^2 |S| when it stages
 * the plane and cales_get_field(CALES_NUT) / the statistics materialise it on demand; 0: nu_t is written after every evaluation),
 * "rhs_variant" (staged momentum kernel -- 1 (default): halo planes moved by 8-byte cp.async, 0: by tiled TMA copies),
 * "correct_pairs" (projection/correction kernel -- 1 (default): two x-neighbours per thread with 16-byte loads and stores, 0: one
 * point per thread),
 * "correct_band" (launch order of that kernel: CTAs sweep k inside bands of this many 8-row CTA rows so that the phi plane k+1 is re-read
 * from L2; 1: plane by plane; 0 (default): chosen from the grid),
 * "rhs_prefetch" (staged momentum kernel -- R^{k-1} of the next plane prefetched while a plane is computed: 1 (default) to L1, 2 to L2,
 * 0 off), "rhs_planes_per_cta" (k-planes per CTA of that kernel; 0 (default): chosen from the grid),
 * "dsm_col_variant" (column march of the dynamic model -- 0: register window, rows staged by TMA bulk copies; 1: the
 * shared-memory-ring form; 2: register window, direct loads; with the 3-D test filter 0: staged rows + register window, 1 / 2: the
 * shared-memory-ring march),
 * "fft_x_lines" / "fft_y_cols" (lines per CTA of the x transforms / columns per CTA tile of the y transforms; defaults: the forward x
 * transform that forms the divergence about 32-64 threads per CTA, the inverse about 64-256, the y tiles 8 or 16 columns),
 * "fft_stage" (2 (default): the first passes of the inverse transforms and the divergence of the forward x transform read shared
 * memory staged by bulk / 16-byte asynchronous copies and batched loads; 1: the inverse y tile is staged through registers instead;
 * 0: they read global memory directly), "poisson_cp_table" (walls in z -- 2 (default):
 * the Thomas solve of the Poisson solver reads c' from a table built once at create, two columns per thread with 16-byte accesses; 1: the
 * same with one column per thread; 0: it recomputes and spills c' on every solve).
 * CALES_EINVAL on an unknown key or a value out of range. */
int cales_set_option(cales_solver* s, const char* key, long long value);

/* Number of kernels cales_step launches per call with the current parameters (for bench.py's gpu_launches). */
int cales_launches_per_step(cales_solver* s);

/* max|div|, bulk velocity, kinetic energy, forcing, Newton iterations, NaN count, phase timings.  Synchronises. */
int cales_diagnostics(cales_solver* s, cales_diag* out);

const char* cales_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
