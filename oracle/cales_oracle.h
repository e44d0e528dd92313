/* cales_oracle.h -- C ABI of the CPU ORACLE for the CaLES hot path (arXiv 2411.09364).
 *
 * TEST INFRASTRUCTURE ONLY.  This library is the plain, slow, step-by-step CPU statement of
 * what one low-storage RK3 step of the paper's method computes (Alg. 1-2 at
 * PAPER.md:146-180).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.  It shares no code with the CUDA library (libcales.so);
 * in particular it does NOT include include/cales.h.
 *
 * Conventions: solver axis convention (x streamwise periodic, y spanwise,
 * z wall-normal / stretched / Thomas direction; paper-y == our z).  All arrays hold interior
 * values only, C order [k][j][i], x fastest: idx = i + nx*(j + ny*k).  u on the +x face of cell
 * (i,j,k), v on the +y face, w on the +z face; p, nu_t, S_ij at cell centres.  fp64 everywhere.
 * Every pointer is a HOST pointer; the caller owns every buffer passed in.
 * All functions returning int return 0 on success, non-zero on bad arguments.
 */
#ifndef CALES_ORACLE_H
#define CALES_ORACLE_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_solver oracle_solver;

typedef struct {
  int nx, ny, nz;
  double lx, ly, lz;
  int zstretch;            /* 0 uniform, 1 two-sided tanh (reading S16), 2 user faces */
  double zstretch_factor;
  const double* zf_user;   /* nz+1 faces when zstretch==2 */
  int bc_y, bc_z;          /* 0 periodic, 1 wall */
  double nu;
  int sgs_model;           /* 0 none, 1 static Smagorinsky (Eq. 4), 2 dynamic (Eq. 5-9) */
  double cs;
  int van_driest; double aplus;
  int dsm_avg_xy_plane;    /* 1: <> over x-y planes (c_s(k)); 0: over x lines (c_s(j,k)) */
  int dsm_clip_total;      /* 0: c_s=max(c_s,0); 1: nu_t=max(nu_t,-nu) */
  double dsm_alpha2d;      /* <=0 -> 4^(1/3) */
  int wall_model; double kappa, B, h_wm, wm_tol; int wm_maxit;
  int implicit_z;
  int const_flow_rate; double u_bulk;
  int wall_model_y;        /* log-law wall model on the y walls too (duct WMLES); needs bc_y = wall */
  int dsm_filter3d;        /* 1: 3-D box test filter (x, y and z) with the first-off-wall-layer rule of PAPER.md:128; 0: x-y filter */
  int implicit_xyz;        /* 1: Crank-Nicolson in all three directions, Eq. 17-19; needs periodic y; excludes implicit_z */
} oracle_params;

/* ---- 1-D primitives (pinned against numpy/scipy and O(N^2) definitions in tests) ---- */
/* complex DFT X[m] = sum_j x[j] exp(sign*2*pi*i*m*j/n), sign=-1 forward, +1 inverse (unnormalised) */
int oracle_fft_c2c(int n, const double* re_in, const double* im_in, double* re_out, double* im_out, int sign);
/* DCT-II  X[n] = sum_j x[j] cos(pi*n*(2j+1)/(2N));  DCT-III inverse x[j] = (X[0] + 2 sum_{n>=1} X[n] cos(..))/N */
int oracle_dct2(int n, const double* x, double* X);
int oracle_dct3(int n, const double* X, double* x);
/* tridiagonal a[k] x[k-1] + b[k] x[k] + c[k] x[k+1] = d[k]; a[0], c[n-1] ignored (Thomas) or wrapped (cyclic) */
int oracle_thomas(int n, const double* a, const double* b, const double* c, const double* d, double* x);
int oracle_thomas_cyclic(int n, const double* a, const double* b, const double* c, const double* d, double* x);
/* Log law, Eq. 10: given Re_wm = U h/nu return h+ = u_tau h/nu by Newton (readings S8,S9); *iters = count */
double oracle_loglaw_hplus(double re_wm, double kappa, double B, double tol, int maxit, int* iters);
/* RK3 coefficients: k = 0,1,2 */
void oracle_rk3_coeffs(int k, double* alpha, double* beta, double* gamma);

/* ---- solver ---- */
int  oracle_create(const oracle_params* p, oracle_solver** out);
void oracle_destroy(oracle_solver* s);
const char* oracle_last_error(void);
/* grid: zf (nz+1), zc (nz), dzf (nz), dzc (nz+1 entries: dzc[-1..nz-1] stored at index k+1) */
int oracle_get_grid(oracle_solver* s, double* zf, double* zc, double* dzf, double* dzc);
/* fields: 0 u, 1 v, 2 w, 3 p, 4 nu_t */
int oracle_set_field(oracle_solver* s, int field, const double* src);
int oracle_get_field(oracle_solver* s, int field, double* dst);
/* one full RK3 step (3 substeps of Alg. 1) */
int oracle_step(oracle_solver* s, double dt);
/* one substep rk = 0, 1, 2 of Alg. 1 on its own, and u* / v* / w* (comp 0, 1, 2) of the last substep as it stands after
   Eq. 11 or Eq. 20-21 and before the bulk shift (hooks for the pins of Eq. 21 and Eq. 22) */
int oracle_substep(oracle_solver* s, int rk, double dt);
int oracle_get_ustar(oracle_solver* s, int comp, double* dst);
/* Poisson: L_h phi = rhs with the solver's BCs (Eq. 12); zero weighted-mean gauge (reading S15) */
int oracle_poisson_solve(oracle_solver* s, const double* rhs, double* phi);
/* (1 - c L_jj) q = rhs for velocity component comp (0 u, 1 v, 2 w) with its boundary closure (Eq. 18; needs periodic y) */
int oracle_helmholtz_solve(oracle_solver* s, int comp, double c, const double* rhs, double* out);
/* plain 7-point stencil L_h phi (O-step 3 operator at centres, periodic/Neumann closure) */
int oracle_laplacian(oracle_solver* s, const double* phi, double* out);
/* nu_t from a velocity field (NULL -> internal state); uses the stored wall stresses for van Driest */
int oracle_eddy_viscosity(oracle_solver* s, const double* u, const double* v, const double* w, double* nut);
/* wall stress planes from the internal velocity: tau[wall(0 bottom,1 top)][comp(0 xz at u-points,1 yz at v-points)][ny][nx] */
int oracle_wall_stress(oracle_solver* s, double* tau);
/* y-wall stress planes: tau[wall(0: j=0 side, 1: j=ny-1 side)][comp(0 xy at u-points, 1 zy at w-points)][nz][nx] */
int oracle_wall_stress_y(oracle_solver* s, double* tau);
/* individual explicit terms on the internal velocity / nu_t (each output nz*ny*nx): */
int oracle_advection(oracle_solver* s, double* au, double* av, double* aw);    /* -d_j(u_i u_j) */
int oracle_diffusion(oracle_solver* s, double* du, double* dv, double* dw, int which); /* which: 0 all, 1 x+y only, 2 z only; nu*L u_i */
int oracle_sgs_term(oracle_solver* s, double* su, double* sv, double* sw);     /* d_j(2 nu_t S_ij) */
int oracle_divergence(oracle_solver* s, double* div);                         /* plain divergence of internal u,v,w */
/* strain at centres of the internal velocity: S[6][N] order 11,22,33,12,13,23 ; smag[N] = sqrt(2 Sij Sij) */
int oracle_strain(oracle_solver* s, double* S, double* smag);
/* x-y test filter (1/4,1/2,1/4)^2 of a centred field (reading S11) */
int oracle_filter_xy(oracle_solver* s, const double* q, double* out);
/* the run's test filter (x-y, or x-y-z with dsm_filter3d) of an interior array; kind 0: centred data and u,
   1: v (y-faces), 2: w (z-faces) */
int oracle_test_filter(oracle_solver* s, const double* q, double* out, int kind);
/* dynamic coefficient of the last eddy-viscosity evaluation: cs[nz] (plane) or cs[nz*ny] (x-line) */
int oracle_get_cs(oracle_solver* s, double* cs);
/* L_ij, M_ij (6 x N each, order 11,22,33,12,13,23) of the last dynamic evaluation (Eq. 7-8) */
int oracle_get_dsm_tensors(oracle_solver* s, double* L, double* M);
/* make the internal velocity discretely solenoidal (one projection, gamma*dt = 1) */
int oracle_project(oracle_solver* s);
/* diagnostics of the internal state */
int oracle_diagnostics(oracle_solver* s, double* max_div, double* u_bulk, double* kinetic_energy, double* forcing, int* wm_max_iters);
/* SURVEY.md 8(f) item 4.  dt = cfl / max(|u_c|/dx + |v_c|/dy + |w_c|/dzf), velocities averaged to cell centres (reading S18) */
int oracle_cfl_dt(oracle_solver* s, double cfl, double* dt);
/* x-y plane means per k: out[q][k], q = <u>,<v>,<w>,<uu>,<vv>,<ww>,<uw>,<nu_t> of the centre-averaged velocity */
int oracle_plane_stats(oracle_solver* s, double* out);
/* time-accumulated statistics: accumulate adds weight x (plane means of oracle_plane_stats, wall-shear means);
   get returns the averages prof[8][nz], wall[8] (z walls: tau_xz, tau_yz bottom then top; y walls: tau_xy, tau_zy low then high),
   derived[4] = tau_w, u_tau, Re_tau = u_tau (lz/2)/nu, C_f = 2 tau_w / u_b^2, and the accumulated weight */
int oracle_stats_reset(oracle_solver* s);
int oracle_stats_accumulate(oracle_solver* s, double weight);
int oracle_stats_get(oracle_solver* s, double* prof, double* wall, double* derived, double* weight);
/* threads used by the OpenMP loops */
int oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
