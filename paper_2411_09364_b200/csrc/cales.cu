// cales.cu -- C ABI (include/cales.h) and stream-ordered orchestration of one RK3 step of CaLES on one B200.
//
// Alg. 1 per substep:  K_rhs [-> K_cn_z x3] -> bulk sum -> K_fft_x_fwd(div fused) -> K_fft_y ->
// K_poisson_z -> K_fft_y(inv) -> K_fft_x_inv -> K_correct -> K_wall_stress -> K_smag | K_dsm_*.
// Everything is enqueued on the caller's stream; no host synchronisation inside a step; scalars (bulk shift,
// dynamic coefficients, Newton iteration count) stay in device memory.
#include "../../include/cales.h"
#include "cales_common.cuh"
#include "cales_fft.cuh"
#include "cales_poisson.cuh"
#include "cales_momentum.cuh"
#include "cales_rhs_tile.cuh"
#include "cales_closures.cuh"
#include "cales_smag_tile.cuh"
#include "cales_dsm_col.cuh"
#include "cales_dsm3.cuh"
#ifndef CALES_D3C_TXB
#define CALES_D3C_TXB 64
#endif
#ifndef CALES_D3C_MINB
#define CALES_D3C_MINB 6
#endif
#ifndef CALES_D3T_MINB
#define CALES_D3T_MINB 4
#endif
#ifndef CALES_D3C_NBUF
#define CALES_D3C_NBUF 1
#endif
#include "cales_host.h"

#include <cmath>
#include <cuda.h>
#include <cudaTypedefs.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

using namespace cales;

extern "C" const char* cales_last_error(void) { return g_err.c_str(); }

#define CUDA_TRY(expr)                                                                                     \
  do {                                                                                                     \
    cudaError_t e_ = (expr);                                                                               \
    if (e_ != cudaSuccess) return fail(CALES_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));   \
  } while (0)

struct cales_solver {
  cales_params P;
  Ctx c;
  cudaStream_t st;
  long long N, nxy;
  // fields
  double *u, *v, *w, *p, *nut, *us, *vs, *ws, *Ru, *Rv, *Rw, *W, *CP, *CQ, *smag;
  double *tau, *tau_y;
  // tables
  double *dzf, *dzc, *rdzf, *rdzc, *delta, *zc, *ak, *ck, *lamx, *lamy, *cncoef, *partial, *stage1, *scal, *dsm_part, *dsm_cs;
  double2 *twx, *twy, *dctw;
  int* maxit;
  FftPlan plx, ply;
  PoissonTabs pt;
  WallGeom wg;
  int xB, yTI, y_tish; size_t x_smem, y_smem; int x_threads, y_threads;
  int xBf, xf_threads; size_t xf_smem;      // lines per CTA, threads and shared memory of the forward x transform that forms the divergence
  dim3 pgrid, pblock;   // point kernels
  long long nblk;
  bool fresh;
  long long rhs_tile_min;   // below this many points the momentum kernel runs one thread per point
  long long tile_min;   // grids with at least this many points use the staged z-march for the static model
  int rhs_variant;      // 1 (default): halo planes by 8-byte cp.async (k_rhs_tile); 0: by tiled TMA copies (k_rhs_tile_tma)
  RhsMaps* rmaps; bool rmaps_ok;   // tensor maps of u, v, w, nu_t, p in device memory (workspace)
  bool nut_lazy, nut_valid; int graph_lazy;   // dynamic model: the momentum kernel forms nu_t from |S| and c_s (nut_lazy); s->nut holds it only when nut_valid
  int dsm_col_rows;     // option: output rows per CTA of the column march (0: chosen from the grid)
  double* CPT; int cpt_on;      // static c' table of k_poisson_z (walls in z), option poisson_cp_table
  int fft_stage;        // option: 2 (default) stages the first-pass inputs of the transforms in shared memory (see cales.h); 1: inverse y through registers; 0: off
  int corr_band;        // option: CTA rows per band of k_correct2's launch order (1: plane by plane; 0: chosen from the grid)
  bool part_dirty;      // the partial-sum array may hold entries of another band layout: zero it before the next plane-averaged evaluation
  int corr2;            // option: correction kernel with two points per thread and 16-byte accesses
  int rhs_pf;           // option: R^{k-1} of the next plane prefetched by the staged momentum kernel (0 off, 1 to L1, 2 to L2)
  int rhs_kz;           // option: k-planes per CTA of the staged momentum kernel (0: rt_chunk)
  int lazy_nut;         // option: 1 (default) skips the |S| -> nu_t pass of the dynamic model
  int dsm_col_variant;  // 0: TMA-staged register-window column march (k_dsm_col_tma); 1: shared-ring form of round 1 (k_dsm_col_sm); 2: direct loads (k_dsm_col_rw)
  double rk_dt;   // dt the substep scalar blocks on the device hold (0: none, or a device-side dt)
  double cn_dt;   // dt the Crank-Nicolson tables on the device were built for (0: none, or a device-side dt)
  int use_graph; cudaGraphExec_t gexec;   // the three substeps captured as one CUDA graph (dt lives in device memory: one graph serves every dt)
  double* stats;   // [8 nz + 8 wall + 1 weight] accumulators, the same again as scratch
  double* rks; double* dtdev; double last_dt;   // substep scalar blocks [3][RK_STRIDE], device-side dt of cales_step_adaptive
  int timing; bool ev_valid;
  std::vector<cudaEvent_t> evpool; std::vector<int> evkid; int evn;   // per-launch events of the last timed step
  double kms[32]; int kcnt[32];                                       // per-kernel totals of the last timed step
  int launches;
  int device;
};

// Every entry point runs on the solver's device whatever the caller's current device is, and restores the latter.
struct DevGuard {
  int prev = -1; bool sw = false;
  explicit DevGuard(int dev) { if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) sw = cudaSetDevice(dev) == cudaSuccess; }
  ~DevGuard() { if (sw) cudaSetDevice(prev); }
};
// Switches the per-kernel timing off for launches that are not part of a step; restored on every return path.
struct TimingOff {
  cales_solver* s; int was;
  explicit TimingOff(cales_solver* s_);
  ~TimingOff();
};

TimingOff::TimingOff(cales_solver* s_) : s(s_), was(s_->timing) { s->timing = 0; }
TimingOff::~TimingOff() { s->timing = was; }

static size_t al32(size_t n) { return (n + 31) / 32 * 32; }

// Carve the workspace.  With base == nullptr only the size is computed.
static size_t carve(cales_solver* s, const cales_params* p, double* base) {
  const size_t N = (size_t)p->nx * p->ny * p->nz, nxy = (size_t)p->nx * p->ny;
  size_t off = 0;
  auto take = [&](size_t n) { double* r = base ? base + off : nullptr; off += al32(n); return r; };
  double* f[12];
  for (int q = 0; q < 12; ++q) f[q] = take(N);
  double* CP = take(N);
  double* CQ = p->bc_z == CALES_BC_PERIODIC ? take(N) : nullptr;
  double* CPT = p->bc_z == CALES_BC_WALL ? take(N) : nullptr;      // static c' of the Poisson Thomas solve (k_poisson_cp)
  double* smag = p->sgs_model == CALES_SGS_DSMAG ? take(N) : nullptr;
  double* tau = take(4 * nxy);
  double* tau_y = take(4 * (size_t)p->nx * p->nz);
  double* dzf = take(p->nz + 2); double* dzc = take(p->nz + 2); double* zc = take(p->nz);
  double* rdzf = take(p->nz + 2); double* rdzc = take(p->nz + 2); double* delta = take(p->nz);
  double* ak = take(p->nz); double* ck = take(p->nz);
  double* lamx = take(p->nx); double* lamy = take(p->ny);
  double* twx = take(2 * (size_t)p->nx); double* twy = take(2 * (size_t)p->ny); double* dctw = take(2 * ((size_t)p->ny / 2 + 1));
  double* cncoef = take(18 * (size_t)p->nz);      // Crank-Nicolson coefficient tables of the three substeps
  const size_t nblk = (size_t)((p->nx + 31) / 32) * ((p->ny + 7) / 8) * p->nz;
  double* partial = take(nblk > nxy ? nblk : nxy);
  double* stage1 = take(4 * 1024);
  double* scal = take(32);
  double* stats = take(2 * (8 * (size_t)p->nz + 16));      // on-line statistics: accumulators, then scratch
  double* tmaps = take(128);      // 5 tensor maps of 128 bytes (cales_rhs_tile.cuh)
  const size_t pslots = (size_t)dsm_shape(p->nx).pslots;
  double* dsm_part = p->sgs_model == CALES_SGS_DSMAG ? take((size_t)p->nz * p->ny * pslots * 2) : nullptr;
  double* dsm_cs = p->sgs_model == CALES_SGS_DSMAG ? take((size_t)p->nz * p->ny) : nullptr;
  if (s && base) {
    s->u = f[0]; s->v = f[1]; s->w = f[2]; s->p = f[3]; s->nut = f[4]; s->us = f[5]; s->vs = f[6]; s->ws = f[7];
    s->Ru = f[8]; s->Rv = f[9]; s->Rw = f[10]; s->W = f[11]; s->CP = CP; s->CQ = CQ; s->CPT = CPT; s->smag = smag; s->tau = tau; s->tau_y = tau_y;
    s->dzf = dzf; s->dzc = dzc; s->zc = zc; s->rdzf = rdzf; s->rdzc = rdzc; s->delta = delta; s->ak = ak; s->ck = ck; s->lamx = lamx; s->lamy = lamy;
    s->twx = reinterpret_cast<double2*>(twx); s->twy = reinterpret_cast<double2*>(twy); s->dctw = reinterpret_cast<double2*>(dctw);
    s->cncoef = cncoef; s->partial = partial; s->stage1 = stage1; s->scal = scal; s->maxit = reinterpret_cast<int*>(scal + 16);
    s->rks = scal + 18; s->dtdev = scal + 30;
    s->dsm_part = dsm_part; s->dsm_cs = dsm_cs; s->nblk = (long long)nblk; s->rmaps = reinterpret_cast<RhsMaps*>(tmaps); s->stats = stats;
  }
  return off * sizeof(double);
}

extern "C" void cales_default_params(cales_params* p) {
  if (!p) return;
  std::memset(p, 0, sizeof(*p));
  p->nu = 1e-3; p->cs = 0.17; p->aplus = 25.0; p->dsm_avg_xy_plane = 1; p->kappa = 0.41; p->B = 5.2; p->wm_tol = 1e-4; p->wm_maxit = 50;
}

extern "C" size_t cales_workspace_bytes(const cales_params* p) {
  if (validate(p) != CALES_OK) return 0;
  return carve(nullptr, p, nullptr);
}

// Kernel ids for the per-kernel timing table (cales_kernel_time).
enum { K_RHS = 0, K_CN_COEF, K_CN_Z, K_SUM, K_BULK, K_FFTX_FWD, K_FFTY_FWD, K_POISSON_Z, K_FFTY_INV, K_FFTX_INV, K_CORRECT,
       K_WALL, K_SMAG, K_DSM_PASS1, K_DSM_COL, K_DSM_COEF, K_DSM_NUT, K_FILL, K_TRANSPOSE, K_DIAG, K_DSM3, K_DSM3_COL, K_HELM_Z, K_COUNT };
static const char* const k_names[K_COUNT] = {"k_rhs", "k_cn_coef", "k_cn_z", "k_sum_stage1", "k_bulk_finish", "k_fft_x_fwd", "k_fft_y_fwd",
  "k_poisson_z", "k_fft_y_inv", "k_fft_x_inv", "k_correct", "k_wall_stress", "k_smag", "k_dsm_pass1", "k_dsm_col", "k_dsm_coef", "k_dsm_nut", "k_fill",
  "k_transpose_xy", "k_diag", "k_dsm3_pass1", "k_dsm3_col", "k_helm_z"};

// record an event on the stream tagged with the kernel that just finished (kid < 0: a separator)
static void tick(cales_solver* s, int kid) {
  if (!s->timing) return;
  if (s->evn == (int)s->evpool.size()) { cudaEvent_t e; cudaEventCreate(&e); s->evpool.push_back(e); s->evkid.push_back(-1); }
  s->evkid[s->evn] = kid;
  cudaEventRecord(s->evpool[s->evn], s->st);
  ++s->evn;
}
static int check_launch(cales_solver* s, int kid) {
  ++s->launches;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(CALES_ECUDA, std::string(k_names[kid]) + ": " + cudaGetErrorString(e));
  tick(s, kid);
  return CALES_OK;
}
#define LAUNCH_TRY(kid)                                  \
  do { int rc_ = check_launch(s, kid); if (rc_) return rc_; } while (0)

// Tiled tensor map of an (nx, ny, nz) fp64 field with box (bx, by, 1) (cuTensorMapEncodeTiled through the runtime's driver
// entry point: libcuda is not linked).  False if the driver call is unavailable or rejects the shape.
static bool make_field_map(CUtensorMap* m, const double* base, int nx, int ny, int nz, int bx, int by) {
  static PFN_cuTensorMapEncodeTiled enc = nullptr;
  if (!enc) {
    void* fn = nullptr; cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess || !fn) { cudaGetLastError(); return false; }
    enc = (PFN_cuTensorMapEncodeTiled)fn;
  }
  const cuuint64_t dims[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz};
  const cuuint64_t strides[2] = {(cuuint64_t)nx * 8, (cuuint64_t)nx * ny * 8};
  const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1}, es[3] = {1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Launch shape of an x transform with L lines per CTA; false if the CTA would be too large.
static bool x_launch_shape(const FftPlan& plx, int nx, int L, int* threads, size_t* smem) {
  const int n2 = nx / 2;
  bool has3 = false; for (int q = 0; q < plx.npass; ++q) has3 |= plx.radix[q] == 3;
  const int per_thread = has3 ? 3 * (F2_E / 3) : F2_E;
  long long th = ((long long)L * n2 + per_thread - 1) / per_thread; th = (th + 31) / 32 * 32; if (th < 32) th = 32;
  const size_t sm = (size_t)L * sm_line(n2) * 16;
  if (th > 512 || sm > 200 * 1024 || L < 1 || L > 64 || L > 2 * th) return false;
  *threads = (int)th; *smem = sm;
  return true;
}
static int static_scratch_ptr(int device, double** out);
extern "C" int cales_create(const cales_params* p, cales_solver** out) {
  if (!out) return fail(CALES_EINVAL, "null output pointer");
  *out = nullptr;
  int rc = validate(p);
  if (rc) return rc;
  if (!p->workspace) return fail(CALES_EINVAL, "null workspace");
  if (((size_t)p->workspace) % 256) return fail(CALES_EINVAL, "workspace must be 256-byte aligned");
  const size_t need = carve(nullptr, p, nullptr);
  if (p->workspace_bytes < need) return fail(CALES_EINVAL, "workspace too small");
  DevGuard dg_(p->device);      // the caller's current device is restored on return
  { int cur = -1; if (cudaGetDevice(&cur) != cudaSuccess || cur != p->device) return fail(CALES_ECUDA, "cannot select the device of the workspace"); }
  HostSetup H;
  if ((rc = build_setup(p, H))) return rc;
  cales_solver* s = new cales_solver();
  s->P = H.P;
  s->device = p->device;
  s->st = (cudaStream_t)p->cuda_stream;
  const int nx = p->nx, ny = p->ny, nz = p->nz;
  s->N = (long long)nx * ny * nz; s->nxy = (long long)nx * ny;
  carve(s, p, (double*)p->workspace);
  // ---- upload the tables
  auto up = [&](double* dst, const std::vector<double>& src, size_t n) { return cudaMemcpyAsync(dst, src.data(), n * sizeof(double), cudaMemcpyHostToDevice, s->st); };
  cudaError_t e = cudaSuccess;
  if (e == cudaSuccess) e = cudaMemsetAsync(p->workspace, 0, need, s->st);
  if (e == cudaSuccess) e = up(s->dzf, H.dzf, nz + 2);
  if (e == cudaSuccess) e = up(s->dzc, H.dzc, nz + 1);
  if (e == cudaSuccess) e = up(s->zc, H.zc, nz);
  if (e == cudaSuccess) e = up(s->rdzf, H.rdzf, nz + 2);
  if (e == cudaSuccess) e = up(s->rdzc, H.rdzc, nz + 1);
  if (e == cudaSuccess) e = up(s->delta, H.delta, nz);
  if (e == cudaSuccess) e = up(s->ak, H.ak, nz);
  if (e == cudaSuccess) e = up(s->ck, H.ck, nz);
  if (e == cudaSuccess) e = up(s->lamx, H.lamx, nx);
  if (e == cudaSuccess) e = up(s->lamy, H.lamy, ny);
  if (e == cudaSuccess) e = up(reinterpret_cast<double*>(s->twx), H.twx, H.twx.size());
  if (e == cudaSuccess) e = up(reinterpret_cast<double*>(s->twy), H.twy, H.twy.size());
  if (e == cudaSuccess) e = up(reinterpret_cast<double*>(s->dctw), H.dctw, H.dctw.size());
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->st);
  if (e != cudaSuccess) { delete s; return fail(CALES_ECUDA, std::string("table upload: ") + cudaGetErrorString(e)); }
  s->c = H.c;
  s->c.dzf = s->dzf + 1; s->c.dzc = s->dzc + 1; s->c.zc = s->zc; s->c.rdzf = s->rdzf + 1; s->c.rdzc = s->rdzc + 1; s->c.delta = s->delta; s->c.tau = s->tau; s->c.tau_y = s->tau_y;
  s->pt.ak = s->ak; s->pt.ck = s->ck; s->pt.lamx = s->lamx; s->pt.lamy = s->lamy;
  s->wg = H.wg;
  s->plx = H.plx; s->plx.tw = s->twx;
  s->ply = H.ply; s->ply.tw = s->twy; s->ply.dctw = s->dctw;
  s->xB = H.xB; s->x_smem = H.x_smem; s->x_threads = H.x_threads;
  s->yTI = H.yTI; s->y_tish = H.y_tish; s->y_smem = H.y_smem; s->y_threads = H.y_threads;
  s->xBf = s->xB; s->xf_threads = s->x_threads; s->xf_smem = s->x_smem;
  {
    // Small CTAs for the x transforms (B200, ms per launch).  Forward with the divergence pre-pass -- config 5 (n2 = 768): 5 lines 7.43,
    // 2: 7.04, 1: 6.32; config 4 (512): 8 lines 0.680, 2: 0.510, 1: 0.520; config 3 (128): 32 lines 0.258, 8: 0.125, 4: 0.109, 2: 0.108;
    // config 2 (96): 42 lines 0.053, 4: 0.020.  Its serial phases (batched loads of a line, butterflies, split) overlap across CTAs, not
    // inside one: many CTAs of 32-64 threads hide the load latency that two CTAs of 256 could not.  Inverse (lines staged by bulk
    // copies) -- config 5: 5 lines 4.13, 2: 4.25, 1: 4.52; config 4: 8 lines 0.341, 2: 0.296; config 3: 32 lines 0.0755, 4: 0.063.
    const int n2 = nx / 2;
    const long long nlines = (long long)ny * nz;
    int Lf = 512 / (n2 > 0 ? n2 : 1); if (Lf < 1) Lf = 1; if (Lf > 64) Lf = 64; if (Lf > nlines) Lf = (int)nlines;
    int th; size_t sm;
    if (Lf < s->xB && x_launch_shape(s->plx, nx, Lf, &th, &sm)) { s->xBf = Lf; s->xf_threads = th; s->xf_smem = sm; }      // never more lines than the host plan (small grids: enough CTAs)
    if (n2 < 640) {
      int Li = 1024 / (n2 > 0 ? n2 : 1); if (Li < 1) Li = 1; if (Li > 64) Li = 64; if (Li > nlines) Li = (int)nlines;
      if (Li < s->xB && x_launch_shape(s->plx, nx, Li, &th, &sm)) { s->xB = Li; s->x_threads = th; s->x_smem = sm; }
    }
  }
  e = cudaFuncSetAttribute(k_fft2_x_fwd<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fft2_x_fwd<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fft2_x_inv, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fft2_y, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rhs_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(RT_SMEM_DOUBLES * sizeof(double)));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rhs_tile_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RT_SMEM_TMA_BYTES);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_smag_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(ST_SMEM_DOUBLES * sizeof(double)));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dsm_pass1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(DSM_SMEM_DOUBLES * sizeof(double)));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dsm3_pass1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(D3_SMEM_DOUBLES * sizeof(double)));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dsm3_col_tma<64, CALES_D3T_MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DSM3T_RAW_BYTES);
  if (e != cudaSuccess) { delete s; return fail(CALES_ECUDA, std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e)); }
  s->pblock = dim3(32, 8, 1);
  s->pgrid = dim3((nx + 31) / 32, (ny + 7) / 8, nz);
  s->fresh = false; s->timing = 0; s->ev_valid = false; s->launches = 0; s->evn = 0;
  s->use_graph = 1; s->gexec = nullptr; s->last_dt = 0.0;
  s->cn_dt = 0.0; s->rk_dt = 0.0;
  s->tile_min = 4000000;
  s->rhs_tile_min = 200000;
  s->dsm_col_variant = 0;
  s->nut_lazy = false; s->nut_valid = true; s->graph_lazy = -1; s->lazy_nut = 1; s->dsm_col_rows = 0; s->rhs_kz = 0; s->rhs_pf = 1; s->corr2 = 1; s->part_dirty = false; s->corr_band = 0; s->fft_stage = 2;
  s->rhs_variant = 1;      // measured on B200 at config 5: cp.async ring 22.7 ms, tiled TMA ring 25.1 ms per launch
  {
    const double* fl[RT_NF] = {s->u, s->v, s->w, s->nut, s->p};
    RhsMaps hm;
    s->rmaps_ok = true;
    for (int f = 0; f < RT_NF; ++f) s->rmaps_ok = s->rmaps_ok && make_field_map(&hm.m[f], fl[f], nx, ny, nz, RTT_TW, RT_TH);
    if (s->rmaps_ok && (cudaMemcpyAsync(s->rmaps, &hm, sizeof(hm), cudaMemcpyHostToDevice, s->st) != cudaSuccess || cudaStreamSynchronize(s->st) != cudaSuccess)) { cudaGetLastError(); s->rmaps_ok = false; }
  }
  s->cpt_on = s->CPT ? 2 : 0;
  if (s->CPT) {      // static c' of the Poisson columns (the matrix never changes)
    k_poisson_cp<<<(unsigned)((s->nxy + 127) / 128), 128, 0, s->st>>>(s->c, s->pt, s->CPT);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->st);
    if (e != cudaSuccess) { delete s; return fail(CALES_ECUDA, std::string("k_poisson_cp: ") + cudaGetErrorString(e)); }
  }
  for (int q = 0; q < 32; ++q) { s->kms[q] = 0.0; s->kcnt[q] = 0; }
  { double* ss_ = nullptr; (void)static_scratch_ptr(s->device, &ss_); }      // set-up of cales_cfl_dt_static; a failure is reported by that call
  *out = s;
  return CALES_OK;
}

extern "C" int cales_create_basic(int nx, int ny, int nz, double lx, double ly, double lz, int zstretch, double zstretch_factor,
                                  int bc_y, int bc_z, double nu, int sgs_model, int wall_model, int implicit_z,
                                  void* workspace, size_t workspace_bytes, void* cuda_stream, int device, cales_solver** out) {
  cales_params p; cales_default_params(&p);
  p.nx = nx; p.ny = ny; p.nz = nz; p.lx = lx; p.ly = ly; p.lz = lz; p.zstretch = zstretch; p.zstretch_factor = zstretch_factor;
  p.bc_y = bc_y; p.bc_z = bc_z; p.nu = nu; p.sgs_model = sgs_model; p.wall_model = wall_model; p.implicit_z = implicit_z;
  p.workspace = workspace; p.workspace_bytes = workspace_bytes; p.cuda_stream = cuda_stream; p.device = device;
  return cales_create(&p, out);
}

extern "C" int cales_destroy(cales_solver* s) {
  DevGuard dg_(s ? s->device : -1);
  if (!s) return CALES_OK;
  for (cudaEvent_t e : s->evpool) cudaEventDestroy(e);
  if (s->gexec) cudaGraphExecDestroy(s->gexec);
  delete s;
  return CALES_OK;
}

static int ensure_nut(cales_solver* s);
static double* field_ptr(cales_solver* s, int f) {
  switch (f) { case CALES_U: return s->u; case CALES_V: return s->v; case CALES_W: return s->w; case CALES_P: return s->p; case CALES_NUT: return s->nut; }
  return nullptr;
}

extern "C" int cales_set_field(cales_solver* s, int field, const double* src, int on_device) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !src) return fail(CALES_EINVAL, "null argument");
  double* d = field_ptr(s, field);
  if (!d) return fail(CALES_EINVAL, "bad field id");
  CUDA_TRY(cudaMemcpyAsync(d, src, s->N * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s->st));
  // the wall faces are kept at exactly 0 (include/cales.h; the interior kernels rely on it)
  if (field == CALES_V && s->c.bc_y == BC_WALL)
    CUDA_TRY(cudaMemset2DAsync(d + (size_t)(s->c.ny - 1) * s->c.nx, (size_t)s->nxy * sizeof(double), 0, (size_t)s->c.nx * sizeof(double), (size_t)s->c.nz, s->st));
  if (field == CALES_W && s->c.bc_z == BC_WALL)
    CUDA_TRY(cudaMemsetAsync(d + (size_t)(s->c.nz - 1) * s->nxy, 0, (size_t)s->nxy * sizeof(double), s->st));
  if (!on_device) CUDA_TRY(cudaStreamSynchronize(s->st));
  if (field <= CALES_W) s->fresh = false;
  if (field == CALES_NUT) { s->nut_lazy = false; s->nut_valid = true; }      // the caller's nu_t is taken as it is
  return CALES_OK;
}
extern "C" int cales_get_field(cales_solver* s, int field, double* dst, int on_device) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !dst) return fail(CALES_EINVAL, "null argument");
  double* d = field_ptr(s, field);
  if (!d) return fail(CALES_EINVAL, "bad field id");
  if (field == CALES_NUT) { int rc = ensure_nut(s); if (rc) return rc; }
  CUDA_TRY(cudaMemcpyAsync(dst, d, s->N * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s->st));
  if (!on_device) CUDA_TRY(cudaStreamSynchronize(s->st));
  return CALES_OK;
}

// ---- building blocks ------------------------------------------------------------------------------------------
static int run_transform_x_fwd(cales_solver* s, const double* src, const DivSrc* ds, double* dst) {
  const long long nlines = (long long)s->c.ny * s->c.nz;
  const unsigned grid = (unsigned)((nlines + s->xB - 1) / s->xB);
  if (ds) k_fft2_x_fwd<true><<<(unsigned)((nlines + s->xBf - 1) / s->xBf), s->xf_threads, s->xf_smem, s->st>>>(s->c, s->plx, s->xBf, nullptr, *ds, dst, (s->fft_stage && s->plx.npass > 0) ? 1 : 0);
  else { DivSrc z{nullptr, nullptr, nullptr, 0.0, nullptr}; k_fft2_x_fwd<false><<<grid, s->x_threads, s->x_smem, s->st>>>(s->c, s->plx, s->xB, src, z, dst, 0); }
  LAUNCH_TRY(K_FFTX_FWD);
  return CALES_OK;
}
static int run_transform_x_inv(cales_solver* s, const double* src, double* dst) {
  const long long nlines = (long long)s->c.ny * s->c.nz;
  const unsigned grid = (unsigned)((nlines + s->xB - 1) / s->xB);
  const int staged = s->fft_stage && (((size_t)src) & 15) == 0 && s->plx.npass > 0;
  k_fft2_x_inv<<<grid, s->x_threads, s->x_smem, s->st>>>(s->c, s->plx, s->xB, src, dst, staged);
  LAUNCH_TRY(K_FFTX_INV);
  return CALES_OK;
}
static int run_transform_y(cales_solver* s, double* A, int inverse) {
  dim3 grid((s->c.nx + s->yTI - 1) / s->yTI, s->c.nz);
  const bool stage_ok = s->fft_stage && (((size_t)A) & 15) == 0 && s->ply.npass > 0 && (size_t)s->c.ny * s->yTI * 8 <= s->y_smem;
  const int staged = (stage_ok && inverse) ? (s->fft_stage >= 2 ? 2 : 1) : 0;
  k_fft2_y<<<grid, s->y_threads, s->y_smem, s->st>>>(s->c, s->ply, s->y_tish, s->c.bc_y == BC_WALL ? 1 : 0, inverse, A, staged);
  LAUNCH_TRY(inverse ? K_FFTY_INV : K_FFTY_FWD);
  return CALES_OK;
}
static int run_poisson_z(cales_solver* s, double* A) {
  const int th = (s->nxy / 128 < 4 * 148) ? 64 : 128;      // small planes: smaller CTAs spread over more SMs
  if (s->cpt_on == 2 && s->CPT && (((size_t)A) & 15) == 0) k_poisson_z2<<<(unsigned)((s->nxy / 2 + th - 1) / th), th, 0, s->st>>>(s->c, s->pt, A, s->CP, s->CPT);
  else k_poisson_z<<<(unsigned)((s->nxy + th - 1) / th), th, 0, s->st>>>(s->c, s->pt, A, s->CP, s->CQ, s->cpt_on ? s->CPT : nullptr);
  LAUNCH_TRY(K_POISSON_Z);
  return CALES_OK;
}
// spectral part of the Poisson solve, W already holds the x-transformed right-hand side
static int run_poisson_core(cales_solver* s) {
  int rc;
  if ((rc = run_transform_y(s, s->W, 0))) return rc;
  if ((rc = run_poisson_z(s, s->W))) return rc;
  if ((rc = run_transform_y(s, s->W, 1))) return rc;
  return CALES_OK;
}
static int run_wall_stress(cales_solver* s) {
  if (!s->c.wall_model && !s->c.wall_model_y) return CALES_OK;
  CUDA_TRY(cudaMemsetAsync(s->maxit, 0, sizeof(int), s->st));
  tick(s, -1);
  if (s->c.wall_model) {
    dim3 grid(s->pgrid.x, s->pgrid.y, 4);
    k_wall_stress<<<grid, s->pblock, 0, s->st>>>(s->c, s->wg, s->u, s->v, s->tau, s->maxit);
    LAUNCH_TRY(K_WALL);
  }
  if (s->c.wall_model_y) {
    dim3 grid((s->c.nx + 31) / 32, (s->c.nz + 7) / 8, 4);
    k_wall_stress_y<<<grid, dim3(32, 8), 0, s->st>>>(s->c, s->u, s->w, s->tau_y, s->maxit);
    LAUNCH_TRY(K_WALL);
  }
  return CALES_OK;
}
// the |S| -> nu_t pass can be skipped when the momentum kernel that will consume nu_t forms it itself (every form but the TMA variant)
static bool lazy_ok(const cales_solver* s) { return s->lazy_nut != 0 && !(s->rhs_variant == 0 && s->rmaps_ok && s->N >= s->rhs_tile_min); }
static int run_eddy_viscosity(cales_solver* s, const double* u, const double* v, const double* w, double* nut) {
  if (s->c.sgs == CALES_SGS_NONE) {
    k_fill<<<1184, 256, 0, s->st>>>(nut, s->N, 0.0);
    LAUNCH_TRY(K_FILL);
  } else if (s->c.sgs == CALES_SGS_SMAG) {
    if (s->N >= s->tile_min) {      // HBM-sized grids: staged z-march; launch-bound sizes: one thread per point
      const int kz = rt_chunk(s->c.nx, s->c.ny, s->c.nz);
      const dim3 g((s->c.nx + RT_TX - 1) / RT_TX, (s->c.ny + RT_TY - 1) / RT_TY, (s->c.nz + kz - 1) / kz);
      k_smag_tile<<<g, RT_THREADS, ST_SMEM_DOUBLES * sizeof(double), s->st>>>(s->c, u, v, w, kz, nut);
    } else k_smag<<<s->pgrid, s->pblock, 0, s->st>>>(s->c, u, v, w, nut);
    LAUNCH_TRY(K_SMAG);
  } else {
    // pass 1: the column-marching kernel wherever the test filter is uniform in y; the tile kernel (Eq. 9 literally) on
    // the DSM_TY rows next to each y wall, where filter and strain do not commute
    const Ctx& c = s->c;
    const DsmShape ds = dsm_shape(c.nx);
    if (s->part_dirty) {      // an option changed the band layout of the column marches: their never-written slots must read 0
      CUDA_TRY(cudaMemsetAsync(s->dsm_part, 0, (size_t)c.nz * c.ny * ds.pslots * 2 * sizeof(double), s->st));
      s->part_dirty = false;
    }
    const bool ywall = c.bc_y == BC_WALL;
    const bool split = ywall && c.ny >= 3 * DSM_TY;
    const size_t tile_smem = DSM_SMEM_DOUBLES * sizeof(double);
    const unsigned ntile = (unsigned)((c.nx + DSM_TX - 1) / DSM_TX);
    if (c.dsm_filter3d) {   // 3-D box filter: Eq. 9 literally on 3x3x3 patches, every row
      // column-marching kernel where filter and strain commute (uniform z, two layers away from every wall), the tile
      // kernel on the planes and rows next to the walls (or everywhere on a stretched grid)
      const D3Split sp = d3_split(c, s->P.zstretch == CALES_Z_UNIFORM);
      const dim3 tb(D3_TX, D3_TY);
      const unsigned ntx3 = (unsigned)((c.nx + D3_TX - 1) / D3_TX), nty3 = (unsigned)((c.ny + D3_TY - 1) / D3_TY);
      const size_t sm3 = D3_SMEM_DOUBLES * sizeof(double);
      if (!sp.col) {
        k_dsm3_pass1<<<dim3(ntx3, nty3, c.nz), tb, sm3, s->st>>>(c, u, v, w, c.nz, 0, D3_TY, c.ny, c.ny, ds.pslots, s->smag, s->dsm_part);
        LAUNCH_TRY(K_DSM3);
      } else {
        if (sp.klo > 0) {          // planes 0, 1, nz-2, nz-1: every row
          k_dsm3_pass1<<<dim3(ntx3, nty3, 2 * sp.klo), tb, sm3, s->st>>>(c, u, v, w, sp.klo, c.nz - 2 * sp.klo, D3_TY, c.ny, c.ny, ds.pslots, s->smag, s->dsm_part);
          LAUNCH_TRY(K_DSM3);
        }
        if (sp.jlo > 0) {          // the other planes: rows 0, 1, ny-2, ny-1
          k_dsm3_pass1<<<dim3(ntx3, 2, sp.khi - sp.klo), tb, sm3, s->st>>>(c, u, v, w, 0, sp.klo, c.ny - D3_TY, sp.jlo, sp.jhi, ds.pslots, s->smag, s->dsm_part);
          LAUNCH_TRY(K_DSM3);
        }
        // <threads, min CTAs/SM, row buffers>: measured on B200 (config 4): (64,4,2) 6.46 ms, (64,6,1) 6.16 ms, (64,8,1) 7.45 ms (spills)
        // dsm_col_variant 0 (default): rows staged by bulk copies, y-window in registers (k_dsm3_col_tma; needs 16-byte aligned rows and
        // nx >= 66); otherwise the shared-ring march of round 1
        if (s->dsm_col_variant == 0 && (((size_t)u | (size_t)v | (size_t)w) & 15) == 0 && c.nx >= 66) {
          int ly = s->dsm_col_rows;
          if (ly <= 0) ly = (sp.jhi - sp.jlo >= 512) ? 256 : ((sp.jhi - sp.jlo >= 192) ? 128 : 32);      // B200, config 5: 32: 40.6, 64: 39.5, 128: 38.9, 256: 38.3 ms
          k_dsm3_col_tma<64, CALES_D3T_MINB><<<dim3(ds.nbx, sp.khi - sp.klo, (unsigned)((sp.jhi - sp.jlo + ly - 1) / ly)), 64, DSM3T_RAW_BYTES, s->st>>>(c, u, v, w, sp.klo, sp.jlo, sp.jhi, ly, ds.pslots, s->smag, s->dsm_part);
        } else
          k_dsm3_col<CALES_D3C_TXB, CALES_D3C_MINB, CALES_D3C_NBUF><<<dim3(ds.nbx, (sp.jhi - sp.jlo + DSMC_LY - 1) / DSMC_LY, sp.khi - sp.klo), CALES_D3C_TXB, 0, s->st>>>(c, u, v, w, sp.klo, sp.jlo, sp.jhi, ds.pslots, s->smag, s->dsm_part);
        LAUNCH_TRY(K_DSM3_COL);
      }
    } else if (ywall) {
      if (split) k_dsm_pass1<<<dim3(ntile, 2, c.nz), dim3(DSM_TX, DSM_TY), tile_smem, s->st>>>(c, u, v, w, c.ny - DSM_TY, DSM_TY, c.ny - DSM_TY, ds.pslots, s->smag, s->dsm_part);
      else k_dsm_pass1<<<dim3(ntile, (c.ny + DSM_TY - 1) / DSM_TY, c.nz), dim3(DSM_TX, DSM_TY), tile_smem, s->st>>>(c, u, v, w, DSM_TY, c.ny, c.ny, ds.pslots, s->smag, s->dsm_part);
      LAUNCH_TRY(K_DSM_PASS1);
    }
    if (!c.dsm_filter3d && (!ywall || split)) {
      const int jlo = ywall ? DSM_TY : 0, jhi = ywall ? c.ny - DSM_TY : c.ny;
      dim3 grid(ds.nbx, (jhi - jlo + DSMC_LY - 1) / DSMC_LY, c.nz);
      // register-window form (cales_dsm_col.cuh); the shared-ring form of round 1 stays selectable for A/B timing
      // variant 0 (default): TMA-staged march on the planes without z-wall ghosts, the direct-load march on the others;
      // bulk copies need 16-byte aligned rows (nx is even, so the field pointers decide) and nx >= 66
      const bool tma_ok = s->dsm_col_variant == 0 && (((size_t)u | (size_t)v | (size_t)w) & 15) == 0 && c.nx >= 66;
      // rows per CTA of the register-window marches: every CTA spends two rows filling its y-window, long bands leave a ragged
      // tail.  Measured on B200 (eddy viscosity, ms): config 5 (1024 rows) 32: 22.9, 64: 22.1, 128: 22.4, 256: 23.5; config 4
      // (252 rows) 32: 2.99, 64: 3.38, 128: 4.32
      int ly = s->dsm_col_rows;
      if (ly <= 0) ly = (jhi - jlo >= 512) ? 64 : 32;
      const unsigned nby = (unsigned)((jhi - jlo + ly - 1) / ly);
      if (tma_ok) {
        const int klo = c.bc_z == BC_PER ? 0 : 1, khi = c.bc_z == BC_PER ? c.nz : c.nz - 1;
        k_dsm_col_tma<64, CALES_DSMR_MINB><<<dim3(ds.nbx, khi - klo, nby), 64, 0, s->st>>>(c, u, v, w, klo, jlo, jhi, ly, ds.pslots, s->smag, s->dsm_part);
        if (klo > 0) { LAUNCH_TRY(K_DSM_COL); k_dsm_col_rw<64, CALES_DSMR_MINB><<<dim3(ds.nbx, 2, nby), 64, 0, s->st>>>(c, u, v, w, 0, c.nz - 1, jlo, jhi, ly, ds.pslots, s->smag, s->dsm_part); }
      } else if (s->dsm_col_variant != 1) k_dsm_col_rw<64, CALES_DSMR_MINB><<<dim3(ds.nbx, c.nz, nby), 64, 0, s->st>>>(c, u, v, w, 0, 1, jlo, jhi, ly, ds.pslots, s->smag, s->dsm_part);
      else k_dsm_col_sm<64, 6, 0><<<dim3(ds.nbx, grid.y, grid.z), 64, 0, s->st>>>(c, u, v, w, jlo, jhi, ds.pslots, s->smag, s->dsm_part);
      LAUNCH_TRY(K_DSM_COL);
    }
    k_dsm_coef<<<s->c.nz, 128, 0, s->st>>>(s->c, s->dsm_part, ds.pslots, s->dsm_cs);
    LAUNCH_TRY(K_DSM_COEF);
    if (nut == s->nut && lazy_ok(s)) {
      // the solver's own nu_t stays implicit: |S| in s->smag, c_s in s->dsm_cs; the momentum kernel forms c_s Delta^2 |S| (with the
      // clip) when it stages the plane, cales_get_field / the statistics materialise it on demand (ensure_nut)
      s->nut_lazy = true; s->nut_valid = false;
    } else {
      k_dsm_nut<<<s->pgrid, s->pblock, 0, s->st>>>(s->c, s->dsm_cs, s->smag, nut);
      LAUNCH_TRY(K_DSM_NUT);
      if (nut == s->nut) { s->nut_lazy = false; s->nut_valid = true; }
    }
    return CALES_OK;
  }
  if (nut == s->nut) { s->nut_lazy = false; s->nut_valid = true; }
  return CALES_OK;
}
// s->nut as an array of nu_t values (the lazy dynamic model keeps |S| and c_s instead)
static int ensure_nut(cales_solver* s) {
  if (!s->nut_lazy || s->nut_valid) return CALES_OK;
  TimingOff toff(s);
  k_dsm_nut<<<s->pgrid, s->pblock, 0, s->st>>>(s->c, s->dsm_cs, s->smag, s->nut);
  LAUNCH_TRY(K_DSM_NUT);
  s->nut_valid = true;
  return CALES_OK;
}
// Alg. 2 on the current velocity, then nu_t (Alg. 1 l.2 / l.12)
static int refresh_closures(cales_solver* s) {
  int rc;
  if ((rc = run_wall_stress(s))) return rc;
  if ((rc = run_eddy_viscosity(s, s->u, s->v, s->w, s->nut))) return rc;
  s->fresh = true;
  return CALES_OK;
}

// CTA rows (8 grid rows each) per band of k_correct2's launch order.  A plane of its nine streams that fits L2 keeps the plane order;
// otherwise bands of about 16 MB (B200, config 5, ms per launch: plane order 9.27, 16 rows 9.15, 32: 8.61, 64: 8.54, 128: 8.46, 256: 8.45,
// 512: 8.65; config 4, whose plane is 19 MB: plane order 0.703, banded 0.706-0.741).
static int corr_band(const cales_solver* s) {
  if (s->corr_band > 0) return s->corr_band;
  const double plane = 72.0 * (double)s->nxy;
  if (plane <= 32.0 * 1048576.0) return 1;
  const int b = (int)(16.0 * 1048576.0 / (72.0 * 8.0 * (double)s->c.nx));
  return b < 1 ? 1 : b;
}
static int substep(cales_solver* s, int rk) {
  int rc;
  double al, be, ga; rk3_coeffs(rk, al, be, ga);
  const Ctx& c = s->c;
  const bool cfr = c.const_flow_rate != 0, imp = c.implicit_z == 1, imp3 = c.implicit_z == 2;
  RhsArgs a;
  a.u = s->u; a.v = s->v; a.w = s->w; a.p = s->p; a.nut = s->nut_lazy ? s->smag : s->nut; a.cs = s->nut_lazy ? s->dsm_cs : nullptr;
  a.Ru0 = s->Ru; a.Rv0 = s->Rv; a.Rw0 = s->Rw; a.Ru1 = s->Ru; a.Rv1 = s->Rv; a.Rw1 = s->Rw;
  const double* sc = s->rks + rk * RK_STRIDE;      // dt, gamma dt, 1/(gamma dt), gamma nu dt / 2 of this substep, in device memory
  a.us = s->us; a.vs = s->vs; a.ws = s->ws; a.dt = 0.0; a.al = al; a.be = be; a.ga = ga; a.store_R = rk < 2 ? 1 : 0; a.sc = sc;
  const int kz = s->rhs_kz > 0 ? s->rhs_kz : rt_chunk(c.nx, c.ny, c.nz);
  dim3 rgrid((c.nx + RT_TX - 1) / RT_TX, (c.ny + RT_TY - 1) / RT_TY, (c.nz + kz - 1) / kz);
  if (s->N >= s->rhs_tile_min && s->rhs_variant == 0 && s->rmaps_ok) k_rhs_tile_tma<<<rgrid, RT_THREADS, RT_SMEM_TMA_BYTES, s->st>>>(c, a, s->rmaps, kz, (cfr && !imp && !imp3) ? s->partial : nullptr);
  else if (s->N >= s->rhs_tile_min) k_rhs_tile<<<rgrid, RT_THREADS, RT_SMEM_DOUBLES * sizeof(double), s->st>>>(c, a, kz, (cfr && !imp && !imp3) ? s->partial : nullptr, s->rhs_pf);
  else { rgrid = s->pgrid; k_rhs_point<<<s->pgrid, s->pblock, 0, s->st>>>(c, a, (cfr && !imp && !imp3) ? s->partial : nullptr); }
  LAUNCH_TRY(K_RHS);
  long long npart = (long long)rgrid.x * rgrid.y * rgrid.z;
  if (imp) {
    const int th = (s->nxy / 128 < 4 * 148) ? 64 : 128; const unsigned g = (unsigned)((s->nxy + th - 1) / th);
    k_cn_z<<<dim3(g, 3), th, 0, s->st>>>(c, s->cncoef + (size_t)rk * 6 * c.nz, s->us, s->vs, s->ws, cfr ? s->partial : nullptr); LAUNCH_TRY(K_CN_Z);
    npart = g;
  }
  if (imp3) {
    // Eq. 18: three modified Helmholtz solves with the transforms of the Poisson solver and a shifted tridiagonal system in z;
    // us, vs, ws hold the right-hand sides u** - c L u^k and receive u*
    double* Q[3] = {s->us, s->vs, s->ws};
    const int th = (s->nxy / 128 < 4 * 148) ? 64 : 128;
    for (int comp = 0; comp < 3; ++comp) {
      if ((rc = run_transform_x_fwd(s, Q[comp], nullptr, s->W))) return rc;
      if ((rc = run_transform_y(s, s->W, 0))) return rc;
      k_helm_z<<<(unsigned)((s->nxy + th - 1) / th), th, 0, s->st>>>(c, s->pt, comp == 2 ? 1 : 0, sc, s->W, s->CP, s->CQ);
      LAUNCH_TRY(K_HELM_Z);
      if ((rc = run_transform_y(s, s->W, 1))) return rc;
      if ((rc = run_transform_x_inv(s, s->W, Q[comp]))) return rc;
    }
    if (cfr) {
      k_weighted_sum<<<s->pgrid, s->pblock, 0, s->st>>>(c, s->us, s->partial); LAUNCH_TRY(K_SUM);
      npart = s->nblk;
    }
  }
  if (cfr) {
    const int g1 = (int)(npart < 1024 ? npart : 1024);
    k_sum_stage1<<<g1, 256, 0, s->st>>>(s->partial, npart, s->stage1); LAUNCH_TRY(K_SUM);
    k_bulk_finish<<<1, 256, 0, s->st>>>(c, s->stage1, g1, 0.0, sc, s->scal); LAUNCH_TRY(K_BULK);
  }
  DivSrc ds{s->us, s->vs, s->ws, 0.0, sc};
  if ((rc = run_transform_x_fwd(s, nullptr, &ds, s->W))) return rc;
  if ((rc = run_poisson_core(s))) return rc;
  if ((rc = run_transform_x_inv(s, s->W, s->W))) return rc;
  CorrArgs ca;
  ca.phi = s->W; ca.us = s->us; ca.vs = s->vs; ca.ws = s->ws; ca.u = s->u; ca.v = s->v; ca.w = s->w; ca.p = s->p;
  ca.shift = cfr ? s->scal : nullptr; ca.gdt = 0.0; ca.cimp = (imp || imp3) ? 1.0 : 0.0; ca.cxy = imp3 ? 1.0 : 0.0; ca.update_p = 1; ca.sc = sc;
  if (imp3) k_correct<true><<<s->pgrid, s->pblock, 0, s->st>>>(c, ca);
  else if (s->corr2 && c.nx >= 4) k_correct2<<<dim3((c.nx / 2 + 31) / 32, s->pgrid.y, s->pgrid.z), s->pblock, 0, s->st>>>(c, ca, corr_band(s));
  else k_correct<false><<<s->pgrid, s->pblock, 0, s->st>>>(c, ca);
  LAUNCH_TRY(K_CORRECT);
  if ((rc = run_wall_stress(s))) return rc;
  if ((rc = run_eddy_viscosity(s, s->u, s->v, s->w, s->nut))) return rc;
  return CALES_OK;
}

extern "C" int cales_launches_per_step(cales_solver* s);

// The three substeps on the stream: replayed as one CUDA graph (launch-bound sizes: ~25-120 launches of a few microseconds
// each), or as plain launches while per-kernel timing is on.  dt and everything derived from it live in device memory
// (s->rks), so the captured graph serves every dt and nothing here synchronises.
static int run_substeps(cales_solver* s) {
  int rc;
  if (s->part_dirty && s->dsm_part) {      // outside any capture: the graph must not carry this memset into every replay
    CUDA_TRY(cudaMemsetAsync(s->dsm_part, 0, (size_t)s->c.nz * s->c.ny * dsm_shape(s->c.nx).pslots * 2 * sizeof(double), s->st));
    s->part_dirty = false;
  }
  if (s->use_graph && !s->timing) {
    if (s->gexec && s->graph_lazy != (int)s->nut_lazy) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }   // the first substep's nu_t source is baked in
    if (s->gexec) {
      const bool dsm = s->c.sgs == CALES_SGS_DSMAG;
      if (dsm) { s->nut_lazy = lazy_ok(s); s->nut_valid = !s->nut_lazy; }      // what the replayed substeps leave behind
      CUDA_TRY(cudaGraphLaunch(s->gexec, s->st));
      s->launches += cales_launches_per_step(s);
      return CALES_OK;
    }
    cudaGraph_t g = nullptr;
    if (cudaStreamBeginCapture(s->st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      rc = CALES_OK;
      const int l0 = s->launches;
      s->graph_lazy = (int)s->nut_lazy;
      for (int rk = 0; rk < 3 && rc == CALES_OK; ++rk) rc = substep(s, rk);
      const cudaError_t ee = cudaStreamEndCapture(s->st, &g);
      if (rc == CALES_OK && ee == cudaSuccess && g && cudaGraphInstantiate(&s->gexec, g, 0) == cudaSuccess) {
        cudaGraphDestroy(g);
        CUDA_TRY(cudaGraphLaunch(s->gexec, s->st));
        return CALES_OK;
      }
      s->launches = l0;
      if (g) cudaGraphDestroy(g);
      s->gexec = nullptr; s->use_graph = 0;      // capture unavailable: plain launches from now on
      cudaGetLastError();
      if (rc) return rc;
    } else { s->use_graph = 0; cudaGetLastError(); }
  }
  tick(s, -1);
  for (int rk = 0; rk < 3; ++rk) if ((rc = substep(s, rk))) return rc;
  s->ev_valid = s->timing != 0;
  return CALES_OK;
}

// dt-dependent device tables of a step: the substep scalar blocks and, with implicit z, the Crank-Nicolson tables of Eq. 21
// (the forward elimination of the constant matrix is a serial recurrence over nz levels, one thread per substep).
static int prepare_dt(cales_solver* s, double dt, const double* dt_dev) {
  if (dt_dev || dt != s->rk_dt) {      // the blocks persist in device memory: a repeated host-side dt costs nothing
    k_rk_scalars<<<1, 32, 0, s->st>>>(dt, dt_dev, s->c.nu, s->rks);
    LAUNCH_TRY(K_CN_COEF);
    s->rk_dt = dt_dev ? 0.0 : dt;
  }
  if (s->c.implicit_z == 1 && (dt_dev || dt != s->cn_dt)) {
    k_cn_coef<<<1, 32, 0, s->st>>>(s->c, s->rks, s->cncoef);
    LAUNCH_TRY(K_CN_COEF);
    s->cn_dt = dt_dev ? 0.0 : dt;
  }
  return CALES_OK;
}

extern "C" int cales_step(cales_solver* s, double dt) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !(dt > 0.0)) return fail(CALES_EINVAL, "bad step arguments");
  int rc;
  s->launches = 0; s->evn = 0; s->ev_valid = false;
  if (!s->fresh && (rc = refresh_closures(s))) return rc;
  { TimingOff toff(s); rc = prepare_dt(s, dt, nullptr); }      // the two table kernels are not part of the timed step
  if (rc) return rc;
  if (s->nut_lazy && !lazy_ok(s)) { if ((rc = ensure_nut(s))) return rc; s->nut_lazy = false; }
  s->last_dt = dt;
  return run_substeps(s);
}

// One step with dt = cfl / max(|u_c|/dx + |v_c|/dy + |w_c|/dzf) of the current field (a fixed fraction of the
// stability limit, reading S18), the reduction and everything derived from dt staying on the device: no host synchronisation.
extern "C" int cales_step_adaptive(cales_solver* s, double cfl) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !(cfl > 0.0)) return fail(CALES_EINVAL, "bad step arguments");
  int rc;
  s->launches = 0; s->evn = 0; s->ev_valid = false;
  if (!s->fresh && (rc = refresh_closures(s))) return rc;
  rc = CALES_OK;
  do {
    TimingOff toff(s);
    double* part = s->CP;   // scratch, nblk <= N
    k_cfl_rate<<<s->pgrid, s->pblock, 0, s->st>>>(s->c, s->u, s->v, s->w, part);
    if ((rc = check_launch(s, K_DIAG))) break;
    const long long nb = s->nblk; const int g1 = (int)(nb < 1024 ? nb : 1024);
    k_max_stage<<<g1, 256, 0, s->st>>>(part, nb, s->stage1);
    if ((rc = check_launch(s, K_SUM))) break;
    k_dt_finish<<<1, 256, 0, s->st>>>(s->stage1, g1, cfl, s->dtdev);
    if ((rc = check_launch(s, K_SUM))) break;
    rc = prepare_dt(s, 0.0, s->dtdev);
  } while (0);
  if (rc) return rc;
  if (s->nut_lazy && !lazy_ok(s)) { if ((rc = ensure_nut(s))) return rc; s->nut_lazy = false; }
  s->last_dt = -1.0;      // on the device: cales_last_dt reads it back
  return run_substeps(s);
}

// dt of the last step (HOST output; synchronises when that dt was computed on the device).
extern "C" int cales_last_dt(cales_solver* s, double* dt_host) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !dt_host) return fail(CALES_EINVAL, "null argument");
  if (s->last_dt < 0.0) {
    CUDA_TRY(cudaMemcpyAsync(dt_host, s->dtdev, sizeof(double), cudaMemcpyDeviceToHost, s->st));
    CUDA_TRY(cudaStreamSynchronize(s->st));
  } else *dt_host = s->last_dt;
  return CALES_OK;
}

extern "C" int cales_set_graph(cales_solver* s, int on) {
  DevGuard dg_(s ? s->device : -1);
  if (!s) return fail(CALES_EINVAL, "null solver");
  s->use_graph = on ? 1 : 0;
  if (!on && s->gexec) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }
  return CALES_OK;
}

// Kernel-selection knobs for tests and A/B timing (the defaults are the measured best).
extern "C" int cales_set_option(cales_solver* s, const char* key, long long value) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !key) return fail(CALES_EINVAL, "null argument");
  const std::string k(key);
  if (k == "rhs_tile_min_points") s->rhs_tile_min = value;
  else if (k == "smag_tile_min_points") s->tile_min = value;
  else if (k == "fft_x_lines") {      // lines per CTA of the x transforms (default: ~256 threads per CTA)
    if (value < 1 || value > 64) return fail(CALES_EINVAL, "fft_x_lines must be 1..64");
    const int n2 = s->c.nx / 2; const int L = (int)value;
    bool has3 = false; for (int q = 0; q < s->plx.npass; ++q) has3 |= s->plx.radix[q] == 3;
    const int per_thread = has3 ? 3 * (F2_E / 3) : F2_E;
    long long th = ((long long)L * n2 + per_thread - 1) / per_thread; th = (th + 31) / 32 * 32; if (th < 32) th = 32;
    const size_t sm = (size_t)L * sm_line(n2) * 16;
    if (th > 512 || sm > 200 * 1024) return fail(CALES_EINVAL, "fft_x_lines: CTA too large");
    s->xB = L; s->x_threads = (int)th; s->x_smem = sm;
    s->xBf = L; s->xf_threads = (int)th; s->xf_smem = sm;
  }
  else if (k == "fft_y_cols") {      // columns per CTA tile of the y transforms (power of two; default: ~256 threads per CTA)
    int tish = 0; while ((1LL << tish) < value) ++tish;
    if (value < 1 || (1LL << tish) != value || value > s->c.nx || value > 64) return fail(CALES_EINVAL, "fft_y_cols must be a power of two <= min(nx, 64)");
    const int n2 = s->c.ny / 2;
    bool has3 = false; for (int q = 0; q < s->ply.npass; ++q) has3 |= s->ply.radix[q] == 3;
    const int per_thread = has3 ? 3 * (F2_EY / 3) : F2_EY;
    long long th = ((long long)value * n2 + per_thread - 1) / per_thread; th = (th + 31) / 32 * 32; if (th < 32) th = 32;
    size_t sm = (size_t)value * n2 * 16; if (sm < 16) sm = 16;
    if (th > 512 || sm > 200 * 1024) return fail(CALES_EINVAL, "fft_y_cols: CTA too large");
    s->yTI = (int)value; s->y_tish = tish; s->y_threads = (int)th; s->y_smem = sm;
  }
  else if (k == "dsm_col_rows") { if (value < 0 || value > 4096) return fail(CALES_EINVAL, "dsm_col_rows must be 0..4096"); s->dsm_col_rows = (int)value; s->part_dirty = true; }
  else if (k == "correct_band") { if (value < 0 || value > 1024) return fail(CALES_EINVAL, "correct_band must be 0..1024"); s->corr_band = (int)value; }
  else if (k == "correct_pairs") { if (value < 0 || value > 1) return fail(CALES_EINVAL, "correct_pairs must be 0 or 1"); s->corr2 = (int)value; }
  else if (k == "rhs_prefetch") { if (value < 0 || value > 2) return fail(CALES_EINVAL, "rhs_prefetch must be 0, 1 or 2"); s->rhs_pf = (int)value; }
  else if (k == "rhs_planes_per_cta") { if (value < 0 || value > 65535) return fail(CALES_EINVAL, "rhs_planes_per_cta out of range"); s->rhs_kz = (int)value; }
  else if (k == "fft_stage") { if (value < 0 || value > 2) return fail(CALES_EINVAL, "fft_stage must be 0, 1 or 2"); s->fft_stage = (int)value; }
  else if (k == "poisson_cp_table") { if (value < 0 || value > 2) return fail(CALES_EINVAL, "poisson_cp_table must be 0, 1 or 2"); s->cpt_on = s->CPT ? (int)value : 0; }
  else if (k == "lazy_nut") { if (value < 0 || value > 1) return fail(CALES_EINVAL, "lazy_nut must be 0 or 1"); s->lazy_nut = (int)value; }
  else if (k == "rhs_variant") { if (value < 0 || value > 1) return fail(CALES_EINVAL, "rhs_variant must be 0 or 1"); s->rhs_variant = (int)value; }
  else if (k == "dsm_col_variant") { if (value < 0 || value > 2) return fail(CALES_EINVAL, "dsm_col_variant must be 0, 1 or 2"); s->dsm_col_variant = (int)value; s->part_dirty = true; }
  else return fail(CALES_EINVAL, "unknown option: " + k);
  if (s->gexec) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }      // the captured step holds the old selection
  return CALES_OK;
}

extern "C" int cales_launches_per_step(cales_solver* s) {
  if (!s) return 0;
  const Ctx& c = s->c;
  int per = 1 /*rhs*/ + (c.implicit_z == 1 ? 1 : 0) + (c.implicit_z == 2 ? 15 + (c.const_flow_rate ? 1 : 0) : 0) + (c.const_flow_rate ? 2 : 0) + 5 /*solver*/ + 1 /*correct*/ + (c.wall_model ? 1 : 0) + (c.wall_model_y ? 1 : 0) +
            1 /*static nu_t or fill*/;
  if (c.sgs == CALES_SGS_DSMAG) {
    const bool ywall = c.bc_y == BC_WALL, split = ywall && c.ny >= 3 * DSM_TY;
    const int ncol = (s->dsm_col_variant == 0 && c.nx >= 66 && c.bc_z == BC_WALL) ? 2 : 1;   // staged march + the two wall planes
    int pass1 = (ywall ? 1 : 0) + ((!ywall || split) ? ncol : 0);
    if (c.dsm_filter3d) {
      const D3Split sp = d3_split(c, s->P.zstretch == CALES_Z_UNIFORM);
      pass1 = sp.col ? 1 + (sp.klo > 0 ? 1 : 0) + (sp.jlo > 0 ? 1 : 0) : 1;
    }
    per += -1 + pass1 + (lazy_ok(s) ? 1 : 2);   // pass 1 (tile and/or column kernel), coefficient, nu_t (formed by the momentum kernel when lazy)
  }
  return 3 * per;
}

extern "C" int cales_poisson_solve(cales_solver* s, const double* rhs, double* phi) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !rhs || !phi) return fail(CALES_EINVAL, "null argument");
  int rc;
  if ((rc = run_transform_x_fwd(s, rhs, nullptr, s->W))) return rc;
  if ((rc = run_poisson_core(s))) return rc;
  if ((rc = run_transform_x_inv(s, s->W, phi))) return rc;
  return CALES_OK;
}

extern "C" int cales_eddy_viscosity(cales_solver* s, const double* u, const double* v, const double* w, double* nut) {
  DevGuard dg_(s ? s->device : -1);
  if (!s) return fail(CALES_EINVAL, "null solver");
  const bool own = !u && !v && !w;
  if (!own && (!u || !v || !w)) return fail(CALES_EINVAL, "u, v, w must be all given or all NULL");
  if (!own && !nut) return fail(CALES_EINVAL, "external u, v, w need an external nut: the solver's own nu_t belongs to its own velocity");
  if (nut && nut != s->nut && s->nut_lazy) {      // the evaluation below reuses the |S| / c_s scratch the solver's own lazy nu_t lives in
    int rc = ensure_nut(s);
    if (rc) return rc;
    s->nut_lazy = false;
    if (s->gexec) { cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; }
  }
  return run_eddy_viscosity(s, own ? s->u : u, own ? s->v : v, own ? s->w : w, nut ? nut : s->nut);
}

extern "C" int cales_wall_stress(cales_solver* s, double* tau_dev) {
  DevGuard dg_(s ? s->device : -1);
  if (!s) return fail(CALES_EINVAL, "null solver");
  if (!s->c.wall_model) return fail(CALES_EINVAL, "solver has no wall model");
  int rc = run_wall_stress(s);
  if (rc) return rc;
  if (tau_dev) CUDA_TRY(cudaMemcpyAsync(tau_dev, s->tau, 4 * s->nxy * sizeof(double), cudaMemcpyDeviceToDevice, s->st));
  return CALES_OK;
}

extern "C" int cales_wall_stress_y(cales_solver* s, double* tau_dev) {
  DevGuard dg_(s ? s->device : -1);
  if (!s) return fail(CALES_EINVAL, "null solver");
  if (!s->c.wall_model_y) return fail(CALES_EINVAL, "solver has no wall model on the y walls");
  int rc = run_wall_stress(s);
  if (rc) return rc;
  if (tau_dev) CUDA_TRY(cudaMemcpyAsync(tau_dev, s->tau_y, 4 * (size_t)s->c.nx * s->c.nz * sizeof(double), cudaMemcpyDeviceToDevice, s->st));
  return CALES_OK;
}

extern "C" int cales_project(cales_solver* s) {
  DevGuard dg_(s ? s->device : -1);
  if (!s) return fail(CALES_EINVAL, "null solver");
  int rc;
  DivSrc ds{s->u, s->v, s->w, 1.0, nullptr};
  if ((rc = run_transform_x_fwd(s, nullptr, &ds, s->W))) return rc;
  if ((rc = run_poisson_core(s))) return rc;
  if ((rc = run_transform_x_inv(s, s->W, s->W))) return rc;
  CorrArgs ca;
  ca.phi = s->W; ca.us = s->u; ca.vs = s->v; ca.ws = s->w; ca.u = s->u; ca.v = s->v; ca.w = s->w; ca.p = s->p;
  ca.shift = nullptr; ca.gdt = 1.0; ca.cimp = 0.0; ca.cxy = 0.0; ca.update_p = 0; ca.sc = nullptr;
  k_correct<false><<<s->pgrid, s->pblock, 0, s->st>>>(s->c, ca);
  LAUNCH_TRY(K_CORRECT);
  s->fresh = false;
  return CALES_OK;
}

// adaptive time step (0.95 x the stability limit in the paper; reading S18)
extern "C" int cales_cfl_dt(cales_solver* s, double cfl, double* dt_host) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !dt_host || !(cfl > 0.0)) return fail(CALES_EINVAL, "bad cfl_dt arguments");
  TimingOff toff(s);
  double* part = s->CP;   // scratch, nblk <= N
  k_cfl_rate<<<s->pgrid, s->pblock, 0, s->st>>>(s->c, s->u, s->v, s->w, part);
  LAUNCH_TRY(K_DIAG);
  const long long nb = s->nblk; const int g1 = (int)(nb < 1024 ? nb : 1024);
  k_max_stage<<<g1, 256, 0, s->st>>>(part, nb, s->stage1); LAUNCH_TRY(K_SUM);
  std::vector<double> h(g1);
  CUDA_TRY(cudaMemcpyAsync(h.data(), s->stage1, g1 * sizeof(double), cudaMemcpyDeviceToHost, s->st));
  CUDA_TRY(cudaStreamSynchronize(s->st));
  double r = 0.0; for (int q = 0; q < g1; ++q) r = std::fmax(r, h[q]);
  *dt_host = r > 0.0 ? cfl / r : 0.0;
  return CALES_OK;
}

// ---- allocation-free entry point ---------------------------------------------------------------------------------------------
// cales_cfl_dt_static: the CFL reduction of cales_cfl_dt with its scratch (per-block maxima, first-stage maxima) in a file-scope
// device array instead of the solver's workspace.  The array's name is a host-side stand-in in host code, not a device address:
// static_scratch_ptr() resolves the address once per device (cudaGetSymbolAddress with that device current) and the kernels get
// that pointer.  Every GPU that loads the library holds CALES_STATIC_SCRATCH_BYTES until exit.
enum { STATIC_BLOCKS = CALES_STATIC_SCRATCH_BLOCKS, STATIC_STAGE = 1024, STATIC_MAX_DEVICES = 64 };
static __device__ __align__(256) double g_static_scratch[STATIC_BLOCKS + STATIC_STAGE];
static_assert(sizeof(double) * (STATIC_BLOCKS + STATIC_STAGE) == CALES_STATIC_SCRATCH_BYTES, "header and array disagree");

static int static_scratch_ptr(int device, double** out) {
  static std::mutex mu;
  static double* ptr[STATIC_MAX_DEVICES] = {};
  if (device < 0 || device >= STATIC_MAX_DEVICES) return fail(CALES_EINVAL, "device index beyond the static scratch table");
  std::lock_guard<std::mutex> lk(mu);
  if (!ptr[device]) {      // the caller's DevGuard has made `device` current
    double* d = nullptr;
    CUDA_TRY(cudaGetSymbolAddress((void**)&d, g_static_scratch));
    ptr[device] = d;
  }
  *out = ptr[device];
  return CALES_OK;
}

extern "C" int cales_cfl_dt_static(cales_solver* s, const double* u, const double* v, const double* w, double cfl, double* dt_dev) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !dt_dev || !(cfl > 0.0)) return fail(CALES_EINVAL, "bad cfl_dt_static arguments");
  const bool own = !u && !v && !w;
  if (!own && (!u || !v || !w)) return fail(CALES_EINVAL, "cfl_dt_static: pass all of u, v, w or none");
  if (s->nblk > (long long)STATIC_BLOCKS)
    return fail(CALES_EINVAL, "cfl_dt_static: grid needs " + std::to_string(s->nblk) + " scratch slots (one per 32 x 8 points of a plane), the static array holds " +
                                  std::to_string((long long)STATIC_BLOCKS) + "; use cales_cfl_dt");
  double* part = nullptr;
  { int rc = static_scratch_ptr(s->device, &part); if (rc) return rc; }
  double* stage = part + STATIC_BLOCKS;
  TimingOff toff(s);
  // every slot read below is written first by this call: nothing has to start at zero
  k_cfl_rate<<<s->pgrid, s->pblock, 0, s->st>>>(s->c, own ? s->u : u, own ? s->v : v, own ? s->w : w, part);
  LAUNCH_TRY(K_DIAG);
  const long long nb = s->nblk; const int g1 = (int)(nb < STATIC_STAGE ? nb : STATIC_STAGE);
  k_max_stage<<<g1, 256, 0, s->st>>>(part, nb, stage); LAUNCH_TRY(K_SUM);
  k_dt_finish<<<1, 256, 0, s->st>>>(stage, g1, cfl, dt_dev);
  return check_launch(s, K_SUM);
}

// x-y plane means of u, v, w, uu, vv, ww, uw (centre-averaged) and nu_t: out_dev DEVICE [8][nz] (PAPER.md:237 profiles)
extern "C" int cales_plane_stats(cales_solver* s, double* out_dev) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !out_dev) return fail(CALES_EINVAL, "null argument");
  TimingOff toff(s);
  { int rc = ensure_nut(s); if (rc) return rc; }
  k_plane_stats<<<s->c.nz, 1024, 0, s->st>>>(s->c, s->u, s->v, s->w, s->nut, out_dev);
  return check_launch(s, K_DIAG);
}

// ---- time-accumulated statistics (Tables 3-5) ------------------------------------------
extern "C" int cales_stats_reset(cales_solver* s) {
  DevGuard dg_(s ? s->device : -1);
  if (!s) return fail(CALES_EINVAL, "null solver");
  CUDA_TRY(cudaMemsetAsync(s->stats, 0, (8 * (size_t)s->c.nz + 16) * sizeof(double), s->st));
  return CALES_OK;
}
extern "C" int cales_stats_accumulate(cales_solver* s, double weight) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !(weight > 0.0)) return fail(CALES_EINVAL, "bad stats arguments");
  int rc = CALES_OK;
  TimingOff toff(s);
  do {
    if (!s->fresh && (rc = refresh_closures(s))) break;      // the wall-model planes must belong to the current velocity
    if ((rc = ensure_nut(s))) break;
    const int n = 8 * s->c.nz + 8;
    double* tmp = s->stats + (8 * (size_t)s->c.nz + 16);
    k_plane_stats<<<s->c.nz, 1024, 0, s->st>>>(s->c, s->u, s->v, s->w, s->nut, tmp);
    if ((rc = check_launch(s, K_DIAG))) break;
    k_wall_shear<<<8, 1024, 0, s->st>>>(s->c, s->u, s->v, s->w, tmp + 8 * (size_t)s->c.nz);
    if ((rc = check_launch(s, K_DIAG))) break;
    k_stats_axpy<<<(n + 1 + 255) / 256, 256, 0, s->st>>>(s->stats, tmp, weight, n);
    rc = check_launch(s, K_DIAG);
  } while (0);
  return rc;
}
extern "C" int cales_stats_get(cales_solver* s, double* prof_host, double* wall_host, double* derived_host, double* weight_host) {
  DevGuard dg_(s ? s->device : -1);
  if (!s) return fail(CALES_EINVAL, "null solver");
  const int nz = s->c.nz, n = 8 * nz + 8;
  std::vector<double> h(n + 1), dzf(nz);
  CUDA_TRY(cudaMemcpyAsync(h.data(), s->stats, (n + 1) * sizeof(double), cudaMemcpyDeviceToHost, s->st));
  CUDA_TRY(cudaMemcpyAsync(dzf.data(), s->dzf + 1, nz * sizeof(double), cudaMemcpyDeviceToHost, s->st));
  CUDA_TRY(cudaStreamSynchronize(s->st));
  const double wsum = h[n];
  if (!(wsum > 0.0)) return fail(CALES_EINVAL, "no statistics accumulated");
  for (int q = 0; q < n; ++q) h[q] /= wsum;
  if (prof_host) std::memcpy(prof_host, h.data(), 8 * (size_t)nz * sizeof(double));
  const double* wl = h.data() + 8 * (size_t)nz;
  if (wall_host) std::memcpy(wall_host, wl, 8 * sizeof(double));
  if (derived_host) {
    double tw = 0.0; int nw = 0;
    if (s->c.bc_z == BC_WALL) { tw += wl[0] + wl[2]; nw += 2; }
    if (s->c.bc_y == BC_WALL) { tw += wl[4] + wl[6]; nw += 2; }
    tw = nw ? tw / nw : 0.0;
    double ub = 0.0; for (int k = 0; k < nz; ++k) ub += h[k] * dzf[k];
    ub /= s->c.lz;
    derived_host[0] = tw; derived_host[1] = tw > 0.0 ? std::sqrt(tw) : 0.0; derived_host[2] = derived_host[1] * 0.5 * s->c.lz / s->c.nu;
    derived_host[3] = ub != 0.0 ? 2.0 * tw / (ub * ub) : 0.0;
  }
  if (weight_host) *weight_host = wsum;
  return CALES_OK;
}

// ---- measured fp64 ALU peak (roofline denominator of the ALU-bound kernel) --------------------------------------------------
// 16 independent DFMA chains per thread, 1024 resident threads per SM: nothing but the fp64 pipe limits it.
__global__ void __launch_bounds__(256) k_fp64_peak(double* __restrict__ out, int iters, double a, double b) {
  double x[16];
#pragma unroll
  for (int q = 0; q < 16; ++q) x[q] = 1.0 + 1e-3 * (threadIdx.x + q);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = fma(x[q], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int q = 0; q < 16; ++q) s += x[q];
  if (s == 123.456) out[0] = s;      // never true: keeps the chains alive
}
extern "C" int cales_fp64_peak(cales_solver* s, double* tflops_host) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !tflops_host) return fail(CALES_EINVAL, "null argument");
  TimingOff toff(s);
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, s->device));
  const int blocks = prop.multiProcessorCount * 4, threads = 256, iters = 1 << 16;
  cudaEvent_t e0, e1;
  CUDA_TRY(cudaEventCreate(&e0)); CUDA_TRY(cudaEventCreate(&e1));
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {      // the first is the warm-up
    cudaEventRecord(e0, s->st);
    k_fp64_peak<<<blocks, threads, 0, s->st>>>(s->scal + 31, iters, 0.999999, 1e-6);
    cudaEventRecord(e1, s->st);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
    const double tf = 2.0 * 16.0 * (double)iters * blocks * threads / (ms * 1e-3) / 1e12;
    if (rep > 0 && tf > best) best = tf;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  CUDA_TRY(cudaGetLastError());
  *tflops_host = best;
  return CALES_OK;
}

extern "C" int cales_get_cs(cales_solver* s, double* cs_dev) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !cs_dev) return fail(CALES_EINVAL, "null argument");
  if (s->c.sgs != CALES_SGS_DSMAG) return fail(CALES_EINVAL, "not a dynamic-model solver");
  const size_t n = s->c.dsm_plane ? (size_t)s->c.nz : (size_t)s->c.nz * s->c.ny;
  CUDA_TRY(cudaMemcpyAsync(cs_dev, s->dsm_cs, n * sizeof(double), cudaMemcpyDeviceToDevice, s->st));
  return CALES_OK;
}

extern "C" int cales_transform(cales_solver* s, double* f, int dir, int inverse) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !f) return fail(CALES_EINVAL, "null argument");
  if (dir == 0) return inverse ? run_transform_x_inv(s, f, f) : run_transform_x_fwd(s, f, nullptr, f);
  if (dir == 1) return run_transform_y(s, f, inverse ? 1 : 0);
  return fail(CALES_EINVAL, "dir must be 0 (x) or 1 (y)");
}

extern "C" int cales_transpose_xy(cales_solver* s, const double* src, double* dst) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !src || !dst || src == dst) return fail(CALES_EINVAL, "bad transpose arguments");
  dim3 grid((s->c.nx + 31) / 32, (s->c.ny + 31) / 32, s->c.nz);
  k_transpose_xy<<<grid, dim3(32, 8), 0, s->st>>>(s->c.nx, s->c.ny, src, dst);
  LAUNCH_TRY(K_TRANSPOSE);
  return CALES_OK;
}

// Turn the event list of the last timed step into per-kernel totals (synchronises the stream).
static int collect_times(cales_solver* s) {
  if (!s->ev_valid) return CALES_OK;
  CUDA_TRY(cudaStreamSynchronize(s->st));
  for (int q = 0; q < K_COUNT; ++q) { s->kms[q] = 0.0; s->kcnt[q] = 0; }
  for (int e = 1; e < s->evn; ++e) {
    const int kid = s->evkid[e];
    if (kid < 0) continue;
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, s->evpool[e - 1], s->evpool[e]) == cudaSuccess) { s->kms[kid] += ms; ++s->kcnt[kid]; }
  }
  s->ev_valid = false; s->evn = 0;
  return CALES_OK;
}

extern "C" int cales_kernel_count(void) { return K_COUNT; }

extern "C" int cales_kernel_time(cales_solver* s, int kid, const char** name, double* ms_total, int* launches) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || kid < 0 || kid >= K_COUNT) return fail(CALES_EINVAL, "bad kernel id");
  int rc = collect_times(s);
  if (rc) return rc;
  if (name) *name = k_names[kid];
  if (ms_total) *ms_total = s->kms[kid];
  if (launches) *launches = s->kcnt[kid];
  return CALES_OK;
}

extern "C" int cales_set_timing(cales_solver* s, int on) {
  DevGuard dg_(s ? s->device : -1);
  if (!s) return fail(CALES_EINVAL, "null solver");
  s->timing = on ? 1 : 0; s->ev_valid = false; s->evn = 0;
  return CALES_OK;
}

extern "C" int cales_diagnostics(cales_solver* s, cales_diag* out) {
  DevGuard dg_(s ? s->device : -1);
  if (!s || !out) return fail(CALES_EINVAL, "null argument");
  std::memset(out, 0, sizeof(*out));
  int rc0 = collect_times(s);
  if (rc0) return rc0;
  TimingOff toff(s);   // the diagnostic kernels are not part of a step
  const long long nb = s->nblk;
  double* part = s->CP;   // scratch (4*nblk <= N)
  k_diag<<<s->pgrid, s->pblock, 0, s->st>>>(s->c, s->u, s->v, s->w, s->p, part);
  LAUNCH_TRY(K_DIAG);
  const int g1 = (int)(nb < 1024 ? nb : 1024);
  k_max_stage<<<g1, 256, 0, s->st>>>(part, nb, s->stage1); LAUNCH_TRY(K_SUM);
  for (int q = 1; q < 4; ++q) { k_sum_stage1<<<g1, 256, 0, s->st>>>(part + q * nb, nb, s->stage1 + q * 1024); LAUNCH_TRY(K_SUM); }
  std::vector<double> h(4 * 1024); double scal[4]; int mi = 0;
  CUDA_TRY(cudaMemcpyAsync(h.data(), s->stage1, h.size() * sizeof(double), cudaMemcpyDeviceToHost, s->st));
  CUDA_TRY(cudaMemcpyAsync(scal, s->scal, sizeof(scal), cudaMemcpyDeviceToHost, s->st));
  CUDA_TRY(cudaMemcpyAsync(&mi, s->maxit, sizeof(int), cudaMemcpyDeviceToHost, s->st));
  CUDA_TRY(cudaStreamSynchronize(s->st));
  double md = 0, ub = 0, ke = 0, bad = 0;
  for (int q = 0; q < g1; ++q) { md = std::fmax(md, h[q]); ub += h[1024 + q]; ke += h[2048 + q]; bad += h[3072 + q]; }
  const double vol = (double)s->c.nx * s->c.ny * s->c.lz;
  out->max_div = md; out->u_bulk = ub / vol; out->kinetic_energy = ke / vol; out->nan_count = (int)bad;
  out->forcing = s->c.const_flow_rate ? scal[1] : 0.0; out->wm_max_iters = mi;
  out->ms_rhs = s->kms[K_RHS]; out->ms_implicit = s->kms[K_CN_COEF] + s->kms[K_CN_Z] + s->kms[K_HELM_Z];
  out->ms_solver = s->kms[K_SUM] + s->kms[K_BULK] + s->kms[K_FFTX_FWD] + s->kms[K_FFTY_FWD] + s->kms[K_POISSON_Z] + s->kms[K_FFTY_INV] + s->kms[K_FFTX_INV];
  out->ms_correction = s->kms[K_CORRECT]; out->ms_wall = s->kms[K_WALL];
  out->ms_sgs = s->kms[K_SMAG] + s->kms[K_DSM_PASS1] + s->kms[K_DSM_COL] + s->kms[K_DSM_COEF] + s->kms[K_DSM_NUT] + s->kms[K_FILL] + s->kms[K_DSM3] + s->kms[K_DSM3_COL];
  return CALES_OK;
}
