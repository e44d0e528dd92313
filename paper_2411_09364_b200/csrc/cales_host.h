// cales_host.h -- host-side setup shared by the CUDA library and the host kernel emulator of tests/emu:
// parameter validation, grid metrics, eigenvalues, twiddle tables, wall-model sampling geometry, transform plans
// and launch shapes.  Plain C++ (no CUDA runtime calls); no arithmetic of the time step itself lives here.
#pragma once
#include "../../include/cales.h"
#include "cales_common.cuh"
#include "cales_fft.cuh"
#include "cales_fft2.cuh"
#include "cales_closures.cuh"

#include <cmath>
#include <cstdlib>
#include <string>
#include <vector>

namespace cales {

static thread_local std::string g_err;
static inline int fail(int code, const std::string& m) { g_err = m; return code; }

static inline bool smooth23(int n) { if (n < 1) return false; while (n % 2 == 0) n /= 2; while (n % 3 == 0) n /= 3; return n == 1; }

static inline int validate(const cales_params* p) {
  if (!p) return fail(CALES_EINVAL, "null parameters");
  if (p->nx < 2 || p->ny < 2 || p->nz < 4) return fail(CALES_EINVAL, "grid too small (nx, ny >= 2, nz >= 4)");
  if (!(p->lx > 0.0) || !(p->ly > 0.0) || !(p->lz > 0.0)) return fail(CALES_EINVAL, "box lengths must be positive");
  if (!(p->nu > 0.0)) return fail(CALES_EINVAL, "nu must be positive");
  if (p->nx % 2 || p->ny % 2) return fail(CALES_EUNSUPPORTED, "nx and ny must be even");
  if (!smooth23(p->nx) || !smooth23(p->ny)) return fail(CALES_EUNSUPPORTED, "nx, ny must factor into 2 and 3");
  if (p->nx > 12288 || p->ny > 8192) return fail(CALES_EUNSUPPORTED, "nx <= 12288 and ny <= 8192 (line must fit shared memory)");
  if (p->nz > 65535) return fail(CALES_EUNSUPPORTED, "nz <= 65535");
  if (p->bc_y != CALES_BC_PERIODIC && p->bc_y != CALES_BC_WALL) return fail(CALES_EINVAL, "bad bc_y");
  if (p->bc_z != CALES_BC_PERIODIC && p->bc_z != CALES_BC_WALL) return fail(CALES_EINVAL, "bad bc_z");
  if (p->zstretch < 0 || p->zstretch > 2) return fail(CALES_EINVAL, "bad zstretch");
  if (p->zstretch == CALES_Z_USER && !p->zf_user) return fail(CALES_EINVAL, "zf_user is null");
  if (p->bc_z == CALES_BC_PERIODIC && p->zstretch != CALES_Z_UNIFORM) return fail(CALES_EUNSUPPORTED, "periodic z requires a uniform grid");
  if (p->sgs_model < 0 || p->sgs_model > 2) return fail(CALES_EINVAL, "bad sgs_model");
  if (p->wall_model && p->bc_z != CALES_BC_WALL) return fail(CALES_EUNSUPPORTED, "wall model needs z walls");
  if (p->wall_model_y && p->bc_y != CALES_BC_WALL) return fail(CALES_EUNSUPPORTED, "wall model on y walls needs y walls");
  if (p->dsm_filter3d && p->sgs_model != CALES_SGS_DSMAG) return fail(CALES_EINVAL, "dsm_filter3d needs the dynamic model");
  if (p->implicit_z && p->bc_z != CALES_BC_WALL) return fail(CALES_EUNSUPPORTED, "implicit z needs z walls");
  if (p->implicit_xyz && p->bc_y != CALES_BC_PERIODIC) return fail(CALES_EUNSUPPORTED, "fully implicit diffusion needs periodic y (PAPER.md:136)");
  if (p->implicit_xyz && p->implicit_z) return fail(CALES_EINVAL, "implicit_z and implicit_xyz exclude each other");
  if (p->wall_model && p->h_wm > 0.0 && !(p->h_wm < 0.5 * p->lz)) return fail(CALES_EINVAL, "h_wm must lie below the half height");
  if (p->wall_model_y && p->h_wm > 0.0 && !(p->h_wm < 0.5 * p->ly)) return fail(CALES_EINVAL, "h_wm must lie below the half width");
  if (p->van_driest && (p->bc_z != CALES_BC_WALL || p->bc_y == CALES_BC_WALL || p->wall_model))
    return fail(CALES_EUNSUPPORTED, "van Driest damping: z walls only, no wall model");
  return CALES_OK;
}

// Radix plan of the complex FFT of length n/2: the power of two 2^a split into ceil(a/4) passes of radix 2..16 of
// (nearly) equal size, smallest first (the first passes write with stride R), then the factors of 3.
static inline void make_plan(FftPlan& pl, int n, int E = F2_E) {
  pl.n = n; pl.n2 = n / 2; pl.npass = 0; pl.tw = nullptr; pl.dctw = nullptr;
  int m = pl.n2, n3 = 0;
  while (m % 3 == 0) { ++n3; m /= 3; }
  int a = 0; while (m % 2 == 0) { ++a; m /= 2; }
  if (a > 0) {
    int maxbits = E >= 16 ? 4 : 3;
    const int np = (a + maxbits - 1) / maxbits, base = a / np, extra = a % np;
    for (int q = 0; q < np; ++q) pl.radix[pl.npass++] = 1 << (base + (q >= np - extra ? 1 : 0));
  }
  for (int q = 0; q < n3; ++q) pl.radix[pl.npass++] = 3;
  int Ns = 1;
  for (int p = 0; p < pl.npass; ++p) {
    pl.per[p] = pl.n2 / pl.radix[p]; pl.ns[p] = Ns;
    pl.mper[p] = pl.per[p] > 1 ? (unsigned)((0x100000000ull + pl.per[p] - 1) / pl.per[p]) : 0u;
    pl.mns[p] = Ns > 1 ? (unsigned)((0x100000000ull + Ns - 1) / Ns) : 0u;
    Ns *= pl.radix[p];
  }
}

// Launch shape of the dynamic-model pass 1: block width TXB of the column march,
// its number of x blocks, and the number of partial-sum slots per (k, j) row shared with the tile kernel.
struct DsmShape { int txb, nbx, pslots; };
static inline DsmShape dsm_shape(int nx) {
  DsmShape d{64, 0, 0};   // 64-thread CTAs (62 output columns + 2 halo columns): measured best of 32 / 64 / 96 / 128 on B200
  d.nbx = (nx + d.txb - 3) / (d.txb - 2);
  d.pslots = (nx + DSM_TX - 1) / DSM_TX;
  { const int cs = d.nbx * (d.txb / 32); if (cs > d.pslots) d.pslots = cs; }      // one partial-sum slot per warp of the column march
  return d;
}

struct HostSetup {
  cales_params P;                 // with the defaults filled in
  std::vector<double> dzf, dzc, rdzf, rdzc, delta, zc, ak, ck, lamx, lamy, twx, twy, dctw;   // dzf: index k+1 holds dzf[k], k=-1..nz; dzc: k+1 holds dzc[k], k=-1..nz-1
  Ctx c;                          // table pointers NOT set
  WallGeom wg;
  FftPlan plx, ply;               // twiddle pointers NOT set
  int xB, yTI, y_tish, x_threads, y_threads; size_t x_smem, y_smem;
};

static inline int build_setup(const cales_params* p, HostSetup& H) {
  const double PI_ = 3.14159265358979323846264338327950288;
  int rc = validate(p);
  if (rc) return rc;
  H.P = *p; H.P.zf_user = nullptr;
  if (H.P.wm_tol <= 0.0) H.P.wm_tol = 1e-4;
  if (H.P.wm_maxit <= 0) H.P.wm_maxit = 50;
  if (H.P.kappa <= 0.0) H.P.kappa = 0.41;
  if (H.P.aplus <= 0.0) H.P.aplus = 25.0;
  const int nx = p->nx, ny = p->ny, nz = p->nz;
  // ---- grid (S16 for the tanh map)
  std::vector<double> zf(nz + 1);
  H.zc.assign(nz, 0.0); H.dzf.assign(nz + 2, 0.0); H.dzc.assign(nz + 2, 0.0);
  for (int k = 0; k <= nz; ++k) {
    if (p->zstretch == CALES_Z_UNIFORM) zf[k] = p->lz * (double)k / (double)nz;
    else if (p->zstretch == CALES_Z_TANH) { const double a = p->zstretch_factor; zf[k] = 0.5 * p->lz * (1.0 + std::tanh(a * (2.0 * k / (double)nz - 1.0)) / std::tanh(a)); }
    else zf[k] = p->zf_user[k];
  }
  zf[0] = 0.0; zf[nz] = p->lz;
  for (int k = 0; k < nz; ++k) {
    H.zc[k] = 0.5 * (zf[k] + zf[k + 1]); H.dzf[k + 1] = zf[k + 1] - zf[k];
    if (!(H.dzf[k + 1] > 0.0)) return fail(CALES_EINVAL, "z faces must increase");
  }
  const bool zper = p->bc_z == CALES_BC_PERIODIC;
  if (zper) { H.dzf[0] = H.dzf[nz]; H.dzf[nz + 1] = H.dzf[1]; } else { H.dzf[0] = H.dzf[1]; H.dzf[nz + 1] = H.dzf[nz]; }
  for (int k = 0; k < nz - 1; ++k) H.dzc[k + 1] = H.zc[k + 1] - H.zc[k];
  if (zper) { H.dzc[0] = H.dzf[1]; H.dzc[nz] = H.dzf[1]; } else { H.dzc[0] = 2.0 * H.zc[0]; H.dzc[nz] = 2.0 * (p->lz - H.zc[nz - 1]); }   // mirrored ghost centre
  H.rdzf.assign(nz + 2, 0.0); H.rdzc.assign(nz + 2, 0.0);
  for (int k = 0; k < nz + 2; ++k) { H.rdzf[k] = 1.0 / H.dzf[k]; if (k <= nz) H.rdzc[k] = 1.0 / H.dzc[k]; }
  H.ak.resize(nz); H.ck.resize(nz);
  for (int k = 0; k < nz; ++k) { H.ak[k] = 1.0 / (H.dzf[k + 1] * H.dzc[k]); H.ck[k] = 1.0 / (H.dzf[k + 1] * H.dzc[k + 1]); }
  // ---- eigenvalues of the 3-point operators in the packed layouts (ref. [28])
  const double dx = p->lx / nx, dy = p->ly / ny;
  H.lamx.resize(nx); H.lamy.resize(ny);
  for (int i = 0; i < nx; ++i) {
    const int m = i == 0 ? 0 : (i == 1 ? nx / 2 : i / 2);
    const double sn = std::sin(PI_ * m / (double)nx); H.lamx[i] = -4.0 / (dx * dx) * sn * sn;
  }
  for (int j = 0; j < ny; ++j) {
    double sn;
    if (p->bc_y == CALES_BC_PERIODIC) { const int m = j == 0 ? 0 : (j == 1 ? ny / 2 : j / 2); sn = std::sin(PI_ * m / (double)ny); }
    else sn = std::sin(PI_ * j / (2.0 * ny));
    H.lamy[j] = -4.0 / (dy * dy) * sn * sn;
  }
  H.delta.resize(nz);
  for (int k = 0; k < nz; ++k) H.delta[k] = std::cbrt(dx * dy * H.dzf[k + 1]);
  // ---- twiddles in extended precision, rounded once to fp64
  H.twx.resize(2 * (size_t)nx); H.twy.resize(2 * (size_t)ny); H.dctw.resize(2 * ((size_t)ny / 2 + 1));
  const long double PIL = 3.14159265358979323846264338327950288L;
  for (int q = 0; q < nx; ++q) { const long double a = 2.0L * PIL * q / nx; H.twx[2 * q] = (double)cosl(a); H.twx[2 * q + 1] = (double)(-sinl(a)); }
  for (int q = 0; q < ny; ++q) { const long double a = 2.0L * PIL * q / ny; H.twy[2 * q] = (double)cosl(a); H.twy[2 * q + 1] = (double)(-sinl(a)); }
  for (int m = 0; m <= ny / 2; ++m) { const long double a = PIL * m / (2.0L * ny); H.dctw[2 * m] = (double)cosl(a); H.dctw[2 * m + 1] = (double)(-sinl(a)); }
  // ---- device context (pointers are set by the owner of the tables)
  Ctx& c = H.c;
  c.nx = nx; c.ny = ny; c.nz = nz; c.N = (long long)nx * ny * nz; c.nxy = (long long)nx * ny;
  c.bc_y = p->bc_y; c.bc_z = p->bc_z; c.wall_model = p->wall_model; c.wall_model_y = p->wall_model_y; c.dsm_filter3d = p->dsm_filter3d; c.sgs = p->sgs_model; c.van_driest = p->van_driest;
  c.implicit_z = p->implicit_xyz ? 2 : (p->implicit_z ? 1 : 0); c.dsm_plane = p->dsm_avg_xy_plane; c.dsm_clip_total = p->dsm_clip_total; c.const_flow_rate = p->const_flow_rate;
  c.wm_maxit = H.P.wm_maxit; c.dx = dx; c.dy = dy; c.rdx = 1.0 / dx; c.rdy = 1.0 / dy; c.lz = p->lz; c.nu = p->nu; c.cs = p->cs; c.aplus = H.P.aplus; c.rnuap = 1.0 / (p->nu * H.P.aplus);
  c.alpha = p->dsm_alpha2d > 0.0 ? p->dsm_alpha2d : std::cbrt(4.0);
  c.kappa = H.P.kappa; c.Blog = p->B; c.h_wm = p->h_wm; c.wm_tol = H.P.wm_tol; c.u_bulk = p->u_bulk;
  c.dzf = nullptr; c.dzc = nullptr; c.zc = nullptr; c.rdzf = nullptr; c.rdzc = nullptr; c.delta = nullptr; c.tau = nullptr; c.tau_y = nullptr;
  // ---- wall-model sampling geometry (linear interpolation between locations 1 and 2)
  for (int wall = 0; wall < 2; ++wall) {
    auto dist = [&](int q) { return wall == 0 ? H.zc[q] : p->lz - H.zc[nz - 1 - q]; };
    const double h = p->h_wm > 0.0 ? p->h_wm : dist(0);
    int q1 = 0; while (q1 + 2 < nz / 2 && dist(q1 + 1) <= h) ++q1;
    H.wg.wgt[wall] = (h - dist(q1)) / (dist(q1 + 1) - dist(q1));
    H.wg.ka[wall] = wall == 0 ? q1 : nz - 1 - q1; H.wg.kb[wall] = wall == 0 ? q1 + 1 : nz - 2 - q1; H.wg.h[wall] = h;
  }
  {   // the same for the y walls (uniform spacing): centre number q lies (q + 1/2) dy from its wall
    auto dist = [&](int q) { return (q + 0.5) * dy; };
    const double h = p->h_wm > 0.0 ? p->h_wm : dist(0);
    int q1 = 0; while (q1 + 2 < ny / 2 && dist(q1 + 1) <= h) ++q1;
    c.wy_q1 = q1; c.wy_wgt = (h - dist(q1)) / (dist(q1 + 1) - dist(q1)); c.wy_h = h;
  }
  // ---- transform plans and launch shapes
  make_plan(H.plx, nx);
  make_plan(H.ply, ny, F2_EY);
  // every thread holds 16 complex elements per pass (15 when a radix-3 pass exists): ~256 threads per CTA
  auto threads_for = [](long long elems, const FftPlan& pl, int E = F2_E) {
    bool has3 = false; for (int p = 0; p < pl.npass; ++p) has3 |= pl.radix[p] == 3;
    const int per_thread = has3 ? 3 * (E / 3) : E;
    long long th = (elems + per_thread - 1) / per_thread;
    th = (th + 31) / 32 * 32;
    return (int)(th < 32 ? 32 : th);
  };
  {
    const int n2 = nx / 2;
    int L = 256 * F2_E / n2; if (L < 1) L = 1; if (L > 64) L = 64;
    const long long nlines = (long long)ny * nz; if (L > nlines) L = (int)nlines;
    while (L > 1 && threads_for((long long)L * n2, H.plx) > 256) --L;
    while (L > 1 && (nlines + L - 1) / L < 2 * 148) --L;            // small grids: at least two CTAs per SM if there is work for them
    H.xB = L; H.x_smem = (size_t)L * sm_line(n2) * 16;
    H.x_threads = threads_for((long long)L * n2, H.plx);
  }
  {
    const int n2 = ny / 2;
    int tish = 4;                                                   // TI = 16 columns (B200: config 4 0.322 / 0.337 ms against 0.345 / 0.343 with 32) ...
    while (tish > 3 && (long long)(1 << tish) * n2 > 512 * F2_EY) --tish;   // ... down to 8 (64-byte row segments) for long lines
    while (tish > 0 && (1 << tish) > nx) --tish;
    while (tish > 3 && (long long)((nx + (1 << tish) - 1) >> tish) * nz < 2 * 148) --tish;
    while (tish > 0 && (threads_for((long long)(1 << tish) * n2, H.ply, F2_EY) > 512 || (size_t)(1 << tish) * n2 * 16 > 200 * 1024)) --tish;
    H.yTI = 1 << tish; H.y_tish = tish; H.y_smem = (size_t)(1 << tish) * n2 * 16; if (H.y_smem < 16) H.y_smem = 16;
    H.y_threads = threads_for((long long)(1 << tish) * n2, H.ply, F2_EY);
  }
  if (H.x_threads > 512 || H.y_threads > 512 || H.x_smem > 200 * 1024 || H.y_smem > 200 * 1024)
    return fail(CALES_EUNSUPPORTED, "line too long for the shared-memory transforms");
  return CALES_OK;
}

}  // namespace cales
