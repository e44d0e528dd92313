// cales_momentum.cuh -- fused momentum right-hand side + low-storage RK3 update (Eq. 11 / Eq. 20),
// bulk-velocity forcing, correction and pressure update (Eq. 13, 14, 22).
//
// Spatial discretisation: second-order central differences on the staggered grid, divergence
// form of the convective term (Eq. 15 with the sign of Eq. 2, S1), Laplacian form of the molecular term
// (Eq. 16), full symmetric form of the SGS term d_j(2 nu_t S_ij) with the edge viscosity = mean of the 4
// surrounding centres (S6).  One thread per grid point computes the three momentum equations at the
// three faces (i+1/2,j,k), (i,j+1/2,k), (i,j,k+1/2) that belong to cell (i,j,k).
#pragma once
#include "cales_common.cuh"

namespace cales {

struct RhsArgs {
  const double *u, *v, *w, *p, *nut;     // state at substep k
  const double *Ru0, *Rv0, *Rw0;         // R^{k-1} (read when beta != 0)
  double *Ru1, *Rv1, *Rw1;               // R^k (written when the next substep needs it; may alias Ru0..)
  double *us, *vs, *ws;                  // u* (explicit) or the right-hand side of Eq. 21 (implicit z)
  double dt, al, be, ga;
  int store_R;
  const double* sc;                      // substep scalar block in device memory (RK_*), or nullptr: dt above is used
  const double* cs;                      // dynamic model, lazy nu_t: `nut` holds |S| and nu_t = dsm_nut_value(cs, |S|, j, k) is formed when
                                         // the momentum kernel stages it (saves the |S| -> nu_t pass, 16 B/pt per substep); nullptr: nut is nu_t
};

// Substep scalars kept in device memory so that one captured CUDA graph serves every dt (and dt itself may be computed on the
// device, cales_step_adaptive): block rk holds dt, gamma dt, 1 / (gamma dt), gamma nu dt / 2.
enum { RK_DT = 0, RK_GDT = 1, RK_INV_GDT = 2, RK_CIMP = 3, RK_STRIDE = 4 };
CALES_HD void rk_scalars(int rk, double dt, double nu, double* sc) {
  double al, be, ga; rk3_coeffs(rk, al, be, ga);
  sc[RK_DT] = dt; sc[RK_GDT] = ga * dt; sc[RK_INV_GDT] = 1.0 / (ga * dt); sc[RK_CIMP] = 0.5 * ga * nu * dt;
}

struct CorrArgs {
  const double *phi, *us, *vs, *ws;
  double *u, *v, *w, *p;
  const double* shift;     // device scalar: uniform shift of u* that restores the bulk velocity (0 if no forcing)
  double gdt;              // gamma dt
  double cimp;             // gamma nu dt / 2 if implicit z (or fully implicit) else 0
  double cxy;              // gamma nu dt / 2 if fully implicit (Eq. 19: the x and y parts of L_jj phi) else 0
  int update_p;
  const double* sc;        // substep scalar block (RK_*) or nullptr; when given, gdt / cimp / cxy above only say which terms are on
};

// Eq. 13: u = u* - gamma dt grad(phi) (+ the bulk shift of u*); Eq. 14 / 22: p += phi (- c L_zz phi).
template <bool IMP3 = true>
CALES_HD void correct_point(const Ctx& c, const CorrArgs& a, int i, int j, int k) {
  const long long n = idx3(c, i, j, k);
  // the substep scalars first: a load placed after the stores below could not be moved above them (possible aliasing)
  double gdt, sh = 0.0;
  if (a.sc && a.shift) ld_scalar2(a.shift + 4, sh, gdt);      // k_bulk_finish leaves (shift, gamma dt) side by side: one load
  else { gdt = a.sc ? ld_scalar(a.sc + RK_GDT) : a.gdt; if (a.shift) sh = ld_scalar(a.shift); }
  const double cimp = (a.sc && a.cimp != 0.0) ? ld_scalar(a.sc + RK_CIMP) : a.cimp;
  const double ph = a.phi[n];
  double phx, phy, phz, phm = 0.0;
  if (interior_row(c, j, k)) {
    const Nbr o = neighbours(c, i, j, k);
    phx = a.phi[n + o.ip]; phy = a.phi[n + o.jp]; phz = a.phi[n + o.kp];
    if (a.cimp != 0.0) phm = a.phi[n + o.km];
  } else {
    phx = scalg(c, a.phi, i + 1, j, k, 1.0); phy = scalg(c, a.phi, i, j + 1, k, 1.0); phz = scalg(c, a.phi, i, j, k + 1, 1.0);
    if (a.cimp != 0.0) phm = scalg(c, a.phi, i, j, k - 1, 1.0);
  }
  const bool vact = !(c.bc_y == BC_WALL && j == c.ny - 1);
  const bool wact = !(c.bc_z == BC_WALL && k == c.nz - 1);
  const double rdzc = c.rdzc[k];
  a.u[n] = (a.us[n] + sh) - gdt * (phx - ph) * c.rdx;
  a.v[n] = vact ? a.vs[n] - gdt * (phy - ph) * c.rdy : 0.0;
  a.w[n] = wact ? a.ws[n] - gdt * (phz - ph) * rdzc : 0.0;
  if (a.update_p) {
    double dp = ph;
    if (a.cimp != 0.0) dp -= cimp * (((phz - ph) * rdzc - (ph - phm) * c.rdzc[k - 1]) * c.rdzf[k]);
    if (IMP3 && a.cxy != 0.0) {      // Eq. 19 (periodic x and y)
      const double pxm = scalg(c, a.phi, i - 1, j, k, 1.0), pym = scalg(c, a.phi, i, j - 1, k, 1.0);
      dp -= cimp * ((phx - 2.0 * ph + pxm) * c.rdx * c.rdx + (phy - 2.0 * ph + pym) * c.rdy * c.rdy);
    }
    a.p[n] += dp;
  }
}

CALES_HD double divergence_point(const Ctx& c, const double* u, const double* v, const double* w, int i, int j, int k) {
  return (velg<0>(c, u, i, j, k, GH_STRAIN) - velg<0>(c, u, i - 1, j, k, GH_STRAIN)) * c.rdx +
         (velg<1>(c, v, i, j, k, GH_STRAIN) - velg<1>(c, v, i, j - 1, k, GH_STRAIN)) * c.rdy +
         (velg<2>(c, w, i, j, k, GH_STRAIN) - velg<2>(c, w, i, j, k - 1, GH_STRAIN)) * c.rdzf[k];
}

#ifdef __CUDACC__
// IMP3: the Eq. 19 terms of the fully implicit scheme compiled in (the common kernel stays at 32 registers: 64 warps per SM in
// flight, which is what a streaming kernel lives on -- at 40 registers it ran 10.7 -> 14 ms on B200 at config 5)
template <bool IMP3>
__global__ void __launch_bounds__(256, IMP3 ? 4 : 8) k_correct(Ctx c, CorrArgs a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
  if (i < c.nx && j < c.ny) correct_point<IMP3>(c, a, i, j, k);
}
// Two x-neighbours per thread with 16-byte loads and stores (explicit or implicit-z diffusion, nx even, 16-byte aligned fields): half the
// instructions of k_correct for the same bytes.  grid (ceil(nx/64), ceil(ny/8), nz), block (32, 8).  Rows or planes that need a
// ghost go through correct_point.
// band > 1: CTAs in launch order sweep k inside a band of `band` CTA rows (8 rows each) instead of finishing a plane first, so that the
// phi plane k+1 read for the z difference is still in L2 when the CTAs of plane k+1 read it as their own.
__global__ void __launch_bounds__(256, 4) k_correct2(Ctx c, CorrArgs a, int band) {
  unsigned jb = blockIdx.y, kk = blockIdx.z;
  if (band > 1) {
    const unsigned gy = gridDim.y, bw = (unsigned)band, nfull = gy / bw, per = bw * gridDim.z;
    const unsigned L = blockIdx.y + gy * blockIdx.z;
    if (L < nfull * per) { const unsigned b = L / per, r = L - b * per; kk = r / bw; jb = b * bw + (r - kk * bw); }
    else { const unsigned r = L - nfull * per, rw = gy - nfull * bw; kk = r / rw; jb = nfull * bw + (r - kk * rw); }
  }
  const int i = 2 * (blockIdx.x * blockDim.x + threadIdx.x), j = (int)jb * blockDim.y + threadIdx.y, k = (int)kk;
  if (i >= c.nx || j >= c.ny) return;
  if (!interior_row(c, j, k)) { correct_point<false>(c, a, i, j, k); correct_point<false>(c, a, i + 1, j, k); return; }
  const long long n = idx3(c, i, j, k);
  double gdt, sh = 0.0;
  if (a.sc && a.shift) ld_scalar2(a.shift + 4, sh, gdt);
  else { gdt = a.sc ? ld_scalar(a.sc + RK_GDT) : a.gdt; if (a.shift) sh = ld_scalar(a.shift); }
  const Nbr o = neighbours(c, i, j, k);
  auto l2 = [](const double* q) { return *reinterpret_cast<const double2*>(q); };
  const double2 ph = l2(a.phi + n), phy = l2(a.phi + n + o.jp), phz = l2(a.phi + n + o.kp);
  const double phx1 = a.phi[i + 2 < c.nx ? n + 2 : n + 2 - c.nx];
  const double2 us = l2(a.us + n), vs = l2(a.vs + n), ws = l2(a.ws + n);
  double2 p2 = l2(a.p + n);
  const double rdzc = c.rdzc[k];
  double2 u2, v2, w2;
  u2.x = (us.x + sh) - gdt * (ph.y - ph.x) * c.rdx;  u2.y = (us.y + sh) - gdt * (phx1 - ph.y) * c.rdx;
  v2.x = vs.x - gdt * (phy.x - ph.x) * c.rdy;        v2.y = vs.y - gdt * (phy.y - ph.y) * c.rdy;
  w2.x = ws.x - gdt * (phz.x - ph.x) * rdzc;         w2.y = ws.y - gdt * (phz.y - ph.y) * rdzc;
  *reinterpret_cast<double2*>(a.u + n) = u2; *reinterpret_cast<double2*>(a.v + n) = v2; *reinterpret_cast<double2*>(a.w + n) = w2;
  if (a.update_p) {
    double dx = ph.x, dy = ph.y;
    if (a.cimp != 0.0) {      // Eq. 22: - c L_zz phi
      const double cimp = a.sc ? ld_scalar(a.sc + RK_CIMP) : a.cimp;
      const double2 phm = l2(a.phi + n + o.km);
      const double rm = c.rdzc[k - 1], rf = c.rdzf[k];
      dx -= cimp * (((phz.x - ph.x) * rdzc - (ph.x - phm.x) * rm) * rf);
      dy -= cimp * (((phz.y - ph.y) * rdzc - (ph.y - phm.y) * rm) * rf);
    }
    p2.x += dx; p2.y += dy; *reinterpret_cast<double2*>(a.p + n) = p2;
  }
}
// deterministic two-stage sum of `n` partials: stage 1 -> out1[gridDim.x], stage 2 (one block) -> scalar
__global__ void k_sum_stage1(const double* __restrict__ in, long long n, double* __restrict__ out1) {
  __shared__ double sh[32];
  const long long per = (n + gridDim.x - 1) / gridDim.x;
  const long long b0 = per * blockIdx.x, b1 = min(n, b0 + per);
  double s = 0.0;
  for (long long q = b0 + threadIdx.x; q < b1; q += blockDim.x) s += in[q];
  const double t = block_sum(s, sh);
  if (threadIdx.x == 0) out1[blockIdx.x] = t;
}
// scal[0] = shift = u_bulk - sum/(nx ny lz); scal[1] = forcing = shift / (gamma dt); scal[2] = mean; scal[4], scal[5] = (shift, gamma dt)
// side by side for the correction kernel
__global__ void k_rk_scalars(double dt, const double* __restrict__ dt_dev, double nu, double* __restrict__ sc) {
  if (threadIdx.x < 3) rk_scalars(threadIdx.x, dt_dev ? *dt_dev : dt, nu, sc + threadIdx.x * RK_STRIDE);
}
__global__ void k_bulk_finish(Ctx c, const double* __restrict__ in, int n, double gdt, const double* __restrict__ sc, double* __restrict__ scal) {
  __shared__ double sh[32];
  double s = 0.0;
  for (int q = threadIdx.x; q < n; q += blockDim.x) s += in[q];
  const double t = block_sum(s, sh);
  if (threadIdx.x == 0) {
    const double m = t / ((double)c.nx * (double)c.ny * c.lz);
    const double shf = c.u_bulk - m;
    const double g = sc ? sc[RK_GDT] : gdt;
    scal[0] = shf; scal[1] = shf / g; scal[2] = m; scal[4] = shf; scal[5] = g;
  }
}
// diagnostics: per-block partials of max|div|, sum u dzf, sum ke dzf, non-finite count
__global__ void __launch_bounds__(256) k_diag(Ctx c, const double* u, const double* v, const double* w, const double* p, double* __restrict__ part) {
  __shared__ double sh[32];
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
  double d = 0.0, ub = 0.0, ke = 0.0, bad = 0.0;
  if (i < c.nx && j < c.ny) {
    const long long n = idx3(c, i, j, k);
    d = fabs(divergence_point(c, u, v, w, i, j, k));
    if (!(d == d)) d = 0.0;
    ub = u[n] * c.dzf[k];
    const double uc = 0.5 * (velg<0>(c, u, i - 1, j, k, GH_STRAIN) + u[n]);
    const double vc = 0.5 * (velg<1>(c, v, i, j - 1, k, GH_STRAIN) + velg<1>(c, v, i, j, k, GH_STRAIN));
    const double wc = 0.5 * (velg<2>(c, w, i, j, k - 1, GH_STRAIN) + velg<2>(c, w, i, j, k, GH_STRAIN));
    ke = 0.5 * (uc * uc + vc * vc + wc * wc) * c.dzf[k];
    bad = (isfinite(u[n]) ? 0.0 : 1.0) + (isfinite(v[n]) ? 0.0 : 1.0) + (isfinite(w[n]) ? 0.0 : 1.0) + (isfinite(p[n]) ? 0.0 : 1.0);
  }
  const long long nb = (long long)gridDim.x * gridDim.y * gridDim.z;
  const long long b = blockIdx.x + gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z);
  const double md = block_max(d, sh);
  const double s1 = block_sum(ub, sh), s2 = block_sum(ke, sh), s3 = block_sum(bad, sh);
  if (threadIdx.x == 0 && threadIdx.y == 0) { part[b] = md; part[nb + b] = s1; part[2 * nb + b] = s2; part[3 * nb + b] = s3; }
}
// SURVEY.md 8(f) item 4.  CFL rate |u_c|/dx + |v_c|/dy + |w_c|/dzf at a cell centre (S18)
CALES_HD double cfl_rate_point(const Ctx& c, const double* u, const double* v, const double* w, int i, int j, int k) {
  const double uc = 0.5 * (velg<0>(c, u, i - 1, j, k, GH_STRAIN) + velg<0>(c, u, i, j, k, GH_STRAIN));
  const double vc = 0.5 * (velg<1>(c, v, i, j - 1, k, GH_STRAIN) + velg<1>(c, v, i, j, k, GH_STRAIN));
  const double wc = 0.5 * (velg<2>(c, w, i, j, k - 1, GH_STRAIN) + velg<2>(c, w, i, j, k, GH_STRAIN));
  return fabs(uc) * c.rdx + fabs(vc) * c.rdy + fabs(wc) * c.rdzf[k];
}
// the 8 plane-statistics quantities at a cell centre: u, v, w, uu, vv, ww, uw (centre-averaged velocity), nu_t
CALES_HD void stats_point(const Ctx& c, const double* u, const double* v, const double* w, const double* nut, int i, int j, int k, double* q) {
  const double uc = 0.5 * (velg<0>(c, u, i - 1, j, k, GH_STRAIN) + velg<0>(c, u, i, j, k, GH_STRAIN));
  const double vc = 0.5 * (velg<1>(c, v, i, j - 1, k, GH_STRAIN) + velg<1>(c, v, i, j, k, GH_STRAIN));
  const double wc = 0.5 * (velg<2>(c, w, i, j, k - 1, GH_STRAIN) + velg<2>(c, w, i, j, k, GH_STRAIN));
  q[0] = uc; q[1] = vc; q[2] = wc; q[3] = uc * uc; q[4] = vc * vc; q[5] = wc * wc; q[6] = uc * wc; q[7] = nut[idx3(c, i, j, k)];
}
// per-block max of the CFL rate -> part[block] (grid as the point kernels)
__global__ void __launch_bounds__(256) k_cfl_rate(Ctx c, const double* u, const double* v, const double* w, double* __restrict__ part) {
  __shared__ double sh[32];
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
  double r = 0.0;
  if (i < c.nx && j < c.ny) r = cfl_rate_point(c, u, v, w, i, j, k);
  const double m = block_max(r, sh);
  if (threadIdx.x == 0 && threadIdx.y == 0) part[blockIdx.x + gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z)] = m;
}
// x-y plane means: grid (nz), block 1024; out[q * nz + k] (deterministic: fixed thread -> point assignment and tree order)
__global__ void __launch_bounds__(1024) k_plane_stats(Ctx c, const double* u, const double* v, const double* w, const double* nut, double* __restrict__ out) {
  __shared__ double sh[32];
  const int k = blockIdx.x;
  double a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (long long n = threadIdx.x; n < c.nxy; n += blockDim.x) {
    double q[8];
    stats_point(c, u, v, w, nut, (int)(n % c.nx), (int)(n / c.nx), k, q);
#pragma unroll
    for (int m = 0; m < 8; ++m) a[m] += q[m];
  }
  for (int m = 0; m < 8; ++m) {
    const double t = block_sum(a[m], sh);
    if (threadIdx.x == 0) out[(long long)m * c.nz + k] = t / (double)c.nxy;
  }
}
// Wall-shear means (C_f and Re_tau of Tables 3-5): grid 8, block 1024; out[q], q = 0..3 the z walls ((tau_xz, tau_yz) bottom,
// top), 4..7 the y walls ((tau_xy, tau_zy) low, high; dzf-weighted); 0 in periodic directions.  Modelled walls: mean of the wall-model
// planes; no-slip walls: nu x the one-sided difference to the mirror ghost, 2 nu q_first / (ghost spacing).
__global__ void __launch_bounds__(1024) k_wall_shear(Ctx c, const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w,
                                                     double* __restrict__ out) {
  __shared__ double sh[32];
  const int q = blockIdx.x, wl = (q >> 1) & 1, comp = q & 1;
  double a = 0.0, norm = 1.0;
  if (q < 4) {
    if (c.bc_z == BC_WALL) {
      const double* f = comp == 0 ? u : v;
      const int k0 = wl == 0 ? 0 : c.nz - 1;
      const double fac = 2.0 * c.nu / (wl == 0 ? c.dzc[-1] : c.dzc[c.nz - 1]);
      for (long long n = threadIdx.x; n < c.nxy; n += blockDim.x)
        a += c.wall_model ? c.tau[(long long)(wl * 2 + comp) * c.nxy + n] : fac * f[(long long)k0 * c.nxy + n];
      norm = (double)c.nxy;
    }
  } else if (c.bc_y == BC_WALL) {
    const double* f = comp == 0 ? u : w;
    const int j0 = wl == 0 ? 0 : c.ny - 1;
    const double fac = 2.0 * c.nu * c.rdy;
    const long long nxz = (long long)c.nx * c.nz;
    for (long long n = threadIdx.x; n < nxz; n += blockDim.x) {
      const int k = (int)(n / c.nx), i = (int)(n - (long long)k * c.nx);
      a += (c.wall_model_y ? c.tau_y[(long long)(wl * 2 + comp) * nxz + n] : fac * f[idx3(c, i, j0, k)]) * c.dzf[k];
    }
    norm = (double)c.nx * c.lz;
  }
  const double t = block_sum(a, sh);
  if (threadIdx.x == 0) out[q] = t / norm;
}
// acc[0..n) += weight * tmp[0..n); acc[n] += weight (the accumulated weight)
__global__ void k_stats_axpy(double* __restrict__ acc, const double* __restrict__ tmp, double weight, int n) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q < n) acc[q] += weight * tmp[q];
  if (q == n) acc[q] += weight;
}
__global__ void k_max_stage(const double* __restrict__ in, long long n, double* __restrict__ out) {
  __shared__ double sh[32];
  const long long per = (n + gridDim.x - 1) / gridDim.x;
  const long long b0 = per * blockIdx.x, b1 = min(n, b0 + per);
  double s = 0.0;
  for (long long q = b0 + threadIdx.x; q < b1; q += blockDim.x) s = fmax(s, in[q]);
  const double t = block_max(s, sh);
  if (threadIdx.x == 0) out[blockIdx.x] = t;
}
// dt = cfl / max rate (0 if the field is at rest), one block
__global__ void k_dt_finish(const double* __restrict__ in, int n, double cfl, double* __restrict__ dt_dev) {
  __shared__ double sh[32];
  double s = 0.0;
  for (int q = threadIdx.x; q < n; q += blockDim.x) s = fmax(s, in[q]);
  const double t = block_max(s, sh);
  if (threadIdx.x == 0) *dt_dev = t > 0.0 ? cfl / t : 0.0;
}
#endif

}  // namespace cales
