// cales_closures.cuh -- log-law wall model (Eq. 10; Fig. 1) and eddy viscosity:
// static Smagorinsky with van Driest damping (Eq. 4) and dynamic Smagorinsky with the x-y box
// test filter and Lilly's least squares averaged over the homogeneous directions (Eq. 5-9).
#pragma once
#include "cales_common.cuh"

namespace cales {

// ------------------------------------------------------------------------------------------------------------
// Wall model.  Newton-Raphson on s = ln(h+), h+ = u_tau h / nu (S8):  g(s) = Re e^{-s} - s/kappa - B,
// Re = U h / nu, s_0 = ln(Re)/2.  Stop when the relative change of tau_w, |e^{2 ds} - 1|, is below tol
// (0.01 %), then ONE more update (S9), which makes the result independent of where the
// stopping test fell.
// ------------------------------------------------------------------------------------------------------------
CALES_HD double loglaw_hplus(double re, double kappa, double B, double tol, int maxit, int* iters) {
  *iters = 0;
  if (!(re > 0.0)) return 0.0;
  double s = 0.5 * log(re);
  int it = 0; bool polish = false;
  while (it < maxit) {
    const double e = re * exp(-s);
    const double g = e - s / kappa - B;
    const double dg = -e - 1.0 / kappa;
    const double sn = s - g / dg;
    ++it;
    const double rel = fabs(exp(2.0 * (sn - s)) - 1.0);
    s = sn;
    if (polish) break;
    if (rel < tol) polish = true;
  }
  *iters = it;
  return exp(s);
}

struct WallGeom { int ka[2], kb[2]; double wgt[2], h[2]; };   // sampling planes, interpolation weight, h_wm per wall

// tau[wall][comp][j][i]; comp 0: tau_xz at the u point (i+1/2, j), comp 1: tau_yz at the v point (i, j+1/2).
CALES_HD int wall_stress_point(const Ctx& c, const WallGeom& g, const double* u, const double* v, int wall, int comp, int i, int j, double* tau) {
  const int ka = g.ka[wall], kb = g.kb[wall];
  const double wg = g.wgt[wall], h = g.h[wall];
#define ATU(ii, jj) ((1.0 - wg) * velg<0>(c, u, ii, jj, ka, GH_STRAIN) + wg * velg<0>(c, u, ii, jj, kb, GH_STRAIN))
#define ATV(ii, jj) ((1.0 - wg) * velg<1>(c, v, ii, jj, ka, GH_STRAIN) + wg * velg<1>(c, v, ii, jj, kb, GH_STRAIN))
  double a, b;
  if (comp == 0) { a = ATU(i, j); b = 0.25 * (ATV(i, j) + ATV(i + 1, j) + ATV(i, j - 1) + ATV(i + 1, j - 1)); }
  else { a = ATV(i, j); b = 0.25 * (ATU(i, j) + ATU(i - 1, j) + ATU(i, j + 1) + ATU(i - 1, j + 1)); }
#undef ATU
#undef ATV
  const double U = sqrt(a * a + b * b);
  double t = 0.0; int it = 0;
  if (U > 0.0) {
    const double hp = loglaw_hplus(U * h / c.nu, c.kappa, c.Blog, c.wm_tol, c.wm_maxit, &it);
    const double utau = hp * c.nu / h;
    t = utau * utau * a / U;
  }
  tau[((long long)(wall * 2 + comp) * c.ny + j) * c.nx + i] = t;
  return it;
}

// y walls (duct WMLES): sampled at the first off-wall centre, h = dy/2.  comp 0: tau_xy at the u point
// (i+1/2, k) from u and the 4 surrounding w points; comp 1: tau_zy at the w point (i, k+1/2) from w and the 4 surrounding u.
// tau_y[wall][comp][k][i].
CALES_HD int wall_stress_y_point(const Ctx& c, const double* u, const double* w, int wall, int comp, int i, int k, double* tau_y) {
  const int ja = wall == 0 ? c.wy_q1 : c.ny - 1 - c.wy_q1, jb = wall == 0 ? c.wy_q1 + 1 : c.ny - 2 - c.wy_q1;
  const double wg = c.wy_wgt, h = c.wy_h;
  // linear interpolation in y between the two bracketing centres; wg = 0 at the default h = dy/2
  auto atu = [&](int ii, int kk) { return (1.0 - wg) * velg<0>(c, u, ii, ja, kk, GH_STRAIN) + wg * velg<0>(c, u, ii, jb, kk, GH_STRAIN); };
  auto atw = [&](int ii, int kk) { return (1.0 - wg) * velg<2>(c, w, ii, ja, kk, GH_STRAIN) + wg * velg<2>(c, w, ii, jb, kk, GH_STRAIN); };
  double a, b;
  if (comp == 0) { a = atu(i, k); b = 0.25 * (atw(i, k) + atw(i + 1, k) + atw(i, k - 1) + atw(i + 1, k - 1)); }
  else { a = atw(i, k); b = 0.25 * (atu(i, k) + atu(i - 1, k) + atu(i, k + 1) + atu(i - 1, k + 1)); }
  const double U = sqrt(a * a + b * b);
  double t = 0.0; int it = 0;
  if (U > 0.0) {
    const double hp = loglaw_hplus(U * h / c.nu, c.kappa, c.Blog, c.wm_tol, c.wm_maxit, &it);
    const double utau = hp * c.nu / h;
    t = utau * utau * a / U;
  }
  tau_y[((long long)(wall * 2 + comp) * c.nz + k) * c.nx + i] = t;
  return it;
}

// ------------------------------------------------------------------------------------------------------------
// Strain rate at a cell centre: diagonals directly; off-diagonals at the 4 surrounding edge
// midpoints, then averaged.  U(di,dj,dk), V, W return the face values at offsets from the cell.
// S order: 11 22 33 12 13 23.  Returns |S| = sqrt(2 S_ij S_ij).
// ------------------------------------------------------------------------------------------------------------
template <class GU, class GV, class GW>
CALES_HD double strain_at(GU U, GV V, GW W, double rdx, double rdy, double rdzf, double rdzc, double rdzcm, double* S) {
  const double u000 = U(0, 0, 0), um00 = U(-1, 0, 0), v000 = V(0, 0, 0), v0m0 = V(0, -1, 0), w000 = W(0, 0, 0), w00m = W(0, 0, -1);
  S[0] = (u000 - um00) * rdx;
  S[1] = (v000 - v0m0) * rdy;
  S[2] = (w000 - w00m) * rdzf;
  const double u0p0 = U(0, 1, 0), u0m0 = U(0, -1, 0), ump0 = U(-1, 1, 0), umm0 = U(-1, -1, 0);
  const double vp00 = V(1, 0, 0), vm00 = V(-1, 0, 0), vpm0 = V(1, -1, 0), vmm0 = V(-1, -1, 0);
  const double s12_00 = 0.5 * ((u0p0 - u000) * rdy + (vp00 - v000) * rdx);
  const double s12_m0 = 0.5 * ((ump0 - um00) * rdy + (v000 - vm00) * rdx);
  const double s12_0m = 0.5 * ((u000 - u0m0) * rdy + (vpm0 - v0m0) * rdx);
  const double s12_mm = 0.5 * ((um00 - umm0) * rdy + (v0m0 - vmm0) * rdx);
  S[3] = 0.25 * (s12_00 + s12_m0 + s12_0m + s12_mm);
  const double u00p = U(0, 0, 1), u00m = U(0, 0, -1), um0p = U(-1, 0, 1), um0m = U(-1, 0, -1);
  const double wp00 = W(1, 0, 0), wm00 = W(-1, 0, 0), wp0m = W(1, 0, -1), wm0m = W(-1, 0, -1);
  const double s13_00 = 0.5 * ((u00p - u000) * rdzc + (wp00 - w000) * rdx);
  const double s13_m0 = 0.5 * ((um0p - um00) * rdzc + (w000 - wm00) * rdx);
  const double s13_0m = 0.5 * ((u000 - u00m) * rdzcm + (wp0m - w00m) * rdx);
  const double s13_mm = 0.5 * ((um00 - um0m) * rdzcm + (w00m - wm0m) * rdx);
  S[4] = 0.25 * (s13_00 + s13_m0 + s13_0m + s13_mm);
  const double v00p = V(0, 0, 1), v00m = V(0, 0, -1), v0mp = V(0, -1, 1), v0mm = V(0, -1, -1);
  const double w0p0 = W(0, 1, 0), w0m0 = W(0, -1, 0), w0pm = W(0, 1, -1), w0mm = W(0, -1, -1);
  const double s23_00 = 0.5 * ((v00p - v000) * rdzc + (w0p0 - w000) * rdy);
  const double s23_m0 = 0.5 * ((v0mp - v0m0) * rdzc + (w000 - w0m0) * rdy);
  const double s23_0m = 0.5 * ((v000 - v00m) * rdzcm + (w0pm - w00m) * rdy);
  const double s23_mm = 0.5 * ((v0m0 - v0mm) * rdzcm + (w00m - w0mm) * rdy);
  S[5] = 0.25 * (s23_00 + s23_m0 + s23_0m + s23_mm);
  return sqrt(2.0 * (S[0] * S[0] + S[1] * S[1] + S[2] * S[2]) + 4.0 * (S[3] * S[3] + S[4] * S[4] + S[5] * S[5]));
}

// Static Smagorinsky, Eq. 4: nu_t = (C_s Delta D)^2 |S|, Delta = (dx dy dzf)^(1/3) (S4),
// D = 1 - exp(-d+/A+) with the local u_tau of the nearest z wall (S5).
CALES_HD double smag_point(const Ctx& c, const double* u, const double* v, const double* w, int i, int j, int k) {
  double S[6];
  double smag;
  if (interior_row(c, j, k)) {
    // no wall ghost in reach: direct loads at wrapped offsets
    const long long n = idx3(c, i, j, k);
    const Nbr o = neighbours(c, i, j, k);
    const int im = o.im, ip = o.ip, jm = o.jm, jp = o.jp;
    const long long km = o.km, kp = o.kp;
    auto at = [&](const double* __restrict__ q, int a, int b, int d) {
      return q[n + (d < 0 ? km : (d > 0 ? kp : 0)) + ((a < 0 ? im : (a > 0 ? ip : 0)) + (b < 0 ? jm : (b > 0 ? jp : 0)))];
    };
    auto U = [&](int a, int b, int d) { return at(u, a, b, d); };
    auto V = [&](int a, int b, int d) { return at(v, a, b, d); };
    auto W = [&](int a, int b, int d) { return at(w, a, b, d); };
    smag = strain_at(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], S);
  } else {
    auto U = [&](int a, int b, int d) { return velg<0>(c, u, i + a, j + b, k + d, GH_STRAIN); };
    auto V = [&](int a, int b, int d) { return velg<1>(c, v, i + a, j + b, k + d, GH_STRAIN); };
    auto W = [&](int a, int b, int d) { return velg<2>(c, w, i + a, j + b, k + d, GH_STRAIN); };
    smag = strain_at(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], S);
  }
  const double delta = c.delta[k];
  double D = 1.0;
  if (c.van_driest) {
    const double db = c.zc[k], dt = c.lz - c.zc[k];
    const int kw = (db <= dt) ? 0 : c.nz - 1;
    const double d = (db <= dt) ? db : dt;
    const double d1 = (kw == 0) ? c.zc[0] : c.lz - c.zc[c.nz - 1];
    const double uc = 0.5 * (velg<0>(c, u, i - 1, j, kw, GH_STRAIN) + velg<0>(c, u, i, j, kw, GH_STRAIN));
    const double vc = 0.5 * (velg<1>(c, v, i, j - 1, kw, GH_STRAIN) + velg<1>(c, v, i, j, kw, GH_STRAIN));
    const double tauw = c.nu * sqrt(uc * uc + vc * vc) / d1;
    const double utau = sqrt(tauw);
    D = 1.0 - exp(-(d * utau / c.nu) / c.aplus);
  }
  const double l = c.cs * delta * D;
  return l * l * smag;
}

// ------------------------------------------------------------------------------------------------------------
// Dynamic Smagorinsky, pass 1.  One CTA = one TX x TY tile of one k-plane.  Shared memory holds
//   raw : u, v, w on planes k-1, k, k+1 over the tile + halo 2 (ghosts synthesised by velg, GH_STRAIN mode),
//   flt : the face-wise test-filtered velocity on the same 3 planes over the tile + halo 1 (Eq. 9 needs its strain),
//   mid : centre velocities, |S| S_ij and |S| on plane k over the tile + halo 1 (the test filter reads a 3x3 patch).
// Test filter: separable (1/4,1/2,1/4) in x and y (S11); in a wall-bounded y the first off-wall rows
// keep the identity in y and the filter ratio there is alpha^(1/2) (x-only filter).
// Each output point forms L_ij (Eq. 7), M_ij (Eq. 8, S2), stores |S| and contributes L:M and M:M to the
// per-(k, j, x-tile) partial sums of Eq. 6.
// ------------------------------------------------------------------------------------------------------------
enum { DSM_TX = 32, DSM_TY = 2 /* exactly the two rows next to a y wall where F and the strain do not commute */, DSM_RX = DSM_TX + 4, DSM_RY = DSM_TY + 4, DSM_MX = DSM_TX + 2, DSM_MY = DSM_TY + 2 };
enum { DSM_RAW = 9 * DSM_RX * DSM_RY, DSM_FLT = 9 * DSM_MX * DSM_MY, DSM_MID = 10 * DSM_MX * DSM_MY,
       DSM_SMEM_DOUBLES = DSM_RAW + DSM_FLT + DSM_MID };

CALES_HD int dsm_raw_off(int comp, int pl, int ry, int rx) { return ((comp * 3 + pl) * DSM_RY + ry) * DSM_RX + rx; }
CALES_HD int dsm_mid_off(int q, int my, int mx) { return (q * DSM_MY + my) * DSM_MX + mx; }

// y weights of the test filter for a row with global index gj.  kind 0: centred data and u, w faces; 1: v faces.
CALES_HD void dsm_wy(const Ctx& c, int gj, int kind, double* wy) {
  wy[0] = 0.25; wy[1] = 0.5; wy[2] = 0.25;
  if (c.bc_y == BC_WALL) {
    if (kind == 0) { if (gj <= 0 || gj >= c.ny - 1) { wy[0] = 0.0; wy[1] = 1.0; wy[2] = 0.0; } }
    else { if (gj < 0 || gj >= c.ny - 1) { wy[0] = 0.0; wy[1] = 0.0; wy[2] = 0.0; } }
  }
}

// phase 1: load the raw tile
CALES_HD void dsm_load(int tid, int nth, const Ctx& c, const double* u, const double* v, const double* w, int i0, int j0, int k, double* raw) {
  const int per = DSM_RX * DSM_RY;
  for (int idx = tid; idx < 9 * per; idx += nth) {
    const int cp = idx / per, r = idx % per;
    const int comp = cp / 3, pl = cp % 3, ry = r / DSM_RX, rx = r % DSM_RX;
    const int gi = i0 - 2 + rx, gj = j0 - 2 + ry, gk = k - 1 + pl;
    double val = 0.0;
    if (gi <= c.nx + 1 && gj <= c.ny + 1) {
      if (comp == 0) val = velg<0>(c, u, gi, gj, gk, GH_STRAIN);
      else if (comp == 1) val = velg<1>(c, v, gi, gj, gk, GH_STRAIN);
      else val = velg<2>(c, w, gi, gj, gk, GH_STRAIN);
    }
    raw[idx] = val;
  }
}

// phase 2: filtered face velocities (3 comps x 3 planes) and the centre quantities of plane k on the mid region
CALES_HD void dsm_mid(int tid, int nth, const Ctx& c, int i0, int j0, int k, const double* raw, double* flt, double* mid) {
  const int per = DSM_MX * DSM_MY;
  for (int idx = tid; idx < 9 * per; idx += nth) {
    const int cp = idx / per, r = idx % per;
    const int comp = cp / 3, pl = cp % 3, my = r / DSM_MX, mx = r % DSM_MX;
    const int gj = j0 - 1 + my;
    // filtered face value of mid row m (global row j0 - 1 + m)
    auto fval = [&](int m) {
      double wy[3]; dsm_wy(c, j0 - 1 + m, comp == 1 ? 1 : 0, wy);
      double s = 0.0;
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        const double* row = raw + dsm_raw_off(comp, pl, m + b, mx);
        s += wy[b] * (0.25 * row[0] + 0.5 * row[1] + 0.25 * row[2]);
      }
      return s;
    };
    // Ghost rows of the FILTERED velocity at a wall-model y wall: the boundary condition is applied to the filtered field
    // (one-sided extrapolation of its first two rows), which is not the filter of the extrapolated raw field.
    if (c.bc_y == BC_WALL && c.wall_model_y && comp != 1 && (gj < 0 || gj >= c.ny))
      flt[idx] = gj < 0 ? 2.0 * fval(my + 1) - fval(my + 2) : 2.0 * fval(my - 1) - fval(my - 2);
    else flt[idx] = fval(my);
  }
  const double rdx = c.rdx, rdy = c.rdy, rdzf = c.rdzf[k], rdzc = c.rdzc[k], rdzcm = c.rdzc[k - 1];
  for (int r = tid; r < per; r += nth) {
    const int my = r / DSM_MX, mx = r % DSM_MX;
    auto U = [&](int a, int b, int d) { return raw[dsm_raw_off(0, 1 + d, my + 1 + b, mx + 1 + a)]; };
    auto V = [&](int a, int b, int d) { return raw[dsm_raw_off(1, 1 + d, my + 1 + b, mx + 1 + a)]; };
    auto W = [&](int a, int b, int d) { return raw[dsm_raw_off(2, 1 + d, my + 1 + b, mx + 1 + a)]; };
    double S[6];
    const double smag = strain_at(U, V, W, rdx, rdy, rdzf, rdzc, rdzcm, S);
    mid[dsm_mid_off(0, my, mx)] = 0.5 * (U(-1, 0, 0) + U(0, 0, 0));
    mid[dsm_mid_off(1, my, mx)] = 0.5 * (V(0, -1, 0) + V(0, 0, 0));
    mid[dsm_mid_off(2, my, mx)] = 0.5 * (W(0, 0, -1) + W(0, 0, 0));
#pragma unroll
    for (int q = 0; q < 6; ++q) mid[dsm_mid_off(3 + q, my, mx)] = smag * S[q];
    mid[dsm_mid_off(9, my, mx)] = smag;
  }
}

// phase 3: one output point (tx, ty); returns L:M and M:M through lm, mm and |S| through smag_out.
CALES_HD void dsm_point(const Ctx& c, int i0, int j0, int k, int tx, int ty, const double* flt, const double* mid, double* lm, double* mm, double* smag_out) {
  const int gj = j0 + ty;
  const int mx = tx + 1, my = ty + 1;
  double wy[3]; dsm_wy(c, gj, 0, wy);
  const double wx[3] = {0.25, 0.5, 0.25};
  double Fv[3] = {0, 0, 0}, Fp[6] = {0, 0, 0, 0, 0, 0}, Fs[6] = {0, 0, 0, 0, 0, 0};
#pragma unroll
  for (int b = 0; b < 3; ++b) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double wgt = wy[b] * wx[a];
      const int o = dsm_mid_off(0, my - 1 + b, mx - 1 + a);
      const int st = DSM_MX * DSM_MY;
      const double uc = mid[o], vc = mid[o + st], wc = mid[o + 2 * st];
      Fv[0] += wgt * uc; Fv[1] += wgt * vc; Fv[2] += wgt * wc;
      Fp[0] += wgt * (uc * uc); Fp[1] += wgt * (vc * vc); Fp[2] += wgt * (wc * wc);
      Fp[3] += wgt * (uc * vc); Fp[4] += wgt * (uc * wc); Fp[5] += wgt * (vc * wc);
#pragma unroll
      for (int q = 0; q < 6; ++q) Fs[q] += wgt * mid[o + (3 + q) * st];
    }
  }
  double L[6];
  L[0] = Fp[0] - Fv[0] * Fv[0]; L[1] = Fp[1] - Fv[1] * Fv[1]; L[2] = Fp[2] - Fv[2] * Fv[2];
  L[3] = Fp[3] - Fv[0] * Fv[1]; L[4] = Fp[4] - Fv[0] * Fv[2]; L[5] = Fp[5] - Fv[1] * Fv[2];
  // Eq. 9: strain of the test-filtered velocity
  const int fst = DSM_MX * DSM_MY;
  auto U = [&](int a, int b, int d) { return flt[((0 * 3 + 1 + d) * DSM_MY + my + b) * DSM_MX + mx + a]; };
  auto V = [&](int a, int b, int d) { return flt[((1 * 3 + 1 + d) * DSM_MY + my + b) * DSM_MX + mx + a]; };
  auto W = [&](int a, int b, int d) { return flt[((2 * 3 + 1 + d) * DSM_MY + my + b) * DSM_MX + mx + a]; };
  (void)fst;
  double St[6];
  const double stmag = strain_at(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], St);
  const double d2 = c.delta[k] * c.delta[k];
  double al = c.alpha;
  if (c.bc_y == BC_WALL && (gj == 0 || gj == c.ny - 1)) al = sqrt(c.alpha);
  double ll = 0.0, m2 = 0.0;
#pragma unroll
  for (int q = 0; q < 6; ++q) {
    const double M = 2.0 * d2 * (Fs[q] - al * al * stmag * St[q]);
    const double f = q < 3 ? 1.0 : 2.0;
    ll += f * L[q] * M; m2 += f * M * M;
  }
  *lm = ll; *mm = m2; *smag_out = mid[dsm_mid_off(9, my, mx)];
}

// ------------------------------------------------------------------------------------------------------------
// Dynamic Smagorinsky, pass 1, column-marching form (the production path; the tile kernel above serves the rows
// next to y walls).  Where the test filter has uniform weights, F commutes with the (linear, x-y shift-invariant)
// strain operator, so Eq. 9's strain of the filtered velocity equals the filtered strain, S~_ij = F(S_ij): the
// kernel filters 21 centred quantities  q = (u_i^c [3], u_i^c u_j^c [6], |S| S_ij [6], S_ij [6])  and needs no
// filtered face velocities.  A CTA is one row of TXB threads (TXB-2 output columns plus one halo column each side)
// at a fixed k; it marches over LY+2 rows of y.  Per row: every thread evaluates the 10 base values
// (u^c, v^c, w^c, S_ij, |S|) of its column, publishes them in shared memory, forms q and its x-filter from its two
// neighbours' base values, and keeps the separable y-filter as a two-row sliding window of Fx q in shared memory:
//   xq(r) = Fx q(r);   F q(r-1) = (xq(r-2) + 2 xq(r-1) + xq(r)) / 4.
// ------------------------------------------------------------------------------------------------------------
#ifndef CALES_DSMC_LY
#define CALES_DSMC_LY 32      // rows per CTA of the column march (experiments: -DCALES_DSMC_LY=64)
#endif
enum { DSMC_LY = CALES_DSMC_LY, DSMC_NB = 10, DSMC_NQ = 21 };

// base values of column gi at row gj (both already wrapped / interior): b[0..2] = u^c, v^c, w^c; b[3..8] = S_ij; b[9] = |S|
CALES_HD void dsmc_base(const Ctx& c, const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w,
                        int gi, int gj, int k, double* b) {
  double S[6];
  if (interior_row(c, gj, k)) {
    const long long n = idx3(c, gi, gj, k);
    const Nbr o = neighbours(c, gi, gj, k);
    auto at = [&](const double* __restrict__ q, int a, int bb, int d) {
      return q[n + (d < 0 ? o.km : (d > 0 ? o.kp : 0)) + ((a < 0 ? o.im : (a > 0 ? o.ip : 0)) + (bb < 0 ? o.jm : (bb > 0 ? o.jp : 0)))];
    };
    auto U = [&](int a, int bb, int d) { return at(u, a, bb, d); };
    auto V = [&](int a, int bb, int d) { return at(v, a, bb, d); };
    auto W = [&](int a, int bb, int d) { return at(w, a, bb, d); };
    b[9] = strain_at(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], S);
    b[0] = 0.5 * (U(-1, 0, 0) + U(0, 0, 0)); b[1] = 0.5 * (V(0, -1, 0) + V(0, 0, 0)); b[2] = 0.5 * (W(0, 0, -1) + W(0, 0, 0));
  } else {
    auto U = [&](int a, int bb, int d) { return velg<0>(c, u, gi + a, gj + bb, k + d, GH_STRAIN); };
    auto V = [&](int a, int bb, int d) { return velg<1>(c, v, gi + a, gj + bb, k + d, GH_STRAIN); };
    auto W = [&](int a, int bb, int d) { return velg<2>(c, w, gi + a, gj + bb, k + d, GH_STRAIN); };
    b[9] = strain_at(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], S);
    b[0] = 0.5 * (U(-1, 0, 0) + U(0, 0, 0)); b[1] = 0.5 * (V(0, -1, 0) + V(0, 0, 0)); b[2] = 0.5 * (W(0, 0, -1) + W(0, 0, 0));
  }
#pragma unroll
  for (int q = 0; q < 6; ++q) b[3 + q] = S[q];
}

// q (21 values) from the base values
CALES_HD void dsmc_q(const double* b, double* q) {
  q[0] = b[0]; q[1] = b[1]; q[2] = b[2];
  q[3] = b[0] * b[0]; q[4] = b[1] * b[1]; q[5] = b[2] * b[2]; q[6] = b[0] * b[1]; q[7] = b[0] * b[2]; q[8] = b[1] * b[2];
#pragma unroll
  for (int m = 0; m < 6; ++m) { q[9 + m] = b[9] * b[3 + m]; q[15 + m] = b[3 + m]; }
}

// Lilly contraction at one point from F q: returns L:M and M:M (Eq. 6-8, S2)
CALES_HD void dsmc_contract(const double* Fq, double d2, double alpha, double* lm, double* mm) {
  double L[6];
  L[0] = Fq[3] - Fq[0] * Fq[0]; L[1] = Fq[4] - Fq[1] * Fq[1]; L[2] = Fq[5] - Fq[2] * Fq[2];
  L[3] = Fq[6] - Fq[0] * Fq[1]; L[4] = Fq[7] - Fq[0] * Fq[2]; L[5] = Fq[8] - Fq[1] * Fq[2];
  const double* St = Fq + 15;
  const double stmag = sqrt(2.0 * (St[0] * St[0] + St[1] * St[1] + St[2] * St[2]) + 4.0 * (St[3] * St[3] + St[4] * St[4] + St[5] * St[5]));
  const double a2s = alpha * alpha * stmag;
  double ll = 0.0, m2 = 0.0;
#pragma unroll
  for (int m = 0; m < 6; ++m) {
    const double M = 2.0 * d2 * (Fq[9 + m] - a2s * St[m]);
    const double f = m < 3 ? 1.0 : 2.0;
    ll += f * L[m] * M; m2 += f * M * M;
  }
  *lm = ll; *mm = m2;
}

// Row r of the march for thread t.  Phase A: base values of (column t, row r) into sh[buf][.][t] and regs `b`.
// The global row is gj = wrap(j0 - 1 + r).
CALES_HD void dsmc_phaseA(const Ctx& c, const double* u, const double* v, const double* w, int txb, int t, int i0, int gj, int k,
                          double* shbuf /* [DSMC_NB][txb] */, double* b) {
  const int gi = ((i0 - 1 + t) % c.nx + c.nx) % c.nx;
  dsmc_base(c, u, v, w, gi, gj, k, b);
#pragma unroll
  for (int q = 0; q < DSMC_NB; ++q) shbuf[q * txb + t] = b[q];
}

// Phase B (threads 1..txb-2): x-filter of q from the neighbours' base values, then the y-filter over a window kept in
// SHARED memory: ring[slot][m][txb] holds Fx q of the two previous rows of every column (thread-private slots, so no
// barrier protects them); F q(r-1) = (xq(r-2) + 2 xq(r-1) + xq(r)) / 4.  When r >= 2 the filtered row r-1 is complete:
// returns true and sets *lm, *mm, *smag (of row r-1, this column).  (A register-resident window was measured slower:
// 224 registers per thread, and 19 % of all instructions were register moves of the sliding window.)
// The first NREG quantities keep their window in registers (wreg[2 * NREG]: xq(r-1), xq(r-2)), the rest in the ring.
template <int NREG>
CALES_HD bool dsmc_phaseB_sm(const Ctx& c, int txb, int t, int r, int k, const double* shbuf, const double* b, double* ring, double* wreg,
                             double* smag_prev, double* lm, double* mm, double* smag) {
  double bl[DSMC_NB], br[DSMC_NB];
#pragma unroll
  for (int q = 0; q < DSMC_NB; ++q) { bl[q] = shbuf[q * txb + t - 1]; br[q] = shbuf[q * txb + t + 1]; }
  double qc[DSMC_NQ], ql[DSMC_NQ], qr[DSMC_NQ];
  dsmc_q(b, qc); dsmc_q(bl, ql); dsmc_q(br, qr);
  double* r1 = ring + ((r + 1) & 1) * (DSMC_NQ * txb) + t;     // xq(r-1)
  double* r2 = ring + (r & 1) * (DSMC_NQ * txb) + t;           // xq(r-2); overwritten with xq(r)
  double Fq[DSMC_NQ];
#pragma unroll
  for (int m = 0; m < DSMC_NQ; ++m) {
    const double xq = 0.25 * (ql[m] + qr[m]) + 0.5 * qc[m];
    if (m < NREG) {
      Fq[m] = 0.25 * (wreg[NREG + m] + xq) + 0.5 * wreg[m];
      wreg[NREG + m] = wreg[m]; wreg[m] = xq;
    } else {
      Fq[m] = 0.25 * (r2[m * txb] + xq) + 0.5 * r1[m * txb];
      r2[m * txb] = xq;
    }
  }
  bool done = false;
  if (r >= 2) {
    const double d2 = c.delta[k] * c.delta[k];
    dsmc_contract(Fq, d2, c.alpha, lm, mm);
    *smag = *smag_prev;
    done = true;
  }
  *smag_prev = b[9];
  return done;
}

// Eq. 6 per row (j,k) from the x-tile partials, then per plane if requested; S13: <MM> = 0 -> c_s = 0.
// part: [k][j][ntx][2].  cs: [k] or [k][j].
CALES_HD void dsm_row_sums(const double* part, int ntx, long long row, double* ll, double* mm) {
  double a = 0.0, b = 0.0;
  for (int t = 0; t < ntx; ++t) { a += part[(row * ntx + t) * 2]; b += part[(row * ntx + t) * 2 + 1]; }
  *ll = a; *mm = b;
}

// pass 2: nu_t = c_s Delta^2 |S| with the clip of PAPER.md:128 (c_s >= 0) or of the total viscosity (S14)
CALES_HD double dsm_nut_value(const Ctx& c, const double* cs, double sm, int j, int k) {
  const double cc = c.dsm_plane ? cs[k] : cs[(long long)k * c.ny + j];
  const double d2 = c.delta[k] * c.delta[k];
  if (!c.dsm_clip_total) return (cc < 0.0 ? 0.0 : cc) * d2 * sm;
  const double t = cc * d2 * sm;
  return t < -c.nu ? -c.nu : t;
}
CALES_HD double dsm_nut_point(const Ctx& c, const double* cs, const double* smag, int i, int j, int k) {
  return dsm_nut_value(c, cs, smag[idx3(c, i, j, k)], j, k);
}

#ifdef __CUDACC__
__global__ void k_wall_stress(Ctx c, WallGeom g, const double* __restrict__ u, const double* __restrict__ v, double* __restrict__ tau, int* __restrict__ maxit) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
  const int wall = blockIdx.z >> 1, comp = blockIdx.z & 1;
  int it = 0;
  if (i < c.nx && j < c.ny) it = wall_stress_point(c, g, u, v, wall, comp, i, j, tau);
  it = __reduce_max_sync(0xffffffffu, it);
  if ((threadIdx.x & 31) == 0 && it > 0) atomicMax(maxit, it);
}
// grid (ceil(nx/32), ceil(nz/8), 4), block (32, 8)
__global__ void k_wall_stress_y(Ctx c, const double* __restrict__ u, const double* __restrict__ w, double* __restrict__ tau_y, int* __restrict__ maxit) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y * blockDim.y + threadIdx.y;
  int it = 0;
  if (i < c.nx && k < c.nz) it = wall_stress_y_point(c, u, w, blockIdx.z >> 1, blockIdx.z & 1, i, k, tau_y);
  it = __reduce_max_sync(0xffffffffu, it);
  if ((threadIdx.x & 31) == 0 && it > 0) atomicMax(maxit, it);
}
__global__ void __launch_bounds__(256) k_smag(Ctx c, const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w, double* __restrict__ nut) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
  if (i < c.nx && j < c.ny) nut[idx3(c, i, j, k)] = smag_point(c, u, v, w, i, j, k);
}
__global__ void k_fill(double* __restrict__ q, long long n, double val) {
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) q[t] = val;
}
// grid (ntx, nty, nz), block (32, 8)
// rows: blockIdx.y -> j0 = jtile0 + blockIdx.y * jstride (wall-row tiles of the duct: jtile0 = 0, jstride = ny - DSM_TY);
// only output rows with row_lo <= j < row_hi || j >= row_hi2 are written (the rest belongs to k_dsm_col).
__global__ void __launch_bounds__(256) k_dsm_pass1(Ctx c, const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w,
                                                   int jstride, int row_hi, int row_lo2, int pslots,
                                                   double* __restrict__ smag, double* __restrict__ part) {
  extern __shared__ double dsm_sm[];
  double* raw = dsm_sm; double* flt = raw + DSM_RAW; double* mid = flt + DSM_FLT;
  const int tid = threadIdx.x + DSM_TX * threadIdx.y, nth = DSM_TX * DSM_TY;
  const int i0 = blockIdx.x * DSM_TX, j0 = blockIdx.y * jstride, k = blockIdx.z;
  dsm_load(tid, nth, c, u, v, w, i0, j0, k, raw);
  __syncthreads();
  dsm_mid(tid, nth, c, i0, j0, k, raw, flt, mid);
  __syncthreads();
  const int i = i0 + threadIdx.x, j = j0 + threadIdx.y;
  double lm = 0.0, mm = 0.0;
  const bool mine = j < c.ny && (j < row_hi || j >= row_lo2);      // warp-uniform (one row per warp)
  if (i < c.nx && mine) {
    double sm;
    dsm_point(c, i0, j0, k, threadIdx.x, threadIdx.y, flt, mid, &lm, &mm, &sm);
    smag[idx3(c, i, j, k)] = sm;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { lm += __shfl_down_sync(0xffffffffu, lm, o); mm += __shfl_down_sync(0xffffffffu, mm, o); }
  if (threadIdx.x == 0 && mine) {
    const long long row = (long long)k * c.ny + j;
    part[(row * pslots + blockIdx.x) * 2] = lm;
    part[(row * pslots + blockIdx.x) * 2 + 1] = mm;
  }
}
// Column-marching pass 1.  grid (ceil(nx/(TXB-2)), ceil((jhi-jlo)/DSMC_LY), nz), block TXB (multiple of 32).
// Handles output rows [jlo, jhi); part: [k][j][pslots][2], this kernel fills slots blockIdx.x*nwarps + warp.
template <int TXB, int MINB, int NREG>
__global__ void __launch_bounds__(TXB, MINB) k_dsm_col_sm(const __grid_constant__ Ctx c, const double* __restrict__ u, const double* __restrict__ v,
                                                          const double* __restrict__ w, int jlo, int jhi, int pslots, double* __restrict__ smag,
                                                          double* __restrict__ part) {
  __shared__ double sh[2][DSMC_NB * TXB];
  __shared__ double ring[2 * DSMC_NQ * TXB];
  const int t = threadIdx.x, k = blockIdx.z;
  const int i0 = blockIdx.x * (TXB - 2);
  const int j0 = jlo + blockIdx.y * DSMC_LY;
  const int jend = min(j0 + DSMC_LY, jhi);
  const int nrows = jend - j0 + 2;
  const int gi = i0 - 1 + t;
  const bool outcol = t >= 1 && t <= TXB - 2 && gi < c.nx;
#pragma unroll
  for (int m = 0; m < 2 * DSMC_NQ; ++m) ring[m * TXB + t] = 0.0;
  double smag_prev = 0.0;
  double wreg[2 * NREG + 1];
#pragma unroll
  for (int m = 0; m < 2 * NREG + 1; ++m) wreg[m] = 0.0;
  for (int r = 0; r < nrows; ++r) {
    int gj = j0 - 1 + r;
    gj = gj < 0 ? gj + c.ny : (gj >= c.ny ? gj - c.ny : gj);
    double b[DSMC_NB];
    dsmc_phaseA(c, u, v, w, TXB, t, i0, gj, k, sh[r & 1], b);
    if (r + 2 < nrows && (t & 3) == 0 && k >= 1 && k <= c.nz - 2) {     // the row after next: pull its lines towards L1
      int gp = j0 + 1 + r + 1; gp = gp >= c.ny ? gp - c.ny : gp;
      const long long nn = idx3(c, ((i0 - 1 + t) % c.nx + c.nx) % c.nx, gp, k);
#pragma unroll
      for (int d = -1; d <= 1; ++d) {
        asm volatile("prefetch.global.L1 [%0];" ::"l"(u + nn + d * c.nxy));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(v + nn + d * c.nxy));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(w + nn + d * c.nxy));
      }
    }
    __syncthreads();
    double lm = 0.0, mm = 0.0, sm = 0.0;
    bool done = false;
    if (t >= 1 && t <= TXB - 2) done = dsmc_phaseB_sm<NREG>(c, TXB, t, r, k, sh[r & 1], b, ring, wreg, &smag_prev, &lm, &mm, &sm);
    if (r >= 2) {
      const int jo = j0 + r - 2;
      if (!(done && outcol)) { lm = 0.0; mm = 0.0; }
      else smag[idx3(c, gi, jo, k)] = sm;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) { lm += __shfl_down_sync(0xffffffffu, lm, o); mm += __shfl_down_sync(0xffffffffu, mm, o); }
      if ((t & 31) == 0) {
        const long long slot = ((long long)k * c.ny + jo) * pslots + blockIdx.x * (TXB / 32) + (t >> 5);
        part[slot * 2] = lm; part[slot * 2 + 1] = mm;
      }
    }
  }
}

// grid nz, block 128
__global__ void k_dsm_coef(Ctx c, const double* __restrict__ part, int ntx, double* __restrict__ cs) {
  __shared__ double sh[32];
  const int k = blockIdx.x;
  double pl = 0.0, pm = 0.0;
  for (int j = threadIdx.x; j < c.ny; j += blockDim.x) {
    double ll, mm;
    dsm_row_sums(part, ntx, (long long)k * c.ny + j, &ll, &mm);
    if (!c.dsm_plane) cs[(long long)k * c.ny + j] = (mm > 0.0) ? ll / mm : 0.0;
    pl += ll; pm += mm;
  }
  if (c.dsm_plane) {
    const double a = block_sum(pl, sh), b = block_sum(pm, sh);
    if (threadIdx.x == 0) cs[k] = (b > 0.0) ? a / b : 0.0;
  }
}
__global__ void __launch_bounds__(256) k_dsm_nut(Ctx c, const double* __restrict__ cs, const double* __restrict__ smag, double* __restrict__ nut) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
  if (i < c.nx && j < c.ny) nut[idx3(c, i, j, k)] = dsm_nut_point(c, cs, smag, i, j, k);
}
#endif

}  // namespace cales
