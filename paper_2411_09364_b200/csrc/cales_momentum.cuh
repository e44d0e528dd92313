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
};

// Returns u* at the point (for the bulk-velocity sum).
CALES_HD double rhs_point(const Ctx& c, const RhsArgs& a, int i, int j, int k) {
  const double rdx = c.rdx, rdy = c.rdy;
  const double dzfk = c.dzf[k], dzfp = c.dzf[k + 1], dzck = c.dzc[k], dzcm = c.dzc[k - 1];
  const double rdzf = c.rdzf[k], rdzc = c.rdzc[k], rdzcm = c.rdzc[k - 1], rdzfp = c.rdzf[k + 1];
  (void)dzcm; (void)dzck;
  const long long n = idx3(c, i, j, k);
  const bool vact = !(c.bc_y == BC_WALL && j == c.ny - 1);
  const bool wact = !(c.bc_z == BC_WALL && k == c.nz - 1);
#define UU(di, dj, dk) velg<0>(c, a.u, i + (di), j + (dj), k + (dk), GH_VISC)
#define VV(di, dj, dk) velg<1>(c, a.v, i + (di), j + (dj), k + (dk), GH_VISC)
#define WW(di, dj, dk) velg<2>(c, a.w, i + (di), j + (dj), k + (dk), GH_VISC)
  const double u000 = UU(0, 0, 0), up00 = UU(1, 0, 0), um00 = UU(-1, 0, 0), u0p0 = UU(0, 1, 0), u0m0 = UU(0, -1, 0),
               u00p = UU(0, 0, 1), u00m = UU(0, 0, -1), ump0 = UU(-1, 1, 0), um0p = UU(-1, 0, 1);
  const double v000 = VV(0, 0, 0), vp00 = VV(1, 0, 0), vm00 = VV(-1, 0, 0), v0p0 = VV(0, 1, 0), v0m0 = VV(0, -1, 0),
               v00p = VV(0, 0, 1), v00m = VV(0, 0, -1), vpm0 = VV(1, -1, 0), v0mp = VV(0, -1, 1);
  const double w000 = WW(0, 0, 0), wp00 = WW(1, 0, 0), wm00 = WW(-1, 0, 0), w0p0 = WW(0, 1, 0), w0m0 = WW(0, -1, 0),
               w00p = WW(0, 0, 1), w00m = WW(0, 0, -1), wp0m = WW(1, 0, -1), w0pm = WW(0, 1, -1);
#undef UU
#undef VV
#undef WW
  // ---- convective terms -d_j(u_i u_j) (weights of DESIGN.md S3)
  double Ru, Rv, Rw;
  {
    const double uxp = 0.5 * (u000 + up00), uxm = 0.5 * (um00 + u000);
    const double uyp = 0.5 * (u000 + u0p0), uym = 0.5 * (u0m0 + u000);
    const double vxp = 0.5 * (v000 + vp00), vxm = 0.5 * (v0m0 + vpm0);
    const double uzp = 0.5 * (u000 + u00p), uzm = 0.5 * (u00m + u000);
    const double wxp = 0.5 * (w000 + wp00), wxm = 0.5 * (w00m + wp0m);
    Ru = -((uxp * uxp - uxm * uxm) * rdx + (uyp * vxp - uym * vxm) * rdy + (uzp * wxp - uzm * wxm) * rdzf);
  }
  {
    const double vyp = 0.5 * (v000 + v0p0), vym = 0.5 * (v0m0 + v000);
    const double vxp = 0.5 * (v000 + vp00), vxm = 0.5 * (vm00 + v000);
    const double uyp = 0.5 * (u000 + u0p0), uym = 0.5 * (um00 + ump0);
    const double vzp = 0.5 * (v000 + v00p), vzm = 0.5 * (v00m + v000);
    const double wyp = 0.5 * (w000 + w0p0), wym = 0.5 * (w00m + w0pm);
    Rv = -((vxp * uyp - vxm * uym) * rdx + (vyp * vyp - vym * vym) * rdy + (vzp * wyp - vzm * wym) * rdzf);
  }
  {
    const double rc2 = 0.5 * rdzc;
    const double wzp = 0.5 * (w000 + w00p), wzm = 0.5 * (w00m + w000);
    const double wxp = 0.5 * (w000 + wp00), wxm = 0.5 * (wm00 + w000);
    const double uzp = (u000 * dzfk + u00p * dzfp) * rc2, uzm = (um00 * dzfk + um0p * dzfp) * rc2;
    const double wyp = 0.5 * (w000 + w0p0), wym = 0.5 * (w0m0 + w000);
    const double vzp = (v000 * dzfk + v00p * dzfp) * rc2, vzm = (v0m0 * dzfk + v0mp * dzfp) * rc2;
    Rw = -((wxp * uzp - wxm * uzm) * rdx + (wyp * vzp - wym * vzm) * rdy + (wzp * wzp - wzm * wzm) * rdzc);
  }
  // ---- molecular diffusion nu L u_i, z part kept apart for the Crank-Nicolson split
  const double rdx2 = rdx * rdx, rdy2 = rdy * rdy;
  const double lzu = ((u00p - u000) * rdzc - (u000 - u00m) * rdzcm) * rdzf;
  const double lzv = ((v00p - v000) * rdzc - (v000 - v00m) * rdzcm) * rdzf;
  const double lzw = ((w00p - w000) * rdzfp - (w000 - w00m) * rdzf) * rdzc;
  Ru += c.nu * ((up00 - 2.0 * u000 + um00) * rdx2 + (u0p0 - 2.0 * u000 + u0m0) * rdy2);
  Rv += c.nu * ((vp00 - 2.0 * v000 + vm00) * rdx2 + (v0p0 - 2.0 * v000 + v0m0) * rdy2);
  Rw += c.nu * ((wp00 - 2.0 * w000 + wm00) * rdx2 + (w0p0 - 2.0 * w000 + w0m0) * rdy2);
  if (!c.implicit_z) { Ru += c.nu * lzu; Rv += c.nu * lzv; Rw += c.nu * lzw; }
  // ---- SGS term d_j(2 nu_t S_ij), always explicit
  if (c.sgs) {
#define NT(di, dj, dk) scalg(c, a.nut, i + (di), j + (dj), k + (dk), -1.0)
    const double n000 = NT(0, 0, 0), np00 = NT(1, 0, 0), nm00 = NT(-1, 0, 0), n0p0 = NT(0, 1, 0), n0m0 = NT(0, -1, 0),
                 n00p = NT(0, 0, 1), n00m = NT(0, 0, -1), npp0 = NT(1, 1, 0), npm0 = NT(1, -1, 0), nmp0 = NT(-1, 1, 0),
                 np0p = NT(1, 0, 1), np0m = NT(1, 0, -1), nm0p = NT(-1, 0, 1), n0pp = NT(0, 1, 1), n0pm = NT(0, 1, -1),
                 n0mp = NT(0, -1, 1);
#undef NT
    // edge fluxes nu_edge * 2 S_ij at the edges around the three faces
    const double exy_00 = 0.25 * (n000 + np00 + n0p0 + npp0) * ((u0p0 - u000) * rdy + (vp00 - v000) * rdx);   // (i+1/2, j+1/2)
    const double exy_0m = 0.25 * (n0m0 + npm0 + n000 + np00) * ((u000 - u0m0) * rdy + (vpm0 - v0m0) * rdx);   // (i+1/2, j-1/2)
    const double exy_m0 = 0.25 * (nm00 + n000 + nmp0 + n0p0) * ((ump0 - um00) * rdy + (v000 - vm00) * rdx);   // (i-1/2, j+1/2)
    const double exz_00 = 0.25 * (n000 + np00 + n00p + np0p) * ((u00p - u000) * rdzc + (wp00 - w000) * rdx);  // (i+1/2, k+1/2)
    const double exz_0m = 0.25 * (n00m + np0m + n000 + np00) * ((u000 - u00m) * rdzcm + (wp0m - w00m) * rdx); // (i+1/2, k-1/2)
    const double exz_m0 = 0.25 * (nm00 + n000 + nm0p + n00p) * ((um0p - um00) * rdzc + (w000 - wm00) * rdx);  // (i-1/2, k+1/2)
    const double eyz_00 = 0.25 * (n000 + n0p0 + n00p + n0pp) * ((v00p - v000) * rdzc + (w0p0 - w000) * rdy);  // (j+1/2, k+1/2)
    const double eyz_0m = 0.25 * (n00m + n0pm + n000 + n0p0) * ((v000 - v00m) * rdzcm + (w0pm - w00m) * rdy); // (j+1/2, k-1/2)
    const double eyz_m0 = 0.25 * (n0m0 + n000 + n0mp + n00p) * ((v0mp - v0m0) * rdzc + (w000 - w0m0) * rdy);  // (j-1/2, k+1/2)
    Ru += (2.0 * np00 * (up00 - u000) * rdx - 2.0 * n000 * (u000 - um00) * rdx) * rdx + (exy_00 - exy_0m) * rdy + (exz_00 - exz_0m) * rdzf;
    Rv += (exy_00 - exy_m0) * rdx + (2.0 * n0p0 * (v0p0 - v000) * rdy - 2.0 * n000 * (v000 - v0m0) * rdy) * rdy + (eyz_00 - eyz_0m) * rdzf;
    Rw += (exz_00 - exz_m0) * rdx + (eyz_00 - eyz_m0) * rdy + (2.0 * n00p * (w00p - w000) * rdzfp - 2.0 * n000 * (w000 - w00m) * rdzf) * rdzc;
  }
  // ---- pressure gradient and the RK3 combination
  const double p000 = a.p[n];
  const double gpx = (scalg(c, a.p, i + 1, j, k, 1.0) - p000) * rdx;
  const double gpy = (scalg(c, a.p, i, j + 1, k, 1.0) - p000) * rdy;
  const double gpz = (scalg(c, a.p, i, j, k + 1, 1.0) - p000) * rdzc;
  double ru0 = 0.0, rv0 = 0.0, rw0 = 0.0;
  if (a.be != 0.0) { ru0 = a.Ru0[n]; rv0 = a.Rv0[n]; rw0 = a.Rw0[n]; }
  if (!vact) Rv = 0.0;
  if (!wact) Rw = 0.0;
  double us = u000 + a.dt * (a.al * Ru + a.be * ru0 - a.ga * gpx);
  double vs = v000 + a.dt * (a.al * Rv + a.be * rv0 - a.ga * gpy);
  double ws = w000 + a.dt * (a.al * Rw + a.be * rw0 - a.ga * gpz);
  if (c.implicit_z) {
    // Eq. 20: + gamma nu L_zz u^k explicitly; then the right-hand side of Eq. 21: u** - c L_zz u^k, c = gamma nu dt / 2
    const double cimp = 0.5 * a.ga * c.nu * a.dt;
    us += a.dt * a.ga * c.nu * lzu - cimp * lzu;
    vs += a.dt * a.ga * c.nu * lzv - cimp * lzv;
    ws += a.dt * a.ga * c.nu * lzw - cimp * lzw;
  }
  if (!vact) vs = 0.0;
  if (!wact) ws = 0.0;
  a.us[n] = us; a.vs[n] = vs; a.ws[n] = ws;
  if (a.store_R) { a.Ru1[n] = Ru; a.Rv1[n] = Rv; a.Rw1[n] = Rw; }
  return us;
}

// Same arithmetic as rhs_point for a point whose stencil needs no wall ghost: direct loads at precomputed offsets,
// reciprocal tables instead of divisions, the factors 1/2 and 1/4 of the interpolations folded into the metric terms.
CALES_HD double rhs_point_fast(const Ctx& c, const RhsArgs& a, int i, int j, int k) {
  const long long n = idx3(c, i, j, k);
  const Nbr o = neighbours(c, i, j, k);
  const double rdx = c.rdx, rdy = c.rdy;     // uniform: hoisted by the compiler
  const double dzfk = c.dzf[k], dzfp = c.dzf[k + 1];
  const double rdzf = c.rdzf[k], rdzfp = c.rdzf[k + 1], rdzc = c.rdzc[k], rdzcm = c.rdzc[k - 1];
  const double* __restrict__ U = a.u + n; const double* __restrict__ Um = U + o.km; const double* __restrict__ Up = U + o.kp;
  const double* __restrict__ V = a.v + n; const double* __restrict__ Vm = V + o.km; const double* __restrict__ Vp = V + o.kp;
  const double* __restrict__ W = a.w + n; const double* __restrict__ Wm = W + o.km; const double* __restrict__ Wp = W + o.kp;
  const double u000 = U[0], up00 = U[o.ip], um00 = U[o.im], u0p0 = U[o.jp], u0m0 = U[o.jm], ump0 = U[o.jp + o.im],
               u00p = Up[0], u00m = Um[0], um0p = Up[o.im];
  const double v000 = V[0], vp00 = V[o.ip], vm00 = V[o.im], v0p0 = V[o.jp], v0m0 = V[o.jm], vpm0 = V[o.jm + o.ip],
               v00p = Vp[0], v00m = Vm[0], v0mp = Vp[o.jm];
  const double w000 = W[0], wp00 = W[o.ip], wm00 = W[o.im], w0p0 = W[o.jp], w0m0 = W[o.jm],
               w00p = Wp[0], w00m = Wm[0], wp0m = Wm[o.ip], w0pm = Wm[o.jp];
  const double qx = 0.25 * rdx, qy = 0.25 * rdy, qzf = 0.25 * rdzf, qzc = 0.25 * rdzc;
  double Ru, Rv, Rw;
  {  // -d_j(u u_j): sums instead of means, the 1/4 sits in qx, qy, qzf
    const double uxp = u000 + up00, uxm = um00 + u000, uyp = u000 + u0p0, uym = u0m0 + u000;
    const double vxp = v000 + vp00, vxm = v0m0 + vpm0, uzp = u000 + u00p, uzm = u00m + u000;
    const double wxp = w000 + wp00, wxm = w00m + wp0m;
    Ru = -((uxp * uxp - uxm * uxm) * qx + (uyp * vxp - uym * vxm) * qy + (uzp * wxp - uzm * wxm) * qzf);
    const double vyp = v000 + v0p0, vym = v0m0 + v000, vxq = vm00 + v000, uym2 = um00 + ump0;
    const double vzp = v000 + v00p, vzm = v00m + v000, wyp = w000 + w0p0, wym = w00m + w0pm;
    Rv = -((vxp * uyp - vxq * uym2) * qx + (vyp * vyp - vym * vym) * qy + (vzp * wyp - vzm * wym) * qzf);
    const double wzp = w000 + w00p, wzm = w00m + w000, wxq = wm00 + w000, wyq = w0m0 + w000;
    const double uzP = u000 * dzfk + u00p * dzfp, uzM = um00 * dzfk + um0p * dzfp;      // 2 dzc x the flux-consistent mean
    const double vzP = v000 * dzfk + v00p * dzfp, vzM = v0m0 * dzfk + v0mp * dzfp;
    Rw = -(((wxp * uzP - wxq * uzM) * qx + (wyp * vzP - wyq * vzM) * qy) * rdzc + (wzp * wzp - wzm * wzm) * qzc);
  }
  const double rdx2 = rdx * rdx, rdy2 = rdy * rdy;
  const double lzu = ((u00p - u000) * rdzc - (u000 - u00m) * rdzcm) * rdzf;
  const double lzv = ((v00p - v000) * rdzc - (v000 - v00m) * rdzcm) * rdzf;
  const double lzw = ((w00p - w000) * rdzfp - (w000 - w00m) * rdzf) * rdzc;
  double du = (up00 - 2.0 * u000 + um00) * rdx2 + (u0p0 - 2.0 * u000 + u0m0) * rdy2;
  double dv = (vp00 - 2.0 * v000 + vm00) * rdx2 + (v0p0 - 2.0 * v000 + v0m0) * rdy2;
  double dw = (wp00 - 2.0 * w000 + wm00) * rdx2 + (w0p0 - 2.0 * w000 + w0m0) * rdy2;
  if (!c.implicit_z) { du += lzu; dv += lzv; dw += lzw; }
  Ru += c.nu * du; Rv += c.nu * dv; Rw += c.nu * dw;
  if (c.sgs) {
    const double* __restrict__ N = a.nut + n; const double* __restrict__ Nm = N + o.km; const double* __restrict__ Np = N + o.kp;
    const double n000 = N[0], np00 = N[o.ip], nm00 = N[o.im], n0p0 = N[o.jp], n0m0 = N[o.jm], n00p = Np[0], n00m = Nm[0],
                 npp0 = N[o.jp + o.ip], npm0 = N[o.jm + o.ip], nmp0 = N[o.jp + o.im], np0p = Np[o.ip], np0m = Nm[o.ip],
                 nm0p = Np[o.im], n0pp = Np[o.jp], n0pm = Nm[o.jp], n0mp = Np[o.jm];
    const double nx0 = n000 + np00, ny0 = n000 + n0p0, nz0 = n000 + n00p;
    // 4 x edge viscosity x 2 S_ij at the edges around the three faces
    const double exy_00 = (nx0 + n0p0 + npp0) * ((u0p0 - u000) * rdy + (vp00 - v000) * rdx);
    const double exy_0m = (nx0 + n0m0 + npm0) * ((u000 - u0m0) * rdy + (vpm0 - v0m0) * rdx);
    const double exy_m0 = (ny0 + nm00 + nmp0) * ((ump0 - um00) * rdy + (v000 - vm00) * rdx);
    const double exz_00 = (nx0 + n00p + np0p) * ((u00p - u000) * rdzc + (wp00 - w000) * rdx);
    const double exz_0m = (nx0 + n00m + np0m) * ((u000 - u00m) * rdzcm + (wp0m - w00m) * rdx);
    const double exz_m0 = (nz0 + nm00 + nm0p) * ((um0p - um00) * rdzc + (w000 - wm00) * rdx);
    const double eyz_00 = (ny0 + n00p + n0pp) * ((v00p - v000) * rdzc + (w0p0 - w000) * rdy);
    const double eyz_0m = (ny0 + n00m + n0pm) * ((v000 - v00m) * rdzcm + (w0pm - w00m) * rdy);
    const double eyz_m0 = (nz0 + n0m0 + n0mp) * ((v0mp - v0m0) * rdzc + (w000 - w0m0) * rdy);
    Ru += (np00 * (up00 - u000) - n000 * (u000 - um00)) * (2.0 * rdx2) + (exy_00 - exy_0m) * qy + (exz_00 - exz_0m) * qzf;
    Rv += (exy_00 - exy_m0) * qx + (n0p0 * (v0p0 - v000) - n000 * (v000 - v0m0)) * (2.0 * rdy2) + (eyz_00 - eyz_0m) * qzf;
    Rw += (exz_00 - exz_m0) * qx + (eyz_00 - eyz_m0) * qy + (n00p * (w00p - w000) * rdzfp - n000 * (w000 - w00m) * rdzf) * (2.0 * rdzc);
  }
  const double* __restrict__ P = a.p + n;
  const double p000 = P[0];
  const double gpx = (P[o.ip] - p000) * rdx, gpy = (P[o.jp] - p000) * rdy, gpz = (P[o.kp] - p000) * rdzc;
  double ru0 = 0.0, rv0 = 0.0, rw0 = 0.0;
  if (a.be != 0.0) { ru0 = a.Ru0[n]; rv0 = a.Rv0[n]; rw0 = a.Rw0[n]; }
  double us = u000 + a.dt * (a.al * Ru + a.be * ru0 - a.ga * gpx);
  double vs = v000 + a.dt * (a.al * Rv + a.be * rv0 - a.ga * gpy);
  double ws = w000 + a.dt * (a.al * Rw + a.be * rw0 - a.ga * gpz);
  if (c.implicit_z) {
    const double f = a.dt * a.ga * c.nu - 0.5 * a.ga * c.nu * a.dt;
    us += f * lzu; vs += f * lzv; ws += f * lzw;
  }
  a.us[n] = us; a.vs[n] = vs; a.ws[n] = ws;
  if (a.store_R) { a.Ru1[n] = Ru; a.Rv1[n] = Rv; a.Rw1[n] = Rw; }
  return us;
}

// The point function both the kernel and the host emulator call.
CALES_HD double rhs_any(const Ctx& c, const RhsArgs& a, int i, int j, int k) {
  return interior_row(c, j, k) ? rhs_point_fast(c, a, i, j, k) : rhs_point(c, a, i, j, k);
}

struct CorrArgs {
  const double *phi, *us, *vs, *ws;
  double *u, *v, *w, *p;
  const double* shift;     // device scalar: uniform shift of u* that restores the bulk velocity (0 if no forcing)
  double gdt;              // gamma dt
  double cimp;             // gamma nu dt / 2 if implicit z else 0
  int update_p;
};

// Eq. 13: u = u* - gamma dt grad(phi) (+ the bulk shift of u*); Eq. 14 / 22: p += phi (- c L_zz phi).
CALES_HD void correct_point(const Ctx& c, const CorrArgs& a, int i, int j, int k) {
  const long long n = idx3(c, i, j, k);
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
  const double sh = a.shift ? *a.shift : 0.0;
  const double rdzc = c.rdzc[k];
  a.u[n] = (a.us[n] + sh) - a.gdt * (phx - ph) * c.rdx;
  a.v[n] = vact ? a.vs[n] - a.gdt * (phy - ph) * c.rdy : 0.0;
  a.w[n] = wact ? a.ws[n] - a.gdt * (phz - ph) * rdzc : 0.0;
  if (a.update_p) {
    double dp = ph;
    if (a.cimp != 0.0) dp -= a.cimp * (((phz - ph) * rdzc - (ph - phm) * c.rdzc[k - 1]) * c.rdzf[k]);
    a.p[n] += dp;
  }
}

CALES_HD double divergence_point(const Ctx& c, const double* u, const double* v, const double* w, int i, int j, int k) {
  return (velg<0>(c, u, i, j, k, GH_STRAIN) - velg<0>(c, u, i - 1, j, k, GH_STRAIN)) * c.rdx +
         (velg<1>(c, v, i, j, k, GH_STRAIN) - velg<1>(c, v, i, j - 1, k, GH_STRAIN)) * c.rdy +
         (velg<2>(c, w, i, j, k, GH_STRAIN) - velg<2>(c, w, i, j, k - 1, GH_STRAIN)) * c.rdzf[k];
}

#ifdef __CUDACC__
// wall rows / planes: the generic path, kept out of line so that it does not weigh on the interior path's registers
__device__ __noinline__ double rhs_point_wall(const Ctx& c, const RhsArgs& a, int i, int j, int k) { return rhs_point(c, a, i, j, k); }

// grid (ceil(nx/32), ceil(ny/8), nz), block (32, 8).  partial[block] = sum over the block of u* dzf[k] (or nullptr).
__global__ void __launch_bounds__(256, 2) k_rhs(Ctx c, RhsArgs a, double* __restrict__ partial) {
  __shared__ double sh[32];
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
  double s = 0.0;
  if (i < c.nx && j < c.ny) s = (interior_row(c, j, k) ? rhs_point_fast(c, a, i, j, k) : rhs_point_wall(c, a, i, j, k)) * c.dzf[k];
  if (partial) {
    const double t = block_sum(s, sh);
    if (threadIdx.x == 0 && threadIdx.y == 0) partial[blockIdx.x + gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z)] = t;
  }
}
__global__ void __launch_bounds__(256) k_correct(Ctx c, CorrArgs a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
  if (i < c.nx && j < c.ny) correct_point(c, a, i, j, k);
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
// scal[0] = shift = u_bulk - sum/(nx ny lz); scal[1] = forcing = shift / (gamma dt); scal[2] = mean
__global__ void k_bulk_finish(Ctx c, const double* __restrict__ in, int n, double gdt, double* __restrict__ scal) {
  __shared__ double sh[32];
  double s = 0.0;
  for (int q = threadIdx.x; q < n; q += blockDim.x) s += in[q];
  const double t = block_sum(s, sh);
  if (threadIdx.x == 0) {
    const double m = t / ((double)c.nx * (double)c.ny * c.lz);
    const double shf = c.u_bulk - m;
    scal[0] = shf; scal[1] = shf / gdt; scal[2] = m;
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
__global__ void k_max_stage(const double* __restrict__ in, long long n, double* __restrict__ out) {
  __shared__ double sh[32];
  const long long per = (n + gridDim.x - 1) / gridDim.x;
  const long long b0 = per * blockIdx.x, b1 = min(n, b0 + per);
  double s = 0.0;
  for (long long q = b0 + threadIdx.x; q < b1; q += blockDim.x) s = fmax(s, in[q]);
  const double t = block_max(s, sh);
  if (threadIdx.x == 0) out[blockIdx.x] = t;
}
#endif

}  // namespace cales
