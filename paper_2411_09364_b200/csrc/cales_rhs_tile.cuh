// cales_rhs_tile.cuh -- the production momentum kernel: fused right-hand side + RK3 update of Eq. 11 / Eq. 20
// as a z-marching, shared-memory staged stencil.
//
// A CTA owns an RT_TX x RT_TY tile of (i,j) columns and marches over a chunk of k-planes.  Each plane of
// u, v, w, nu_t, p (tile + halo 1) is staged ONCE into a 4-slot shared-memory ring by asynchronous copies
// (cp.async, LDGSTS) issued one plane ahead of the arithmetic, so every global value is fetched once per CTA, the
// copy of plane k+2 overlaps the arithmetic of plane k, and all 50-odd stencil reads of a point are shared-memory
// reads.  Boundary conditions (Alg. 2) are applied WHEN A HALO ELEMENT IS STAGED: periodic wrap
// is address arithmetic of the async copy; wall ghosts (no-slip mirror, zero wall-normal face, Neumann p, nu_t = -
// interior, wall-model stress ghost) are produced by the generic accessors velg / scalg and stored synchronously.
// The arithmetic itself (rhs_core) is written once over an accessor and is shared with the host emulator.
#pragma once
#include "cales_common.cuh"
#include "cales_momentum.cuh"
#include "cales_closures.cuh"
#ifdef __CUDACC__
#include <cuda.h>
#endif

namespace cales {

#ifndef CALES_RT_TY
#define CALES_RT_TY 16
#endif
#ifndef CALES_RT_MINB
#define CALES_RT_MINB 2
#endif
enum { RT_TX = 32, RT_TY = CALES_RT_TY, RT_RPT = 2, RT_TW = RT_TX + 2, RT_TH = RT_TY + 2, RT_PLANE = RT_TW * RT_TH, RT_NF = 5, RT_NSLOT = 4,
       RT_THREADS = RT_TX * RT_TY / RT_RPT, RT_SMEM_DOUBLES = RT_NSLOT * RT_NF * RT_PLANE,
       RT_EPT = (RT_PLANE + RT_THREADS - 1) / RT_THREADS };   // halo-tile positions per thread

// Momentum right-hand side and RK update at one point over an accessor A with
//   A.U(di,dj,dk), A.V, A.W : velocity components incl. ghosts (viscous-flux ghost at wall-model walls),
//   A.NT(di,dj,dk)          : nu_t incl. ghosts,   A.P(di,dj,dk): pressure incl. ghosts.
// Second-order central, divergence-form advection (S1, S3); the factors 1/2, 1/4 of the interpolations are folded into
// the metric terms.  Returns u* at the point.
// z metrics of one plane, loaded once per plane by the marching kernel
struct ZMet { double dzfk, dzfp, rdzf, rdzfp, rdzc, rdzcm; };
CALES_HD ZMet zmet_at(const Ctx& c, int k) { return ZMet{c.dzf[k], c.dzf[k + 1], c.rdzf[k], c.rdzf[k + 1], c.rdzc[k], c.rdzc[k - 1]}; }

// ru0, rv0, rw0: R^{k-1} at the point (read by the caller ahead of the stencil arithmetic so that the loads are in flight early)
template <class A>
CALES_HD double rhs_core_r(const Ctx& c, const RhsArgs& a, const A& q, int i, int j, int k, const ZMet& zm, double ru0, double rv0, double rw0) {
  const long long n = idx3(c, i, j, k);
  const double rdx = c.rdx, rdy = c.rdy;
  const double dzfk = zm.dzfk, dzfp = zm.dzfp, rdzf = zm.rdzf, rdzfp = zm.rdzfp, rdzc = zm.rdzc, rdzcm = zm.rdzcm;
  const bool vact = !(c.bc_y == BC_WALL && j == c.ny - 1);
  const bool wact = !(c.bc_z == BC_WALL && k == c.nz - 1);
  const double u000 = q.U(0, 0, 0), up00 = q.U(1, 0, 0), um00 = q.U(-1, 0, 0), u0p0 = q.U(0, 1, 0), u0m0 = q.U(0, -1, 0),
               ump0 = q.U(-1, 1, 0), u00p = q.U(0, 0, 1), u00m = q.U(0, 0, -1), um0p = q.U(-1, 0, 1);
  const double v000 = q.V(0, 0, 0), vp00 = q.V(1, 0, 0), vm00 = q.V(-1, 0, 0), v0p0 = q.V(0, 1, 0), v0m0 = q.V(0, -1, 0),
               vpm0 = q.V(1, -1, 0), v00p = q.V(0, 0, 1), v00m = q.V(0, 0, -1), v0mp = q.V(0, -1, 1);
  const double w000 = q.W(0, 0, 0), wp00 = q.W(1, 0, 0), wm00 = q.W(-1, 0, 0), w0p0 = q.W(0, 1, 0), w0m0 = q.W(0, -1, 0),
               w00p = q.W(0, 0, 1), w00m = q.W(0, 0, -1), wp0m = q.W(1, 0, -1), w0pm = q.W(0, 1, -1);
  const double qx = 0.25 * rdx, qy = 0.25 * rdy, qzf = 0.25 * rdzf, qzc = 0.25 * rdzc;
  double Ru, Rv, Rw;
  {  // -d_j(u_i u_j), weights of DESIGN.md S3
    const double uxp = u000 + up00, uxm = um00 + u000, uyp = u000 + u0p0, uym = u0m0 + u000;
    const double vxp = v000 + vp00, vxm = v0m0 + vpm0, uzp = u000 + u00p, uzm = u00m + u000;
    const double wxp = w000 + wp00, wxm = w00m + wp0m;
    Ru = -((uxp * uxp - uxm * uxm) * qx + (uyp * vxp - uym * vxm) * qy + (uzp * wxp - uzm * wxm) * qzf);
    const double vyp = v000 + v0p0, vym = v0m0 + v000, vxq = vm00 + v000, uym2 = um00 + ump0;
    const double vzp = v000 + v00p, vzm = v00m + v000, wyp = w000 + w0p0, wym = w00m + w0pm;
    Rv = -((vxp * uyp - vxq * uym2) * qx + (vyp * vyp - vym * vym) * qy + (vzp * wyp - vzm * wym) * qzf);
    const double wzp = w000 + w00p, wzm = w00m + w000, wxq = wm00 + w000, wyq = w0m0 + w000;
    const double uzP = u000 * dzfk + u00p * dzfp, uzM = um00 * dzfk + um0p * dzfp;
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
  const double lxu = du, lxv = dv, lxw = dw;      // (L_xx + L_yy) u_i
  if (!c.implicit_z) { du += lzu; dv += lzv; dw += lzw; }
  if (c.implicit_z != 2) { Ru += c.nu * du; Rv += c.nu * dv; Rw += c.nu * dw; }      // Eq. 17: all of nu L_jj u goes with gamma
  if (c.sgs) {   // d_j(2 nu_t S_ij), edge viscosity = mean of the 4 surrounding centres (S6)
    const double n000 = q.NT(0, 0, 0), np00 = q.NT(1, 0, 0), nm00 = q.NT(-1, 0, 0), n0p0 = q.NT(0, 1, 0), n0m0 = q.NT(0, -1, 0),
                 n00p = q.NT(0, 0, 1), n00m = q.NT(0, 0, -1), npp0 = q.NT(1, 1, 0), npm0 = q.NT(1, -1, 0), nmp0 = q.NT(-1, 1, 0),
                 np0p = q.NT(1, 0, 1), np0m = q.NT(1, 0, -1), nm0p = q.NT(-1, 0, 1), n0pp = q.NT(0, 1, 1), n0pm = q.NT(0, 1, -1),
                 n0mp = q.NT(0, -1, 1);
    const double nx0 = n000 + np00, ny0 = n000 + n0p0, nz0 = n000 + n00p;
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
  const double p000 = q.P(0, 0, 0);
  const double gpx = (q.P(1, 0, 0) - p000) * rdx, gpy = (q.P(0, 1, 0) - p000) * rdy, gpz = (q.P(0, 0, 1) - p000) * rdzc;
  if (!vact) Rv = 0.0;
  if (!wact) Rw = 0.0;
  const double dt = a.sc ? ld_scalar(a.sc + RK_DT) : a.dt;
  double us = u000 + dt * (a.al * Ru + a.be * ru0 - a.ga * gpx);
  double vs = v000 + dt * (a.al * Rv + a.be * rv0 - a.ga * gpy);
  double ws = w000 + dt * (a.al * Rw + a.be * rw0 - a.ga * gpz);
  if (c.implicit_z) {   // Eq. 20 explicit half + right-hand side of Eq. 21
    const double fe = dt * a.ga * c.nu, fi = 0.5 * a.ga * c.nu * dt;
    double ltu = lzu, ltv = lzv;        // L_zz of the implicit operator applied to u^k
    if (c.wall_model) {                 // zero-flux closure: the modelled wall stress is a source outside the implicit operator
      const double up = (k < c.nz - 1) ? 1.0 : 0.0, lo = (k > 0) ? 1.0 : 0.0;
      ltu = (up * (u00p - u000) * rdzc - lo * (u000 - u00m) * rdzcm) * rdzf;
      ltv = (up * (v00p - v000) * rdzc - lo * (v000 - v00m) * rdzcm) * rdzf;
    }
    us += fe * lzu - fi * ltu; vs += fe * lzv - fi * ltv; ws += (fe - fi) * lzw;
    if (c.implicit_z == 2) { us += (fe - fi) * lxu; vs += (fe - fi) * lxv; ws += (fe - fi) * lxw; }   // Eq. 17 explicit half + right-hand side of Eq. 18
  }
  if (!vact) vs = 0.0;
  if (!wact) ws = 0.0;
  a.us[n] = us; a.vs[n] = vs; a.ws[n] = ws;
  if (a.store_R) { a.Ru1[n] = Ru; a.Rv1[n] = Rv; a.Rw1[n] = Rw; }
  return us;
}

template <class A>
CALES_HD double rhs_core(const Ctx& c, const RhsArgs& a, const A& q, int i, int j, int k, const ZMet& zm) {
  double ru0 = 0.0, rv0 = 0.0, rw0 = 0.0;
  if (a.be != 0.0) { const long long n = idx3(c, i, j, k); ru0 = a.Ru0[n]; rv0 = a.Rv0[n]; rw0 = a.Rw0[n]; }
  return rhs_core_r(c, a, q, i, j, k, zm, ru0, rv0, rw0);
}

// nu_t with ghosts (ghost = -interior at walls, S7; periodic wrap otherwise).  With the lazy dynamic model (a.cs) the
// array holds |S| and the value is formed here from the coefficient of the row / plane the (possibly mirrored) element lies in.
CALES_HD double nutg(const Ctx& c, const RhsArgs& a, int i, int j, int k) {
  i = wrapi(i, c.nx);
  double s = 1.0;
  if (c.bc_y == BC_PER) j = wrapi(j, c.ny);
  else { if (j < 0) { j = 0; s = -s; } else if (j >= c.ny) { j = c.ny - 1; s = -s; } }
  if (c.bc_z == BC_PER) k = wrapi(k, c.nz);
  else { if (k < 0) { k = 0; s = -s; } else if (k >= c.nz) { k = c.nz - 1; s = -s; } }
  const double q = a.nut[idx3(c, i, j, k)];
  return s * (a.cs ? dsm_nut_value(c, a.cs, q, j, k) : q);
}

// Accessor over the generic boundary-condition accessors (any point, any boundary).
struct GhostAcc {
  const Ctx& c; const RhsArgs& a; int i, j, k;
  CALES_HD double U(int di, int dj, int dk) const { return velg<0>(c, a.u, i + di, j + dj, k + dk, GH_VISC); }
  CALES_HD double V(int di, int dj, int dk) const { return velg<1>(c, a.v, i + di, j + dj, k + dk, GH_VISC); }
  CALES_HD double W(int di, int dj, int dk) const { return velg<2>(c, a.w, i + di, j + dj, k + dk, GH_VISC); }
  CALES_HD double NT(int di, int dj, int dk) const { return nutg(c, a, i + di, j + dj, k + dk); }
  CALES_HD double P(int di, int dj, int dk) const { return scalg(c, a.p, i + di, j + dj, k + dk, 1.0); }
};

// Value staged for field f (0 u, 1 v, 2 w, 3 nu_t, 4 p) at (gi,gj,gk), -1 <= gi <= nx, -1 <= gj <= ny, -1 <= gk <= nz.
CALES_HD double rt_elem(const Ctx& c, const RhsArgs& a, int f, int gi, int gj, int gk) {
  switch (f) {
    case 0: return velg<0>(c, a.u, gi, gj, gk, GH_VISC);
    case 1: return velg<1>(c, a.v, gi, gj, gk, GH_VISC);
    case 2: return velg<2>(c, a.w, gi, gj, gk, GH_VISC);
    case 3: return c.sgs ? nutg(c, a, gi, gj, gk) : 0.0;
    default: return scalg(c, a.p, gi, gj, gk, 1.0);
  }
}

// Accessor over three staged planes (k-1, k, k+1): sl[d] points at field 0 of the slot, ctr = (ly+1)*RT_TW + lx+1.
template <int FSTRIDE, int PITCH>
struct TileAccT {
  const double* sl[3]; int ctr;
  CALES_HD double at(int f, int di, int dj, int dk) const { return sl[dk + 1][f * FSTRIDE + ctr + dj * PITCH + di]; }
  CALES_HD double U(int di, int dj, int dk) const { return at(0, di, dj, dk); }
  CALES_HD double V(int di, int dj, int dk) const { return at(1, di, dj, dk); }
  CALES_HD double W(int di, int dj, int dk) const { return at(2, di, dj, dk); }
  CALES_HD double NT(int di, int dj, int dk) const { return at(3, di, dj, dk); }
  CALES_HD double P(int di, int dj, int dk) const { return at(4, di, dj, dk); }
};
typedef TileAccT<RT_PLANE, RT_TW> TileAcc;

// k-planes per CTA: enough chunks for ~8 waves of 2 CTAs/SM on 148 SMs, at least 8 planes per chunk
static inline int rt_chunk(int nx, int ny, int nz) {
  const long long tiles = (long long)((nx + RT_TX - 1) / RT_TX) * ((ny + RT_TY - 1) / RT_TY);
  long long want = (8 * 296 + tiles - 1) / tiles;
  const long long maxc = nz / 8 > 0 ? nz / 8 : 1;
  if (want > maxc) want = maxc;
  if (want < 1) want = 1;
  // at most ~96 planes per CTA: neighbouring CTAs that march a whole tall column drift apart by more planes than L2 holds, and the halo
  // they share comes from DRAM twice (ncu, config 5, nz = 512: 66.8 GB read per launch with one chunk, 54.3 GB with chunks of 64 for
  // 51.5 GB of fields; 24.56 -> 23.59 ms, interleaved A/B; 16 planes: 24.60, the two extra halo planes per chunk take over)
  const long long cap = (nz + 95) / 96;
  if (want < cap) want = cap;
  return (int)((nz + want - 1) / want);
}

#ifdef __CUDACC__
// Launch-bound grids (config 1: 32^3): one thread per point through the generic boundary accessors; a z-marching CTA has
// too few planes to amortise its pipeline fill there.  grid (ceil(nx/32), ceil(ny/8), nz), block (32, 8).
__global__ void __launch_bounds__(256) k_rhs_point(const __grid_constant__ Ctx c, const __grid_constant__ RhsArgs a, double* __restrict__ partial) {
  __shared__ double red[32];
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
  double s = 0.0;
  if (i < c.nx && j < c.ny) { const GhostAcc q{c, a, i, j, k}; s = rhs_core(c, a, q, i, j, k, zmet_at(c, k)) * c.dzf[k]; }
  if (partial) {
    const double t = block_sum(s, red);
    if (threadIdx.x == 0 && threadIdx.y == 0) partial[blockIdx.x + gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z)] = t;
  }
}

// grid (ceil(nx/RT_TX), ceil(ny/RT_TY), ceil(nz/kz)), block RT_THREADS, dynamic smem RT_SMEM_DOUBLES*8.
// partial[linear block id] = sum over the CTA's points of u* dzf[k] (or nullptr).
__global__ void __launch_bounds__(RT_THREADS, CALES_RT_MINB) k_rhs_tile(const __grid_constant__ Ctx c, const __grid_constant__ RhsArgs a, int kz,
                                                            double* __restrict__ partial, int pf) {
  extern __shared__ double rt_sm[];
  __shared__ double red[32];
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const int i0 = blockIdx.x * RT_TX, j0 = blockIdx.y * RT_TY, k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  // ---- this thread's halo-tile positions (the same for every plane and field)
  int goff[RT_EPT], soff[RT_EPT];      // in-plane global offset (>= 0: async copy; -1: unused; -2: y ghost, generic path)
#pragma unroll
  for (int e = 0; e < RT_EPT; ++e) {
    const int pos = tid + e * RT_THREADS;
    soff[e] = pos; goff[e] = -1;
    if (pos < RT_PLANE) {
      const int ry = pos / RT_TW, rx = pos - ry * RT_TW;
      int gi = i0 - 1 + rx, gj = j0 - 1 + ry;
      if (gi <= c.nx && gj <= c.ny) {
        gi = gi < 0 ? c.nx - 1 : (gi == c.nx ? 0 : gi);
        if (c.bc_y == BC_PER) { gj = gj < 0 ? c.ny - 1 : (gj == c.ny ? 0 : gj); goff[e] = gj * c.nx + gi; }
        else goff[e] = (gj < 0 || gj >= c.ny) ? -2 : gj * c.nx + gi;
      }
    }
  }
  const double* fld[RT_NF] = {a.u, a.v, a.w, a.nut, a.p};
  auto issue = [&](int kk) {
    double* slot = rt_sm + ((kk + 4) & 3) * (RT_NF * RT_PLANE);
    const bool zreg = c.bc_z == BC_PER || (kk >= 0 && kk < c.nz);
    const long long kw = (long long)(kk < 0 ? kk + c.nz : (kk >= c.nz ? kk - c.nz : kk)) * c.nxy;
#pragma unroll
    for (int e = 0; e < RT_EPT; ++e) {
      if (goff[e] == -1) continue;
      if (zreg && goff[e] >= 0) {
#pragma unroll
        for (int f = 0; f < RT_NF; ++f) if (f != 3 || c.sgs) cp_async8(slot + f * RT_PLANE + soff[e], fld[f] + kw + goff[e]);
      } else {
        const int ry = soff[e] / RT_TW, rx = soff[e] - ry * RT_TW;
#pragma unroll
        for (int f = 0; f < RT_NF; ++f) slot[f * RT_PLANE + soff[e]] = rt_elem(c, a, f, i0 - 1 + rx, j0 - 1 + ry, kk);
      }
    }
  };
  // the elements of plane kk this thread copied asynchronously (the synchronous ghost path has formed nu_t already)
  auto scale_nut = [&](int kk) {
    if (!(c.bc_z == BC_PER || (kk >= 0 && kk < c.nz))) return;
    double* pl = rt_sm + ((kk + 4) & 3) * (RT_NF * RT_PLANE) + 3 * RT_PLANE;
    const int kw = kk < 0 ? kk + c.nz : (kk >= c.nz ? kk - c.nz : kk);
#pragma unroll
    for (int e = 0; e < RT_EPT; ++e) {
      if (goff[e] < 0) continue;
      const int gj = c.dsm_plane ? 0 : (int)((unsigned)goff[e] / (unsigned)c.nx);
      pl[soff[e]] = dsm_nut_value(c, a.cs, pl[soff[e]], gj, kw);
    }
  };
  issue(k0 - 1); issue(k0);
  if (k0 + 1 <= k1) issue(k0 + 1);
  cp_async_commit();
  double acc = 0.0;
  ZMet zm = zmet_at(c, k0);
  for (int k = k0; k < k1; ++k) {
    // the metrics of the next plane are read one plane ahead; R^{k-1} is read inside rhs_core (early, pinned loads of it were
    // measured: no gain at 12 more live registers)
    const ZMet zn = zmet_at(c, k + 1 < k1 ? k + 1 : k);
    cp_async_wait_all();
    if (a.cs && c.sgs) {      // lazy dynamic model: this thread's |S| elements of the planes that have just landed become nu_t
#pragma unroll 1
      for (int kk = (k == k0) ? k0 - 1 : k + 1; kk <= k + 1; ++kk) scale_nut(kk);
    }
    __syncthreads();
    if (k + 2 <= k1) issue(k + 2);
    cp_async_commit();
    if (pf && a.be != 0.0 && k + 1 < k1) {     // R^{k-1} of the next plane: pull its sectors towards the SM while this plane is computed
#pragma unroll
      for (int r = 0; r < RT_RPT; ++r) {
        const int i = i0 + tx, j = j0 + ty * RT_RPT + r;
        if (i < c.nx && j < c.ny && (tx & 3) == 0) {
          const long long nn = idx3(c, i, j, k + 1);
          if (pf == 1) {
            asm volatile("prefetch.global.L1 [%0];" ::"l"(a.Ru0 + nn)); asm volatile("prefetch.global.L1 [%0];" ::"l"(a.Rv0 + nn));
            asm volatile("prefetch.global.L1 [%0];" ::"l"(a.Rw0 + nn));
          } else {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Ru0 + nn)); asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Rv0 + nn));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Rw0 + nn));
          }
        }
      }
    }
    TileAcc q;
    q.sl[0] = rt_sm + ((k + 3) & 3) * (RT_NF * RT_PLANE); q.sl[1] = rt_sm + (k & 3) * (RT_NF * RT_PLANE); q.sl[2] = rt_sm + ((k + 1) & 3) * (RT_NF * RT_PLANE);
    const double dz = zm.dzfk;
#pragma unroll
    for (int r = 0; r < RT_RPT; ++r) {
      const int ly = ty * RT_RPT + r, i = i0 + tx, j = j0 + ly;   // adjacent rows: their stencils share shared-memory loads
      if (i < c.nx && j < c.ny) {
        q.ctr = (ly + 1) * RT_TW + tx + 1;
        acc += rhs_core(c, a, q, i, j, k, zm) * dz;
      }
    }
    zm = zn;
  }
  if (partial) {
    const double t = block_sum(acc, red);
    if (tid == 0) partial[blockIdx.x + gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z)] = t;
  }
}

// ---- the same kernel with the halo planes moved by the TMA engine -----------------------------------------------------------
// ncu on k_rhs_tile (profiles/r1_ncu_full.md): 16 warps per SM, top stalls long scoreboard and wait, L1 pipe 59 % -- every
// plane costs each thread 12 eight-byte LDGSTS with their address arithmetic.  Here thread 0 issues ONE tiled tensor copy per
// field and plane (cp.async.bulk.tensor.3d, box 36 x 18 x 1 at (i0-2, j0-1, k), SASS UTMALDG), completing on an mbarrier two
// planes ahead of its use.  (The box starts one column left of the halo because the TMA engine wants the innermost
// coordinate on a 16-byte boundary -- an odd fp64 column is an illegal instruction, measured on B200.)  Elements outside the array arrive as zeros and are then overwritten with the boundary rule of
// Alg. 2 (periodic wrap, wall ghosts) by the threads that own them -- only tiles on the edge of the x-y plane have any.
// Planes beyond a z wall are filled by the generic path as before.  Field planes are padded to RT_FS doubles (128-byte slots).
enum { RTT_TW = RT_TX + 4, RTT_PLANE = RTT_TW * RT_TH, RT_FS = 656, RT_SMEM_TMA_BYTES = RT_NSLOT * RT_NF * RT_FS * 8 + 128,
       RTT_EPT = (RTT_PLANE + RT_THREADS - 1) / RT_THREADS };
struct RhsMaps { CUtensorMap m[RT_NF]; };      // u, v, w, nu_t, p as (nx, ny, nz) fp64 tensors, box (RTT_TW, RT_TH, 1); lives in device memory

__global__ void __launch_bounds__(RT_THREADS, 2) k_rhs_tile_tma(const __grid_constant__ Ctx c, const __grid_constant__ RhsArgs a,
                                                                const RhsMaps* __restrict__ maps, int kz, double* __restrict__ partial) {
  extern __shared__ double rt_sm_raw[];
  __shared__ double red[32];
  __shared__ unsigned long long full[RT_NSLOT];
  double* rt_sm = reinterpret_cast<double*>((reinterpret_cast<size_t>(rt_sm_raw) + 127) & ~(size_t)127);
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const int i0 = blockIdx.x * RT_TX, j0 = blockIdx.y * RT_TY, k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  // tiles on the edge of the x-y plane hold elements outside the array (zeros from the TMA, replaced in land())
  const bool edge = i0 == 0 || i0 + RT_TX >= c.nx || j0 == 0 || j0 + RT_TY >= c.ny;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < RT_NSLOT; ++s) mbar_init(&full[s], 1);
    mbar_fence_init();
  }
  __syncthreads();
  // plane kk (k0-1 <= kk <= k1) lives in slot q & 3, q = kk - (k0 - 1); its barrier phase is (q >> 2) & 1
  auto issue = [&](int kk) {
    const int q = kk - (k0 - 1);
    double* slot = rt_sm + (q & 3) * (RT_NF * RT_FS);
    const bool zreg = c.bc_z == BC_PER || (kk >= 0 && kk < c.nz);
    if (zreg) {
      if (tid == 0) {
        const int kw = kk < 0 ? kk + c.nz : (kk >= c.nz ? kk - c.nz : kk);
        const int nf = c.sgs ? RT_NF : RT_NF - 1;
        mbar_expect_tx(&full[q & 3], (unsigned)(nf * RTT_PLANE * sizeof(double)));
#pragma unroll
        for (int f = 0; f < RT_NF; ++f) if (f != 3 || c.sgs) tma_load_3d(slot + f * RT_FS, &maps->m[f], i0 - 2, j0 - 1, kw, &full[q & 3]);
      }
    } else {
      for (int pos = tid; pos < RTT_PLANE; pos += RT_THREADS) {
        const int ry = pos / RTT_TW, rx = pos - ry * RTT_TW, gi = i0 - 2 + rx, gj = j0 - 1 + ry;
        if (rx < 1 || gi > c.nx || gj > c.ny) continue;
        for (int f = 0; f < RT_NF; ++f) slot[f * RT_FS + pos] = rt_elem(c, a, f, gi, gj, kk);
      }
      if (tid == 0) mbar_arrive(&full[q & 3]);       // keeps the phase count of the slot in step
    }
  };
  // wait for plane kk and replace the out-of-array zeros (x / y ghosts) of a TMA plane
  auto land = [&](int kk) {
    const int q = kk - (k0 - 1);
    mbar_wait(&full[q & 3], (q >> 2) & 1);
    const bool zreg = c.bc_z == BC_PER || (kk >= 0 && kk < c.nz);
    if (!zreg || !edge) return;
    double* slot = rt_sm + (q & 3) * (RT_NF * RT_FS);
    for (int pos = tid; pos < RTT_PLANE; pos += RT_THREADS) {
      const int ry = pos / RTT_TW, rx = pos - ry * RTT_TW, gi = i0 - 2 + rx, gj = j0 - 1 + ry;
      if (rx < 1 || gi > c.nx || gj > c.ny || (gi >= 0 && gi < c.nx && gj >= 0 && gj < c.ny)) continue;
      for (int f = 0; f < RT_NF; ++f) slot[f * RT_FS + pos] = rt_elem(c, a, f, gi, gj, kk);
    }
  };
  issue(k0 - 1); issue(k0);
  if (k0 + 1 <= k1) issue(k0 + 1);
  land(k0 - 1); land(k0);
  double acc = 0.0;
  for (int k = k0; k < k1; ++k) {
    land(k + 1);
    __syncthreads();
    if (k + 2 <= k1) issue(k + 2);
    if (a.be != 0.0 && k + 1 < k1) {     // R^{k-1} of the next plane: pull the lines towards L1 while this plane is computed
#pragma unroll
      for (int r = 0; r < RT_RPT; ++r) {
        const int i = i0 + tx, j = j0 + ty * RT_RPT + r;
        if (i < c.nx && j < c.ny && (tx & 3) == 0) {
          const long long nn = idx3(c, i, j, k + 1);
          asm volatile("prefetch.global.L1 [%0];" ::"l"(a.Ru0 + nn));
          asm volatile("prefetch.global.L1 [%0];" ::"l"(a.Rv0 + nn));
          asm volatile("prefetch.global.L1 [%0];" ::"l"(a.Rw0 + nn));
        }
      }
    }
    const int qc = k - (k0 - 1);
    TileAccT<RT_FS, RTT_TW> q;
    q.sl[0] = rt_sm + ((qc - 1) & 3) * (RT_NF * RT_FS); q.sl[1] = rt_sm + (qc & 3) * (RT_NF * RT_FS); q.sl[2] = rt_sm + ((qc + 1) & 3) * (RT_NF * RT_FS);
    const ZMet zm = zmet_at(c, k);
    const double dz = zm.dzfk;
#pragma unroll
    for (int r = 0; r < RT_RPT; ++r) {
      const int ly = ty * RT_RPT + r, i = i0 + tx, j = j0 + ly;
      if (i < c.nx && j < c.ny) {
        q.ctr = (ly + 1) * RTT_TW + tx + 2;
        acc += rhs_core(c, a, q, i, j, k, zm) * dz;
      }
    }
  }
  if (partial) {
    const double t = block_sum(acc, red);
    if (tid == 0) partial[blockIdx.x + gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z)] = t;
  }
}
#endif

}  // namespace cales
