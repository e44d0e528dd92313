// cales_dsm3.cuh -- dynamic Smagorinsky, pass 1, with the 3-D box test filter.
// The filter is separable (1/4,1/2,1/4) in x, y and z ("assumes uniform grid spacing").  In the first
// off-wall layer of a wall-bounded direction that direction keeps the identity (the paper's "linear extrapolation to the
// ghost points, followed by the 3D filter") and the filter-width ratio is the cube root of the volume ratio of the
// directions actually filtered: 8^(1/3) = 2 inside, 4^(1/3) in the first layer, 2^(1/3) in a duct corner.
//
// One CTA = one D3_TX x D3_TY tile of one k-plane.  Shared memory holds
//   raw : u, v, w on planes k-2 .. k+2 over the tile + halo 2 (ghosts by velg, GH_STRAIN mode),
//   flt : the face-wise test-filtered velocity on planes k-1, k, k+1 over the tile + halo 1 (Eq. 9 takes its strain);
//         its ghosts are the boundary condition applied to the FILTERED field (S24), z before y (S25),
//   mid : centre velocities, |S| S_ij and |S| on planes k-1, k, k+1 over the tile + halo 1 (the filter reads 3x3x3).
// Eq. 9 is evaluated literally (strain of the filtered velocity), so the kernel is valid next to walls in y and z.
#pragma once
#include "cales_common.cuh"
#include "cales_closures.cuh"
#include "cales_dsm_col.cuh"

namespace cales {

enum { D3_TX = 32, D3_TY = 8, D3_RX = D3_TX + 4, D3_RY = D3_TY + 4, D3_MX = D3_TX + 2, D3_MY = D3_TY + 2 };
enum { D3_RAW = 15 * D3_RX * D3_RY, D3_FLT = 9 * D3_MX * D3_MY, D3_MID = 30 * D3_MX * D3_MY,
       D3_SMEM_DOUBLES = D3_RAW + D3_FLT + D3_MID };

CALES_HD int d3_raw_off(int comp, int pl /* 0..4 <-> plane k-2+pl */, int ry, int rx) { return ((comp * 5 + pl) * D3_RY + ry) * D3_RX + rx; }
CALES_HD int d3_flt_off(int comp, int pl /* 0..2 <-> plane k-1+pl */, int my, int mx) { return ((comp * 3 + pl) * D3_MY + my) * D3_MX + mx; }
CALES_HD int d3_mid_off(int q, int pl /* 0..2 <-> plane k-1+pl */, int my, int mx) { return ((q * 3 + pl) * D3_MY + my) * D3_MX + mx; }

// z weights of the test filter for plane gk.  kind 0: data centred in z (u, v, centre quantities); 1: w faces.
CALES_HD void d3_wz(const Ctx& c, int gk, int kind, double* wz) {
  wz[0] = 0.25; wz[1] = 0.5; wz[2] = 0.25;
  if (c.bc_z == BC_WALL) {
    if (kind == 0) { if (gk <= 0 || gk >= c.nz - 1) { wz[0] = 0.0; wz[1] = 1.0; wz[2] = 0.0; } }
    else { if (gk < 0 || gk >= c.nz - 1) { wz[0] = 0.0; wz[1] = 0.0; wz[2] = 0.0; } }
  }
}

// phase 1: the raw tile, 3 components x 5 planes
CALES_HD void d3_load(int tid, int nth, const Ctx& c, const double* u, const double* v, const double* w, int i0, int j0, int k, double* raw) {
  const int per = D3_RX * D3_RY;
  for (int idx = tid; idx < 15 * per; idx += nth) {
    const int cp = idx / per, r = idx % per;
    const int comp = cp / 5, pl = cp % 5, ry = r / D3_RX, rx = r % D3_RX;
    const int gi = i0 - 2 + rx, gj = j0 - 2 + ry;
    int gk = k - 2 + pl;
    double val = 0.0;
    bool ok = gi <= c.nx + 1 && gj <= c.ny + 1;
    if (c.bc_z == BC_PER) gk = wrapi(gk, c.nz);
    else if (gk < -1 || gk > c.nz) ok = false;            // beyond the ghost layer: never read with a non-zero weight
    if (ok) {
      if (comp == 0) val = velg<0>(c, u, gi, gj, gk, GH_STRAIN);
      else if (comp == 1) val = velg<1>(c, v, gi, gj, gk, GH_STRAIN);
      else val = velg<2>(c, w, gi, gj, gk, GH_STRAIN);
    }
    raw[idx] = val;
  }
}

// phase 2: filtered face velocities (3 components x 3 planes) and the centre quantities on the mid region
CALES_HD void d3_mid(int tid, int nth, const Ctx& c, int i0, int j0, int k, const double* raw, double* flt, double* mid) {
  const int per = D3_MX * D3_MY;
  for (int idx = tid; idx < 9 * per; idx += nth) {
    const int cp = idx / per, r = idx % per;
    const int comp = cp / 3, pl = cp % 3, my = r / D3_MX, mx = r % D3_MX;
    const int gj = j0 - 1 + my, gk = k - 1 + pl;
    // 3-D filtered face value on raw plane index p (global plane k-2+p, interior or periodic), mid row m
    auto f0 = [&](int p, int m) {
      double wz[3]; d3_wz(c, k - 2 + p, comp == 2 ? 1 : 0, wz);
      double wy[3]; dsm_wy(c, j0 - 1 + m, comp == 1 ? 1 : 0, wy);
      double s = 0.0;
      for (int d = 0; d < 3; ++d) {
        if (wz[d] == 0.0) continue;
        double t = 0.0;
        for (int b = 0; b < 3; ++b) {
          const double* row = raw + d3_raw_off(comp, p - 1 + d, m + b, mx);
          t += wy[b] * (0.25 * row[0] + 0.5 * row[1] + 0.25 * row[2]);
        }
        s += wz[d] * t;
      }
      return s;
    };
    // plane gk including the z ghosts of the filtered field: w = 0 on and beyond the wall faces; u, v no-slip mirror
    // or, at a wall-model wall, the one-sided extrapolation of the first two filtered layers (as velg_z, GH_STRAIN)
    auto fz = [&](int m) {
      if (c.bc_z == BC_PER || (gk >= 0 && gk < c.nz)) return f0(pl + 1, m);
      if (comp == 2) return 0.0;
      const bool bottom = gk < 0;
      const double q0 = f0(bottom ? pl + 2 : pl, m);
      if (!c.wall_model) return -q0;
      const double q1 = f0(bottom ? pl + 3 : pl - 1, m);
      const double rr = bottom ? c.dzc[-1] / c.dzc[0] : c.dzc[c.nz - 1] / c.dzc[c.nz - 2];
      return q0 + (q0 - q1) * rr;
    };
    // y ghost rows of the filtered u, w at a wall-model y wall: the same rule in y (after z)
    if (c.bc_y == BC_WALL && c.wall_model_y && comp != 1 && (gj < 0 || gj >= c.ny))
      flt[idx] = gj < 0 ? 2.0 * fz(my + 1) - fz(my + 2) : 2.0 * fz(my - 1) - fz(my - 2);
    else flt[idx] = fz(my);
  }
  double wzc[3]; d3_wz(c, k, 0, wzc);
  const double rdx = c.rdx, rdy = c.rdy;
  for (int idx = tid; idx < 3 * per; idx += nth) {
    const int pl = idx / per, r = idx % per, my = r / D3_MX, mx = r % D3_MX;
    if (wzc[pl] == 0.0) {                                  // plane outside the filter stencil (first off-wall layer)
      for (int q = 0; q < 10; ++q) mid[d3_mid_off(q, pl, my, mx)] = 0.0;
      continue;
    }
    const int kk = c.bc_z == BC_PER ? wrapi(k - 1 + pl, c.nz) : k - 1 + pl;
    auto U = [&](int a, int b, int d) { return raw[d3_raw_off(0, 1 + pl + d, my + 1 + b, mx + 1 + a)]; };
    auto V = [&](int a, int b, int d) { return raw[d3_raw_off(1, 1 + pl + d, my + 1 + b, mx + 1 + a)]; };
    auto W = [&](int a, int b, int d) { return raw[d3_raw_off(2, 1 + pl + d, my + 1 + b, mx + 1 + a)]; };
    double S[6];
    const double smag = strain_at(U, V, W, rdx, rdy, c.rdzf[kk], c.rdzc[kk], c.rdzc[kk - 1], S);
    mid[d3_mid_off(0, pl, my, mx)] = 0.5 * (U(-1, 0, 0) + U(0, 0, 0));
    mid[d3_mid_off(1, pl, my, mx)] = 0.5 * (V(0, -1, 0) + V(0, 0, 0));
    mid[d3_mid_off(2, pl, my, mx)] = 0.5 * (W(0, 0, -1) + W(0, 0, 0));
    for (int q = 0; q < 6; ++q) mid[d3_mid_off(3 + q, pl, my, mx)] = smag * S[q];
    mid[d3_mid_off(9, pl, my, mx)] = smag;
  }
}

// phase 3: one output point (tx, ty); L:M and M:M through lm, mm and |S| through smag_out
CALES_HD void d3_point(const Ctx& c, int j0, int k, int tx, int ty, const double* flt, const double* mid, double* lm, double* mm, double* smag_out) {
  const int gj = j0 + ty;
  const int mx = tx + 1, my = ty + 1;
  double wy[3]; dsm_wy(c, gj, 0, wy);
  double wz[3]; d3_wz(c, k, 0, wz);
  const double wx[3] = {0.25, 0.5, 0.25};
  double Fv[3] = {0, 0, 0}, Fp[6] = {0, 0, 0, 0, 0, 0}, Fs[6] = {0, 0, 0, 0, 0, 0};
  const int st = 3 * D3_MX * D3_MY;                        // stride between quantities
  for (int d = 0; d < 3; ++d) {
    if (wz[d] == 0.0) continue;
#pragma unroll
    for (int b = 0; b < 3; ++b) {
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        const double wgt = wz[d] * (wy[b] * wx[a]);
        const int o = d3_mid_off(0, d, my - 1 + b, mx - 1 + a);
        const double uc = mid[o], vc = mid[o + st], wc = mid[o + 2 * st];
        Fv[0] += wgt * uc; Fv[1] += wgt * vc; Fv[2] += wgt * wc;
        Fp[0] += wgt * (uc * uc); Fp[1] += wgt * (vc * vc); Fp[2] += wgt * (wc * wc);
        Fp[3] += wgt * (uc * vc); Fp[4] += wgt * (uc * wc); Fp[5] += wgt * (vc * wc);
#pragma unroll
        for (int q = 0; q < 6; ++q) Fs[q] += wgt * mid[o + (3 + q) * st];
      }
    }
  }
  double L[6];
  L[0] = Fp[0] - Fv[0] * Fv[0]; L[1] = Fp[1] - Fv[1] * Fv[1]; L[2] = Fp[2] - Fv[2] * Fv[2];
  L[3] = Fp[3] - Fv[0] * Fv[1]; L[4] = Fp[4] - Fv[0] * Fv[2]; L[5] = Fp[5] - Fv[1] * Fv[2];
  // Eq. 9: strain of the test-filtered velocity
  auto U = [&](int a, int b, int d) { return flt[d3_flt_off(0, 1 + d, my + b, mx + a)]; };
  auto V = [&](int a, int b, int d) { return flt[d3_flt_off(1, 1 + d, my + b, mx + a)]; };
  auto W = [&](int a, int b, int d) { return flt[d3_flt_off(2, 1 + d, my + b, mx + a)]; };
  double St[6];
  const double stmag = strain_at(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], St);
  const double d2 = c.delta[k] * c.delta[k];
  int nf = 1;                                               // directions filtered at this point
  if (!(c.bc_y == BC_WALL && (gj == 0 || gj == c.ny - 1))) ++nf;
  if (!(c.bc_z == BC_WALL && (k == 0 || k == c.nz - 1))) ++nf;
  const double al = nf == 2 ? c.alpha : (nf == 1 ? sqrt(c.alpha) : c.alpha * sqrt(c.alpha));
  double ll = 0.0, m2 = 0.0;
#pragma unroll
  for (int q = 0; q < 6; ++q) {
    const double M = 2.0 * d2 * (Fs[q] - al * al * stmag * St[q]);
    const double f = q < 3 ? 1.0 : 2.0;
    ll += f * L[q] * M; m2 += f * M * M;
  }
  *lm = ll; *mm = m2; *smag_out = mid[d3_mid_off(9, 1, my, mx)];
}

// ------------------------------------------------------------------------------------------------------------
// Column-marching form (the production path where the 27 filter weights are uniform and the z grid is uniform: there F
// commutes with the strain operator, S~_ij = F(S_ij), as in k_dsm_col_sm).  Same march as the x-y kernel, with the z part
// of the separable filter applied first, point-wise: every thread evaluates the base values of its column on planes
// k-1, k, k+1, forms  zq = (q(k-1) + 2 q(k) + q(k+1)) / 4  of the 21 quantities and publishes zq; the x-filter reads the
// neighbours' zq, the y-filter is the two-row window in shared memory.  Planes / rows next to a wall (two of each: the
// first-layer rule changes the weights of the layer itself and of its neighbour's stencil) go to k_dsm3_pass1.
// ------------------------------------------------------------------------------------------------------------
struct D3Split { int col, klo, khi, jlo, jhi; };    // col = 0: the tile kernel everywhere
CALES_HD D3Split d3_split(const Ctx& c, int z_uniform) {
  D3Split s; s.col = 0; s.klo = 0; s.khi = c.nz; s.jlo = 0; s.jhi = c.ny;
  if (!z_uniform) return s;
  if (c.bc_z == BC_WALL) { s.klo = 2; s.khi = c.nz - 2; }
  if (c.bc_y == BC_WALL) { s.jlo = 2; s.jhi = c.ny - 2; }
  if (s.khi - s.klo < 2 || (c.bc_y == BC_WALL && c.ny < 2 * D3_TY)) return s;
  s.col = 1;
  return s;
}

// phase A: zq of (column t, row gj) into shbuf[.][t] and the registers zq; |S| of plane k through smag_c
CALES_HD void d3c_phaseA(const Ctx& c, const double* u, const double* v, const double* w, int txb, int t, int i0, int gj, int k,
                         double* shbuf /* [DSMC_NQ][txb] */, double* zq, double* smag_c) {
  const int gi = ((i0 - 1 + t) % c.nx + c.nx) % c.nx;
#pragma unroll
  for (int m = 0; m < DSMC_NQ; ++m) zq[m] = 0.0;
  // planes k-2 .. k+2 without wrap or ghost (and a row whose y neighbours are plain): one set of in-plane neighbour offsets
  // and plane offsets that are multiples of nxy, so the loads shared by the three strain stencils are issued once
  const bool plain = k >= 2 && k <= c.nz - 3 && (c.bc_y == BC_PER || (gj >= 1 && gj <= c.ny - 2));
  auto add = [&](const double* b, int d) {
    double q[DSMC_NQ];
    dsmc_q(b, q);
    const double wgt = d == 0 ? 0.5 : 0.25;
#pragma unroll
    for (int m = 0; m < DSMC_NQ; ++m) zq[m] += wgt * q[m];
    if (d == 0) *smag_c = b[9];
  };
  if (plain) {
    const long long n = idx3(c, gi, gj, k);
    const Nbr o = neighbours(c, gi, gj, k);
#pragma unroll
    for (int d = -1; d <= 1; ++d) {
      auto at = [&](const double* __restrict__ f, int a, int bb, int dd) {
        return f[n + (long long)(d + dd) * c.nxy + ((a < 0 ? o.im : (a > 0 ? o.ip : 0)) + (bb < 0 ? o.jm : (bb > 0 ? o.jp : 0)))];
      };
      auto U = [&](int a, int bb, int dd) { return at(u, a, bb, dd); };
      auto V = [&](int a, int bb, int dd) { return at(v, a, bb, dd); };
      auto W = [&](int a, int bb, int dd) { return at(w, a, bb, dd); };
      double b[DSMC_NB], S[6];
      b[9] = strain_at(U, V, W, c.rdx, c.rdy, c.rdzf[k + d], c.rdzc[k + d], c.rdzc[k + d - 1], S);
      b[0] = 0.5 * (U(-1, 0, 0) + U(0, 0, 0)); b[1] = 0.5 * (V(0, -1, 0) + V(0, 0, 0)); b[2] = 0.5 * (W(0, 0, -1) + W(0, 0, 0));
#pragma unroll
      for (int m = 0; m < 6; ++m) b[3 + m] = S[m];
      add(b, d);
    }
  } else {
    for (int d = -1; d <= 1; ++d) {
      double b[DSMC_NB];
      dsmc_base(c, u, v, w, gi, gj, c.bc_z == BC_PER ? wrapi(k + d, c.nz) : k + d, b);
      add(b, d);
    }
  }
#pragma unroll
  for (int m = 0; m < DSMC_NQ; ++m) shbuf[m * txb + t] = zq[m];
}

// phase B (threads 1..txb-2): x-filter from the neighbours' zq, y-filter over the shared-memory window (as dsmc_phaseB_sm)
CALES_HD bool d3c_phaseB(const Ctx& c, int txb, int t, int r, int k, const double* shbuf, const double* zq, double* ring,
                         double* smag_prev, double smag_c, double* lm, double* mm, double* smag) {
  double* r1 = ring + ((r + 1) & 1) * (DSMC_NQ * txb) + t;     // xq(r-1)
  double* r2 = ring + (r & 1) * (DSMC_NQ * txb) + t;           // xq(r-2); overwritten with xq(r)
  double Fq[DSMC_NQ];
#pragma unroll
  for (int m = 0; m < DSMC_NQ; ++m) {
    const double xq = 0.25 * (shbuf[m * txb + t - 1] + shbuf[m * txb + t + 1]) + 0.5 * zq[m];
    Fq[m] = 0.25 * (r2[m * txb] + xq) + 0.5 * r1[m * txb];
    r2[m * txb] = xq;
  }
  bool done = false;
  if (r >= 2) {
    const double d2 = c.delta[k] * c.delta[k];
    dsmc_contract(Fq, d2, c.alpha * sqrt(c.alpha), lm, mm);      // three filtered directions: alpha = 8^(1/3)
    *smag = *smag_prev;
    done = true;
  }
  *smag_prev = smag_c;
  return done;
}

// ---- the column march in the register-window form of cales_dsm_col.cuh ------------------------------------------------------
// One row for an output column: zq = the thread's own z-filtered 21 quantities, UNNORMALISED (zq' = q(k-1) + q(k+1) + 2 q(k) = 4 Fz q);
// shbuf = the row's zq' of all columns ([DSMC_NQ][txb]).  x: xq' = l + r + 2 c = 16 Fx Fz q; y over the register window:
// F' = w2 + xq' + 2 w1 = 64 F q.  With L' = 64 F'(u_i u_j) - F'(u_i) F'(u_j) = 4096 L and M' = 64 F'(|S| S_ij) - a2 |S~|' S~'_ij =
// 4096 M / (2 Delta^2) the powers of two go into the constants of the contraction.  a2 = alpha^2 of three filtered directions.
template <int PAR>
CALES_HD void dsm3r_row(const double* shbuf, int txb, int t, const double* zq, DsmrWin& w, bool emit, double d2, double a2, double* lm, double* mm) {
  const double* sl = shbuf + t - 1;
  const double* sr = shbuf + t + 1;
  double* w1 = w.q[1 - PAR];     // row r-1
  double* w2 = w.q[PAR];         // row r-2, then row r
  double F[DSMC_NQ];
#pragma unroll
  for (int m = 0; m < DSMC_NQ; ++m) {
    const double x = (sl[m * txb] + sr[m * txb]) + 2.0 * zq[m];
    const double ts = w2[m] + 2.0 * w1[m]; w2[m] = x; F[m] = ts + x;      // old window value consumed first (no moves)
  }
  if (!emit) return;
  const double* St = F + 15;
  const double stmag = sqrt(2.0 * (St[0] * St[0] + St[1] * St[1] + St[2] * St[2]) + 4.0 * (St[3] * St[3] + St[4] * St[4] + St[5] * St[5]));
  const double a2s = a2 * stmag;
  double Mp[6];
#pragma unroll
  for (int m = 0; m < 6; ++m) Mp[m] = 64.0 * F[9 + m] - a2s * St[m];
  const double md = Mp[0] * Mp[0] + Mp[1] * Mp[1] + Mp[2] * Mp[2], mo = Mp[3] * Mp[3] + Mp[4] * Mp[4] + Mp[5] * Mp[5];
  const double ld = (64.0 * F[3] - F[0] * F[0]) * Mp[0] + (64.0 * F[4] - F[1] * F[1]) * Mp[1] + (64.0 * F[5] - F[2] * F[2]) * Mp[2];
  const double lo = (64.0 * F[6] - F[0] * F[1]) * Mp[3] + (64.0 * F[7] - F[0] * F[2]) * Mp[4] + (64.0 * F[8] - F[1] * F[2]) * Mp[5];
  const double sc = 2.0 * d2 * (1.0 / 4096.0);
  *lm = (ld + 2.0 * lo) * (sc * (1.0 / 4096.0));
  *mm = (md + 2.0 * mo) * (sc * sc);
}

// zq' of one column from accessors to the raw velocities around (column, row) on planes k-2 .. k+2: U(a, b, d) = u at column offset a,
// row offset b, plane k + d (the same for V, W).  Returns |S| of plane k.
template <class GU, class GV, class GW>
CALES_HD double dsm3r_zq(GU U, GV V, GW W, double rdx, double rdy, const double* rdzf3 /* k-1, k, k+1 */, const double* rdzc4 /* k-2 .. k+1 */, double* zq) {
  double smag_c = 0.0;
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    const int d = s == 0 ? -1 : (s == 1 ? 1 : 0);      // the two outer planes first, the centre plane (weight 2) last
    auto Ud = [&](int a, int b, int dd) { return U(a, b, d + dd); };
    auto Vd = [&](int a, int b, int dd) { return V(a, b, d + dd); };
    auto Wd = [&](int a, int b, int dd) { return W(a, b, d + dd); };
    double b[DSMC_NB], q[DSMC_NQ];
    dsmr_base_from(Ud, Vd, Wd, rdx, rdy, rdzf3[1 + d], rdzc4[2 + d], rdzc4[1 + d], b);
    dsmc_q(b, q);
#pragma unroll
    for (int m = 0; m < DSMC_NQ; ++m) zq[m] = s == 0 ? q[m] : (s == 1 ? zq[m] + q[m] : zq[m] + 2.0 * q[m]);
    if (d == 0) smag_c = b[9];
  }
  return smag_c;
}

#ifdef __CUDACC__
// grid (ceil(nx/D3_TX), row tiles, planes), block (D3_TX, D3_TY), dynamic smem D3_SMEM_DOUBLES*8.
// planes: k = blockIdx.z (+ kskip when blockIdx.z >= ksplit); rows: j0 = blockIdx.y * jstride, of which only the rows
// j < row_hi || j >= row_lo2 are written (the others belong to k_dsm3_col).
// part: [k][j][pslots][2]; this kernel fills slot blockIdx.x of its rows (the other slots stay 0).
__global__ void __launch_bounds__(D3_TX * D3_TY) k_dsm3_pass1(const __grid_constant__ Ctx c, const double* __restrict__ u, const double* __restrict__ v,
                                                               const double* __restrict__ w, int ksplit, int kskip, int jstride, int row_hi, int row_lo2,
                                                               int pslots, double* __restrict__ smag, double* __restrict__ part) {
  extern __shared__ double d3_sm[];
  double* raw = d3_sm; double* flt = raw + D3_RAW; double* mid = flt + D3_FLT;
  const int tid = threadIdx.x + D3_TX * threadIdx.y, nth = D3_TX * D3_TY;
  const int i0 = blockIdx.x * D3_TX, j0 = blockIdx.y * jstride, k = (int)blockIdx.z + ((int)blockIdx.z >= ksplit ? kskip : 0);
  d3_load(tid, nth, c, u, v, w, i0, j0, k, raw);
  __syncthreads();
  d3_mid(tid, nth, c, i0, j0, k, raw, flt, mid);
  __syncthreads();
  const int i = i0 + threadIdx.x, j = j0 + threadIdx.y;
  double lm = 0.0, mm = 0.0;
  const bool mine = j < c.ny && (j < row_hi || j >= row_lo2);      // warp-uniform (one row per warp)
  if (i < c.nx && mine) {
    double sm;
    d3_point(c, j0, k, threadIdx.x, threadIdx.y, flt, mid, &lm, &mm, &sm);
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
// grid (ceil(nx/(TXB-2)), ceil((jhi-jlo)/DSMC_LY), khi-klo), block TXB; output rows [jlo, jhi) of planes [klo, khi).
// part: slots blockIdx.x * (TXB/32) + warp.
template <int TXB, int MINB, int NBUF>
__global__ void __launch_bounds__(TXB, MINB) k_dsm3_col(const __grid_constant__ Ctx c, const double* __restrict__ u, const double* __restrict__ v,
                                                        const double* __restrict__ w, int klo, int jlo, int jhi, int pslots, double* __restrict__ smag,
                                                        double* __restrict__ part) {
  __shared__ double sh[NBUF][DSMC_NQ * TXB];
  __shared__ double ring[2 * DSMC_NQ * TXB];
  const int t = threadIdx.x, k = klo + blockIdx.z;
  const int i0 = blockIdx.x * (TXB - 2);
  const int j0 = jlo + blockIdx.y * DSMC_LY;
  const int jend = min(j0 + DSMC_LY, jhi);
  const int nrows = jend - j0 + 2;
  const int gi = i0 - 1 + t;
  const bool outcol = t >= 1 && t <= TXB - 2 && gi < c.nx;
#pragma unroll
  for (int m = 0; m < 2 * DSMC_NQ; ++m) ring[m * TXB + t] = 0.0;
  double smag_prev = 0.0;
  for (int r = 0; r < nrows; ++r) {
    int gj = j0 - 1 + r;
    gj = gj < 0 ? gj + c.ny : (gj >= c.ny ? gj - c.ny : gj);
    double zq[DSMC_NQ], smag_c;
    if (NBUF == 1) __syncthreads();     // the previous row's neighbours have read the buffer
    d3c_phaseA(c, u, v, w, TXB, t, i0, gj, k, sh[r & (NBUF - 1)], zq, &smag_c);
    __syncthreads();
    double lm = 0.0, mm = 0.0, sm = 0.0;
    bool done = false;
    if (t >= 1 && t <= TXB - 2) done = d3c_phaseB(c, TXB, t, r, k, sh[r & (NBUF - 1)], zq, ring, &smag_prev, smag_c, &lm, &mm, &sm);
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

// ---- the same march with the raw rows staged by the TMA engine and the y-window in registers (as k_dsm_col_tma) -----------
// 14 lines per raw row: u on planes k-2 .. k+2, v on k-2 .. k+2, w on k-2 .. k+1, columns i0-2 .. i0+TXB-1, in a ring of DSMT_NS rows
// filled by cp.async.bulk copies (seven producer lanes in each of the two warps) that complete on mbarriers two rows ahead.  Every
// thread evaluates the strain rate of its column on the three planes from shared memory (immediate offsets), forms the unnormalised
// zq', publishes it, and dsm3r_row runs the x filter, the register y-window and the contraction.
// grid (ceil(nx/(TXB-2)), khi-klo, ceil((jhi-jlo)/ly)), block TXB = 64.  Needs nx >= TXB + 2, 16-byte aligned fields, planes klo-2 ..
// khi+1 and rows jlo-2 .. jhi+1 plain (in the array or periodic wrap): the region d3_split gives the column march.
enum { DSM3T_NL = 14, DSM3T_RAW_BYTES = DSMT_NS * DSM3T_NL * 66 * 8 };      // for TXB = 64
template <int TXB, int MINB>
__global__ void __launch_bounds__(TXB, MINB) k_dsm3_col_tma(const __grid_constant__ Ctx c, const double* __restrict__ u, const double* __restrict__ v,
                                                            const double* __restrict__ w, int klo, int jlo, int jhi, int ly, int pslots,
                                                            double* __restrict__ smag, double* __restrict__ part) {
  constexpr int LW = TXB + 2;
  constexpr int STAGE = DSM3T_NL * LW;
  extern __shared__ __align__(128) double d3t_raw[];      // DSMT_NS * STAGE doubles (dynamic: with `sh` the CTA is past 48 KB)
  double* raw = d3t_raw;
  __shared__ double sh[2][DSMC_NQ * TXB];
  __shared__ unsigned long long full[DSMT_NS];
  const int t = threadIdx.x, k = klo + blockIdx.y;
  const int i0 = blockIdx.x * (TXB - 2);
  const int j0 = jlo + blockIdx.z * ly;
  const int jend = min(j0 + ly, jhi);
  const int nrows = jend - j0 + 2;             // base rows j0-1 .. jend; raw rows j0-2 .. jend+1
  const int nraw = nrows + 2;
  const int gi = i0 - 1 + t;
  const bool inner = t >= 1 && t <= TXB - 2;
  const bool outcol = inner && gi < c.nx;
  const double d2 = c.delta[k] * c.delta[k], a2 = c.alpha * c.alpha * c.alpha;      // alpha = 8^(1/3) x the 2-D ratio^(1/2): (alpha^(3/2))^2
  const double rdx = c.rdx, rdy = c.rdy;
  auto wz = [&](int kk) { return kk < 0 ? kk + c.nz : (kk >= c.nz ? kk - c.nz : kk); };
  const double rdzf3[3] = {c.rdzf[wz(k - 1)], c.rdzf[k], c.rdzf[wz(k + 1)]};
  const double rdzc4[4] = {c.rdzc[wz(k - 2)], c.rdzc[wz(k - 1)], c.rdzc[k], c.rdzc[wz(k + 1)]};
  // ---- producer state (lanes 0..6 of warps 0 and 1: seven lines each)
  const double* src = nullptr; int gj_next = 0, segA = 0;
  const bool producer = (t & 31) < DSM3T_NL / 2 && t < 64;
  const int line = (t & 31) + (t >> 5) * (DSM3T_NL / 2);
  if (producer) {
    const int l = line;
    const double* f = l < 5 ? u : (l < 10 ? v : w);
    const int kk = wz(k - 2 + (l < 5 ? l : (l < 10 ? l - 5 : l - 10)));
    gj_next = j0 - 2; gj_next = gj_next < 0 ? gj_next + c.ny : gj_next;
    src = f + ((long long)kk * c.ny + gj_next) * c.nx;
    const int cw0 = (((i0 - 2) % c.nx) + c.nx) % c.nx;
    segA = min(LW, c.nx - cw0);
    src += cw0;
  }
  auto issue = [&](int slot) {
    unsigned long long* bar = &full[slot];
    if (t == 0) mbar_expect_tx(bar, STAGE * (unsigned)sizeof(double));
    double* dst = raw + slot * STAGE + line * LW;
    bulk_g2s(dst, src, (unsigned)segA * 8u, bar);
    if (segA < LW) bulk_g2s(dst + segA, src - (c.nx - segA), (unsigned)(LW - segA) * 8u, bar);
    ++gj_next;
    if (gj_next == c.ny) { gj_next = 0; src -= (long long)(c.ny - 1) * c.nx; } else src += c.nx;
  };
  if (t == 0) {
#pragma unroll
    for (int s = 0; s < DSMT_NS; ++s) mbar_init(&full[s], 1);
    mbar_fence_init();
  }
  __syncthreads();
  if (producer) {
#pragma unroll
    for (int s = 0; s < DSMT_NS; ++s) if (s < nraw) issue(s);
  }
  DsmrWin win;
  dsmr_win_init(win);
  double* sm_out = smag + idx3(c, gi < c.nx ? gi : 0, j0, k);           // |S| of output row j0, bumped by nx per emitted row
  long long pslot = ((long long)k * c.ny + j0) * pslots + blockIdx.x * (TXB / 32) + (t >> 5);
  const double* Rt = raw + t + 1;
  auto row = [&](auto ph, int r) {
    constexpr int PH = decltype(ph)::value;    // r & 3
    constexpr int PAR = PH & 1, S0 = PH, S1 = (PH + 1) & 3, S2 = (PH + 2) & 3;
    if (r == 0) { mbar_wait(&full[0], 0); mbar_wait(&full[1], 0); }
    mbar_wait(&full[S2], ((r + 2) >> 2) & 1);
    double zq[DSMC_NQ], smag_c;
    {
      const double* R0 = Rt + S0 * STAGE;      // raw row below the base row
      const double* R1 = Rt + S1 * STAGE;      // the base row
      const double* R2 = Rt + S2 * STAGE;      // the row above
      auto U = [&](int a, int bb, int d) { return (bb < 0 ? R0 : (bb > 0 ? R2 : R1))[(2 + d) * LW + a]; };
      auto V = [&](int a, int bb, int d) { return (bb < 0 ? R0 : (bb > 0 ? R2 : R1))[(7 + d) * LW + a]; };
      auto W = [&](int a, int bb, int d) { return (bb < 0 ? R0 : (bb > 0 ? R2 : R1))[(12 + d) * LW + a]; };
      smag_c = dsm3r_zq(U, V, W, rdx, rdy, rdzf3, rdzc4, zq);
    }
#pragma unroll
    for (int q = 0; q < DSMC_NQ; ++q) sh[PAR][q * TXB + t] = zq[q];
    __syncthreads();
    if (producer && r + DSMT_NS < nraw) issue(S0);     // the slot of raw row r: every thread is past its last read
    double lm = 0.0, mm = 0.0;
    const bool emit = r >= 2;
    if (inner) dsm3r_row<PAR>(sh[PAR], TXB, t, zq, win, emit, d2, a2, &lm, &mm);
    if (emit) {
      if (outcol) *sm_out = win.smag_prev;
      else { lm = 0.0; mm = 0.0; }
      sm_out += c.nx;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) { lm += __shfl_down_sync(0xffffffffu, lm, o); mm += __shfl_down_sync(0xffffffffu, mm, o); }
      if ((t & 31) == 0) { part[pslot * 2] = lm; part[pslot * 2 + 1] = mm; }
      pslot += pslots;
    }
    win.smag_prev = smag_c;
  };
  for (int r = 0; r < nrows; r += 4) {
    row(std::integral_constant<int, 0>{}, r);
    if (r + 1 < nrows) row(std::integral_constant<int, 1>{}, r + 1);
    if (r + 2 < nrows) row(std::integral_constant<int, 2>{}, r + 2);
    if (r + 3 < nrows) row(std::integral_constant<int, 3>{}, r + 3);
  }
}
#endif


}  // namespace cales
