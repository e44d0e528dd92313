// cales_dsm_col.cuh -- dynamic Smagorinsky, pass 1, x-y test filter, column march with a REGISTER y-window
// (Eq. 5-9; filter, averaging and clipping rules of PAPER.md:128).
//
// Same mathematics as k_dsm_col_sm (cales_closures.cuh): where the test filter has uniform weights it commutes with the
// strain operator, so the kernel filters the 21 centred quantities
//     q = (u_i^c [3], u_i^c u_j^c [6], |S| S_ij [6], S_ij [6])
// with the separable (1/4,1/2,1/4) weights in x and y and contracts L_ij M_ij, M_ij M_ij at every point.
// What differs is where the data live.  ncu on the shared-ring form (profiles/r1_ncu_full.md): 80 % L1/shared pipe, 6.0 G
// shared wavefronts per launch, fp64 pipe 40 % -- the y-window of Fx q (21 quantities x (2 loads + 1 store) per point) was
// two thirds of that traffic.  Here
//   * the y-window is 2 x 21 doubles per thread IN REGISTERS; the row loop is unrolled by two with the row parity a template
//     parameter, so window slots are compile-time names and nothing is ever moved;
//   * the filters run unnormalised (xq' = ql + qr + 2 qc = 4 Fx q;  Fq' = w2 + xq' + 2 w1 = 16 F q): two fp64 instructions per
//     quantity and direction instead of three, the powers of 16 go into the constants of the contraction;
//   * the strain rate uses the summed form of the four-edge average (S_12 = [rdy (sum of 4 du) + rdx (sum of 4 dv)] / 8,
//     PAPER.md:128 "evaluated at the edge midpoints, then averaged") -- 38 instead of 75 fp64 instructions;
//   * with plane averaging (c_s(k)) the two sums are carried in registers over the CTA's rows and reduced once, not per row;
//   * the grid is (x-blocks, k, y-bands): consecutive CTAs sweep k inside one y-band, so the planes k-1, k, k+1 every CTA
//     reads are shared inside a wave through L2 (the (x, y, k) order re-read every plane three times from DRAM).
// Shared memory carries only the 10 base values of a row to the x-neighbours (10 stores + 20 loads per point).
#pragma once
#include "cales_closures.cuh"

namespace cales {

#ifndef CALES_DSMR_MINB
#define CALES_DSMR_MINB 5
#endif

// Strain rate at a centre in summed form, plus the centre velocities (needs the same 30 face values as strain_at).
// b[0..2] = u^c, v^c, w^c; b[3..8] = S_11 S_22 S_33 S_12 S_13 S_23; b[9] = |S|.
template <class GU, class GV, class GW>
CALES_HD void dsmr_base_from(GU U, GV V, GW W, double rdx, double rdy, double rdzf, double rdzc, double rdzcm, double* b) {
  const double u000 = U(0, 0, 0), um00 = U(-1, 0, 0), v000 = V(0, 0, 0), v0m0 = V(0, -1, 0), w000 = W(0, 0, 0), w00m = W(0, 0, -1);
  b[0] = 0.5 * (u000 + um00); b[1] = 0.5 * (v000 + v0m0); b[2] = 0.5 * (w000 + w00m);
  const double s11 = (u000 - um00) * rdx, s22 = (v000 - v0m0) * rdy, s33 = (w000 - w00m) * rdzf;
  const double ex = 0.125 * rdx, ey = 0.125 * rdy, ez = 0.125 * rdzc, ezm = 0.125 * rdzcm;
  // the four edges around the centre share their inner values: only the outer ones survive the sum
  const double s12 = ey * ((U(0, 1, 0) - U(0, -1, 0)) + (U(-1, 1, 0) - U(-1, -1, 0))) + ex * ((V(1, 0, 0) - V(-1, 0, 0)) + (V(1, -1, 0) - V(-1, -1, 0)));
  const double s13 = ez * ((U(0, 0, 1) - u000) + (U(-1, 0, 1) - um00)) + ezm * ((u000 - U(0, 0, -1)) + (um00 - U(-1, 0, -1))) +
                     ex * ((W(1, 0, 0) - W(-1, 0, 0)) + (W(1, 0, -1) - W(-1, 0, -1)));
  const double s23 = ez * ((V(0, 0, 1) - v000) + (V(0, -1, 1) - v0m0)) + ezm * ((v000 - V(0, 0, -1)) + (v0m0 - V(0, -1, -1))) +
                     ey * ((W(0, 1, 0) - W(0, -1, 0)) + (W(0, 1, -1) - W(0, -1, -1)));
  b[3] = s11; b[4] = s22; b[5] = s33; b[6] = s12; b[7] = s13; b[8] = s23;
  b[9] = sqrt(2.0 * (s11 * s11 + s22 * s22 + s33 * s33) + 4.0 * (s12 * s12 + s13 * s13 + s23 * s23));
}

// base values of column gi at row gj (both wrapped / interior)
CALES_HD void dsmr_base(const Ctx& c, const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w,
                        int gi, int gj, int k, double* b) {
  if (interior_row(c, gj, k)) {
    const long long n = idx3(c, gi, gj, k);
    const Nbr o = neighbours(c, gi, gj, k);
    auto at = [&](const double* __restrict__ q, int a, int bb, int d) {
      return q[n + (d < 0 ? o.km : (d > 0 ? o.kp : 0)) + ((a < 0 ? o.im : (a > 0 ? o.ip : 0)) + (bb < 0 ? o.jm : (bb > 0 ? o.jp : 0)))];
    };
    auto U = [&](int a, int bb, int d) { return at(u, a, bb, d); };
    auto V = [&](int a, int bb, int d) { return at(v, a, bb, d); };
    auto W = [&](int a, int bb, int d) { return at(w, a, bb, d); };
    dsmr_base_from(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], b);
  } else if (c.bc_z == BC_WALL && c.nz >= 3 && (k == 0 || k == c.nz - 1) && (c.bc_y == BC_PER || (gj >= 1 && gj <= c.ny - 2))) {
    // a plane next to a z wall, row plain in y: in-plane neighbours by offsets, only the plane beyond the wall is a ghost -- the
    // velg_z rules written out (w = 0 beyond and on the wall; u, v: no-slip mirror, or the linear extrapolation of GH_STRAIN with
    // the wall model).  The generic accessors below cost 1660 instructions per point on these two planes (ncu, r2b).
    const long long n = idx3(c, gi, gj, k);
    const Nbr o = neighbours(c, gi, gj, k);
    const bool bottom = k == 0;
    const int dg = bottom ? -1 : 1;                                   // the ghost plane
    const long long in1 = bottom ? c.nxy : -c.nxy;                    // towards the interior
    const double r = bottom ? c.dzc[-1] / c.dzc[0] : c.dzc[c.nz - 1] / c.dzc[c.nz - 2];
    auto off = [&](int a, int bb) { return (long long)((a < 0 ? o.im : (a > 0 ? o.ip : 0)) + (bb < 0 ? o.jm : (bb > 0 ? o.jp : 0))); };
    auto uv = [&](const double* __restrict__ q, int a, int bb, int d) {
      const long long m = n + off(a, bb);
      if (d != dg) return q[m + (long long)d * c.nxy];
      const double q0 = q[m];
      if (!c.wall_model) return -q0;
      return q0 + (q0 - q[m + in1]) * r;
    };
    auto U = [&](int a, int bb, int d) { return uv(u, a, bb, d); };
    auto V = [&](int a, int bb, int d) { return uv(v, a, bb, d); };
    auto W = [&](int a, int bb, int d) {      // d is 0 or -1; w[nz-1] is stored as 0
      if (bottom && d < 0) return 0.0;
      return w[n + off(a, bb) + (long long)d * c.nxy];
    };
    dsmr_base_from(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], b);
  } else {
    auto U = [&](int a, int bb, int d) { return velg<0>(c, u, gi + a, gj + bb, k + d, GH_STRAIN); };
    auto V = [&](int a, int bb, int d) { return velg<1>(c, v, gi + a, gj + bb, k + d, GH_STRAIN); };
    auto W = [&](int a, int bb, int d) { return velg<2>(c, w, gi + a, gj + bb, k + d, GH_STRAIN); };
    dsmr_base_from(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], b);
  }
}

// y-window of one thread: q[s][m] = 4 Fx q_m of an earlier row.  At row r (parity PAR = r & 1) slot 1-PAR holds row r-1 and
// slot PAR holds row r-2, which is overwritten with row r.
struct DsmrWin { double q[2][DSMC_NQ]; double smag_prev; };

CALES_HD void dsmr_win_init(DsmrWin& w) {
#pragma unroll
  for (int m = 0; m < DSMC_NQ; ++m) { w.q[0][m] = 0.0; w.q[1][m] = 0.0; }
  w.smag_prev = 0.0;
}

// One row of the march for an output column: b = own base values (row r), shbuf = the row's base values of all columns
// ([DSMC_NB][txb]).  Pushes row r into the window; when emit, returns the two contractions of Eq. 6 at row r-1:
//   *lm = L_ij M_ij,  *mm = M_ij M_ij  (sums over the 9 pairs), with d2 = Delta_k^2, a2 = alpha^2.
template <int PAR>
CALES_HD void dsmr_row(const double* shbuf, int txb, int t, const double* b, DsmrWin& w, bool emit, double d2, double a2, double* lm, double* mm) {
  const double* sl = shbuf + t - 1;
  const double* sr = shbuf + t + 1;
  double* w1 = w.q[1 - PAR];     // row r-1
  double* w2 = w.q[PAR];         // row r-2, then row r
  // --- strain rate and |S| S_ij (q 15..20 and 9..14): St' = 16 F(S_ij), Fp = 16 F(|S| S_ij) of row r-1
  double St[6], Mp[6];
  {
    const double ml = sl[9 * txb], mr = sr[9 * txb], mc2 = 2.0 * b[9];
#pragma unroll
    for (int m = 0; m < 6; ++m) {
      const double l = sl[(3 + m) * txb], r = sr[(3 + m) * txb], cc = b[3 + m];
      const double xs = (l + r) + 2.0 * cc;
      const double xp = mc2 * cc + (ml * l + mr * r);
      // old window value consumed first, so the new one can be formed in its register (no moves at the loop's merge points)
      const double ts = w2[15 + m] + 2.0 * w1[15 + m]; w2[15 + m] = xs; St[m] = ts + xs;
      const double tp = w2[9 + m] + 2.0 * w1[9 + m]; w2[9 + m] = xp; Mp[m] = tp + xp;
    }
  }
  double md = 0.0, mo = 0.0;
  if (emit) {   // M' = 256 M / (2 Delta^2) = 16 Fp - alpha^2 (16 |S~|) St'
    const double stmag = sqrt(2.0 * (St[0] * St[0] + St[1] * St[1] + St[2] * St[2]) + 4.0 * (St[3] * St[3] + St[4] * St[4] + St[5] * St[5]));
    const double a2s = a2 * stmag;
#pragma unroll
    for (int m = 0; m < 6; ++m) Mp[m] = 16.0 * Mp[m] - a2s * St[m];
    md = Mp[0] * Mp[0] + Mp[1] * Mp[1] + Mp[2] * Mp[2]; mo = Mp[3] * Mp[3] + Mp[4] * Mp[4] + Mp[5] * Mp[5];
  }
  // --- velocities and their products (q 0..8): L' = 256 L = 16 (16 F(u_i u_j)) - (16 F u_i)(16 F u_j), contracted with M' on the fly
  const double ul = sl[0], ur = sr[0], vl = sl[txb], vr = sr[txb], wl = sl[2 * txb], wr = sr[2 * txb];
  const double uc = b[0], vc = b[1], wc = b[2], uc2 = 2.0 * uc, vc2 = 2.0 * vc, wc2 = 2.0 * wc;
  double x, Fu, Fv, Fw, ld = 0.0, lo = 0.0;
#define DSMR_PUSH(m, expr) x = w2[m] + 2.0 * w1[m]; w2[m] = (expr); const double F##m = x + w2[m];
  DSMR_PUSH(0, (ul + ur) + uc2) Fu = F0;
  DSMR_PUSH(1, (vl + vr) + vc2) Fv = F1;
  DSMR_PUSH(2, (wl + wr) + wc2) Fw = F2;
  DSMR_PUSH(3, uc2 * uc + (ul * ul + ur * ur)) ld += (16.0 * F3 - Fu * Fu) * Mp[0];
  DSMR_PUSH(4, vc2 * vc + (vl * vl + vr * vr)) ld += (16.0 * F4 - Fv * Fv) * Mp[1];
  DSMR_PUSH(5, wc2 * wc + (wl * wl + wr * wr)) ld += (16.0 * F5 - Fw * Fw) * Mp[2];
  DSMR_PUSH(6, uc2 * vc + (ul * vl + ur * vr)) lo += (16.0 * F6 - Fu * Fv) * Mp[3];
  DSMR_PUSH(7, uc2 * wc + (ul * wl + ur * wr)) lo += (16.0 * F7 - Fu * Fw) * Mp[4];
  DSMR_PUSH(8, vc2 * wc + (vl * wl + vr * wr)) lo += (16.0 * F8 - Fv * Fw) * Mp[5];
#undef DSMR_PUSH
  if (!emit) return;
  const double sc = 2.0 * d2 * (1.0 / 256.0);
  *lm = (ld + 2.0 * lo) * (sc * (1.0 / 256.0));
  *mm = (md + 2.0 * mo) * (sc * sc);
}

#ifdef __CUDACC__
// grid (ceil(nx/(TXB-2)), planes, ceil((jhi-jlo)/ly)), block TXB (multiple of 32); ly = output rows per CTA.  Planes k0 + blockIdx.y * kstride,
// output rows [jlo, jhi).
// part: [k][j][pslots][2]; this kernel fills slots blockIdx.x*(TXB/32) + warp of its rows: per row with x-line averaging, the
// CTA's total in its first row with plane averaging (the others are left at the zeros the host guarantees).
template <int TXB, int MINB>
__global__ void __launch_bounds__(TXB, MINB) k_dsm_col_rw(const __grid_constant__ Ctx c, const double* __restrict__ u, const double* __restrict__ v,
                                                          const double* __restrict__ w, int k0, int kstride, int jlo, int jhi, int ly, int pslots,
                                                          double* __restrict__ smag, double* __restrict__ part) {
  __shared__ double sh[2][DSMC_NB * TXB];
  const int t = threadIdx.x, k = k0 + blockIdx.y * kstride;
  const int i0 = blockIdx.x * (TXB - 2);
  const int j0 = jlo + blockIdx.z * ly;
  const int jend = min(j0 + ly, jhi);
  const int nrows = jend - j0 + 2;
  const int gi = i0 - 1 + t;
  const int gw = ((gi % c.nx) + c.nx) % c.nx;
  const bool inner = t >= 1 && t <= TXB - 2;
  const bool outcol = inner && gi < c.nx;
  const bool zplain = k >= 1 && k <= c.nz - 2;
  const double d2 = c.delta[k] * c.delta[k], a2 = c.alpha * c.alpha;
  const long long pslot0 = ((long long)k * c.ny) * pslots + blockIdx.x * (TXB / 32) + (t >> 5);
  DsmrWin win;
  dsmr_win_init(win);
  double accl = 0.0, accm = 0.0;
  auto row = [&](auto par, int r) {
    constexpr int PAR = decltype(par)::value;
    int gj = j0 - 1 + r;
    gj = gj < 0 ? gj + c.ny : (gj >= c.ny ? gj - c.ny : gj);
    double b[DSMC_NB];
    dsmr_base(c, u, v, w, gw, gj, k, b);
#pragma unroll
    for (int q = 0; q < DSMC_NB; ++q) sh[PAR][q * TXB + t] = b[q];
    if (r + 2 < nrows && (t & 3) == 0 && zplain) {     // the row after next: pull its lines towards L1
      int gp = j0 + 1 + r + 1; gp = gp >= c.ny ? gp - c.ny : gp;
      const long long nn = idx3(c, gw, gp, k);
#pragma unroll
      for (int d = -1; d <= 1; ++d) {
        asm volatile("prefetch.global.L1 [%0];" ::"l"(u + nn + d * c.nxy));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(v + nn + d * c.nxy));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(w + nn + d * c.nxy));
      }
    }
    __syncthreads();
    double lm = 0.0, mm = 0.0;
    const bool emit = r >= 2;
    if (inner) dsmr_row<PAR>(sh[PAR], TXB, t, b, win, emit, d2, a2, &lm, &mm);
    if (emit) {
      const int jo = j0 + r - 2;
      if (outcol) smag[idx3(c, gi, jo, k)] = win.smag_prev;
      else { lm = 0.0; mm = 0.0; }
      if (c.dsm_plane) { accl += lm; accm += mm; }
      else {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { lm += __shfl_down_sync(0xffffffffu, lm, o); mm += __shfl_down_sync(0xffffffffu, mm, o); }
        if ((t & 31) == 0) { const long long slot = pslot0 + (long long)jo * pslots; part[slot * 2] = lm; part[slot * 2 + 1] = mm; }
      }
    }
    win.smag_prev = b[9];
  };
  for (int r = 0; r < nrows; r += 2) {
    row(std::integral_constant<int, 0>{}, r);
    if (r + 1 < nrows) row(std::integral_constant<int, 1>{}, r + 1);
  }
  if (c.dsm_plane) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { accl += __shfl_down_sync(0xffffffffu, accl, o); accm += __shfl_down_sync(0xffffffffu, accm, o); }
    if ((t & 31) == 0)
      {      // the CTA's total in the slot of its first row.  The slots of its other rows are never written: they are zero since create (or
             // since the host re-zeroed the array after an option changed the band layout), which saves 0.4 GB of scattered 16-byte
             // stores per launch at config 5 (18.75 -> 18.40 ms per evaluation)
        const long long slot = pslot0 + (long long)j0 * pslots;
        part[slot * 2] = accl; part[slot * 2 + 1] = accm;
      }
  }
}

// ---- the same march with the raw velocity rows staged by the TMA engine ---------------------------------------------------
// ncu on k_dsm_col_rw (profiles/r2_ncu_dsm.md): 577 instructions per warp and row of which only 219 are fp64 -- the rest is
// 64-bit address arithmetic of 30 strided loads per point, wrap selects and branches -- and the warps wait on those loads.
// Here eight lanes keep a ring of DSMT_NS = 4 raw ROWS in shared memory, DSMT_NL = 8 lines each (u on planes k-1, k, k+1; v on
// k-1, k, k+1; w on k-1, k), filled by cp.async.bulk (UBLKCP) copies that complete on an mbarrier two rows ahead of their
// first use: each producer lane issues one line, periodic wrap in x splits a line into two copies, wrap in y / z is pointer arithmetic of
// the issuing lane.  The row loop is unrolled by four, so ring slots and window parity are compile-time and the strain
// stencil is 30 shared-memory loads at immediate offsets.  Planes next to a z wall (wall ghosts) are left to k_dsm_col_rw.
enum { DSMT_NS = 4, DSMT_NL = 8 };

// grid (ceil(nx/(TXB-2)), khi-klo, ceil((jhi-jlo)/ly)), block TXB = 64; planes [klo, khi), output rows [jlo, jhi).
// Needs nx >= TXB + 2, 16-byte aligned fields, and every base row jlo-1 .. jhi an interior row (periodic y, or 1 <= j <= ny-2).
template <int TXB, int MINB>
__global__ void __launch_bounds__(TXB, MINB) k_dsm_col_tma(const __grid_constant__ Ctx c, const double* __restrict__ u, const double* __restrict__ v,
                                                           const double* __restrict__ w, int klo, int jlo, int jhi, int ly, int pslots,
                                                           double* __restrict__ smag, double* __restrict__ part) {
  constexpr int LW = TXB + 2;                  // columns i0-2 .. i0+TXB-1 of a line
  constexpr int STAGE = DSMT_NL * LW;
  __shared__ __align__(128) double raw[DSMT_NS * STAGE];
  __shared__ double sh[2][DSMC_NB * TXB];
  __shared__ unsigned long long full[DSMT_NS];
  const int t = threadIdx.x, k = klo + blockIdx.y;
  const int i0 = blockIdx.x * (TXB - 2);
  const int j0 = jlo + blockIdx.z * ly;
  const int jend = min(j0 + ly, jhi);
  const int nrows = jend - j0 + 2;             // base rows j0-1 .. jend; raw rows j0-2 .. jend+1 (nrows + 2 of them)
  const int nraw = nrows + 2;
  const int gi = i0 - 1 + t;
  const bool inner = t >= 1 && t <= TXB - 2;
  const bool outcol = inner && gi < c.nx;
  const double d2 = c.delta[k] * c.delta[k], a2 = c.alpha * c.alpha;
  const double rdx = c.rdx, rdy = c.rdy, rdzf = c.rdzf[k], rdzc = c.rdzc[k], rdzcm = c.rdzc[k - 1];
  // ---- producer state (lanes 0..7 of warp 0): source pointer of this lane's line at the next raw row, x segments
  const double* src = nullptr; int gj_next = 0, segA = 0;
  const bool producer = (t & 31) < DSMT_NL / 2 && t < 64;      // lanes 0..3 of warps 0 and 1: four lines each
  const int line = (t & 31) + (t >> 5) * (DSMT_NL / 2);
  if (producer) {
    const int l = line;
    const double* f = l < 3 ? u : (l < 6 ? v : w);
    const int km = k == 0 ? c.nz - 1 : k - 1, kp = k == c.nz - 1 ? 0 : k + 1;
    const int kk = (l == 1 || l == 4 || l == 7) ? k : ((l == 2 || l == 5) ? kp : km);
    gj_next = j0 - 2; gj_next = gj_next < 0 ? gj_next + c.ny : gj_next;
    src = f + ((long long)kk * c.ny + gj_next) * c.nx;
    const int cw0 = (((i0 - 2) % c.nx) + c.nx) % c.nx;
    segA = min(LW, c.nx - cw0);
    src += cw0;                                // segment A starts at column cw0, segment B (if any) at column 0 of the row
  }
  auto issue = [&](int slot) {                 // next raw row into `slot` (called by the eight producer lanes)
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
  double accl = 0.0, accm = 0.0;
  double* sm_out = smag + idx3(c, gi < c.nx ? gi : 0, j0, k);           // |S| of output row j0, bumped by nx per emitted row
  long long pslot = ((long long)k * c.ny + j0) * pslots + blockIdx.x * (TXB / 32) + (t >> 5);
  const double* Rt = raw + t + 1;
  auto row = [&](auto ph, int r) {
    constexpr int PH = decltype(ph)::value;    // r & 3
    constexpr int PAR = PH & 1, S0 = PH, S1 = (PH + 1) & 3, S2 = (PH + 2) & 3;
    if (r == 0) { mbar_wait(&full[0], 0); mbar_wait(&full[1], 0); }
    mbar_wait(&full[S2], ((r + 2) >> 2) & 1);
    double b[DSMC_NB];
    {
      const double* R0 = Rt + S0 * STAGE;      // raw row below the base row
      const double* R1 = Rt + S1 * STAGE;      // the base row
      const double* R2 = Rt + S2 * STAGE;      // the row above
      auto U = [&](int a, int bb, int d) { return (bb < 0 ? R0 : (bb > 0 ? R2 : R1))[(1 + d) * LW + a]; };
      auto V = [&](int a, int bb, int d) { return (bb < 0 ? R0 : (bb > 0 ? R2 : R1))[(4 + d) * LW + a]; };
      auto W = [&](int a, int bb, int d) { return (bb < 0 ? R0 : (bb > 0 ? R2 : R1))[(7 + d) * LW + a]; };
      dsmr_base_from(U, V, W, rdx, rdy, rdzf, rdzc, rdzcm, b);
    }
#pragma unroll
    for (int q = 0; q < DSMC_NB; ++q) sh[PAR][q * TXB + t] = b[q];
    __syncthreads();
    if (producer && r + DSMT_NS < nraw) issue(S0);     // the slot of raw row r: every thread is past its last read
    double lm = 0.0, mm = 0.0;
    const bool emit = r >= 2;
    if (inner) dsmr_row<PAR>(sh[PAR], TXB, t, b, win, emit, d2, a2, &lm, &mm);
    if (emit) {
      if (outcol) *sm_out = win.smag_prev;
      else { lm = 0.0; mm = 0.0; }
      sm_out += c.nx;
      if (c.dsm_plane) { accl += lm; accm += mm; }
      else {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { lm += __shfl_down_sync(0xffffffffu, lm, o); mm += __shfl_down_sync(0xffffffffu, mm, o); }
        if ((t & 31) == 0) { part[pslot * 2] = lm; part[pslot * 2 + 1] = mm; }
        pslot += pslots;
      }
    }
    win.smag_prev = b[9];
  };
  for (int r = 0; r < nrows; r += 4) {
    row(std::integral_constant<int, 0>{}, r);
    if (r + 1 < nrows) row(std::integral_constant<int, 1>{}, r + 1);
    if (r + 2 < nrows) row(std::integral_constant<int, 2>{}, r + 2);
    if (r + 3 < nrows) row(std::integral_constant<int, 3>{}, r + 3);
  }
  if (c.dsm_plane) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { accl += __shfl_down_sync(0xffffffffu, accl, o); accm += __shfl_down_sync(0xffffffffu, accm, o); }
    if ((t & 31) == 0)
      { part[pslot * 2] = accl; part[pslot * 2 + 1] = accm; }      // the CTA's total in its first row; the slots of its other rows stay 0 (see k_dsm_col_rw)
  }
}
#endif

}  // namespace cales
