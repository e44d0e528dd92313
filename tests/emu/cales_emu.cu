// cales_emu.cu -- HOST EMULATOR of the CUDA kernels of libcales.so.  TEST INFRASTRUCTURE ONLY.
//
// Purpose: the box that runs `pytest -m "not gpu"` has no GPU.  The kernels of paper_2411_09364_b200/csrc are
// written as __host__ __device__ phase functions of (tid, nth) / per-point functions, with the block barriers in
// the __global__ wrappers only.  This file steps those SAME functions on the host -- block by block, phase by
// phase, thread by thread -- in the order cales.cu launches them, so that the device code's arithmetic and index
// logic can be compared with the CPU oracle without a GPU.  It is NOT a fallback: nothing in the package loads
// it, it is built only by tests/emu/build.py, and it is orders of magnitude slower than the oracle.
// Not covered here (GPU tests only): launch shapes, shared-memory sizes, warp-shuffle reductions, stream order.
#include "../../paper_2411_09364_b200/csrc/cales_host.h"
#include "../../paper_2411_09364_b200/csrc/cales_poisson.cuh"
#include "../../paper_2411_09364_b200/csrc/cales_momentum.cuh"
#include "../../paper_2411_09364_b200/csrc/cales_rhs_tile.cuh"
#include "../../paper_2411_09364_b200/csrc/cales_smag_tile.cuh"
#include "../../paper_2411_09364_b200/csrc/cales_dsm_col.cuh"
#include "../../paper_2411_09364_b200/csrc/cales_dsm3.cuh"

#include <cstring>
#include <vector>

using namespace cales;

struct emu_solver {
  HostSetup H;
  Ctx c;
  FftPlan plx, ply;
  PoissonTabs pt;
  long long N, nxy;
  std::vector<double> u, v, w, p, nut, us, vs, ws, Ru, Rv, Rw, W, CP, CQ, smag, tau, tau_y, cncoef, dsm_part, dsm_cs;
  double scal[4];
  int maxit;
  bool fresh;
};

extern "C" const char* emu_last_error(void) { return g_err.c_str(); }

extern "C" int emu_create(const cales_params* p, emu_solver** out) {
  emu_solver* s = new emu_solver();
  int rc = build_setup(p, s->H);
  if (rc) { delete s; return rc; }
  HostSetup& H = s->H;
  s->c = H.c; s->N = H.c.N; s->nxy = H.c.nxy;
  const size_t N = (size_t)s->N;
  for (auto* f : {&s->u, &s->v, &s->w, &s->p, &s->nut, &s->us, &s->vs, &s->ws, &s->Ru, &s->Rv, &s->Rw, &s->W, &s->CP, &s->CQ, &s->smag}) f->assign(N, 0.0);
  s->tau.assign(4 * (size_t)s->nxy, 0.0);
  s->tau_y.assign(4 * (size_t)p->nx * p->nz, 0.0);
  s->cncoef.assign(6 * (size_t)p->nz, 0.0);
  s->dsm_part.assign((size_t)p->nz * p->ny * dsm_shape(p->nx).pslots * 2, 0.0);
  s->dsm_cs.assign((size_t)p->nz * p->ny, 0.0);
  s->c.dzf = H.dzf.data() + 1; s->c.dzc = H.dzc.data() + 1; s->c.zc = H.zc.data(); s->c.rdzf = H.rdzf.data() + 1; s->c.rdzc = H.rdzc.data() + 1; s->c.delta = H.delta.data(); s->c.tau = s->tau.data(); s->c.tau_y = s->tau_y.data();
  s->plx = H.plx; s->plx.tw = reinterpret_cast<const double2*>(H.twx.data());
  s->ply = H.ply; s->ply.tw = reinterpret_cast<const double2*>(H.twy.data()); s->ply.dctw = reinterpret_cast<const double2*>(H.dctw.data());
  s->pt.ak = H.ak.data(); s->pt.ck = H.ck.data(); s->pt.lamx = H.lamx.data(); s->pt.lamy = H.lamy.data();
  s->scal[0] = s->scal[1] = s->scal[2] = 0.0; s->maxit = 0; s->fresh = false;
  *out = s;
  return 0;
}
extern "C" void emu_destroy(emu_solver* s) { delete s; }

static std::vector<double>* fld(emu_solver* s, int f) {
  switch (f) { case 0: return &s->u; case 1: return &s->v; case 2: return &s->w; case 3: return &s->p; case 4: return &s->nut; }
  return nullptr;
}
extern "C" int emu_set_field(emu_solver* s, int f, const double* src) {
  std::memcpy(fld(s, f)->data(), src, s->N * sizeof(double));
  const Ctx& c = s->c;
  if (f == 1 && c.bc_y == BC_WALL) for (int k = 0; k < c.nz; ++k) for (int i = 0; i < c.nx; ++i) s->v[idx3(c, i, c.ny - 1, k)] = 0.0;
  if (f == 2 && c.bc_z == BC_WALL) for (long long q = 0; q < s->nxy; ++q) s->w[(long long)(c.nz - 1) * s->nxy + q] = 0.0;
  if (f <= 2) s->fresh = false;
  return 0;
}
extern "C" int emu_get_field(emu_solver* s, int f, double* dst) { std::memcpy(dst, fld(s, f)->data(), s->N * sizeof(double)); return 0; }

// ---- kernel emulations: same block decomposition and phase order as the __global__ wrappers ----
// f2_passes (cales_fft2.cuh) stepped on the host: one register file of F2_E complex numbers per emulated thread, the
// phases separated where the kernel has its block barriers.
template <bool TO_GLOBAL, int E = F2_E, class FIRST, class LAST>
static void emu_f2_passes(const Fft2Lay& lay, const FftPlan& pl, int sign, double2* buf, int nth, FIRST first, LAST last) {
  const int np = pl.npass;
  std::vector<double2> regs((size_t)nth * E);
  F2SmemLd sld{buf, lay}; F2SmemSt sst{buf, lay};
  if (np == 0) {
    std::vector<double2> z(lay.L);
    for (int b = 0; b < lay.L && b < 2 * nth; ++b) z[b] = first(b, 0);       // thread tid owns lines tid and tid + nth
    for (int b = 0; b < lay.L && b < 2 * nth; ++b) { if (TO_GLOBAL) last(b, 0, z[b]); else sst(b, 0, z[b]); }
    return;
  }
  for (int p = 0; p < np; ++p) {
    for (int tid = 0; tid < nth; ++tid) {
      if (p == 0) f2_load_any<E>(lay, pl, 0, tid, nth, first, &regs[(size_t)tid * E]);
      else f2_load_any<E>(lay, pl, p, tid, nth, sld, &regs[(size_t)tid * E]);
    }
    for (int tid = 0; tid < nth; ++tid) {
      if (TO_GLOBAL && p == np - 1) f2_bfly_any<E>(lay, pl, p, sign, tid, nth, &regs[(size_t)tid * E], last);
      else f2_bfly_any<E>(lay, pl, p, sign, tid, nth, &regs[(size_t)tid * E], sst);
    }
  }
}
static void emu_fft_x_fwd(emu_solver* s, const double* src, const DivSrc* ds, double* dst) {
  const Ctx& c = s->c; const FftPlan& pl = s->plx; const int L = s->H.xB, nth = s->H.x_threads;
  const Fft2Lay lay{L, sm_line(pl.n2), 0, false};
  std::vector<double2> sm((size_t)L * lay.ls);
  const long long nlines = (long long)c.ny * c.nz;
  DivSrc none{nullptr, nullptr, nullptr, 0.0, nullptr};
  for (long long l0 = 0; l0 < nlines; l0 += L) {
    const int nb = (int)std::min<long long>(L, nlines - l0);
    F2XFwdLd first{c, pl, l0, nb, src, ds ? *ds : none, ds != nullptr, ds ? ds->inv_gdt : 0.0};
    emu_f2_passes<false>(lay, pl, -1, sm.data(), nth, first, F2SmemSt{sm.data(), lay});
    for (int tid = 0; tid < nth; ++tid) f2x_split_store(tid, nth, pl, lay, l0, nb, sm.data(), dst);
  }
}
static void emu_fft_x_inv(emu_solver* s, const double* src, double* dst) {
  const Ctx& c = s->c; const FftPlan& pl = s->plx; const int L = s->H.xB, nth = s->H.x_threads;
  const Fft2Lay lay{L, sm_line(pl.n2), 0, false};
  std::vector<double2> sm((size_t)L * lay.ls);
  const long long nlines = (long long)c.ny * c.nz;
  for (long long l0 = 0; l0 < nlines; l0 += L) {
    const int nb = (int)std::min<long long>(L, nlines - l0);
    F2XInvLd first{pl, l0, nb, src};
    F2XInvSt last{pl, l0, nb, dst, 1.0 / (double)pl.n2};
    emu_f2_passes<true>(lay, pl, +1, sm.data(), nth, first, last);
  }
}
static void emu_fft_y(emu_solver* s, double* A, int inverse) {
  const Ctx& c = s->c; const FftPlan& pl = s->ply; const int TI = s->H.yTI, nth = s->H.y_threads;
  const bool dct = c.bc_y == BC_WALL;
  const Fft2Lay lay{TI, 0, s->H.y_tish, true};
  std::vector<double2> sm((size_t)TI * std::max(pl.n2, 1));
  for (int k = 0; k < c.nz; ++k) for (int i0 = 0; i0 < c.nx; i0 += TI) {
    const int nb = std::min(TI, c.nx - i0);
    double* base = A + (long long)k * c.nxy + i0;
    if (!inverse) {
      F2YFwdLd first{c, pl, base, nb, dct};
      emu_f2_passes<false, F2_EY>(lay, pl, -1, sm.data(), nth, first, F2SmemSt{sm.data(), lay});
      for (int tid = 0; tid < nth; ++tid) f2y_split_store(tid, nth, c, pl, lay, dct, base, nb, sm.data());
    } else {
      F2YInvLd first{c, pl, base, nb, dct};
      F2YInvSt last{c, pl, base, nb, dct, 1.0 / (double)pl.n2};
      emu_f2_passes<true, F2_EY>(lay, pl, +1, sm.data(), nth, first, last);
    }
  }
}
static void emu_poisson_core(emu_solver* s) {
  emu_fft_y(s, s->W.data(), 0);
  for (int j = 0; j < s->c.ny; ++j) for (int i = 0; i < s->c.nx; ++i) poisson_column(s->c, s->pt, i, j, s->W.data(), s->CP.data(), s->CQ.data());
  emu_fft_y(s, s->W.data(), 1);
}
static void emu_tau(emu_solver* s) {
  if (s->c.wall_model_y) {
    if (!s->c.wall_model) s->maxit = 0;
    std::vector<double> ty(s->tau_y.size());      // all stresses come from the velocity only: order of evaluation is immaterial
    for (int z = 0; z < 4; ++z) for (int k = 0; k < s->c.nz; ++k) for (int i = 0; i < s->c.nx; ++i)
      wall_stress_y_point(s->c, s->u.data(), s->w.data(), z >> 1, z & 1, i, k, ty.data());
    s->tau_y = ty; s->c.tau_y = s->tau_y.data();
  }
  if (!s->c.wall_model) return;
  s->maxit = 0;
  for (int z = 0; z < 4; ++z) for (int j = 0; j < s->c.ny; ++j) for (int i = 0; i < s->c.nx; ++i) {
    const int it = wall_stress_point(s->c, s->H.wg, s->u.data(), s->v.data(), z >> 1, z & 1, i, j, s->tau.data());
    if (it > s->maxit) s->maxit = it;
  }
}
static void emu_nut(emu_solver* s, const double* u, const double* v, const double* w, double* nut) {
  const Ctx& c = s->c;
  if (c.sgs == 0) { for (long long n = 0; n < s->N; ++n) nut[n] = 0.0; return; }
  if (c.sgs == 1) {
    // k_smag_tile: stage the three halo planes with the kernel's staging rule (st_elem), evaluate through the tile accessor
    std::vector<double> ring(3 * ST_NF * RT_PLANE);
    for (int j0 = 0; j0 < c.ny; j0 += RT_TY) for (int i0 = 0; i0 < c.nx; i0 += RT_TX) for (int k = 0; k < c.nz; ++k) {
      for (int d = 0; d < 3; ++d) for (int f = 0; f < ST_NF; ++f) for (int pos = 0; pos < RT_PLANE; ++pos) {
        const int ry = pos / RT_TW, rx = pos % RT_TW, gi = i0 - 1 + rx, gj = j0 - 1 + ry;
        ring[(d * ST_NF + f) * RT_PLANE + pos] = (gi <= c.nx && gj <= c.ny) ? st_elem(c, u, v, w, f, gi, gj, k - 1 + d) : 0.0;
      }
      const double* sl[3] = {ring.data(), ring.data() + ST_NF * RT_PLANE, ring.data() + 2 * ST_NF * RT_PLANE};
      for (int ly = 0; ly < RT_TY; ++ly) for (int tx = 0; tx < RT_TX; ++tx) {
        const int i = i0 + tx, j = j0 + ly;
        if (i >= c.nx || j >= c.ny) continue;
        double tauw[2] = {0.0, 0.0};
        if (c.van_driest) smag_wall_shear(c, u, v, i, j, tauw);
        nut[idx3(c, i, j, k)] = smag_tile_point(c, sl, (ly + 1) * RT_TW + tx + 1, k, tauw);
      }
    }
    return;
  }
  const DsmShape dsh = dsm_shape(c.nx);
  const int ntx = dsh.pslots;
  const bool ywall = c.bc_y == BC_WALL, split = ywall && c.ny >= 3 * DSM_TY;
  std::fill(s->dsm_part.begin(), s->dsm_part.end(), 0.0);
  if (c.dsm_filter3d) {   // k_dsm3_pass1: phases separated by the block barrier
    const int ntile = (c.nx + D3_TX - 1) / D3_TX, nth = D3_TX * D3_TY;
    std::vector<double> sm(D3_SMEM_DOUBLES);
    double* raw = sm.data(); double* flt = raw + D3_RAW; double* mid = flt + D3_FLT;
    const D3Split sp = d3_split(c, s->H.P.zstretch == CALES_Z_UNIFORM);
    // the tile kernel's launches: (planes, row tiles, jstride, row_hi, row_lo2)
    struct TL { int k0, k1, nby, jstride, row_hi, row_lo2; };
    std::vector<TL> tl;
    if (!sp.col) tl.push_back({0, c.nz, (c.ny + D3_TY - 1) / D3_TY, D3_TY, c.ny, c.ny});
    else {
      if (sp.klo > 0) { tl.push_back({0, sp.klo, (c.ny + D3_TY - 1) / D3_TY, D3_TY, c.ny, c.ny}); tl.push_back({sp.khi, c.nz, (c.ny + D3_TY - 1) / D3_TY, D3_TY, c.ny, c.ny}); }
      if (sp.jlo > 0) tl.push_back({sp.klo, sp.khi, 2, c.ny - D3_TY, sp.jlo, sp.jhi});
    }
    for (const TL& L : tl)
    for (int k = L.k0; k < L.k1; ++k) for (int by = 0; by < L.nby; ++by) for (int bx = 0; bx < ntile; ++bx) {
      const int i0 = bx * D3_TX, j0 = by * L.jstride;
      for (int tid = 0; tid < nth; ++tid) d3_load(tid, nth, c, u, v, w, i0, j0, k, raw);
      for (int tid = 0; tid < nth; ++tid) d3_mid(tid, nth, c, i0, j0, k, raw, flt, mid);
      for (int ty = 0; ty < D3_TY; ++ty) {
        const int j = j0 + ty;
        if (!(j < c.ny && (j < L.row_hi || j >= L.row_lo2))) continue;
        double lm = 0.0, mm = 0.0;
        for (int tx = 0; tx < D3_TX; ++tx) {
          const int i = i0 + tx;
          if (i < c.nx) {
            double a, b, sg;
            d3_point(c, j0, k, tx, ty, flt, mid, &a, &b, &sg);
            s->smag[idx3(c, i, j, k)] = sg; lm += a; mm += b;
          }
        }
        const long long row = (long long)k * c.ny + j;
        s->dsm_part[(row * ntx + bx) * 2] = lm; s->dsm_part[(row * ntx + bx) * 2 + 1] = mm;
      }
    }
    if (sp.col && c.nx >= 66) {   // k_dsm3_col_tma: register window per emulated thread, zq' from the raw velocities on planes k-2 .. k+2
      const int T = dsh.txb;
      std::vector<double> sh(2 * DSMC_NQ * T), zq((size_t)T * DSMC_NQ), smc(T);
      std::vector<DsmrWin> win(T);
      auto wr = [](int a, int n) { return a < 0 ? a + n : (a >= n ? a - n : a); };
      for (int k = sp.klo; k < sp.khi; ++k) for (int by = 0; by * DSMC_LY < sp.jhi - sp.jlo; ++by) for (int bx = 0; bx < dsh.nbx; ++bx) {
        const int i0 = bx * (T - 2), j0 = sp.jlo + by * DSMC_LY, jend = std::min(j0 + DSMC_LY, sp.jhi), nrows = jend - j0 + 2;
        const double d2 = c.delta[k] * c.delta[k], a2 = c.alpha * c.alpha * c.alpha;
        const double rdzf3[3] = {c.rdzf[wr(k - 1, c.nz)], c.rdzf[k], c.rdzf[wr(k + 1, c.nz)]};
        const double rdzc4[4] = {c.rdzc[wr(k - 2, c.nz)], c.rdzc[wr(k - 1, c.nz)], c.rdzc[k], c.rdzc[wr(k + 1, c.nz)]};
        for (int t = 0; t < T; ++t) dsmr_win_init(win[t]);
        for (int r = 0; r < nrows; ++r) {
          const int gj = wr(j0 - 1 + r, c.ny);
          double* buf = sh.data() + (r & 1) * DSMC_NQ * T;
          for (int t = 0; t < T; ++t) {
            const int gw = (((i0 - 1 + t) % c.nx) + c.nx) % c.nx;
            auto at = [&](const double* f, int a, int b, int d) { return f[idx3(c, wr(gw + a, c.nx), wr(gj + b, c.ny), wr(k + d, c.nz))]; };
            auto U = [&](int a, int b, int d) { return at(u, a, b, d); };
            auto V = [&](int a, int b, int d) { return at(v, a, b, d); };
            auto W = [&](int a, int b, int d) { return at(w, a, b, d); };
            smc[t] = dsm3r_zq(U, V, W, c.rdx, c.rdy, rdzf3, rdzc4, &zq[(size_t)t * DSMC_NQ]);
            for (int q = 0; q < DSMC_NQ; ++q) buf[q * T + t] = zq[(size_t)t * DSMC_NQ + q];
          }
          std::vector<double> wl(T / 32, 0.0), wm(T / 32, 0.0);
          for (int t = 0; t < T; ++t) {
            double lm = 0.0, mm = 0.0;
            const bool inner = t >= 1 && t <= T - 2, emit = r >= 2;
            if (inner) {
              if (r & 1) dsm3r_row<1>(buf, T, t, &zq[(size_t)t * DSMC_NQ], win[t], emit, d2, a2, &lm, &mm);
              else dsm3r_row<0>(buf, T, t, &zq[(size_t)t * DSMC_NQ], win[t], emit, d2, a2, &lm, &mm);
            }
            const int gi = i0 - 1 + t;
            if (emit && inner && gi < c.nx) { s->smag[idx3(c, gi, j0 + r - 2, k)] = win[t].smag_prev; wl[t >> 5] += lm; wm[t >> 5] += mm; }
            win[t].smag_prev = smc[t];
          }
          if (r >= 2) for (int wq = 0; wq < T / 32; ++wq) {
            const long long slot = ((long long)k * c.ny + (j0 + r - 2)) * ntx + bx * (T / 32) + wq;
            s->dsm_part[slot * 2] = wl[wq]; s->dsm_part[slot * 2 + 1] = wm[wq];
          }
        }
      }
    } else
    if (sp.col) {   // k_dsm3_col, stepped row by row with the block barrier between the phases
      const int T = dsh.txb;
      std::vector<double> sh(2 * DSMC_NQ * T), zq((size_t)T * DSMC_NQ), smc(T), ring(2 * DSMC_NQ * T), smprev(T);
      for (int k = sp.klo; k < sp.khi; ++k) for (int by = 0; by * DSMC_LY < sp.jhi - sp.jlo; ++by) for (int bx = 0; bx < dsh.nbx; ++bx) {
        const int i0 = bx * (T - 2), j0 = sp.jlo + by * DSMC_LY, jend = std::min(j0 + DSMC_LY, sp.jhi), nrows = jend - j0 + 2;
        std::fill(ring.begin(), ring.end(), 0.0); std::fill(smprev.begin(), smprev.end(), 0.0);
        for (int r = 0; r < nrows; ++r) {
          int gj = j0 - 1 + r; gj = gj < 0 ? gj + c.ny : (gj >= c.ny ? gj - c.ny : gj);
          double* buf = sh.data() + (r & 1) * DSMC_NQ * T;
          for (int t = 0; t < T; ++t) d3c_phaseA(c, u, v, w, T, t, i0, gj, k, buf, &zq[(size_t)t * DSMC_NQ], &smc[t]);
          std::vector<double> wl(T / 32, 0.0), wm(T / 32, 0.0);
          for (int t = 1; t <= T - 2; ++t) {
            double lm = 0.0, mm = 0.0, sg = 0.0;
            const bool done = d3c_phaseB(c, T, t, r, k, buf, &zq[(size_t)t * DSMC_NQ], ring.data(), &smprev[t], smc[t], &lm, &mm, &sg);
            const int gi = i0 - 1 + t;
            if (r >= 2 && done && gi < c.nx) { s->smag[idx3(c, gi, j0 + r - 2, k)] = sg; wl[t >> 5] += lm; wm[t >> 5] += mm; }
          }
          if (r >= 2) for (int wq = 0; wq < T / 32; ++wq) {
            const long long slot = ((long long)k * c.ny + (j0 + r - 2)) * ntx + bx * (T / 32) + wq;
            s->dsm_part[slot * 2] = wl[wq]; s->dsm_part[slot * 2 + 1] = wm[wq];
          }
        }
      }
    }
  } else if (ywall) {   // tile kernel: all rows, or the DSM_TY rows next to each y wall
    const int ntile = (c.nx + DSM_TX - 1) / DSM_TX, nth = DSM_TX * DSM_TY;
    const int nby = split ? 2 : (c.ny + DSM_TY - 1) / DSM_TY, jstride = split ? c.ny - DSM_TY : DSM_TY;
    const int row_hi = split ? DSM_TY : c.ny, row_lo2 = split ? c.ny - DSM_TY : c.ny;
    std::vector<double> sm(DSM_SMEM_DOUBLES);
    double* raw = sm.data(); double* flt = raw + DSM_RAW; double* mid = flt + DSM_FLT;
    for (int k = 0; k < c.nz; ++k) for (int by = 0; by < nby; ++by) for (int bx = 0; bx < ntile; ++bx) {
      const int i0 = bx * DSM_TX, j0 = by * jstride;
      for (int tid = 0; tid < nth; ++tid) dsm_load(tid, nth, c, u, v, w, i0, j0, k, raw);
      for (int tid = 0; tid < nth; ++tid) dsm_mid(tid, nth, c, i0, j0, k, raw, flt, mid);
      for (int ty = 0; ty < DSM_TY; ++ty) {
        const int j = j0 + ty;
        const bool mine = j < c.ny && (j < row_hi || j >= row_lo2);
        if (!mine) continue;
        double lm = 0.0, mm = 0.0;
        for (int tx = 0; tx < DSM_TX; ++tx) {
          const int i = i0 + tx;
          if (i < c.nx) {
            double a, b, sg;
            dsm_point(c, i0, j0, k, tx, ty, flt, mid, &a, &b, &sg);
            s->smag[idx3(c, i, j, k)] = sg; lm += a; mm += b;
          }
        }
        const long long row = (long long)k * c.ny + j;
        s->dsm_part[(row * ntx + bx) * 2] = lm; s->dsm_part[(row * ntx + bx) * 2 + 1] = mm;
      }
    }
  }
  if (!c.dsm_filter3d && (!ywall || split)) {   // k_dsm_col_rw: stepped row by row with the block barrier between the phases; one register window per emulated thread
    const int T = dsh.txb, jlo = ywall ? DSM_TY : 0, jhi = ywall ? c.ny - DSM_TY : c.ny;
    std::vector<double> sh(2 * DSMC_NB * T), breg((size_t)T * DSMC_NB);
    std::vector<DsmrWin> win(T);
    for (int k = 0; k < c.nz; ++k) for (int by = 0; by * DSMC_LY < jhi - jlo; ++by) for (int bx = 0; bx < dsh.nbx; ++bx) {
      const int i0 = bx * (T - 2), j0 = jlo + by * DSMC_LY, jend = std::min(j0 + DSMC_LY, jhi), nrows = jend - j0 + 2;
      const double d2 = c.delta[k] * c.delta[k], a2 = c.alpha * c.alpha;
      for (int t = 0; t < T; ++t) dsmr_win_init(win[t]);
      std::vector<double> accl(T / 32, 0.0), accm(T / 32, 0.0);
      for (int r = 0; r < nrows; ++r) {
        int gj = j0 - 1 + r; gj = gj < 0 ? gj + c.ny : (gj >= c.ny ? gj - c.ny : gj);
        double* buf = sh.data() + (r & 1) * DSMC_NB * T;
        for (int t = 0; t < T; ++t) {
          const int gw = (((i0 - 1 + t) % c.nx) + c.nx) % c.nx;
          dsmr_base(c, u, v, w, gw, gj, k, &breg[(size_t)t * DSMC_NB]);
          for (int q = 0; q < DSMC_NB; ++q) buf[q * T + t] = breg[(size_t)t * DSMC_NB + q];
        }
        std::vector<double> wl(T / 32, 0.0), wm(T / 32, 0.0);
        for (int t = 0; t < T; ++t) {
          double lm = 0.0, mm = 0.0;
          const bool inner = t >= 1 && t <= T - 2, emit = r >= 2;
          if (inner) {
            if (r & 1) dsmr_row<1>(buf, T, t, &breg[(size_t)t * DSMC_NB], win[t], emit, d2, a2, &lm, &mm);
            else dsmr_row<0>(buf, T, t, &breg[(size_t)t * DSMC_NB], win[t], emit, d2, a2, &lm, &mm);
          }
          const int gi = i0 - 1 + t;
          if (emit && inner && gi < c.nx) { s->smag[idx3(c, gi, j0 + r - 2, k)] = win[t].smag_prev; wl[t >> 5] += lm; wm[t >> 5] += mm; }
          win[t].smag_prev = breg[(size_t)t * DSMC_NB + 9];
        }
        if (r >= 2) for (int wq = 0; wq < T / 32; ++wq) {
          const long long slot = ((long long)k * c.ny + (j0 + r - 2)) * ntx + bx * (T / 32) + wq;
          if (c.dsm_plane) { accl[wq] += wl[wq]; accm[wq] += wm[wq]; s->dsm_part[slot * 2] = 0.0; s->dsm_part[slot * 2 + 1] = 0.0; }
          else { s->dsm_part[slot * 2] = wl[wq]; s->dsm_part[slot * 2 + 1] = wm[wq]; }
        }
      }
      if (c.dsm_plane) for (int wq = 0; wq < T / 32; ++wq) {
        const long long slot = ((long long)k * c.ny + j0) * ntx + bx * (T / 32) + wq;
        s->dsm_part[slot * 2] = accl[wq]; s->dsm_part[slot * 2 + 1] = accm[wq];
      }
    }
  }
  for (int k = 0; k < c.nz; ++k) {
    double pl = 0.0, pm = 0.0;
    for (int j = 0; j < c.ny; ++j) {
      double ll, mm;
      dsm_row_sums(s->dsm_part.data(), ntx, (long long)k * c.ny + j, &ll, &mm);
      if (!c.dsm_plane) s->dsm_cs[(long long)k * c.ny + j] = (mm > 0.0) ? ll / mm : 0.0;
      pl += ll; pm += mm;
    }
    if (c.dsm_plane) s->dsm_cs[k] = (pm > 0.0) ? pl / pm : 0.0;
  }
  for (int k = 0; k < c.nz; ++k) for (int j = 0; j < c.ny; ++j) for (int i = 0; i < c.nx; ++i)
    nut[idx3(c, i, j, k)] = dsm_nut_point(c, s->dsm_cs.data(), s->smag.data(), i, j, k);
}
static void emu_refresh(emu_solver* s) {
  emu_tau(s);
  emu_nut(s, s->u.data(), s->v.data(), s->w.data(), s->nut.data());
  s->fresh = true;
}
static void emu_substep(emu_solver* s, int rk, double dt) {
  const Ctx& c = s->c;
  double al, be, ga; rk3_coeffs(rk, al, be, ga);
  const bool cfr = c.const_flow_rate != 0, imp = c.implicit_z == 1;      // the fully implicit scheme (implicit_z == 2) is covered on the GPU only
  RhsArgs a;
  a.u = s->u.data(); a.v = s->v.data(); a.w = s->w.data(); a.p = s->p.data(); a.nut = s->nut.data();
  a.Ru0 = s->Ru.data(); a.Rv0 = s->Rv.data(); a.Rw0 = s->Rw.data(); a.Ru1 = s->Ru.data(); a.Rv1 = s->Rv.data(); a.Rw1 = s->Rw.data();
  a.us = s->us.data(); a.vs = s->vs.data(); a.ws = s->ws.data(); a.dt = dt; a.al = al; a.be = be; a.ga = ga; a.store_R = rk < 2 ? 1 : 0; a.sc = nullptr; a.cs = nullptr;
  double sum = 0.0;
  {  // k_rhs_tile: per CTA tile and plane, stage the three halo planes with the staging rule of the kernel (rt_elem), then
     // evaluate rhs_core through the shared-memory accessor
    std::vector<double> ring(3 * RT_NF * RT_PLANE);
    for (int j0 = 0; j0 < c.ny; j0 += RT_TY) for (int i0 = 0; i0 < c.nx; i0 += RT_TX) for (int k = 0; k < c.nz; ++k) {
      for (int d = 0; d < 3; ++d) for (int f = 0; f < RT_NF; ++f) for (int pos = 0; pos < RT_PLANE; ++pos) {
        const int ry = pos / RT_TW, rx = pos % RT_TW, gi = i0 - 1 + rx, gj = j0 - 1 + ry;
        ring[(d * RT_NF + f) * RT_PLANE + pos] = (gi <= c.nx && gj <= c.ny) ? rt_elem(c, a, f, gi, gj, k - 1 + d) : 0.0;
      }
      TileAcc q; for (int d = 0; d < 3; ++d) q.sl[d] = ring.data() + d * RT_NF * RT_PLANE;
      for (int ly = 0; ly < RT_TY; ++ly) for (int tx = 0; tx < RT_TX; ++tx) {
        const int i = i0 + tx, j = j0 + ly;
        if (i < c.nx && j < c.ny) { q.ctr = (ly + 1) * RT_TW + tx + 1; sum += rhs_core(c, a, q, i, j, k, zmet_at(c, k)) * c.dzf[k]; }
      }
    }
  }
  if (imp) {
    const double cimp = 0.5 * ga * c.nu * dt;
    cn_coefficients(c, cimp, s->cncoef.data());
    sum = 0.0;
    for (long long col = 0; col < s->nxy; ++col) {
      const int j = (int)(col / c.nx);
      sum += cn_column(c, s->cncoef.data(), c.nz, col, s->us.data());
      if (!(c.bc_y == BC_WALL && j == c.ny - 1)) cn_column(c, s->cncoef.data(), c.nz, col, s->vs.data());
      cn_column(c, s->cncoef.data() + 3 * c.nz, c.nz - 1, col, s->ws.data());
    }
  }
  if (cfr) {
    const double m = sum / ((double)c.nx * (double)c.ny * c.lz);
    s->scal[0] = c.u_bulk - m; s->scal[1] = s->scal[0] / (ga * dt); s->scal[2] = m;
  }
  DivSrc ds{s->us.data(), s->vs.data(), s->ws.data(), 1.0 / (ga * dt), nullptr};
  emu_fft_x_fwd(s, nullptr, &ds, s->W.data());
  emu_poisson_core(s);
  emu_fft_x_inv(s, s->W.data(), s->W.data());
  CorrArgs ca;
  ca.phi = s->W.data(); ca.us = s->us.data(); ca.vs = s->vs.data(); ca.ws = s->ws.data();
  ca.u = s->u.data(); ca.v = s->v.data(); ca.w = s->w.data(); ca.p = s->p.data();
  ca.shift = cfr ? s->scal : nullptr; ca.gdt = ga * dt; ca.cimp = imp ? 0.5 * ga * c.nu * dt : 0.0; ca.cxy = 0.0; ca.update_p = 1; ca.sc = nullptr;
  for (int k = 0; k < c.nz; ++k) for (int j = 0; j < c.ny; ++j) for (int i = 0; i < c.nx; ++i) correct_point(c, ca, i, j, k);
  emu_refresh(s);
}
extern "C" int emu_step(emu_solver* s, double dt) {
  if (!s->fresh) emu_refresh(s);
  for (int rk = 0; rk < 3; ++rk) emu_substep(s, rk, dt);
  return 0;
}
extern "C" int emu_poisson_solve(emu_solver* s, const double* rhs, double* phi) {
  emu_fft_x_fwd(s, rhs, nullptr, s->W.data());
  emu_poisson_core(s);
  emu_fft_x_inv(s, s->W.data(), phi);
  return 0;
}
extern "C" int emu_eddy_viscosity(emu_solver* s, const double* u, const double* v, const double* w, double* nut) {
  if (u) emu_nut(s, u, v, w, nut); else emu_nut(s, s->u.data(), s->v.data(), s->w.data(), nut);
  return 0;
}
extern "C" int emu_wall_stress(emu_solver* s, double* tau) { emu_tau(s); std::memcpy(tau, s->tau.data(), s->tau.size() * sizeof(double)); return 0; }
extern "C" int emu_get_cs(emu_solver* s, double* cs) { const size_t n = s->c.dsm_plane ? s->c.nz : (size_t)s->c.nz * s->c.ny; std::memcpy(cs, s->dsm_cs.data(), n * sizeof(double)); return 0; }
extern "C" int emu_transform(emu_solver* s, double* f, int dir, int inverse) {
  if (dir == 0) { if (inverse) emu_fft_x_inv(s, f, f); else emu_fft_x_fwd(s, f, nullptr, f); }
  else emu_fft_y(s, f, inverse);
  return 0;
}
extern "C" int emu_project(emu_solver* s) {
  const Ctx& c = s->c;
  DivSrc ds{s->u.data(), s->v.data(), s->w.data(), 1.0, nullptr};
  emu_fft_x_fwd(s, nullptr, &ds, s->W.data());
  emu_poisson_core(s);
  emu_fft_x_inv(s, s->W.data(), s->W.data());
  CorrArgs ca;
  ca.phi = s->W.data(); ca.us = s->u.data(); ca.vs = s->v.data(); ca.ws = s->w.data();
  ca.u = s->u.data(); ca.v = s->v.data(); ca.w = s->w.data(); ca.p = s->p.data();
  ca.shift = nullptr; ca.gdt = 1.0; ca.cimp = 0.0; ca.cxy = 0.0; ca.update_p = 0; ca.sc = nullptr;
  for (int k = 0; k < c.nz; ++k) for (int j = 0; j < c.ny; ++j) for (int i = 0; i < c.nx; ++i) correct_point(c, ca, i, j, k);
  s->fresh = false;
  return 0;
}
extern "C" double emu_max_div(emu_solver* s) {
  const Ctx& c = s->c; double md = 0.0;
  for (int k = 0; k < c.nz; ++k) for (int j = 0; j < c.ny; ++j) for (int i = 0; i < c.nx; ++i)
    md = std::fmax(md, std::fabs(divergence_point(c, s->u.data(), s->v.data(), s->w.data(), i, j, k)));
  return md;
}
extern "C" double emu_cfl_dt(emu_solver* s, double cfl) {
  const Ctx& c = s->c; double r = 0.0;
  for (int k = 0; k < c.nz; ++k) for (int j = 0; j < c.ny; ++j) for (int i = 0; i < c.nx; ++i)
    r = std::fmax(r, cfl_rate_point(c, s->u.data(), s->v.data(), s->w.data(), i, j, k));
  return r > 0.0 ? cfl / r : 0.0;
}
extern "C" int emu_plane_stats(emu_solver* s, double* out) {
  const Ctx& c = s->c;
  for (int k = 0; k < c.nz; ++k) {
    double a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (long long n = 0; n < c.nxy; ++n) {
      double q[8]; stats_point(c, s->u.data(), s->v.data(), s->w.data(), s->nut.data(), (int)(n % c.nx), (int)(n / c.nx), k, q);
      for (int m = 0; m < 8; ++m) a[m] += q[m];
    }
    for (int m = 0; m < 8; ++m) out[(long long)m * c.nz + k] = a[m] / (double)c.nxy;
  }
  return 0;
}
extern "C" int emu_wall_stress_y(emu_solver* s, double* tau) { emu_tau(s); std::memcpy(tau, s->tau_y.data(), s->tau_y.size() * sizeof(double)); return 0; }
