// cales_oracle.cpp -- CPU ORACLE of the CaLES hot path (arXiv 2411.09364).  TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, step-by-step statement of one low-storage RK3 step of the paper's incompressible
// staggered-grid LES (Alg. 1; Alg. 2), written the
// plain way: explicit ghost layers, one loop nest per term, a separate array for every intermediate,
// no fusion, fp64, no fast-math.  OpenMP "parallel for" over k-planes / line batches only.
// It shares no code with the CUDA library.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load it.
//
// Axis convention: solver convention: z is the (possibly stretched) wall-normal / Thomas
// direction.  Paper-y == our z, paper L_22 == our L_zz.
//
// Where the paper is silent/garbled the readings S1..S23 of DESIGN.md are taken; each use is marked.
//
// PARITY UNPINNED: the *combination* of wall model + SGS near the wall (S7 and the
// one-sided strain), the van Driest u_tau choice (S5), the filter treatment at duct y-walls (S11) and the
// forcing mechanism (S12) are readings pinned only by their own invariants, not by numbers in the paper.
#include "cales_oracle.h"
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
static const double PI = 3.14159265358979323846264338327950288;
static thread_local std::string g_err;
static int fail(const char* m) { g_err = m; return 1; }
extern "C" const char* oracle_last_error(void) { return g_err.c_str(); }
extern "C" int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ------------------------------------------------------------------------------------------------
// RK3 coefficients: alpha = (8/15, 5/12, 3/4), beta = (0, -17/60, -5/12), gamma = alpha+beta
// ------------------------------------------------------------------------------------------------
extern "C" void oracle_rk3_coeffs(int k, double* alpha, double* beta, double* gamma) {
  const double al[3] = {8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0};
  const double be[3] = {0.0, -17.0 / 60.0, -5.0 / 12.0};
  *alpha = al[k]; *beta = be[k]; *gamma = al[k] + be[k];
}

// ------------------------------------------------------------------------------------------------
// 1-D transforms.  Recursive decimation-in-time Cooley-Tukey with radices 2 and 3 and a plain O(r^2)
// DFT for any other prime factor.  (The paper uses cuFFT; the transform itself is the
// textbook DFT, which the tests pin against the O(N^2) definition and numpy.)
// ------------------------------------------------------------------------------------------------
static void fft_rec(int n, int stride, const cd* in, cd* out, const cd* tw, int tws, int N) {
  if (n == 1) { out[0] = in[0]; return; }
  int r = (n % 2 == 0) ? 2 : (n % 3 == 0) ? 3 : n;
  if (r == n) {  // prime length: definition
    for (int k = 0; k < n; ++k) {
      cd s = 0;
      for (int j = 0; j < n; ++j) s += in[j * stride] * tw[(int)(((long long)j * k * tws) % N)];
      out[k] = s;
    }
    return;
  }
  int m = n / r;
  for (int q = 0; q < r; ++q) fft_rec(m, stride * r, in + q * stride, out + q * m, tw, tws * r, N);
  cd t[3];
  for (int k = 0; k < m; ++k) {
    for (int q = 0; q < r; ++q) t[q] = out[q * m + k] * tw[(int)(((long long)q * k * tws) % N)];
    for (int s = 0; s < r; ++s) {
      cd acc = 0;
      for (int q = 0; q < r; ++q) acc += t[q] * tw[(int)(((long long)q * s * m * tws) % N)];
      out[k + m * s] = acc;
    }
  }
}
struct FftPlan {
  int n; std::vector<cd> twf, twb;  // exp(-/+ 2 pi i k / n)
  explicit FftPlan(int n_) : n(n_), twf(n_), twb(n_) {
    for (int k = 0; k < n; ++k) {
      double a = 2.0 * PI * (double)k / (double)n;
      twf[k] = cd(std::cos(a), -std::sin(a)); twb[k] = cd(std::cos(a), std::sin(a));
    }
  }
  void run(const cd* in, cd* out, int sign) const { fft_rec(n, 1, in, out, sign < 0 ? twf.data() : twb.data(), 1, n); }
};
extern "C" int oracle_fft_c2c(int n, const double* re_in, const double* im_in, double* re_out, double* im_out, int sign) {
  if (n < 1) return fail("fft: n<1");
  FftPlan pl(n); std::vector<cd> a(n), b(n);
  for (int i = 0; i < n; ++i) a[i] = cd(re_in[i], im_in ? im_in[i] : 0.0);
  pl.run(a.data(), b.data(), sign);
  for (int i = 0; i < n; ++i) { re_out[i] = b[i].real(); im_out[i] = b[i].imag(); }
  return 0;
}
// DCT-II by the 2N-point FFT of the even extension y = [x, reverse(x)]:
//   Y[n] = e^{i pi n/(2N)} * 2 sum_j x[j] cos(pi n (2j+1)/(2N))  =>  X[n] = Re(e^{-i pi n/(2N)} Y[n]) / 2.
struct DctPlan {
  int n; FftPlan f2;
  explicit DctPlan(int n_) : n(n_), f2(2 * n_) {}
  void dct2(const double* x, double* X) const {
    std::vector<cd> y(2 * n), Y(2 * n);
    for (int j = 0; j < n; ++j) { y[j] = x[j]; y[2 * n - 1 - j] = x[j]; }
    f2.run(y.data(), Y.data(), -1);
    for (int k = 0; k < n; ++k) {
      double a = PI * (double)k / (2.0 * n);
      X[k] = 0.5 * (cd(std::cos(a), -std::sin(a)) * Y[k]).real();
    }
  }
  // inverse: rebuild the Hermitian 2N spectrum, inverse FFT, keep the first N samples.
  void dct3(const double* X, double* x) const {
    std::vector<cd> Y(2 * n), y(2 * n);
    for (int k = 0; k < n; ++k) {
      double a = PI * (double)k / (2.0 * n);
      Y[k] = 2.0 * X[k] * cd(std::cos(a), std::sin(a));
    }
    Y[n] = 0.0;
    for (int k = 1; k < n; ++k) Y[2 * n - k] = std::conj(Y[k]);
    f2.run(Y.data(), y.data(), +1);
    for (int j = 0; j < n; ++j) x[j] = y[j].real() / (2.0 * n);
  }
};
extern "C" int oracle_dct2(int n, const double* x, double* X) { if (n < 1) return fail("dct: n<1"); DctPlan(n).dct2(x, X); return 0; }
extern "C" int oracle_dct3(int n, const double* X, double* x) { if (n < 1) return fail("dct: n<1"); DctPlan(n).dct3(X, x); return 0; }

// ------------------------------------------------------------------------------------------------
// Thomas algorithm and its cyclic variant (Sherman-Morrison), textbook form.
// ------------------------------------------------------------------------------------------------
extern "C" int oracle_thomas(int n, const double* a, const double* b, const double* c, const double* d, double* x) {
  if (n < 1) return fail("thomas: n<1");
  std::vector<double> cp(n), dp(n);
  cp[0] = c[0] / b[0]; dp[0] = d[0] / b[0];
  for (int k = 1; k < n; ++k) {
    double den = b[k] - a[k] * cp[k - 1];
    cp[k] = c[k] / den; dp[k] = (d[k] - a[k] * dp[k - 1]) / den;
  }
  x[n - 1] = dp[n - 1];
  for (int k = n - 2; k >= 0; --k) x[k] = dp[k] - cp[k] * x[k + 1];
  return 0;
}
extern "C" int oracle_thomas_cyclic(int n, const double* a, const double* b, const double* c, const double* d, double* x) {
  if (n < 3) return fail("cyclic thomas: n<3");
  // A = T + u v^T with u = (g,0,..,0,c[n-1])^T, v = (1,0,..,0,a[0]/g)^T, g = -b[0]
  double g = -b[0];
  std::vector<double> bb(b, b + n), uu(n, 0.0), y(n), q(n);
  bb[0] = b[0] - g; bb[n - 1] = b[n - 1] - a[0] * c[n - 1] / g;
  uu[0] = g; uu[n - 1] = c[n - 1];
  oracle_thomas(n, a, bb.data(), c, d, y.data());
  oracle_thomas(n, a, bb.data(), c, uu.data(), q.data());
  double vy = y[0] + a[0] * y[n - 1] / g, vq = q[0] + a[0] * q[n - 1] / g;
  double f = vy / (1.0 + vq);
  for (int k = 0; k < n; ++k) x[k] = y[k] - f * q[k];
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Log law, Eq. 10: U/u_tau = ln(u_tau h/nu)/kappa + B.  Newton-Raphson on
// s = ln(h+), h+ = u_tau h/nu (reading S8):  g(s) = Re e^{-s} - s/kappa - B, Re = U h/nu, s_0 = ln(Re)/2.
// Stop when the relative change of tau_w = u_tau^2, |e^{2(s_new-s_old)} - 1|, is below tol (PAPER.md:130:
// 0.01 %), then take ONE more Newton update (reading S9).
// ------------------------------------------------------------------------------------------------
extern "C" double oracle_loglaw_hplus(double re_wm, double kappa, double B, double tol, int maxit, int* iters) {
  if (iters) *iters = 0;
  if (!(re_wm > 0.0)) return 0.0;  // reading S10
  double s = 0.5 * std::log(re_wm);
  int it = 0; bool polish = false;
  while (it < maxit) {
    double e = re_wm * std::exp(-s);
    double g = e - s / kappa - B;
    double dg = -e - 1.0 / kappa;
    double sn = s - g / dg;
    ++it;
    double rel = std::fabs(std::exp(2.0 * (sn - s)) - 1.0);
    s = sn;
    if (polish) break;
    if (rel < tol) polish = true;
  }
  if (iters) *iters = it;
  return std::exp(s);
}

// ------------------------------------------------------------------------------------------------
// Ghosted 3-D array: interior 0..n-1 plus one ghost layer on every side.
// ------------------------------------------------------------------------------------------------
struct F3 {
  int nx = 0, ny = 0, nz = 0; std::vector<double> a;
  F3() {}
  F3(int x, int y, int z) : nx(x), ny(y), nz(z), a((size_t)(x + 2) * (y + 2) * (z + 2), 0.0) {}
  inline double& operator()(int i, int j, int k) { return a[(size_t)(i + 1) + (size_t)(nx + 2) * ((size_t)(j + 1) + (size_t)(ny + 2) * (size_t)(k + 1))]; }
  inline double operator()(int i, int j, int k) const { return a[(size_t)(i + 1) + (size_t)(nx + 2) * ((size_t)(j + 1) + (size_t)(ny + 2) * (size_t)(k + 1))]; }
  void from(const double* src) {
#pragma omp parallel for
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) (*this)(i, j, k) = src[i + (size_t)nx * (j + (size_t)ny * k)];
  }
  void to(double* dst) const {
#pragma omp parallel for
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) dst[i + (size_t)nx * (j + (size_t)ny * k)] = (*this)(i, j, k);
  }
};

enum { BC_PER = 0, BC_WALL = 1 };
enum { GH_VISC = 0, GH_STRAIN = 1 };   // which ghost the wall-model walls get
enum { SC_NEUMANN = 0, SC_NEG = 1 };

struct oracle_solver {
  oracle_params P;
  int nx, ny, nz; size_t N;
  double dx, dy;
  std::vector<double> zf, zc, dzf_, dzc_;     // dzf_[k+1] = dzf[k], k=-1..nz ; dzc_[k+1] = dzc[k], k=-1..nz-1
  inline double dzf(int k) const { return dzf_[k + 1]; }
  inline double dzc(int k) const { return dzc_[k + 1]; }
  F3 u, v, w, p, nut;
  std::vector<double> Ru, Rv, Rw;             // R^{k-1}
  std::vector<double> tau;                    // [wall][comp][ny][nx]
  std::vector<double> tauy;                   // y walls: [wall][comp (0 tau_xy at u points, 1 tau_zy at w points)][nz][nx]
  std::vector<double> cs;                     // dynamic coefficient per k or per (k,j)
  std::vector<double> Lij, Mij;               // tensors of the last dynamic evaluation (for the pins)
  std::vector<double> st_prof, st_wall; double st_weight = 0.0;   // time accumulators of the on-line statistics
  std::vector<double> ust, vst, wst;          // u*, v*, w* of the last substep, after O-step 6, before the bulk shift (for the pins)
  bool fresh = false;                         // wall stress + nu_t consistent with the velocity
  double forcing = 0.0; int wm_max_iters = 0;
  double alpha2d;
  FftPlan* plx = nullptr; FftPlan* ply = nullptr; DctPlan* pdy = nullptr;
  ~oracle_solver() { delete plx; delete ply; delete pdy; }
  inline size_t id(int i, int j, int k) const { return (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k); }
  inline double& tw(int wall, int comp, int i, int j) { return tau[((size_t)(wall * 2 + comp) * ny + j) * nx + i]; }
  // y-wall stress seen from any (i,k) incl. ghosts: i periodic, k clamped to the interior
  inline double& twy(int wall, int comp, int i, int k) {
    int ii = i < 0 ? i + nx : (i >= nx ? i - nx : i), kk = k < 0 ? 0 : (k >= nz ? nz - 1 : k);
    return tauy[((size_t)(wall * 2 + comp) * nz + kk) * nx + ii];
  }
};

// ------------------------------------------------------------------------------------------------
// Boundary conditions (Alg. 2; O-step 1 of DESIGN.md).
// Fill order z, x, y so that edge ghosts are consistent.
// ------------------------------------------------------------------------------------------------
static void wrap_x(F3& q) {
  int nx = q.nx;
  for (int k = -1; k <= q.nz; ++k) for (int j = 0; j < q.ny; ++j) { q(-1, j, k) = q(nx - 1, j, k); q(nx, j, k) = q(0, j, k); }
}
static void wrap_y(F3& q) {
  int ny = q.ny;
  for (int k = -1; k <= q.nz; ++k) for (int i = -1; i <= q.nx; ++i) { q(i, -1, k) = q(i, ny - 1, k); q(i, ny, k) = q(i, 0, k); }
}
static void mirror_y(F3& q, double sgn) {
  int ny = q.ny;
  for (int k = -1; k <= q.nz; ++k) for (int i = -1; i <= q.nx; ++i) { q(i, -1, k) = sgn * q(i, 0, k); q(i, ny, k) = sgn * q(i, ny - 1, k); }
}
static void bc_scalar(const oracle_solver& S, F3& q, int kind) {
  double sgn = (kind == SC_NEUMANN) ? 1.0 : -1.0;   // Neumann for p, phi; nu_t ghost = -interior at walls (reading S7)
  int nz = S.nz;
  for (int j = 0; j < S.ny; ++j) for (int i = 0; i < S.nx; ++i) {
    if (S.P.bc_z == BC_PER) { q(i, j, -1) = q(i, j, nz - 1); q(i, j, nz) = q(i, j, 0); }
    else { q(i, j, -1) = sgn * q(i, j, 0); q(i, j, nz) = sgn * q(i, j, nz - 1); }
  }
  wrap_x(q);
  if (S.P.bc_y == BC_PER) wrap_y(q); else mirror_y(q, sgn);
}
// velocity ghosts.  mode selects the ghost a wall-model wall gives the wall-parallel components:
//  GH_VISC   : u_g = u[0] - tau_xz * dzc[-1] / nu     (the modelled stress IS the wall viscous flux)
//  GH_STRAIN : u_g = linear extrapolation of u[0], u[1] (one-sided derivative for the strain rate)
static void bc_velocity(oracle_solver& S, F3& u, F3& v, F3& w, int mode) {
  int nx = S.nx, ny = S.ny, nz = S.nz;
  // --- z
  for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    if (S.P.bc_z == BC_PER) {
      u(i, j, -1) = u(i, j, nz - 1); u(i, j, nz) = u(i, j, 0);
      v(i, j, -1) = v(i, j, nz - 1); v(i, j, nz) = v(i, j, 0);
      w(i, j, -1) = w(i, j, nz - 1); w(i, j, nz) = w(i, j, 0);
    } else {
      w(i, j, nz - 1) = 0.0; w(i, j, -1) = 0.0; w(i, j, nz) = 0.0;   // impermeable wall faces
      if (!S.P.wall_model) {                                          // no-slip: mirror
        u(i, j, -1) = -u(i, j, 0); u(i, j, nz) = -u(i, j, nz - 1);
        v(i, j, -1) = -v(i, j, 0); v(i, j, nz) = -v(i, j, nz - 1);
      } else if (mode == GH_VISC) {
        u(i, j, -1) = u(i, j, 0) - S.tw(0, 0, i, j) * S.dzc(-1) / S.P.nu;
        v(i, j, -1) = v(i, j, 0) - S.tw(0, 1, i, j) * S.dzc(-1) / S.P.nu;
        u(i, j, nz) = u(i, j, nz - 1) - S.tw(1, 0, i, j) * S.dzc(nz - 1) / S.P.nu;
        v(i, j, nz) = v(i, j, nz - 1) - S.tw(1, 1, i, j) * S.dzc(nz - 1) / S.P.nu;
      } else {
        u(i, j, -1) = u(i, j, 0) - (u(i, j, 1) - u(i, j, 0)) * S.dzc(-1) / S.dzc(0);
        v(i, j, -1) = v(i, j, 0) - (v(i, j, 1) - v(i, j, 0)) * S.dzc(-1) / S.dzc(0);
        u(i, j, nz) = u(i, j, nz - 1) + (u(i, j, nz - 1) - u(i, j, nz - 2)) * S.dzc(nz - 1) / S.dzc(nz - 2);
        v(i, j, nz) = v(i, j, nz - 1) + (v(i, j, nz - 1) - v(i, j, nz - 2)) * S.dzc(nz - 1) / S.dzc(nz - 2);
      }
    }
  }
  // --- x (always periodic)
  wrap_x(u); wrap_x(v); wrap_x(w);
  // --- y
  if (S.P.bc_y == BC_PER) { wrap_y(u); wrap_y(v); wrap_y(w); }
  else {
    if (!S.P.wall_model_y) { mirror_y(u, -1.0); mirror_y(w, -1.0); }
    else {
      // SURVEY.md 8(f) item 1 (duct WMLES): the y walls carry the wall model too; same two ghost kinds as in z,
      // with the uniform spacing dy (ghost centre mirrored at distance dy from the first centre)
      const double dy = S.dy, nu = S.P.nu;
      for (int k = -1; k <= nz; ++k) for (int i = -1; i <= nx; ++i) {
        if (mode == GH_VISC) {
          u(i, -1, k) = u(i, 0, k) - S.twy(0, 0, i, k) * dy / nu; u(i, ny, k) = u(i, ny - 1, k) - S.twy(1, 0, i, k) * dy / nu;
          w(i, -1, k) = w(i, 0, k) - S.twy(0, 1, i, k) * dy / nu; w(i, ny, k) = w(i, ny - 1, k) - S.twy(1, 1, i, k) * dy / nu;
        } else {
          u(i, -1, k) = 2.0 * u(i, 0, k) - u(i, 1, k); u(i, ny, k) = 2.0 * u(i, ny - 1, k) - u(i, ny - 2, k);
          w(i, -1, k) = 2.0 * w(i, 0, k) - w(i, 1, k); w(i, ny, k) = 2.0 * w(i, ny - 1, k) - w(i, ny - 2, k);
        }
      }
    }
    for (int k = -1; k <= nz; ++k) for (int i = -1; i <= nx; ++i) { v(i, ny - 1, k) = 0.0; v(i, -1, k) = 0.0; v(i, ny, k) = 0.0; }
  }
}

// ------------------------------------------------------------------------------------------------
// Wall model (Eq. 10, 130, Fig. 1; O-step 8).  For each modelled wall and each u-point:
// u_wm = u interpolated linearly in z to h_wm, v_wm = the 4 surrounding v-points averaged to the u-point
// (each interpolated to h_wm), U = sqrt(u_wm^2+v_wm^2), Newton for u_tau, tau_xz = u_tau^2 u_wm / U.
// Same at v-points with u interpolated -> tau_yz.  Needs x/y ghosts of u, v (call after bc_velocity).
// ------------------------------------------------------------------------------------------------
// y walls (duct WMLES): sampled at h_wm from the wall, linear interpolation between the two bracketing centres as in z
// (default: the first off-wall centre, h = dy/2).  tau_xy at the u points (i+1/2, k) from u and the
// 4 surrounding w points; tau_zy at the w points (i, k+1/2) from w and the 4 surrounding u points.
static void wall_stress_y(oracle_solver& S, int& maxit) {
  int nx = S.nx, ny = S.ny, nz = S.nz;
  auto dist = [&](int q) { return (q + 0.5) * S.dy; };        // centre number q counted from the wall
  const double h = S.P.h_wm > 0.0 ? S.P.h_wm : dist(0);
  int q1 = 0; while (q1 + 2 < ny / 2 && dist(q1 + 1) <= h) ++q1;
  const double wgt = (h - dist(q1)) / (dist(q1 + 1) - dist(q1));
  for (int wall = 0; wall < 2; ++wall) {
    const int ja = wall == 0 ? q1 : ny - 1 - q1, jb = wall == 0 ? q1 + 1 : ny - 2 - q1;
    auto at = [&](const F3& q, int ii, int kk) { return (1.0 - wgt) * q(ii, ja, kk) + wgt * q(ii, jb, kk); };
    for (int k = 0; k < nz; ++k) for (int i = 0; i < nx; ++i) for (int comp = 0; comp < 2; ++comp) {
      double a, b;
      if (comp == 0) { a = at(S.u, i, k); b = 0.25 * (at(S.w, i, k) + at(S.w, i + 1, k) + at(S.w, i, k - 1) + at(S.w, i + 1, k - 1)); }
      else { a = at(S.w, i, k); b = 0.25 * (at(S.u, i, k) + at(S.u, i - 1, k) + at(S.u, i, k + 1) + at(S.u, i - 1, k + 1)); }
      double U = std::sqrt(a * a + b * b), t = 0.0;
      if (U > 0.0) {
        int it = 0;
        double hp = oracle_loglaw_hplus(U * h / S.P.nu, S.P.kappa, S.P.B, S.P.wm_tol, S.P.wm_maxit, &it);
        double utau = hp * S.P.nu / h;
        t = utau * utau * a / U;
        if (it > maxit) maxit = it;
      }
      S.tauy[((size_t)(wall * 2 + comp) * nz + k) * nx + i] = t;
    }
  }
}
static void wall_stress(oracle_solver& S) {
  int maxit = 0;
  if (S.P.wall_model_y) wall_stress_y(S, maxit);
  if (!S.P.wall_model) { if (S.P.wall_model_y) S.wm_max_iters = maxit; return; }
  int nx = S.nx, ny = S.ny, nz = S.nz;
  for (int wall = 0; wall < 2; ++wall) {
    // distance of centre number q (counted from this wall) to the wall
    auto dist = [&](int q) { return wall == 0 ? S.zc[q] : S.P.lz - S.zc[nz - 1 - q]; };
    double h = S.P.h_wm > 0.0 ? S.P.h_wm : dist(0);          // reading S21: default = first off-wall centre
    int q1 = 0; while (q1 + 2 < nz / 2 && dist(q1 + 1) <= h) ++q1;   // bracketing centres: dist(q1) <= h <= dist(q1+1)
    double wgt = (h - dist(q1)) / (dist(q1 + 1) - dist(q1));  // linear interpolation between locations 1 and 2
    int ka = wall == 0 ? q1 : nz - 1 - q1, kb = wall == 0 ? q1 + 1 : nz - 2 - q1;
#pragma omp parallel for reduction(max : maxit)
    for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
      auto at = [&](const F3& q, int ii, int jj) { return (1.0 - wgt) * q(ii, jj, ka) + wgt * q(ii, jj, kb); };
      for (int comp = 0; comp < 2; ++comp) {
        double a, b;  // a = own component at its point, b = the other component interpolated to it
        if (comp == 0) { a = at(S.u, i, j); b = 0.25 * (at(S.v, i, j) + at(S.v, i + 1, j) + at(S.v, i, j - 1) + at(S.v, i + 1, j - 1)); }
        else { a = at(S.v, i, j); b = 0.25 * (at(S.u, i, j) + at(S.u, i - 1, j) + at(S.u, i, j + 1) + at(S.u, i - 1, j + 1)); }
        double U = std::sqrt(a * a + b * b);
        double t = 0.0;
        if (U > 0.0) {
          int it = 0;
          double hp = oracle_loglaw_hplus(U * h / S.P.nu, S.P.kappa, S.P.B, S.P.wm_tol, S.P.wm_maxit, &it);
          double utau = hp * S.P.nu / h;
          t = utau * utau * a / U;
          if (it > maxit) maxit = it;
        }
        S.tw(wall, comp, i, j) = t;
      }
    }
  }
  S.wm_max_iters = maxit;
}

// ------------------------------------------------------------------------------------------------
// Explicit terms (O-steps 2-4).  Inputs ghosted; outputs interior arrays.
// ------------------------------------------------------------------------------------------------
// -d_j(u_i u_j), divergence form, Harlow-Welch (PAPER.md:38, 88, 102 with sign reading S1; weights reading S3)
static void advection(const oracle_solver& S, const F3& u, const F3& v, const F3& w, double* au, double* av, double* aw) {
  int nx = S.nx, ny = S.ny, nz = S.nz; double dx = S.dx, dy = S.dy;
  int kwmax = (S.P.bc_z == BC_WALL) ? nz - 1 : nz;   // w faces that are unknowns
  int jvmax = (S.P.bc_y == BC_WALL) ? ny - 1 : ny;
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    // ---- u at (i+1/2, j, k)
    {
      double uxp = 0.5 * (u(i, j, k) + u(i + 1, j, k)), uxm = 0.5 * (u(i - 1, j, k) + u(i, j, k));      // u at centres i+1, i
      double uyp = 0.5 * (u(i, j, k) + u(i, j + 1, k)), uym = 0.5 * (u(i, j - 1, k) + u(i, j, k));      // u at edges j+-1/2
      double vxp = 0.5 * (v(i, j, k) + v(i + 1, j, k)), vxm = 0.5 * (v(i, j - 1, k) + v(i + 1, j - 1, k));
      double uzp = 0.5 * (u(i, j, k) + u(i, j, k + 1)), uzm = 0.5 * (u(i, j, k - 1) + u(i, j, k));      // u at edges k+-1/2
      double wxp = 0.5 * (w(i, j, k) + w(i + 1, j, k)), wxm = 0.5 * (w(i, j, k - 1) + w(i + 1, j, k - 1));
      au[S.id(i, j, k)] = -((uxp * uxp - uxm * uxm) / dx + (uyp * vxp - uym * vxm) / dy + (uzp * wxp - uzm * wxm) / S.dzf(k));
    }
    // ---- v at (i, j+1/2, k)
    if (j < jvmax) {
      double vyp = 0.5 * (v(i, j, k) + v(i, j + 1, k)), vym = 0.5 * (v(i, j - 1, k) + v(i, j, k));
      double vxp = 0.5 * (v(i, j, k) + v(i + 1, j, k)), vxm = 0.5 * (v(i - 1, j, k) + v(i, j, k));
      double uyp = 0.5 * (u(i, j, k) + u(i, j + 1, k)), uym = 0.5 * (u(i - 1, j, k) + u(i - 1, j + 1, k));
      double vzp = 0.5 * (v(i, j, k) + v(i, j, k + 1)), vzm = 0.5 * (v(i, j, k - 1) + v(i, j, k));
      double wyp = 0.5 * (w(i, j, k) + w(i, j + 1, k)), wym = 0.5 * (w(i, j, k - 1) + w(i, j + 1, k - 1));
      av[S.id(i, j, k)] = -((vxp * uyp - vxm * uym) / dx + (vyp * vyp - vym * vym) / dy + (vzp * wyp - vzm * wym) / S.dzf(k));
    } else av[S.id(i, j, k)] = 0.0;
    // ---- w at (i, j, k+1/2)
    if (k < kwmax) {
      double f0 = S.dzf(k), f1 = S.dzf(k + 1), c2 = 2.0 * S.dzc(k);
      double wzp = 0.5 * (w(i, j, k) + w(i, j, k + 1)), wzm = 0.5 * (w(i, j, k - 1) + w(i, j, k));      // w at centres k+1, k
      double wxp = 0.5 * (w(i, j, k) + w(i + 1, j, k)), wxm = 0.5 * (w(i - 1, j, k) + w(i, j, k));
      // advecting velocity: dzf-weighted mean (reading S3) so that the staggered control volume inherits continuity
      double uzp = (u(i, j, k) * f0 + u(i, j, k + 1) * f1) / c2, uzm = (u(i - 1, j, k) * f0 + u(i - 1, j, k + 1) * f1) / c2;
      double wyp = 0.5 * (w(i, j, k) + w(i, j + 1, k)), wym = 0.5 * (w(i, j - 1, k) + w(i, j, k));
      double vzp = (v(i, j, k) * f0 + v(i, j, k + 1) * f1) / c2, vzm = (v(i, j - 1, k) * f0 + v(i, j - 1, k + 1) * f1) / c2;
      aw[S.id(i, j, k)] = -((wxp * uzp - wxm * uzm) / dx + (wyp * vzp - wym * vzm) / dy + (wzp * wzp - wzm * wzm) / S.dzc(k));
    } else aw[S.id(i, j, k)] = 0.0;
  }
}
// nu * L_jj u_i (Eq. 16; reading S22).  which: 0 = all directions, 1 = x and y only, 2 = z only.
static void diffusion(const oracle_solver& S, const F3& u, const F3& v, const F3& w, double* du, double* dv, double* dw, int which) {
  int nx = S.nx, ny = S.ny, nz = S.nz; double dx = S.dx, dy = S.dy, nu = S.P.nu;
  int kwmax = (S.P.bc_z == BC_WALL) ? nz - 1 : nz, jvmax = (S.P.bc_y == BC_WALL) ? ny - 1 : ny;
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t n = S.id(i, j, k);
    double lxy, lz;
    lxy = (u(i + 1, j, k) - 2.0 * u(i, j, k) + u(i - 1, j, k)) / (dx * dx) + (u(i, j + 1, k) - 2.0 * u(i, j, k) + u(i, j - 1, k)) / (dy * dy);
    lz = ((u(i, j, k + 1) - u(i, j, k)) / S.dzc(k) - (u(i, j, k) - u(i, j, k - 1)) / S.dzc(k - 1)) / S.dzf(k);
    du[n] = nu * ((which != 2 ? lxy : 0.0) + (which != 1 ? lz : 0.0));
    if (j < jvmax) {
      lxy = (v(i + 1, j, k) - 2.0 * v(i, j, k) + v(i - 1, j, k)) / (dx * dx) + (v(i, j + 1, k) - 2.0 * v(i, j, k) + v(i, j - 1, k)) / (dy * dy);
      lz = ((v(i, j, k + 1) - v(i, j, k)) / S.dzc(k) - (v(i, j, k) - v(i, j, k - 1)) / S.dzc(k - 1)) / S.dzf(k);
      dv[n] = nu * ((which != 2 ? lxy : 0.0) + (which != 1 ? lz : 0.0));
    } else dv[n] = 0.0;
    if (k < kwmax) {
      lxy = (w(i + 1, j, k) - 2.0 * w(i, j, k) + w(i - 1, j, k)) / (dx * dx) + (w(i, j + 1, k) - 2.0 * w(i, j, k) + w(i, j - 1, k)) / (dy * dy);
      lz = ((w(i, j, k + 1) - w(i, j, k)) / S.dzf(k + 1) - (w(i, j, k) - w(i, j, k - 1)) / S.dzf(k)) / S.dzc(k);
      dw[n] = nu * ((which != 2 ? lxy : 0.0) + (which != 1 ? lz : 0.0));
    } else dw[n] = 0.0;
  }
}
// d_j(2 nu_t S_ij) (Eq. 3, 15; sign reading S1; edge viscosity = mean of the 4 surrounding centres, reading S6)
static void sgs_term(const oracle_solver& S, const F3& u, const F3& v, const F3& w, const F3& nt, double* su, double* sv, double* sw) {
  int nx = S.nx, ny = S.ny, nz = S.nz; double dx = S.dx, dy = S.dy;
  int kwmax = (S.P.bc_z == BC_WALL) ? nz - 1 : nz, jvmax = (S.P.bc_y == BC_WALL) ? ny - 1 : ny;
  // edge quantities nu_edge * (2 S_ij) at the three edge families, as lambdas of the edge's lower-left indices
  auto exy = [&](int i, int j, int k) {   // edge (i+1/2, j+1/2, k)
    double ne = 0.25 * (nt(i, j, k) + nt(i + 1, j, k) + nt(i, j + 1, k) + nt(i + 1, j + 1, k));
    return ne * ((u(i, j + 1, k) - u(i, j, k)) / dy + (v(i + 1, j, k) - v(i, j, k)) / dx);
  };
  auto exz = [&](int i, int j, int k) {   // edge (i+1/2, j, k+1/2)
    double ne = 0.25 * (nt(i, j, k) + nt(i + 1, j, k) + nt(i, j, k + 1) + nt(i + 1, j, k + 1));
    return ne * ((u(i, j, k + 1) - u(i, j, k)) / S.dzc(k) + (w(i + 1, j, k) - w(i, j, k)) / dx);
  };
  auto eyz = [&](int i, int j, int k) {   // edge (i, j+1/2, k+1/2)
    double ne = 0.25 * (nt(i, j, k) + nt(i, j + 1, k) + nt(i, j, k + 1) + nt(i, j + 1, k + 1));
    return ne * ((v(i, j, k + 1) - v(i, j, k)) / S.dzc(k) + (w(i, j + 1, k) - w(i, j, k)) / dy);
  };
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t n = S.id(i, j, k);
    su[n] = (2.0 * nt(i + 1, j, k) * (u(i + 1, j, k) - u(i, j, k)) / dx - 2.0 * nt(i, j, k) * (u(i, j, k) - u(i - 1, j, k)) / dx) / dx
          + (exy(i, j, k) - exy(i, j - 1, k)) / dy + (exz(i, j, k) - exz(i, j, k - 1)) / S.dzf(k);
    if (j < jvmax)
      sv[n] = (exy(i, j, k) - exy(i - 1, j, k)) / dx
            + (2.0 * nt(i, j + 1, k) * (v(i, j + 1, k) - v(i, j, k)) / dy - 2.0 * nt(i, j, k) * (v(i, j, k) - v(i, j - 1, k)) / dy) / dy
            + (eyz(i, j, k) - eyz(i, j, k - 1)) / S.dzf(k);
    else sv[n] = 0.0;
    if (k < kwmax)
      sw[n] = (exz(i, j, k) - exz(i - 1, j, k)) / dx + (eyz(i, j, k) - eyz(i, j - 1, k)) / dy
            + (2.0 * nt(i, j, k + 1) * (w(i, j, k + 1) - w(i, j, k)) / S.dzf(k + 1) - 2.0 * nt(i, j, k) * (w(i, j, k) - w(i, j, k - 1)) / S.dzf(k)) / S.dzc(k);
    else sw[n] = 0.0;
  }
}
static void divergence(const oracle_solver& S, const F3& u, const F3& v, const F3& w, double* d) {
#pragma omp parallel for
  for (int k = 0; k < S.nz; ++k) for (int j = 0; j < S.ny; ++j) for (int i = 0; i < S.nx; ++i)
    d[S.id(i, j, k)] = (u(i, j, k) - u(i - 1, j, k)) / S.dx + (v(i, j, k) - v(i, j - 1, k)) / S.dy + (w(i, j, k) - w(i, j, k - 1)) / S.dzf(k);
}

// ------------------------------------------------------------------------------------------------
// Poisson solver by eigenfunction expansion (ref. [28]; O-step 7): DFT along x, DFT (periodic)
// or DCT-II (Neumann) along y, tridiagonal solve along z for every (m, n).  The full complex spectrum is
// kept (no half-complex packing) -- plain, not fast.
// ------------------------------------------------------------------------------------------------
static double lam_x(const oracle_solver& S, int m) { double s = std::sin(PI * m / (double)S.nx); return -4.0 / (S.dx * S.dx) * s * s; }
static double lam_y(const oracle_solver& S, int n) {
  double s = (S.P.bc_y == BC_PER) ? std::sin(PI * n / (double)S.ny) : std::sin(PI * n / (2.0 * S.ny));
  return -4.0 / (S.dy * S.dy) * s * s;
}
// z system of the Poisson equation for mode (i, j): a_k phi[k-1] + b_k phi[k] + c_k phi[k+1] = f, a_k = 1/(dzf[k] dzc[k-1]),
// c_k = 1/(dzf[k] dzc[k]), b_k = -(a_k + c_k) + lam_x + lam_y; Neumann: a_0, c_{nz-1} dropped from b; periodic z: cyclic.
static void poisson_zsolve(const oracle_solver& S, int i, int j, double* dr, double* di) {
  int nz = S.nz;
  std::vector<double> a(nz), b(nz), c(nz), xr(nz), xi(nz);
  double lam = lam_x(S, i) + lam_y(S, j);
  for (int k = 0; k < nz; ++k) {
    a[k] = 1.0 / (S.dzf(k) * S.dzc(k - 1)); c[k] = 1.0 / (S.dzf(k) * S.dzc(k));
    double aa = a[k], cc = c[k];
    if (S.P.bc_z == BC_WALL) { if (k == 0) aa = 0.0; if (k == nz - 1) cc = 0.0; }
    b[k] = -(aa + cc) + lam;
  }
  bool cyclic = (S.P.bc_z == BC_PER);
  if (i == 0 && j == 0) {
    // singular zero mode (reading S15): drop the dzf-weighted mean of f, pin phi[0] = 0, solve, then
    // shift to zero dzf-weighted mean.
    double mr = 0, mi = 0;
    for (int k = 0; k < nz; ++k) { mr += dr[k] * S.dzf(k); mi += di[k] * S.dzf(k); }
    mr /= S.P.lz; mi /= S.P.lz;
    for (int k = 0; k < nz; ++k) { dr[k] -= mr; di[k] -= mi; }
    b[0] = 1.0; c[0] = 0.0; dr[0] = 0.0; di[0] = 0.0;   // row 0: phi[0] = 0 (this also breaks the cycle)
    oracle_thomas(nz, a.data(), b.data(), c.data(), dr, xr.data());
    oracle_thomas(nz, a.data(), b.data(), c.data(), di, xi.data());
    double sr = 0, si = 0;
    for (int k = 0; k < nz; ++k) { sr += xr[k] * S.dzf(k); si += xi[k] * S.dzf(k); }
    sr /= S.P.lz; si /= S.P.lz;
    for (int k = 0; k < nz; ++k) { xr[k] -= sr; xi[k] -= si; }
  } else if (cyclic) {
    oracle_thomas_cyclic(nz, a.data(), b.data(), c.data(), dr, xr.data());
    oracle_thomas_cyclic(nz, a.data(), b.data(), c.data(), di, xi.data());
  } else {
    oracle_thomas(nz, a.data(), b.data(), c.data(), dr, xr.data());
    oracle_thomas(nz, a.data(), b.data(), c.data(), di, xi.data());
  }
  for (int k = 0; k < nz; ++k) { dr[k] = xr[k]; di[k] = xi[k]; }
}
// The transform scaffold shared by the Poisson solve (Eq. 12) and the Helmholtz solves of Eq. 18: forward DFT along x, forward
// DFT / DCT-II along y, zsolve(i, j, re[nz], im[nz]) overwrites the z column of mode (i, j) with its solution, inverse y, inverse x.
template <class ZSolve>
static void eigen_expansion_solve(const oracle_solver& S, const double* rhs, double* phi, ZSolve zsolve) {
  int nx = S.nx, ny = S.ny, nz = S.nz;
  std::vector<cd> A(S.N);
  // forward x
#pragma omp parallel
  {
    std::vector<cd> a(nx), b(nx);
#pragma omp for
    for (int l = 0; l < ny * nz; ++l) {
      for (int i = 0; i < nx; ++i) a[i] = rhs[(size_t)l * nx + i];
      S.plx->run(a.data(), b.data(), -1);
      for (int i = 0; i < nx; ++i) A[(size_t)l * nx + i] = b[i];
    }
  }
  // forward y
#pragma omp parallel
  {
    std::vector<cd> a(ny), b(ny); std::vector<double> r(ny), q(ny), R(ny), Q(ny);
#pragma omp for
    for (int l = 0; l < nx * nz; ++l) {
      int i = l % nx, k = l / nx;
      if (S.P.bc_y == BC_PER) {
        for (int j = 0; j < ny; ++j) a[j] = A[S.id(i, j, k)];
        S.ply->run(a.data(), b.data(), -1);
        for (int j = 0; j < ny; ++j) A[S.id(i, j, k)] = b[j];
      } else {
        for (int j = 0; j < ny; ++j) { r[j] = A[S.id(i, j, k)].real(); q[j] = A[S.id(i, j, k)].imag(); }
        S.pdy->dct2(r.data(), R.data()); S.pdy->dct2(q.data(), Q.data());
        for (int j = 0; j < ny; ++j) A[S.id(i, j, k)] = cd(R[j], Q[j]);
      }
    }
  }
  // z: one tridiagonal system per mode (i, j), real and imaginary parts share the matrix
#pragma omp parallel
  {
    std::vector<double> dr(nz), di(nz);
#pragma omp for
    for (int l = 0; l < nx * ny; ++l) {
      int i = l % nx, j = l / nx;
      for (int k = 0; k < nz; ++k) { dr[k] = A[S.id(i, j, k)].real(); di[k] = A[S.id(i, j, k)].imag(); }
      zsolve(i, j, dr.data(), di.data());
      for (int k = 0; k < nz; ++k) A[S.id(i, j, k)] = cd(dr[k], di[k]);
    }
  }
  // inverse y
#pragma omp parallel
  {
    std::vector<cd> a(ny), b(ny); std::vector<double> r(ny), q(ny), R(ny), Q(ny);
#pragma omp for
    for (int l = 0; l < nx * nz; ++l) {
      int i = l % nx, k = l / nx;
      if (S.P.bc_y == BC_PER) {
        for (int j = 0; j < ny; ++j) a[j] = A[S.id(i, j, k)];
        S.ply->run(a.data(), b.data(), +1);
        for (int j = 0; j < ny; ++j) A[S.id(i, j, k)] = b[j] / (double)ny;
      } else {
        for (int j = 0; j < ny; ++j) { R[j] = A[S.id(i, j, k)].real(); Q[j] = A[S.id(i, j, k)].imag(); }
        S.pdy->dct3(R.data(), r.data()); S.pdy->dct3(Q.data(), q.data());
        for (int j = 0; j < ny; ++j) A[S.id(i, j, k)] = cd(r[j], q[j]);
      }
    }
  }
  // inverse x
#pragma omp parallel
  {
    std::vector<cd> a(nx), b(nx);
#pragma omp for
    for (int l = 0; l < ny * nz; ++l) {
      for (int i = 0; i < nx; ++i) a[i] = A[(size_t)l * nx + i];
      S.plx->run(a.data(), b.data(), +1);
      for (int i = 0; i < nx; ++i) phi[(size_t)l * nx + i] = b[i].real() / (double)nx;
    }
  }
}

static void poisson(const oracle_solver& S, const double* rhs, double* phi) {
  eigen_expansion_solve(S, rhs, phi, [&](int i, int j, double* dr, double* di) { poisson_zsolve(S, i, j, dr, di); });
}

// Modified Helmholtz equation of the fully implicit Crank-Nicolson scheme, Eq. 18 ("solved with the same
// direct solver used for the Poisson equation"):  (1 - c L_jj) q = rhs  for velocity component comp (0 u, 1 v: centred in z;
// 2 w: on z faces), c = gamma nu dt / 2.  x and y are periodic (the transforms need homogeneous conditions there), so
// the eigenvalues are those of the Poisson solve; the z system carries the component's wall closure: no-slip mirror ghost for
// u, v (or the zero-flux closure with the wall model, whose lagged stress is a source outside the operator), w = 0 on the wall
// faces (unknowns k = 0 .. nz-2), cyclic when z is periodic.
static void helmholtz(const oracle_solver& S, int comp, double c, const double* rhs, double* out) {
  int nz = S.nz;
  bool per = S.P.bc_z == BC_PER;
  eigen_expansion_solve(S, rhs, out, [&](int i, int j, double* dr, double* di) {
    double lam = lam_x(S, i) + lam_y(S, j);
    int m = (comp == 2 && !per) ? nz - 1 : nz;
    std::vector<double> a(m), b(m), cc(m), xr(m), xi(m);
    for (int k = 0; k < m; ++k) {
      double ak, ck;
      if (comp < 2) { ak = 1.0 / (S.dzf(k) * S.dzc(k - 1)); ck = 1.0 / (S.dzf(k) * S.dzc(k)); }
      else { ak = 1.0 / (S.dzc(k) * S.dzf(k)); ck = 1.0 / (S.dzc(k) * S.dzf(k + 1)); }
      a[k] = -c * ak; cc[k] = -c * ck; b[k] = 1.0 + c * (ak + ck) - c * lam;
      if (!per && comp < 2) {
        double sg = S.P.wall_model ? -1.0 : 1.0;          // mirror ghost q[-1] = -q[0], or zero flux q[-1] = q[0]
        if (k == 0) b[k] += sg * c * ak;
        if (k == nz - 1) b[k] += sg * c * ck;
      }
    }
    if (per) {
      oracle_thomas_cyclic(m, a.data(), b.data(), cc.data(), dr, xr.data());
      oracle_thomas_cyclic(m, a.data(), b.data(), cc.data(), di, xi.data());
    } else {
      oracle_thomas(m, a.data(), b.data(), cc.data(), dr, xr.data());
      oracle_thomas(m, a.data(), b.data(), cc.data(), di, xi.data());
    }
    for (int k = 0; k < m; ++k) { dr[k] = xr[k]; di[k] = xi[k]; }
    for (int k = m; k < nz; ++k) { dr[k] = 0.0; di[k] = 0.0; }       // the wall face of w
  });
}

// ------------------------------------------------------------------------------------------------
// Strain rate at cell centres: diagonals directly at centres; off-diagonals at the edge
// midpoints, then averaged (4 edges) to the centre; |S| = sqrt(2 S_ij S_ij).  Velocity must be ghosted.
// ------------------------------------------------------------------------------------------------
static void strain(const oracle_solver& S, const F3& u, const F3& v, const F3& w, double* Sij /*6N*/, double* smag) {
  int nx = S.nx, ny = S.ny, nz = S.nz; double dx = S.dx, dy = S.dy; size_t N = S.N;
  auto s12 = [&](int i, int j, int k) { return 0.5 * ((u(i, j + 1, k) - u(i, j, k)) / dy + (v(i + 1, j, k) - v(i, j, k)) / dx); };       // edge (i+1/2,j+1/2)
  auto s13 = [&](int i, int j, int k) { return 0.5 * ((u(i, j, k + 1) - u(i, j, k)) / S.dzc(k) + (w(i + 1, j, k) - w(i, j, k)) / dx); }; // edge (i+1/2,k+1/2)
  auto s23 = [&](int i, int j, int k) { return 0.5 * ((v(i, j, k + 1) - v(i, j, k)) / S.dzc(k) + (w(i, j + 1, k) - w(i, j, k)) / dy); }; // edge (j+1/2,k+1/2)
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t n = S.id(i, j, k);
    double a11 = (u(i, j, k) - u(i - 1, j, k)) / dx;
    double a22 = (v(i, j, k) - v(i, j - 1, k)) / dy;
    double a33 = (w(i, j, k) - w(i, j, k - 1)) / S.dzf(k);
    double a12 = 0.25 * (s12(i, j, k) + s12(i - 1, j, k) + s12(i, j - 1, k) + s12(i - 1, j - 1, k));
    double a13 = 0.25 * (s13(i, j, k) + s13(i - 1, j, k) + s13(i, j, k - 1) + s13(i - 1, j, k - 1));
    double a23 = 0.25 * (s23(i, j, k) + s23(i, j - 1, k) + s23(i, j, k - 1) + s23(i, j - 1, k - 1));
    Sij[0 * N + n] = a11; Sij[1 * N + n] = a22; Sij[2 * N + n] = a33; Sij[3 * N + n] = a12; Sij[4 * N + n] = a13; Sij[5 * N + n] = a23;
    smag[n] = std::sqrt(2.0 * (a11 * a11 + a22 * a22 + a33 * a33) + 4.0 * (a12 * a12 + a13 * a13 + a23 * a23));
  }
}

// x-y test filter, separable (1/4,1/2,1/4) per filtered direction (reading S11).  In a wall-bounded y the
// first off-wall layers (j = 0, ny-1) keep the identity in y (linear extrapolation to the
// ghost followed by the symmetric 3-point filter is the identity).  Acts on interior arrays of centred data.
static void filter_xy_centre(const oracle_solver& S, const double* q, double* out) {
  int nx = S.nx, ny = S.ny, nz = S.nz;
  std::vector<double> t(S.N);
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    int im = (i + nx - 1) % nx, ip = (i + 1) % nx;
    t[S.id(i, j, k)] = 0.25 * q[S.id(im, j, k)] + 0.5 * q[S.id(i, j, k)] + 0.25 * q[S.id(ip, j, k)];
  }
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    if (S.P.bc_y == BC_WALL && (j == 0 || j == ny - 1)) { out[S.id(i, j, k)] = t[S.id(i, j, k)]; continue; }
    int jm = (j + ny - 1) % ny, jp = (j + 1) % ny;
    out[S.id(i, j, k)] = 0.25 * t[S.id(i, jm, k)] + 0.5 * t[S.id(i, j, k)] + 0.25 * t[S.id(i, jp, k)];
  }
}
// the same filter for v, which lives on y-faces: with y-walls the faces j = -1 and ny-1 are the walls (value 0),
// every interior face j = 0..ny-2 has both neighbours, so the full 3-point filter applies; the wall face stays 0.
static void filter_xy_vface(const oracle_solver& S, const double* q, double* out) {
  if (S.P.bc_y == BC_PER) { filter_xy_centre(S, q, out); return; }   // same as the centred filter when y is periodic
  int nx = S.nx, ny = S.ny, nz = S.nz; std::vector<double> t(S.N);
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    int im = (i + nx - 1) % nx, ip = (i + 1) % nx;
    t[S.id(i, j, k)] = 0.25 * q[S.id(im, j, k)] + 0.5 * q[S.id(i, j, k)] + 0.25 * q[S.id(ip, j, k)];
  }
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    if (j == ny - 1) { out[S.id(i, j, k)] = 0.0; continue; }
    double lo = (j == 0) ? 0.0 : t[S.id(i, j - 1, k)];
    double hi = (j == ny - 2) ? 0.0 : t[S.id(i, j + 1, k)];
    out[S.id(i, j, k)] = 0.25 * lo + 0.5 * t[S.id(i, j, k)] + 0.25 * hi;
  }
}

// z part of the 3-D box test filter ("2D or 3D box filters ... assumes uniform grid spacing"): the same
// (1/4,1/2,1/4) weights along z.  "The 3D box filter cannot be used in the first off-wall layer, hence a 2D box filter
// is applied through linear extrapolation ... to the ghost points, followed by ... a 3D filter": extrapolation followed
// by the symmetric 3-point filter is the identity, so layers k = 0 and nz-1 of a wall-bounded z keep the identity in z.
// wface = 1: data on z-faces (w): the wall faces k = -1, nz-1 hold 0, every interior face has both neighbours.
static void filter_z(const oracle_solver& S, const double* q, double* out, int wface) {
  int nx = S.nx, ny = S.ny, nz = S.nz;
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t n = S.id(i, j, k);
    if (S.P.bc_z == BC_PER) { out[n] = 0.25 * q[S.id(i, j, (k + nz - 1) % nz)] + 0.5 * q[n] + 0.25 * q[S.id(i, j, (k + 1) % nz)]; continue; }
    if (!wface) {
      if (k == 0 || k == nz - 1) out[n] = q[n];
      else out[n] = 0.25 * q[S.id(i, j, k - 1)] + 0.5 * q[n] + 0.25 * q[S.id(i, j, k + 1)];
    } else {
      if (k == nz - 1) { out[n] = 0.0; continue; }
      double lo = (k == 0) ? 0.0 : q[S.id(i, j, k - 1)];
      double hi = (k == nz - 2) ? 0.0 : q[S.id(i, j, k + 1)];
      out[n] = 0.25 * lo + 0.5 * q[n] + 0.25 * hi;
    }
  }
}
// the test filter of the run: x-y (dsm_filter3d = 0) or x-y-z.  kind 0: centred data and u; 1: v (y-faces); 2: w (z-faces)
static void test_filter(const oracle_solver& S, const double* q, double* out, int kind) {
  if (!S.P.dsm_filter3d) { if (kind == 1) filter_xy_vface(S, q, out); else filter_xy_centre(S, q, out); return; }
  std::vector<double> t(S.N);
  if (kind == 1) filter_xy_vface(S, q, t.data()); else filter_xy_centre(S, q, t.data());
  filter_z(S, t.data(), out, kind == 2);
}

// ------------------------------------------------------------------------------------------------
// Eddy viscosity (O-step 9).  u,v,w ghosted in GH_STRAIN mode by the caller.
// ------------------------------------------------------------------------------------------------
static void eddy_viscosity(oracle_solver& S, F3& u, F3& v, F3& w, double* nut) {
  int nx = S.nx, ny = S.ny, nz = S.nz; size_t N = S.N; double dx = S.dx, dy = S.dy, nu = S.P.nu;
  if (S.P.sgs_model == 0) { for (size_t n = 0; n < N; ++n) nut[n] = 0.0; return; }
  std::vector<double> Sij(6 * N), smag(N);
  strain(S, u, v, w, Sij.data(), smag.data());
  if (S.P.sgs_model == 1) {
    // Eq. 4: nu_t = (C_s Delta D)^2 |S|, Delta = (dx dy dzf)^(1/3) (reading S4),
    // D = 1 - exp(-d+/A+) with the local u_tau of the nearest z-wall (reading S5)
#pragma omp parallel for
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
      double delta = std::cbrt(dx * dy * S.dzf(k));
      double D = 1.0;
      if (S.P.van_driest) {
        double db = S.zc[k], dt = S.P.lz - S.zc[k];
        int kw = (db <= dt) ? 0 : nz - 1; double d = (db <= dt) ? db : dt;
        double d1 = (kw == 0) ? S.zc[0] : S.P.lz - S.zc[nz - 1];
        double uc = 0.5 * (u(i - 1, j, kw) + u(i, j, kw)), vc = 0.5 * (v(i, j - 1, kw) + v(i, j, kw));
        double tauw = nu * std::sqrt(uc * uc + vc * vc) / d1;
        double utau = std::sqrt(tauw);
        D = 1.0 - std::exp(-(d * utau / nu) / S.P.aplus);
      }
      double l = S.P.cs * delta * D;
      nut[S.id(i, j, k)] = l * l * smag[S.id(i, j, k)];
    }
    return;
  }
  // ---- dynamic Smagorinsky, Eq. 5-9, x-y test filter (readings S2, S11)
  std::vector<double> uc(N), vc(N), wc(N);
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {   // velocities averaged to centres
    size_t n = S.id(i, j, k);
    uc[n] = 0.5 * (u(i - 1, j, k) + u(i, j, k)); vc[n] = 0.5 * (v(i, j - 1, k) + v(i, j, k)); wc[n] = 0.5 * (w(i, j, k - 1) + w(i, j, k));
  }
  const double* vel[3] = {uc.data(), vc.data(), wc.data()};
  std::vector<double> fvel(3 * N), prod(N), fprod(N);
  for (int c = 0; c < 3; ++c) test_filter(S, vel[c], &fvel[c * N], 0);
  const int pa[6] = {0, 1, 2, 0, 0, 1}, pb[6] = {0, 1, 2, 1, 2, 2};   // 11 22 33 12 13 23
  std::vector<double> L(6 * N), M(6 * N);
  for (int c = 0; c < 6; ++c) {   // Eq. 7: L_ij = F(u_i u_j) - F(u_i) F(u_j)
    for (size_t n = 0; n < N; ++n) prod[n] = vel[pa[c]][n] * vel[pb[c]][n];
    test_filter(S, prod.data(), fprod.data(), 0);
    for (size_t n = 0; n < N; ++n) L[c * N + n] = fprod[n] - fvel[pa[c] * N + n] * fvel[pb[c] * N + n];
  }
  // Eq. 9: test-filtered strain from the face-wise filtered velocity, ghosted by the same BC routine
  F3 uf(nx, ny, nz), vf(nx, ny, nz), wf(nx, ny, nz);
  {
    std::vector<double> a(N), b(N);
    u.to(a.data()); test_filter(S, a.data(), b.data(), 0); uf.from(b.data());
    v.to(a.data()); test_filter(S, a.data(), b.data(), 1); vf.from(b.data());
    w.to(a.data()); test_filter(S, a.data(), b.data(), 2); wf.from(b.data());
  }
  bc_velocity(S, uf, vf, wf, GH_STRAIN);
  std::vector<double> St(6 * N), stmag(N);
  strain(S, uf, vf, wf, St.data(), stmag.data());
  for (int c = 0; c < 6; ++c) {   // Eq. 8 (reading S2): M_ij = 2 Delta^2 [F(|S| S_ij) - alpha^2 |S~| S~_ij]
    for (size_t n = 0; n < N; ++n) prod[n] = smag[n] * Sij[c * N + n];
    test_filter(S, prod.data(), fprod.data(), 0);
#pragma omp parallel for
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
      size_t n = S.id(i, j, k);
      double d2 = std::pow(dx * dy * S.dzf(k), 2.0 / 3.0);
      // filter-width ratio: (volume ratio)^(1/3) of the directions actually filtered at this point (PAPER.md:128:
      // 4^(1/3) for a 2-D filter, 8^(1/3) = 2 for the 3-D one; reading S11: 2^(1/3) where only x is filtered)
      int nf = 1;
      if (!(S.P.bc_y == BC_WALL && (j == 0 || j == ny - 1))) ++nf;
      if (S.P.dsm_filter3d && !(S.P.bc_z == BC_WALL && (k == 0 || k == nz - 1))) ++nf;
      double al = nf == 2 ? S.alpha2d : (nf == 1 ? std::sqrt(S.alpha2d) : S.alpha2d * std::sqrt(S.alpha2d));
      M[c * N + n] = 2.0 * d2 * (fprod[n] - al * al * stmag[n] * St[c * N + n]);
    }
  }
  S.Lij = L; S.Mij = M;
  // Eq. 6: c_s = <M_ij L_ij>/<M_ij M_ij>, sum over the 9 (i,j) pairs and the homogeneous directions
  int per_plane = S.P.dsm_avg_xy_plane;
  S.cs.assign(per_plane ? nz : (size_t)nz * ny, 0.0);
  for (int k = 0; k < nz; ++k) {
    double pl = 0, pm = 0;
    for (int j = 0; j < ny; ++j) {
      double ll = 0, mm = 0;
      for (int i = 0; i < nx; ++i) {
        size_t n = S.id(i, j, k);
        for (int c = 0; c < 6; ++c) { double f = c < 3 ? 1.0 : 2.0; ll += f * L[c * N + n] * M[c * N + n]; mm += f * M[c * N + n] * M[c * N + n]; }
      }
      if (!per_plane) S.cs[(size_t)k * ny + j] = (mm > 0.0) ? ll / mm : 0.0;   // reading S13
      pl += ll; pm += mm;
    }
    if (per_plane) S.cs[k] = (pm > 0.0) ? pl / pm : 0.0;
  }
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t n = S.id(i, j, k);
    double c = per_plane ? S.cs[k] : S.cs[(size_t)k * ny + j];
    double d2 = std::pow(dx * dy * S.dzf(k), 2.0 / 3.0);
    if (!S.P.dsm_clip_total) { if (c < 0.0) c = 0.0; nut[n] = c * d2 * smag[n]; }          // PAPER.md:128 clip
    else { double t = c * d2 * smag[n]; nut[n] = (t < -nu) ? -nu : t; }                      // reading S14 (config 4)
  }
}

// ------------------------------------------------------------------------------------------------
// solver object
// ------------------------------------------------------------------------------------------------
static bool smooth23(int n) { while (n % 2 == 0) n /= 2; while (n % 3 == 0) n /= 3; return n == 1; }
extern "C" int oracle_create(const oracle_params* p, oracle_solver** out) {
  if (!p || !out) return fail("null argument");
  if (p->nx < 2 || p->ny < 2 || p->nz < 4) return fail("grid too small");
  if (p->nx % 2) return fail("nx must be even");
  if (!smooth23(p->nx) || !smooth23(p->ny)) return fail("nx, ny must factor into 2 and 3");
  if (p->bc_z == BC_PER && p->zstretch != 0) return fail("periodic z requires a uniform grid");
  if (p->wall_model && p->bc_z != BC_WALL) return fail("wall model needs z walls");
  if (p->wall_model_y && p->bc_y != BC_WALL) return fail("wall model on y walls needs y walls");
  if (p->implicit_z && p->bc_z != BC_WALL) return fail("implicit z needs z walls");
  if (p->implicit_xyz && p->bc_y != BC_PER) return fail("fully implicit diffusion needs periodic y (PAPER.md:136)");
  if (p->implicit_xyz && p->implicit_z) return fail("implicit_z and implicit_xyz exclude each other");
  if (p->wall_model && p->h_wm > 0.0 && !(p->h_wm < 0.5 * p->lz)) return fail("h_wm must lie below the half height");
  if (p->wall_model_y && p->h_wm > 0.0 && !(p->h_wm < 0.5 * p->ly)) return fail("h_wm must lie below the half width");
  if (p->van_driest && (p->bc_z != BC_WALL || p->bc_y == BC_WALL || p->wall_model)) return fail("van Driest: z walls only, no wall model");
  oracle_solver* S = new oracle_solver();
  S->P = *p; S->nx = p->nx; S->ny = p->ny; S->nz = p->nz; S->N = (size_t)p->nx * p->ny * p->nz;
  S->dx = p->lx / p->nx; S->dy = p->ly / p->ny;
  int nz = p->nz;
  S->zf.resize(nz + 1); S->zc.resize(nz); S->dzf_.resize(nz + 2); S->dzc_.resize(nz + 1);
  for (int k = 0; k <= nz; ++k) {
    if (p->zstretch == 0) S->zf[k] = p->lz * (double)k / (double)nz;
    else if (p->zstretch == 1) { double a = p->zstretch_factor; S->zf[k] = 0.5 * p->lz * (1.0 + std::tanh(a * (2.0 * k / (double)nz - 1.0)) / std::tanh(a)); }  // reading S16
    else S->zf[k] = p->zf_user[k];
  }
  S->zf[0] = 0.0; S->zf[nz] = p->lz;
  for (int k = 0; k < nz; ++k) { S->zc[k] = 0.5 * (S->zf[k] + S->zf[k + 1]); S->dzf_[k + 1] = S->zf[k + 1] - S->zf[k]; }
  if (p->bc_z == BC_PER) { S->dzf_[0] = S->dzf_[nz]; S->dzf_[nz + 1] = S->dzf_[1]; }
  else { S->dzf_[0] = S->dzf_[1]; S->dzf_[nz + 1] = S->dzf_[nz]; }
  for (int k = 0; k < nz - 1; ++k) S->dzc_[k + 1] = S->zc[k + 1] - S->zc[k];
  if (p->bc_z == BC_PER) { S->dzc_[0] = S->dzf_[1]; S->dzc_[nz] = S->dzf_[1]; }
  else { S->dzc_[0] = 2.0 * S->zc[0]; S->dzc_[nz] = 2.0 * (p->lz - S->zc[nz - 1]); }   // mirrored ghost centre
  S->u = F3(p->nx, p->ny, nz); S->v = S->u; S->w = S->u; S->p = S->u; S->nut = S->u;
  S->Ru.assign(S->N, 0.0); S->Rv.assign(S->N, 0.0); S->Rw.assign(S->N, 0.0);
  S->tau.assign((size_t)4 * p->nx * p->ny, 0.0);
  S->tauy.assign((size_t)4 * p->nx * p->nz, 0.0);
  S->alpha2d = p->dsm_alpha2d > 0.0 ? p->dsm_alpha2d : std::cbrt(4.0);
  if (S->P.wm_tol <= 0.0) S->P.wm_tol = 1e-4;
  if (S->P.wm_maxit <= 0) S->P.wm_maxit = 50;
  if (S->P.kappa <= 0.0) S->P.kappa = 0.41;
  if (S->P.aplus <= 0.0) S->P.aplus = 25.0;
  S->plx = new FftPlan(p->nx);
  if (p->bc_y == BC_PER) S->ply = new FftPlan(p->ny); else S->pdy = new DctPlan(p->ny);
  *out = S; return 0;
}
extern "C" void oracle_destroy(oracle_solver* s) { delete s; }
extern "C" int oracle_get_grid(oracle_solver* S, double* zf, double* zc, double* dzf, double* dzc) {
  if (!S) return fail("null");
  if (zf) for (int k = 0; k <= S->nz; ++k) zf[k] = S->zf[k];
  if (zc) for (int k = 0; k < S->nz; ++k) zc[k] = S->zc[k];
  if (dzf) for (int k = 0; k < S->nz; ++k) dzf[k] = S->dzf(k);
  if (dzc) for (int k = -1; k < S->nz; ++k) dzc[k + 1] = S->dzc(k);
  return 0;
}
static F3* field_of(oracle_solver* S, int f) { switch (f) { case 0: return &S->u; case 1: return &S->v; case 2: return &S->w; case 3: return &S->p; case 4: return &S->nut; } return nullptr; }
extern "C" int oracle_set_field(oracle_solver* S, int f, const double* src) {
  F3* q = S ? field_of(S, f) : nullptr; if (!q || !src) return fail("bad field");
  q->from(src); if (f <= 2) S->fresh = false; return 0;
}
extern "C" int oracle_get_field(oracle_solver* S, int f, double* dst) {
  F3* q = S ? field_of(S, f) : nullptr; if (!q || !dst) return fail("bad field");
  q->to(dst); return 0;
}

// Alg. 2 on the current velocity, then nu_t (Alg. 1 l.2 / l.12)
static void refresh_closures(oracle_solver& S) {
  bc_velocity(S, S.u, S.v, S.w, GH_STRAIN);   // steps 1-2: periodic + ordinary BCs (x/y ghosts are mode-independent)
  wall_stress(S);                             // step 3
  // step 4 (wall-model ghosts) happens inside bc_velocity wherever a ghost is consumed
  std::vector<double> nt(S.N);
  eddy_viscosity(S, S.u, S.v, S.w, nt.data());
  S.nut.from(nt.data());
  S.fresh = true;
}

static void substep(oracle_solver& S, int rk, double dt) {
  int nx = S.nx, ny = S.ny, nz = S.nz; size_t N = S.N; double dx = S.dx, dy = S.dy, nu = S.P.nu;
  double al, be, ga; oracle_rk3_coeffs(rk, &al, &be, &ga);
  int kwmax = (S.P.bc_z == BC_WALL) ? nz - 1 : nz, jvmax = (S.P.bc_y == BC_WALL) ? ny - 1 : ny;
  // O-step 1: ghosts
  bc_velocity(S, S.u, S.v, S.w, GH_VISC);
  bc_scalar(S, S.p, SC_NEUMANN);
  bc_scalar(S, S.nut, SC_NEG);
  // O-steps 2-4
  std::vector<double> au(N), av(N), aw(N), dxu(N), dxv(N), dxw(N), dzu(N), dzv(N), dzw(N), su(N), sv(N), sw(N);
  advection(S, S.u, S.v, S.w, au.data(), av.data(), aw.data());
  diffusion(S, S.u, S.v, S.w, dxu.data(), dxv.data(), dxw.data(), 1);
  diffusion(S, S.u, S.v, S.w, dzu.data(), dzv.data(), dzw.data(), 2);
  if (S.P.sgs_model != 0) sgs_term(S, S.u, S.v, S.w, S.nut, su.data(), sv.data(), sw.data());
  // O-step 5: R^k and the RK update, Eq. 11 (explicit) / Eq. 20 (implicit z)
  F3 us(nx, ny, nz), vs(nx, ny, nz), ws(nx, ny, nz);
  bool imp = S.P.implicit_z != 0, imp3 = S.P.implicit_xyz != 0;
  // Eq. 11: R = H + nu L_jj u;  Eq. 20: R = H + nu (L_xx + L_yy) u, the z part goes with gamma;  Eq. 17: R = H, all of nu L_jj u
  // goes with gamma (H = advection + SGS, Eq. 15)
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t n = S.id(i, j, k);
    double Ru = au[n] + su[n] + (imp3 ? 0.0 : dxu[n]) + ((imp || imp3) ? 0.0 : dzu[n]);
    double Rv = av[n] + sv[n] + (imp3 ? 0.0 : dxv[n]) + ((imp || imp3) ? 0.0 : dzv[n]);
    double Rw = aw[n] + sw[n] + (imp3 ? 0.0 : dxw[n]) + ((imp || imp3) ? 0.0 : dzw[n]);
    double gpx = (S.p(i + 1, j, k) - S.p(i, j, k)) / dx, gpy = (S.p(i, j + 1, k) - S.p(i, j, k)) / dy, gpz = (S.p(i, j, k + 1) - S.p(i, j, k)) / S.dzc(k);
    double gu = imp ? dzu[n] : (imp3 ? dxu[n] + dzu[n] : 0.0), gv = imp ? dzv[n] : (imp3 ? dxv[n] + dzv[n] : 0.0), gw = imp ? dzw[n] : (imp3 ? dxw[n] + dzw[n] : 0.0);
    us(i, j, k) = S.u(i, j, k) + dt * (al * Ru + be * S.Ru[n] - ga * gpx + ga * gu);
    vs(i, j, k) = (j < jvmax) ? S.v(i, j, k) + dt * (al * Rv + be * S.Rv[n] - ga * gpy + ga * gv) : 0.0;
    ws(i, j, k) = (k < kwmax) ? S.w(i, j, k) + dt * (al * Rw + be * S.Rw[n] - ga * gpz + ga * gw) : 0.0;
    S.Ru[n] = Ru; S.Rv[n] = (j < jvmax) ? Rv : 0.0; S.Rw[n] = (k < kwmax) ? Rw : 0.0;
  }
  // O-step 6: (1 - c L_zz) u* = u** - c L_zz u^k, c = gamma nu dt / 2 (Eq. 21), plain Thomas per (i,j)
  double cimp = ga * nu * dt / 2.0;
  if (imp) {
#pragma omp parallel
    {
      std::vector<double> a(nz), b(nz), c(nz), d(nz), x(nz);
#pragma omp for
      for (int l = 0; l < nx * ny; ++l) {
        int i = l % nx, j = l / nx;
        for (int comp = 0; comp < 2; ++comp) {     // u, v: centred in z, no-slip ghost folded into the diagonal
          F3& q = comp == 0 ? us : vs; const double* lz = comp == 0 ? dzu.data() : dzv.data();
          if (comp == 1 && j >= jvmax) continue;
          const F3& q0 = comp == 0 ? S.u : S.v;
          for (int k = 0; k < nz; ++k) {
            double ak = 1.0 / (S.dzf(k) * S.dzc(k - 1)), ck = 1.0 / (S.dzf(k) * S.dzc(k));
            a[k] = -cimp * ak; c[k] = -cimp * ck; b[k] = 1.0 + cimp * (ak + ck);
            if (!S.P.wall_model) {
              if (k == 0) b[k] += cimp * ak;           // u[-1] = -u[0]
              if (k == nz - 1) b[k] += cimp * ck;      // u[nz] = -u[nz-1]
              d[k] = q(i, j, k) - cimp * (lz[S.id(i, j, k)] / nu);
            } else {
              // with the wall model the wall flux is the prescribed, lagged stress: it
              // is a source s in L_zz u = Lt u + s that appears on both sides of Eq. 21 and cancels; the implicit operator
              // Lt has the zero-flux (Neumann) closure at the walls, and the right-hand side uses Lt u^k.
              if (k == 0) b[k] -= cimp * ak;
              if (k == nz - 1) b[k] -= cimp * ck;
              double lt = ((k < nz - 1 ? (q0(i, j, k + 1) - q0(i, j, k)) / S.dzc(k) : 0.0) - (k > 0 ? (q0(i, j, k) - q0(i, j, k - 1)) / S.dzc(k - 1) : 0.0)) / S.dzf(k);
              d[k] = q(i, j, k) - cimp * lt;
            }
          }
          oracle_thomas(nz, a.data(), b.data(), c.data(), d.data(), x.data());
          for (int k = 0; k < nz; ++k) q(i, j, k) = x[k];
        }
        {                                            // w: faces k = 0..nz-2 unknown, w = 0 on the wall faces
          int m = nz - 1;
          for (int k = 0; k < m; ++k) {
            double ak = 1.0 / (S.dzc(k) * S.dzf(k)), ck = 1.0 / (S.dzc(k) * S.dzf(k + 1));
            a[k] = -cimp * ak; c[k] = -cimp * ck; b[k] = 1.0 + cimp * (ak + ck);
            d[k] = ws(i, j, k) - cimp * (dzw[S.id(i, j, k)] / nu);
          }
          oracle_thomas(m, a.data(), b.data(), c.data(), d.data(), x.data());
          for (int k = 0; k < m; ++k) ws(i, j, k) = x[k];
        }
      }
    }
  }
  // Eq. 18: (1 - c L_jj) u* = u** - c L_jj u^k, three modified Helmholtz solves by the eigen-expansion solver.
  // With the wall model (z walls only) the lagged stress is a source outside the implicit operator, as in Eq. 21:
  // the right-hand side uses the zero-flux z operator applied to u^k.
  if (imp3) {
    std::vector<double> rhs(N), sol(N);
    for (int comp = 0; comp < 3; ++comp) {
      F3& q = comp == 0 ? us : (comp == 1 ? vs : ws);
      const F3& q0 = comp == 0 ? S.u : (comp == 1 ? S.v : S.w);
      const double* lxy = comp == 0 ? dxu.data() : (comp == 1 ? dxv.data() : dxw.data());
      const double* lz = comp == 0 ? dzu.data() : (comp == 1 ? dzv.data() : dzw.data());
#pragma omp parallel for
      for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        size_t n = S.id(i, j, k);
        double lzz = lz[n] / nu;
        if (S.P.wall_model && comp < 2)
          lzz = ((k < nz - 1 ? (q0(i, j, k + 1) - q0(i, j, k)) / S.dzc(k) : 0.0) - (k > 0 ? (q0(i, j, k) - q0(i, j, k - 1)) / S.dzc(k - 1) : 0.0)) / S.dzf(k);
        rhs[n] = q(i, j, k) - cimp * (lxy[n] / nu + lzz);
      }
      helmholtz(S, comp, cimp, rhs.data(), sol.data());
      q.from(sol.data());
    }
  }
  S.ust.resize(N); S.vst.resize(N); S.wst.resize(N);     // kept for the pins of Eq. 21 / Eq. 22 (oracle_get_ustar)
  us.to(S.ust.data()); vs.to(S.vst.data()); ws.to(S.wst.data());
  // O-step 7a: constant flow rate (reading S12): uniform shift of u* to the target bulk velocity
  S.forcing = 0.0;
  if (S.P.const_flow_rate) {
    double m = 0.0;
    for (int k = 0; k < nz; ++k) { double pl = 0.0; for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) pl += us(i, j, k); m += pl * S.dzf(k); }
    m /= ((double)nx * (double)ny * S.P.lz);
    double sh = S.P.u_bulk - m;
#pragma omp parallel for
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) us(i, j, k) += sh;
    S.forcing = sh / (ga * dt);
  }
  // BC on u* (PAPER.md:142); the wall-model ghosts of u* are never read (O-step 8 note), any mode will do
  bc_velocity(S, us, vs, ws, GH_STRAIN);
  // O-step 7b: Eq. 12
  std::vector<double> f(N), phi(N);
  divergence(S, us, vs, ws, f.data());
  for (size_t n = 0; n < N; ++n) f[n] /= (ga * dt);
  poisson(S, f.data(), phi.data());
  F3 ph(nx, ny, nz); ph.from(phi.data());
  bc_scalar(S, ph, SC_NEUMANN);
  // Eq. 13 correction; Eq. 14 / Eq. 22 pressure update
#pragma omp parallel for
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    S.u(i, j, k) = us(i, j, k) - ga * dt * (ph(i + 1, j, k) - ph(i, j, k)) / dx;
    S.v(i, j, k) = (j < jvmax) ? vs(i, j, k) - ga * dt * (ph(i, j + 1, k) - ph(i, j, k)) / dy : 0.0;
    S.w(i, j, k) = (k < kwmax) ? ws(i, j, k) - ga * dt * (ph(i, j, k + 1) - ph(i, j, k)) / S.dzc(k) : 0.0;
    double lzz = ((ph(i, j, k + 1) - ph(i, j, k)) / S.dzc(k) - (ph(i, j, k) - ph(i, j, k - 1)) / S.dzc(k - 1)) / S.dzf(k);
    double lxy = (ph(i + 1, j, k) - 2.0 * ph(i, j, k) + ph(i - 1, j, k)) / (dx * dx) + (ph(i, j + 1, k) - 2.0 * ph(i, j, k) + ph(i, j - 1, k)) / (dy * dy);
    S.p(i, j, k) += ph(i, j, k) - (imp ? cimp * lzz : 0.0) - (imp3 ? cimp * (lxy + lzz) : 0.0);     // Eq. 14 / Eq. 22 / Eq. 19
  }
  // O-steps 8-9
  refresh_closures(S);
}

extern "C" int oracle_step(oracle_solver* S, double dt) {
  if (!S || !(dt > 0.0)) return fail("bad step arguments");
  if (!S->fresh) refresh_closures(*S);   // Alg. 1 l.1-2
  for (int rk = 0; rk < 3; ++rk) substep(*S, rk, dt);
  return 0;
}
// One substep rk = 0, 1, 2 of Alg. 1 on its own (for the pins; a step is the three in order).
extern "C" int oracle_substep(oracle_solver* S, int rk, double dt) {
  if (!S || !(dt > 0.0) || rk < 0 || rk > 2) return fail("bad substep arguments");
  if (!S->fresh) refresh_closures(*S);
  substep(*S, rk, dt);
  return 0;
}
// u* (comp 0), v* (1), w* (2) of the last substep: after the Crank-Nicolson solve of Eq. 21 (if any), before the bulk shift
extern "C" int oracle_get_ustar(oracle_solver* S, int comp, double* dst) {
  if (!S || !dst || comp < 0 || comp > 2) return fail("bad argument");
  const std::vector<double>& q = comp == 0 ? S->ust : (comp == 1 ? S->vst : S->wst);
  if (q.size() != S->N) return fail("no substep yet");
  std::memcpy(dst, q.data(), S->N * sizeof(double));
  return 0;
}
extern "C" int oracle_poisson_solve(oracle_solver* S, const double* rhs, double* phi) {
  if (!S || !rhs || !phi) return fail("null"); poisson(*S, rhs, phi); return 0;
}
extern "C" int oracle_helmholtz_solve(oracle_solver* S, int comp, double c, const double* rhs, double* out) {
  if (!S || !rhs || !out || comp < 0 || comp > 2) return fail("bad argument");
  if (S->P.bc_y != BC_PER) return fail("helmholtz: periodic y only");
  helmholtz(*S, comp, c, rhs, out); return 0;
}
extern "C" int oracle_laplacian(oracle_solver* S, const double* phi, double* out) {
  if (!S || !phi || !out) return fail("null");
  F3 q(S->nx, S->ny, S->nz); q.from(phi); bc_scalar(*S, q, SC_NEUMANN);
  double dx = S->dx, dy = S->dy;
  for (int k = 0; k < S->nz; ++k) for (int j = 0; j < S->ny; ++j) for (int i = 0; i < S->nx; ++i)
    out[S->id(i, j, k)] = (q(i + 1, j, k) - 2.0 * q(i, j, k) + q(i - 1, j, k)) / (dx * dx) + (q(i, j + 1, k) - 2.0 * q(i, j, k) + q(i, j - 1, k)) / (dy * dy)
                        + ((q(i, j, k + 1) - q(i, j, k)) / S->dzc(k) - (q(i, j, k) - q(i, j, k - 1)) / S->dzc(k - 1)) / S->dzf(k);
  return 0;
}
extern "C" int oracle_eddy_viscosity(oracle_solver* S, const double* u, const double* v, const double* w, double* nut) {
  if (!S || !nut) return fail("null");
  if (u && v && w) {
    F3 a(S->nx, S->ny, S->nz), b(S->nx, S->ny, S->nz), c(S->nx, S->ny, S->nz);
    a.from(u); b.from(v); c.from(w);
    bc_velocity(*S, a, b, c, GH_STRAIN);
    eddy_viscosity(*S, a, b, c, nut);
  } else {
    bc_velocity(*S, S->u, S->v, S->w, GH_STRAIN);
    eddy_viscosity(*S, S->u, S->v, S->w, nut);
  }
  return 0;
}
extern "C" int oracle_wall_stress(oracle_solver* S, double* tau) {
  if (!S || !tau) return fail("null");
  bc_velocity(*S, S->u, S->v, S->w, GH_STRAIN);
  wall_stress(*S);
  std::memcpy(tau, S->tau.data(), S->tau.size() * sizeof(double));
  return 0;
}
extern "C" int oracle_wall_stress_y(oracle_solver* S, double* tauy) {
  if (!S || !tauy) return fail("null");
  bc_velocity(*S, S->u, S->v, S->w, GH_STRAIN);
  wall_stress(*S);
  std::memcpy(tauy, S->tauy.data(), S->tauy.size() * sizeof(double));
  return 0;
}
extern "C" int oracle_advection(oracle_solver* S, double* au, double* av, double* aw) {
  if (!S) return fail("null"); bc_velocity(*S, S->u, S->v, S->w, GH_VISC); advection(*S, S->u, S->v, S->w, au, av, aw); return 0;
}
extern "C" int oracle_diffusion(oracle_solver* S, double* du, double* dv, double* dw, int which) {
  if (!S) return fail("null"); bc_velocity(*S, S->u, S->v, S->w, GH_VISC); diffusion(*S, S->u, S->v, S->w, du, dv, dw, which); return 0;
}
extern "C" int oracle_sgs_term(oracle_solver* S, double* su, double* sv, double* sw) {
  if (!S) return fail("null");
  bc_velocity(*S, S->u, S->v, S->w, GH_VISC); bc_scalar(*S, S->nut, SC_NEG);
  sgs_term(*S, S->u, S->v, S->w, S->nut, su, sv, sw); return 0;
}
extern "C" int oracle_divergence(oracle_solver* S, double* d) {
  if (!S || !d) return fail("null"); bc_velocity(*S, S->u, S->v, S->w, GH_STRAIN); divergence(*S, S->u, S->v, S->w, d); return 0;
}
extern "C" int oracle_strain(oracle_solver* S, double* Sij, double* smag) {
  if (!S) return fail("null"); bc_velocity(*S, S->u, S->v, S->w, GH_STRAIN); strain(*S, S->u, S->v, S->w, Sij, smag); return 0;
}
extern "C" int oracle_filter_xy(oracle_solver* S, const double* q, double* out) { if (!S) return fail("null"); filter_xy_centre(*S, q, out); return 0; }
extern "C" int oracle_test_filter(oracle_solver* S, const double* q, double* out, int kind) { if (!S || kind < 0 || kind > 2) return fail("bad argument"); test_filter(*S, q, out, kind); return 0; }
extern "C" int oracle_get_cs(oracle_solver* S, double* cs) {
  if (!S || !cs) return fail("null"); for (size_t n = 0; n < S->cs.size(); ++n) cs[n] = S->cs[n]; return 0;
}
extern "C" int oracle_get_dsm_tensors(oracle_solver* S, double* L, double* M) {
  if (!S || S->Lij.size() != 6 * S->N) return fail("no dynamic evaluation yet");
  if (L) std::memcpy(L, S->Lij.data(), 6 * S->N * sizeof(double));
  if (M) std::memcpy(M, S->Mij.data(), 6 * S->N * sizeof(double));
  return 0;
}
extern "C" int oracle_project(oracle_solver* S) {
  if (!S) return fail("null");
  int nx = S->nx, ny = S->ny, nz = S->nz;
  int kwmax = (S->P.bc_z == BC_WALL) ? nz - 1 : nz, jvmax = (S->P.bc_y == BC_WALL) ? ny - 1 : ny;
  bc_velocity(*S, S->u, S->v, S->w, GH_STRAIN);
  std::vector<double> f(S->N), phi(S->N);
  divergence(*S, S->u, S->v, S->w, f.data());
  poisson(*S, f.data(), phi.data());
  F3 ph(nx, ny, nz); ph.from(phi.data()); bc_scalar(*S, ph, SC_NEUMANN);
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    S->u(i, j, k) -= (ph(i + 1, j, k) - ph(i, j, k)) / S->dx;
    S->v(i, j, k) = (j < jvmax) ? S->v(i, j, k) - (ph(i, j + 1, k) - ph(i, j, k)) / S->dy : 0.0;
    S->w(i, j, k) = (k < kwmax) ? S->w(i, j, k) - (ph(i, j, k + 1) - ph(i, j, k)) / S->dzc(k) : 0.0;
  }
  S->fresh = false;
  return 0;
}
extern "C" int oracle_diagnostics(oracle_solver* S, double* max_div, double* u_bulk, double* ke, double* forcing, int* wm_max_iters) {
  if (!S) return fail("null");
  int nx = S->nx, ny = S->ny, nz = S->nz;
  bc_velocity(*S, S->u, S->v, S->w, GH_STRAIN);
  std::vector<double> d(S->N); divergence(*S, S->u, S->v, S->w, d.data());
  double md = 0, ub = 0, e = 0;
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    double a = std::fabs(d[S->id(i, j, k)]); if (a > md) md = a;
    ub += S->u(i, j, k) * S->dzf(k);
    double uc = 0.5 * (S->u(i - 1, j, k) + S->u(i, j, k)), vc = 0.5 * (S->v(i, j - 1, k) + S->v(i, j, k)), wc = 0.5 * (S->w(i, j, k - 1) + S->w(i, j, k));
    e += 0.5 * (uc * uc + vc * vc + wc * wc) * S->dzf(k);
  }
  double vol = (double)nx * ny * S->P.lz;
  if (max_div) *max_div = md; if (u_bulk) *u_bulk = ub / vol; if (ke) *ke = e / vol;
  if (forcing) *forcing = S->forcing; if (wm_max_iters) *wm_max_iters = S->wm_max_iters;
  return 0;
}

// ---- adaptive time step and on-line plane statistics -----------------------------------------
// dt = cfl / max over cells of (|u_c|/dx + |v_c|/dy + |w_c|/dzf) with the velocities averaged to the cell centre
// (reading S18; "0.95 x the stability limit", formula silent).
extern "C" int oracle_cfl_dt(oracle_solver* S, double cfl, double* dt) {
  if (!S || !dt) return fail("null");
  int nx = S->nx, ny = S->ny, nz = S->nz;
  bc_velocity(*S, S->u, S->v, S->w, GH_STRAIN);
  double rmax = 0.0;
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    double uc = 0.5 * (S->u(i - 1, j, k) + S->u(i, j, k)), vc = 0.5 * (S->v(i, j - 1, k) + S->v(i, j, k)), wc = 0.5 * (S->w(i, j, k - 1) + S->w(i, j, k));
    double r = std::fabs(uc) / S->dx + std::fabs(vc) / S->dy + std::fabs(wc) / S->dzf(k);
    if (r > rmax) rmax = r;
  }
  *dt = rmax > 0.0 ? cfl / rmax : 0.0;
  return 0;
}
// Plane (x-y) means per k of the centre-averaged velocity, its products and nu_t (the profiles of PAPER.md:237):
// out[q][k], q = 0 <u>, 1 <v>, 2 <w>, 3 <uu>, 4 <vv>, 5 <ww>, 6 <uw>, 7 <nu_t>.
extern "C" int oracle_plane_stats(oracle_solver* S, double* out) {
  if (!S || !out) return fail("null");
  int nx = S->nx, ny = S->ny, nz = S->nz;
  bc_velocity(*S, S->u, S->v, S->w, GH_STRAIN);
  for (int k = 0; k < nz; ++k) {
    double a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
      double uc = 0.5 * (S->u(i - 1, j, k) + S->u(i, j, k)), vc = 0.5 * (S->v(i, j - 1, k) + S->v(i, j, k)), wc = 0.5 * (S->w(i, j, k - 1) + S->w(i, j, k));
      a[0] += uc; a[1] += vc; a[2] += wc; a[3] += uc * uc; a[4] += vc * vc; a[5] += wc * wc; a[6] += uc * wc; a[7] += S->nut(i, j, k);
    }
    for (int q = 0; q < 8; ++q) out[(size_t)q * nz + k] = a[q] / ((double)nx * ny);
  }
  return 0;
}

// ---- on-line statistics accumulated in time ("mean quantities"; Tables 3-5 report C_f and Re_tau) ------------------
// Instantaneous wall shear stress, averaged over each wall.  wall[0..3]: z walls, (tau_xz, tau_yz) at the bottom then the top;
// wall[4..7]: y walls, (tau_xy, tau_zy) at the j = 0 side then the j = ny-1 side; 0 in periodic directions.  Sign: positive when
// the wall retards a flow in the positive direction (the convention of the wall-model planes).  Modelled walls: the mean of the
// wall-model stress planes; no-slip walls: nu times the one-sided difference to the mirror ghost, 2 nu q_first / (ghost spacing).
static void wall_shear_means(oracle_solver& S, double* wall) {
  int nx = S.nx, ny = S.ny, nz = S.nz; double nu = S.P.nu;
  for (int q = 0; q < 8; ++q) wall[q] = 0.0;
  if (S.P.bc_z == BC_WALL) {
    for (int wl = 0; wl < 2; ++wl) for (int comp = 0; comp < 2; ++comp) {
      const F3& f = comp == 0 ? S.u : S.v;
      int k0 = wl == 0 ? 0 : nz - 1; double dz = wl == 0 ? S.dzc(-1) : S.dzc(nz - 1);
      double a = 0.0;
      for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) a += S.P.wall_model ? S.tw(wl, comp, i, j) : 2.0 * nu * f(i, j, k0) / dz;
      wall[wl * 2 + comp] = a / ((double)nx * ny);
    }
  }
  if (S.P.bc_y == BC_WALL) {
    for (int wl = 0; wl < 2; ++wl) for (int comp = 0; comp < 2; ++comp) {
      const F3& f = comp == 0 ? S.u : S.w;
      int j0 = wl == 0 ? 0 : ny - 1;
      double a = 0.0;
      for (int k = 0; k < nz; ++k) for (int i = 0; i < nx; ++i)
        a += (S.P.wall_model_y ? S.tauy[((size_t)(wl * 2 + comp) * nz + k) * nx + i] : 2.0 * nu * f(i, j0, k) / S.dy) * S.dzf(k);
      wall[4 + wl * 2 + comp] = a / ((double)nx * S.P.lz);
    }
  }
}
extern "C" int oracle_stats_reset(oracle_solver* S) {
  if (!S) return fail("null");
  S->st_prof.assign((size_t)8 * S->nz, 0.0); S->st_wall.assign(8, 0.0); S->st_weight = 0.0; return 0;
}
// adds weight x (the instantaneous plane means of oracle_plane_stats, the wall-shear means) to the accumulators
extern "C" int oracle_stats_accumulate(oracle_solver* S, double weight) {
  if (!S || !(weight > 0.0)) return fail("bad argument");
  if (S->st_prof.empty()) oracle_stats_reset(S);
  if (!S->fresh) refresh_closures(*S);       // the wall-model planes must belong to the current velocity
  std::vector<double> pr((size_t)8 * S->nz); double wl[8];
  oracle_plane_stats(S, pr.data());
  wall_shear_means(*S, wl);
  for (size_t q = 0; q < pr.size(); ++q) S->st_prof[q] += weight * pr[q];
  for (int q = 0; q < 8; ++q) S->st_wall[q] += weight * wl[q];
  S->st_weight += weight;
  return 0;
}
// time averages: prof[8][nz], wall[8]; derived[0] = tau_w (mean of the x components on the z walls, or on all four walls of a
// duct), [1] = u_tau = sqrt(tau_w), [2] = Re_tau = u_tau (lz/2) / nu, [3] = C_f = 2 tau_w / u_b^2 with u_b the dzf-weighted mean
// of the averaged <u> profile; *weight = accumulated weight
extern "C" int oracle_stats_get(oracle_solver* S, double* prof, double* wall, double* derived, double* weight) {
  if (!S || !(S->st_weight > 0.0)) return fail("no statistics accumulated");
  double w = S->st_weight; int nz = S->nz;
  std::vector<double> pr(S->st_prof); for (double& q : pr) q /= w;
  double wl[8]; for (int q = 0; q < 8; ++q) wl[q] = S->st_wall[q] / w;
  if (prof) std::memcpy(prof, pr.data(), pr.size() * sizeof(double));
  if (wall) std::memcpy(wall, wl, sizeof(wl));
  if (derived) {
    double tw = 0.0; int nw = 0;
    if (S->P.bc_z == BC_WALL) { tw += wl[0] + wl[2]; nw += 2; }
    if (S->P.bc_y == BC_WALL) { tw += wl[4] + wl[6]; nw += 2; }
    tw = nw ? tw / nw : 0.0;
    double ub = 0.0; for (int k = 0; k < nz; ++k) ub += pr[k] * S->dzf(k); ub /= S->P.lz;
    derived[0] = tw; derived[1] = tw > 0.0 ? std::sqrt(tw) : 0.0; derived[2] = derived[1] * 0.5 * S->P.lz / S->P.nu;
    derived[3] = ub != 0.0 ? 2.0 * tw / (ub * ub) : 0.0;
  }
  if (weight) *weight = w;
  return 0;
}
