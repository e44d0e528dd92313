// cales_poisson.cuh -- tridiagonal solves along z: the Thomas step of the eigenfunction-expansion Poisson
// solver and the Crank-Nicolson z solve of Eq. 21.
//
// One thread per (i,j) column, consecutive threads on consecutive i, so every load and store of a k-level is
// coalesced.  The forward sweep leaves d' in place and c' in a scratch field; the backward sweep overwrites d'
// with the solution.
#pragma once
#include "cales_common.cuh"

namespace cales {

struct PoissonTabs {
  const double* ak;    // a_k = 1/(dzf[k] dzc[k-1])
  const double* ck;    // c_k = 1/(dzf[k] dzc[k])
  const double* lamx;  // eigenvalue of slot i of the packed half-complex x spectrum
  const double* lamy;  // eigenvalue of row j (packed half-complex, or DCT-II mode j)
};

// Poisson column (i,j): [a_k, b_k, c_k] phi = f with b_k = -(a_k + c_k) + lam_x + lam_y, a_0 and c_{nz-1} dropped from
// b at walls (Neumann) or wrapped (periodic z: cyclic Thomas via Sherman-Morrison).  The singular (0,0) mode drops the
// dzf-weighted mean of f, pins phi[0] = 0, and returns the solution with zero dzf-weighted mean (S15).
// CPT (walls in z only): c' of every column, computed once at set-up by poisson_cp_column -- the matrix does not depend on the right-
// hand side, so the forward sweep need not spill c' (8 of its 46 B/pt of DRAM traffic) and the backward sweep reads the table.
CALES_HD void poisson_column(const Ctx& c, const PoissonTabs& T, int i, int j, double* __restrict__ A, double* __restrict__ CP, double* __restrict__ CQ,
                             const double* __restrict__ CPT = nullptr) {
  const int nz = c.nz;
  const long long col = (long long)i + (long long)c.nx * j, st = c.nxy;
  const double lam = T.lamx[i] + T.lamy[j];
  const bool per = c.bc_z == BC_PER;
  const bool zero = (i == 0 && j == 0);
  if (zero || !per) {
    double mean = 0.0;
    if (zero) {
      for (int k = 0; k < nz; ++k) mean += A[col + st * k] * c.dzf[k];
      mean /= c.lz;
    }
    // Both sweeps read their inputs TZ levels at a time into registers before the recurrence touches them, so that TZ
    // independent loads per array are in flight per thread (the recurrence itself is a serial chain).
    enum { TZ = 8 };
    double cp = 0.0, dp = 0.0;
    for (int k0 = 0; k0 < nz; k0 += TZ) {
      double dd[TZ];
#pragma unroll
      for (int q = 0; q < TZ; ++q) dd[q] = (k0 + q < nz) ? A[col + st * (k0 + q)] : 0.0;
#pragma unroll
      for (int q = 0; q < TZ; ++q) {
        const int k = k0 + q;
        if (k < nz) {
          const double a = T.ak[k], cc = T.ck[k];
          const double b = lam - ((k > 0 || per) ? a : 0.0) - ((k < nz - 1 || per) ? cc : 0.0);
          const double d = dd[q] - mean;
          if (zero && k == 0) { cp = 0.0; dp = 0.0; }   // row 0: phi[0] = 0
          else {
            const double r = 1.0 / (b - a * cp);
            cp = cc * r; dp = (d - a * dp) * r;
          }
          if (!CPT) CP[col + st * k] = cp;
          A[col + st * k] = dp;
        }
      }
    }
    const double* __restrict__ CR = CPT ? CPT : CP;
    double x = dp;
    double s = x * c.dzf[nz - 1];
    for (int k0 = nz - 2; k0 >= 0; k0 -= TZ) {
      double dd[TZ], cc[TZ];
#pragma unroll
      for (int q = 0; q < TZ; ++q) {
        const int k = k0 - q;
        dd[q] = k >= 0 ? A[col + st * k] : 0.0; cc[q] = k >= 0 ? CR[col + st * k] : 0.0;
      }
#pragma unroll
      for (int q = 0; q < TZ; ++q) {
        const int k = k0 - q;
        if (k >= 0) {
          x = dd[q] - cc[q] * x;
          A[col + st * k] = x;
          s += x * c.dzf[k];
        }
      }
    }
    if (zero) {
      s /= c.lz;
      for (int k = 0; k < nz; ++k) A[col + st * k] -= s;
    }
    return;
  }
  // cyclic: A = T + u v^T, u = (g,0,..,0,c[n-1])^T, v = (1,0,..,0,a[0]/g)^T, g = -b[0]
  const double a0 = T.ak[0], cn = T.ck[nz - 1];
  const double b0 = lam - T.ak[0] - T.ck[0];
  const double g = -b0;
  double cp = 0.0, dp = 0.0, qp = 0.0;
  for (int k = 0; k < nz; ++k) {
    const double a = T.ak[k], cc = T.ck[k];
    double b = lam - a - cc;
    if (k == 0) b -= g;
    if (k == nz - 1) b -= a0 * cn / g;
    const double uu = k == 0 ? g : (k == nz - 1 ? cn : 0.0);
    const double d = A[col + st * k];
    const double r = 1.0 / (k == 0 ? b : b - a * cp);
    cp = cc * r;
    dp = (k == 0 ? d : d - a * dp) * r;
    qp = (k == 0 ? uu : uu - a * qp) * r;
    CP[col + st * k] = cp; A[col + st * k] = dp; CQ[col + st * k] = qp;
  }
  double y = dp, q = qp;
  const double yn = y, qn = q;
  for (int k = nz - 2; k >= 0; --k) {
    const double cpk = CP[col + st * k];
    y = A[col + st * k] - cpk * y;
    q = CQ[col + st * k] - cpk * q;
    A[col + st * k] = y; CQ[col + st * k] = q;
  }
  const double vy = y + a0 * yn / g, vq = q + a0 * qn / g;
  const double f = vy / (1.0 + vq);
  for (int k = 0; k < nz; ++k) A[col + st * k] -= f * CQ[col + st * k];
}

// c' of column (i,j) exactly as poisson_column's forward sweep forms it (same operations in the same order: the table holds the same
// bits the sweep would have spilled).  Non-periodic z only.
CALES_HD void poisson_cp_column(const Ctx& c, const PoissonTabs& T, int i, int j, double* __restrict__ CPT) {
  const int nz = c.nz;
  const long long col = (long long)i + (long long)c.nx * j, st = c.nxy;
  const double lam = T.lamx[i] + T.lamy[j];
  const bool zero = (i == 0 && j == 0);
  double cp = 0.0;
  for (int k = 0; k < nz; ++k) {
    const double a = T.ak[k], cc = T.ck[k];
    const double b = lam - (k > 0 ? a : 0.0) - (k < nz - 1 ? cc : 0.0);
    if (zero && k == 0) cp = 0.0;
    else { const double r = 1.0 / (b - a * cp); cp = cc * r; }
    CPT[col + st * k] = cp;
  }
}

// Helmholtz column (i,j) of Eq. 18: (1 - c (L_zz + lam_x + lam_y)) q = d in place, for a velocity
// component in the spectral (packed real) layout.  fam 0: centred in z (u, v) with the no-slip mirror ghost folded into the
// diagonal, or the zero-flux closure with the wall model (its lagged stress is a source outside the operator);
// fam 1: on z faces (w), unknowns k = 0..nz-2, w = 0 on the wall faces.  Periodic z: cyclic Thomas (Sherman-Morrison).
CALES_HD void helm_column(const Ctx& c, const PoissonTabs& T, int fam, double cimp, int i, int j, double* __restrict__ A,
                          double* __restrict__ CP, double* __restrict__ CQ) {
  const int nz = c.nz;
  const long long col = (long long)i + (long long)c.nx * j, st = c.nxy;
  const bool per = c.bc_z == BC_PER;
  const int m = (fam == 1 && !per) ? nz - 1 : nz;
  const double e = fam == 1 ? 1.0 : (c.wall_model ? 0.0 : 2.0);
  const double sh = 1.0 - cimp * (T.lamx[i] + T.lamy[j]);
  auto ak = [&](int k) { return fam == 0 ? T.ak[k] : c.rdzc[k] * c.rdzf[k]; };
  auto ck = [&](int k) { return fam == 0 ? T.ck[k] : c.rdzc[k] * c.rdzf[k + 1]; };
  auto diag = [&](int k) { return sh + cimp * (((k == 0 && !per) ? e : 1.0) * ak(k) + ((k == m - 1 && !per) ? e : 1.0) * ck(k)); };
  if (!per) {
    double cp = 0.0, dp = 0.0;
    for (int k = 0; k < m; ++k) {
      const double lo = -cimp * ak(k), up = -cimp * ck(k);
      const double r = 1.0 / (k == 0 ? diag(k) : diag(k) - lo * cp);
      cp = up * r; dp = (k == 0 ? A[col + st * k] : A[col + st * k] - lo * dp) * r;
      CP[col + st * k] = cp; A[col + st * k] = dp;
    }
    double x = dp;
    for (int k = m - 2; k >= 0; --k) { x = A[col + st * k] - CP[col + st * k] * x; A[col + st * k] = x; }
    for (int k = m; k < nz; ++k) A[col + st * k] = 0.0;
    return;
  }
  const double l0 = -cimp * ak(0), un = -cimp * ck(nz - 1);
  const double g = -diag(0);
  double cp = 0.0, dp = 0.0, qp = 0.0;
  for (int k = 0; k < nz; ++k) {
    const double lo = -cimp * ak(k), up = -cimp * ck(k);
    double b = diag(k);
    if (k == 0) b -= g;
    if (k == nz - 1) b -= l0 * un / g;
    const double uu = k == 0 ? g : (k == nz - 1 ? un : 0.0);
    const double d = A[col + st * k];
    const double r = 1.0 / (k == 0 ? b : b - lo * cp);
    cp = up * r;
    dp = (k == 0 ? d : d - lo * dp) * r;
    qp = (k == 0 ? uu : uu - lo * qp) * r;
    CP[col + st * k] = cp; A[col + st * k] = dp; CQ[col + st * k] = qp;
  }
  double y = dp, q = qp;
  const double yn = y, qn = q;
  for (int k = nz - 2; k >= 0; --k) {
    const double cpk = CP[col + st * k];
    y = A[col + st * k] - cpk * y;
    q = CQ[col + st * k] - cpk * q;
    A[col + st * k] = y; CQ[col + st * k] = q;
  }
  const double vy = y + l0 * yn / g, vq = q + l0 * qn / g;
  const double f = vy / (1.0 + vq);
  for (int k = 0; k < nz; ++k) A[col + st * k] -= f * CQ[col + st * k];
}

// Crank-Nicolson coefficients of Eq. 21 for substep constant cimp = gamma nu dt / 2, computed once per substep by one
// thread: for the centred components (u, v; no-slip ghost folded into the diagonal) and for w (faces 0..nz-2).
// Layout of `coef`: [0] lower a, [1] c' (modified upper), [2] 1/den for u,v; [3],[4],[5] the same for w.
CALES_HD void cn_coefficients(const Ctx& c, double cimp, double* coef) {
  const int nz = c.nz;
  double cp = 0.0;
  for (int k = 0; k < nz; ++k) {
    const double ak = 1.0 / (c.dzf[k] * c.dzc[k - 1]), ck = 1.0 / (c.dzf[k] * c.dzc[k]);
    double b = 1.0 + cimp * (ak + ck);
    // walls: no-slip ghost folded into the diagonal, or -- with the wall model, whose lagged stress is a source that cancels in
    // Eq. 21 -- the zero-flux closure
    if (k == 0) b += c.wall_model ? -cimp * ak : cimp * ak;
    if (k == nz - 1) b += c.wall_model ? -cimp * ck : cimp * ck;
    const double a = -cimp * ak, cc = -cimp * ck;
    const double r = 1.0 / (k == 0 ? b : b - a * cp);
    cp = cc * r;
    coef[0 * nz + k] = a; coef[1 * nz + k] = cp; coef[2 * nz + k] = r;
  }
  cp = 0.0;
  for (int k = 0; k < nz - 1; ++k) {
    const double ak = 1.0 / (c.dzc[k] * c.dzf[k]), ck = 1.0 / (c.dzc[k] * c.dzf[k + 1]);
    const double b = 1.0 + cimp * (ak + ck);
    const double a = -cimp * ak, cc = -cimp * ck;
    const double r = 1.0 / (k == 0 ? b : b - a * cp);
    cp = cc * r;
    coef[3 * nz + k] = a; coef[4 * nz + k] = cp; coef[5 * nz + k] = r;
  }
  coef[3 * nz + nz - 1] = 0.0; coef[4 * nz + nz - 1] = 0.0; coef[5 * nz + nz - 1] = 0.0;
}

// Solve (1 - c L_zz) q* = d in place for one column; m = number of unknowns (nz for u, v; nz-1 for w).
// Returns sum_k q*[k] dzf[k] (used for the bulk velocity of u*).
CALES_HD double cn_column(const Ctx& c, const double* coef, int m, long long col, double* __restrict__ Q) {
  const int nz = c.nz; const long long st = c.nxy;
  const double* a = coef; const double* cp = coef + nz; const double* r = coef + 2 * nz;
  enum { TZ = 8 };
  double dp = 0.0;
  for (int k0 = 0; k0 < m; k0 += TZ) {
    double dd[TZ];
#pragma unroll
    for (int q = 0; q < TZ; ++q) dd[q] = (k0 + q < m) ? Q[col + st * (k0 + q)] : 0.0;
#pragma unroll
    for (int q = 0; q < TZ; ++q) {
      const int k = k0 + q;
      if (k < m) {
        dp = (k == 0 ? dd[q] : dd[q] - a[k] * dp) * r[k];
        Q[col + st * k] = dp;
      }
    }
  }
  double x = dp, s = x * c.dzf[m - 1];
  for (int k0 = m - 2; k0 >= 0; k0 -= TZ) {
    double dd[TZ];
#pragma unroll
    for (int q = 0; q < TZ; ++q) dd[q] = (k0 - q >= 0) ? Q[col + st * (k0 - q)] : 0.0;
#pragma unroll
    for (int q = 0; q < TZ; ++q) {
      const int k = k0 - q;
      if (k >= 0) {
        x = dd[q] - cp[k] * x;
        Q[col + st * k] = x;
        s += x * c.dzf[k];
      }
    }
  }
  return s;
}

#ifdef __CUDACC__
__global__ void k_poisson_z(Ctx c, PoissonTabs T, double* __restrict__ A, double* __restrict__ CP, double* __restrict__ CQ, const double* __restrict__ CPT) {
  const long long col = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= c.nxy) return;
  poisson_column(c, T, (int)(col % c.nx), (int)(col / c.nx), A, CP, CQ, CPT);
}
// Two adjacent columns (i, i+1), i even, per thread with 16-byte loads and stores: the non-periodic solve with the static c' table
// (poisson_column's arithmetic on both lanes of a double2; k_correct gained 20 % from the wider accesses alone).  The thread that owns
// the singular column (0,0) falls back to poisson_column for its two columns.  grid over nxy/2 pairs.
__global__ void k_poisson_z2(Ctx c, PoissonTabs T, double* __restrict__ A, double* __restrict__ CP, const double* __restrict__ CPT) {
  const long long pr = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (pr >= c.nxy / 2) return;
  const int hx = c.nx / 2;
  const int j = (int)(pr / hx), i = 2 * (int)(pr - (long long)j * hx);
  if (i == 0 && j == 0) { poisson_column(c, T, 0, 0, A, CP, nullptr, CPT); poisson_column(c, T, 1, 0, A, CP, nullptr, CPT); return; }
  const int nz = c.nz;
  const long long col = (long long)i + (long long)c.nx * j, st = c.nxy;
  const double lam0 = T.lamx[i] + T.lamy[j], lam1 = T.lamx[i + 1] + T.lamy[j];
  enum { TZ = 8 };
  auto L2 = [](const double* q) { return *reinterpret_cast<const double2*>(q); };
  double cp0 = 0.0, cp1 = 0.0, dp0 = 0.0, dp1 = 0.0;
  for (int k0 = 0; k0 < nz; k0 += TZ) {
    double2 dd[TZ];
#pragma unroll
    for (int q = 0; q < TZ; ++q) dd[q] = (k0 + q < nz) ? L2(A + col + st * (k0 + q)) : make_double2(0.0, 0.0);
#pragma unroll
    for (int q = 0; q < TZ; ++q) {
      const int k = k0 + q;
      if (k < nz) {
        const double a = T.ak[k], cc = T.ck[k];
        const double off = (k > 0 ? a : 0.0) + (k < nz - 1 ? cc : 0.0);
        const double b0 = lam0 - (k > 0 ? a : 0.0) - (k < nz - 1 ? cc : 0.0), b1 = lam1 - (k > 0 ? a : 0.0) - (k < nz - 1 ? cc : 0.0);
        (void)off;
        const double r0 = 1.0 / (b0 - a * cp0), r1 = 1.0 / (b1 - a * cp1);
        cp0 = cc * r0; dp0 = (dd[q].x - a * dp0) * r0;
        cp1 = cc * r1; dp1 = (dd[q].y - a * dp1) * r1;
        *reinterpret_cast<double2*>(A + col + st * k) = make_double2(dp0, dp1);
      }
    }
  }
  double x0 = dp0, x1 = dp1;
  for (int k0 = nz - 2; k0 >= 0; k0 -= TZ) {
    double2 dd[TZ], cc[TZ];
#pragma unroll
    for (int q = 0; q < TZ; ++q) {
      const int k = k0 - q;
      dd[q] = k >= 0 ? L2(A + col + st * k) : make_double2(0.0, 0.0); cc[q] = k >= 0 ? L2(CPT + col + st * k) : make_double2(0.0, 0.0);
    }
#pragma unroll
    for (int q = 0; q < TZ; ++q) {
      const int k = k0 - q;
      if (k >= 0) {
        x0 = dd[q].x - cc[q].x * x0; x1 = dd[q].y - cc[q].y * x1;
        *reinterpret_cast<double2*>(A + col + st * k) = make_double2(x0, x1);
      }
    }
  }
}
__global__ void k_poisson_cp(Ctx c, PoissonTabs T, double* __restrict__ CPT) {
  const long long col = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= c.nxy) return;
  poisson_cp_column(c, T, (int)(col % c.nx), (int)(col / c.nx), CPT);
}
__global__ void k_helm_z(Ctx c, PoissonTabs T, int fam, const double* __restrict__ sc, double* __restrict__ A, double* __restrict__ CP, double* __restrict__ CQ) {
  const long long col = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= c.nxy) return;
  helm_column(c, T, fam, sc[3], (int)(col % c.nx), (int)(col / c.nx), A, CP, CQ);
}
// Crank-Nicolson tables of the three substeps built on the device from the substep scalar blocks (one thread per substep: the
// forward elimination of the constant matrix is a serial recurrence over nz levels).  coef: [3][6][nz], sc: [3][4].
__global__ void k_cn_coef(Ctx c, const double* __restrict__ sc, double* __restrict__ coef) {
  if (threadIdx.x < 3) cn_coefficients(c, sc[threadIdx.x * 4 + 3], coef + (size_t)threadIdx.x * 6 * c.nz);
}
// partial[block] = sum over the block's points of q dzf[k] (bulk velocity of u* after the Helmholtz solves); grid/block of the point kernels
__global__ void __launch_bounds__(256) k_weighted_sum(Ctx c, const double* __restrict__ q, double* __restrict__ partial) {
  __shared__ double red[32];
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
  const double s = (i < c.nx && j < c.ny) ? q[idx3(c, i, j, k)] * c.dzf[k] : 0.0;
  const double t = block_sum(s, red);
  if (threadIdx.x == 0 && threadIdx.y == 0) partial[blockIdx.x + gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z)] = t;
}
// grid (ceil(nxy / blockDim), 3): blockIdx.y = component (0 u, 1 v, 2 w), one launch for the three independent solves so that
// small planes still fill the machine.  For u the dzf-weighted column sums are reduced per block into partial[blockIdx.x].
__global__ void k_cn_z(Ctx c, const double* __restrict__ coef, double* __restrict__ us, double* __restrict__ vs, double* __restrict__ ws,
                       double* __restrict__ partial) {
  __shared__ double sh[32];
  const int comp = blockIdx.y;
  double* Q = comp == 0 ? us : (comp == 1 ? vs : ws);
  const long long col = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double s = 0.0;
  if (col < c.nxy) {
    const int j = (int)(col / c.nx);
    const bool skip = (comp == 1 && c.bc_y == BC_WALL && j == c.ny - 1);   // the +y wall face stays 0
    if (!skip) s = cn_column(c, comp == 2 ? coef + 3 * c.nz : coef, comp == 2 ? c.nz - 1 : c.nz, col, Q);
  }
  if (comp == 0 && partial) {
    const double t = block_sum(s, sh);
    if (threadIdx.x == 0) partial[blockIdx.x] = t;
  }
}
#endif

}  // namespace cales
