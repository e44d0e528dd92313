// cales_smag_tile.cuh -- static Smagorinsky eddy viscosity (Eq. 4) as a z-marching, shared-memory staged
// stencil: the same staging scheme as the momentum kernel (cales_rhs_tile.cuh) for the three velocity components with
// the strain-rate ghosts (GH_STRAIN: no-slip mirror, or one-sided extrapolation at a wall-model wall).
// Every velocity value is fetched once per CTA by cp.async one plane ahead; the 36 stencil reads of the strain rate
// are shared-memory reads.
#pragma once
#include "cales_common.cuh"
#include "cales_closures.cuh"
#include "cales_rhs_tile.cuh"

namespace cales {

enum { ST_NF = 3, ST_SMEM_DOUBLES = RT_NSLOT * ST_NF * RT_PLANE };

// velocity component f (0 u, 1 v, 2 w) at (gi,gj,gk) incl. ghosts, as the strain rate sees it
CALES_HD double st_elem(const Ctx& c, const double* u, const double* v, const double* w, int f, int gi, int gj, int gk) {
  if (f == 0) return velg<0>(c, u, gi, gj, gk, GH_STRAIN);
  if (f == 1) return velg<1>(c, v, gi, gj, gk, GH_STRAIN);
  return velg<2>(c, w, gi, gj, gk, GH_STRAIN);
}

// nu_t at one point from three staged planes (sl[d] -> field 0 of plane k-1+d; ctr as in TileAcc);
// tauw[0], tauw[1]: u_tau = sqrt(nu |u_c| / d1) at the bottom / top wall of this column (van Driest only, S5)
CALES_HD double smag_tile_point(const Ctx& c, const double* const* sl, int ctr, int k, const double* tauw) {
  auto at = [&](int f, int a, int b, int d) { return sl[d + 1][f * RT_PLANE + ctr + b * RT_TW + a]; };
  auto U = [&](int a, int b, int d) { return at(0, a, b, d); };
  auto V = [&](int a, int b, int d) { return at(1, a, b, d); };
  auto W = [&](int a, int b, int d) { return at(2, a, b, d); };
  double S[6];
  const double smag = strain_at(U, V, W, c.rdx, c.rdy, c.rdzf[k], c.rdzc[k], c.rdzc[k - 1], S);
  double D = 1.0;
  if (c.van_driest) {
    const double db = c.zc[k], dt = c.lz - c.zc[k];
    const double d = (db <= dt) ? db : dt;
    const double utau = (db <= dt) ? tauw[0] : tauw[1];          // u_tau of the nearer wall (precomputed per column)
    D = 1.0 - exp(-(d * utau) * c.rnuap);
  }
  const double l = c.cs * c.delta[k] * D;
  return l * l * smag;
}

// local friction velocity of the van Driest damping for column (i,j): tauw[0] bottom, tauw[1] top (as in smag_point)
CALES_HD void smag_wall_shear(const Ctx& c, const double* u, const double* v, int i, int j, double* tauw) {
  for (int wl = 0; wl < 2; ++wl) {
    const int kw = wl == 0 ? 0 : c.nz - 1;
    const double d1 = wl == 0 ? c.zc[0] : c.lz - c.zc[c.nz - 1];
    const double uc = 0.5 * (velg<0>(c, u, i - 1, j, kw, GH_STRAIN) + velg<0>(c, u, i, j, kw, GH_STRAIN));
    const double vc = 0.5 * (velg<1>(c, v, i, j - 1, kw, GH_STRAIN) + velg<1>(c, v, i, j, kw, GH_STRAIN));
    tauw[wl] = sqrt(c.nu * sqrt(uc * uc + vc * vc) / d1);        // u_tau = sqrt(tau_w)
  }
}

#ifdef __CUDACC__
// grid (ceil(nx/RT_TX), ceil(ny/RT_TY), ceil(nz/kz)), block RT_THREADS, dynamic smem ST_SMEM_DOUBLES*8
__global__ void __launch_bounds__(RT_THREADS, 3) k_smag_tile(const __grid_constant__ Ctx c, const double* __restrict__ u, const double* __restrict__ v,
                                                             const double* __restrict__ w, int kz, double* __restrict__ nut) {
  extern __shared__ double st_sm[];
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const int i0 = blockIdx.x * RT_TX, j0 = blockIdx.y * RT_TY, k0 = blockIdx.z * kz, k1 = min(k0 + kz, c.nz);
  int goff[RT_EPT];      // in-plane global offset (>= 0: async copy; -1: unused; -2: y ghost, generic path)
#pragma unroll
  for (int e = 0; e < RT_EPT; ++e) {
    const int pos = tid + e * RT_THREADS;
    goff[e] = -1;
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
  const double* fld[ST_NF] = {u, v, w};
  auto issue = [&](int kk) {
    double* slot = st_sm + ((kk + 4) & 3) * (ST_NF * RT_PLANE);
    const bool zreg = c.bc_z == BC_PER || (kk >= 0 && kk < c.nz);
    const long long kw = (long long)(kk < 0 ? kk + c.nz : (kk >= c.nz ? kk - c.nz : kk)) * c.nxy;
#pragma unroll
    for (int e = 0; e < RT_EPT; ++e) {
      const int pos = tid + e * RT_THREADS;
      if (goff[e] == -1) continue;
      if (zreg && goff[e] >= 0) {
#pragma unroll
        for (int f = 0; f < ST_NF; ++f) cp_async8(slot + f * RT_PLANE + pos, fld[f] + kw + goff[e]);
      } else {
        const int ry = pos / RT_TW, rx = pos - ry * RT_TW;
#pragma unroll
        for (int f = 0; f < ST_NF; ++f) slot[f * RT_PLANE + pos] = st_elem(c, u, v, w, f, i0 - 1 + rx, j0 - 1 + ry, kk);
      }
    }
  };
  issue(k0 - 1); issue(k0);
  if (k0 + 1 <= k1) issue(k0 + 1);
  cp_async_commit();
  double tauw[RT_RPT][2];
#pragma unroll
  for (int r = 0; r < RT_RPT; ++r) {
    tauw[r][0] = tauw[r][1] = 0.0;
    const int i = i0 + tx, j = j0 + ty * RT_RPT + r;
    if (c.van_driest && i < c.nx && j < c.ny) smag_wall_shear(c, u, v, i, j, tauw[r]);
  }
  for (int k = k0; k < k1; ++k) {
    cp_async_wait_all();
    __syncthreads();
    if (k + 2 <= k1) issue(k + 2);
    cp_async_commit();
    const double* sl[3] = {st_sm + ((k + 3) & 3) * (ST_NF * RT_PLANE), st_sm + (k & 3) * (ST_NF * RT_PLANE), st_sm + ((k + 1) & 3) * (ST_NF * RT_PLANE)};
#pragma unroll
    for (int r = 0; r < RT_RPT; ++r) {
      const int ly = ty * RT_RPT + r, i = i0 + tx, j = j0 + ly;   // adjacent rows: their stencils share shared-memory loads
      if (i < c.nx && j < c.ny) nut[idx3(c, i, j, k)] = smag_tile_point(c, sl, (ly + 1) * RT_TW + tx + 1, k, tauw[r]);
    }
  }
}
#endif

}  // namespace cales
