// cales_common.cuh -- device-side context, boundary-condition accessors and small reductions.
//
// The GPU keeps NO ghost layers: every array holds interior values only,
// [k][j][i] with x fastest, and the boundary conditions of PAPER.md:142 / Alg. 2 are
// applied by index arithmetic when a neighbour is read.  The accessors below are the single place where
// that happens.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#define CALES_HD __host__ __device__ __forceinline__

namespace cales {

enum { BC_PER = 0, BC_WALL = 1 };
enum { GH_VISC = 0, GH_STRAIN = 1 };  // ghost of the wall-parallel velocity at a wall-model wall

// Grid, options and table pointers, passed by value to every kernel.
struct Ctx {
  int nx, ny, nz;
  int bc_y, bc_z, wall_model, wall_model_y, sgs, van_driest, implicit_z, dsm_plane, dsm_clip_total, dsm_filter3d, const_flow_rate;
  int wm_maxit;   // implicit_z above: 0 explicit diffusion, 1 Crank-Nicolson in z (Eq. 20-22), 2 in all three directions (Eq. 17-19)
  int wy_q1;       // y-wall model: the sample lies between centres wy_q1 and wy_q1 + 1 counted from the wall
  long long N;     // nx*ny*nz
  long long nxy;   // nx*ny
  double dx, dy, rdx, rdy, rnuap /* 1/(nu A+) */, lz, nu, cs, aplus, alpha, kappa, Blog, h_wm, wm_tol, u_bulk, wy_wgt /* interpolation weight */, wy_h /* sampling distance */;
  // 1-D grid tables in device memory, offset so that the ghost entries are addressable:
  const double* dzf;   // dzf[-1 .. nz]   cell heights (ghost = neighbour's / wrapped)
  const double* dzc;   // dzc[-1 .. nz-1] centre spacings across face k+1 (mirrored ghost centre at walls)
  const double* zc;    // zc[0 .. nz-1]
  const double* rdzf;  // 1/dzf[-1 .. nz]
  const double* rdzc;  // 1/dzc[-1 .. nz-1]
  const double* delta; // filter width Delta_k = (dx dy dzf[k])^(1/3), k = 0..nz-1 (S4)
  const double* tau;   // wall stress planes [wall][comp][ny][nx]
  const double* tau_y; // y-wall stress planes [wall][comp (0 tau_xy at u points, 1 tau_zy at w points)][nz][nx]
};

CALES_HD long long idx3(const Ctx& c, int i, int j, int k) { return (long long)i + (long long)c.nx * ((long long)j + (long long)c.ny * (long long)k); }
CALES_HD int wrapi(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

// Velocity component COMP (0 u, 1 v, 2 w) at (i,j,k) with -1 <= i <= nx, -1 <= j <= ny, -1 <= k <= nz.
// Ghosts compose in the order z, then x, then y (as an explicit ghost fill would):
//   x periodic;  y periodic, or walls: u, w mirrored (no slip), v = 0 on the wall faces and beyond;
//   z periodic, or walls: w = 0 on the wall faces and beyond; u, v: no-slip mirror, or with the wall model
//   GH_VISC   ghost = q0 - tau * dzc_wall / nu       (the modelled stress is the wall viscous flux)
//   GH_STRAIN ghost = linear extrapolation of q0, q1 (one-sided derivative for the strain rate).
// x already wrapped, 0 <= j < ny: periodic wrap or wall ghosts in z only
template <int COMP>
CALES_HD double velg_z(const Ctx& c, const double* __restrict__ q, int i, int j, int k, int mode) {
  if (c.bc_z == BC_PER) return q[idx3(c, i, j, wrapi(k, c.nz))];
  if (COMP == 2) { if (k < 0 || k >= c.nz - 1) return 0.0; return q[idx3(c, i, j, k)]; }
  if (k >= 0 && k < c.nz) return q[idx3(c, i, j, k)];
  const bool bottom = k < 0;
  const int k0 = bottom ? 0 : c.nz - 1;
  const double q0 = q[idx3(c, i, j, k0)];
  if (!c.wall_model) return -q0;
  if (mode == GH_VISC) {
    const double t = c.tau[((long long)((bottom ? 0 : 2) + COMP) * c.ny + j) * c.nx + i];
    const double dz = bottom ? c.dzc[-1] : c.dzc[c.nz - 1];
    return q0 - t * dz / c.nu;
  }
  const int k1 = bottom ? 1 : c.nz - 2;
  const double q1 = q[idx3(c, i, j, k1)];
  const double r = bottom ? c.dzc[-1] / c.dzc[0] : c.dzc[c.nz - 1] / c.dzc[c.nz - 2];
  return q0 + (q0 - q1) * r;
}
template <int COMP>
CALES_HD double velg(const Ctx& c, const double* __restrict__ q, int i, int j, int k, int mode) {
  i = wrapi(i, c.nx);
  if (c.bc_y == BC_PER) return velg_z<COMP>(c, q, i, wrapi(j, c.ny), k, mode);
  if (COMP == 1) { if (j < 0 || j >= c.ny - 1) return 0.0; return velg_z<COMP>(c, q, i, j, k, mode); }
  if (j >= 0 && j < c.ny) return velg_z<COMP>(c, q, i, j, k, mode);
  const bool low = j < 0;
  const int j0 = low ? 0 : c.ny - 1;
  const double q0 = velg_z<COMP>(c, q, i, j0, k, mode);
  if (!c.wall_model_y) return -q0;                       // no-slip mirror
  // wall model on the y walls (duct WMLES): same two ghost kinds as in z, uniform spacing dy
  if (mode == GH_VISC) {
    const int kk = k < 0 ? 0 : (k >= c.nz ? c.nz - 1 : k);
    const double t = c.tau_y[((long long)((low ? 0 : 2) + (COMP == 0 ? 0 : 1)) * c.nz + kk) * c.nx + i];
    return q0 - t * c.dy / c.nu;
  }
  return 2.0 * q0 - velg_z<COMP>(c, q, i, low ? 1 : c.ny - 2, k, mode);
}

// Cell-centred scalar with ghost = sgn * interior at walls (sgn = +1: Neumann, p and phi; sgn = -1: nu_t,
// which makes the edge viscosity and hence the SGS flux vanish on a wall) and periodic wrap otherwise.
CALES_HD double scalg(const Ctx& c, const double* __restrict__ q, int i, int j, int k, double sgn) {
  i = wrapi(i, c.nx);
  double s = 1.0;
  if (c.bc_y == BC_PER) j = wrapi(j, c.ny);
  else { if (j < 0) { j = 0; s *= sgn; } else if (j >= c.ny) { j = c.ny - 1; s *= sgn; } }
  if (c.bc_z == BC_PER) k = wrapi(k, c.nz);
  else { if (k < 0) { k = 0; s *= sgn; } else if (k >= c.nz) { k = c.nz - 1; s *= sgn; } }
  return s * q[idx3(c, i, j, k)];
}

// True when none of the neighbours of (.,j,k) read by the momentum / strain-rate stencils needs a wall ghost: periodic wrap is
// plain index arithmetic, wall rows/planes go through the generic accessors.  Relies on the library keeping the wall
// faces v[.][ny-1][.] and w[nz-1] at exactly 0 (cales_set_field zeroes them).
CALES_HD bool interior_row(const Ctx& c, int j, int k) {
  const bool yok = c.bc_y == BC_PER || (j >= 1 && j <= c.ny - 2);
  const bool zok = c.bc_z == BC_PER || (k >= 1 && k <= c.nz - 2);
  return yok && zok;
}

// Neighbour offsets of an interior point (periodic wrap only).
struct Nbr { int im, ip, jm, jp; long long km, kp; };
CALES_HD Nbr neighbours(const Ctx& c, int i, int j, int k) {
  Nbr o;
  o.im = (i == 0) ? c.nx - 1 : -1;
  o.ip = (i == c.nx - 1) ? -(c.nx - 1) : 1;
  o.jm = (j == 0) ? (c.ny - 1) * c.nx : -c.nx;
  o.jp = (j == c.ny - 1) ? -(c.ny - 1) * c.nx : c.nx;
  o.km = (k == 0) ? (long long)(c.nz - 1) * c.nxy : -c.nxy;
  o.kp = (k == c.nz - 1) ? -(long long)(c.nz - 1) * c.nxy : c.nxy;
  return o;
}

// A scalar that every thread of a large grid reads from the same device address (substep scalars, bulk shift): through the
// read-only path with the L1 evict-last policy, so that the line stays resident in each SM's (small, streamed-through) L1 and the
// one L2 slice that owns it is not hammered by every warp of the grid (measured on B200: k_correct 10.7 -> 16 ms with plain loads).
CALES_HD double ld_scalar(const double* p) {
#ifdef __CUDA_ARCH__
  double v;
  asm("ld.global.nc.L1::evict_last.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
#else
  return *p;
#endif
}

// two adjacent scalars (16-byte aligned) in one load
CALES_HD void ld_scalar2(const double* p, double& a, double& b) {
#ifdef __CUDA_ARCH__
  asm("ld.global.nc.L1::evict_last.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "l"(p));
#else
  a = p[0]; b = p[1];
#endif
}

// RK3 coefficients of PAPER.md:100.
CALES_HD void rk3_coeffs(int rk, double& al, double& be, double& ga) {
  al = rk == 0 ? 8.0 / 15.0 : (rk == 1 ? 5.0 / 12.0 : 3.0 / 4.0);
  be = rk == 0 ? 0.0 : (rk == 1 ? -17.0 / 60.0 : -5.0 / 12.0);
  ga = al + be;
}

#ifdef __CUDACC__
// 8-byte asynchronous global -> shared copies (LDGSTS)
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(gsrc) : "memory");
}
// 16-byte form (LDGSTS.128, L2 only): both addresses 16-byte aligned
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// A global load the compiler may not sink below later volatile asm (barriers, cp.async waits): used to put long-latency loads in
// flight ahead of a wait.  Read-only path (.nc): the address must not be written by another thread during the kernel.
__device__ __forceinline__ double ldg_early(const double* p) {
  double v;
  asm volatile("ld.global.nc.f64 %0, [%1];\n" : "=d"(v) : "l"(p));
  return v;
}

// ---- mbarrier + 1-D bulk asynchronous copies (cp.async.bulk, the TMA engine without a tensor map; SASS: UBLKCP / SYNCS).
// One thread arms the barrier with the byte count and issues the copies; every consumer waits on the phase parity.
// Source, destination and size must be multiples of 16 bytes.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// plain arrival (no bytes expected): flips the phase of a barrier of count 1
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
// 3-D tiled TMA load (cp.async.bulk.tensor, SASS: UTMALDG): box of the tensor map at element coordinates (c0, c1, c2) into
// shared memory (128-byte aligned), completing on the mbarrier; out-of-range elements arrive as zeros.
__device__ __forceinline__ void tma_load_3d(void* smem_dst, const void* tmap, int c0, int c1, int c2, unsigned long long* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n"
               ::"r"(smem_u32(smem_dst)), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

// Sum over the thread block (result valid in thread 0).  blockDim.x*y*z <= 1024, multiple of 32.
__device__ __forceinline__ double block_sum(double v, double* sh /* >= 32 doubles */) {
  const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
  const int nth = blockDim.x * blockDim.y * blockDim.z;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((tid & 31) == 0) sh[tid >> 5] = v;
  __syncthreads();
  double r = 0.0;
  if (tid < 32) {
    r = (tid < (nth + 31) / 32) ? sh[tid] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
  }
  __syncthreads();
  return r;
}
__device__ __forceinline__ double block_max(double v, double* sh) {
  const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
  const int nth = blockDim.x * blockDim.y * blockDim.z;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
  if ((tid & 31) == 0) sh[tid >> 5] = v;
  __syncthreads();
  double r = 0.0;
  if (tid < 32) {
    r = (tid < (nth + 31) / 32) ? sh[tid] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r = fmax(r, __shfl_down_sync(0xffffffffu, r, o));
  }
  __syncthreads();
  return r;
}
#endif

}  // namespace cales
