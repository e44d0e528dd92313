// cales_fft.cuh -- hand-written batched real transforms of the eigenfunction-expansion Poisson solver
// (FFT-based eigenfunction expansion; the paper calls cuFFT, this path does not).
//
// Formulation: everything is REAL-to-REAL in "packed half-complex" form, so the
// spectral array has exactly nx*ny*nz doubles and every (i,j) column is one real tridiagonal system:
//   a real line x[0..n-1] (n even) -> h[0] = X[0], h[1] = X[n/2], h[2m] = Re X[m], h[2m+1] = Im X[m], 0<m<n/2,
//   X[m] = sum_j x[j] exp(-2 pi i m j / n).  Re and Im of an x-mode transform independently along y.
//   Neumann (wall) y: DCT-II  X[n] = sum_j x[j] cos(pi n (2j+1)/(2N)), row n holds mode n; inverse DCT-III.
// A real transform of length n is one complex Stockham FFT of length n2 = n/2 on z[t] = x[2t] + i x[2t+1] plus a
// split (forward) or merge (inverse) step; the DCT adds the even/odd permutation and a quarter-wave twiddle.  All
// twiddles come from host-built tables (long double, rounded once).  This header holds the plan, the small in-register
// DFTs (radix 2, 3, 4, 8, 16), the forward split and the standalone tiled transpose; the kernels are in cales_fft2.cuh.
//
// Every phase is a __host__ __device__ function of (tid, nth) so that the identical code can be stepped phase by
// phase on the host by the test emulator (tests/emu); __syncthreads() sits between phases in the kernels only.
#pragma once
#include "cales_common.cuh"

namespace cales {

struct FftPlan {
  int n;            // real length
  int n2;           // n/2, length of the complex FFT
  int npass;
  int radix[20];
  int per[20], ns[20];          // butterflies per line and product of the previous radices, per pass
  unsigned mper[20], mns[20];   // ceil(2^32 / per), ceil(2^32 / ns) for the division-free index split (cales_fft2.cuh)
  const double2* tw;    // tw[q] = exp(-2 pi i q / n), q = 0..n-1
  const double2* dctw;  // dctw[m] = exp(-i pi m / (2 n)), m = 0..n/2   (DCT only)
};

CALES_HD double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
CALES_HD double2 cmulc(double2 a, double2 b) { return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }  // a * conj(b)
CALES_HD double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
CALES_HD double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }

// Shared-memory view of B lines of n2 complex numbers.  x layout (bfast = false): line b is contiguous with one padding
// slot per 8 elements (element t at b*ls + t + t/8), which makes the stride-R writes of the first Stockham passes
// bank-conflict free for R <= 8; y layout (bfast = true): element (b, t) at t*es + b, consecutive threads on consecutive b.
struct SmView { int es, ls, B; bool bfast; };
CALES_HD int sm_pad(int t) { return t + (t >> 3); }
CALES_HD int sm_off(const SmView& v, int b, int t) { return v.bfast ? b * v.ls + t * v.es : b * v.ls + sm_pad(t); }
CALES_HD int sm_line(int n2) { return sm_pad(n2) + 1; }   // line stride of the x layout

// ---- small in-register DFTs, natural order in and out, s = -1 forward / +1 inverse --------------------------------
CALES_HD double2 cmul_i(double2 a, int s) { return s < 0 ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x); }   // a * (s i)
CALES_HD void dft2(double2& a, double2& b) { const double2 t = a; a = cadd(t, b); b = csub(t, b); }
CALES_HD void dft3(double2& a, double2& b, double2& c, int s) {
  const double s3 = 0.86602540378443864676372317075294;
  const double2 t1 = cadd(b, c);
  const double2 t2 = make_double2(a.x - 0.5 * t1.x, a.y - 0.5 * t1.y);
  const double2 d = csub(b, c);
  const double2 id = make_double2(-s3 * d.y, s3 * d.x);   // i * s3 * d
  a = cadd(a, t1);
  b = s < 0 ? csub(t2, id) : cadd(t2, id);
  c = s < 0 ? cadd(t2, id) : csub(t2, id);
}
CALES_HD void dft4(double2& v0, double2& v1, double2& v2, double2& v3, int s) {
  const double2 a0 = cadd(v0, v2), a1 = csub(v0, v2), a2 = cadd(v1, v3), a3 = cmul_i(csub(v1, v3), s);
  v0 = cadd(a0, a2); v1 = cadd(a1, a3); v2 = csub(a0, a2); v3 = csub(a1, a3);
}
// a * exp(s i pi m / 8) for the constants the radix-8 / radix-16 butterflies need
template <int M>
CALES_HD double2 cmul_w16(double2 a, int s) {
  const double c1 = 0.92387953251128675612818318939679, s1 = 0.38268343236508977172845998403040, r2 = 0.70710678118654752440084436210485;
  const double sg = s < 0 ? -1.0 : 1.0;
  if (M == 0) return a;
  if (M == 4) return cmul_i(a, s);
  double cr, ci;
  if (M == 1) { cr = c1; ci = s1; } else if (M == 2) { cr = r2; ci = r2; } else if (M == 3) { cr = s1; ci = c1; }
  else if (M == 6) { cr = -r2; ci = r2; } else /* M == 9 */ { cr = -c1; ci = -s1; }
  ci *= sg;
  return make_double2(a.x * cr - a.y * ci, a.x * ci + a.y * cr);
}
CALES_HD void dft8(double2* v, int s) {
  dft4(v[0], v[2], v[4], v[6], s);
  dft4(v[1], v[3], v[5], v[7], s);
  const double2 o1 = cmul_w16<2>(v[3], s), o2 = cmul_i(v[5], s), o3 = cmul_w16<6>(v[7], s);
  const double2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
  v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
  v[1] = cadd(e1, o1); v[5] = csub(e1, o1);
  v[2] = cadd(e2, o2); v[6] = csub(e2, o2);
  v[3] = cadd(e3, o3); v[7] = csub(e3, o3);
}
CALES_HD void dft16(double2* v, int s) {
  // n = 4a + b: step 1, DFT-4 over a for each b; step 2, twiddle W16^(b t1); step 3, DFT-4 over b for each t1
#pragma unroll
  for (int b = 0; b < 4; ++b) dft4(v[b], v[4 + b], v[8 + b], v[12 + b], s);      // v[4 t1 + b] = Y_b[t1]
  v[5] = cmul_w16<1>(v[5], s); v[6] = cmul_w16<2>(v[6], s); v[7] = cmul_w16<3>(v[7], s);
  v[9] = cmul_w16<2>(v[9], s); v[10] = cmul_w16<4>(v[10], s); v[11] = cmul_w16<6>(v[11], s);
  v[13] = cmul_w16<3>(v[13], s); v[14] = cmul_w16<6>(v[14], s); v[15] = cmul_w16<9>(v[15], s);
#pragma unroll
  for (int t1 = 0; t1 < 4; ++t1) dft4(v[4 * t1], v[4 * t1 + 1], v[4 * t1 + 2], v[4 * t1 + 3], s);   // v[4 t1 + t2] = X[t1 + 4 t2]
  // to natural order: X[m], m = t1 + 4 t2, sits at 4 t1 + t2 (a 4x4 transpose)
#pragma unroll
  for (int t1 = 0; t1 < 4; ++t1)
#pragma unroll
    for (int t2 = t1 + 1; t2 < 4; ++t2) { const double2 t = v[4 * t1 + t2]; v[4 * t1 + t2] = v[4 * t2 + t1]; v[4 * t2 + t1] = t; }
}
template <int R> CALES_HD void dft_small(double2* v, int s) {
  if (R == 2) dft2(v[0], v[1]);
  else if (R == 3) dft3(v[0], v[1], v[2], s);
  else if (R == 4) dft4(v[0], v[1], v[2], v[3], s);
  else if (R == 8) dft8(v, s);
  else dft16(v, s);
}

// ---- forward split: Z (complex FFT of the packed line) -> half-complex X[m]; thread handles (b, m), m = 0..n2-1.
// Returns through `emit(b, slotA, valA, slotB, valB)`: two real outputs per (b, m).
//   FFT mode: slots (2m, 2m+1) (m = 0: X[0], X[n2]).
//   DCT mode: slots (m, N-m)   (m = 0: modes 0 and N/2).
template <class Emit>
CALES_HD void split_forward(int tid, int nth, const double2* Z, const SmView& sv, const FftPlan& pl, bool dct, int nbvalid, Emit emit) {
  const int n2 = pl.n2, total = n2 * sv.B;
  for (int idx = tid; idx < total; idx += nth) {
    int b, m;
    if (sv.bfast) { b = idx % sv.B; m = idx / sv.B; } else { m = idx % n2; b = idx / n2; }
    if (b >= nbvalid) continue;
    if (m == 0) {
      const double2 z0 = Z[sm_off(sv, b, 0)];
      const double x0 = z0.x + z0.y, xn = z0.x - z0.y;
      if (!dct) emit(b, 0, x0, 1, xn);
      else emit(b, 0, x0, n2, xn * 0.70710678118654752440084436210485);
      continue;
    }
    const double2 zm = Z[sm_off(sv, b, m)];
    double2 zc = Z[sm_off(sv, b, n2 - m)]; zc.y = -zc.y;
    const double2 e = make_double2(0.5 * (zm.x + zc.x), 0.5 * (zm.y + zc.y));
    const double2 d = make_double2(0.5 * (zm.x - zc.x), 0.5 * (zm.y - zc.y));
    // X = e - i * W^m * d
    const double2 wd = cmul(pl.tw[m], d);
    const double2 X = make_double2(e.x + wd.y, e.y - wd.x);
    if (!dct) emit(b, 2 * m, X.x, 2 * m + 1, X.y);
    else { const double2 t = cmul(pl.dctw[m], X); emit(b, m, t.x, pl.n - m, -t.y); }
  }
}

// position in the packed complex line of real sample r of the (possibly DCT-permuted) input:
//   FFT: v = x.   DCT-II: v[q] = x[2q] (q < N/2), v[N-1-q'] = x[2q'+1].
CALES_HD int perm_fwd(int r, int n, bool dct) {
  if (!dct) return r;
  return (r & 1) ? (n - 1 - (r >> 1)) : (r >> 1);
}

// ------------------------------------------------------------------------------------------------------------
// x transforms: lines are contiguous in memory.  One CTA transforms B lines.  The forward kernel can build its
// input on the fly as the Poisson right-hand side f = div(u*)/(gamma dt) (Eq. 12), so the
// divergence never touches HBM.  Phases (load / passes / store) are separated by block barriers.
// ------------------------------------------------------------------------------------------------------------
struct DivSrc { const double* us; const double* vs; const double* ws; double inv_gdt; const double* sc; };   // sc: substep scalar block (1/(gamma dt) at index 2) or nullptr

CALES_HD double2 ld2(const double* p, int t) { return reinterpret_cast<const double2*>(p)[t]; }

#ifdef __CUDACC__
// Tiled shared-memory transpose of every k-plane: dst[k][i][j] = src[k][j][i]  (32x32 tiles, padded).
__global__ void k_transpose_xy(int nx, int ny, const double* __restrict__ src, double* __restrict__ dst) {
  __shared__ double tile[32][33];
  const long long plane = (long long)nx * ny;
  const double* s = src + plane * blockIdx.z;
  double* d = dst + plane * blockIdx.z;
  const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    const int i = i0 + threadIdx.x, j = j0 + r;
    if (i < nx && j < ny) tile[r][threadIdx.x] = s[(long long)j * nx + i];
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    const int j = j0 + threadIdx.x, i = i0 + r;
    if (i < nx && j < ny) d[(long long)i * ny + j] = tile[threadIdx.x][r];
  }
}
#endif  // __CUDACC__

}  // namespace cales
