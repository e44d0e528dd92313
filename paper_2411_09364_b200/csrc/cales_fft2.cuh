// cales_fft2.cuh -- production transform kernels of the Poisson solver: in-place, register-resident
// Stockham passes.
//
// A CTA owns L lines (x: L whole lines, contiguous, padded; y: a [ny x TI] tile whose rows are TI-column segments, so
// the x<->y transpose of the pencil solver is fused into the load and the store).  Every thread keeps F2_E = 16 complex
// elements of the current pass in registers (one radix-16, two radix-8, four radix-4, eight radix-2 or five radix-3
// butterflies), so a pass is:   registers <- source;  barrier;  butterflies + twiddles;  registers -> destination.
// The FIRST pass reads straight from global memory (for the forward x transform it builds the divergence of u* on
// the fly, Eq. 12; for the inverse transforms it applies the half-complex / DCT-III merge on the fly) and the LAST
// pass of an inverse transform writes straight to global memory, so shared memory holds ONE buffer per line, is
// touched once per pass, and 2-4 CTAs per SM overlap their global-load, butterfly and store phases.
// Everything except the barriers is __host__ __device__ so that tests/emu can step the same code.
#pragma once
#include "cales_fft.cuh"

namespace cales {

#ifndef CALES_F2_E
#define CALES_F2_E 16
#endif
enum { F2_E = CALES_F2_E };     // complex elements per thread per pass (16: radix <= 16; 8: radix <= 8, half the registers)
#ifndef CALES_F2_EY
#define CALES_F2_EY 8
#endif
// the y transforms: 8 (64 registers, twice the warps per SM): B200, config 5, 3.85 / 4.52 ms against 4.3 / 4.6 with 16; the x transforms
// lose with 8 (8.6 / 4.9 against 6.3 / 4.2 ms)
enum { F2_EY = CALES_F2_EY };

struct Fft2Lay { int L, ls, tish; bool ylay; };     // x: line stride ls (padded); y: TI = 1 << tish columns
CALES_HD int f2_off(const Fft2Lay& g, int b, int t) { return g.ylay ? (t << g.tish) + b : b * g.ls + sm_pad(t); }

// floor(n / d) by a precomputed magic = ceil(2^32 / d) (exact for n * d < 2^32; d == 1 has magic 0)
CALES_HD unsigned f2_div(unsigned n, unsigned d, unsigned magic) {
  if (d == 1u) return n;
#ifdef __CUDA_ARCH__
  return __umulhi(n, magic);
#else
  return (unsigned)(((unsigned long long)n * magic) >> 32);
#endif
}

template <int R, int E = F2_E> struct F2G { enum { G = (R == 3) ? E / 3 : (E / R > 0 ? E / R : 1) }; };

// butterfly g of this thread in pass p -> (line b, butterfly index j); false if beyond the work of the pass
CALES_HD bool f2_item(const Fft2Lay& lay, const FftPlan& pl, int p, int tid, int nth, int g, int& b, int& j) {
  const unsigned per = (unsigned)pl.per[p];
  const unsigned idx = (unsigned)(tid + g * nth);
  if (idx >= per * (unsigned)lay.L) return false;
  if (lay.ylay) { b = (int)(idx & ((1u << lay.tish) - 1u)); j = (int)(idx >> lay.tish); }
  else { const unsigned q = f2_div(idx, per, pl.mper[p]); b = (int)q; j = (int)(idx - q * per); }
  return true;
}

// registers <- LD(b, element) for the butterflies of pass p
template <int R, int E, class LD>
CALES_HD void f2_load(const Fft2Lay& lay, const FftPlan& pl, int p, int tid, int nth, LD ld, double2* v) {
  const int per = pl.per[p];
#pragma unroll
  for (int g = 0; g < F2G<R, E>::G; ++g) {
    int b, j;
    if (!f2_item(lay, pl, p, tid, nth, g, b, j)) continue;
#pragma unroll
    for (int t = 0; t < R; ++t) v[g * R + t] = ld(b, j + t * per);
  }
}

// twiddles + radix-R butterflies of pass p on the registers, then ST(b, element, value)
template <int R, int E, class ST>
CALES_HD void f2_bfly_store(const Fft2Lay& lay, const FftPlan& pl, int p, int sign, int tid, int nth, double2* v, ST st) {
  const int Ns = pl.ns[p];
  const int tws = pl.n / (Ns * R);
#pragma unroll
  for (int g = 0; g < F2G<R, E>::G; ++g) {
    int b, j;
    if (!f2_item(lay, pl, p, tid, nth, g, b, j)) continue;
    const int k = j - (int)f2_div((unsigned)j, (unsigned)Ns, pl.mns[p]) * Ns;
    const int j0 = (j - k) * R + k;
    double2* x = v + g * R;
    if (k != 0) {
      double2 w[R];
      w[1] = pl.tw[k * tws];
      if (R > 2) w[2] = pl.tw[2 * k * tws];
      if (R > 3) w[3] = pl.tw[3 * k * tws];
      if (R > 4) { w[4] = cmul(w[2], w[2]); w[5] = cmul(w[4], w[1]); w[6] = cmul(w[4], w[2]); w[7] = cmul(w[4], w[3]); }
      if (R > 8) {
        w[8] = cmul(w[4], w[4]); w[9] = cmul(w[8], w[1]); w[10] = cmul(w[8], w[2]); w[11] = cmul(w[8], w[3]);
        w[12] = cmul(w[8], w[4]); w[13] = cmul(w[12], w[1]); w[14] = cmul(w[12], w[2]); w[15] = cmul(w[12], w[3]);
      }
#pragma unroll
      for (int t = 1; t < R; ++t) x[t] = sign < 0 ? cmul(x[t], w[t]) : cmulc(x[t], w[t]);
    }
    dft_small<R>(x, sign);
#pragma unroll
    for (int t = 0; t < R; ++t) st(b, j0 + t * Ns, x[t]);
  }
}

// dispatch on the radix of pass p
template <int E = F2_E, class LD>
CALES_HD void f2_load_any(const Fft2Lay& lay, const FftPlan& pl, int p, int tid, int nth, LD ld, double2* v) {
  switch (pl.radix[p]) {
    case 2: f2_load<2, E>(lay, pl, p, tid, nth, ld, v); break;
    case 3: f2_load<3, E>(lay, pl, p, tid, nth, ld, v); break;
    case 4: f2_load<4, E>(lay, pl, p, tid, nth, ld, v); break;
    case 8: f2_load<8, E>(lay, pl, p, tid, nth, ld, v); break;
    default: f2_load<16, E>(lay, pl, p, tid, nth, ld, v); break;
  }
}
template <int E = F2_E, class ST>
CALES_HD void f2_bfly_any(const Fft2Lay& lay, const FftPlan& pl, int p, int sign, int tid, int nth, double2* v, ST st) {
  switch (pl.radix[p]) {
    case 2: f2_bfly_store<2, E>(lay, pl, p, sign, tid, nth, v, st); break;
    case 3: f2_bfly_store<3, E>(lay, pl, p, sign, tid, nth, v, st); break;
    case 4: f2_bfly_store<4, E>(lay, pl, p, sign, tid, nth, v, st); break;
    case 8: f2_bfly_store<8, E>(lay, pl, p, sign, tid, nth, v, st); break;
    default: f2_bfly_store<16, E>(lay, pl, p, sign, tid, nth, v, st); break;
  }
}

// packed position q of the (DCT-permuted) input line -> row r with perm_fwd(r) == q
CALES_HD int perm_inv(int q, int n, bool dct) {
  if (!dct) return q;
  return q < n / 2 ? 2 * q : 2 * (n - 1 - q) + 1;
}

// Z[m] of the inverse transforms from the half-complex (or DCT) modes: Z = e + i conj(W^m) d (X_m = E_m + W^m O_m inverted for the packed line z = even + i odd)
CALES_HD double2 f2_merge(const FftPlan& pl, int m, double2 xm, double2 xc /* mode n2 - m, NOT yet conjugated */) {
  xc.y = -xc.y;
  const double2 e = make_double2(0.5 * (xm.x + xc.x), 0.5 * (xm.y + xc.y));
  const double2 d = make_double2(0.5 * (xm.x - xc.x), 0.5 * (xm.y - xc.y));
  const double2 o = cmulc(d, pl.tw[m]);
  return make_double2(e.x - o.y, e.y + o.x);
}

// ---- accessors: shared memory -----------------------------------------------------------------------------------
struct F2SmemLd { const double2* buf; const Fft2Lay& lay; CALES_HD double2 operator()(int b, int t) const { return buf[f2_off(lay, b, t)]; } };
struct F2SmemSt { double2* buf; const Fft2Lay& lay; CALES_HD void operator()(int b, int t, double2 z) const { buf[f2_off(lay, b, t)] = z; } };

// ---- accessors: x transforms (lines contiguous in global memory) ---------------------------------------------------
// forward: packed complex element t of line l0+b, either from src or as the divergence of u* / (gamma dt) (Eq. 12)
struct F2XFwdLd {
  const Ctx& c; const FftPlan& pl; long long l0; int nb; const double* src; const DivSrc& ds; bool div; double inv;   // inv = 1 / (gamma dt)
  CALES_HD double2 operator()(int b, int t) const {
    if (b >= nb) return make_double2(0.0, 0.0);
    const int n = pl.n; const long long l = l0 + b;
    if (!div) return ld2(src + l * n, t);
    const int k = (int)((unsigned)l / (unsigned)c.ny), j = (int)l - k * c.ny;      // ny * nz < 2^31
    const double* ul = ds.us + l * n; const double* vl = ds.vs + l * n; const double* wl = ds.ws + l * n;
    const double* vm = nullptr; const double* wm = nullptr;          // v(j-1), w(k-1): ghosts of u*
    if (j > 0) vm = vl - n; else if (c.bc_y == BC_PER) vm = vl + (long long)(c.ny - 1) * n;
    if (k > 0) wm = wl - c.nxy; else if (c.bc_z == BC_PER) wm = wl + (long long)(c.nz - 1) * c.nxy;
    const double rdx = c.rdx, rdy = c.rdy, rdz = c.rdzf[k];
    const double2 uu = ld2(ul, t);
    const double um = ul[t == 0 ? n - 1 : 2 * t - 1];
    const double2 vv = ld2(vl, t), ww = ld2(wl, t);
    const double2 vvm = vm ? ld2(vm, t) : make_double2(0.0, 0.0), wwm = wm ? ld2(wm, t) : make_double2(0.0, 0.0);
    return make_double2(((uu.x - um) * rdx + (vv.x - vvm.x) * rdy + (ww.x - wwm.x) * rdz) * inv,
                        ((uu.y - uu.x) * rdx + (vv.y - vvm.y) * rdy + (ww.y - wwm.y) * rdz) * inv);
  }
};
// forward from lines staged in shared memory: packed complex element t of line b at buf[b * ls + t]
struct F2XFwdLdS {
  int nb; const double2* buf; int ls;
  CALES_HD double2 operator()(int b, int t) const { return b < nb ? buf[b * ls + t] : make_double2(0.0, 0.0); }
};
// inverse: Z[t] merged on the fly from the packed half-complex line (h[0] = X0, h[1] = X_{n/2}, h[2m], h[2m+1] = X_m)
struct F2XInvLd {
  const FftPlan& pl; long long l0; int nb; const double* src;
  CALES_HD double2 mode(const double* h, int m) const {
    if (m == 0) return make_double2(h[0], 0.0);
    if (m == pl.n2) return make_double2(h[1], 0.0);
    return ld2(h, m);
  }
  CALES_HD double2 operator()(int b, int t) const {
    if (b >= nb) return make_double2(0.0, 0.0);
    const double* h = src + (l0 + b) * pl.n;
    return f2_merge(pl, t, mode(h, t), mode(h, pl.n2 - t));
  }
};
// the same from lines staged in shared memory (raw packed layout, `stride` doubles between lines)
struct F2XInvLdS {
  const FftPlan& pl; int nb; const double* base; int stride;
  CALES_HD double2 mode(const double* h, int m) const {
    if (m == 0) return make_double2(h[0], 0.0);
    if (m == pl.n2) return make_double2(h[1], 0.0);
    return ld2(h, m);
  }
  CALES_HD double2 operator()(int b, int t) const {
    if (b >= nb) return make_double2(0.0, 0.0);
    const double* h = base + b * stride;
    return f2_merge(pl, t, mode(h, t), mode(h, pl.n2 - t));
  }
};
struct F2XInvSt {
  const FftPlan& pl; long long l0; int nb; double* dst; double sc;
  CALES_HD void operator()(int b, int t, double2 z) const {
    if (b < nb) reinterpret_cast<double2*>(dst + (l0 + b) * pl.n)[t] = make_double2(z.x * sc, z.y * sc);
  }
};

// ---- accessors: y transforms (element (row r, column b) at base[r * nx + b]) ---------------------------------------
struct F2YFwdLd {
  const Ctx& c; const FftPlan& pl; const double* base; int nb; bool dct;
  CALES_HD double2 operator()(int b, int t) const {
    if (b >= nb) return make_double2(0.0, 0.0);
    return make_double2(base[(long long)perm_inv(2 * t, pl.n, dct) * c.nx + b], base[(long long)perm_inv(2 * t + 1, pl.n, dct) * c.nx + b]);
  }
};
struct F2YInvLd {
  const Ctx& c; const FftPlan& pl; const double* base; int nb; bool dct;
  CALES_HD double row(int r, int b) const { return base[(long long)r * c.nx + b]; }
  CALES_HD double2 mode(int m, int b) const {      // X[m] (FFT rows) or V[m] (DCT rows), see hc_mode
    if (m == 0) return make_double2(row(0, b), 0.0);
    if (!dct) return m == pl.n2 ? make_double2(row(1, b), 0.0) : make_double2(row(2 * m, b), row(2 * m + 1, b));
    return cmulc(make_double2(row(m, b), -row(pl.n - m, b)), pl.dctw[m]);
  }
  CALES_HD double2 operator()(int b, int t) const {
    if (b >= nb) return make_double2(0.0, 0.0);
    return f2_merge(pl, t, mode(t, b), mode(pl.n2 - t, b));
  }
};
// the same from a tile staged in shared memory (row r, column b at base[r * rs + b])
struct F2YInvLdS {
  const FftPlan& pl; const double* base; int rs; int nb; bool dct;
  CALES_HD double row(int r, int b) const { return base[r * rs + b]; }
  CALES_HD double2 mode(int m, int b) const {
    if (m == 0) return make_double2(row(0, b), 0.0);
    if (!dct) return m == pl.n2 ? make_double2(row(1, b), 0.0) : make_double2(row(2 * m, b), row(2 * m + 1, b));
    return cmulc(make_double2(row(m, b), -row(pl.n - m, b)), pl.dctw[m]);
  }
  CALES_HD double2 operator()(int b, int t) const {
    if (b >= nb) return make_double2(0.0, 0.0);
    return f2_merge(pl, t, mode(t, b), mode(pl.n2 - t, b));
  }
};
struct F2YInvSt {
  const Ctx& c; const FftPlan& pl; double* base; int nb; bool dct; double sc;
  CALES_HD void operator()(int b, int t, double2 z) const {
    if (b >= nb) return;
    base[(long long)perm_inv(2 * t, pl.n, dct) * c.nx + b] = z.x * sc;
    base[(long long)perm_inv(2 * t + 1, pl.n, dct) * c.nx + b] = z.y * sc;
  }
};

// forward split of the finished complex FFT (shared memory) into the packed spectrum in global memory
CALES_HD void f2x_split_store(int tid, int nth, const FftPlan& pl, const Fft2Lay& lay, long long l0, int nb, const double2* Z, double* dst) {
  SmView sv{1, lay.ls, lay.L, false};
  const int n = pl.n;
  split_forward(tid, nth, Z, sv, pl, false, nb, [&](int b, int sa, double va, int sb, double vb) {
    reinterpret_cast<double2*>(dst + (l0 + b) * n)[sa >> 1] = make_double2(va, vb); (void)sb;
  });
}
CALES_HD void f2y_split_store(int tid, int nth, const Ctx& c, const FftPlan& pl, const Fft2Lay& lay, bool dct, double* base, int nb, const double2* Z) {
  SmView sv{1 << lay.tish, 1, 1 << lay.tish, true};
  split_forward(tid, nth, Z, sv, pl, dct, nb, [&](int b, int sa, double va, int sb, double vb) {
    base[(long long)sa * c.nx + b] = va;
    base[(long long)sb * c.nx + b] = vb;
  });
}

#ifdef __CUDACC__
// The pass loop shared by the four kernels.  FIRST reads the pass-0 inputs, LAST (inverse only) consumes the outputs
// of the final pass; forward transforms leave the complex FFT in shared memory for the split.
template <bool TO_GLOBAL, int E = F2_E, class FIRST, class LAST>
__device__ __forceinline__ void f2_passes(const Fft2Lay& lay, const FftPlan& pl, int sign, double2* buf, FIRST first, LAST last) {
  const int tid = threadIdx.x, nth = blockDim.x, np = pl.npass;
  double2 v[E];
  F2SmemLd sld{buf, lay}; F2SmemSt sst{buf, lay};
  if (np == 0) {                 // n = 2: a single complex element per line (lines b = tid, tid + nth, ...; L <= 64 <= 2 * nth)
    double2 z0 = make_double2(0.0, 0.0), z1 = z0;
    if (tid < lay.L) z0 = first(tid, 0);
    if (tid + nth < lay.L) z1 = first(tid + nth, 0);
    __syncthreads();
    if (tid < lay.L) { if (TO_GLOBAL) last(tid, 0, z0); else sst(tid, 0, z0); }
    if (tid + nth < lay.L) { if (TO_GLOBAL) last(tid + nth, 0, z1); else sst(tid + nth, 0, z1); }
    __syncthreads();
    return;
  }
  for (int p = 0; p < np; ++p) {
    if (p == 0) f2_load_any<E>(lay, pl, 0, tid, nth, first, v); else f2_load_any<E>(lay, pl, p, tid, nth, sld, v);
    __syncthreads();             // in-place passes (and in-place global transforms): all reads before any write
    if (TO_GLOBAL && p == np - 1) f2_bfly_any<E>(lay, pl, p, sign, tid, nth, v, last);
    else { f2_bfly_any<E>(lay, pl, p, sign, tid, nth, v, sst); __syncthreads(); }
  }
}

// staged != 0 (DIV only): the divergence of u* / (gamma dt) of the CTA's lines is first formed into the line slots by a pre-pass whose
// loads are batched four elements deep (24 independent loads in flight per thread) instead of one load -> use chain per element inside
// the first butterfly pass; that pass then reads shared memory.
template <bool DIV>
__global__ void __launch_bounds__(512) k_fft2_x_fwd(const __grid_constant__ Ctx c, const __grid_constant__ FftPlan pl, int L, const double* __restrict__ src,
                                                       DivSrc ds, double* __restrict__ dst, int staged) {
  extern __shared__ double2 f2_sm[];
  const Fft2Lay lay{L, sm_line(pl.n2), 0, false};
  const long long nlines = (long long)c.ny * c.nz, l0 = (long long)blockIdx.x * L;
  const int nb = (int)min((long long)L, nlines - l0);
  if (DIV && staged) {
    const int n = pl.n, n2 = pl.n2, nth = blockDim.x;
    const double inv = ds.sc ? ds.sc[2] : ds.inv_gdt, rdx = c.rdx, rdy = c.rdy;
    enum { UB = 4 };
    for (int b = 0; b < nb; ++b) {
      const long long l = l0 + b;
      const int k = (int)((unsigned)l / (unsigned)c.ny), j = (int)l - k * c.ny;
      const double* ul = ds.us + l * n; const double* vl = ds.vs + l * n; const double* wl = ds.ws + l * n;
      const double* vm = nullptr; const double* wm = nullptr;          // v(j-1), w(k-1): ghosts of u*
      if (j > 0) vm = vl - n; else if (c.bc_y == BC_PER) vm = vl + (long long)(c.ny - 1) * n;
      if (k > 0) wm = wl - c.nxy; else if (c.bc_z == BC_PER) wm = wl + (long long)(c.nz - 1) * c.nxy;
      const double rdz = c.rdzf[k];
      double2* out = f2_sm + b * lay.ls;
      for (int t0 = threadIdx.x; t0 < n2; t0 += UB * nth) {
        double2 uu[UB], vv[UB], ww[UB], vvm[UB], wwm[UB]; double um[UB];
#pragma unroll
        for (int q = 0; q < UB; ++q) {
          const int t = t0 + q * nth;
          if (t < n2) {
            uu[q] = ld2(ul, t); um[q] = ul[t == 0 ? n - 1 : 2 * t - 1]; vv[q] = ld2(vl, t); ww[q] = ld2(wl, t);
            vvm[q] = vm ? ld2(vm, t) : make_double2(0.0, 0.0); wwm[q] = wm ? ld2(wm, t) : make_double2(0.0, 0.0);
          }
        }
#pragma unroll
        for (int q = 0; q < UB; ++q) {
          const int t = t0 + q * nth;
          if (t < n2) out[t] = make_double2(((uu[q].x - um[q]) * rdx + (vv[q].x - vvm[q].x) * rdy + (ww[q].x - wwm[q].x) * rdz) * inv,
                                            ((uu[q].y - uu[q].x) * rdx + (vv[q].y - vvm[q].y) * rdy + (ww[q].y - wwm[q].y) * rdz) * inv);
        }
      }
    }
    __syncthreads();
    F2XFwdLdS first{nb, f2_sm, lay.ls};
    f2_passes<false>(lay, pl, -1, f2_sm, first, F2SmemSt{f2_sm, lay});
  } else {
    F2XFwdLd first{c, pl, l0, nb, src, ds, DIV, DIV ? (ds.sc ? ds.sc[2] : ds.inv_gdt) : 0.0};
    f2_passes<false>(lay, pl, -1, f2_sm, first, F2SmemSt{f2_sm, lay});
  }
  f2x_split_store(threadIdx.x, blockDim.x, pl, lay, l0, nb, f2_sm, dst);
}
// staged != 0: the CTA's packed lines are first brought into their shared-memory line slots by one cp.async.bulk copy each (whole
// lines are contiguous; 16-byte aligned because n is even), so the merge of the first pass reads shared memory.  ncu on the direct
// form (profiles/r2_ncu_full.md): 45 % of all stall samples sat on the sixteen load -> merge dependencies of that pass, one global
// latency each; the transforms run at the same rate on L2-resident data, i.e. they were never DRAM-bound.
__global__ void __launch_bounds__(512) k_fft2_x_inv(const __grid_constant__ Ctx c, const __grid_constant__ FftPlan pl, int L, const double* __restrict__ src,
                                                       double* __restrict__ dst, int staged) {
  extern __shared__ double2 f2_sm[];
  __shared__ unsigned long long bar;
  const Fft2Lay lay{L, sm_line(pl.n2), 0, false};
  const long long nlines = (long long)c.ny * c.nz, l0 = (long long)blockIdx.x * L;
  const int nb = (int)min((long long)L, nlines - l0);
  F2XInvSt last{pl, l0, nb, dst, 1.0 / (double)pl.n2};
  if (staged) {
    if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
    __syncthreads();
    if (threadIdx.x == 0) {
      mbar_expect_tx(&bar, (unsigned)nb * (unsigned)pl.n * 8u);
      for (int b = 0; b < nb; ++b) bulk_g2s(f2_sm + b * lay.ls, src + (l0 + b) * pl.n, (unsigned)pl.n * 8u, &bar);
    }
    mbar_wait(&bar, 0);
    F2XInvLdS first{pl, nb, reinterpret_cast<const double*>(f2_sm), 2 * lay.ls};
    f2_passes<true>(lay, pl, +1, f2_sm, first, last);
  } else {
    F2XInvLd first{pl, l0, nb, src};
    f2_passes<true>(lay, pl, +1, f2_sm, first, last);
  }
}
// grid (ceil(nx/TI), nz); in place on A
// staged != 0 (inverse only): the raw [ny x TI] tile is first copied into the (equally large) shared buffer -- bit 1: by 16-byte
// asynchronous copies (cp.async.cg: the whole tile in flight at once, no registers; 5.34 -> 4.57 ms at config 5), bit 0: by batched,
// dependency-free loads through registers -- and the merge of the first pass reads shared memory, same reason as in k_fft2_x_inv.
// The forward transform gains nothing from either (4.25 vs 4.23 ms): its first pass already issues 32 independent loads per thread.
__global__ void __launch_bounds__(512) k_fft2_y(const __grid_constant__ Ctx c, const __grid_constant__ FftPlan pl, int tish, int dct, int inverse, double* __restrict__ A,
                                                   int staged) {
  extern __shared__ double2 f2_sm[];
  const int TI = 1 << tish;
  const Fft2Lay lay{TI, 0, tish, true};
  const int i0 = blockIdx.x * TI, k = blockIdx.y;
  const int nb = min(TI, c.nx - i0);
  double* base = A + (long long)k * c.nxy + i0;
  if (!inverse) {
    F2YFwdLd first{c, pl, base, nb, dct != 0};
    f2_passes<false, F2_EY>(lay, pl, -1, f2_sm, first, F2SmemSt{f2_sm, lay});
    f2y_split_store(threadIdx.x, blockDim.x, c, pl, lay, dct != 0, base, nb, f2_sm);
  } else if ((staged & 3) && nb == TI && TI >= 2) {
    F2YInvSt last{c, pl, base, nb, dct != 0, 1.0 / (double)pl.n2};
    const int hsh = tish - 1, total = pl.n << hsh;            // double2 elements of the tile: ny rows of TI/2
    enum { UB = 8 };
    if (staged & 2) {      // the whole tile in flight at once, no registers: 16-byte asynchronous copies
      for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
        const int r = idx >> hsh, cq = idx & ((1 << hsh) - 1);
        cp_async16(f2_sm + idx, base + (long long)r * c.nx + 2 * cq);
      }
      cp_async_commit();
      cp_async_wait_all();
    } else
    for (int i0b = threadIdx.x; i0b < total; i0b += UB * blockDim.x) {
      double2 tmp[UB];
#pragma unroll
      for (int q = 0; q < UB; ++q) {
        const int idx = i0b + q * blockDim.x;
        if (idx < total) { const int r = idx >> hsh, cq = idx & ((1 << hsh) - 1); tmp[q] = *reinterpret_cast<const double2*>(base + (long long)r * c.nx + 2 * cq); }
      }
#pragma unroll
      for (int q = 0; q < UB; ++q) { const int idx = i0b + q * blockDim.x; if (idx < total) f2_sm[idx] = tmp[q]; }
    }
    __syncthreads();
    F2YInvLdS first{pl, reinterpret_cast<const double*>(f2_sm), TI, nb, dct != 0};
    f2_passes<true, F2_EY>(lay, pl, +1, f2_sm, first, last);
  } else {
    F2YInvLd first{c, pl, base, nb, dct != 0};
    F2YInvSt last{c, pl, base, nb, dct != 0, 1.0 / (double)pl.n2};
    f2_passes<true, F2_EY>(lay, pl, +1, f2_sm, first, last);
  }
}
#endif

}  // namespace cales
