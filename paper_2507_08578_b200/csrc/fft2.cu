// fft2.cu -- K2, register-resident path: every 1-D transform of the five pruned passes (fft.cu header,
// SURVEY.md 8(a) S3-S7; PAPER.md :475 "local part using fast Fourier transforms", :436 batched over bands)
// is ONE two-stage decomposition n = R1 * R2 done in registers with a single shared-memory exchange:
//
//   type I  (G -> r, w = exp(+2 pi i/n)):  j = j2 + R2 j1,  k = k1 + R1 k2
//       thread j2:  Y[k1] = sum_j1 x[j2 + R2 j1] w_R1^(j1 k1);   Z[k1] = Y[k1] w_n^(j2 k1)      (radix R1, R2 threads)
//       exchange;   thread k1:  X[k1 + R1 k2] = sum_j2 Z_j2[k1] w_R2^(j2 k2)                    (radix R2, R1 threads)
//   type II (r -> G, w = exp(-2 pi i/n)):  j = a + R1 b,    k = c + R2 d
//       thread a:   Y[c] = sum_b x[a + R1 b] w_R2^(b c);         Z[c] = Y[c] w_n^(a c)          (radix R2, R1 threads)
//       exchange;   thread c:   X[c + R2 d] = sum_a Z_a[c] w_R1^(a d)                           (radix R1, R2 threads)
//
// Type II consumes exactly the register layout type I produces (thread k1 holds k1 + R1 k2) and returns
// the layout type I reads (thread j2 holds j2 + R2 j1), so pass C (forward along z, times V(r)/N,
// inverse along z) touches shared memory twice per line instead of twelve times, and every global
// access goes straight from/to registers: along y and z a warp's lanes are consecutive x (contiguous runs
// of XT complex numbers); along x the lanes are the consecutive slots j2 / k1 / a / c of one line.
// Pruning: the occupied x of a column, y of a plane and z of the box are (at most) two runs of
// consecutive box indices each (the sphere is convex), so "is this input non-zero / is this output
// kept" is two range checks (struct Run) and the sphere <-> box maps need no index list.
#include "fft_codelets.cuh"
#include "internal.h"
#include "ptx.cuh"

namespace dftb200 {

__device__ __forceinline__ int run_map(const Run &r, int x) {
  unsigned d = (unsigned)(x - r.lo);
  if (d < (unsigned)r.nlo) return r.base + (int)d;
  d = (unsigned)(x - r.hi);
  if (d < (unsigned)r.nhi) return r.base + r.nlo + (int)d;
  return -1;
}
__device__ __forceinline__ Run load_run(const Run *p) {
  const int4 *q = reinterpret_cast<const int4 *>(p);
  int4 a = __ldg(q), b = __ldg(q + 1);
  Run r; r.base = a.x; r.lo = a.y; r.nlo = a.z; r.hi = a.w; r.nhi = b.x; r.aux0 = b.y; r.aux1 = b.z; r.pad = b.w;
  return r;
}
__device__ __forceinline__ cplx ldtw(const cplx *tw, int i) {
  return __ldg(tw + i);
}
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {   // a * conj(b)
  return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
constexpr int F2_THREADS = 256;
#ifndef F2C_THREADS_N
#define F2C_THREADS_N 256
#endif
constexpr int F2C_THREADS = F2C_THREADS_N;   // pass C ring kernel: threads per CTA (tile = F2C_THREADS / max radix lines, a multiple of 8)
constexpr int F2C_PER_SM = F2C_THREADS_N <= 128 ? 4 : 2;
__host__ __device__ constexpr int imax(int a, int b) { return a > b ? a : b; }
__host__ __device__ constexpr int pad8(int len, int want) { return len + (((want - len) % 8) + 8) % 8; }   // smallest >= len congruent to want mod 8

struct Fft2Geom {
  int n1, n2, n3, npw, mpw, ncol, nplane;
  const Run *col_run, *plane_run;
  Run zrun;
  const cplx *tw1, *tw2, *tw3;
  int64_t t1_band, t2_band;   // complex elements per band of T1 [ncol][n1] and T2 [nplane][n2][n1]
};

// Several k-points in one launch (BATCH): blockIdx.y = k-point, geometry read from a device array, per-k strides of
// the caller's arrays and of the scratch; grid.x is sized for the k-point with the most columns / planes.
struct Fft2Batch {
  const Fft2Geom *Gs;
  int64_t ks_psi, ks_t1, ks_t2;   // complex elements between consecutive k-points
};

// ---- pass A: sphere -> x-lines (type I).  block = lpc lines x NS slots, slot fastest; grid = nb * ntile.
//      Three CTAs per SM (80 registers): the gather from psi is latency-bound, a third CTA buys 42 -> 53 % of HBM peak.
template <int R1, int R2, bool BATCH, bool EXTRA>
__global__ void __launch_bounds__(F2_THREADS, 3)
fft2_a_fwd_kernel(Fft2Geom G0, Fft2Batch B, const cplx *__restrict__ psi, cplx *__restrict__ T1, int lpc, int ntile,
                  const double *__restrict__ pre) {
  const Fft2Geom G = BATCH ? B.Gs[blockIdx.y] : G0;
  if (BATCH) { psi += (size_t)blockIdx.y * B.ks_psi; T1 += (size_t)blockIdx.y * B.ks_t1; }
  constexpr int NS = imax(R1, R2), KS = R2 | 1, LS = pad8(R1 * KS, NS);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx *sm = reinterpret_cast<cplx *>(smem_raw);
  const int t = threadIdx.x, s = t % NS, l = t / NS;
  const int tile = blockIdx.x % ntile, b = blockIdx.x / ntile;
  const int c = tile * lpc + l;
  const bool ok = c < G.ncol;
  Run r = load_run(G.col_run + (ok ? c : 0));
  cplx v[NS];
  if (s < R2) {
    const cplx *src = psi + (size_t)b * G.mpw;
#pragma unroll
    for (int j1 = 0; j1 < R1; j1++) {
      int g = ok ? run_map(r, s + R2 * j1) : -1;
      v[j1] = g >= 0 ? src[g] : make_double2(0.0, 0.0);
      if (EXTRA && pre && g >= 0) v[j1] = cscale(v[j1], __ldg(pre + g));     // diagonal factor in G space before the transform
    }
    Dft<R1, +1>::run(v);
#pragma unroll
    for (int k1 = 1; k1 < R1; k1++) v[k1] = cmul(v[k1], ldtw(G.tw1, s * k1));
#pragma unroll
    for (int k1 = 0; k1 < R1; k1++) sm[l * LS + k1 * KS + s] = v[k1];
  }
  __syncthreads();
  if (s < R1) {
#pragma unroll
    for (int j2 = 0; j2 < R2; j2++) v[j2] = sm[l * LS + s * KS + j2];
    Dft<R2, +1>::run(v);
    if (ok) {
      cplx *dst = T1 + (size_t)b * G.t1_band + (size_t)c * G.n1 + s;
#pragma unroll
      for (int k2 = 0; k2 < R2; k2++) dst[R1 * k2] = v[k2];
    }
  }
}

// ---- pass A^-1: x-lines -> sphere (type II) + zero the pad entries ipw >= npw of the band
template <int R1, int R2, bool BATCH, bool EXTRA>
__global__ void __launch_bounds__(F2_THREADS, 2)
fft2_a_inv_kernel(Fft2Geom G0, Fft2Batch B, const cplx *__restrict__ T1, cplx *__restrict__ hpsi, int lpc, int ntile,
                  const double *__restrict__ post, int accumulate) {
  const Fft2Geom G = BATCH ? B.Gs[blockIdx.y] : G0;
  if (BATCH) { hpsi += (size_t)blockIdx.y * B.ks_psi; T1 += (size_t)blockIdx.y * B.ks_t1; }
  constexpr int NS = imax(R1, R2), KS = R1 | 1, LS = pad8(R2 * KS, NS);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx *sm = reinterpret_cast<cplx *>(smem_raw);
  const int t = threadIdx.x, s = t % NS, l = t / NS;
  const int tile = blockIdx.x % ntile, b = blockIdx.x / ntile;
  const int c = tile * lpc + l;
  const bool ok = c < G.ncol;
  Run r = load_run(G.col_run + (ok ? c : 0));
  cplx v[NS];
  if (s < R1) {
    const cplx *src = T1 + (size_t)b * G.t1_band + (size_t)(ok ? c : 0) * G.n1 + s;
#pragma unroll
    for (int b2 = 0; b2 < R2; b2++) v[b2] = ok ? src[R1 * b2] : make_double2(0.0, 0.0);
    Dft<R2, -1>::run(v);
#pragma unroll
    for (int cc = 1; cc < R2; cc++) v[cc] = cmulc(v[cc], ldtw(G.tw1, s * cc));
#pragma unroll
    for (int cc = 0; cc < R2; cc++) sm[l * LS + cc * KS + s] = v[cc];
  }
  __syncthreads();
  cplx *dst = hpsi + (size_t)b * G.mpw;
  if (s < R2) {
#pragma unroll
    for (int a = 0; a < R1; a++) v[a] = sm[l * LS + s * KS + a];
    Dft<R1, -1>::run(v);
#pragma unroll
    for (int d = 0; d < R1; d++) {
      int g = ok ? run_map(r, s + R2 * d) : -1;
      if (g >= 0) {
        cplx o = v[d];
        if (EXTRA) {
          if (post) o = cscale(o, __ldg(post + g));                  // diagonal factor in G space after the transform
          if (accumulate) { cplx h = dst[g]; o.x += h.x; o.y += h.y; }
        }
        dst[g] = o;
      }
    }
  }
  if (tile == ntile - 1 && !(EXTRA && accumulate))
    for (int g = G.npw + t; g < G.mpw; g += blockDim.x) dst[g] = make_double2(0.0, 0.0);
}

// ---- pass B: along y on the occupied planes (type I).  block = NS slots x XT consecutive x, x fastest;
//      grid = nb * nplane * nxt.  Shared exchange element (k1, j2, px) at k1*KS + j2*XT + px.
template <int R1, int R2, bool BATCH>
__global__ void __launch_bounds__(F2_THREADS, 2)
fft2_b_fwd_kernel(Fft2Geom G0, Fft2Batch B, const cplx *__restrict__ T1, cplx *__restrict__ T2, int XT, int nxt, int nb) {
  const Fft2Geom G = BATCH ? B.Gs[blockIdx.y] : G0;
  if (BATCH) { T1 += (size_t)blockIdx.y * B.ks_t1; T2 += (size_t)blockIdx.y * B.ks_t2; }
  if (BATCH && (int)(blockIdx.x / (nxt * G.nplane)) >= nb) return;   // grid sized for the k-point with most planes
  constexpr int NS = imax(R1, R2);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx *sm = reinterpret_cast<cplx *>(smem_raw);
  const int t = threadIdx.x, px = t % XT, s = t / XT;
  const int xt = blockIdx.x % nxt, p = (blockIdx.x / nxt) % G.nplane, b = blockIdx.x / (nxt * G.nplane);
  const int x = xt * XT + px;
  const bool xok = x < G.n1;
  const int KS = pad8(R2 * XT, XT);
  Run r = load_run(G.plane_run + p);
  cplx v[NS];
  if (s < R2) {
    const cplx *src = T1 + (size_t)b * G.t1_band + x;
#pragma unroll
    for (int j1 = 0; j1 < R1; j1++) {
      int c = xok ? run_map(r, s + R2 * j1) : -1;
      v[j1] = c >= 0 ? src[(size_t)c * G.n1] : make_double2(0.0, 0.0);
    }
    Dft<R1, +1>::run(v);
#pragma unroll
    for (int k1 = 1; k1 < R1; k1++) v[k1] = cmul(v[k1], ldtw(G.tw2, s * k1));
#pragma unroll
    for (int k1 = 0; k1 < R1; k1++) sm[k1 * KS + s * XT + px] = v[k1];
  }
  __syncthreads();
  if (s < R1) {
#pragma unroll
    for (int j2 = 0; j2 < R2; j2++) v[j2] = sm[s * KS + j2 * XT + px];
    Dft<R2, +1>::run(v);
    if (xok) {
      cplx *dst = T2 + (size_t)b * G.t2_band + ((size_t)p * G.n2 + s) * G.n1 + x;
#pragma unroll
      for (int k2 = 0; k2 < R2; k2++) dst[(size_t)(R1 * k2) * G.n1] = v[k2];
    }
  }
}

// ---- pass B^-1: inverse along y, keep the non-empty columns (type II)
template <int R1, int R2, bool BATCH>
__global__ void __launch_bounds__(F2_THREADS, 2)
fft2_b_inv_kernel(Fft2Geom G0, Fft2Batch B, cplx *__restrict__ T1, const cplx *__restrict__ T2, int XT, int nxt, int nb) {
  const Fft2Geom G = BATCH ? B.Gs[blockIdx.y] : G0;
  if (BATCH) { T1 += (size_t)blockIdx.y * B.ks_t1; T2 += (size_t)blockIdx.y * B.ks_t2; }
  if (BATCH && (int)(blockIdx.x / (nxt * G.nplane)) >= nb) return;
  constexpr int NS = imax(R1, R2);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx *sm = reinterpret_cast<cplx *>(smem_raw);
  const int t = threadIdx.x, px = t % XT, s = t / XT;
  const int xt = blockIdx.x % nxt, p = (blockIdx.x / nxt) % G.nplane, b = blockIdx.x / (nxt * G.nplane);
  const int x = xt * XT + px;
  const bool xok = x < G.n1;
  const int KS = pad8(R1 * XT, XT);
  Run r = load_run(G.plane_run + p);
  cplx v[NS];
  if (s < R1) {
    const cplx *src = T2 + (size_t)b * G.t2_band + ((size_t)p * G.n2 + s) * G.n1 + (xok ? x : 0);
#pragma unroll
    for (int b2 = 0; b2 < R2; b2++) v[b2] = xok ? src[(size_t)(R1 * b2) * G.n1] : make_double2(0.0, 0.0);
    Dft<R2, -1>::run(v);
#pragma unroll
    for (int cc = 1; cc < R2; cc++) v[cc] = cmulc(v[cc], ldtw(G.tw2, s * cc));
#pragma unroll
    for (int cc = 0; cc < R2; cc++) sm[cc * KS + s * XT + px] = v[cc];
  }
  __syncthreads();
  if (s < R2) {
#pragma unroll
    for (int a = 0; a < R1; a++) v[a] = sm[s * KS + a * XT + px];
    Dft<R1, -1>::run(v);
    cplx *dst = T1 + (size_t)b * G.t1_band + x;
#pragma unroll
    for (int d = 0; d < R1; d++) {
      int c = xok ? run_map(r, s + R2 * d) : -1;
      if (c >= 0) dst[(size_t)c * G.n1] = v[d];
    }
  }
}

// ---- pass C: along z (type I), times V(r)/N, inverse along z (type II), in place on the occupied planes.
//      grid = ntile * nb with the BAND fastest, so the nb CTAs that need the same V tile run together
//      and V is fetched from DRAM once per band chunk.
template <int R1, int R2, bool BATCH>
__global__ void __launch_bounds__(F2_THREADS, 2)
fft2_c_kernel(Fft2Geom G0, Fft2Batch B, cplx *__restrict__ T2, const double *__restrict__ vloc, int XT, int nxt, int nb) {
  const Fft2Geom G = BATCH ? B.Gs[blockIdx.y] : G0;
  if (BATCH) T2 += (size_t)blockIdx.y * B.ks_t2;
  constexpr int NS = imax(R1, R2);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx *sm = reinterpret_cast<cplx *>(smem_raw);
  const int t = threadIdx.x, px = t % XT, s = t / XT;
  const int b = blockIdx.x % nb, tile = blockIdx.x / nb, xt = tile % nxt, y = tile / nxt;
  const int x = xt * XT + px;
  const bool xok = x < G.n1;
  const int KSa = pad8(R2 * XT, XT), KSb = pad8(R1 * XT, XT);
  const size_t pstride = (size_t)G.n2 * G.n1;
  cplx *base = T2 + (size_t)b * G.t2_band + (size_t)y * G.n1 + (xok ? x : 0);
  cplx v[NS];
  if (s < R2) {
#pragma unroll
    for (int j1 = 0; j1 < R1; j1++) {
      int p = xok ? run_map(G.zrun, s + R2 * j1) : -1;
      v[j1] = p >= 0 ? base[(size_t)p * pstride] : make_double2(0.0, 0.0);
    }
    Dft<R1, +1>::run(v);
#pragma unroll
    for (int k1 = 1; k1 < R1; k1++) v[k1] = cmul(v[k1], ldtw(G.tw3, s * k1));
#pragma unroll
    for (int k1 = 0; k1 < R1; k1++) sm[k1 * KSa + s * XT + px] = v[k1];
  }
  __syncthreads();
  if (s < R1) {
#pragma unroll
    for (int j2 = 0; j2 < R2; j2++) v[j2] = sm[s * KSa + j2 * XT + px];
  }
  __syncthreads();   // every read of the forward exchange is done before the buffer is reused
  if (s < R1) {
    Dft<R2, +1>::run(v);
    // thread s now holds psi(r) at z = s + R1 k2
    const double *vp = vloc + (size_t)s * pstride + (size_t)y * G.n1 + (xok ? x : 0);
#pragma unroll
    for (int k2 = 0; k2 < R2; k2++) {
      double w = xok ? __ldg(vp + (size_t)(R1 * k2) * pstride) : 0.0;
      v[k2] = cscale(v[k2], w);
    }
    Dft<R2, -1>::run(v);
#pragma unroll
    for (int cc = 1; cc < R2; cc++) v[cc] = cmulc(v[cc], ldtw(G.tw3, s * cc));
#pragma unroll
    for (int cc = 0; cc < R2; cc++) sm[cc * KSb + s * XT + px] = v[cc];
  }
  __syncthreads();
  if (s < R2) {
#pragma unroll
    for (int a = 0; a < R1; a++) v[a] = sm[s * KSb + a * XT + px];
    Dft<R1, -1>::run(v);
#pragma unroll
    for (int d = 0; d < R1; d++) {
      int p = xok ? run_map(G.zrun, s + R2 * d) : -1;
      if (p >= 0) base[(size_t)p * pstride] = v[d];
    }
  }
}

// ---- pass C for two-component spinors (PAPER.md :448; reading 27): the rows of T2 come in pairs (2 j, 2 j + 1) =
//      (up, down) component of spinor band j, and the potential is the Hermitian 2 x 2 matrix V^{ss'}(r), given as the four
//      real fields v4 = (V_upup, V_dndn, Re V_updn, Im V_updn) / N:
//          out_up = V_upup psi_up + V_updn psi_dn,     out_dn = conj(V_updn) psi_up + V_dndn psi_dn     at every point r.
//      A tile is 8 consecutive x of BOTH components: lanes px = 0..7 hold the up component, px = 8..15 the down component of
//      the same points, so after the forward transform the partner value sits in lane ^ 8 of the same warp and one
//      shuffle per number replaces any second pass over the data: one local application for the whole 2 x 2 matrix
//      instead of the four of the Pauli decomposition (spinor.cu).  Same exchanges and twiddles as fft2_c_kernel.
//      The CTAs are persistent: each walks a contiguous range of (tile, spinor band) pairs with the band fastest and keeps
//      the four fields of its tile, [4][n3][8] doubles, and the twiddles in shared memory (with the fields read straight
//      from L2 in the multiply loop, 45 dependent-latency loads per thread, the pass took 109 ms per 1024 rows at c4).
template <int R1, int R2>
__global__ void __launch_bounds__(F2_THREADS, 2)
fft2_c_spinor_kernel(Fft2Geom G, cplx *__restrict__ T2, const double *__restrict__ v4, int nxt, int nsb, int ntiles) {
  constexpr int NS = imax(R1, R2), XT = 16;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int KSa = pad8(R2 * XT, XT), KSb = pad8(R1 * XT, XT), exn = imax(R1 * KSa, R2 * KSb);
  cplx *sm = reinterpret_cast<cplx *>(smem_raw);
  cplx *tws = sm + exn;                                       // exp(+2 pi i j / n3), j < n3
  double *vs = reinterpret_cast<double *>(tws + G.n3);        // [4][n3][8]
  const int t = threadIdx.x, px = t % XT, s = t / XT, comp = px >> 3, xq = px & 7;
  for (int i = t; i < G.n3; i += blockDim.x) tws[i] = __ldg(G.tw3 + i);
  const int first = (int)(((int64_t)ntiles * blockIdx.x) / gridDim.x);
  const int nmine = (int)(((int64_t)ntiles * (blockIdx.x + 1)) / gridDim.x) - first;
  const size_t pstride = (size_t)G.n2 * G.n1, nbox = (size_t)G.n3 * pstride;
  int sb = first % nsb, g = first / nsb;
  bool newgroup = true;
  const unsigned half = 0xffffu << (t & 16);      // the 16 lanes that share this thread's s
  const double sgn = comp ? -1.0 : 1.0;           // the down row of the matrix holds conj(V_updn)
  const double *vown = vs + (size_t)comp * G.n3 * 8 + xq, *vre = vs + (size_t)2 * G.n3 * 8 + xq, *vim = vs + (size_t)3 * G.n3 * 8 + xq;
  for (int it = 0; it < nmine; it++) {
    const int xt = g % nxt, y = g / nxt, x = xt * 8 + xq;
    const bool xok = x < G.n1;
    if (newgroup) {
      __syncthreads();       // every read of the previous tile's fields (and the twiddle fill, the first time) is done
      const double *vp = v4 + (size_t)y * G.n1 + xt * 8;
      for (int i = t; i < 4 * G.n3 * 8; i += blockDim.x) {
        const int f = i / (G.n3 * 8), r = i - f * (G.n3 * 8), z = r >> 3, xx = r & 7;
        vs[i] = (xt * 8 + xx < G.n1) ? __ldg(vp + (size_t)f * nbox + (size_t)z * pstride + xx) : 0.0;
      }
      newgroup = false;      // the barrier after the first exchange orders these writes before the reads of stage 2
    }
    cplx *base = T2 + (size_t)(2 * sb + comp) * G.t2_band + (size_t)y * G.n1 + (xok ? x : 0);
    cplx v[NS];
    if (s < R2) {
#pragma unroll
      for (int j1 = 0; j1 < R1; j1++) {
        int p = xok ? run_map(G.zrun, s + R2 * j1) : -1;
        v[j1] = p >= 0 ? base[(size_t)p * pstride] : make_double2(0.0, 0.0);
      }
      Dft<R1, +1>::run(v);
#pragma unroll
      for (int k1 = 1; k1 < R1; k1++) v[k1] = cmul(v[k1], tws[s * k1]);
#pragma unroll
      for (int k1 = 0; k1 < R1; k1++) sm[k1 * KSa + s * XT + px] = v[k1];
    }
    __syncthreads();
    if (s < R1) {
      // in-place second exchange as in fft2_c_ring_kernel: this thread overwrites exactly the slots it read
#pragma unroll
      for (int j2 = 0; j2 < R2; j2++) v[j2] = sm[s * KSa + j2 * XT + px];
      Dft<R2, +1>::run(v);
      // thread s now holds psi_comp(r) at z = s + R1 k2; its partner lane (^ 8) holds the other component at the same points.
      // The 16 lanes of a half-warp share s, so the branch is uniform per half-warp and the shuffle names that half only.
#pragma unroll
      for (int k2 = 0; k2 < R2; k2++) {
        const int o = (s + R1 * k2) * 8;
        const double a = vown[o], cr = vre[o], ci = sgn * vim[o];
        const double ox = __shfl_xor_sync(half, v[k2].x, 8), oy = __shfl_xor_sync(half, v[k2].y, 8);
        v[k2] = make_double2(a * v[k2].x + (cr * ox - ci * oy), a * v[k2].y + (cr * oy + ci * ox));
      }
      Dft<R2, -1>::run(v);
#pragma unroll
      for (int cc = 1; cc < R2; cc++) v[cc] = cmulc(v[cc], tws[s * cc]);
#pragma unroll
      for (int cc = 0; cc < R2; cc++) sm[s * KSa + cc * XT + px] = v[cc];
    }
    __syncthreads();
    if (s < R2) {
#pragma unroll
      for (int a = 0; a < R1; a++) v[a] = sm[a * KSa + s * XT + px];
      Dft<R1, -1>::run(v);
#pragma unroll
      for (int d = 0; d < R1; d++) {
        int p = xok ? run_map(G.zrun, s + R2 * d) : -1;
        if (p >= 0) base[(size_t)p * pstride] = v[d];
      }
    }
    if (++sb == nsb) { sb = 0; newgroup = true; g++; }
  }
}

// ------------------------------------------------------------------------------------------
// TMA-ring variants of the three strided passes (B, C, B^-1).  Same arithmetic, same register
// layout; what changes is how a tile's INPUT reaches the registers.  Above, every thread issues its own
// R loads and then waits for them, so with 2 CTAs of ~6 warps per SM the kernel is exposed to DRAM
// latency for a large part of each tile (ncu r1: 17 % warps active, long-scoreboard stalls, 25-50 % of
// HBM peak).  Here a CTA is persistent, walks a list of tiles, and lane 0 keeps S-1 tiles in flight with
// cp.async.bulk.tensor (one box = all occupied rows of the tile x XT consecutive x) into a
// shared-memory ring guarded by mbarriers; the threads read their strided inputs from the ring
// (consecutive lanes -> consecutive 16-byte words, conflict-free) and DRAM latency is off the critical
// path.  Outputs still go from registers straight to global memory (stores do not stall).
// ------------------------------------------------------------------------------------------
struct RingParams {
  int XT, nxt, ntiles, S, nb;
  uint32_t stage_stride, box_bytes;   // bytes; stage_stride is box_bytes rounded up to 128
};
__device__ __forceinline__ int run_local(const Run &r, int x) {   // row inside the tile's box (box row 0 = r.base)
  unsigned d = (unsigned)(x - r.lo);
  if (d < (unsigned)r.nlo) return (int)d;
  d = (unsigned)(x - r.hi);
  if (d < (unsigned)r.nhi) return r.nlo + (int)d;
  return -1;
}

// ---- pass B (type I along y): box {XT x, HB columns starting at the plane's first column} of T1
template <int R1, int R2>
__global__ void __launch_bounds__(F2_THREADS, 2)
fft2_b_fwd_ring_kernel(const __grid_constant__ CUtensorMap mapT1, Fft2Geom G, cplx *__restrict__ T2, RingParams Q) {
  constexpr int NS = imax(R1, R2);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int XT = Q.XT, KS = pad8(R2 * XT, XT);
  unsigned char *stages = smem_raw;
  cplx *sm = reinterpret_cast<cplx *>(stages + (size_t)Q.S * Q.stage_stride);
  Run *runs = reinterpret_cast<Run *>(sm + R1 * KS);
  uint64_t *full = reinterpret_cast<uint64_t *>(runs + G.nplane);
  const int t = threadIdx.x, px = t % XT, s = t / XT;
  for (int i = t; i < G.nplane * 2; i += blockDim.x)
    reinterpret_cast<int4 *>(runs)[i] = __ldg(reinterpret_cast<const int4 *>(G.plane_run) + i);
  if (t == 0) {
    for (int i = 0; i < Q.S; i++) mbar_init(&full[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // contiguous range of tiles (x-tile fastest, then plane, then band), decoded incrementally
  const int first = (int)(((int64_t)Q.ntiles * blockIdx.x) / gridDim.x);
  const int nmine = (int)(((int64_t)Q.ntiles * (blockIdx.x + 1)) / gridDim.x) - first;
  int xt = first % Q.nxt, p = (first / Q.nxt) % G.nplane, b = first / (Q.nxt * G.nplane);
  int ixt = xt, ip = p, ib = b, ist = 0;      // producer's copy (lane 0 only), runs S-1 tiles ahead
  auto issue = [&]() {
    mbar_expect_tx(&full[ist], Q.box_bytes);
    tma_load_3d(stages + (size_t)ist * Q.stage_stride, &mapT1, &full[ist], 2 * ixt * XT, runs[ip].base, ib);
    if (++ist == Q.S) ist = 0;
    if (++ixt == Q.nxt) { ixt = 0; if (++ip == G.nplane) { ip = 0; ib++; } }
  };
  if (t == 0)
    for (int j = 0; j < Q.S - 1 && j < nmine; j++) issue();
  int st = 0; uint32_t ph = 0;
  for (int it = 0; it < nmine; it++) {
    if (t == 0 && it + Q.S - 1 < nmine) issue();
    const int x = xt * XT + px;
    const bool xok = x < G.n1;
    const Run r = runs[p];
    const cplx *in = reinterpret_cast<const cplx *>(stages + (size_t)st * Q.stage_stride) + px;
    mbar_wait(&full[st], ph);
    cplx v[NS];
    if (s < R2) {
#pragma unroll
      for (int j1 = 0; j1 < R1; j1++) {
        int c = run_local(r, s + R2 * j1);
        v[j1] = c >= 0 ? in[c * XT] : make_double2(0.0, 0.0);
      }
      Dft<R1, +1>::run(v);
#pragma unroll
      for (int k1 = 1; k1 < R1; k1++) v[k1] = cmul(v[k1], ldtw(G.tw2, s * k1));   // (shared-memory twiddles: slower here, 13.5 -> 13.9 ms at c4)
#pragma unroll
      for (int k1 = 0; k1 < R1; k1++) sm[k1 * KS + s * XT + px] = v[k1];
    }
    __syncthreads();
    if (s < R1) {
#pragma unroll
      for (int j2 = 0; j2 < R2; j2++) v[j2] = sm[s * KS + j2 * XT + px];
      Dft<R2, +1>::run(v);
      if (xok) {
        cplx *dst = T2 + (size_t)b * G.t2_band + ((size_t)p * G.n2 + s) * G.n1 + x;
#pragma unroll
        for (int k2 = 0; k2 < R2; k2++) dst[(size_t)(R1 * k2) * G.n1] = v[k2];
      }
    }
    __syncthreads();   // the exchange buffer is rewritten by the next tile
    if (++st == Q.S) { st = 0; ph ^= 1; }
    if (++xt == Q.nxt) { xt = 0; if (++p == G.nplane) { p = 0; b++; } }
  }
}

// ---- pass B^-1 (type II along y): box {XT x, n2 y} of one plane of T2
template <int R1, int R2>
__global__ void __launch_bounds__(F2_THREADS, 2)
fft2_b_inv_ring_kernel(const __grid_constant__ CUtensorMap mapT2, Fft2Geom G, cplx *__restrict__ T1, RingParams Q) {
  constexpr int NS = imax(R1, R2);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int XT = Q.XT, KS = pad8(R1 * XT, XT);
  unsigned char *stages = smem_raw;
  cplx *sm = reinterpret_cast<cplx *>(stages + (size_t)Q.S * Q.stage_stride);
  Run *runs = reinterpret_cast<Run *>(sm + R2 * KS);
  cplx *tws = reinterpret_cast<cplx *>(runs + G.nplane);      // twiddles exp(+2 pi i j / n2) in shared memory: loading them from
  uint64_t *full = reinterpret_cast<uint64_t *>(tws + G.n2);  // L2 in every tile sat on the critical path (12.25 -> 10.6 ms at c4)
  const int t = threadIdx.x, px = t % XT, s = t / XT;
  for (int i = t; i < G.nplane * 2; i += blockDim.x)
    reinterpret_cast<int4 *>(runs)[i] = __ldg(reinterpret_cast<const int4 *>(G.plane_run) + i);
  for (int i = t; i < G.n2; i += blockDim.x) tws[i] = __ldg(G.tw2 + i);
  if (t == 0) {
    for (int i = 0; i < Q.S; i++) mbar_init(&full[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // contiguous range of tiles (x-tile fastest, then plane, then band), decoded incrementally
  const int first = (int)(((int64_t)Q.ntiles * blockIdx.x) / gridDim.x);
  const int nmine = (int)(((int64_t)Q.ntiles * (blockIdx.x + 1)) / gridDim.x) - first;
  int xt = first % Q.nxt, p = (first / Q.nxt) % G.nplane, b = first / (Q.nxt * G.nplane);
  int ixt = xt, ip = p, ib = b, ist = 0;      // producer's copy (lane 0 only), runs S-1 tiles ahead
  auto issue = [&]() {
    mbar_expect_tx(&full[ist], Q.box_bytes);
    tma_load_4d(stages + (size_t)ist * Q.stage_stride, &mapT2, &full[ist], 2 * ixt * XT, 0, ip, ib);
    if (++ist == Q.S) ist = 0;
    if (++ixt == Q.nxt) { ixt = 0; if (++ip == G.nplane) { ip = 0; ib++; } }
  };
  if (t == 0)
    for (int j = 0; j < Q.S - 1 && j < nmine; j++) issue();
  int st = 0; uint32_t ph = 0;
  for (int it = 0; it < nmine; it++) {
    if (t == 0 && it + Q.S - 1 < nmine) issue();
    const int x = xt * XT + px;
    const bool xok = x < G.n1;
    const Run r = runs[p];
    const cplx *in = reinterpret_cast<const cplx *>(stages + (size_t)st * Q.stage_stride) + px;
    mbar_wait(&full[st], ph);
    cplx v[NS];
    if (s < R1) {
#pragma unroll
      for (int b2 = 0; b2 < R2; b2++) v[b2] = in[(s + R1 * b2) * XT];
      Dft<R2, -1>::run(v);
#pragma unroll
      for (int cc = 1; cc < R2; cc++) v[cc] = cmulc(v[cc], tws[s * cc]);
#pragma unroll
      for (int cc = 0; cc < R2; cc++) sm[cc * KS + s * XT + px] = v[cc];
    }
    __syncthreads();
    if (s < R2) {
#pragma unroll
      for (int a = 0; a < R1; a++) v[a] = sm[s * KS + a * XT + px];
      Dft<R1, -1>::run(v);
      cplx *dst = T1 + (size_t)b * G.t1_band + x;
#pragma unroll
      for (int d = 0; d < R1; d++) {
        int c = xok ? run_map(r, s + R2 * d) : -1;
        if (c >= 0) dst[(size_t)c * G.n1] = v[d];
      }
    }
    __syncthreads();
    if (++st == Q.S) { st = 0; ph ^= 1; }
    if (++xt == Q.nxt) { xt = 0; if (++p == G.nplane) { p = 0; b++; } }
  }
}

// ---- pass C: box {XT x, one y, all occupied planes} of T2; a CTA owns a contiguous range of tiles with the
//      band fastest, so its V(r)/N tile [n3][XT] is staged in shared memory once per (y, x-tile) group.
template <int R1, int R2>
__global__ void __launch_bounds__(F2C_THREADS, F2C_PER_SM)
fft2_c_ring_kernel(const __grid_constant__ CUtensorMap mapT2, Fft2Geom G, cplx *__restrict__ T2,
                   const double *__restrict__ vloc, RingParams Q) {
  constexpr int NS = imax(R1, R2);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int XT = (F2C_THREADS / NS) & ~7;     // a function of the radices only: all tile addressing is immediate
  constexpr int KSa = pad8(R2 * XT, XT), KSb = pad8(R1 * XT, XT);
  constexpr int exn = imax(R1 * KSa, R2 * KSb);
  unsigned char *stages = smem_raw;
  cplx *sm = reinterpret_cast<cplx *>(stages + (size_t)Q.S * Q.stage_stride);
  double *vs = reinterpret_cast<double *>(sm + exn);
  cplx *tws = reinterpret_cast<cplx *>(vs + ((G.n3 * XT + 1) & ~1));   // twiddles exp(+2 pi i j / n3), j < n3
  uint64_t *full = reinterpret_cast<uint64_t *>(tws + G.n3);
  const int t = threadIdx.x, px = t % XT, s = t / XT;
  for (int i = t; i < G.n3; i += blockDim.x) tws[i] = __ldg(G.tw3 + i);
  if (t == 0) {
    for (int i = 0; i < Q.S; i++) mbar_init(&full[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int first = (int)(((int64_t)Q.ntiles * blockIdx.x) / gridDim.x);
  const int nmine = (int)(((int64_t)Q.ntiles * (blockIdx.x + 1)) / gridDim.x) - first;
  // the (x, y) plane is one flat index xy = x + n1 y (x-lines are contiguous in T2 and V), tiled XT at a time
  const size_t pstride = (size_t)G.n2 * G.n1;
  int b = first % Q.nb, g = first / Q.nb;
  int ib = b, ig = g, ist = 0;      // producer's copy (lane 0 only), runs S-1 tiles ahead
  auto issue = [&]() {
    mbar_expect_tx(&full[ist], Q.box_bytes);
    tma_load_3d(stages + (size_t)ist * Q.stage_stride, &mapT2, &full[ist], 2 * ig * XT, 0, ib);
    if (++ist == Q.S) ist = 0;
    if (++ib == Q.nb) { ib = 0; ig++; }
  };
  if (t == 0)
    for (int j = 0; j < Q.S - 1 && j < nmine; j++) issue();
  int st = 0; uint32_t ph = 0;
  bool newgroup = true;
  // which of this thread's z = s + R2 j are occupied planes, and in which of the two runs: fixed for the whole kernel
  unsigned vmask = 0, hmask = 0;
#pragma unroll
  for (int j1 = 0; j1 < R1; j1++) {
    const int z = s + R2 * j1;
    if (run_map(G.zrun, z) >= 0) vmask |= 1u << j1;
    if ((unsigned)(z - G.zrun.hi) < (unsigned)G.zrun.nhi) hmask |= 1u << j1;
  }
  const int off1 = (s - G.zrun.lo) * XT, off2 = (s - G.zrun.hi + G.zrun.nlo) * XT;   // plane ordinal * XT minus R2 j XT
  for (int it = 0; it < nmine; it++) {
    if (t == 0 && it + Q.S - 1 < nmine) issue();
    const size_t xy = (size_t)g * XT + px;
    const bool xok = xy < pstride;
    if (newgroup) {
      // every read of the previous V tile happened before the barrier that ended the last iteration
      const double *vp = vloc + (size_t)g * XT;
      for (int i = t; i < G.n3 * XT; i += blockDim.x) {
        int z = i / XT, xx = i - z * XT;
        vs[i] = ((size_t)g * XT + xx < pstride) ? __ldg(vp + (size_t)z * pstride + xx) : 0.0;
      }
      newgroup = false;
    }
    const cplx *in = reinterpret_cast<const cplx *>(stages + (size_t)st * Q.stage_stride) + px;
    mbar_wait(&full[st], ph);
    cplx v[NS];
    if (s < R2) {
#pragma unroll
      for (int j1 = 0; j1 < R1; j1++) {
        const cplx *src = in + ((hmask >> j1) & 1 ? off2 : off1) + R2 * j1 * XT;
        v[j1] = (vmask >> j1) & 1 ? *src : make_double2(0.0, 0.0);
      }
      Dft<R1, +1>::run(v);
#pragma unroll
      for (int k1 = 1; k1 < R1; k1++) v[k1] = cmul(v[k1], tws[s * k1]);
#pragma unroll
      for (int k1 = 0; k1 < R1; k1++) sm[k1 * KSa + s * XT + px] = v[k1];
    }
    __syncthreads();
    if (s < R1) {
      // The second exchange is IN PLACE: this thread writes its R2 results exactly where it read its R2 inputs
      // (row s, slots j2), so no other thread's pending read is overwritten and no barrier is needed before the
      // writes; the last stage then reads sm[a][s] -- the slots the same thread fills again in the next tile's first
      // stage -- so the barrier at the end of the tile is not needed either: two CTA barriers per tile instead of four.
#pragma unroll
      for (int j2 = 0; j2 < R2; j2++) v[j2] = sm[s * KSa + j2 * XT + px];
      Dft<R2, +1>::run(v);
#pragma unroll
      for (int k2 = 0; k2 < R2; k2++) v[k2] = cscale(v[k2], vs[(s + R1 * k2) * XT + px]);
      Dft<R2, -1>::run(v);
#pragma unroll
      for (int cc = 1; cc < R2; cc++) v[cc] = cmulc(v[cc], tws[s * cc]);
#pragma unroll
      for (int cc = 0; cc < R2; cc++) sm[s * KSa + cc * XT + px] = v[cc];
    }
    __syncthreads();
    if (s < R2) {
#pragma unroll
      for (int a = 0; a < R1; a++) v[a] = sm[a * KSa + s * XT + px];
      Dft<R1, -1>::run(v);
      cplx *base = T2 + (size_t)b * G.t2_band + xy;
#pragma unroll
      const unsigned smask = xok ? vmask : 0u;
      cplx *base1 = base + (ptrdiff_t)(s - G.zrun.lo) * (ptrdiff_t)pstride, *base2 = base + (ptrdiff_t)(s - G.zrun.hi + G.zrun.nlo) * (ptrdiff_t)pstride;
#pragma unroll
      for (int d = 0; d < R1; d++)
        if ((smask >> d) & 1) ((hmask >> d) & 1 ? base2 : base1)[(size_t)(R2 * d) * pstride] = v[d];
    }
    if (++st == Q.S) { st = 0; ph ^= 1; }
    if (++b == Q.nb) { b = 0; newgroup = true; g++; }
  }
}

// ---- pass C with two barrier domains per CTA (16-line tiles, NS <= 16): warps 0-3 work on the first eight lines of a
//      tile, warps 4-7 on the other eight, each group with its own named barrier, its own half of the V tile and its own
//      pace; ring, exchange buffer and twiddles are shared.  The kernel above synchronises all eight warps twice per tile,
//      so a CTA's shared-memory phases and FP64 phases alternate (ncu: their times ADD UP to the kernel time); with four
//      barrier domains per SM instead of two, one domain's exchanges can overlap another's transforms.  A ring slot is
//      written by the TMA for both groups, so it is released by an `empty` mbarrier that both groups arrive on after their
//      reads; the producer lane (thread 0) waits for it before re-filling the slot.
template <int R1, int R2>
__global__ void __launch_bounds__(256, 2)
fft2_c_ring2_kernel(const __grid_constant__ CUtensorMap mapT2, Fft2Geom G, cplx *__restrict__ T2,
                    const double *__restrict__ vloc, RingParams Q) {
  constexpr int NS = imax(R1, R2);
  static_assert(NS <= 16, "sixteen slot rows per group");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int XT = 16, HX = 8;
  constexpr int KSa = pad8(R2 * XT, XT), KSb = pad8(R1 * XT, XT);
  constexpr int exn = imax(R1 * KSa, R2 * KSb);
  unsigned char *stages = smem_raw;
  cplx *sm = reinterpret_cast<cplx *>(stages + (size_t)Q.S * Q.stage_stride);
  double *vs = reinterpret_cast<double *>(sm + exn);
  cplx *tws = reinterpret_cast<cplx *>(vs + ((G.n3 * XT + 1) & ~1));   // twiddles exp(+2 pi i j / n3), j < n3
  uint64_t *full = reinterpret_cast<uint64_t *>(tws + G.n3), *empty = full + Q.S;
  const int t = threadIdx.x, grp = t >> 7, tl = t & 127, px = grp * HX + (tl & 7), s = tl >> 3;
  for (int i = t; i < G.n3; i += blockDim.x) tws[i] = __ldg(G.tw3 + i);
  if (t == 0) {
    for (int i = 0; i < Q.S; i++) { mbar_init(&full[i], 1); mbar_init(&empty[i], 2); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int first = (int)(((int64_t)Q.ntiles * blockIdx.x) / gridDim.x);
  const int nmine = (int)(((int64_t)Q.ntiles * (blockIdx.x + 1)) / gridDim.x) - first;
  const size_t pstride = (size_t)G.n2 * G.n1;
  int b = first % Q.nb, g = first / Q.nb;
  int ib = b, ig = g, ist = 0, iround = 0;      // producer's copy (thread 0 only), runs S-1 tiles ahead
  auto issue = [&]() {
    if (iround > 0) mbar_wait(&empty[ist], (uint32_t)((iround - 1) & 1));
    mbar_expect_tx(&full[ist], Q.box_bytes);
    tma_load_3d(stages + (size_t)ist * Q.stage_stride, &mapT2, &full[ist], 2 * ig * XT, 0, ib);
    if (++ist == Q.S) { ist = 0; iround++; }
    if (++ib == Q.nb) { ib = 0; ig++; }
  };
  if (t == 0)
    for (int j = 0; j < Q.S - 1 && j < nmine; j++) issue();
  int st = 0; uint32_t ph = 0;
  bool newgroup = true;
  unsigned vmask = 0, hmask = 0;
#pragma unroll
  for (int j1 = 0; j1 < R1; j1++) {
    const int z = s + R2 * j1;
    if (run_map(G.zrun, z) >= 0) vmask |= 1u << j1;
    if ((unsigned)(z - G.zrun.hi) < (unsigned)G.zrun.nhi) hmask |= 1u << j1;
  }
  const int off1 = (s - G.zrun.lo) * XT, off2 = (s - G.zrun.hi + G.zrun.nlo) * XT;
  for (int it = 0; it < nmine; it++) {
    if (t == 0 && it + Q.S - 1 < nmine) issue();
    const size_t xy = (size_t)g * XT + px;
    const bool xok = xy < pstride;
    if (newgroup) {
      // this group's half of the V tile; its reads of the previous one ended before its second barrier of the last tile
      const double *vp = vloc + (size_t)g * XT + grp * HX;
      for (int i = tl; i < G.n3 * HX; i += 128) {
        const int z = i >> 3, xx = i & 7;
        vs[z * XT + grp * HX + xx] = ((size_t)g * XT + grp * HX + xx < pstride) ? __ldg(vp + (size_t)z * pstride + xx) : 0.0;
      }
      newgroup = false;
    }
    const cplx *in = reinterpret_cast<const cplx *>(stages + (size_t)st * Q.stage_stride) + px;
    mbar_wait(&full[st], ph);
    cplx v[NS];
    if (s < R2) {
#pragma unroll
      for (int j1 = 0; j1 < R1; j1++) {
        const cplx *src = in + ((hmask >> j1) & 1 ? off2 : off1) + R2 * j1 * XT;
        v[j1] = (vmask >> j1) & 1 ? *src : make_double2(0.0, 0.0);
      }
      Dft<R1, +1>::run(v);
#pragma unroll
      for (int k1 = 1; k1 < R1; k1++) v[k1] = cmul(v[k1], tws[s * k1]);
#pragma unroll
      for (int k1 = 0; k1 < R1; k1++) sm[k1 * KSa + s * XT + px] = v[k1];
    }
    if (grp == 0) asm volatile("bar.sync 1, 128;" ::: "memory"); else asm volatile("bar.sync 2, 128;" ::: "memory");
    if (tl == 0) mbar_arrive(&empty[st]);          // this group has read its half of the ring slot
    if (s < R1) {
#pragma unroll
      for (int j2 = 0; j2 < R2; j2++) v[j2] = sm[s * KSa + j2 * XT + px];
      Dft<R2, +1>::run(v);
#pragma unroll
      for (int k2 = 0; k2 < R2; k2++) v[k2] = cscale(v[k2], vs[(s + R1 * k2) * XT + px]);
      Dft<R2, -1>::run(v);
#pragma unroll
      for (int cc = 1; cc < R2; cc++) v[cc] = cmulc(v[cc], tws[s * cc]);
#pragma unroll
      for (int cc = 0; cc < R2; cc++) sm[s * KSa + cc * XT + px] = v[cc];
    }
    if (grp == 0) asm volatile("bar.sync 1, 128;" ::: "memory"); else asm volatile("bar.sync 2, 128;" ::: "memory");
    if (s < R2) {
#pragma unroll
      for (int a = 0; a < R1; a++) v[a] = sm[a * KSa + s * XT + px];
      Dft<R1, -1>::run(v);
      cplx *base = T2 + (size_t)b * G.t2_band + xy;
      const unsigned smask = xok ? vmask : 0u;
      cplx *base1 = base + (ptrdiff_t)(s - G.zrun.lo) * (ptrdiff_t)pstride, *base2 = base + (ptrdiff_t)(s - G.zrun.hi + G.zrun.nlo) * (ptrdiff_t)pstride;
#pragma unroll
      for (int d = 0; d < R1; d++)
        if ((smask >> d) & 1) ((hmask >> d) & 1 ? base2 : base1)[(size_t)(R2 * d) * pstride] = v[d];
    }
    if (++st == Q.S) { st = 0; ph ^= 1; }
    if (++b == Q.nb) { b = 0; newgroup = true; g++; }
  }
}

// ---- density (Eq. 6, :140: n(r) = sum_nk w_nk |psi_nk(r)|^2): the forward half of pass C, then
//      rho(r) += sum_b w_b |psi_b(r)|^2.  A CTA owns WHOLE groups (one flat-xy tile, all bands of the launch), keeps the
//      running sum over the bands in registers and adds it to rho once per group: no atomics, fixed summation order.
template <int R1, int R2>
__global__ void __launch_bounds__(F2_THREADS, 2)
fft2_density_kernel(const __grid_constant__ CUtensorMap mapT2, Fft2Geom G, const double *__restrict__ wgt,
                    double *__restrict__ rho, RingParams Q) {
  constexpr int NS = imax(R1, R2);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int XT = (F2_THREADS / NS) & ~7;
  constexpr int KSa = pad8(R2 * XT, XT);
  unsigned char *stages = smem_raw;
  cplx *sm = reinterpret_cast<cplx *>(stages + (size_t)Q.S * Q.stage_stride);
  cplx *tws = sm + R1 * KSa;
  uint64_t *full = reinterpret_cast<uint64_t *>(tws + G.n3);
  const int t = threadIdx.x, px = t % XT, s = t / XT;
  for (int i = t; i < G.n3; i += blockDim.x) tws[i] = __ldg(G.tw3 + i);
  if (t == 0) {
    for (int i = 0; i < Q.S; i++) mbar_init(&full[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int g0 = (int)(((int64_t)Q.nxt * blockIdx.x) / gridDim.x), g1 = (int)(((int64_t)Q.nxt * (blockIdx.x + 1)) / gridDim.x);
  const int nmine = (g1 - g0) * Q.nb;
  const size_t pstride = (size_t)G.n2 * G.n1;
  int b = 0, g = g0;
  int ib = 0, ig = g0, ist = 0;
  auto issue = [&]() {
    mbar_expect_tx(&full[ist], Q.box_bytes);
    tma_load_3d(stages + (size_t)ist * Q.stage_stride, &mapT2, &full[ist], 2 * ig * XT, 0, ib);
    if (++ist == Q.S) ist = 0;
    if (++ib == Q.nb) { ib = 0; ig++; }
  };
  if (t == 0)
    for (int j = 0; j < Q.S - 1 && j < nmine; j++) issue();
  int st = 0; uint32_t ph = 0;
  double acc[R2];
#pragma unroll
  for (int k2 = 0; k2 < R2; k2++) acc[k2] = 0.0;
  for (int it = 0; it < nmine; it++) {
    if (t == 0 && it + Q.S - 1 < nmine) issue();
    const cplx *in = reinterpret_cast<const cplx *>(stages + (size_t)st * Q.stage_stride) + px;
    mbar_wait(&full[st], ph);
    cplx v[NS];
    if (s < R2) {
#pragma unroll
      for (int j1 = 0; j1 < R1; j1++) {
        int p = run_map(G.zrun, s + R2 * j1);
        v[j1] = p >= 0 ? in[p * XT] : make_double2(0.0, 0.0);
      }
      Dft<R1, +1>::run(v);
#pragma unroll
      for (int k1 = 1; k1 < R1; k1++) v[k1] = cmul(v[k1], tws[s * k1]);
#pragma unroll
      for (int k1 = 0; k1 < R1; k1++) sm[k1 * KSa + s * XT + px] = v[k1];
    }
    __syncthreads();
    if (s < R1) {
#pragma unroll
      for (int j2 = 0; j2 < R2; j2++) v[j2] = sm[s * KSa + j2 * XT + px];
      Dft<R2, +1>::run(v);
      const double wb = __ldg(wgt + b);
#pragma unroll
      for (int k2 = 0; k2 < R2; k2++) acc[k2] += wb * (v[k2].x * v[k2].x + v[k2].y * v[k2].y);   // psi(r) at z = s + R1 k2
    }
    __syncthreads();   // the exchange buffer is rewritten by the next tile
    if (++st == Q.S) { st = 0; ph ^= 1; }
    if (++b == Q.nb) {
      const size_t xy = (size_t)g * XT + px;
      if (s < R1 && xy < pstride) {
        double *dst = rho + (size_t)s * pstride + xy;
#pragma unroll
        for (int k2 = 0; k2 < R2; k2++) { dst[(size_t)(R1 * k2) * pstride] += acc[k2]; acc[k2] = 0.0; }
      }
      b = 0; g++;
    }
  }
}

// ------------------------------------------------------------------------------------------
// host side: pair table, launch geometry
// ------------------------------------------------------------------------------------------
// (R1, R2) with R1 <= R2, both radices available as register codelets
// The file is compiled four times (-DFFT2_PART=0..3, see _build.py): each translation unit instantiates the kernels of
// a part of the pairs and exports the three dispatch functions below under a part-specific name; part 0 also holds the
// entry points, which try the parts in turn.
#ifndef FFT2_PART
#define FFT2_PART 0
#endif
#define FFT2_PAIRS_0(X) X(3, 3) X(4, 4) X(4, 5) X(4, 6) X(5, 5) X(5, 6) X(4, 8) X(6, 6) X(5, 8) X(12, 15)
#define FFT2_PAIRS_1(X) X(6, 8) X(5, 10) X(6, 10) X(8, 8) X(8, 9) X(8, 10) X(9, 9) X(9, 10) X(8, 12) X(8, 16) X(5, 9) X(6, 9)
#define FFT2_PAIRS_2(X) X(10, 10) X(9, 12) X(10, 12) X(12, 12) X(10, 15) X(10, 16) X(12, 16) X(15, 15) X(15, 16) X(16, 16) X(5, 15) X(9, 15)
// radices 18 = 2 x 9 and 20 = 4 x 5 (prime-factor codelets): 162, 200, 216, 270, 288, 300, 320, 324, 360, 400
#define FFT2_PAIRS_3(X) X(9, 18) X(10, 20) X(12, 18) X(15, 18) X(16, 18) X(15, 20) X(16, 20) X(18, 18) X(18, 20) X(20, 20) X(16, 24) X(18, 24) X(20, 24) X(24, 24)
#define FFT2_PAIRS_ALL(X) FFT2_PAIRS_0(X) FFT2_PAIRS_1(X) FFT2_PAIRS_2(X) FFT2_PAIRS_3(X)
#if FFT2_PART == 0
#define FFT2_PAIRS(X) FFT2_PAIRS_0(X)
#define FFT2_PARTFN(name) name##_p0
#elif FFT2_PART == 1
#define FFT2_PAIRS(X) FFT2_PAIRS_1(X)
#define FFT2_PARTFN(name) name##_p1
#elif FFT2_PART == 2
#define FFT2_PAIRS(X) FFT2_PAIRS_2(X)
#define FFT2_PARTFN(name) name##_p2
#else
#define FFT2_PAIRS(X) FFT2_PAIRS_3(X)
#define FFT2_PARTFN(name) name##_p3
#endif
constexpr int FFT2_NOT_MINE = 0x7f000001;   // "this pair is instantiated in another part"
struct Fft2PassArgs {      // arguments of one pass launch, the same for every part
  dft_plan *p; const Fft2Geom *G; const Fft2Batch *B; int nk, pass;
  const cplx *psi; cplx *hpsi, *T1, *T2; const double *vpot; int nb, hb, max_ncol, max_nplane; cudaStream_t st;
  const FftExtra *X; const double *wgt; double *rho;
};
#define FFT2_DECL(part) \
  int fft2_pass_##part(const Fft2PassArgs &a, int r1, int r2); \
  int fft2_batched_pass_##part(const Fft2PassArgs &a, int r1, int r2); \
  int fft2_density_pass_##part(const Fft2PassArgs &a, int r1, int r2);
FFT2_DECL(p0) FFT2_DECL(p1) FFT2_DECL(p2) FFT2_DECL(p3)

#if FFT2_PART == 0
bool fft2_pair(int n, int *r1, int *r2) {
  int best1 = 0, best2 = 0;
#define X(a, b) if ((a) * (b) == n && (best2 == 0 || (b) < best2)) { best1 = (a); best2 = (b); }
  FFT2_PAIRS_ALL(X)
#undef X
  if (!best2) return false;
  if (r1) *r1 = best1;
  if (r2) *r2 = best2;
  return true;
}
#endif

static int choose_xt2(int n1, int ns) {
  int cap = F2_THREADS / ns;
  if (cap > n1) cap = n1;
  for (int d = cap; d >= 4; d--)
    if (n1 % d == 0 && d % 2 == 0) return d;
  return cap < 1 ? 1 : cap;
}

static Fft2Geom make_geom2(const dft_plan *p, int ik, int64_t t1_band, int64_t t2_band) {
  const KPoint &kp = p->kp[ik];
  Fft2Geom G;
  G.n1 = p->n[0]; G.n2 = p->n[1]; G.n3 = p->n[2];
  G.npw = kp.npw; G.mpw = p->mpw; G.ncol = kp.ncol; G.nplane = kp.nplane;
  G.col_run = kp.col_run; G.plane_run = kp.plane_run; G.zrun = kp.zrun;
  G.tw1 = reinterpret_cast<const cplx *>(p->d_tw[0]);
  G.tw2 = reinterpret_cast<const cplx *>(p->d_tw[1]);
  G.tw3 = reinterpret_cast<const cplx *>(p->d_tw[2]);
  G.t1_band = t1_band; G.t2_band = t2_band;
  return G;
}

template <typename K>
static int set_smem(K kernel, size_t bytes) {
  if (bytes > 48 * 1024) DFT_CUDA_CHECK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return DFT_OK;
}

typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                             const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// FP64 tensor map of rank `rank` (dims/strides innermost first, strides in bytes for dims 1..), no swizzle, OOB = 0
static int encode_map(dft_plan *p, CUtensorMap *m, void *base, int rank, const cuuint64_t *dims, const cuuint64_t *strides,
                      const cuuint32_t *box) {
  cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  for (int i = 0; i < rank; i++)
    if (box[i] == 0 || box[i] > 256) return DFT_ERR_UNSUPPORTED;
  CUresult r = ((EncodeFn)p->encode_fn)(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, rank, base, dims, strides, box, estr,
                                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                        CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? DFT_OK : DFT_ERR_UNSUPPORTED;
}

// Ring launch of pass 1 (B), 2 (C) or 3 (B^-1).  Returns DFT_ERR_UNSUPPORTED (without setting the error text)
// when the tile does not fit a TMA box or two CTAs' shared memory; the caller then uses the plain kernels.
template <int R1, int R2>
static int launch_ring(dft_plan *p, const Fft2Geom &G, int pass, cplx *T1, cplx *T2, const double *vloc, int nb, int hb,
                       cudaStream_t st) {
  constexpr int NS = imax(R1, R2);
  if (!p->encode_fn) return DFT_ERR_UNSUPPORTED;
  // passes B / B^-1 tile x; pass C tiles the flat (x, y) plane, so its XT need not divide n1: the largest multiple of 8
  // (128-byte runs, 8 full warps for NS = 15, 16) that fits the block
  int XT = choose_xt2(G.n1, NS), nxt = (G.n1 + XT - 1) / XT;
  if (pass == 2) {
    XT = (F2C_THREADS / NS) & ~7;
    if (XT < 8) return DFT_ERR_UNSUPPORTED;
    int64_t nxy = (int64_t)G.n1 * G.n2;
    if (XT > nxy) return DFT_ERR_UNSUPPORTED;    // tiny planes: the plain kernel
    nxt = (int)((nxy + XT - 1) / XT);
  }
  if (XT * NS > F2_THREADS) return DFT_ERR_UNSUPPORTED;
  const int rows = pass == 1 ? hb : (pass == 2 ? G.nplane : G.n2);
  const int KSa = pad8(R2 * XT, XT), KSb = pad8(R1 * XT, XT);
  size_t ex = sizeof(cplx) * (size_t)(pass == 1 ? R1 * KSa : (pass == 3 ? R2 * KSb : imax(R1 * KSa, R2 * KSb)));
  size_t extra = pass == 2 ? sizeof(double) * (size_t)((G.n3 * XT + 1) & ~1) + sizeof(cplx) * (size_t)G.n3
                           : sizeof(Run) * (size_t)G.nplane + (pass == 3 ? sizeof(cplx) * (size_t)G.n2 : 0);
  RingParams Q;
  Q.XT = XT; Q.nxt = nxt; Q.nb = nb;
  Q.box_bytes = (uint32_t)((size_t)rows * XT * 16);
  Q.stage_stride = (Q.box_bytes + 127u) & ~127u;
  int64_t ntiles = (int64_t)nb * nxt * (pass == 2 ? 1 : G.nplane);
  if (ntiles > 0x7fffffffLL) return DFT_ERR_UNSUPPORTED;
  Q.ntiles = (int)ntiles;
  const size_t fixed = ex + extra + 8 * 8;
  const size_t budget2 = (size_t)(p->smem_per_sm / 2) - 1024, budget1 = (size_t)p->smem_optin;
  int S = 0, per_sm = 2;
  if (pass == 2 && F2C_PER_SM > 2)        // small pass-C tiles: as many CTAs per SM as shared memory allows (each is its own barrier domain)
    for (int c = F2C_PER_SM; c > 2 && !S; c--)
      if (fixed + 2 * (size_t)Q.stage_stride <= (size_t)(p->smem_per_sm / c) - 1024) { S = 2; per_sm = c; }
  for (int s = 4; s >= 2 && !S; s--)
    if (fixed + (size_t)s * Q.stage_stride <= budget2) S = s;
  if (!S) {
    per_sm = 1;
    for (int s = 4; s >= 2 && !S; s--)
      if (fixed + (size_t)s * Q.stage_stride <= budget1) S = s;
  }
  if (!S) return DFT_ERR_UNSUPPORTED;
  Q.S = S;
  const size_t smem = fixed + (size_t)S * Q.stage_stride;
  CUtensorMap map;
  int rc;
  if (pass == 1) {
    cuuint64_t dims[3] = {2 * (cuuint64_t)G.n1, (cuuint64_t)G.ncol, (cuuint64_t)nb};
    cuuint64_t strides[2] = {(cuuint64_t)G.n1 * 16, (cuuint64_t)G.t1_band * 16};
    cuuint32_t box[3] = {2 * (cuuint32_t)XT, (cuuint32_t)rows, 1};
    if ((rc = encode_map(p, &map, T1, 3, dims, strides, box))) return rc;
  } else if (pass == 2) {
    cuuint64_t dims[3] = {2 * (cuuint64_t)G.n1 * G.n2, (cuuint64_t)G.nplane, (cuuint64_t)nb};
    cuuint64_t strides[2] = {(cuuint64_t)G.n1 * G.n2 * 16, (cuuint64_t)G.t2_band * 16};
    cuuint32_t box[3] = {2 * (cuuint32_t)XT, (cuuint32_t)rows, 1};
    if ((rc = encode_map(p, &map, T2, 3, dims, strides, box))) return rc;
  } else {
    cuuint64_t dims[4] = {2 * (cuuint64_t)G.n1, (cuuint64_t)G.n2, (cuuint64_t)G.nplane, (cuuint64_t)nb};
    cuuint64_t strides[3] = {(cuuint64_t)G.n1 * 16, (cuuint64_t)G.n1 * G.n2 * 16, (cuuint64_t)G.t2_band * 16};
    cuuint32_t box[4] = {2 * (cuuint32_t)XT, (cuuint32_t)rows, 1, 1};
    if ((rc = encode_map(p, &map, T2, 4, dims, strides, box))) return rc;
  }
  int grid = per_sm * p->sm_count;
  if (grid > Q.ntiles) grid = Q.ntiles;
  if (pass == 1) {
    if ((rc = set_smem(fft2_b_fwd_ring_kernel<R1, R2>, smem))) return rc;
    fft2_b_fwd_ring_kernel<R1, R2><<<grid, XT * NS, smem, st>>>(map, G, T2, Q);
  } else if (pass == 3) {
    if ((rc = set_smem(fft2_b_inv_ring_kernel<R1, R2>, smem))) return rc;
    fft2_b_inv_ring_kernel<R1, R2><<<grid, XT * NS, smem, st>>>(map, G, T1, Q);
  } else {
    if constexpr (NS <= 16) {
      // two barrier domains per CTA: pays where a tile carries enough arithmetic per exchange (both radices >= 12: 180, 192,
      // 225, 256: -4 .. -10 %; neutral at 160 / 240; slower at 128 = 8 x 16, +23 %), hence the automatic choice (2)
      if ((p->fft_c_split == 1 || (p->fft_c_split == 2 && R1 >= 12 && R2 >= 12)) && XT == 16 && F2C_THREADS == 256) {
        if ((rc = set_smem(fft2_c_ring2_kernel<R1, R2>, smem))) return rc;
        fft2_c_ring2_kernel<R1, R2><<<grid, 256, smem, st>>>(map, G, T2, vloc, Q);
        DFT_CUDA_CHECK(cudaGetLastError());
        return DFT_OK;
      }
    }
    if ((rc = set_smem(fft2_c_ring_kernel<R1, R2>, smem))) return rc;
    fft2_c_ring_kernel<R1, R2><<<grid, XT * NS, smem, st>>>(map, G, T2, vloc, Q);
  }
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

template <int R1, int R2>
static int launch_pass(dft_plan *p, const Fft2Geom &G, int pass, const cplx *psi, cplx *hpsi, cplx *T1, cplx *T2, const double *vloc,
                       int nb, int hb, cudaStream_t st, const FftExtra &X) {
  constexpr int NS = imax(R1, R2);
  int rc;
  if (pass == 2 && X.vspin) {       // two-component spinors: rows in (up, down) pairs, 2 x 2 potential
    if (16 * NS > F2_THREADS) { set_error("the fused spinor pass serves radices up to 16 (box length %d)", G.n3); return DFT_ERR_UNSUPPORTED; }
    if (nb & 1) { set_error("the spinor local term needs an even number of rows per launch (got %d)", nb); return DFT_ERR_INVALID_ARG; }
    const int nxt = (G.n1 + 7) / 8;
    const size_t sm = sizeof(cplx) * (size_t)(imax(pad8(R2 * 16, 16) * R1, pad8(R1 * 16, 16) * R2) + G.n3) + sizeof(double) * 4 * (size_t)G.n3 * 8;
    const int64_t ntiles = (int64_t)(nb / 2) * nxt * G.n2;
    if (ntiles > 0x7fffffffLL) { set_error("FFT grid too large"); return DFT_ERR_UNSUPPORTED; }
    if (sm > (size_t)p->smem_optin) { set_error("the spinor pass needs %zu bytes of shared memory", sm); return DFT_ERR_UNSUPPORTED; }
    int grid = 2 * p->sm_count;
    if (grid > ntiles) grid = (int)ntiles;
    if ((rc = set_smem(fft2_c_spinor_kernel<R1, R2>, sm))) return rc;
    fft2_c_spinor_kernel<R1, R2><<<grid, 16 * NS, sm, st>>>(G, T2, X.vspin, nxt, nb / 2, (int)ntiles);
    DFT_CUDA_CHECK(cudaGetLastError());
    return DFT_OK;
  }
  if (pass >= 1 && pass <= 3 && (p->fft_path == 0 || p->fft_path == 4)) {
    rc = launch_ring<R1, R2>(p, G, pass, T1, T2, vloc, nb, hb, st);
    if (rc != DFT_ERR_UNSUPPORTED) return rc;
  }
  if (pass == 0 || pass == 4) {
    int lpc = F2_THREADS / NS;
    if (lpc > G.ncol) lpc = G.ncol;
    int ntile = (G.ncol + lpc - 1) / lpc;
    constexpr int LSf = pad8(R1 * (R2 | 1), NS), LSi = pad8(R2 * (R1 | 1), NS);
    size_t sm = sizeof(cplx) * (size_t)lpc * (pass == 0 ? LSf : LSi);
    int64_t grid = (int64_t)nb * ntile;
    if (grid > 0x7fffffffLL) { set_error("FFT grid too large"); return DFT_ERR_UNSUPPORTED; }
    if (pass == 0) {
      if (X.pre) {
        if ((rc = set_smem(fft2_a_fwd_kernel<R1, R2, false, true>, sm))) return rc;
        fft2_a_fwd_kernel<R1, R2, false, true><<<(unsigned)grid, lpc * NS, sm, st>>>(G, Fft2Batch(), psi, T1, lpc, ntile, X.pre);
      } else {
        if ((rc = set_smem(fft2_a_fwd_kernel<R1, R2, false, false>, sm))) return rc;
        fft2_a_fwd_kernel<R1, R2, false, false><<<(unsigned)grid, lpc * NS, sm, st>>>(G, Fft2Batch(), psi, T1, lpc, ntile, nullptr);
      }
    } else {
      if (X.post || X.accumulate) {
        if ((rc = set_smem(fft2_a_inv_kernel<R1, R2, false, true>, sm))) return rc;
        fft2_a_inv_kernel<R1, R2, false, true><<<(unsigned)grid, lpc * NS, sm, st>>>(G, Fft2Batch(), T1, hpsi, lpc, ntile, X.post, X.accumulate);
      } else {
        if ((rc = set_smem(fft2_a_inv_kernel<R1, R2, false, false>, sm))) return rc;
        fft2_a_inv_kernel<R1, R2, false, false><<<(unsigned)grid, lpc * NS, sm, st>>>(G, Fft2Batch(), T1, hpsi, lpc, ntile, nullptr, 0);
      }
    }
  } else {
    int XT = choose_xt2(G.n1, NS), nxt = (G.n1 + XT - 1) / XT;
    size_t sm = sizeof(cplx) * (size_t)(pad8(R2 * XT, XT) * R1 > pad8(R1 * XT, XT) * R2 ? pad8(R2 * XT, XT) * R1 : pad8(R1 * XT, XT) * R2);
    int64_t grid = (int64_t)nb * nxt * (pass == 2 ? G.n2 : G.nplane);
    if (grid > 0x7fffffffLL) { set_error("FFT grid too large"); return DFT_ERR_UNSUPPORTED; }
    if (pass == 1) {
      if ((rc = set_smem(fft2_b_fwd_kernel<R1, R2, false>, sm))) return rc;
      fft2_b_fwd_kernel<R1, R2, false><<<(unsigned)grid, XT * NS, sm, st>>>(G, Fft2Batch(), T1, T2, XT, nxt, nb);
    } else if (pass == 3) {
      if ((rc = set_smem(fft2_b_inv_kernel<R1, R2, false>, sm))) return rc;
      fft2_b_inv_kernel<R1, R2, false><<<(unsigned)grid, XT * NS, sm, st>>>(G, Fft2Batch(), T1, T2, XT, nxt, nb);
    } else {
      if ((rc = set_smem(fft2_c_kernel<R1, R2, false>, sm))) return rc;
      fft2_c_kernel<R1, R2, false><<<(unsigned)grid, XT * NS, sm, st>>>(G, Fft2Batch(), T2, vloc, XT, nxt, nb);
    }
  }
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

// ---- several k-points per launch (small boxes, e.g. 32 k-points of a 32^3 box: one launch per pass instead of 32)
template <int R1, int R2>
static int launch_pass_batched(const Fft2Geom &G, const Fft2Batch &B, int nk, int pass, const cplx *psi, cplx *hpsi, cplx *T1,
                               cplx *T2, const double *vloc, int nb, int max_ncol, int max_nplane, cudaStream_t st) {
  constexpr int NS = imax(R1, R2);
  int rc;
  if (pass == 0 || pass == 4) {
    int lpc = F2_THREADS / NS;
    if (lpc > max_ncol) lpc = max_ncol;
    int ntile = (max_ncol + lpc - 1) / lpc;
    constexpr int LSf = pad8(R1 * (R2 | 1), NS), LSi = pad8(R2 * (R1 | 1), NS);
    size_t sm = sizeof(cplx) * (size_t)lpc * (pass == 0 ? LSf : LSi);
    int64_t grid = (int64_t)nb * ntile;
    if (grid > 0x7fffffffLL) return DFT_ERR_UNSUPPORTED;
    if (pass == 0) {
      if ((rc = set_smem(fft2_a_fwd_kernel<R1, R2, true, false>, sm))) return rc;
      fft2_a_fwd_kernel<R1, R2, true, false><<<dim3((unsigned)grid, nk), lpc * NS, sm, st>>>(G, B, psi, T1, lpc, ntile, nullptr);
    } else {
      if ((rc = set_smem(fft2_a_inv_kernel<R1, R2, true, false>, sm))) return rc;
      fft2_a_inv_kernel<R1, R2, true, false><<<dim3((unsigned)grid, nk), lpc * NS, sm, st>>>(G, B, T1, hpsi, lpc, ntile, nullptr, 0);
    }
  } else {
    int XT = choose_xt2(G.n1, NS), nxt = (G.n1 + XT - 1) / XT;
    size_t sm = sizeof(cplx) * (size_t)(pad8(R2 * XT, XT) * R1 > pad8(R1 * XT, XT) * R2 ? pad8(R2 * XT, XT) * R1 : pad8(R1 * XT, XT) * R2);
    int64_t grid = (int64_t)nb * nxt * (pass == 2 ? G.n2 : max_nplane);
    if (grid > 0x7fffffffLL) return DFT_ERR_UNSUPPORTED;
    if (pass == 1) {
      if ((rc = set_smem(fft2_b_fwd_kernel<R1, R2, true>, sm))) return rc;
      fft2_b_fwd_kernel<R1, R2, true><<<dim3((unsigned)grid, nk), XT * NS, sm, st>>>(G, B, T1, T2, XT, nxt, nb);
    } else if (pass == 3) {
      if ((rc = set_smem(fft2_b_inv_kernel<R1, R2, true>, sm))) return rc;
      fft2_b_inv_kernel<R1, R2, true><<<dim3((unsigned)grid, nk), XT * NS, sm, st>>>(G, B, T1, T2, XT, nxt, nb);
    } else {
      if ((rc = set_smem(fft2_c_kernel<R1, R2, true>, sm))) return rc;
      fft2_c_kernel<R1, R2, true><<<dim3((unsigned)grid, nk), XT * NS, sm, st>>>(G, B, T2, vloc, XT, nxt, nb);
    }
  }
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

// ---- the three dispatch functions of this part
int FFT2_PARTFN(fft2_batched_pass)(const Fft2PassArgs &a, int r1, int r2) {
#define X(q, r) if (r1 == (q) && r2 == (r)) return launch_pass_batched<q, r>(*a.G, *a.B, a.nk, a.pass, a.psi, a.hpsi, a.T1, a.T2, a.vpot, a.nb, a.max_ncol, a.max_nplane, a.st);
  FFT2_PAIRS(X)
#undef X
  return FFT2_NOT_MINE;
}

#if FFT2_PART == 0
typedef int (*PartFn)(const Fft2PassArgs &, int, int);
static int try_parts(PartFn f0, PartFn f1, PartFn f2, PartFn f3, const Fft2PassArgs &a, int r1, int r2) {
  int rc = f0(a, r1, r2);
  if (rc == FFT2_NOT_MINE) rc = f1(a, r1, r2);
  if (rc == FFT2_NOT_MINE) rc = f2(a, r1, r2);
  if (rc == FFT2_NOT_MINE) rc = f3(a, r1, r2);
  return rc == FFT2_NOT_MINE ? DFT_ERR_UNSUPPORTED : rc;
}

bool fft2_batch_ok(const dft_plan *p) {
  if (p->nkpt < 2 || p->nkpt > 65535 || p->fft_path == 1) return false;
  for (int c = 0; c < 3; c++)
    if (!fft2_pair(p->n[c], nullptr, nullptr)) return false;
  for (int ik = 0; ik < p->nkpt; ik++)
    if (!p->kp[ik].runs_ok || p->kp[ik].npw == 0) return false;
  return true;
}

// V_loc psi for `nb` bands of EVERY k-point: psi/hpsi point at the first of those bands of k-point 0, consecutive
// k-points are nband_total bands apart; ws holds T1 [nkpt][nb] then T2 [nkpt][nb] with the per-band strides of
// fft_ws_bytes_per_band's maxima.
int fft2_apply_batched(dft_plan *p, const double *psi, double *hpsi, int nb, int nband_total, void *ws, cudaStream_t st) {
  const int nk = p->nkpt;
  int64_t t1b = 0, t2b = 0;
  int max_ncol = 0, max_nplane = 0;
  for (int ik = 0; ik < nk; ik++) {
    const KPoint &kp = p->kp[ik];
    int64_t a = ((int64_t)kp.ncol * p->n[0] * 16 + 255) / 256 * 256, b = ((int64_t)kp.nplane * p->n[1] * p->n[0] * 16 + 255) / 256 * 256;
    if (a > t1b) t1b = a;
    if (b > t2b) t2b = b;
    if (kp.ncol > max_ncol) max_ncol = kp.ncol;
    if (kp.nplane > max_nplane) max_nplane = kp.nplane;
  }
  t1b /= 16; t2b /= 16;
  if (!p->d_geom2) {
    std::vector<Fft2Geom> g(nk);
    for (int ik = 0; ik < nk; ik++) g[ik] = make_geom2(p, ik, t1b, t2b);
    if (cudaMalloc(&p->d_geom2, sizeof(Fft2Geom) * nk) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the k-point geometry array"); return DFT_ERR_ALLOC; }
    DFT_CUDA_CHECK(cudaMemcpy(p->d_geom2, g.data(), sizeof(Fft2Geom) * nk, cudaMemcpyHostToDevice));
  }
  Fft2Geom G = make_geom2(p, 0, t1b, t2b);
  Fft2Batch B;
  B.Gs = reinterpret_cast<const Fft2Geom *>(p->d_geom2);
  B.ks_psi = (int64_t)nband_total * p->mpw; B.ks_t1 = (int64_t)nb * t1b; B.ks_t2 = (int64_t)nb * t2b;
  cplx *T1 = reinterpret_cast<cplx *>(ws), *T2 = T1 + (size_t)nk * nb * t1b;
  const cplx *cpsi = reinterpret_cast<const cplx *>(psi);
  cplx *chpsi = reinterpret_cast<cplx *>(hpsi);
  const int axis_of[5] = {0, 1, 2, 1, 0};
  for (int pass = 0; pass < 5; pass++) {
    int r1, r2, rc = DFT_ERR_UNSUPPORTED;
    fft2_pair(p->n[axis_of[pass]], &r1, &r2);
    phase_begin(p, pass, st);
    Fft2PassArgs a = {p, &G, &B, nk, pass, cpsi, chpsi, T1, T2, p->d_vloc, nb, 0, max_ncol, max_nplane, st, nullptr, nullptr, nullptr};
    rc = try_parts(fft2_batched_pass_p0, fft2_batched_pass_p1, fft2_batched_pass_p2, fft2_batched_pass_p3, a, r1, r2);
    phase_end(p, pass, st, 1);
    if (rc) { if (rc == DFT_ERR_UNSUPPORTED) set_error("batched FFT pass %d cannot be launched", pass); return rc; }
  }
  return DFT_OK;
}
#endif   // FFT2_PART == 0

template <int R1, int R2>
static int launch_density(dft_plan *p, const Fft2Geom &G, cplx *T2, const double *wgt, double *rho, int nb, cudaStream_t st) {
  constexpr int NS = imax(R1, R2);
  if (!p->encode_fn || G.nplane > 256) return DFT_ERR_UNSUPPORTED;
  int XT = (F2_THREADS / NS) & ~7;
  if (XT < 8) return DFT_ERR_UNSUPPORTED;
  const int64_t nxy = (int64_t)G.n1 * G.n2;
  if (XT > nxy) return DFT_ERR_UNSUPPORTED;
  RingParams Q;
  Q.XT = XT; Q.nxt = (int)((nxy + XT - 1) / XT); Q.nb = nb; Q.ntiles = 0;
  Q.box_bytes = (uint32_t)((size_t)G.nplane * XT * 16);
  Q.stage_stride = (Q.box_bytes + 127u) & ~127u;
  const size_t fixed = sizeof(cplx) * (size_t)R1 * pad8(R2 * XT, XT) + sizeof(cplx) * (size_t)G.n3 + 8 * 8;
  const size_t budget2 = (size_t)(p->smem_per_sm / 2) - 1024, budget1 = (size_t)p->smem_optin;
  int S = 0, per_sm = 2;
  for (int sg = 4; sg >= 2 && !S; sg--)
    if (fixed + (size_t)sg * Q.stage_stride <= budget2) S = sg;
  if (!S) {
    per_sm = 1;
    for (int sg = 4; sg >= 2 && !S; sg--)
      if (fixed + (size_t)sg * Q.stage_stride <= budget1) S = sg;
  }
  if (!S) return DFT_ERR_UNSUPPORTED;
  Q.S = S;
  const size_t smem = fixed + (size_t)S * Q.stage_stride;
  CUtensorMap map;
  cuuint64_t dims[3] = {2 * (cuuint64_t)nxy, (cuuint64_t)G.nplane, (cuuint64_t)nb};
  cuuint64_t strides[2] = {(cuuint64_t)nxy * 16, (cuuint64_t)G.t2_band * 16};
  cuuint32_t box[3] = {2 * (cuuint32_t)XT, (cuuint32_t)G.nplane, 1};
  int rc;
  if ((rc = encode_map(p, &map, T2, 3, dims, strides, box))) return rc;
  if ((rc = set_smem(fft2_density_kernel<R1, R2>, smem))) return rc;
  int grid = per_sm * p->sm_count;
  if (grid > Q.nxt) grid = Q.nxt;
  fft2_density_kernel<R1, R2><<<grid, XT * NS, smem, st>>>(map, G, wgt, rho, Q);
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

int FFT2_PARTFN(fft2_density_pass)(const Fft2PassArgs &a, int r1, int r2) {
#define X(q, r) if (r1 == (q) && r2 == (r)) return launch_density<q, r>(a.p, *a.G, a.T2, a.wgt, a.rho, a.nb, a.st);
  FFT2_PAIRS(X)
#undef X
  return FFT2_NOT_MINE;
}

int FFT2_PARTFN(fft2_pass)(const Fft2PassArgs &a, int r1, int r2) {
#define X(q, r) if (r1 == (q) && r2 == (r)) return launch_pass<q, r>(a.p, *a.G, a.pass, a.psi, a.hpsi, a.T1, a.T2, a.vpot, a.nb, a.hb, a.st, *a.X);
  FFT2_PAIRS(X)
#undef X
  return FFT2_NOT_MINE;
}

#if FFT2_PART == 0
// rho(r) += sum_b wgt[b] |psi_b(r)|^2 for nb bands of k-point ik: passes A and B as in H psi, then the density kernel.
// Only the register path has it: DFT_ERR_UNSUPPORTED for box lengths without a two-radix factorisation.
int fft2_density(dft_plan *p, int ik, const double *psi, const double *wgt_dev, double *rho, int nb, void *ws, cudaStream_t st,
                 const double *pre) {
  const KPoint &kp = p->kp[ik];
  if (kp.npw == 0 || nb == 0) return DFT_OK;
  int r1, r2;
  for (int c = 0; c < 3; c++)
    if (!fft2_pair(p->n[c], &r1, &r2) || !kp.runs_ok) {
      set_error("dft_accumulate_density needs box lengths with a two-radix factorisation (got %d)", p->n[c]);
      return DFT_ERR_UNSUPPORTED;
    }
  int64_t t1b = ((int64_t)kp.ncol * p->n[0] * 16 + 255) / 256 * 256, t2b = ((int64_t)kp.nplane * p->n[1] * p->n[0] * 16 + 255) / 256 * 256;
  cplx *T1 = reinterpret_cast<cplx *>(ws);
  cplx *T2 = reinterpret_cast<cplx *>(reinterpret_cast<char *>(ws) + t1b * nb);
  int rc;
  for (int pass = 0; pass < 2; pass++) {
    phase_begin(p, pass, st);
    FftExtra X;
    X.pre = pre;      // optional diagonal factor in G space (gradient component for the kinetic-energy density)
    rc = fft2_launch(p, ik, pass, psi, nullptr, T1, T2, t1b / 16, t2b / 16, nb, st, &X);
    phase_end(p, pass, st, 1);
    if (rc) return rc;
  }
  Fft2Geom G = make_geom2(p, ik, t1b / 16, t2b / 16);
  fft2_pair(p->n[2], &r1, &r2);
  rc = DFT_ERR_UNSUPPORTED;
  phase_begin(p, 2, st);
  {
    Fft2PassArgs a = {p, &G, nullptr, 1, 2, nullptr, nullptr, T1, T2, nullptr, nb, 0, 0, 0, st, nullptr, wgt_dev, rho};
    rc = try_parts(fft2_density_pass_p0, fft2_density_pass_p1, fft2_density_pass_p2, fft2_density_pass_p3, a, r1, r2);
  }
  phase_end(p, 2, st, 1);
  if (rc == DFT_ERR_UNSUPPORTED) set_error("density kernel: tile does not fit (nplane = %d)", kp.nplane);
  return rc;
}

// pass: 0 A, 1 B, 2 C, 3 B^-1, 4 A^-1.  The pair is that of the axis the pass transforms.
int fft2_launch(dft_plan *p, int ik, int pass, const double *psi, double *hpsi, void *T1, void *T2, int64_t t1_band,
                int64_t t2_band, int nb, cudaStream_t st, const FftExtra *extra) {
  FftExtra X;
  if (extra) X = *extra;
  const double *vpot = X.vpot ? X.vpot : p->d_vloc;
  int axis = (pass == 0 || pass == 4) ? 0 : (pass == 2 ? 2 : 1);
  int r1, r2;
  if (!fft2_pair(p->n[axis], &r1, &r2)) { set_error("no two-stage factorisation of %d", p->n[axis]); return DFT_ERR_UNSUPPORTED; }
  Fft2Geom G = make_geom2(p, ik, t1_band, t2_band);
  const cplx *cpsi = reinterpret_cast<const cplx *>(psi);
  cplx *chpsi = reinterpret_cast<cplx *>(hpsi), *t1 = reinterpret_cast<cplx *>(T1), *t2 = reinterpret_cast<cplx *>(T2);
  const int hb = p->kp[ik].max_cols_per_plane;
  Fft2PassArgs a = {p, &G, nullptr, 1, pass, cpsi, chpsi, t1, t2, vpot, nb, hb, 0, 0, st, &X, nullptr, nullptr};
  return try_parts(fft2_pass_p0, fft2_pass_p1, fft2_pass_p2, fft2_pass_p3, a, r1, r2);
}
#endif   // FFT2_PART == 0

}  // namespace dftb200
