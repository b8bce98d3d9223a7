// fft_small.cuh -- pieces shared by the two fused small-box kernels of the local term (fft_small.cu: any supported box,
// sizes dispatched at run time; fft_small2.cu: compile-time box sizes, persistent CTAs): the pair-of-lanes line
// transforms and the kernel parameter blocks.  See fft_small.cu for the layouts.  Nothing here is shared with the CPU checker.
#pragma once
#include "fft_codelets.cuh"
#include "fft_tw_literals.cuh"
#include "internal.h"

namespace dftb200 {
namespace {

constexpr int SB_THREADS = 512;

__device__ __forceinline__ int sb_run_map(const Run &r, int x) {
  unsigned d = (unsigned)(x - r.lo);
  if (d < (unsigned)r.nlo) return r.base + (int)d;
  d = (unsigned)(x - r.hi);
  if (d < (unsigned)r.nhi) return r.base + r.nlo + (int)d;
  return -1;
}

template <int N> struct Line {
  static constexpr int NT = (N % 2 == 0 && N >= 8) ? 2 : 1;
  static constexpr int R = N / NT;
  static constexpr int H = NT == 2 ? (R + 1) / 2 : N;
  static constexpr int NV = NT == 2 ? 2 * H : N;
  // box index of time-layout slot i (i < R) and of freq-layout slot i (i < NV); freq_ok: the slot exists
  static __device__ __forceinline__ int time_idx(int a, int i) { return a + NT * i; }
  static __device__ __forceinline__ int freq_idx(int a, int i) { return NT == 1 ? i : (i < H ? a * H + i : R + a * H + (i - H)); }
  static __device__ __forceinline__ bool freq_ok(int a, int i) { return NT == 1 ? true : (a * H + (i < H ? i : i - H) < R); }
};

__device__ __forceinline__ cplx shfl16(cplx v) {
  return make_double2(__shfl_xor_sync(0xffffffffu, v.x, 16), __shfl_xor_sync(0xffffffffu, v.y, 16));
}
__device__ __forceinline__ double flip_if(double v, int a) {   // a ? -v : v, on the integer pipe
  return __hiloint2double(__double2hiint(v) ^ (a << 31), __double2loint(v));
}

// time layout -> freq layout, w = exp(S 2 pi i / N)
template <int N, int S> __device__ __forceinline__ void t2f(cplx (&v)[Line<N>::NV], int a) {
  typedef Line<N> L;
  if constexpr (L::NT == 1) { Dft<N, S>::run(v); return; } else {
  constexpr int R = L::R, H = L::H;
  Dft<R, S>::run(v);
#pragma unroll
  for (int k = 1; k < R; k++) {
    const double c = a ? tw_cos(N, k) : 1.0, s = a ? S * tw_sin(N, k) : 0.0;
    v[k] = make_double2(v[k].x * c - v[k].y * s, v[k].x * s + v[k].y * c);
  }
#pragma unroll
  for (int i = 0; i < H; i++) {
    const cplx lo = v[i], hi = v[H + i < R ? H + i : R - 1];
    const cplx own = a ? hi : lo, send = a ? lo : hi;
    const cplx recv = shfl16(send);
    v[i] = make_double2(own.x + recv.x, own.y + recv.y);
    v[H + i] = make_double2(flip_if(own.x - recv.x, a), flip_if(own.y - recv.y, a));
  }
  }
}

// freq layout -> time layout, w = exp(S 2 pi i / N)
template <int N, int S> __device__ __forceinline__ void f2t(cplx (&v)[Line<N>::NV], int a) {
  typedef Line<N> L;
  if constexpr (L::NT == 1) { Dft<N, S>::run(v); return; } else {
  constexpr int R = L::R, H = L::H;
#pragma unroll
  for (int i = 0; i < H; i++) {
    const cplx x0 = v[i], x1 = v[H + i];
    const cplx s = make_double2(x0.x + x1.x, x0.y + x1.y), d0 = make_double2(x0.x - x1.x, x0.y - x1.y);
    const int k1 = H + i < R ? H + i : R - 1;
    const double c = a ? tw_cos(N, k1) : tw_cos(N, i), sn = a ? S * tw_sin(N, k1) : S * tw_sin(N, i);
    const cplx d = make_double2(d0.x * c - d0.y * sn, d0.x * sn + d0.y * c);
    const cplx send = a ? s : d, keep = a ? d : s;
    const cplx recv = shfl16(send);
    v[i] = a ? recv : keep;
    if (H + i < R) v[H + i] = a ? keep : recv;
  }
  Dft<R, S>::run(v);
  }
}

struct SbGeom {      // per k-point, device memory
  int npw, ncol, nplane, pad;
  const Run *col_run, *plane_run;
  Run zrun;
};

struct SbParams {
  const SbGeom *geom;
  const cplx *psi; cplx *hpsi;
  const double *vpot;                 // [n3][n2][n1], pre-scaled by 1/N
  const double *pre, *post;           // optional diagonal factors in G space (per k-point: + ik * kstride_pp), null = 1
  int64_t kstride_psi, kstride_pp;    // complex / double elements between consecutive k-points
  int n1, n2, n3, mpw, XS, P1, accumulate, ik0;
  int off_sl, off_runs;               // byte offsets of the slab / staging region and of the run tables in shared memory
  // fft_small2.cu only: position (column * P1 + x) of every plane wave in T1, [nkpt][mpw]; work items = nk * nb (k, band) pairs
  const int32_t *dstmap;
  int nitems, nb;
};

}  // namespace
}  // namespace dftb200
