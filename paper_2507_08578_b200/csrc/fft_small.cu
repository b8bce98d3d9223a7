// fft_small.cu -- K2s, the small-box path of the local term ("for c0 and c3 the box fits in one SM's
// shared memory, so the denominator there is the compulsory 2a"; PAPER.md :475 "local part using fast Fourier
// transforms", :436 "multiple concurrent Fourier transforms using an array of wave functions").
//
// When one band's pruned working set fits the shared memory of one SM, the whole local application
//
//     hpsi = FFT^-1[ V(r)/N . FFT[psi] ]        (scatter, three forward passes, V, three inverse passes, gather)
//
// is ONE kernel with one CTA per (k-point, band); HBM sees psi in, hpsi out and V (L2-resident) only:
//
//   stage psi[npw] into shared memory (coalesced)
//   A    : every non-empty (i2,i3) column: zero-padded transform along x           -> T1 [ncol][n1+1]       (shared)
//   for each slab of XS consecutive x (the y- and z-transforms act at fixed x):
//     B  : every (occupied plane, x): transform along y of the plane's columns     -> SL [nplane][n2][XS]   (shared)
//     C  : every (y, x): pad s3 -> n3, transform along z, times V(r)/N, inverse, keep the s3 occupied planes (in place)
//     B' : every (plane, x): inverse along y, keep the plane's columns              -> T1 (in place, this slab's x)
//   A'   : every column: inverse along x, gather the sphere entries                 -> staged, then stored coalesced
//
// A 1-D transform is done by ONE thread (odd n) or by a PAIR of threads (even n = 2R, lanes l and l^16 of a warp):
// each thread holds R complex numbers in registers, runs one radix-R codelet (fft_codelets.cuh) and the pair finishes
// with a radix-2 step whose operands cross by warp shuffle -- no shared-memory exchange at all, so the shared-memory
// traffic is only the pass-to-pass hand-over (what T1/T2 are in HBM for the big boxes).
//   time layout  : thread a (0/1) holds x[a + 2 i], i < R
//   freq layout  : thread a holds X[a H + i] (slot i < H) and X[R + a H + i] (slot H + i), H = ceil(R/2)
//   t2f (DIT)    : Y_a = DFT_R(x[a + 2 i]); Z_a[k] = Y_a[k] w_n^(a k); X[k] = Z_0[k] + Z_1[k], X[k + R] = Z_0[k] - Z_1[k]
//   f2t (DIF)    : y0[j] = x[j] + x[j + R], y1[j] = (x[j] - x[j + R]) w_n^j; X[2k] = DFT_R(y0)[k], X[2k + 1] = DFT_R(y1)[k]
// f2t consumes exactly what t2f produces, so pass C chains forward transform, V multiply and inverse in registers.
// Partner lanes are 16 apart so that a quarter-warp (the unit a 16-byte shared-memory access is served in) is eight
// different lines with the same a: consecutive lines are consecutive x, i.e. conflict-free.
//
// Nothing here is shared with the CPU checker.
#include "fft_small.cuh"

namespace dftb200 {

namespace {

struct SbCtx {       // what a phase needs, by value (the phases are separate functions)
  cplx *T1, *SL;
  const Run *cruns, *pruns;
  Run zrun;
  int ncol, nplane, n1, n2, XS, P1;
};

// lines are dealt to threads (NT = 1) or to lane pairs (NT = 2: 16 lines per warp, a = lane >> 4); every thread of a
// warp makes the same number of rounds (the shuffles need the whole warp), lines >= nlines compute on zeros.
template <int N> __device__ __forceinline__ void sb_line_of(int &line, int &a, int &stride) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (Line<N>::NT == 2) { line = warp * 16 + (lane & 15); a = lane >> 4; stride = (SB_THREADS / 32) * 16; }
  else { line = tid; a = 0; stride = SB_THREADS; }
}

// ---- A: sphere coefficients (staged in SL) -> x-lines in T1
template <int N> __device__ __noinline__ void sb_phase_a(SbCtx C) {
  typedef Line<N> L;
  int line, a, stride;
  sb_line_of<N>(line, a, stride);
  const cplx *src = C.SL;
  for (int c0 = 0; c0 < C.ncol; c0 += stride, line += stride) {
    const bool ok = line < C.ncol;
    const Run r = C.cruns[ok ? line : 0];
    cplx v[L::NV];
#pragma unroll
    for (int i = 0; i < L::R; i++) {
      const int g = ok ? sb_run_map(r, L::time_idx(a, i)) : -1;
      v[i] = g >= 0 ? src[g] : make_double2(0.0, 0.0);
    }
    t2f<N, +1>(v, a);
    if (ok) {
      cplx *dst = C.T1 + (size_t)line * C.P1;
#pragma unroll
      for (int i = 0; i < L::NV; i++)
        if (L::freq_ok(a, i)) dst[L::freq_idx(a, i)] = v[i];
    }
  }
}

// ---- B: along y, the columns of each occupied plane at the slab's x -> SL [plane][y][xs]
template <int N> __device__ __noinline__ void sb_phase_b(SbCtx C, int x0, int nxs) {
  typedef Line<N> L;
  int line, a, stride;
  sb_line_of<N>(line, a, stride);
  const int nlines = C.nplane * nxs;
  for (int l0 = 0; l0 < nlines; l0 += stride, line += stride) {
    const bool ok = line < nlines;
    const int p = ok ? line / nxs : 0, xs = ok ? line - p * nxs : 0;
    const Run r = C.pruns[p];
    const cplx *src = C.T1 + x0 + xs;
    cplx v[L::NV];
#pragma unroll
    for (int i = 0; i < L::R; i++) {
      const int c = ok ? sb_run_map(r, L::time_idx(a, i)) : -1;
      v[i] = c >= 0 ? src[(size_t)c * C.P1] : make_double2(0.0, 0.0);
    }
    t2f<N, +1>(v, a);
    if (ok) {
      cplx *dst = C.SL + (size_t)p * C.n2 * C.XS + xs;
#pragma unroll
      for (int i = 0; i < L::NV; i++)
        if (L::freq_ok(a, i)) dst[L::freq_idx(a, i) * C.XS] = v[i];
    }
  }
}

// ---- C: along z (pad s3 -> n3), times V(r)/N, inverse along z, keep the occupied planes; in place in SL
template <int N> __device__ __noinline__ void sb_phase_c(SbCtx C, int x0, int nxs, const double *__restrict__ vpot) {
  typedef Line<N> L;
  int line, a, stride;
  sb_line_of<N>(line, a, stride);
  const int nlines = C.n2 * nxs;
  const size_t pstride = (size_t)C.n2 * C.XS, vstride = (size_t)C.n2 * C.n1;
  for (int l0 = 0; l0 < nlines; l0 += stride, line += stride) {
    const bool ok = line < nlines;
    const int y = ok ? line / nxs : 0, xs = ok ? line - y * nxs : 0;
    cplx *base = C.SL + (size_t)y * C.XS + xs;
    const double *vp = vpot + (size_t)y * C.n1 + x0 + xs;
    double w[L::NV];
#pragma unroll
    for (int i = 0; i < L::NV; i++) w[i] = (ok && L::freq_ok(a, i)) ? __ldg(vp + (size_t)L::freq_idx(a, i) * vstride) : 0.0;
    cplx v[L::NV];
#pragma unroll
    for (int i = 0; i < L::R; i++) {
      const int p = ok ? sb_run_map(C.zrun, L::time_idx(a, i)) : -1;
      v[i] = p >= 0 ? base[(size_t)p * pstride] : make_double2(0.0, 0.0);
    }
    t2f<N, +1>(v, a);
#pragma unroll
    for (int i = 0; i < L::NV; i++) v[i] = make_double2(v[i].x * w[i], v[i].y * w[i]);   // w = 0 on slots that do not exist
    f2t<N, -1>(v, a);
    if (ok) {
#pragma unroll
      for (int i = 0; i < L::R; i++) {
        const int p = sb_run_map(C.zrun, L::time_idx(a, i));
        if (p >= 0) base[(size_t)p * pstride] = v[i];
      }
    }
  }
}

// ---- B': inverse along y, keep the plane's non-empty columns -> T1 (this slab's x)
template <int N> __device__ __noinline__ void sb_phase_binv(SbCtx C, int x0, int nxs) {
  typedef Line<N> L;
  int line, a, stride;
  sb_line_of<N>(line, a, stride);
  const int nlines = C.nplane * nxs;
  for (int l0 = 0; l0 < nlines; l0 += stride, line += stride) {
    const bool ok = line < nlines;
    const int p = ok ? line / nxs : 0, xs = ok ? line - p * nxs : 0;
    const Run r = C.pruns[p];
    const cplx *src = C.SL + (size_t)p * C.n2 * C.XS + xs;
    cplx v[L::NV];
#pragma unroll
    for (int i = 0; i < L::NV; i++) v[i] = (ok && L::freq_ok(a, i)) ? src[L::freq_idx(a, i) * C.XS] : make_double2(0.0, 0.0);
    f2t<N, -1>(v, a);
    if (ok) {
      cplx *dst = C.T1 + x0 + xs;
#pragma unroll
      for (int i = 0; i < L::R; i++) {
        const int c = sb_run_map(r, L::time_idx(a, i));
        if (c >= 0) dst[(size_t)c * C.P1] = v[i];
      }
    }
  }
}

// ---- A': inverse along x, gather the sphere entries into the staging area (SL)
template <int N> __device__ __noinline__ void sb_phase_ainv(SbCtx C) {
  typedef Line<N> L;
  int line, a, stride;
  sb_line_of<N>(line, a, stride);
  cplx *dst = C.SL;
  for (int c0 = 0; c0 < C.ncol; c0 += stride, line += stride) {
    const bool ok = line < C.ncol;
    const Run r = C.cruns[ok ? line : 0];
    const cplx *src = C.T1 + (size_t)(ok ? line : 0) * C.P1;
    cplx v[L::NV];
#pragma unroll
    for (int i = 0; i < L::NV; i++) v[i] = (ok && L::freq_ok(a, i)) ? src[L::freq_idx(a, i)] : make_double2(0.0, 0.0);
    f2t<N, -1>(v, a);
    if (ok) {
#pragma unroll
      for (int i = 0; i < L::R; i++) {
        const int g = sb_run_map(r, L::time_idx(a, i));
        if (g >= 0) dst[g] = v[i];
      }
    }
  }
}

// box lengths this path has a line transform for: 9 (one thread per line) and the even lengths 2R whose R is a codelet
#define SB_SIZES(X) X(8) X(9) X(10) X(12) X(16) X(18) X(20) X(24) X(30) X(32) X(36)

__global__ void __launch_bounds__(SB_THREADS, 1) vloc_small_kernel(SbParams Q) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int ik = blockIdx.y, b = blockIdx.x, tid = threadIdx.x;
  const SbGeom G = Q.geom[Q.ik0 + ik];
  SbCtx C;
  C.T1 = reinterpret_cast<cplx *>(smem_raw);
  C.SL = reinterpret_cast<cplx *>(smem_raw + Q.off_sl);
  Run *runs = reinterpret_cast<Run *>(smem_raw + Q.off_runs);
  C.cruns = runs; C.pruns = runs + G.ncol; C.zrun = G.zrun;
  C.ncol = G.ncol; C.nplane = G.nplane; C.n1 = Q.n1; C.n2 = Q.n2; C.XS = Q.XS; C.P1 = Q.P1;
  const size_t row = (size_t)ik * Q.kstride_psi + (size_t)b * Q.mpw;
  const cplx *psi = Q.psi + row;
  cplx *hpsi = Q.hpsi + row;
  const double *pre = Q.pre ? Q.pre + (size_t)ik * Q.kstride_pp : nullptr, *post = Q.post ? Q.post + (size_t)ik * Q.kstride_pp : nullptr;
  // run tables and the band's coefficients into shared memory
  for (int i = tid; i < G.ncol * 2; i += SB_THREADS) reinterpret_cast<int4 *>(runs)[i] = __ldg(reinterpret_cast<const int4 *>(G.col_run) + i);
  for (int i = tid; i < G.nplane * 2; i += SB_THREADS)
    reinterpret_cast<int4 *>(runs + G.ncol)[i] = __ldg(reinterpret_cast<const int4 *>(G.plane_run) + i);
  for (int g = tid; g < G.npw; g += SB_THREADS) {
    cplx v = psi[g];
    if (pre) { const double f = __ldg(pre + g); v.x *= f; v.y *= f; }
    C.SL[g] = v;
  }
  __syncthreads();
  switch (Q.n1) {
#define X(n) case n: sb_phase_a<n>(C); break;
    SB_SIZES(X)
#undef X
  }
  __syncthreads();
  for (int x0 = 0; x0 < Q.n1; x0 += Q.XS) {
    const int nxs = Q.n1 - x0 < Q.XS ? Q.n1 - x0 : Q.XS;
    switch (Q.n2) {
#define X(n) case n: sb_phase_b<n>(C, x0, nxs); break;
      SB_SIZES(X)
#undef X
    }
    __syncthreads();
    switch (Q.n3) {
#define X(n) case n: sb_phase_c<n>(C, x0, nxs, Q.vpot); break;
      SB_SIZES(X)
#undef X
    }
    __syncthreads();
    switch (Q.n2) {
#define X(n) case n: sb_phase_binv<n>(C, x0, nxs); break;
      SB_SIZES(X)
#undef X
    }
    __syncthreads();
  }
  switch (Q.n1) {
#define X(n) case n: sb_phase_ainv<n>(C); break;
    SB_SIZES(X)
#undef X
  }
  __syncthreads();
  // staged result -> hpsi (coalesced); pad entries ipw >= npw are written as 0 unless accumulating
  for (int g = tid; g < G.npw; g += SB_THREADS) {
    cplx o = C.SL[g];
    if (post) { const double f = __ldg(post + g); o.x *= f; o.y *= f; }
    if (Q.accumulate) { const cplx h = hpsi[g]; o.x += h.x; o.y += h.y; }
    hpsi[g] = o;
  }
  if (!Q.accumulate)
    for (int g = G.npw + tid; g < Q.mpw; g += SB_THREADS) hpsi[g] = make_double2(0.0, 0.0);
}

bool sb_size_ok(int n) {
  switch (n) {
#define X(m) case m: return true;
    SB_SIZES(X)
#undef X
  }
  return false;
}

struct SbLayout { int XS, P1, off_sl, off_runs; size_t smem; };

// shared-memory layout for the plan's largest k-point: T1 [max ncol][n1 + 1], then max(slab, psi staging), then the run tables
bool sb_layout(const dft_plan *p, SbLayout *out) {
  int max_ncol = 0, max_nplane = 0;
  for (const KPoint &kp : p->kp) {
    if (kp.ncol > max_ncol) max_ncol = kp.ncol;
    if (kp.nplane > max_nplane) max_nplane = kp.nplane;
  }
  const int n1 = p->n[0], n2 = p->n[1];
  const int P1 = n1 | 1;      // odd row pitch: column-per-lane accesses of passes A / A' are conflict-free
  const size_t t1 = ((size_t)max_ncol * P1 * 16 + 127) & ~(size_t)127;
  const size_t runs = (size_t)(max_ncol + max_nplane) * sizeof(Run);
  const size_t stage = (size_t)p->mpw * 16;
  // the whole x range in one slab if it fits, else the largest multiple of 8 that does
  for (int xs = n1; xs >= 1; xs = (xs == n1 ? ((n1 - 1) & ~7) : xs - 8)) {
    size_t slab = (size_t)max_nplane * n2 * xs * 16;
    if (slab < stage) slab = stage;
    slab = (slab + 127) & ~(size_t)127;
    const size_t tot = t1 + slab + runs;
    if (tot <= (size_t)p->smem_optin) {
      out->XS = xs; out->P1 = P1; out->off_sl = (int)t1; out->off_runs = (int)(t1 + slab); out->smem = tot;
      return true;
    }
    if (xs <= 8) break;
  }
  return false;
}

}  // namespace

// Can the fused small-box kernel serve this plan?  (every box length has a line transform, every k-point's occupied
// sets are runs, and the largest k-point's working set fits one CTA's shared memory)
bool fft_small_ok(const dft_plan *p) {
  if (p->nkpt < 1 || p->nkpt > 65535 || p->mpw == 0) return false;
  for (int c = 0; c < 3; c++)
    if (!sb_size_ok(p->n[c])) return false;
  for (const KPoint &kp : p->kp)
    if (!kp.runs_ok || kp.npw == 0) return false;
  SbLayout L;
  return sb_layout(p, &L);
}

// V_loc psi for `nb` bands of k-points ik0 .. ik0 + nk - 1 in one launch; psi/hpsi point at the first of those bands of
// k-point ik0, consecutive k-points are nband_total bands apart.  No scratch in device memory.
int fft_small_apply(dft_plan *p, int ik0, int nk, const double *psi, double *hpsi, int nb, int nband_total, cudaStream_t st,
                    const FftExtra *extra) {
  SbLayout L;
  if (!sb_layout(p, &L)) { set_error("small-box FFT path: the working set does not fit in shared memory"); return DFT_ERR_UNSUPPORTED; }
  if (!p->d_geom_small) {
    std::vector<SbGeom> g(p->nkpt);
    for (int ik = 0; ik < p->nkpt; ik++) {
      const KPoint &kp = p->kp[ik];
      g[ik].npw = kp.npw; g[ik].ncol = kp.ncol; g[ik].nplane = kp.nplane; g[ik].pad = 0;
      g[ik].col_run = kp.col_run; g[ik].plane_run = kp.plane_run; g[ik].zrun = kp.zrun;
    }
    if (cudaMalloc(&p->d_geom_small, sizeof(SbGeom) * p->nkpt) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the k-point geometry array"); return DFT_ERR_ALLOC; }
    DFT_CUDA_CHECK(cudaMemcpy(p->d_geom_small, g.data(), sizeof(SbGeom) * p->nkpt, cudaMemcpyHostToDevice));
  }
  if (!p->small_attr_done) {
    DFT_CUDA_CHECK(cudaFuncSetAttribute(vloc_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_optin));
    p->small_attr_done = true;
  }
  SbParams Q;
  Q.geom = reinterpret_cast<const SbGeom *>(p->d_geom_small);
  Q.psi = reinterpret_cast<const cplx *>(psi); Q.hpsi = reinterpret_cast<cplx *>(hpsi);
  Q.vpot = (extra && extra->vpot) ? extra->vpot : p->d_vloc;
  Q.pre = extra ? extra->pre : nullptr; Q.post = extra ? extra->post : nullptr;
  Q.kstride_psi = (int64_t)nband_total * p->mpw; Q.kstride_pp = (int64_t)3 * p->mpw;
  Q.n1 = p->n[0]; Q.n2 = p->n[1]; Q.n3 = p->n[2]; Q.mpw = p->mpw; Q.XS = L.XS; Q.P1 = L.P1;
  Q.accumulate = extra ? extra->accumulate : 0; Q.ik0 = ik0;
  Q.off_sl = L.off_sl; Q.off_runs = L.off_runs;
  Q.dstmap = nullptr; Q.nitems = 0; Q.nb = nb;
  if (p->fft_path != 5) {      // box shapes with a compile-time-size kernel (fft_small2.cu)
    bool handled = false;
    int rc = fft_small2_launch(p, &Q, nk, nb, st, &handled);
    if (rc || handled) return rc;
  }
  phase_begin(p, 8, st);
  vloc_small_kernel<<<dim3((unsigned)nb, (unsigned)nk), SB_THREADS, L.smem, st>>>(Q);
  phase_end(p, 8, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

}  // namespace dftb200
