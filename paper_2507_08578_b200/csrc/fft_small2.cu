// fft_small2.cu -- K2s with compile-time box sizes: the fused small-box local term of fft_small.cu (same phases, same
// pair-of-lanes line transforms, SURVEY.md 8(d) "the box fits in one SM's shared memory"; PAPER.md :475, :436) for the box
// shapes of the BASELINE cells and of the parity cells, as PERSISTENT CTAs (one per SM, 8 warps, up to 255 registers):
//
//   * every box length, the slab width XS and the row pitch are template constants: all shared-memory addressing is
//     LDS/STS with immediate offsets, no division, no switch, no local memory;
//   * the sphere coefficients are scattered straight into zeroed x-lines T1[column][x] (a per-plane-wave position table),
//     so passes A and A' are DENSE in-place line transforms without any run logic, and the result is gathered from T1
//     straight to hpsi: no staging copy;
//   * V(r)/N of a thread's next z-line is fetched from L2 into registers one phase ahead of its use;
//   * a CTA walks (k-point, band) items with stride gridDim.x and keeps the run tables of its k-point in shared memory.
//
// Selected automatically by fft_small_apply when the plan's box is one of SB2_BOXES; option fft_path = 5 keeps the
// run-time-dispatched kernel of fft_small.cu (A/B tests).  Nothing here is shared with the CPU checker.
#include "fft_small.cuh"

namespace dftb200 {

namespace {

#ifndef SB2_THREADS_N
#define SB2_THREADS_N 256
#endif
constexpr int SB2_THREADS = SB2_THREADS_N;

// lines are dealt to lane pairs (NT = 2: 16 lines per warp, a = lane >> 4) or to threads (NT = 1)
template <int N> __device__ __forceinline__ void sb2_line_of(int &line, int &a, int &stride) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (Line<N>::NT == 2) { line = warp * 16 + (lane & 15); a = lane >> 4; stride = (SB2_THREADS / 32) * 16; }
  else { line = tid; a = 0; stride = SB2_THREADS; }
}
// first line of this thread's warp in a round starting at l0 (a whole warp skips a round when it is >= nlines)
template <int N> __device__ __forceinline__ int sb2_warp_first(int l0) {
  const int warp = threadIdx.x >> 5;
  return l0 + (Line<N>::NT == 2 ? warp * 16 : warp * 32);
}

// position of box index y of a two-run set: [lo, lo + nlo) -> base + (y - lo), [hi, hi + nhi) -> base + nlo + (y - hi), else -1
__device__ __forceinline__ int sb2_map(const Run &r, int y) {
  const unsigned d0 = (unsigned)(y - r.lo), d1 = (unsigned)(y - r.hi);
  int c = -1;
  if (d1 < (unsigned)r.nhi) c = r.base + r.nlo + (int)d1;
  if (d0 < (unsigned)r.nlo) c = r.base + (int)d0;
  return c;
}

template <int N1, int N2, int N3, int XS>
__global__ void __launch_bounds__(SB2_THREADS, 1) vloc_small2_kernel(SbParams Q) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int P1 = N1 | 1;
  static_assert(N1 % XS == 0, "the slab width must divide n1");
  typedef Line<N1> L1;
  typedef Line<N2> L2;
  typedef Line<N3> L3;
  cplx *T1 = reinterpret_cast<cplx *>(smem_raw);
  cplx *SL = reinterpret_cast<cplx *>(smem_raw + Q.off_sl);
  Run *runs = reinterpret_cast<Run *>(smem_raw + Q.off_runs);
  const int tid = threadIdx.x;
  int cur_ik = -1, ncol = 0, nplane = 0, npw = 0;
  Run zrun = {0, 0, 0, 0, 0, 0, 0, 0};
  const double *__restrict__ vpot = Q.vpot;
  constexpr size_t vstride = (size_t)N2 * N1;

  // a CTA takes a contiguous range of items (mostly one k-point: run tables stay, the next band can be prefetched)
  const int per = (Q.nitems + gridDim.x - 1) / gridDim.x;
  const int it0 = blockIdx.x * per, it1 = it0 + per < Q.nitems ? it0 + per : Q.nitems;
  // the first PF * 256 coefficients of a band and their positions in T1 travel through registers, fetched one item ahead
  constexpr int PF = 8;
  cplx pf[PF];
  int dn[PF];
  if (it0 < it1) {
    const int ik = it0 / Q.nb, b = it0 - ik * Q.nb;
    const cplx *src = Q.psi + (size_t)ik * Q.kstride_psi + (size_t)b * Q.mpw;
    const int32_t *dm = Q.dstmap + (size_t)(Q.ik0 + ik) * Q.mpw;
#pragma unroll
    for (int j = 0; j < PF; j++) {
      const int g = tid + j * SB2_THREADS;
      pf[j] = g < Q.mpw ? src[g] : make_double2(0.0, 0.0);
      dn[j] = g < Q.mpw ? __ldg(dm + g) : 0;
    }
  }
  for (int item = it0; item < it1; item++) {
    const int ik = item / Q.nb, b = item - ik * Q.nb;
    if (ik != cur_ik) {
      __syncthreads();
      const SbGeom G = Q.geom[Q.ik0 + ik];
      ncol = G.ncol; nplane = G.nplane; npw = G.npw; zrun = G.zrun;
      for (int i = tid; i < ncol * 2; i += SB2_THREADS) reinterpret_cast<int4 *>(runs)[i] = __ldg(reinterpret_cast<const int4 *>(G.col_run) + i);
      for (int i = tid; i < nplane * 2; i += SB2_THREADS)
        reinterpret_cast<int4 *>(runs + ncol)[i] = __ldg(reinterpret_cast<const int4 *>(G.plane_run) + i);
      cur_ik = ik;
    }
    const Run *pruns = runs + ncol;
    const size_t row = (size_t)ik * Q.kstride_psi + (size_t)b * Q.mpw;
    const cplx *__restrict__ psi = Q.psi + row;
    cplx *__restrict__ hpsi = Q.hpsi + row;
    const int32_t *__restrict__ dst = Q.dstmap + (size_t)(Q.ik0 + ik) * Q.mpw;
    const double *pre = Q.pre ? Q.pre + (size_t)ik * Q.kstride_pp : nullptr, *post = Q.post ? Q.post + (size_t)ik * Q.kstride_pp : nullptr;

    // ---- zero the x-lines, scatter the sphere coefficients into them
    for (int i = tid; i < ncol * P1; i += SB2_THREADS) T1[i] = make_double2(0.0, 0.0);
    __syncthreads();
#pragma unroll
    for (int j = 0; j < PF; j++) {
      const int g = tid + j * SB2_THREADS;
      if (g < npw) {
        cplx v = pf[j];
        if (pre) { const double f = __ldg(pre + g); v.x *= f; v.y *= f; }
        T1[dn[j]] = v;
      }
    }
    for (int g = tid + PF * SB2_THREADS; g < npw; g += SB2_THREADS) {
      cplx v = psi[g];
      if (pre) { const double f = __ldg(pre + g); v.x *= f; v.y *= f; }
      T1[__ldg(dst + g)] = v;
    }
    __syncthreads();

    // ---- A: dense transform along x of every non-empty column, in place
    {
      int line, a, stride;
      sb2_line_of<N1>(line, a, stride);
      for (int l0 = 0; l0 < ncol; l0 += stride, line += stride) {
        if (sb2_warp_first<N1>(l0) >= ncol) break;
        const bool ok = line < ncol;
        cplx *rowp = T1 + (size_t)(ok ? line : 0) * P1;
        cplx v[L1::NV];
#pragma unroll
        for (int i = 0; i < L1::R; i++) v[i] = rowp[L1::time_idx(a, i)];
        t2f<N1, +1>(v, a);
        if (ok) {
#pragma unroll
          for (int i = 0; i < L1::NV; i++)
            if (L1::freq_ok(a, i)) rowp[L1::freq_idx(a, i)] = v[i];
        }
      }
    }
    __syncthreads();

    for (int x0 = 0; x0 < N1; x0 += XS) {
      // V(r)/N of this thread's first z-line of the slab: in flight during pass B
      int cline, ca, cstride;
      sb2_line_of<N3>(cline, ca, cstride);
      constexpr int nlines_c = N2 * XS;
      double w[L3::NV];
      {
        const bool ok = cline < nlines_c;
        const int y = ok ? cline / XS : 0, xs = ok ? cline - y * XS : 0;
        const double *vp = vpot + (size_t)y * N1 + x0 + xs;
#pragma unroll
        for (int i = 0; i < L3::NV; i++) w[i] = (ok && L3::freq_ok(ca, i)) ? __ldg(vp + (size_t)L3::freq_idx(ca, i) * vstride) : 0.0;
      }
      // ---- B: along y, the columns of each occupied plane at the slab's x -> SL [plane][y][XS]
      {
        int line, a, stride;
        sb2_line_of<N2>(line, a, stride);
        const int nlines = nplane * XS;
        for (int l0 = 0; l0 < nlines; l0 += stride, line += stride) {
          if (sb2_warp_first<N2>(l0) >= nlines) break;
          const bool ok = line < nlines;
          const int p = ok ? line / XS : 0, xs = ok ? line - p * XS : 0;
          const Run r = pruns[p];
          const cplx *src = T1 + x0 + xs;
          cplx v[L2::NV];
#pragma unroll
          for (int i = 0; i < L2::R; i++) {
            const int c = ok ? sb2_map(r, L2::time_idx(a, i)) : -1;
            v[i] = c >= 0 ? src[(size_t)c * P1] : make_double2(0.0, 0.0);
          }
          t2f<N2, +1>(v, a);
          if (ok) {
            cplx *dstp = SL + (size_t)p * N2 * XS + xs;
#pragma unroll
            for (int i = 0; i < L2::NV; i++)
              if (L2::freq_ok(a, i)) dstp[L2::freq_idx(a, i) * XS] = v[i];
          }
        }
      }
      __syncthreads();
      // ---- C: along z (pad s3 -> n3), times V(r)/N, inverse along z, keep the occupied planes; in place in SL
      {
        constexpr size_t pstride = (size_t)N2 * XS;
        for (int l0 = 0; l0 < nlines_c; l0 += cstride, cline += cstride) {
          if (sb2_warp_first<N3>(l0) >= nlines_c) break;
          const bool ok = cline < nlines_c;
          const int y = ok ? cline / XS : 0, xs = ok ? cline - y * XS : 0;
          cplx *base = SL + (size_t)y * XS + xs;
          // next round's potential values (in flight during this round's transforms)
          constexpr bool MULTI = nlines_c > (L3::NT == 2 ? SB2_THREADS / 2 : SB2_THREADS);   // more than one round per slab
          double wn[MULTI ? L3::NV : 1];
          if (MULTI) {
            const int nl = cline + cstride;
            const bool okn = nl < nlines_c;
            const int yn = okn ? nl / XS : 0, xn = okn ? nl - yn * XS : 0;
            const double *vp = vpot + (size_t)yn * N1 + x0 + xn;
#pragma unroll
            for (int i = 0; i < L3::NV; i++) wn[i] = (okn && L3::freq_ok(ca, i)) ? __ldg(vp + (size_t)L3::freq_idx(ca, i) * vstride) : 0.0;
          }
          cplx v[L3::NV];
#pragma unroll
          for (int i = 0; i < L3::R; i++) {
            const int p = ok ? sb2_map(zrun, L3::time_idx(ca, i)) : -1;
            v[i] = p >= 0 ? base[(size_t)p * pstride] : make_double2(0.0, 0.0);
          }
          t2f<N3, +1>(v, ca);
#pragma unroll
          for (int i = 0; i < L3::NV; i++) v[i] = make_double2(v[i].x * w[i], v[i].y * w[i]);   // w = 0 on slots that do not exist
          f2t<N3, -1>(v, ca);
          if (ok) {
#pragma unroll
            for (int i = 0; i < L3::R; i++) {
              const int p = sb2_map(zrun, L3::time_idx(ca, i));
              if (p >= 0) base[(size_t)p * pstride] = v[i];
            }
          }
          if (MULTI) {
#pragma unroll
            for (int i = 0; i < L3::NV; i++) w[i] = wn[i];
          }
        }
      }
      __syncthreads();
      // ---- B': inverse along y, keep the plane's non-empty columns -> T1 (this slab's x)
      {
        int line, a, stride;
        sb2_line_of<N2>(line, a, stride);
        const int nlines = nplane * XS;
        for (int l0 = 0; l0 < nlines; l0 += stride, line += stride) {
          if (sb2_warp_first<N2>(l0) >= nlines) break;
          const bool ok = line < nlines;
          const int p = ok ? line / XS : 0, xs = ok ? line - p * XS : 0;
          const Run r = pruns[p];
          const cplx *src = SL + (size_t)p * N2 * XS + xs;
          cplx v[L2::NV];
#pragma unroll
          for (int i = 0; i < L2::NV; i++) v[i] = (ok && L2::freq_ok(a, i)) ? src[L2::freq_idx(a, i) * XS] : make_double2(0.0, 0.0);
          f2t<N2, -1>(v, a);
          if (ok) {
            cplx *dstp = T1 + x0 + xs;
#pragma unroll
            for (int i = 0; i < L2::R; i++) {
              const int c = sb2_map(r, L2::time_idx(a, i));
              if (c >= 0) dstp[(size_t)c * P1] = v[i];
            }
          }
        }
      }
      __syncthreads();
    }

    // next item's coefficients and this item's gather positions: in flight during pass A'
    cplx pfn[PF];
    int dnn[PF], dg[PF];
    {
      const bool more = item + 1 < it1;
      const int ikn = more ? (item + 1) / Q.nb : ik, bn = more ? (item + 1) - ikn * Q.nb : b;
      const cplx *src = Q.psi + (size_t)ikn * Q.kstride_psi + (size_t)bn * Q.mpw;
      const int32_t *dm = Q.dstmap + (size_t)(Q.ik0 + ikn) * Q.mpw;
#pragma unroll
      for (int j = 0; j < PF; j++) {
        const int g = tid + j * SB2_THREADS;
        const bool in = g < Q.mpw;
        pfn[j] = (more && in) ? src[g] : make_double2(0.0, 0.0);
        dnn[j] = (more && in) ? __ldg(dm + g) : 0;
        dg[j] = in ? __ldg(dst + g) : 0;
      }
    }
    // ---- A': dense inverse along x, in place
    {
      int line, a, stride;
      sb2_line_of<N1>(line, a, stride);
      for (int l0 = 0; l0 < ncol; l0 += stride, line += stride) {
        if (sb2_warp_first<N1>(l0) >= ncol) break;
        const bool ok = line < ncol;
        cplx *rowp = T1 + (size_t)(ok ? line : 0) * P1;
        cplx v[L1::NV];
#pragma unroll
        for (int i = 0; i < L1::NV; i++) v[i] = L1::freq_ok(a, i) ? rowp[L1::freq_idx(a, i)] : make_double2(0.0, 0.0);
        f2t<N1, -1>(v, a);
        if (ok) {
#pragma unroll
          for (int i = 0; i < L1::R; i++) rowp[L1::time_idx(a, i)] = v[i];
        }
      }
    }
    __syncthreads();
    // ---- gather the sphere entries (coalesced stores); pad entries ipw >= npw are written as 0 unless accumulating
#pragma unroll
    for (int j = 0; j < PF; j++) {
      const int g = tid + j * SB2_THREADS;
      if (g < npw) {
        cplx o = T1[dg[j]];
        if (post) { const double f = __ldg(post + g); o.x *= f; o.y *= f; }
        if (Q.accumulate) { const cplx h = hpsi[g]; o.x += h.x; o.y += h.y; }
        hpsi[g] = o;
      }
    }
    for (int g = tid + PF * SB2_THREADS; g < npw; g += SB2_THREADS) {
      cplx o = T1[__ldg(dst + g)];
      if (post) { const double f = __ldg(post + g); o.x *= f; o.y *= f; }
      if (Q.accumulate) { const cplx h = hpsi[g]; o.x += h.x; o.y += h.y; }
      hpsi[g] = o;
    }
    if (!Q.accumulate)
      for (int g = npw + tid; g < Q.mpw; g += SB2_THREADS) hpsi[g] = make_double2(0.0, 0.0);
#pragma unroll
    for (int j = 0; j < PF; j++) { pf[j] = pfn[j]; dn[j] = dnn[j]; }
    __syncthreads();
  }
}

// box shapes with an instantiation: (n1, n2, n3, slab width).  A narrower slab is taken when the wide one does not fit.
#define SB2_BOXES(X) X(20, 20, 20, 20) X(20, 20, 20, 10) X(32, 32, 32, 8) X(30, 30, 30, 10) X(36, 36, 36, 12) X(20, 24, 30, 10)

struct Sb2Layout { int off_sl, off_runs; size_t smem; };

bool sb2_layout(const dft_plan *p, int xs, Sb2Layout *out) {
  int max_ncol = 0, max_nplane = 0;
  for (const KPoint &kp : p->kp) {
    if (kp.ncol > max_ncol) max_ncol = kp.ncol;
    if (kp.nplane > max_nplane) max_nplane = kp.nplane;
  }
  const int n1 = p->n[0], n2 = p->n[1], P1 = n1 | 1;
  const size_t t1 = ((size_t)max_ncol * P1 * 16 + 127) & ~(size_t)127;
  const size_t slab = ((size_t)max_nplane * n2 * xs * 16 + 127) & ~(size_t)127;
  const size_t runs = (size_t)(max_ncol + max_nplane) * sizeof(Run);
  out->off_sl = (int)t1; out->off_runs = (int)(t1 + slab); out->smem = t1 + slab + runs;
  return out->smem <= (size_t)p->smem_optin;
}

}  // namespace

// Launches the compile-time-size kernel if the plan's box has one; *handled tells whether it did.
int fft_small2_launch(dft_plan *p, void *params, int nk, int nb, cudaStream_t st, bool *handled) {
  SbParams Q = *reinterpret_cast<SbParams *>(params);
  *handled = false;
  if (!p->d_dstmap) {
    // position of every plane wave in T1: column ordinal * P1 + x (columns are contiguous runs of the ascending list)
    const int P1 = p->n[0] | 1;
    std::vector<int32_t> m((size_t)p->nkpt * p->mpw, 0);
    for (int ik = 0; ik < p->nkpt; ik++) {
      const KPoint &kp = p->kp[ik];
      int col = -1; int64_t last = -1;
      for (int g = 0; g < kp.npw; g++) {
        const int64_t idx = kp.h_igfft[g], c = idx / p->n[0];
        if (c != last) { col++; last = c; }
        m[(size_t)ik * p->mpw + g] = col * P1 + (int)(idx % p->n[0]);
      }
    }
    if (cudaMalloc(&p->d_dstmap, sizeof(int32_t) * (m.size() ? m.size() : 1)) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the scatter map"); return DFT_ERR_ALLOC; }
    DFT_CUDA_CHECK(cudaMemcpy(p->d_dstmap, m.data(), sizeof(int32_t) * m.size(), cudaMemcpyHostToDevice));
  }
  Q.dstmap = p->d_dstmap; Q.nitems = nk * nb; Q.nb = nb;
  int grid = Q.nitems < p->sm_count ? Q.nitems : p->sm_count;
  { const int per = (Q.nitems + grid - 1) / grid; grid = (Q.nitems + per - 1) / per; }   // contiguous item ranges, none empty
  Sb2Layout L;
#define X(a, b, c, xs)                                                                                              \
  if (!*handled && p->n[0] == a && p->n[1] == b && p->n[2] == c && sb2_layout(p, xs, &L)) {                         \
    if (!(p->small2_attr_mask & (1u << slot))) {                                                                     \
      DFT_CUDA_CHECK(cudaFuncSetAttribute(vloc_small2_kernel<a, b, c, xs>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_optin)); \
      p->small2_attr_mask |= 1u << slot;                                                                             \
    }                                                                                                                \
    Q.off_sl = L.off_sl; Q.off_runs = L.off_runs; Q.XS = xs; Q.P1 = a | 1;                                           \
    phase_begin(p, 8, st);                                                                                           \
    vloc_small2_kernel<a, b, c, xs><<<grid, SB2_THREADS, L.smem, st>>>(Q);                                           \
    phase_end(p, 8, st, 1);                                                                                          \
    *handled = true;                                                                                                 \
  }                                                                                                                  \
  slot++;
  int slot = 0;
  SB2_BOXES(X)
#undef X
  if (*handled) DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

}  // namespace dftb200
