// fft.cu -- K2: the local term  V_loc psi = FFT^-1[ V_loc(r) . FFT[psi] ]  (PAPER.md :475 "local part
// using fast Fourier transforms", :436 "multiple concurrent Fourier transforms using an array of
// wave functions"), as a sphere-pruned, batched complex128 3-D transform in five passes
// (SURVEY.md 8(a) steps S3-S7):
//
//   A    scatter sphere -> zero-padded x-lines, transform along x, only the ncol non-empty (i2,i3) columns
//   B    transform along y for every x, only the s3 non-empty i3 planes
//   C    per (x,y) line: pad s3 -> n3, transform along z, multiply by V(r)/N, inverse transform, keep s3
//   B^-1 inverse along y, keep only the non-empty columns
//   A^-1 inverse along x, gather the sphere entries -> hpsi
//
// Reading 4: G->r uses exp(+2 pi i m.j/n) unscaled, r->G uses exp(-...) and 1/N; the
// 1/N is folded into the stored potential by dft_set_vloc.  The pruned sequence is an exact
// re-arrangement of the full-box transform (skipped lines are identically zero on the way in and
// are never read on the way out).
//
// Every pass stages its lines in shared memory and runs Stockham autosort radix passes
// (radices 2,3,4,5,8,9) with one butterfly per thread; strided passes (B, C) keep x fastest so
// that global accesses are contiguous runs of XT complex numbers and shared accesses are
// conflict-free.
#include <math.h>

#include "fft_codelets.cuh"
#include "internal.h"

namespace dftb200 {

// ------------------------------------------------------------------------------------------
// factorisation of a 1-D length into the radices the butterflies below implement
// ------------------------------------------------------------------------------------------
bool factorize(int n, FftFactors *f) {
  f->n = n; f->nfac = 0;
  if (n < 1) return false;
  int e2 = 0, e3 = 0, e5 = 0, m = n;
  while (m % 2 == 0) { m /= 2; e2++; }
  while (m % 3 == 0) { m /= 3; e3++; }
  while (m % 5 == 0) { m /= 5; e5++; }
  if (m != 1) return false;
  auto push = [&](int r) { f->radix[f->nfac++] = r; };
  while (e3 >= 2) { push(9); e3 -= 2; }
  if (e3) push(3);
  for (int i = 0; i < e5; i++) push(5);
  if (e2 == 1) push(2);
  else if (e2 % 3 == 1) { push(4); push(4); e2 -= 4; }
  else if (e2 % 3 == 2) { push(4); e2 -= 2; }
  if (e2 >= 3) while (e2 > 0) { push(8); e2 -= 3; }
  return f->nfac <= 12;
}

struct FacDev { int nfac; int radix[12]; };

// One Stockham pass of radix R over `nlines` lines held in shared memory.
// element j of line l sits at buf[l*ls + j*es]; tw[j] = exp(+2 pi i j/n).
template <int R, int S>
__device__ __forceinline__ void stockham_pass(const cplx *__restrict__ in, cplx *__restrict__ out, const cplx *__restrict__ tw,
                                              int n, int Ns, int nlines, int es, int ls) {
  const int nb = n / R;             // butterflies per line
  const int tstep = n / (Ns * R);   // twiddle exp(S 2 pi i r k/(Ns R)) = tw[r k tstep]
  for (int w = threadIdx.x; w < nb * nlines; w += blockDim.x) {
    int l = w % nlines, j = w / nlines;
    int k = j % Ns;
    cplx v[R];
    const cplx *src = in + l * ls + j * es;
#pragma unroll
    for (int r = 0; r < R; r++) v[r] = src[r * nb * es];
    if (Ns > 1) {
#pragma unroll
      for (int r = 1; r < R; r++) {
        cplx t = tw[r * k * tstep];
        if (S < 0) t.y = -t.y;
        v[r] = cmul(v[r], t);
      }
    }
    Dft<R, S>::run(v);
    int j0 = (j / Ns) * Ns * R + k;
    cplx *dst = out + l * ls + j0 * es;
#pragma unroll
    for (int r = 0; r < R; r++) dst[r * Ns * es] = v[r];
  }
}

// Full 1-D transform of all lines; ping-pongs between a and b, returns the buffer holding the result.
template <int S>
__device__ __forceinline__ cplx *fft_lines(cplx *a, cplx *b, const cplx *tw, int n, const FacDev &F, int nlines, int es, int ls) {
  int Ns = 1;
  for (int f = 0; f < F.nfac; f++) {
    int R = F.radix[f];
    __syncthreads();
    switch (R) {
      case 2: stockham_pass<2, S>(a, b, tw, n, Ns, nlines, es, ls); break;
      case 3: stockham_pass<3, S>(a, b, tw, n, Ns, nlines, es, ls); break;
      case 4: stockham_pass<4, S>(a, b, tw, n, Ns, nlines, es, ls); break;
      case 5: stockham_pass<5, S>(a, b, tw, n, Ns, nlines, es, ls); break;
      case 8: stockham_pass<8, S>(a, b, tw, n, Ns, nlines, es, ls); break;
      default: stockham_pass<9, S>(a, b, tw, n, Ns, nlines, es, ls); break;
    }
    Ns *= R;
    cplx *t = a; a = b; b = t;
  }
  __syncthreads();
  return a;
}

__device__ __forceinline__ void load_twiddles(cplx *tws, const double *tw, int n) {
  const cplx *g = reinterpret_cast<const cplx *>(tw);
  for (int j = threadIdx.x; j < n; j += blockDim.x) tws[j] = g[j];
}

struct FftGeom {
  int n1, n2, n3, n1p;         // n1p: odd line stride used by the x passes
  int npw, mpw, ncol, nplane;
  int XT, nxt;                 // x-tile width of the strided passes, number of tiles
  int CL;                      // columns per CTA in the x passes
  const int32_t *col_start, *col_i2, *col_plane, *pw_i1, *plane_i3, *plane_col0;
  const double *tw1, *tw2, *tw3;
  FacDev f1, f2, f3;
  int64_t t1_band, t2_band;    // complex elements per band of T1 [ncol][n1] and T2 [nplane][n2][n1]
};

constexpr int FFT_THREADS = 256;

// ---- pass A: scatter + transform along x.  grid (ceil(ncol/CL), nb) -------------------------------
// pre: optional real diagonal factor in G space ([npw], meta-GGA term), applied while scattering
__global__ void __launch_bounds__(FFT_THREADS) fft_pass_a_kernel(FftGeom G, const cplx *__restrict__ psi, cplx *__restrict__ T1,
                                                                 const double *__restrict__ pre) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *tws = reinterpret_cast<cplx *>(smem_raw);
  cplx *bufa = tws + G.n1, *bufb = bufa + G.CL * G.n1p;
  int c0 = blockIdx.x * G.CL, nc = min(G.CL, G.ncol - c0), b = blockIdx.y;
  load_twiddles(tws, G.tw1, G.n1);
  for (int i = threadIdx.x; i < G.CL * G.n1p; i += blockDim.x) bufa[i] = make_double2(0.0, 0.0);
  __syncthreads();
  const cplx *src = psi + (size_t)b * G.mpw;
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
  for (int lc = warp; lc < nc; lc += nwarp) {
    int g0 = G.col_start[c0 + lc], g1 = G.col_start[c0 + lc + 1];
    for (int g = g0 + lane; g < g1; g += 32) {
      cplx v = src[g];
      if (pre) { const double f = pre[g]; v.x *= f; v.y *= f; }
      bufa[lc * G.n1p + G.pw_i1[g]] = v;
    }
  }
  cplx *res = fft_lines<+1>(bufa, bufb, tws, G.n1, G.f1, G.CL, 1, G.n1p);
  cplx *dst = T1 + (size_t)b * G.t1_band + (size_t)c0 * G.n1;
  for (int i = threadIdx.x; i < nc * G.n1; i += blockDim.x) dst[i] = res[(i / G.n1) * G.n1p + (i % G.n1)];
}

// ---- pass A^-1: inverse along x + gather.  grid (ceil(ncol/CL), nb) ---------------------------------
// post: optional real diagonal factor applied while gathering; accumulate: hpsi += result (pad entries untouched)
__global__ void __launch_bounds__(FFT_THREADS) fft_pass_ainv_kernel(FftGeom G, const cplx *__restrict__ T1, cplx *__restrict__ hpsi,
                                                                    const double *__restrict__ post, int accumulate) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *tws = reinterpret_cast<cplx *>(smem_raw);
  cplx *bufa = tws + G.n1, *bufb = bufa + G.CL * G.n1p;
  int c0 = blockIdx.x * G.CL, nc = min(G.CL, G.ncol - c0), b = blockIdx.y;
  load_twiddles(tws, G.tw1, G.n1);
  const cplx *src = T1 + (size_t)b * G.t1_band + (size_t)c0 * G.n1;
  for (int i = threadIdx.x; i < G.CL * G.n1; i += blockDim.x) {
    int lc = i / G.n1, x = i % G.n1;
    bufa[lc * G.n1p + x] = (lc < nc) ? src[i] : make_double2(0.0, 0.0);
  }
  cplx *res = fft_lines<-1>(bufa, bufb, tws, G.n1, G.f1, G.CL, 1, G.n1p);
  cplx *dst = hpsi + (size_t)b * G.mpw;
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
  for (int lc = warp; lc < nc; lc += nwarp) {
    int g0 = G.col_start[c0 + lc], g1 = G.col_start[c0 + lc + 1];
    for (int g = g0 + lane; g < g1; g += 32) {
      cplx v = res[lc * G.n1p + G.pw_i1[g]];
      if (post) { const double f = post[g]; v.x *= f; v.y *= f; }
      if (accumulate) { const cplx h = dst[g]; v.x += h.x; v.y += h.y; }
      dst[g] = v;
    }
  }
  // entries ipw >= npw of the band are defined to be 0 on output
  if (blockIdx.x == gridDim.x - 1 && !accumulate)
    for (int g = G.npw + threadIdx.x; g < G.mpw; g += blockDim.x) dst[g] = make_double2(0.0, 0.0);
}

// ---- pass B: transform along y.  grid (nxt, nplane, nb) -------------------------------------------
template <int S>
__global__ void __launch_bounds__(FFT_THREADS) fft_pass_b_kernel(FftGeom G, cplx *__restrict__ T1, cplx *__restrict__ T2) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *tws = reinterpret_cast<cplx *>(smem_raw);
  cplx *bufa = tws + G.n2, *bufb = bufa + G.n2 * G.XT;
  int x0 = blockIdx.x * G.XT, nx = min(G.XT, G.n1 - x0), p = blockIdx.y, b = blockIdx.z;
  int ca = G.plane_col0[p], cb = G.plane_col0[p + 1];
  load_twiddles(tws, G.tw2, G.n2);
  cplx *t1 = T1 + (size_t)b * G.t1_band;
  cplx *t2 = T2 + (size_t)b * G.t2_band + (size_t)p * G.n2 * G.n1;
  if (S > 0) {
    for (int i = threadIdx.x; i < G.n2 * G.XT; i += blockDim.x) bufa[i] = make_double2(0.0, 0.0);
    __syncthreads();
    for (int i = threadIdx.x; i < (cb - ca) * G.XT; i += blockDim.x) {
      int c = ca + i / G.XT, xt = i % G.XT;
      if (xt < nx) bufa[G.col_i2[c] * G.XT + xt] = t1[(size_t)c * G.n1 + x0 + xt];
    }
  } else {
    for (int i = threadIdx.x; i < G.n2 * G.XT; i += blockDim.x) {
      int y = i / G.XT, xt = i % G.XT;
      bufa[i] = (xt < nx) ? t2[(size_t)y * G.n1 + x0 + xt] : make_double2(0.0, 0.0);
    }
  }
  cplx *res = fft_lines<S>(bufa, bufb, tws, G.n2, G.f2, G.XT, G.XT, 1);
  if (S > 0) {
    for (int i = threadIdx.x; i < G.n2 * G.XT; i += blockDim.x) {
      int y = i / G.XT, xt = i % G.XT;
      if (xt < nx) t2[(size_t)y * G.n1 + x0 + xt] = res[i];
    }
  } else {
    for (int i = threadIdx.x; i < (cb - ca) * G.XT; i += blockDim.x) {
      int c = ca + i / G.XT, xt = i % G.XT;
      if (xt < nx) t1[(size_t)c * G.n1 + x0 + xt] = res[G.col_i2[c] * G.XT + xt];
    }
  }
}

// ---- pass C: along z, times V/N, inverse along z.  grid (nxt, n2, nb) ------------------------------
__global__ void __launch_bounds__(FFT_THREADS) fft_pass_c_kernel(FftGeom G, cplx *__restrict__ T2, const double *__restrict__ vloc) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *tws = reinterpret_cast<cplx *>(smem_raw);
  cplx *bufa = tws + G.n3, *bufb = bufa + G.n3 * G.XT;
  int x0 = blockIdx.x * G.XT, nx = min(G.XT, G.n1 - x0), y = blockIdx.y, b = blockIdx.z;
  load_twiddles(tws, G.tw3, G.n3);
  cplx *t2 = T2 + (size_t)b * G.t2_band + (size_t)y * G.n1 + x0;
  size_t pstride = (size_t)G.n2 * G.n1;
  for (int i = threadIdx.x; i < G.n3 * G.XT; i += blockDim.x) bufa[i] = make_double2(0.0, 0.0);
  __syncthreads();
  for (int i = threadIdx.x; i < G.nplane * G.XT; i += blockDim.x) {
    int p = i / G.XT, xt = i % G.XT;
    if (xt < nx) bufa[G.plane_i3[p] * G.XT + xt] = t2[p * pstride + xt];
  }
  cplx *res = fft_lines<+1>(bufa, bufb, tws, G.n3, G.f3, G.XT, G.XT, 1);
  cplx *other = (res == bufa) ? bufb : bufa;
  const double *v = vloc + (size_t)y * G.n1 + x0;
  for (int i = threadIdx.x; i < G.n3 * G.XT; i += blockDim.x) {
    int z = i / G.XT, xt = i % G.XT;
    double s = (xt < nx) ? v[z * pstride + xt] : 0.0;
    res[i] = make_double2(res[i].x * s, res[i].y * s);
  }
  res = fft_lines<-1>(res, other, tws, G.n3, G.f3, G.XT, G.XT, 1);
  for (int i = threadIdx.x; i < G.nplane * G.XT; i += blockDim.x) {
    int p = i / G.XT, xt = i % G.XT;
    if (xt < nx) t2[p * pstride + xt] = res[G.plane_i3[p] * G.XT + xt];
  }
}

// ---- density on the generic path (Eq. 6, :140): the forward half of pass C, then rho += sum_b w_b |psi_b(r)|^2.
//      grid (nxt, n2); a CTA owns its (x tile, y) lines for ALL bands of the launch, keeps the running sum in shared memory
//      and adds it to rho once: no atomics, fixed summation order (the register path has its own kernel in fft2.cu).
__global__ void __launch_bounds__(FFT_THREADS) fft_density_c_kernel(FftGeom G, const cplx *__restrict__ T2, const double *__restrict__ wgt,
                                                                    double *__restrict__ rho, int nb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx *tws = reinterpret_cast<cplx *>(smem_raw);
  cplx *bufa = tws + G.n3, *bufb = bufa + G.n3 * G.XT;
  double *acc = reinterpret_cast<double *>(bufb + G.n3 * G.XT);
  int x0 = blockIdx.x * G.XT, nx = min(G.XT, G.n1 - x0), y = blockIdx.y;
  load_twiddles(tws, G.tw3, G.n3);
  size_t pstride = (size_t)G.n2 * G.n1;
  for (int i = threadIdx.x; i < G.n3 * G.XT; i += blockDim.x) acc[i] = 0.0;
  for (int b = 0; b < nb; b++) {
    const cplx *t2 = T2 + (size_t)b * G.t2_band + (size_t)y * G.n1 + x0;
    __syncthreads();
    for (int i = threadIdx.x; i < G.n3 * G.XT; i += blockDim.x) bufa[i] = make_double2(0.0, 0.0);
    __syncthreads();
    for (int i = threadIdx.x; i < G.nplane * G.XT; i += blockDim.x) {
      int p = i / G.XT, xt = i % G.XT;
      if (xt < nx) bufa[G.plane_i3[p] * G.XT + xt] = t2[p * pstride + xt];
    }
    cplx *res = fft_lines<+1>(bufa, bufb, tws, G.n3, G.f3, G.XT, G.XT, 1);
    const double w = wgt[b];
    for (int i = threadIdx.x; i < G.n3 * G.XT; i += blockDim.x) acc[i] += w * (res[i].x * res[i].x + res[i].y * res[i].y);
  }
  double *dst = rho + (size_t)y * G.n1 + x0;
  for (int i = threadIdx.x; i < G.n3 * G.XT; i += blockDim.x) {
    int z = i / G.XT, xt = i % G.XT;
    if (xt < nx) dst[z * pstride + xt] += acc[i];
  }
}

__global__ void zero_kernel(double *p, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = 0.0;
}

int zero_fill(double *hpsi, int64_t ndouble, cudaStream_t st) {
  if (ndouble <= 0) return DFT_OK;
  int grid = (int)((ndouble + 255) / 256 < 148 * 8 ? (ndouble + 255) / 256 : 148 * 8);
  zero_kernel<<<grid, 256, 0, st>>>(hpsi, ndouble);
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
static const size_t SMEM_BUDGET = 200 * 1024;

static int choose_xt(int n1, int nmax) {
  int cap = (int)(SMEM_BUDGET / (32 * (size_t)nmax));   // two buffers of n*XT complex
  if (cap < 1) cap = 1;
  int xt = 0;
  for (int d = 16; d <= 40; d += 2)
    if (n1 % d == 0) { xt = d; break; }
  if (!xt) xt = n1 <= 40 ? n1 : 16;
  return xt < cap ? xt : cap;
}
static int choose_cl(int n1p) {
  int cap = (int)(SMEM_BUDGET / (32 * (size_t)n1p));
  return cap < 16 ? (cap < 1 ? 1 : cap) : 16;
}

static FftGeom make_geom(const dft_plan *p, int ik) {
  const KPoint &kp = p->kp[ik];
  FftGeom G;
  G.n1 = p->n[0]; G.n2 = p->n[1]; G.n3 = p->n[2]; G.n1p = G.n1 | 1;
  G.npw = kp.npw; G.mpw = p->mpw; G.ncol = kp.ncol; G.nplane = kp.nplane;
  int nmax = G.n2 > G.n3 ? G.n2 : G.n3;
  G.XT = choose_xt(G.n1, nmax); G.nxt = (G.n1 + G.XT - 1) / G.XT;
  G.CL = choose_cl(G.n1p);
  G.col_start = kp.col_start; G.col_i2 = kp.col_i2; G.col_plane = kp.col_plane; G.pw_i1 = kp.pw_i1;
  G.plane_i3 = kp.plane_i3; G.plane_col0 = kp.plane_col0;
  G.tw1 = p->d_tw[0]; G.tw2 = p->d_tw[1]; G.tw3 = p->d_tw[2];
  const FftFactors *f[3] = {&p->fac[0], &p->fac[1], &p->fac[2]};
  FacDev *d[3] = {&G.f1, &G.f2, &G.f3};
  for (int c = 0; c < 3; c++) {
    d[c]->nfac = f[c]->nfac;
    for (int i = 0; i < 12; i++) d[c]->radix[i] = f[c]->radix[i];
  }
  G.t1_band = (int64_t)kp.ncol * G.n1;
  G.t2_band = (int64_t)kp.nplane * G.n2 * G.n1;
  return G;
}

// scratch per band: T1 [ncol][n1] + T2 [nplane][n2][n1] complex (max over k-points), 256-byte rounded
int64_t fft_ws_bytes_per_band(const dft_plan *p) {
  int64_t mx = 0;
  for (int ik = 0; ik < p->nkpt; ik++) {
    const KPoint &kp = p->kp[ik];
    int64_t t1 = ((int64_t)kp.ncol * p->n[0] * 16 + 255) / 256 * 256;
    int64_t t2 = ((int64_t)kp.nplane * p->n[1] * p->n[0] * 16 + 255) / 256 * 256;
    if (t1 + t2 > mx) mx = t1 + t2;
  }
  return mx;
}

// scratch per band of the all-k-points-per-launch path (fft2_apply_batched): T1 [nkpt][nb][max_k t1] then T2 [nkpt][nb][max_k t2],
// i.e. the two maxima taken SEPARATELY (the k-point with most columns need not be the one with most planes)
int64_t fft_ws_bytes_per_band_batched(const dft_plan *p) {
  int64_t m1 = 0, m2 = 0;
  for (int ik = 0; ik < p->nkpt; ik++) {
    const KPoint &kp = p->kp[ik];
    int64_t t1 = ((int64_t)kp.ncol * p->n[0] * 16 + 255) / 256 * 256;
    int64_t t2 = ((int64_t)kp.nplane * p->n[1] * p->n[0] * 16 + 255) / 256 * 256;
    if (t1 > m1) m1 = t1;
    if (t2 > m2) m2 = t2;
  }
  return (m1 + m2) * p->nkpt;
}

static int set_attrs() {
  // set unconditionally (cheap): a per-process flag would miss a plan on a second device
  int mx = (int)(SMEM_BUDGET + 24 * 1024);
  DFT_CUDA_CHECK(cudaFuncSetAttribute(fft_pass_a_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
  DFT_CUDA_CHECK(cudaFuncSetAttribute(fft_pass_ainv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
  DFT_CUDA_CHECK(cudaFuncSetAttribute(fft_pass_b_kernel<+1>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
  DFT_CUDA_CHECK(cudaFuncSetAttribute(fft_pass_b_kernel<-1>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
  DFT_CUDA_CHECK(cudaFuncSetAttribute(fft_pass_c_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, mx));
  return DFT_OK;
}

int fft_apply_vloc(dft_plan *p, int ik, const double *psi, double *hpsi, int nb, void *ws, cudaStream_t st,
                   const FftExtra *extra) {
  int rc = set_attrs();
  if (rc) return rc;
  const KPoint &kp = p->kp[ik];
  if (kp.npw == 0 || nb == 0) return (extra && extra->accumulate) ? DFT_OK : zero_fill(hpsi, (int64_t)nb * p->mpw * 2, st);
  FftGeom G = make_geom(p, ik);
  int64_t t1b = ((int64_t)G.t1_band * 16 + 255) / 256 * 256;
  cplx *T1 = reinterpret_cast<cplx *>(ws);
  cplx *T2 = reinterpret_cast<cplx *>(reinterpret_cast<char *>(ws) + t1b * nb);
  // T1 is addressed with the rounded per-band stride
  G.t1_band = t1b / 16;
  G.t2_band = (((int64_t)G.t2_band * 16 + 255) / 256 * 256) / 16;
  const cplx *cpsi = reinterpret_cast<const cplx *>(psi);
  cplx *chpsi = reinterpret_cast<cplx *>(hpsi);
  size_t sm_a = sizeof(cplx) * ((size_t)G.n1 + 2 * (size_t)G.CL * G.n1p);
  size_t sm_b = sizeof(cplx) * ((size_t)G.n2 + 2 * (size_t)G.n2 * G.XT);
  size_t sm_c = sizeof(cplx) * ((size_t)G.n3 + 2 * (size_t)G.n3 * G.XT);
  dim3 ga((G.ncol + G.CL - 1) / G.CL, nb), gb(G.nxt, G.nplane, nb), gc(G.nxt, G.n2, nb);
  // per pass: the register-resident two-stage kernel (fft2.cu) when the axis length factorises into two
  // codelet radices and the sphere's occupied sets are runs; otherwise the generic Stockham kernel
  bool fast[3];
  for (int c = 0; c < 3; c++) fast[c] = p->fft_path != 1 && kp.runs_ok && fft2_pair(p->n[c], nullptr, nullptr);
  const double *vpot = (extra && extra->vpot) ? extra->vpot : p->d_vloc;
  if (extra && extra->vspin && !(fast[0] && fast[1] && fast[2])) {
    set_error("the fused spinor pass needs box lengths with a two-radix factorisation (register FFT path)");
    return DFT_ERR_UNSUPPORTED;
  }
  const int axis_of[5] = {0, 1, 2, 1, 0};
  for (int pass = 0; pass < 5; pass++) {
    phase_begin(p, pass, st);
    if (fast[axis_of[pass]]) {
      if ((rc = fft2_launch(p, ik, pass, psi, hpsi, T1, T2, G.t1_band, G.t2_band, nb, st, extra))) return rc;
    } else if (pass == 0) fft_pass_a_kernel<<<ga, FFT_THREADS, sm_a, st>>>(G, cpsi, T1, extra ? extra->pre : nullptr);
    else if (pass == 1) fft_pass_b_kernel<+1><<<gb, FFT_THREADS, sm_b, st>>>(G, T1, T2);
    else if (pass == 2) fft_pass_c_kernel<<<gc, FFT_THREADS, sm_c, st>>>(G, T2, vpot);
    else if (pass == 3) fft_pass_b_kernel<-1><<<gb, FFT_THREADS, sm_b, st>>>(G, T1, T2);
    else fft_pass_ainv_kernel<<<ga, FFT_THREADS, sm_a, st>>>(G, T1, chpsi, extra ? extra->post : nullptr, extra ? extra->accumulate : 0);
    phase_end(p, pass, st, 1);
  }
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

// rho(r) += sum_b wgt[b] |psi_b(r)|^2 for nb bands of k-point ik on ANY box the plan accepts: passes A and B as in
// fft_apply_vloc (register kernels where the axis length has a two-radix factorisation, generic ones elsewhere), then the
// generic density kernel.  fft2_density (register path, faster) is preferred by the caller where all three axes have it.
int fft_density_generic(dft_plan *p, int ik, const double *psi, const double *wgt_dev, double *rho, int nb, void *ws, cudaStream_t st,
                        const double *pre) {
  int rc = set_attrs();
  if (rc) return rc;
  const KPoint &kp = p->kp[ik];
  if (kp.npw == 0 || nb == 0) return DFT_OK;
  FftGeom G = make_geom(p, ik);
  int64_t t1b = ((int64_t)G.t1_band * 16 + 255) / 256 * 256;
  cplx *T1 = reinterpret_cast<cplx *>(ws);
  cplx *T2 = reinterpret_cast<cplx *>(reinterpret_cast<char *>(ws) + t1b * nb);
  G.t1_band = t1b / 16;
  G.t2_band = (((int64_t)G.t2_band * 16 + 255) / 256 * 256) / 16;
  const cplx *cpsi = reinterpret_cast<const cplx *>(psi);
  size_t sm_a = sizeof(cplx) * ((size_t)G.n1 + 2 * (size_t)G.CL * G.n1p);
  size_t sm_b = sizeof(cplx) * ((size_t)G.n2 + 2 * (size_t)G.n2 * G.XT);
  size_t sm_d = sizeof(cplx) * ((size_t)G.n3 + 2 * (size_t)G.n3 * G.XT) + sizeof(double) * (size_t)G.n3 * G.XT;
  dim3 ga((G.ncol + G.CL - 1) / G.CL, nb), gb(G.nxt, G.nplane, nb), gd(G.nxt, G.n2);
  FftExtra X;
  X.pre = pre;
  for (int pass = 0; pass < 2; pass++) {
    phase_begin(p, pass, st);
    const bool fast = p->fft_path != 1 && kp.runs_ok && fft2_pair(p->n[pass], nullptr, nullptr);
    if (fast) {
      if ((rc = fft2_launch(p, ik, pass, psi, nullptr, T1, T2, G.t1_band, G.t2_band, nb, st, &X))) return rc;
    } else if (pass == 0) fft_pass_a_kernel<<<ga, FFT_THREADS, sm_a, st>>>(G, cpsi, T1, pre);
    else fft_pass_b_kernel<+1><<<gb, FFT_THREADS, sm_b, st>>>(G, T1, T2);
    phase_end(p, pass, st, 1);
  }
  if (sm_d > 48 * 1024) DFT_CUDA_CHECK(cudaFuncSetAttribute(fft_density_c_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_d));
  phase_begin(p, 2, st);
  fft_density_c_kernel<<<gd, FFT_THREADS, sm_d, st>>>(G, T2, wgt_dev, rho, nb);
  phase_end(p, 2, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

}  // namespace dftb200
