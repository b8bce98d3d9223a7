// plan.cu -- the C ABI of include/dft.h: plan construction, setters, and dft_apply_h, which enqueues
//
//   fft_A(scatter) -> fft_B -> fft_C.V.C^-1 -> fft_B^-1 -> fft_A^-1(gather)      (fft.cu,  V_loc psi)
//   gemm1 (cprj = P^H psi) -> dij -> gemm2 (+ kinetic epilogue, accumulates)     (nonlocal.cu)
//
// on the caller's stream without any host synchronisation (PAPER.md :438 "minimize host-device and
// device-host transfers"; :456 the operation itself).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "internal.h"

namespace dftb200 {

static thread_local char g_err[512] = "";
void set_error(const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

void phase_begin(dft_plan *p, int phase, cudaStream_t st) {
  if (!p->timer.on) return;
  cudaEvent_t a, b;
  auto &pool = p->timer.pool;   // events are reused: dft_plan_phase_ms hands them back
  if (pool.size() >= 2) { a = pool.back(); pool.pop_back(); b = pool.back(); pool.pop_back(); }
  else { cudaEventCreate(&a); cudaEventCreate(&b); }
  cudaEventRecord(a, st);
  p->timer.ev[phase].push_back({a, b});
}
void phase_end(dft_plan *p, int phase, cudaStream_t st, int launches) {
  p->last_launches += launches;
  if (!p->timer.on) return;
  cudaEventRecord(p->timer.ev[phase].back().second, st);
  p->timer.launches[phase] += launches;
}

template <typename T>
static int to_device(T **dst, const T *src, size_t count) {
  DFT_CUDA_CHECK(cudaMalloc((void **)dst, (count ? count : 1) * sizeof(T)));
  if (count) DFT_CUDA_CHECK(cudaMemcpy(*dst, src, count * sizeof(T), cudaMemcpyHostToDevice));
  return DFT_OK;
}

__global__ void scale_copy_kernel(const double *__restrict__ src, double *__restrict__ dst, int64_t n, double s) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) dst[i] = src[i] * s;
}

static void free_kpoint(KPoint &k) {
  cudaFree(k.kg); cudaFree(k.igfft); cudaFree(k.kin); cudaFree(k.col_start); cudaFree(k.col_i2); cudaFree(k.col_plane);
  cudaFree(k.pw_i1); cudaFree(k.plane_i3); cudaFree(k.plane_col0); cudaFree(k.col_run); cudaFree(k.plane_run);
}

static void destroy_plan(dft_plan *p) {
  if (!p) return;
  for (auto &k : p->kp) free_kpoint(k);
  cudaFree(p->d_f); cudaFree(p->d_f2); cudaFree(p->d_typat); cudaFree(p->d_nlmn); cudaFree(p->d_lmn_l); cudaFree(p->d_lmn_m);
  cudaFree(p->d_lmn_irad); cudaFree(p->d_atom_first); cudaFree(p->d_nq); cudaFree(p->d_dq); cudaFree(p->d_xred);
  cudaFree(p->d_blk_atom); cudaFree(p->d_blk_frow); cudaFree(p->d_blk_first); cudaFree(p->d_blk_nl);
  cudaFree(p->d_stab); cudaFree(p->d_fytab); cudaFree(p->d_vtau); cudaFree(p->d_qcart); cudaFree(p->d_qhalf); cudaFree(p->d_wgt); cudaFree(p->d_geom2); cudaFree(p->d_geom_small); cudaFree(p->d_dstmap); cudaFree(p->d_kina); cudaFree((void *)p->d_kinaptr); cudaFree(p->d_dij); cudaFree(p->d_sij); cudaFree(p->d_ones); cudaFree((void *)p->d_oneptr); cudaFree(p->d_ptab); cudaFree(p->d_npw); cudaFree((void *)p->d_kinptr); cudaFree(p->d_vloc);
  for (int c = 0; c < 3; c++) cudaFree(p->d_tw[c]);
  cudaFree(p->ws_own); cudaFree(p->d_part); cudaFree(p->d_cprj); cudaFree(p->d_stage_in); cudaFree(p->d_stage_out);
  gamma_free(p);
  nl_maps_free(p);
  cudaFree(p->d_symx);
  cudaFree(p->d_vpauli); cudaFree(p->d_dspin); cudaFree(p->d_spin_tmp);
  if (p->host_stream) cudaStreamDestroy(p->host_stream);
  if (p->h2d_stream) cudaStreamDestroy(p->h2d_stream);
  if (p->d2h_stream) cudaStreamDestroy(p->d2h_stream);
  for (int ph = 0; ph < NPHASE; ph++)
    for (auto &e : p->timer.ev[ph]) { cudaEventDestroy(e.first); cudaEventDestroy(e.second); }
  for (cudaEvent_t e : p->timer.pool) cudaEventDestroy(e);
  cudaGetLastError();
  delete p;
}

static int create_impl(dft_plan *p, const double rprimd[9], int32_t nkpt, const double *kpt, double ecut, const int32_t ngfft[3],
                       int32_t natom, const int32_t *typat, const double *xred, int32_t ntypat, const dft_proj_table *tables,
                       const double *dij) {
  int dev_count = 0;
  if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0) {
    cudaGetLastError();
    set_error("no CUDA device available (this library has no CPU path)");
    return DFT_ERR_CUDA;
  }
  int dev = 0;
  DFT_CUDA_CHECK(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  DFT_CUDA_CHECK(cudaGetDeviceProperties(&prop, dev));
  if (prop.major < 10) { set_error("device %s is sm_%d%d; this library is built for sm_100a only", prop.name, prop.major, prop.minor); return DFT_ERR_CUDA; }
  p->sm_count = prop.multiProcessorCount;
  p->smem_per_sm = (int)prop.sharedMemPerMultiprocessor;
  p->smem_optin = (int)prop.sharedMemPerBlockOptin;

  // ---- lattice (reading 1)
  for (int i = 0; i < 9; i++) {
    if (!isfinite(rprimd[i])) { set_error("rprimd has a non-finite entry"); return DFT_ERR_INVALID_ARG; }
    p->rprimd[i] = rprimd[i];
  }
  double det;
  lattice_algebra(p->rprimd, p->bm, p->gmet, &det);
  if (!(fabs(det) > 0.0) || !isfinite(det)) { set_error("lattice vectors are coplanar (det = %g)", det); return DFT_ERR_INVALID_ARG; }
  p->ecut = ecut;
  for (int c = 0; c < 3; c++) {
    p->n[c] = ngfft[c];
    if (ngfft[c] < 1 || ngfft[c] > 1024) { set_error("ngfft[%d] = %d outside 1..1024", c, ngfft[c]); return DFT_ERR_INVALID_ARG; }
    if (!factorize(ngfft[c], &p->fac[c])) { set_error("ngfft[%d] = %d has a prime factor > 5", c, ngfft[c]); return DFT_ERR_UNSUPPORTED; }
  }
  p->nbox = (int64_t)p->n[0] * p->n[1] * p->n[2];
  if (p->nbox >= ((int64_t)1 << 31)) { set_error("FFT box too large"); return DFT_ERR_UNSUPPORTED; }

  // ---- atoms / projector metadata
  p->natom = natom; p->ntypat = natom > 0 ? ntypat : 0;
  p->lmax = 0; p->nrad_max = 0; p->nq_max = 0;
  for (int t = 0; t < p->ntypat; t++) {
    const dft_proj_table &T = tables[t];
    if (T.nlmn < 0 || T.nlmn > 16) { set_error("type %d: nlmn = %d outside 0..16", t, T.nlmn); return DFT_ERR_INVALID_ARG; }
    if (T.nlmn > 0 && (!T.l || !T.m || !T.irad || !T.f || !T.f2 || T.nrad < 1 || T.nq < 2 || !(T.dq > 0.0))) {
      set_error("type %d: incomplete projector table", t); return DFT_ERR_INVALID_ARG;
    }
    for (int i = 0; i < T.nlmn; i++) {
      if (T.l[i] < 0 || T.l[i] > 2) { set_error("type %d projector %d: l = %d unsupported (0..2)", t, i, T.l[i]); return DFT_ERR_UNSUPPORTED; }
      if (T.m[i] < -T.l[i] || T.m[i] > T.l[i]) { set_error("type %d projector %d: m = %d outside -l..l", t, i, T.m[i]); return DFT_ERR_INVALID_ARG; }
      if (T.irad[i] < 0 || T.irad[i] >= T.nrad) { set_error("type %d projector %d: irad = %d outside 0..nrad-1", t, i, T.irad[i]); return DFT_ERR_INVALID_ARG; }
    }
    if (T.nlmn > p->lmax) p->lmax = T.nlmn;
    if (T.nlmn > 0) { if (T.nrad > p->nrad_max) p->nrad_max = T.nrad; if (T.nq > p->nq_max) p->nq_max = T.nq; }
  }
  p->typat.assign(typat, typat + natom);
  p->xred.assign(xred, xred + 3 * (size_t)natom);
  p->nlmn.resize(p->ntypat); p->nq.resize(p->ntypat); p->dq.resize(p->ntypat);
  size_t lm = (size_t)p->ntypat * (p->lmax ? p->lmax : 1);
  p->lmn_l.assign(lm, 0); p->lmn_m.assign(lm, 0); p->lmn_irad.assign(lm, 0);
  std::vector<double> hf((size_t)p->ntypat * p->nrad_max * p->nq_max, 0.0), hf2(hf.size(), 0.0);
  for (int t = 0; t < p->ntypat; t++) {
    const dft_proj_table &T = tables[t];
    p->nlmn[t] = T.nlmn; p->nq[t] = T.nlmn ? T.nq : 2; p->dq[t] = T.nlmn ? T.dq : 1e300;
    for (int i = 0; i < T.nlmn; i++) { p->lmn_l[t * p->lmax + i] = T.l[i]; p->lmn_m[t * p->lmax + i] = T.m[i]; p->lmn_irad[t * p->lmax + i] = T.irad[i]; }
    if (T.nlmn)
      for (int r = 0; r < T.nrad; r++)
        for (int j = 0; j < T.nq; j++) {
          hf[((size_t)t * p->nrad_max + r) * p->nq_max + j] = T.f[(size_t)r * T.nq + j];
          hf2[((size_t)t * p->nrad_max + r) * p->nq_max + j] = T.f2[(size_t)r * T.nq + j];
        }
  }
  p->atom_first.resize(natom + 1);
  p->nproj = 0;
  for (int a = 0; a < natom; a++) {
    if (typat[a] < 0 || typat[a] >= ntypat) { set_error("typat[%d] = %d outside 0..ntypat-1", a, typat[a]); return DFT_ERR_INVALID_ARG; }
    for (int c = 0; c < 3; c++) if (!isfinite(xred[3 * a + c])) { set_error("xred of atom %d is not finite", a); return DFT_ERR_INVALID_ARG; }
    p->atom_first[a] = p->nproj; p->nproj += p->nlmn[typat[a]];
  }
  p->atom_first[natom] = p->nproj;
  if (natom > 65535) { set_error("natom > 65535 unsupported"); return DFT_ERR_UNSUPPORTED; }

  // ---- K1: spheres
  p->nkpt = nkpt;
  p->kp.resize(nkpt);
  p->mpw = 0;
  const double TWO_PI = 6.283185307179586;
  for (int ik = 0; ik < nkpt; ik++) {
    KPoint &K = p->kp[ik];
    for (int c = 0; c < 3; c++) {
      K.k[c] = kpt[3 * ik + c];
      if (!isfinite(K.k[c])) { set_error("k-point %d is not finite", ik); return DFT_ERR_INVALID_ARG; }
    }
    // |(k+m)_j| = |a_j . q|/(2 pi) <= |a_j| sqrt(2 ecut)/(2 pi): integer cube that surely contains the sphere
    int bound[3], mmin[3], mmax[3];
    for (int j = 0; j < 3; j++) {
      const double *a = p->rprimd + 3 * j;
      double len = sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
      double b = ceil(len * sqrt(2.0 * ecut) / TWO_PI + fabs(K.k[j])) + 1.0;
      if (!(b < 4096.0)) { set_error("sphere extent along axis %d is too large", j); return DFT_ERR_UNSUPPORTED; }
      bound[j] = (int)b;
    }
    int rc = sphere_extent(p->gmet, K.k, ecut, bound, mmin, mmax);
    if (rc) return rc;
    for (int j = 0; j < 3; j++)
      if (mmin[j] <= mmax[j] && (mmin[j] < -(p->n[j] / 2) || mmax[j] > (p->n[j] - 1) / 2)) {
        set_error("k-point %d: sphere spans m_%d in [%d, %d], FFT box n = %d holds [%d, %d]", ik, j + 1, mmin[j], mmax[j], p->n[j],
                  -(p->n[j] / 2), (p->n[j] - 1) / 2);
        return DFT_ERR_GRID_TOO_SMALL;
      }
    rc = sphere_build(p->gmet, p->n, ecut, &K);
    if (rc) return rc;
    if (K.npw > p->mpw) p->mpw = K.npw;
  }
  {
    std::vector<int32_t> npw(nkpt);
    std::vector<const double *> kin(nkpt);
    for (int ik = 0; ik < nkpt; ik++) { npw[ik] = p->kp[ik].npw; kin[ik] = p->kp[ik].kin; }
    int rc;
    if ((rc = to_device(&p->d_npw, npw.data(), nkpt))) return rc;
    if ((rc = to_device((const double ***)&p->d_kinptr, kin.data(), nkpt))) return rc;
  }

  // ---- device copies of the atom data, D_ij, projector table (S1)
  int rc;
  if ((rc = to_device(&p->d_typat, p->typat.data(), natom))) return rc;
  if ((rc = to_device(&p->d_nlmn, p->nlmn.data(), p->ntypat))) return rc;
  if ((rc = to_device(&p->d_lmn_l, p->lmn_l.data(), p->lmn_l.size()))) return rc;
  if ((rc = to_device(&p->d_lmn_m, p->lmn_m.data(), p->lmn_m.size()))) return rc;
  if ((rc = to_device(&p->d_lmn_irad, p->lmn_irad.data(), p->lmn_irad.size()))) return rc;
  if ((rc = to_device(&p->d_atom_first, p->atom_first.data(), p->atom_first.size()))) return rc;
  if ((rc = to_device(&p->d_nq, p->nq.data(), p->ntypat))) return rc;
  if ((rc = to_device(&p->d_dq, p->dq.data(), p->ntypat))) return rc;
  if ((rc = to_device(&p->d_xred, p->xred.data(), p->xred.size()))) return rc;
  if ((rc = to_device(&p->d_f, hf.data(), hf.size()))) return rc;
  if ((rc = to_device(&p->d_f2, hf2.data(), hf2.size()))) return rc;
  size_t ndij = (size_t)natom * p->lmax * p->lmax;
  if (ndij) {
    if (!dij) { set_error("dij is NULL"); return DFT_ERR_INVALID_ARG; }
    if ((rc = to_device(&p->d_dij, dij, ndij))) return rc;
    std::vector<double> zero(ndij, 0.0);
    if ((rc = to_device(&p->d_sij, zero.data(), ndij))) return rc;
  }
  if (p->mpw > 0) {   // unit diagonal of the overlap operator, addressed like the kinetic energies
    std::vector<double> ones((size_t)p->mpw, 1.0);
    if ((rc = to_device(&p->d_ones, ones.data(), ones.size()))) return rc;
    std::vector<const double *> optr((size_t)nkpt, p->d_ones);
    if ((rc = to_device((const double ***)&p->d_oneptr, optr.data(), nkpt))) return rc;
  }
  size_t tab = (size_t)nkpt * p->nproj * p->mpw * 16;
  if (tab && !p->skip_table_at_create) {     // dft_plan_create_opts with proj_mode = 1: the table is never built (19.4 GB at c4)
    if (cudaMalloc(&p->d_ptab, tab + 256) != cudaSuccess) {
      cudaGetLastError();
      set_error("cannot allocate the projector table (%zu bytes)", tab);
      return DFT_ERR_ALLOC;
    }
  }
  for (int ik = 0; ik < nkpt; ik++) {
    double maxq;
    if ((rc = build_projector_table(p, ik, &maxq))) return rc;
  }

  // ---- twiddles exp(+2 pi i j/n) from long double
  for (int c = 0; c < 3; c++) {
    int n = p->n[c];
    std::vector<double> tw(2 * (size_t)n);
    const long double PI_L = 3.14159265358979323846264338327950288L;
    for (int j = 0; j < n; j++) {
      long double ang = 2.0L * PI_L * (long double)j / (long double)n;
      tw[2 * j] = (double)cosl(ang); tw[2 * j + 1] = (double)sinl(ang);
    }
    if ((rc = to_device(&p->d_tw[c], tw.data(), tw.size()))) return rc;
  }
  DFT_CUDA_CHECK(cudaMalloc(&p->d_vloc, sizeof(double) * (size_t)p->nbox));

  // ---- TMA descriptor encoder (driver entry point; no link against libcuda)
  cudaDriverEntryPointQueryResult qres;
  void *fn = nullptr;
  DFT_CUDA_CHECK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
  if (!fn || qres != cudaDriverEntryPointSuccess) { set_error("cuTensorMapEncodeTiled not available in this driver"); return DFT_ERR_CUDA; }
  p->encode_fn = fn;
  DFT_CUDA_CHECK(cudaDeviceSynchronize());
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

static int ensure_workspace(dft_plan *p, int64_t per_band, int nband, int *chunk_out, void **ws_out, cudaStream_t st) {
  int chunk = p->band_chunk > 0 ? p->band_chunk : 0;
  if (p->ws_user) {
    int64_t fit = per_band > 0 ? p->ws_user_bytes / per_band : nband;
    if (fit < 1) { set_error("workspace of %lld bytes is smaller than one band (%lld bytes)", (long long)p->ws_user_bytes, (long long)per_band); return DFT_ERR_ALLOC; }
    if (chunk == 0 || chunk > fit) chunk = (int)(fit < 65535 ? fit : 65535);
    if (chunk > nband) chunk = nband;
    *chunk_out = chunk; *ws_out = p->ws_user;
    return DFT_OK;
  }
  if (chunk == 0) {
    int64_t target = (int64_t)8 << 30;   // about 8 GiB of pass-to-pass scratch (c4: 139 bands per chunk; fewer, longer launches)
    int64_t fit = per_band > 0 ? target / per_band : nband;
    chunk = (int)(fit < 1 ? 1 : (fit > 4096 ? 4096 : fit));
  }
  if (chunk > nband) chunk = nband;
  if (chunk > 65535) chunk = 65535;
  int64_t need = per_band * chunk;
  if (need > p->ws_own_bytes) {
    if (p->ws_own) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->ws_own); p->ws_own = nullptr; p->ws_own_bytes = 0; }
    if (cudaMalloc(&p->ws_own, need) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes of FFT scratch", (long long)need); return DFT_ERR_ALLOC; }
    p->ws_own_bytes = need;
  }
  *chunk_out = chunk; *ws_out = p->ws_own;
  return DFT_OK;
}

static int ensure_qcart_ready(dft_plan *p) {
  if (!p->d_qcart || !p->d_qhalf) { set_error("the k+G arrays of the meta-GGA term are missing"); return DFT_ERR_NOT_READY; }
  return DFT_OK;
}

// hpsi = V_loc psi (extra: another potential, diagonal factors with k-stride 3 mpw, accumulation) for [nkpt][nband][mpw] blocks
int local_term(dft_plan *p, const double *psi, double *hpsi, int nband, cudaStream_t st, const FftExtra *extra) {
  int rc;
  const size_t band_stride = (size_t)p->mpw * 2;
  const bool small = (p->fft_path == 0 || p->fft_path == 3 || p->fft_path == 5) && fft_small_ok(p);
  if (small)   // the box fits one SM's shared memory: the whole local term of all k-points and bands is ONE launch, no scratch
    return fft_small_apply(p, 0, p->nkpt, psi, hpsi, nband, nband, st, extra);
  int chunk; void *ws;
  if (!extra && fft2_batch_ok(p) && (!p->ws_user || p->ws_user_bytes >= fft_ws_bytes_per_band_batched(p))) {
    // small boxes, many k-points: every pass is one launch over all k-points (blockIdx.y = k-point)
    if ((rc = ensure_workspace(p, fft_ws_bytes_per_band_batched(p), nband, &chunk, &ws, st))) return rc;
    for (int b0 = 0; b0 < nband; b0 += chunk) {
      int nb = nband - b0 < chunk ? nband - b0 : chunk;
      if ((rc = fft2_apply_batched(p, psi + (size_t)b0 * band_stride, hpsi + (size_t)b0 * band_stride, nb, nband, ws, st))) return rc;
    }
    return DFT_OK;
  }
  if ((rc = ensure_workspace(p, fft_ws_bytes_per_band(p), nband, &chunk, &ws, st))) return rc;
  if (extra && extra->vspin) {      // rows are (up, down) pairs: a chunk holds whole spinor bands
    chunk &= ~1;
    if (chunk < 2) { set_error("the workspace holds fewer than the two rows of one spinor band"); return DFT_ERR_ALLOC; }
  }
  for (int ik = 0; ik < p->nkpt; ik++)
    for (int b0 = 0; b0 < nband; b0 += chunk) {
      int nb = nband - b0 < chunk ? nband - b0 : chunk;
      size_t off = ((size_t)ik * nband + b0) * band_stride;
      FftExtra X;
      if (extra) {
        X = *extra;
        if (X.pre) X.pre += (size_t)ik * 3 * p->mpw;
        if (X.post) X.post += (size_t)ik * 3 * p->mpw;
      }
      if ((rc = fft_apply_vloc(p, ik, psi + off, hpsi + off, nb, ws, st, extra ? &X : nullptr))) return rc;
    }
  return DFT_OK;
}

static int apply_impl(dft_plan *p, const double *psi, double *hpsi, int32_t nband, cudaStream_t st, const Recurrence *rec = nullptr,
                      double *spsi = nullptr) {
  p->last_launches = 0;
  if (nband == 0 || p->mpw == 0 || p->nkpt == 0) return DFT_OK;
  const bool loc = (p->terms & 2) != 0, kin = (p->terms & 1) != 0, nl = (p->terms & 4) != 0 && p->nproj > 0;
  if (loc && !p->vloc_set) { set_error("dft_apply_h called before dft_set_vloc"); return DFT_ERR_NOT_READY; }
  int rc;
  const size_t band_stride = (size_t)p->mpw * 2;
  const bool small = (p->fft_path == 0 || p->fft_path == 3 || p->fft_path == 5) && fft_small_ok(p);
  if (loc) {
    if ((rc = local_term(p, psi, hpsi, nband, st, nullptr))) return rc;
  } else {
    phase_begin(p, 4, st);
    if ((rc = zero_fill(hpsi, (int64_t)p->nkpt * nband * band_stride, st))) return rc;
    phase_end(p, 4, st, 1);
  }
  if ((p->terms & 8) && p->vtau_set) {
    // meta-GGA term (Eq. 8): hpsi += 1/2 sum_d q_d . FFT^-1[ v_tau(r) FFT[ q_d psi ] ], q = k + G Cartesian;
    // three more local applications with diagonal factors fused into the scatter and gather passes
    int chunk = 0; void *ws = nullptr;
    if (small) {
      if ((rc = ensure_qcart_ready(p))) return rc;
      for (int d = 0; d < 3; d++) {
        FftExtra X;
        X.vpot = p->d_vtau;
        X.pre = p->d_qcart + (size_t)d * p->mpw;      // k-point ik: + ik * 3 * mpw (inside the kernel)
        X.post = p->d_qhalf + (size_t)d * p->mpw;
        X.accumulate = 1;
        if ((rc = fft_small_apply(p, 0, p->nkpt, psi, hpsi, nband, nband, st, &X))) return rc;
      }
    } else if ((rc = ensure_workspace(p, fft_ws_bytes_per_band(p), nband, &chunk, &ws, st))) return rc;
    for (int ik = 0; ik < p->nkpt && !small; ik++)
      for (int b0 = 0; b0 < nband; b0 += chunk) {
        int nb = nband - b0 < chunk ? nband - b0 : chunk;
        size_t off = ((size_t)ik * nband + b0) * band_stride;
        for (int d = 0; d < 3; d++) {
          FftExtra X;
          X.vpot = p->d_vtau;
          X.pre = p->d_qcart + ((size_t)ik * 3 + d) * p->mpw;
          X.post = p->d_qhalf + ((size_t)ik * 3 + d) * p->mpw;
          X.accumulate = 1;
          if ((rc = fft_apply_vloc(p, ik, psi + off, hpsi + off, nb, ws, st, &X))) return rc;
        }
      }
  }
  if (kin || nl || rec || spsi)
    if ((rc = nonlocal_apply(p, psi, hpsi, nband, true, kin, nl, st, nullptr, p->vecpot_on ? p->d_kinaptr : nullptr, nullptr, rec,
                             spsi))) return rc;
  return DFT_OK;
}

}  // namespace dftb200

using namespace dftb200;

#define DFT_GUARD_BEGIN try {
#define DFT_GUARD_END                                          \
  } catch (const std::bad_alloc &) {                           \
    set_error("host allocation failed");                       \
    return DFT_ERR_ALLOC;                                      \
  } catch (...) {                                              \
    set_error("unexpected internal error");                    \
    return DFT_ERR_INVALID_ARG;                                \
  }

extern "C" {

const char *dft_last_error(void) { return g_err; }

int dft_plan_create(dft_plan **out, const double rprimd[9], int32_t nkpt, const double *kpt, double ecut, const int32_t ngfft[3],
                    int32_t natom, const int32_t *typat, const double *xred, int32_t ntypat, const dft_proj_table *tables,
                    const double *dij) {
  DFT_GUARD_BEGIN
  if (!out || !rprimd || !kpt || !ngfft) { set_error("null argument"); return DFT_ERR_INVALID_ARG; }
  if (nkpt < 1) { set_error("nkpt = %d must be >= 1", nkpt); return DFT_ERR_INVALID_ARG; }
  if (!(ecut > 0.0) || !isfinite(ecut)) { set_error("ecut = %g must be positive and finite", ecut); return DFT_ERR_INVALID_ARG; }
  if (natom < 0 || ntypat < 0) { set_error("negative natom/ntypat"); return DFT_ERR_INVALID_ARG; }
  if (natom > 0 && (!typat || !xred || !tables || ntypat < 1)) { set_error("atoms given without typat/xred/tables"); return DFT_ERR_INVALID_ARG; }
  dft_plan *p = new dft_plan();
  int rc = create_impl(p, rprimd, nkpt, kpt, ecut, ngfft, natom, typat, xred, ntypat, tables, dij);
  if (rc != DFT_OK) { destroy_plan(p); return rc; }
  *out = p;
  return DFT_OK;
  DFT_GUARD_END
}

int dft_plan_create_opts(dft_plan **out, const double rprimd[9], int32_t nkpt, const double *kpt, double ecut, const int32_t ngfft[3],
                         int32_t natom, const int32_t *typat, const double *xred, int32_t ntypat, const dft_proj_table *tables,
                         const double *dij, int32_t nopt, const char *const *keys, const int64_t *values) {
  DFT_GUARD_BEGIN
  if (!out || !rprimd || !kpt || !ngfft) { set_error("null argument"); return DFT_ERR_INVALID_ARG; }
  if (nkpt < 1) { set_error("nkpt = %d must be >= 1", nkpt); return DFT_ERR_INVALID_ARG; }
  if (!(ecut > 0.0) || !isfinite(ecut)) { set_error("ecut = %g must be positive and finite", ecut); return DFT_ERR_INVALID_ARG; }
  if (natom < 0 || ntypat < 0) { set_error("negative natom/ntypat"); return DFT_ERR_INVALID_ARG; }
  if (natom > 0 && (!typat || !xred || !tables || ntypat < 1)) { set_error("atoms given without typat/xred/tables"); return DFT_ERR_INVALID_ARG; }
  if (nopt < 0 || (nopt > 0 && (!keys || !values))) { set_error("nopt = %d without keys/values", nopt); return DFT_ERR_INVALID_ARG; }
  for (int i = 0; i < nopt; i++) if (!keys[i]) { set_error("option %d has a null key", i); return DFT_ERR_INVALID_ARG; }
  dft_plan *p = new dft_plan();
  // the last value given for proj_mode decides whether the materialised table is built at all
  for (int i = 0; i < nopt; i++) if (!strcmp(keys[i], "proj_mode")) p->skip_table_at_create = (values[i] == 1);
  int rc = create_impl(p, rprimd, nkpt, kpt, ecut, ngfft, natom, typat, xred, ntypat, tables, dij);
  for (int i = 0; i < nopt && rc == DFT_OK; i++) rc = dft_plan_set_option(p, keys[i], values[i]);
  if (rc != DFT_OK) { destroy_plan(p); return rc; }
  *out = p;
  return DFT_OK;
  DFT_GUARD_END
}

int dft_plan_get_info(const dft_plan *p, int32_t *nkpt, int32_t *npw, int32_t *mpw, int32_t *nproj, int64_t *ws_per_band) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nkpt) *nkpt = p->nkpt;
  if (npw) for (int ik = 0; ik < p->nkpt; ik++) npw[ik] = p->kp[ik].npw;
  if (mpw) *mpw = p->mpw;
  if (nproj) *nproj = p->nproj;
  if (ws_per_band) *ws_per_band = fft_ws_bytes_per_band(p);
  return DFT_OK;
}

int dft_plan_get_kg(const dft_plan *p, int32_t ik, int32_t *kg, int32_t *igfft, double *kin) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (ik < 0 || ik >= p->nkpt) { set_error("ik = %d outside 0..%d", ik, p->nkpt - 1); return DFT_ERR_INVALID_ARG; }
  const KPoint &K = p->kp[ik];
  if (kg && K.npw) memcpy(kg, K.h_kg.data(), sizeof(int32_t) * 3 * (size_t)K.npw);
  if (igfft && K.npw) memcpy(igfft, K.h_igfft.data(), sizeof(int32_t) * (size_t)K.npw);
  if (kin && K.npw) memcpy(kin, K.h_kin.data(), sizeof(double) * (size_t)K.npw);
  return DFT_OK;
}

int dft_plan_get_projectors(const dft_plan *p, int32_t ik, double *ptab) {
  if (!p || !ptab) { set_error("null argument"); return DFT_ERR_INVALID_ARG; }
  if (ik < 0 || ik >= p->nkpt) { set_error("ik = %d outside 0..%d", ik, p->nkpt - 1); return DFT_ERR_INVALID_ARG; }
  int npw = p->kp[ik].npw;
  if (p->nproj == 0 || npw == 0) return DFT_OK;
  if (!p->d_ptab) { set_error("the projector table is not materialised while proj_mode = 1"); return DFT_ERR_NOT_READY; }
  const double *src = p->d_ptab + (size_t)ik * p->nproj * p->mpw * 2;
  DFT_CUDA_CHECK(cudaMemcpy2D(ptab, (size_t)npw * 16, src, (size_t)p->mpw * 16, (size_t)npw * 16, p->nproj, cudaMemcpyDeviceToHost));
  return DFT_OK;
}

int dft_plan_copy_projectors_device(const dft_plan *p, int32_t ik, double *ptab_dev, void *stream) {
  if (!p || !ptab_dev) { set_error("null argument"); return DFT_ERR_INVALID_ARG; }
  if (ik < 0 || ik >= p->nkpt) { set_error("ik = %d outside 0..%d", ik, p->nkpt - 1); return DFT_ERR_INVALID_ARG; }
  if (p->nproj == 0 || p->mpw == 0) return DFT_OK;
  if (!p->d_ptab) { set_error("the projector table is not materialised while proj_mode = 1"); return DFT_ERR_NOT_READY; }
  const double *src = p->d_ptab + (size_t)ik * p->nproj * p->mpw * 2;
  DFT_CUDA_CHECK(cudaMemcpyAsync(ptab_dev, src, (size_t)p->nproj * p->mpw * 16, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return DFT_OK;
}

int dft_set_dij(dft_plan *p, const double *dij) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  size_t n = (size_t)p->natom * p->lmax * p->lmax;
  if (n == 0) return DFT_OK;
  if (!dij) { set_error("dij is NULL"); return DFT_ERR_INVALID_ARG; }
  if (p->gamma_on) { int rcg = gamma_check_dij(p, dij); if (rcg) return rcg; }
  // an apply enqueued earlier on a non-blocking stream may still read D_ij: wait for the device before replacing it
  DFT_CUDA_CHECK(cudaDeviceSynchronize());
  DFT_CUDA_CHECK(cudaMemcpy(p->d_dij, dij, n * sizeof(double), cudaMemcpyHostToDevice));
  return DFT_OK;
}

int dft_set_vloc(dft_plan *p, const double *V_r, void *stream) {
  if (!p || !V_r) { set_error("null argument"); return DFT_ERR_INVALID_ARG; }
  cudaStream_t st = (cudaStream_t)stream;
  int64_t n = p->nbox;
  int grid = (int)((n + 255) / 256 < 148 * 8 ? (n + 255) / 256 : 148 * 8);
  scale_copy_kernel<<<grid, 256, 0, st>>>(V_r, p->d_vloc, n, 1.0 / (double)n);
  DFT_CUDA_CHECK(cudaGetLastError());
  p->vloc_set = true;
  return DFT_OK;
}

}  // extern "C"
namespace dftb200 {
// Cartesian q = 2 pi (k + m) Bm per plane wave: out[d][g] = q_d, half[d][g] = q_d / 2 (rows mpw apart)
__global__ void qcart_kernel(const int32_t *__restrict__ kg, int npw, int mpw, double k1, double k2, double k3,
                             const double *__restrict__ bm9, double *__restrict__ out, double *__restrict__ half) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= npw) return;
  const double twopi = 6.283185307179586476925286766559;
  double t1 = k1 + (double)kg[3 * g], t2 = k2 + (double)kg[3 * g + 1], t3 = k3 + (double)kg[3 * g + 2];
  for (int d = 0; d < 3; d++) {
    double q = twopi * (t1 * bm9[d] + t2 * bm9[3 + d] + t3 * bm9[6 + d]);
    out[(size_t)d * mpw + g] = q; half[(size_t)d * mpw + g] = 0.5 * q;
  }
}
}  // namespace dftb200
extern "C" {

static int ensure_qcart(dft_plan *p) {
  if (!p->d_qcart && p->mpw > 0) {
    size_t cnt = (size_t)p->nkpt * 3 * p->mpw;
    if (cudaMalloc(&p->d_qcart, sizeof(double) * cnt) != cudaSuccess || cudaMalloc(&p->d_qhalf, sizeof(double) * cnt) != cudaSuccess) {
      cudaGetLastError(); set_error("cannot allocate the k+G arrays"); return DFT_ERR_ALLOC;
    }
    DFT_CUDA_CHECK(cudaMemset(p->d_qcart, 0, sizeof(double) * cnt));
    DFT_CUDA_CHECK(cudaMemset(p->d_qhalf, 0, sizeof(double) * cnt));
    double *d_bm = nullptr;
    int rc;
    if ((rc = to_device(&d_bm, p->bm, 9))) return rc;
    for (int ik = 0; ik < p->nkpt; ik++) {
      const KPoint &K = p->kp[ik];
      if (K.npw == 0) continue;
      qcart_kernel<<<(K.npw + 255) / 256, 256>>>(K.kg, K.npw, p->mpw, K.k[0], K.k[1], K.k[2], d_bm,
                                                p->d_qcart + (size_t)ik * 3 * p->mpw, p->d_qhalf + (size_t)ik * 3 * p->mpw);
    }
    cudaError_t e = cudaDeviceSynchronize();
    cudaFree(d_bm);
    if (e != cudaSuccess) { set_error("qcart_kernel failed: %s", cudaGetErrorString(e)); return DFT_ERR_CUDA; }
  }
  return DFT_OK;
}

int dft_set_vtau(dft_plan *p, const double *vtau_r, void *stream) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (!vtau_r) { p->vtau_set = false; return DFT_OK; }
  cudaStream_t st = (cudaStream_t)stream;
  int64_t n = p->nbox;
  if (!p->d_vtau && cudaMalloc(&p->d_vtau, sizeof(double) * n) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate v_tau"); return DFT_ERR_ALLOC; }
  { int rcq = ensure_qcart(p); if (rcq) return rcq; }
  int grid = (int)((n + 255) / 256 < 148 * 8 ? (n + 255) / 256 : 148 * 8);
  scale_copy_kernel<<<grid, 256, 0, st>>>(vtau_r, p->d_vtau, n, 1.0 / (double)n);
  DFT_CUDA_CHECK(cudaGetLastError());
  p->vtau_set = true;
  return DFT_OK;
  DFT_GUARD_END
}

int dft_set_workspace(dft_plan *p, void *dev_ptr, int64_t bytes) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (dev_ptr && (bytes <= 0 || ((uintptr_t)dev_ptr & 255))) { set_error("workspace must be 256-byte aligned with bytes > 0"); return DFT_ERR_INVALID_ARG; }
  if (dev_ptr && bytes < fft_ws_bytes_per_band(p)) { set_error("workspace smaller than one band (%lld bytes needed)", (long long)fft_ws_bytes_per_band(p)); return DFT_ERR_ALLOC; }
  p->ws_user = dev_ptr; p->ws_user_bytes = dev_ptr ? bytes : 0;
  return DFT_OK;
}

int dft_plan_workspace_bytes(const dft_plan *p, int32_t nband, int64_t *min_bytes, int64_t *full_bytes) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  if (min_bytes) *min_bytes = fft_ws_bytes_per_band(p);
  if (full_bytes) *full_bytes = (fft2_batch_ok(p) ? fft_ws_bytes_per_band_batched(p) : fft_ws_bytes_per_band(p)) * (int64_t)nband;
  return DFT_OK;
}

int dft_plan_set_option(dft_plan *p, const char *key, int64_t value) {
  if (!p || !key) { set_error("null argument"); return DFT_ERR_INVALID_ARG; }
  if (!strcmp(key, "band_chunk")) {
    if (value < 0 || value > 65535) { set_error("band_chunk = %lld outside 0..65535", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->band_chunk = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "terms")) {
    if (value < 0 || value > 15) { set_error("terms = %lld outside 0..15", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->terms = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "fft_path")) {
    if (value < 0 || value > 5) { set_error("fft_path = %lld outside 0..5", (long long)value); return DFT_ERR_INVALID_ARG; }
    if ((value == 3 || value == 5) && !fft_small_ok(p)) { set_error("fft_path = 3: the fused small-box kernel cannot serve this plan (box lengths or shared memory)"); return DFT_ERR_UNSUPPORTED; }
    p->fft_path = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "fft_c_split")) {
    if (value < 0 || value > 2) { set_error("fft_c_split = %lld outside 0..2", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->fft_c_split = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "gemm2_merge")) {
    if (value < 0 || value > 1) { set_error("gemm2_merge = %lld outside 0..1", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->gemm2_merge = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "nl_tiny")) {
    if (value < 0 || value > 1) { set_error("nl_tiny = %lld outside 0..1", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->nl_tiny = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "spinor_fused")) {
    if (value < 0 || value > 1) { set_error("spinor_fused = %lld outside 0..1", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->spinor_fused = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "proj_mode")) {
    if (value < 0 || value > 1) { set_error("proj_mode = %lld outside 0..1", (long long)value); return DFT_ERR_INVALID_ARG; }
    if (value == 1 && p->nproj > 0) {
      if (!p->d_stab || !p->d_fytab) {
        int rc = build_factor_tables(p);
        if (rc) return rc;
      }
      // the materialised table is not needed in this mode: give its memory back (19.4 GB at c4)
      DFT_CUDA_CHECK(cudaDeviceSynchronize());
      cudaFree(p->d_ptab); p->d_ptab = nullptr;
    }
    if (value == 0 && p->nproj > 0 && p->mpw > 0 && !p->d_ptab) {
      size_t tab = (size_t)p->nkpt * p->nproj * p->mpw * 16;
      if (cudaMalloc(&p->d_ptab, tab + 256) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the projector table (%zu bytes)", tab); return DFT_ERR_ALLOC; }
      for (int ik = 0; ik < p->nkpt; ik++) {
        double maxq;
        int rc = build_projector_table(p, ik, &maxq);
        if (rc) return rc;
      }
      DFT_CUDA_CHECK(cudaDeviceSynchronize());
    }
    p->proj_mode = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "gamma_real")) {
    if (value < 0 || value > 1) { set_error("gamma_real = %lld outside 0..1", (long long)value); return DFT_ERR_INVALID_ARG; }
    if (value == 1) {
      int rcg = gamma_build(p, true);
      if (rcg) return rcg;
      p->gamma_on = true;
      return DFT_OK;
    }
    p->gamma_on = false;     // the tables stay: the symmetric-table GEMMs of dft_apply_h use them too
    return DFT_OK;
  }
  if (!strcmp(key, "gemm_strassen")) {
    if (value < 0 || value > 2) { set_error("gemm_strassen = %lld outside 0..2", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->gemm_strassen = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "gemm_sym")) {
    if (value < 0 || value > 2) { set_error("gemm_sym = %lld outside 0..2", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->gemm_sym = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "host_groups")) {
    if (value < 1 || value > 64) { set_error("host_groups = %lld outside 1..64", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->host_groups = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "gemm_3m")) {
    if (value < 0 || value > 1) { set_error("gemm_3m = %lld outside 0..1", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->gemm_3m = (int)value; return DFT_OK;
  }
  if (!strcmp(key, "splitk")) {
    if (value < 0 || value > 4096) { set_error("splitk = %lld outside 0..4096", (long long)value); return DFT_ERR_INVALID_ARG; }
    p->splitk = (int)value; return DFT_OK;
  }
  set_error("unknown option '%s'", key);
  return DFT_ERR_INVALID_ARG;
}

int dft_apply_h(dft_plan *p, const double *psi, double *hpsi, int32_t nband, void *stream) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  if (nband > 0 && p->mpw > 0 && (!psi || !hpsi)) { set_error("null psi/hpsi"); return DFT_ERR_INVALID_ARG; }
  if (((uintptr_t)psi & 15) || ((uintptr_t)hpsi & 15)) { set_error("psi/hpsi must be 16-byte aligned"); return DFT_ERR_INVALID_ARG; }
  return apply_impl(p, psi, hpsi, nband, (cudaStream_t)stream);
  DFT_GUARD_END
}

int dft_plan_get_kg_gamma(const dft_plan *p, int32_t *nhalf, int32_t *kg, int32_t *igfft, double *kin) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (!p->gam || !p->gamma_on) { set_error("Gamma storage is not enabled (dft_plan_set_option gamma_real = 1)"); return DFT_ERR_NOT_READY; }
  const GammaData &G = *p->gam;
  if (nhalf) *nhalf = G.nh;
  if (kg && G.nh) memcpy(kg, G.h_kg.data(), sizeof(int32_t) * 3 * (size_t)G.nh);
  if (igfft && G.nh) memcpy(igfft, G.h_igfft.data(), sizeof(int32_t) * (size_t)G.nh);
  if (kin && G.nh) memcpy(kin, G.h_kin.data(), sizeof(double) * (size_t)G.nh);
  return DFT_OK;
}

int dft_apply_h_gamma(dft_plan *p, const double *psi, double *hpsi, int32_t nband, void *stream) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  if (nband > 0 && p->gam && p->gam->nh > 0 && (!psi || !hpsi)) { set_error("null psi/hpsi"); return DFT_ERR_INVALID_ARG; }
  if (((uintptr_t)psi & 15) || ((uintptr_t)hpsi & 15)) { set_error("psi/hpsi must be 16-byte aligned"); return DFT_ERR_INVALID_ARG; }
  return gamma_apply(p, psi, hpsi, nband, (cudaStream_t)stream);
  DFT_GUARD_END
}

int dft_set_vloc_spinor(dft_plan *p, const double *v4, void *stream) {
  DFT_GUARD_BEGIN
  if (!p || !v4) { set_error("null argument"); return DFT_ERR_INVALID_ARG; }
  return spinor_set_vloc(p, v4, (cudaStream_t)stream);
  DFT_GUARD_END
}

int dft_set_dij_spinor(dft_plan *p, const double *dspin) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (!dspin) { p->dspin_set = false; return DFT_OK; }     // back to the scalar D_ij on both components
  const size_t n = (size_t)p->natom * 4 * p->lmax * p->lmax * 2;
  if (n == 0) return DFT_OK;
  DFT_CUDA_CHECK(cudaDeviceSynchronize());                  // an apply enqueued earlier may still read the old matrix
  if (!p->d_dspin && cudaMalloc(&p->d_dspin, n * sizeof(double)) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the spinor D_ij"); return DFT_ERR_ALLOC; }
  DFT_CUDA_CHECK(cudaMemcpy(p->d_dspin, dspin, n * sizeof(double), cudaMemcpyHostToDevice));
  p->dspin_set = true;
  return DFT_OK;
  DFT_GUARD_END
}

int dft_apply_h_spinor(dft_plan *p, const double *psi, double *hpsi, int32_t nband, void *stream) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  if (nband > 0 && p->mpw > 0 && (!psi || !hpsi)) { set_error("null psi/hpsi"); return DFT_ERR_INVALID_ARG; }
  if (((uintptr_t)psi & 15) || ((uintptr_t)hpsi & 15)) { set_error("psi/hpsi must be 16-byte aligned"); return DFT_ERR_INVALID_ARG; }
  if (2 * (int64_t)nband > 65535 * 2) { set_error("nband too large"); return DFT_ERR_INVALID_ARG; }
  return spinor_apply(p, psi, hpsi, nband, (cudaStream_t)stream);
  DFT_GUARD_END
}

}  // extern "C"
namespace dftb200 {
// 1/2 |k + G + A|^2 for the plane waves of one k-point: q = 2 pi (k + m) Bm (Cartesian), A Cartesian, atomic units
__global__ void kin_vecpot_kernel(const int32_t *__restrict__ kg, int npw, double k1, double k2, double k3, const double *__restrict__ bm9,
                                  double a1, double a2, double a3, double *__restrict__ out) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= npw) return;
  const double twopi = 6.283185307179586476925286766559;
  double t1 = k1 + (double)kg[3 * g], t2 = k2 + (double)kg[3 * g + 1], t3 = k3 + (double)kg[3 * g + 2];
  double q1 = twopi * (t1 * bm9[0] + t2 * bm9[3] + t3 * bm9[6]) + a1;
  double q2 = twopi * (t1 * bm9[1] + t2 * bm9[4] + t3 * bm9[7]) + a2;
  double q3 = twopi * (t1 * bm9[2] + t2 * bm9[5] + t3 * bm9[8]) + a3;
  out[g] = 0.5 * (q1 * q1 + q2 * q2 + q3 * q3);
}
}  // namespace dftb200
extern "C" {

int dft_set_vector_potential(dft_plan *p, const double *a_cart) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (!a_cart || (a_cart[0] == 0.0 && a_cart[1] == 0.0 && a_cart[2] == 0.0)) { p->vecpot_on = false; return DFT_OK; }
  for (int c = 0; c < 3; c++)
    if (!(a_cart[c] == a_cart[c]) || a_cart[c] - a_cart[c] != 0.0) { set_error("vector potential is not finite"); return DFT_ERR_INVALID_ARG; }
  if (p->mpw == 0 || p->nkpt == 0) return DFT_OK;
  int rc;
  if (!p->d_kina) {
    if (cudaMalloc(&p->d_kina, sizeof(double) * (size_t)p->nkpt * p->mpw) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the kinetic array"); return DFT_ERR_ALLOC; }
    std::vector<const double *> ptr(p->nkpt);
    for (int ik = 0; ik < p->nkpt; ik++) ptr[ik] = p->d_kina + (size_t)ik * p->mpw;
    if ((rc = to_device((const double ***)&p->d_kinaptr, ptr.data(), p->nkpt))) return rc;
  }
  double *d_bm = nullptr;
  if ((rc = to_device(&d_bm, p->bm, 9))) return rc;
  DFT_CUDA_CHECK(cudaMemset(p->d_kina, 0, sizeof(double) * (size_t)p->nkpt * p->mpw));
  for (int ik = 0; ik < p->nkpt; ik++) {
    const KPoint &K = p->kp[ik];
    if (K.npw == 0) continue;
    kin_vecpot_kernel<<<(K.npw + 255) / 256, 256>>>(K.kg, K.npw, K.k[0], K.k[1], K.k[2], d_bm, a_cart[0], a_cart[1], a_cart[2],
                                                   p->d_kina + (size_t)ik * p->mpw);
  }
  cudaError_t e = cudaDeviceSynchronize();
  cudaFree(d_bm);
  if (e != cudaSuccess) { set_error("kin_vecpot_kernel failed: %s", cudaGetErrorString(e)); return DFT_ERR_CUDA; }
  p->vecpot_on = true;
  return DFT_OK;
  DFT_GUARD_END
}

}  // extern "C"
// the three-term recurrence around any of the apply functions (full sphere or Gamma storage); n = doubles per psi-sized array
template <typename Apply>
static int chebyshev_impl(dft_plan *p, double *psi, double *work, size_t n, int32_t degree, double center, double halfwidth,
                          cudaStream_t st, Apply apply) {
  // three psi-sized arrays rotate: x = T_{j-1}, y = T_j, w receives T_{j+1} from the GEMM-2 epilogue
  double *buf[3] = {psi, work, work + n};
  int ix = 2, iy = 0, iw = 1;
  int64_t launches = 0;
  for (int j = 0; j < degree; j++) {
    Recurrence rec;
    if (j == 0) { rec.sh = 1.0 / halfwidth; rec.sy = -center / halfwidth; rec.sx = 0.0; rec.xprev = nullptr; }
    else { rec.sh = 2.0 / halfwidth; rec.sy = -2.0 * center / halfwidth; rec.sx = -1.0; rec.xprev = buf[ix]; }
    // T_{j+1} goes to the third array: the FFT passes store V_loc T_j there before the epilogue reads T_{j-1}
    int rc = apply(buf[iy], buf[iw], &rec);
    if (rc) return rc;
    launches += p->last_launches;
    int t = ix; ix = iy; iy = iw; iw = t;
  }
  p->last_launches = launches;
  if (buf[iy] != psi) DFT_CUDA_CHECK(cudaMemcpyAsync(psi, buf[iy], n * sizeof(double), cudaMemcpyDeviceToDevice, st));
  return DFT_OK;
}

static int chebyshev_args(dft_plan *p, const double *psi, const double *work, int32_t nband, int32_t degree, double center, double halfwidth) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0 || degree < 0) { set_error("nband = %d, degree = %d: negative", nband, degree); return DFT_ERR_INVALID_ARG; }
  if (!(halfwidth > 0.0) || !(center == center)) { set_error("halfwidth must be > 0 and center finite"); return DFT_ERR_INVALID_ARG; }
  if (((uintptr_t)psi & 15) || ((uintptr_t)work & 15)) { set_error("psi/work must be 16-byte aligned"); return DFT_ERR_INVALID_ARG; }
  return DFT_OK;
}

extern "C" {

int dft_chebyshev_filter(dft_plan *p, double *psi, double *work, int32_t nband, int32_t degree, double center,
                         double halfwidth, void *stream) {
  DFT_GUARD_BEGIN
  int rc = chebyshev_args(p, psi, work, nband, degree, center, halfwidth);
  if (rc) return rc;
  p->last_launches = 0;
  const size_t n = (size_t)p->nkpt * nband * p->mpw * 2;   // doubles per psi-sized array
  if (n == 0 || degree == 0) return DFT_OK;
  if (!psi || !work) { set_error("null psi/work"); return DFT_ERR_INVALID_ARG; }
  cudaStream_t st = (cudaStream_t)stream;
  return chebyshev_impl(p, psi, work, n, degree, center, halfwidth, st,
                        [&](const double *x, double *y, const Recurrence *rec) { return apply_impl(p, x, y, nband, st, rec); });
  DFT_GUARD_END
}

int dft_chebyshev_filter_gamma(dft_plan *p, double *psi, double *work, int32_t nband, int32_t degree, double center,
                               double halfwidth, void *stream) {
  DFT_GUARD_BEGIN
  int rc = chebyshev_args(p, psi, work, nband, degree, center, halfwidth);
  if (rc) return rc;
  if (!p->gam || !p->gamma_on) { set_error("Gamma storage is not enabled (dft_plan_set_option gamma_real = 1)"); return DFT_ERR_NOT_READY; }
  p->last_launches = 0;
  const size_t n = (size_t)nband * p->gam->nh * 2;
  if (n == 0 || degree == 0) return DFT_OK;
  if (!psi || !work) { set_error("null psi/work"); return DFT_ERR_INVALID_ARG; }
  cudaStream_t st = (cudaStream_t)stream;
  return chebyshev_impl(p, psi, work, n, degree, center, halfwidth, st,
                        [&](const double *x, double *y, const Recurrence *rec) { return gamma_apply(p, x, y, nband, st, rec); });
  DFT_GUARD_END
}

static int accumulate_impl(dft_plan *p, const double *psi, const double *weights, double *rho, int32_t nband, void *stream, bool tau) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  p->last_launches = 0;
  if (nband == 0 || p->mpw == 0 || p->nkpt == 0) return DFT_OK;
  if (!psi || !weights || !rho) { set_error("null psi/weights/rho"); return DFT_ERR_INVALID_ARG; }
  if ((uintptr_t)psi & 15) { set_error("psi must be 16-byte aligned"); return DFT_ERR_INVALID_ARG; }
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t nw = (int64_t)p->nkpt * nband;
  if (nw > p->wgt_count) {
    if (p->d_wgt) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->d_wgt); p->d_wgt = nullptr; p->wgt_count = 0; }
    if (cudaMalloc(&p->d_wgt, sizeof(double) * nw) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the weight array"); return DFT_ERR_ALLOC; }
    p->wgt_count = nw;
  }
  // weights are HOST memory and must be consumed before the call returns: copy on the stream, then wait for it
  std::vector<double> wh(weights, weights + nw);
  if (tau) {   // tau(r) = 1/2 sum w |grad psi|^2: three gradient components, each a density with half the weight
    for (auto &v : wh) v *= 0.5;
    int rcq = ensure_qcart(p);
    if (rcq) return rcq;
  }
  DFT_CUDA_CHECK(cudaMemcpyAsync(p->d_wgt, wh.data(), sizeof(double) * nw, cudaMemcpyHostToDevice, st));
  DFT_CUDA_CHECK(cudaStreamSynchronize(st));
  int chunk; void *ws; int rc;
  if ((rc = ensure_workspace(p, fft_ws_bytes_per_band(p), nband, &chunk, &ws, st))) return rc;
  const size_t band_stride = (size_t)p->mpw * 2;
  for (int ik = 0; ik < p->nkpt; ik++)
    for (int b0 = 0; b0 < nband; b0 += chunk) {
      int nb = nband - b0 < chunk ? nband - b0 : chunk;
      size_t off = ((size_t)ik * nband + b0) * band_stride;
      bool regpath = p->fft_path != 1 && p->kp[ik].runs_ok;
      for (int c = 0; c < 3 && regpath; c++) regpath = fft2_pair(p->n[c], nullptr, nullptr);
      for (int d = 0; d < (tau ? 3 : 1); d++) {
        const double *pre = tau ? p->d_qcart + ((size_t)ik * 3 + d) * p->mpw : nullptr;
        rc = regpath ? fft2_density(p, ik, psi + off, p->d_wgt + (size_t)ik * nband + b0, rho, nb, ws, st, pre)
                     : fft_density_generic(p, ik, psi + off, p->d_wgt + (size_t)ik * nband + b0, rho, nb, ws, st, pre);
        if (rc == DFT_ERR_UNSUPPORTED && regpath)      // e.g. a tile that does not fit the register kernel: the generic passes
          rc = fft_density_generic(p, ik, psi + off, p->d_wgt + (size_t)ik * nband + b0, rho, nb, ws, st, pre);
        if (rc) return rc;
      }
    }
  return DFT_OK;
  DFT_GUARD_END
}

int dft_accumulate_density(dft_plan *p, const double *psi, const double *weights, double *rho, int32_t nband, void *stream) {
  return accumulate_impl(p, psi, weights, rho, nband, stream, false);
}

int dft_accumulate_tau(dft_plan *p, const double *psi, const double *weights, double *tau, int32_t nband, void *stream) {
  return accumulate_impl(p, psi, weights, tau, nband, stream, true);
}

int dft_set_sij(dft_plan *p, const double *sij) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  size_t n = (size_t)p->natom * p->lmax * p->lmax;
  if (n == 0) return DFT_OK;
  if (!sij) { set_error("sij is NULL"); return DFT_ERR_INVALID_ARG; }
  DFT_CUDA_CHECK(cudaDeviceSynchronize());   // see dft_set_dij
  DFT_CUDA_CHECK(cudaMemcpy(p->d_sij, sij, n * sizeof(double), cudaMemcpyHostToDevice));
  return DFT_OK;
}

int dft_apply_s(dft_plan *p, const double *psi, double *spsi, int32_t nband, void *stream) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  if (nband > 0 && p->mpw > 0 && (!psi || !spsi)) { set_error("null psi/spsi"); return DFT_ERR_INVALID_ARG; }
  if (((uintptr_t)psi & 15) || ((uintptr_t)spsi & 15)) { set_error("psi/spsi must be 16-byte aligned"); return DFT_ERR_INVALID_ARG; }
  p->last_launches = 0;
  if (nband == 0 || p->mpw == 0 || p->nkpt == 0) return DFT_OK;
  // S psi = psi + sum_a sum_ij |p_a,i> s^a_ij <p_a,j|psi>: the non-local path with s_ij for D_ij and a unit diagonal
  bool ragged = false;
  for (int ik = 0; ik < p->nkpt; ik++) ragged |= p->kp[ik].npw < p->mpw;
  if (ragged) DFT_CUDA_CHECK(cudaMemsetAsync(spsi, 0, (size_t)p->nkpt * nband * p->mpw * 16, (cudaStream_t)stream));   // pad entries = 0
  return nonlocal_apply(p, psi, spsi, nband, false, true, p->nproj > 0, (cudaStream_t)stream, p->d_sij, p->d_oneptr, nullptr);
  DFT_GUARD_END
}

int dft_apply_hs(dft_plan *p, const double *psi, double *hpsi, double *spsi, int32_t nband, void *stream) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  if (nband > 0 && p->mpw > 0 && (!psi || !hpsi || !spsi)) { set_error("null psi/hpsi/spsi"); return DFT_ERR_INVALID_ARG; }
  if (((uintptr_t)psi & 15) || ((uintptr_t)hpsi & 15) || ((uintptr_t)spsi & 15)) { set_error("psi/hpsi/spsi must be 16-byte aligned"); return DFT_ERR_INVALID_ARG; }
  if (nband > 0 && p->mpw > 0) {
    if ((p->terms & 4) == 0) { set_error("dft_apply_hs needs the non-local term switched on (terms bit 2)"); return DFT_ERR_INVALID_ARG; }
    bool ragged = false;
    for (int ik = 0; ik < p->nkpt; ik++) ragged |= p->kp[ik].npw < p->mpw;
    if (ragged) DFT_CUDA_CHECK(cudaMemsetAsync(spsi, 0, (size_t)p->nkpt * nband * p->mpw * 16, (cudaStream_t)stream));
  }
  return apply_impl(p, psi, hpsi, nband, (cudaStream_t)stream, nullptr, spsi);
  DFT_GUARD_END
}

int dft_get_cprj(dft_plan *p, const double *psi, double *cprj, int32_t nband, void *stream) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  p->last_launches = 0;
  if (nband == 0 || p->mpw == 0 || p->nkpt == 0 || p->nproj == 0) return DFT_OK;
  if (!psi || !cprj) { set_error("null psi/cprj"); return DFT_ERR_INVALID_ARG; }
  if (((uintptr_t)psi & 15) || ((uintptr_t)cprj & 15)) { set_error("psi/cprj must be 16-byte aligned"); return DFT_ERR_INVALID_ARG; }
  return nonlocal_apply(p, psi, nullptr, nband, false, false, true, (cudaStream_t)stream, nullptr, nullptr, cprj);
  DFT_GUARD_END
}

int dft_apply_h_host(dft_plan *p, const double *psi_host, double *hpsi_host, int32_t nband) {
  DFT_GUARD_BEGIN
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  int64_t bytes = (int64_t)p->nkpt * nband * p->mpw * 16;
  if (bytes == 0) return DFT_OK;
  if (!psi_host || !hpsi_host) { set_error("null psi/hpsi"); return DFT_ERR_INVALID_ARG; }
  if (!p->host_stream) DFT_CUDA_CHECK(cudaStreamCreateWithFlags(&p->host_stream, cudaStreamNonBlocking));
  if (bytes > p->stage_bytes) {
    cudaFree(p->d_stage_in); cudaFree(p->d_stage_out); p->d_stage_in = p->d_stage_out = nullptr; p->stage_bytes = 0;
    if (cudaMalloc(&p->d_stage_in, bytes) != cudaSuccess || cudaMalloc(&p->d_stage_out, bytes) != cudaSuccess) {
      cudaGetLastError(); cudaFree(p->d_stage_in); p->d_stage_in = nullptr;
      set_error("cannot allocate 2 x %lld bytes of device staging", (long long)bytes);
      return DFT_ERR_ALLOC;
    }
    p->stage_bytes = bytes;
  }
  cudaStream_t st = p->host_stream;
  // One k-point: the band block is cut into groups that go through the whole path one after the other, so
  // that the host->device copy of group g+1 and the device->host copy of group g-1 overlap the kernels of
  // group g (three streams, events between them).  Several k-points: one copy in, one pass, one copy out.
  int ngroup = 1;
  if (p->nkpt == 1 && p->host_groups > 1 && nband >= 2 * 64) {
    ngroup = p->host_groups;
    if (nband / ngroup < 64) ngroup = nband / 64;
  }
  if (ngroup <= 1) {
    DFT_CUDA_CHECK(cudaMemcpyAsync(p->d_stage_in, psi_host, bytes, cudaMemcpyHostToDevice, st));
    int rc = apply_impl(p, p->d_stage_in, p->d_stage_out, nband, st);
    if (rc) return rc;
    DFT_CUDA_CHECK(cudaMemcpyAsync(hpsi_host, p->d_stage_out, bytes, cudaMemcpyDeviceToHost, st));
    DFT_CUDA_CHECK(cudaStreamSynchronize(st));
    return DFT_OK;
  }
  if (!p->h2d_stream) DFT_CUDA_CHECK(cudaStreamCreateWithFlags(&p->h2d_stream, cudaStreamNonBlocking));
  if (!p->d2h_stream) DFT_CUDA_CHECK(cudaStreamCreateWithFlags(&p->d2h_stream, cudaStreamNonBlocking));
  // group sizes in whole GEMM band tiles of 64.  Only the copy-in of the first group and the copy-out of the last one
  // are exposed, so with enough bands those two groups are one tile each and the rest is split evenly.
  std::vector<int> sizes;
  {
    const int per = ((nband + ngroup - 1) / ngroup + 63) / 64 * 64;
    if (ngroup >= 6 && nband >= 128 * ngroup) {
      // ramp: 64, 128, middle groups in whole pairs of tiles, 128, 64.  A group's host->device copy runs under the kernels
      // of the group before it and its device->host copy under those of the group after it, and 256 bands take longer to
      // copy (22 ms at 55 GB/s at c4) than 64 bands take to compute (20 ms): the second and the second-last group are
      // therefore half as large as the middle ones.
      const int mid = ngroup - 4, rest = nband - 384, permid = ((rest + mid - 1) / mid + 127) / 128 * 128;
      sizes.push_back(64); sizes.push_back(128);
      for (int left = rest; left > 0; left -= permid) sizes.push_back(left < permid ? left : permid);
      sizes.push_back(128); sizes.push_back(64);
    } else if (ngroup >= 4 && nband >= 64 * 2 * ngroup) {
      const int mid = ngroup - 2, rest = nband - 128, permid = ((rest + mid - 1) / mid + 63) / 64 * 64;
      sizes.push_back(64);
      for (int left = rest; left > 0; left -= permid) sizes.push_back(left < permid ? left : permid);
      sizes.push_back(64);
    } else {
      for (int left = nband; left > 0; left -= per) sizes.push_back(left < per ? left : per);
    }
  }
  std::vector<cudaEvent_t> ev;
  int64_t launches = 0;
  int rc = DFT_OK;
  int b0 = 0;
  for (size_t gi = 0; gi < sizes.size() && rc == DFT_OK; b0 += sizes[gi], gi++) {
    const int nb = sizes[gi];
    const size_t off = (size_t)b0 * p->mpw * 2, gbytes = (size_t)nb * p->mpw * 16;
    cudaEvent_t in_done, k_done;
    if (cudaEventCreateWithFlags(&in_done, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&k_done, cudaEventDisableTiming) != cudaSuccess) { set_error("cudaEventCreate failed"); rc = DFT_ERR_CUDA; break; }
    ev.push_back(in_done); ev.push_back(k_done);
    if (cudaMemcpyAsync(p->d_stage_in + off, psi_host + off, gbytes, cudaMemcpyHostToDevice, p->h2d_stream) != cudaSuccess ||
        cudaEventRecord(in_done, p->h2d_stream) != cudaSuccess || cudaStreamWaitEvent(st, in_done, 0) != cudaSuccess) {
      set_error("host->device copy of bands %d.. failed: %s", b0, cudaGetErrorString(cudaGetLastError())); rc = DFT_ERR_CUDA; break;
    }
    if ((rc = apply_impl(p, p->d_stage_in + off, p->d_stage_out + off, nb, st))) break;
    launches += p->last_launches;
    if (cudaEventRecord(k_done, st) != cudaSuccess || cudaStreamWaitEvent(p->d2h_stream, k_done, 0) != cudaSuccess ||
        cudaMemcpyAsync(hpsi_host + off, p->d_stage_out + off, gbytes, cudaMemcpyDeviceToHost, p->d2h_stream) != cudaSuccess) {
      set_error("device->host copy of bands %d.. failed: %s", b0, cudaGetErrorString(cudaGetLastError())); rc = DFT_ERR_CUDA; break;
    }
  }
  cudaError_t e1 = cudaStreamSynchronize(p->h2d_stream), e2 = cudaStreamSynchronize(st), e3 = cudaStreamSynchronize(p->d2h_stream);
  for (cudaEvent_t e : ev) cudaEventDestroy(e);
  p->last_launches = launches;
  if (rc) return rc;
  if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess) { set_error("dft_apply_h_host: stream synchronisation failed"); return DFT_ERR_CUDA; }
  return DFT_OK;
  DFT_GUARD_END
}

int64_t dft_plan_last_launches(const dft_plan *p) { return p ? p->last_launches : 0; }

int dft_plan_set_timing(dft_plan *p, int32_t on) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  p->timer.on = on != 0;
  return DFT_OK;
}

int dft_plan_phase_ms(dft_plan *p, int32_t phase, double *ms, int64_t *launches) {
  if (!p || phase < 0 || phase >= NPHASE) { set_error("bad phase"); return DFT_ERR_INVALID_ARG; }
  double tot = 0.0;
  for (auto &e : p->timer.ev[phase]) {
    DFT_CUDA_CHECK(cudaEventSynchronize(e.second));
    float t = 0.f;
    DFT_CUDA_CHECK(cudaEventElapsedTime(&t, e.first, e.second));
    tot += t;
    p->timer.pool.push_back(e.first); p->timer.pool.push_back(e.second);
  }
  p->timer.ev[phase].clear();
  if (ms) *ms = tot;
  if (launches) *launches = p->timer.launches[phase];
  p->timer.launches[phase] = 0;
  return DFT_OK;
}

int dft_plan_destroy(dft_plan *p) {
  if (!p) return DFT_OK;
  cudaDeviceSynchronize();
  destroy_plan(p);
  return DFT_OK;
}

}  // extern "C"
