// projtab.cu -- S1: materialise the non-local projectors of Eq. 26 (PAPER.md :470) in device memory,
// the "projectors ... computed and stored in memory" variant of :479.
//
//   p_{a,i}(m) = F_{t(a),irad_i}(|q|) . Y_{l_i m_i}(q^) . exp(-2 pi i (k+m).x_a),   q = 2 pi (k+m)^T Bm
//
// Readings: 6 form of the projector, 7 cubic-spline evaluation of the radial
// table, 8 real spherical harmonics without Condon-Shortley sign, m = -l..l, 11 phase argument
// reduced mod 1.  Layout: P[ik][row][mpw] complex128, row = atom_first[a] + i, zero for ipw >= npw_k,
// i.e. K-contiguous for GEMM-1 and M-contiguous for GEMM-2 (nonlocal.cu).
#include <math.h>

#include <vector>

#include "internal.h"

namespace dftb200 {

struct ProjParams {
  double bm[9];
  double k[3];
  int npw, mpw, natom, lmax, nrad_max, nq_max;
  const int32_t *kg;
  const int32_t *typat, *nlmn, *lmn_l, *lmn_m, *lmn_irad, *atom_first, *nq;
  const double *dq, *xred, *f, *f2;
  double *ptab;   // this k-point's [nproj][mpw] complex
  int rot_odd;    // 1: rows of odd l are multiplied by i (Gamma storage, reading 26)
};

// reading 7
__device__ __forceinline__ double spline_eval(int nq, double dq, const double *f, const double *f2, double q) {
  int j = (int)floor(q / dq);
  if (j > nq - 2) j = nq - 2;
  if (j < 0) j = 0;
  double A = ((double)(j + 1) * dq - q) / dq, B = 1.0 - A;
  return A * f[j] + B * f[j + 1] + ((A * A * A - A) * f2[j] + (B * B * B - B) * f2[j + 1]) * (dq * dq) / 6.0;
}

// reading 8: orthonormal real harmonics; (x,y,z) = q vector, qn = |q|.  l > 0 at q = 0 gives 0.
__device__ __forceinline__ double real_ylm(int l, int m, double x, double y, double z, double qn) {
  const double PI = 3.14159265358979323846;
  if (l == 0) return 0.5 / sqrt(PI);
  if (qn == 0.0) return 0.0;
  if (l == 1) {
    double c = sqrt(3.0 / (4.0 * PI));
    double v = (m == -1) ? y : ((m == 0) ? z : x);
    return c * v / qn;
  }
  double q2 = qn * qn;
  double c1 = 0.5 * sqrt(15.0 / PI), c0 = 0.25 * sqrt(5.0 / PI), c2 = 0.25 * sqrt(15.0 / PI);
  switch (m) {
    case -2: return c1 * x * y / q2;
    case -1: return c1 * y * z / q2;
    case 0:  return c0 * (3.0 * z * z - q2) / q2;
    case 1:  return c1 * x * z / q2;
    default: return c2 * (x * x - y * y) / q2;
  }
}

constexpr int PT_THREADS = 128;
constexpr int PT_MAXRAD = 8;

// grid: (ceil(mpw / PT_THREADS), natom); one thread = one plane wave of one atom, writes nlmn rows
__global__ void __launch_bounds__(PT_THREADS) projtab_kernel(ProjParams P) {
  int g = blockIdx.x * PT_THREADS + threadIdx.x;
  int a = blockIdx.y;
  if (g >= P.mpw) return;
  int t = P.typat[a], nl = P.nlmn[t];
  double2 *dst = reinterpret_cast<double2 *>(P.ptab) + (size_t)P.atom_first[a] * P.mpw + g;
  if (g >= P.npw) {
    for (int i = 0; i < nl; i++) dst[(size_t)i * P.mpw] = make_double2(0.0, 0.0);
    return;
  }
  const double TWO_PI = 6.283185307179586;
  double t0 = P.k[0] + (double)P.kg[3 * g], t1 = P.k[1] + (double)P.kg[3 * g + 1], t2 = P.k[2] + (double)P.kg[3 * g + 2];
  double qx = TWO_PI * (t0 * P.bm[0] + t1 * P.bm[3] + t2 * P.bm[6]);
  double qy = TWO_PI * (t0 * P.bm[1] + t1 * P.bm[4] + t2 * P.bm[7]);
  double qz = TWO_PI * (t0 * P.bm[2] + t1 * P.bm[5] + t2 * P.bm[8]);
  double qn = sqrt(qx * qx + qy * qy + qz * qz);
  // reading 11: exp(-2 pi i frac((k+m).x_a))
  const double *x = P.xred + 3 * a;
  double arg = t0 * x[0] + t1 * x[1] + t2 * x[2];
  arg -= floor(arg);
  double sn, cs;
  sincospi(2.0 * arg, &sn, &cs);
  sn = -sn;
  double frad[PT_MAXRAD];
  bool have[PT_MAXRAD];
#pragma unroll
  for (int r = 0; r < PT_MAXRAD; r++) have[r] = false;
  for (int i = 0; i < nl; i++) {
    int ir = P.lmn_irad[t * P.lmax + i];
    double F;
    if (ir < PT_MAXRAD && have[ir]) {
      F = frad[ir];
    } else {
      size_t off = ((size_t)t * P.nrad_max + ir) * P.nq_max;
      F = spline_eval(P.nq[t], P.dq[t], P.f + off, P.f2 + off, qn);
      if (ir < PT_MAXRAD) { frad[ir] = F; have[ir] = true; }
    }
    const int l = P.lmn_l[t * P.lmax + i];
    double fy = F * real_ylm(l, P.lmn_m[t * P.lmax + i], qx, qy, qz, qn);
    dst[(size_t)i * P.mpw] = (P.rot_odd && (l & 1)) ? make_double2(-(fy * sn), fy * cs) : make_double2(fy * cs, fy * sn);
  }
}

int build_projector_table(dft_plan *p, int ik, double *maxq_out) {
  KPoint &kp = p->kp[ik];
  // max |k+G| (host, O(npw)) for the table-range check of the boundary
  double mx = 0.0;
  const double TWO_PI = 6.283185307179586;
  for (int g = 0; g < kp.npw; g++) {
    double t0 = kp.k[0] + kp.h_kg[3 * g], t1 = kp.k[1] + kp.h_kg[3 * g + 1], t2 = kp.k[2] + kp.h_kg[3 * g + 2];
    double q2 = 0.0;
    for (int c = 0; c < 3; c++) {
      double q = TWO_PI * (t0 * p->bm[c] + t1 * p->bm[3 + c] + t2 * p->bm[6 + c]);
      q2 += q * q;
    }
    if (q2 > mx) mx = q2;
  }
  *maxq_out = sqrt(mx);
  if (p->natom == 0 || p->nproj == 0 || p->mpw == 0) return DFT_OK;
  for (int t = 0; t < p->ntypat; t++)
    if (*maxq_out > (p->nq[t] - 1) * p->dq[t]) {
      set_error("k-point %d: max|k+G| = %.6f exceeds the radial table range (nq-1)*dq = %.6f of type %d", ik,
                *maxq_out, (p->nq[t] - 1) * p->dq[t], t);
      return DFT_ERR_TABLE_RANGE;
    }
  if (!p->d_ptab) return DFT_OK;      // plan created in factorised mode: the range check above is all that is needed here
  ProjParams P;
  for (int i = 0; i < 9; i++) P.bm[i] = p->bm[i];
  for (int i = 0; i < 3; i++) P.k[i] = kp.k[i];
  P.npw = kp.npw; P.mpw = p->mpw; P.natom = p->natom; P.lmax = p->lmax; P.nrad_max = p->nrad_max; P.nq_max = p->nq_max;
  P.kg = kp.kg; P.typat = p->d_typat; P.nlmn = p->d_nlmn; P.lmn_l = p->d_lmn_l; P.lmn_m = p->d_lmn_m;
  P.lmn_irad = p->d_lmn_irad; P.atom_first = p->d_atom_first; P.nq = p->d_nq; P.dq = p->d_dq; P.xred = p->d_xred;
  P.f = p->d_f; P.f2 = p->d_f2;
  P.ptab = p->d_ptab + (size_t)ik * p->nproj * p->mpw * 2;
  P.rot_odd = 0;
  dim3 grid((p->mpw + PT_THREADS - 1) / PT_THREADS, p->natom);
  projtab_kernel<<<grid, PT_THREADS>>>(P);
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

// The same table on another plane-wave list (device kg [npw][3]), rows mpw apart, into d_out [nproj][mpw] complex
int build_projector_table_on(dft_plan *p, const int32_t *d_kg, int npw, int mpw, const double k[3], double *d_out, int rot_odd) {
  if (p->natom == 0 || p->nproj == 0 || mpw == 0) return DFT_OK;
  ProjParams P;
  for (int i = 0; i < 9; i++) P.bm[i] = p->bm[i];
  for (int i = 0; i < 3; i++) P.k[i] = k[i];
  P.npw = npw; P.mpw = mpw; P.natom = p->natom; P.lmax = p->lmax; P.nrad_max = p->nrad_max; P.nq_max = p->nq_max;
  P.kg = d_kg; P.typat = p->d_typat; P.nlmn = p->d_nlmn; P.lmn_l = p->d_lmn_l; P.lmn_m = p->d_lmn_m;
  P.lmn_irad = p->d_lmn_irad; P.atom_first = p->d_atom_first; P.nq = p->d_nq; P.dq = p->d_dq; P.xred = p->d_xred;
  P.f = p->d_f; P.f2 = p->d_f2;
  P.ptab = d_out; P.rot_odd = rot_odd;
  projtab_kernel<<<dim3((mpw + PT_THREADS - 1) / PT_THREADS, p->natom), PT_THREADS>>>(P);
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}


// ------------------------------------------------------------------------------------------
// Factorised projectors (PAPER.md :477 "computed on-the-fly"): p_{a,i}(m) = FY_{t(a),i}(m) . S_a(m)
// with FY = F.Y real (one row per projector of an atom TYPE) and S_a(m) = exp(-2 pi i (k+m).x_a) (one row per ATOM).
// The two small tables replace the [nproj][mpw] complex one: S [natom][mpw] complex, FY [ntypat*8][ldf] real
// (whole 8-row blocks per type, rows >= nlmn zero), zero for ipw >= npw_k.  Row r of S belongs to atom srow_atom[r]: the
// atoms in the order of the block list (by type group, see build_factor_tables), so that the 16 blocks of a GEMM-1 tile
// read 16 consecutive S rows whatever the order of the types in typat.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(PT_THREADS) stab_kernel(ProjParams P, double2 *__restrict__ stab, const int32_t *__restrict__ srow_atom) {
  int g = blockIdx.x * PT_THREADS + threadIdx.x, a = srow_atom[blockIdx.y];
  if (g >= P.mpw) return;
  double2 v = make_double2(0.0, 0.0);
  if (g < P.npw) {
    double t0 = P.k[0] + (double)P.kg[3 * g], t1 = P.k[1] + (double)P.kg[3 * g + 1], t2 = P.k[2] + (double)P.kg[3 * g + 2];
    const double *x = P.xred + 3 * a;
    double arg = t0 * x[0] + t1 * x[1] + t2 * x[2];
    arg -= floor(arg);
    double sn, cs;
    sincospi(2.0 * arg, &sn, &cs);
    v = make_double2(cs, -sn);
  }
  stab[(size_t)blockIdx.y * P.mpw + g] = v;
}

__global__ void __launch_bounds__(PT_THREADS) fytab_kernel(ProjParams P, double *__restrict__ fy, int ldf,
                                                           const int32_t *__restrict__ type_row0, const int32_t *__restrict__ type_rows) {
  int g = blockIdx.x * PT_THREADS + threadIdx.x, t = blockIdx.y;
  if (g >= ldf) return;
  int nl = P.nlmn[t];
  const int nrows = type_rows[t];                 // 8 * ceil(nlmn / 8): whole 8-row blocks, rows >= nlmn are zero
  double *dst = fy + (size_t)type_row0[t] * ldf + g;
  if (g >= P.npw) {
    for (int i = 0; i < nrows; i++) dst[(size_t)i * ldf] = 0.0;
    return;
  }
  const double TWO_PI = 6.283185307179586;
  double t0 = P.k[0] + (double)P.kg[3 * g], t1 = P.k[1] + (double)P.kg[3 * g + 1], t2 = P.k[2] + (double)P.kg[3 * g + 2];
  double qx = TWO_PI * (t0 * P.bm[0] + t1 * P.bm[3] + t2 * P.bm[6]);
  double qy = TWO_PI * (t0 * P.bm[1] + t1 * P.bm[4] + t2 * P.bm[7]);
  double qz = TWO_PI * (t0 * P.bm[2] + t1 * P.bm[5] + t2 * P.bm[8]);
  double qn = sqrt(qx * qx + qy * qy + qz * qz);
  for (int i = 0; i < nrows; i++) {
    double v = 0.0;
    if (i < nl) {
      int ir = P.lmn_irad[t * P.lmax + i];
      size_t off = ((size_t)t * P.nrad_max + ir) * P.nq_max;
      double F = spline_eval(P.nq[t], P.dq[t], P.f + off, P.f2 + off, qn);
      v = F * real_ylm(P.lmn_l[t * P.lmax + i], P.lmn_m[t * P.lmax + i], qx, qy, qz, qn);
    }
    dst[(size_t)i * ldf] = v;
  }
}

// Builds (or rebuilds) both tables for every k-point, and the list of projector BLOCKS the factorised GEMMs walk: an atom
// with nlmn projectors contributes ceil(nlmn / 8) blocks of up to 8 rows (M = 8 of the DMMA shape).  The kernels keep the
// FY rows they need in shared memory, at most FAC_MAX_FROWS of them, so the atom types are cut into GROUPS of consecutive
// types whose rows (8 or 16 per type) fit; the block list is ordered by group and both GEMMs run once per group on that
// group's blocks and FY rows (one group for up to 32 rows, e.g. four types of 8 projectors).
template <typename T>
static int upload_vec(T **dst, const std::vector<T> &v) {
  cudaFree(*dst); *dst = nullptr;
  if (v.empty()) return DFT_OK;
  DFT_CUDA_CHECK(cudaMalloc(dst, v.size() * sizeof(T)));
  DFT_CUDA_CHECK(cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
  return DFT_OK;
}

int build_factor_tables(dft_plan *p) {
  if (p->natom == 0 || p->nproj == 0 || p->mpw == 0) return DFT_OK;
  std::vector<int32_t> row0(p->ntypat), rows(p->ntypat);
  std::vector<int> grp(p->ntypat, 0);
  int nfrow = 0;
  p->fac_groups.clear();
  for (int t = 0; t < p->ntypat; t++) {
    row0[t] = nfrow; rows[t] = (p->nlmn[t] + 7) / 8 * 8; nfrow += rows[t];
    if (rows[t] == 0) { grp[t] = -1; continue; }
    if (p->fac_groups.empty() || p->fac_groups.back().nfrow + rows[t] > FAC_MAX_FROWS) {
      FacGroup g; g.frow0 = row0[t]; g.nfrow = 0; g.blk0 = 0; g.nblk = 0;
      p->fac_groups.push_back(g);
    }
    p->fac_groups.back().nfrow += rows[t];
    grp[t] = (int)p->fac_groups.size() - 1;
  }
  std::vector<int32_t> b_atom, b_frow, b_first, b_nl, srow_atom;
  for (size_t g = 0; g < p->fac_groups.size(); g++) {
    FacGroup &G = p->fac_groups[g];
    G.blk0 = (int)b_atom.size();
    for (int a = 0; a < p->natom; a++) {
      int t = p->typat[a], nl = p->nlmn[t];
      if (grp[t] != (int)g) continue;
      const int srow = (int)srow_atom.size();
      srow_atom.push_back(a);
      for (int mb = 0; mb * 8 < nl; mb++) {
        b_atom.push_back(srow); b_frow.push_back(row0[t] - G.frow0 + 8 * mb); b_first.push_back(p->atom_first[a] + 8 * mb);
        b_nl.push_back(nl - 8 * mb < 8 ? nl - 8 * mb : 8);
      }
    }
    G.nblk = (int)b_atom.size() - G.blk0;
  }
  for (int a = 0; a < p->natom; a++)          // atoms without projectors: rows nobody reads, kept so that the table has natom rows
    if (p->nlmn[p->typat[a]] == 0) srow_atom.push_back(a);
  p->nblk = (int)b_atom.size(); p->nfrow = nfrow;
  int rc;
  int32_t *d_row0 = nullptr, *d_rows = nullptr, *d_srow = nullptr;
  if ((rc = upload_vec(&p->d_blk_atom, b_atom)) || (rc = upload_vec(&p->d_blk_frow, b_frow)) ||
      (rc = upload_vec(&p->d_blk_first, b_first)) || (rc = upload_vec(&p->d_blk_nl, b_nl)) ||
      (rc = upload_vec(&d_row0, row0)) || (rc = upload_vec(&d_rows, rows)) || (rc = upload_vec(&d_srow, srow_atom))) return rc;
  p->ldf = (p->mpw + 7) / 8 * 8;
  size_t sbytes = (size_t)p->nkpt * p->natom * p->mpw * 16 + 256, fbytes = (size_t)p->nkpt * nfrow * p->ldf * 8 + 256;
  if (!p->d_stab && cudaMalloc(&p->d_stab, sbytes) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the structure-factor table (%zu bytes)", sbytes); return DFT_ERR_ALLOC; }
  if (!p->d_fytab && cudaMalloc(&p->d_fytab, fbytes) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the form-factor table (%zu bytes)", fbytes); return DFT_ERR_ALLOC; }
  for (int ik = 0; ik < p->nkpt; ik++) {
    KPoint &kp = p->kp[ik];
    ProjParams P;
    for (int i = 0; i < 9; i++) P.bm[i] = p->bm[i];
    for (int i = 0; i < 3; i++) P.k[i] = kp.k[i];
    P.npw = kp.npw; P.mpw = p->mpw; P.natom = p->natom; P.lmax = p->lmax; P.nrad_max = p->nrad_max; P.nq_max = p->nq_max;
    P.kg = kp.kg; P.typat = p->d_typat; P.nlmn = p->d_nlmn; P.lmn_l = p->d_lmn_l; P.lmn_m = p->d_lmn_m;
    P.lmn_irad = p->d_lmn_irad; P.atom_first = p->d_atom_first; P.nq = p->d_nq; P.dq = p->d_dq; P.xred = p->d_xred;
    P.f = p->d_f; P.f2 = p->d_f2; P.ptab = nullptr; P.rot_odd = 0;
    stab_kernel<<<dim3((p->mpw + PT_THREADS - 1) / PT_THREADS, p->natom), PT_THREADS>>>(
        P, reinterpret_cast<double2 *>(p->d_stab) + (size_t)ik * p->natom * p->mpw, d_srow);
    fytab_kernel<<<dim3((p->ldf + PT_THREADS - 1) / PT_THREADS, p->ntypat), PT_THREADS>>>(
        P, p->d_fytab + (size_t)ik * nfrow * p->ldf, p->ldf, d_row0, d_rows);
  }
  cudaError_t e = cudaDeviceSynchronize();
  cudaFree(d_row0); cudaFree(d_rows); cudaFree(d_srow);
  if (e != cudaSuccess) { set_error("factor-table kernels failed: %s", cudaGetErrorString(e)); return DFT_ERR_CUDA; }
  return DFT_OK;
}

}  // namespace dftb200
