// sphere.cu -- K1: the G-sphere index builder (readings 1-3).
//
//   S_k = { m in Z^3 : kin(m) <= ecut },  kin(m) = 2 pi^2 (k+m)^T gmet (k+m) = 1/2|k+G|^2  (Hartree)
//
// The paper only says "plane-wave basis sets" with a "cutoff energy" (PAPER.md :46, :489); the
// criterion (inclusive <=) is BASELINE.json's.  The plane waves are listed in ascending FFT-box
// index idx = i1 + n1*(i2 + n2*i3), i_j = m_j mod n_j, which makes the list unique and the
// sphere<->box maps monotone.  Bit-exactness rule (reading 1): t_c = k_c + (double)m_c;
// s = (t1 t1) g11 + (t2 t2) g22 + (t3 t3) g33 + 2((t1 t2) g12) + 2((t1 t3) g13) + 2((t2 t3) g23),
// summed left to right, every product and sum rounded separately (no FMA); kin = (2 pi^2) * s.
#include <math.h>
#include <stdio.h>

#include "internal.h"

namespace dftb200 {

// Reading 1: Bm = (A^-1)^T by cofactors (rows b_i, a_i . b_j = delta_ij, no 2 pi), gmet = Bm Bm^T.
// Operation order is part of the rule: cofactor c_ij = x*y - z*w as written, det = (a11 c11 +
// a12 c12) + a13 c13, bm = c/det, gmet_ij = (b_i1 b_j1 + b_i2 b_j2) + b_i3 b_j3.  Compiled with
// -ffp-contract=off on the host.
void lattice_algebra(const double *a, double *bm, double *gmet, double *det_out) {
  double c[9];
  c[0] = a[4] * a[8] - a[5] * a[7];
  c[1] = a[5] * a[6] - a[3] * a[8];
  c[2] = a[3] * a[7] - a[4] * a[6];
  c[3] = a[2] * a[7] - a[1] * a[8];
  c[4] = a[0] * a[8] - a[2] * a[6];
  c[5] = a[1] * a[6] - a[0] * a[7];
  c[6] = a[1] * a[5] - a[2] * a[4];
  c[7] = a[2] * a[3] - a[0] * a[5];
  c[8] = a[0] * a[4] - a[1] * a[3];
  double det = (a[0] * c[0] + a[1] * c[1]) + a[2] * c[2];
  *det_out = det;
  for (int i = 0; i < 9; i++) bm[i] = c[i] / det;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++)
      gmet[3 * i + j] = (bm[3 * i] * bm[3 * j] + bm[3 * i + 1] * bm[3 * j + 1]) + bm[3 * i + 2] * bm[3 * j + 2];
}

struct SphereParams {
  double g11, g22, g33, g12, g13, g23;
  double k1, k2, k3;
  double ecut;
  int n1, n2, n3;
};

// 2 pi^2 rounded to nearest double (19.739208802178716)
#define DFT_TWO_PI_SQ 0x1.3bd3cc9be45dep+4

__device__ __forceinline__ double kin_of(const SphereParams &P, int m1, int m2, int m3) {
  double t1 = __dadd_rn(P.k1, (double)m1), t2 = __dadd_rn(P.k2, (double)m2), t3 = __dadd_rn(P.k3, (double)m3);
  double s = __dmul_rn(__dmul_rn(t1, t1), P.g11);
  s = __dadd_rn(s, __dmul_rn(__dmul_rn(t2, t2), P.g22));
  s = __dadd_rn(s, __dmul_rn(__dmul_rn(t3, t3), P.g33));
  s = __dadd_rn(s, __dmul_rn(2.0, __dmul_rn(__dmul_rn(t1, t2), P.g12)));
  s = __dadd_rn(s, __dmul_rn(2.0, __dmul_rn(__dmul_rn(t1, t3), P.g13)));
  s = __dadd_rn(s, __dmul_rn(2.0, __dmul_rn(__dmul_rn(t2, t3), P.g23)));
  return __dmul_rn(DFT_TWO_PI_SQ, s);
}

// reading 3: i <= floor((n-1)/2) -> m = i, else m = i - n  (Nyquist index n/2 maps to -n/2)
__device__ __forceinline__ int unwrap_index(int i, int n) { return (i <= (n - 1) / 2) ? i : i - n; }

constexpr int SPH_THREADS = 1024;

// pass 1: number of sphere points in each block of SPH_THREADS consecutive box indices
__global__ void __launch_bounds__(SPH_THREADS) sphere_count_kernel(SphereParams P, int64_t nbox, int32_t *blk_count) {
  int64_t idx = (int64_t)blockIdx.x * SPH_THREADS + threadIdx.x;
  int in = 0;
  if (idx < nbox) {
    int i1 = (int)(idx % P.n1), i2 = (int)((idx / P.n1) % P.n2), i3 = (int)(idx / ((int64_t)P.n1 * P.n2));
    double e = kin_of(P, unwrap_index(i1, P.n1), unwrap_index(i2, P.n2), unwrap_index(i3, P.n3));
    in = (e <= P.ecut);
  }
  int tot = __syncthreads_count(in);
  if (threadIdx.x == 0) blk_count[blockIdx.x] = tot;
}

// pass 2: ordered compaction (ascending box index) given the exclusive scan of the block counts
__global__ void __launch_bounds__(SPH_THREADS) sphere_fill_kernel(SphereParams P, int64_t nbox, const int32_t *blk_off,
                                                                  int32_t *kg, int32_t *igfft, double *kin) {
  __shared__ int warp_tot[SPH_THREADS / 32];
  int64_t idx = (int64_t)blockIdx.x * SPH_THREADS + threadIdx.x;
  int in = 0, m1 = 0, m2 = 0, m3 = 0;
  double e = 0.0;
  if (idx < nbox) {
    int i1 = (int)(idx % P.n1), i2 = (int)((idx / P.n1) % P.n2), i3 = (int)(idx / ((int64_t)P.n1 * P.n2));
    m1 = unwrap_index(i1, P.n1); m2 = unwrap_index(i2, P.n2); m3 = unwrap_index(i3, P.n3);
    e = kin_of(P, m1, m2, m3);
    in = (e <= P.ecut);
  }
  unsigned bal = __ballot_sync(0xffffffffu, in);
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) warp_tot[w] = __popc(bal);
  __syncthreads();
  int before = 0;
  for (int i = 0; i < w; i++) before += warp_tot[i];
  if (in) {
    int pos = blk_off[blockIdx.x] + before + __popc(bal & ((1u << lane) - 1u));
    kg[3 * pos] = m1; kg[3 * pos + 1] = m2; kg[3 * pos + 2] = m3;
    igfft[pos] = (int32_t)idx;
    kin[pos] = e;
  }
}

// extents of the true sphere over the integer cube |m_j| <= bound_j (for DFT_ERR_GRID_TOO_SMALL)
__global__ void sphere_extent_kernel(SphereParams P, int b1, int b2, int b3, int *ext /* min[3], max[3] */) {
  int64_t tot = (int64_t)(2 * b1 + 1) * (2 * b2 + 1) * (2 * b3 + 1);
  int mn[3] = {INT_MAX, INT_MAX, INT_MAX}, mx[3] = {INT_MIN, INT_MIN, INT_MIN};
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < tot; t += (int64_t)gridDim.x * blockDim.x) {
    int m1 = (int)(t % (2 * b1 + 1)) - b1, m2 = (int)((t / (2 * b1 + 1)) % (2 * b2 + 1)) - b2;
    int m3 = (int)(t / ((int64_t)(2 * b1 + 1) * (2 * b2 + 1))) - b3;
    if (kin_of(P, m1, m2, m3) <= P.ecut) {
      mn[0] = min(mn[0], m1); mx[0] = max(mx[0], m1);
      mn[1] = min(mn[1], m2); mx[1] = max(mx[1], m2);
      mn[2] = min(mn[2], m3); mx[2] = max(mx[2], m3);
    }
  }
  for (int j = 0; j < 3; j++) {
    if (mn[j] != INT_MAX) atomicMin(&ext[j], mn[j]);
    if (mx[j] != INT_MIN) atomicMax(&ext[3 + j], mx[j]);
  }
}

static SphereParams make_params(const double *gmet, const double *k, double ecut, const int n[3]) {
  SphereParams P;
  P.g11 = gmet[0]; P.g22 = gmet[4]; P.g33 = gmet[8]; P.g12 = gmet[1]; P.g13 = gmet[2]; P.g23 = gmet[5];
  P.k1 = k[0]; P.k2 = k[1]; P.k3 = k[2]; P.ecut = ecut;
  P.n1 = n ? n[0] : 1; P.n2 = n ? n[1] : 1; P.n3 = n ? n[2] : 1;
  return P;
}

int sphere_extent(const double *gmet, const double *k, double ecut, const int bound[3], int mmin[3], int mmax[3]) {
  SphereParams P = make_params(gmet, k, ecut, nullptr);
  int *d_ext = nullptr;
  DFT_CUDA_CHECK(cudaMalloc(&d_ext, 6 * sizeof(int)));
  int init[6] = {INT_MAX, INT_MAX, INT_MAX, INT_MIN, INT_MIN, INT_MIN};
  cudaMemcpy(d_ext, init, sizeof(init), cudaMemcpyHostToDevice);
  int64_t tot = (int64_t)(2 * bound[0] + 1) * (2 * bound[1] + 1) * (2 * bound[2] + 1);
  int grid = (int)((tot + 255) / 256 < 148 * 16 ? (tot + 255) / 256 : 148 * 16);
  sphere_extent_kernel<<<grid, 256>>>(P, bound[0], bound[1], bound[2], d_ext);
  int h[6];
  cudaError_t e = cudaMemcpy(h, d_ext, sizeof(h), cudaMemcpyDeviceToHost);
  cudaFree(d_ext);
  DFT_CUDA_CHECK(e);
  DFT_CUDA_CHECK(cudaGetLastError());
  for (int j = 0; j < 3; j++) { mmin[j] = h[j]; mmax[j] = h[3 + j]; }
  return DFT_OK;
}

template <typename T>
static int upload(T **dst, const std::vector<T> &src) {
  size_t bytes = (src.size() ? src.size() : 1) * sizeof(T);
  DFT_CUDA_CHECK(cudaMalloc((void **)dst, bytes));
  if (!src.empty()) DFT_CUDA_CHECK(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
  return DFT_OK;
}

int sphere_build(const double *gmet, const int n[3], double ecut, KPoint *kp) {
  SphereParams P = make_params(gmet, kp->k, ecut, n);
  int64_t nbox = (int64_t)n[0] * n[1] * n[2];
  int nblk = (int)((nbox + SPH_THREADS - 1) / SPH_THREADS);
  int32_t *d_cnt = nullptr;
  DFT_CUDA_CHECK(cudaMalloc(&d_cnt, sizeof(int32_t) * nblk));
  sphere_count_kernel<<<nblk, SPH_THREADS>>>(P, nbox, d_cnt);
  std::vector<int32_t> cnt(nblk);
  cudaError_t e = cudaMemcpy(cnt.data(), d_cnt, sizeof(int32_t) * nblk, cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) { cudaFree(d_cnt); DFT_CUDA_CHECK(e); }
  int64_t tot = 0;
  for (int i = 0; i < nblk; i++) { int c = cnt[i]; cnt[i] = (int32_t)tot; tot += c; }
  if (tot > INT32_MAX / 4) { cudaFree(d_cnt); set_error("sphere too large (%lld plane waves)", (long long)tot); return DFT_ERR_UNSUPPORTED; }
  kp->npw = (int)tot;
  cudaMemcpy(d_cnt, cnt.data(), sizeof(int32_t) * nblk, cudaMemcpyHostToDevice);
  size_t np = tot ? (size_t)tot : 1;
  DFT_CUDA_CHECK(cudaMalloc(&kp->kg, np * 3 * sizeof(int32_t)));
  DFT_CUDA_CHECK(cudaMalloc(&kp->igfft, np * sizeof(int32_t)));
  DFT_CUDA_CHECK(cudaMalloc(&kp->kin, np * sizeof(double)));
  sphere_fill_kernel<<<nblk, SPH_THREADS>>>(P, nbox, d_cnt, kp->kg, kp->igfft, kp->kin);
  kp->h_kg.resize(3 * (size_t)tot); kp->h_igfft.resize(tot); kp->h_kin.resize(tot);
  if (tot) {
    cudaMemcpy(kp->h_kg.data(), kp->kg, 3 * tot * sizeof(int32_t), cudaMemcpyDeviceToHost);
    cudaMemcpy(kp->h_igfft.data(), kp->igfft, tot * sizeof(int32_t), cudaMemcpyDeviceToHost);
    cudaMemcpy(kp->h_kin.data(), kp->kin, tot * sizeof(double), cudaMemcpyDeviceToHost);
  }
  cudaFree(d_cnt);
  DFT_CUDA_CHECK(cudaDeviceSynchronize());
  DFT_CUDA_CHECK(cudaGetLastError());

  // ---- pruned-FFT geometry (host, O(npw)): columns are maximal runs of equal (i2,i3) in the list
  std::vector<int32_t> col_start, col_i2, col_plane, pw_i1(tot), plane_i3, plane_col0;
  int n1 = n[0], n2 = n[1];
  int last_col = -1, last_i3 = -1;
  for (int64_t g = 0; g < tot; g++) {
    int idx = kp->h_igfft[g];
    int i1 = idx % n1, i2 = (idx / n1) % n2, i3 = idx / (n1 * n2);
    pw_i1[g] = i1;
    int colid = i2 + n2 * i3;
    if (colid != last_col) {
      if (i3 != last_i3) { plane_i3.push_back(i3); plane_col0.push_back((int32_t)col_start.size()); last_i3 = i3; }
      col_start.push_back((int32_t)g); col_i2.push_back(i2); col_plane.push_back((int32_t)plane_i3.size() - 1);
      last_col = colid;
    }
  }
  kp->ncol = (int)col_start.size();
  kp->nplane = (int)plane_i3.size();
  col_start.push_back((int32_t)tot);
  plane_col0.push_back(kp->ncol);
  // the same geometry as runs of consecutive box indices
  auto make_run = [](const int32_t *idx, int cnt, int base, Run *r) -> bool {
    r->base = base; r->lo = cnt ? idx[0] : 0; r->nlo = 0; r->hi = 0; r->nhi = 0; r->aux0 = r->aux1 = r->pad = 0;
    int i = 0;
    while (i < cnt && idx[i] == r->lo + i) i++;
    r->nlo = i;
    if (i < cnt) {
      r->hi = idx[i];
      int j = i;
      while (j < cnt && idx[j] == r->hi + (j - i)) j++;
      r->nhi = j - i;
      if (j < cnt) return false;
    }
    return true;
  };
  std::vector<Run> col_run(kp->ncol), plane_run(kp->nplane);
  bool runs_ok = true;
  for (int c = 0; c < kp->ncol; c++) {
    runs_ok &= make_run(pw_i1.data() + col_start[c], col_start[c + 1] - col_start[c], col_start[c], &col_run[c]);
    col_run[c].aux0 = col_i2[c]; col_run[c].aux1 = col_plane[c];
  }
  for (int p = 0; p < kp->nplane; p++) {
    runs_ok &= make_run(col_i2.data() + plane_col0[p], plane_col0[p + 1] - plane_col0[p], plane_col0[p], &plane_run[p]);
    plane_run[p].aux0 = plane_i3[p];
  }
  runs_ok &= make_run(plane_i3.data(), kp->nplane, 0, &kp->zrun);
  kp->runs_ok = runs_ok;
  kp->max_cols_per_plane = 0;
  for (int p = 0; p < kp->nplane; p++)
    if (plane_col0[p + 1] - plane_col0[p] > kp->max_cols_per_plane) kp->max_cols_per_plane = plane_col0[p + 1] - plane_col0[p];
  int rc;
  if ((rc = upload(&kp->col_run, col_run))) return rc;
  if ((rc = upload(&kp->plane_run, plane_run))) return rc;
  if ((rc = upload(&kp->col_start, col_start))) return rc;
  if ((rc = upload(&kp->col_i2, col_i2))) return rc;
  if ((rc = upload(&kp->col_plane, col_plane))) return rc;
  if ((rc = upload(&kp->pw_i1, pw_i1))) return rc;
  if ((rc = upload(&kp->plane_i3, plane_i3))) return rc;
  if ((rc = upload(&kp->plane_col0, plane_col0))) return rc;
  return DFT_OK;
}

}  // namespace dftb200
