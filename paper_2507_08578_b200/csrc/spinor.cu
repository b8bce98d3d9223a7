// spinor.cu -- two-component spinor wave functions (PAPER.md :448 "all types of magnetism":
// non-collinear magnetism, spin-orbit coupling; reading 27).
//
//   psi = (psi_up, psi_dn), stored [nkpt][nband][2][mpw];   H = kin (x) 1 + V^{ss'}(r) + sum |p_a,i> D^{a,ss'}_ij <p_a,j|
//
// Non-local term: the two components are two more "bands" for both GEMMs (rows 2 b + s of a [2 nband][mpw] block, the
// kernels of nonlocal.cu unchanged); only the small step between them mixes the spins (dij_spinor_kernel).  The
// kinetic diagonal is the same for both components (GEMM-2's epilogue).
// Local term: V = V0 + Vx sigma_x + Vy sigma_y + Vz sigma_z (Pauli decomposition of the Hermitian 2x2 matrix:
// V0 = (V_upup + V_dndn)/2, Vz = (V_upup - V_dndn)/2, Vx = Re V_updn, Vy = -Im V_updn), and every V_mu is a REAL field, so
//   V psi = Loc_V0(psi) + sum_mu Loc_Vmu(sigma_mu psi):
// four applications of the scalar local term (pruned FFT passes of fft2.cu / fft_small.cu, unchanged), the last three
// on sigma_mu psi (one elementwise kernel each) accumulating onto the first.  That form serves every box.  Where all three
// box lengths have a two-radix factorisation and the box is too large for the fused small-box kernel (the five-pass
// register path of fft2.cu), ONE local application does it all: the rows (band, s) go through passes A and B like 2 nband
// scalar bands, pass C multiplies the 2 x 2 matrix in real space (fft2_c_spinor_kernel: the two components of a point
// sit in partner lanes of a warp), and passes B^-1, A^-1 bring both components back -- a quarter of the transforms
// (option spinor_fused, default 1).  Nothing here is shared with the CPU checker.
#include "internal.h"

namespace dftb200 {

namespace {

// out[0..3][j] = (V0, Vx, Vy, Vz)(r_j) / N and out[4..7][j] = v4 / N from v4 = (V_upup, V_dndn, Re V_updn, Im V_updn)
__global__ void pauli_split_kernel(const double *__restrict__ v4, double *__restrict__ out, int64_t n, double s) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double uu = v4[i], dd = v4[n + i], re = v4[2 * n + i], im = v4[3 * n + i];
    out[i] = 0.5 * (uu + dd) * s; out[n + i] = re * s; out[2 * n + i] = -im * s; out[3 * n + i] = 0.5 * (uu - dd) * s;
    out[4 * n + i] = uu * s; out[5 * n + i] = dd * s; out[6 * n + i] = re * s; out[7 * n + i] = im * s;   // the matrix itself / N
  }
}

// out = sigma_mu psi on rows (band, s): mu = 1: (dn, up); 2: (-i dn, i up); 3: (up, -dn).  grid (ceil(mpw/256), rows/2)
__global__ void pauli_apply_kernel(const double2 *__restrict__ psi, double2 *__restrict__ out, int mpw, int mu) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= mpw) return;
  const size_t r = (size_t)blockIdx.y * 2 * mpw + g;
  const double2 u = psi[r], d = psi[r + mpw];
  double2 ou, od;
  if (mu == 1) { ou = d; od = u; }
  else if (mu == 2) { ou = make_double2(d.y, -d.x); od = make_double2(-u.y, u.x); }
  else { ou = u; od = make_double2(-d.x, -d.y); }
  out[r] = ou; out[r + mpw] = od;
}

}  // namespace

int spinor_set_vloc(dft_plan *p, const double *v4, cudaStream_t st) {
  const int64_t n = p->nbox;
  if (!p->d_vpauli && cudaMalloc(&p->d_vpauli, sizeof(double) * 8 * n) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the spinor potential"); return DFT_ERR_ALLOC; }
  const int grid = (int)((n + 255) / 256 < 148 * 8 ? (n + 255) / 256 : 148 * 8);
  pauli_split_kernel<<<grid, 256, 0, st>>>(v4, p->d_vpauli, n, 1.0 / (double)n);
  DFT_CUDA_CHECK(cudaGetLastError());
  p->vspin_set = true;
  return DFT_OK;
}

// psi, hpsi: [nkpt][nband][2][mpw] complex (device)
int spinor_apply(dft_plan *p, const double *psi, double *hpsi, int nband, cudaStream_t st) {
  p->last_launches = 0;
  if (nband == 0 || p->mpw == 0 || p->nkpt == 0) return DFT_OK;
  const bool loc = (p->terms & 2) != 0, kin = (p->terms & 1) != 0, nl = (p->terms & 4) != 0 && p->nproj > 0;
  if (loc && !p->vspin_set) { set_error("dft_apply_h_spinor called before dft_set_vloc_spinor"); return DFT_ERR_NOT_READY; }
  if ((p->terms & 8) && p->vtau_set) { set_error("dft_apply_h_spinor: the meta-GGA term is not available for spinors (option terms, bit 3)"); return DFT_ERR_UNSUPPORTED; }
  int rc;
  const int rows = 2 * nband;
  const int64_t n = p->nbox;
  // one application with the 2 x 2 matrix in pass C where the five-pass register path serves the box
  bool fused = p->spinor_fused && p->fft_path != 1 && !((p->fft_path == 0 || p->fft_path == 3 || p->fft_path == 5) && fft_small_ok(p));
  for (int c = 0; c < 3 && fused; c++) fused = fft2_pair(p->n[c], nullptr, nullptr);
  { int r1 = 0, r2 = 0; if (fused && fft2_pair(p->n[2], &r1, &r2) && r2 > 16) fused = false; }   // the 2 x 2 pass holds 16 lanes per slot row
  for (int ik = 0; ik < p->nkpt && fused; ik++) fused = p->kp[ik].runs_ok;
  if (loc && fused) {
    FftExtra X;
    X.vspin = p->d_vpauli + 4 * n;
    if ((rc = local_term(p, psi, hpsi, rows, st, &X))) return rc;
  } else if (loc) {
    const int64_t need = (int64_t)p->nkpt * rows * p->mpw * 16;
    if (need > p->spin_tmp_bytes) {
      if (p->d_spin_tmp) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->d_spin_tmp); p->d_spin_tmp = nullptr; p->spin_tmp_bytes = 0; }
      if (cudaMalloc(&p->d_spin_tmp, need) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes for sigma psi", (long long)need); return DFT_ERR_ALLOC; }
      p->spin_tmp_bytes = need;
    }
    FftExtra X;
    X.vpot = p->d_vpauli;                                  // V0
    if ((rc = local_term(p, psi, hpsi, rows, st, &X))) return rc;
    for (int mu = 1; mu <= 3; mu++) {
      phase_begin(p, 9, st);
      pauli_apply_kernel<<<dim3((p->mpw + 255) / 256, p->nkpt * nband), 256, 0, st>>>(
          reinterpret_cast<const double2 *>(psi), reinterpret_cast<double2 *>(p->d_spin_tmp), p->mpw, mu);
      phase_end(p, 9, st, 1);
      DFT_CUDA_CHECK(cudaGetLastError());
      FftExtra Y;
      Y.vpot = p->d_vpauli + (size_t)mu * n; Y.accumulate = 1;
      if ((rc = local_term(p, p->d_spin_tmp, hpsi, rows, st, &Y))) return rc;
    }
  } else {
    phase_begin(p, 4, st);
    if ((rc = zero_fill(hpsi, (int64_t)p->nkpt * rows * p->mpw * 2, st))) return rc;
    phase_end(p, 4, st, 1);
  }
  if (kin || nl)
    if ((rc = nonlocal_apply_spinor(p, psi, hpsi, nband, true, kin, nl, st))) return rc;
  return DFT_OK;
}

}  // namespace dftb200
