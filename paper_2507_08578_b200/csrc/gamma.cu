// gamma.cu -- Gamma-point real-symmetry storage (PAPER.md :407 "time-reversal symmetry";
// DESIGN.md reading 26).
//
// At k = 0 a band whose psi(r) is real has c(-G) = conj(c(G)); the caller stores one plane wave of every pair
// (m3 > 0, or m3 = 0 and m2 > 0, or m3 = m2 = 0 and m1 >= 0; ascending box index; nh = (npw + 1)/2).  The operator is
// the full one on the symmetric vector, restricted again.  Here it is computed WITHOUT expanding:
//
//   local term : two stored bands A, B are packed into ONE complex full-sphere vector f = c_A + i c_B (f(-G) =
//                conj(c_A(G)) + i conj(c_B(G))), i.e. psi_A(r) + i psi_B(r) with both real; one pruned complex FFT
//                round trip (the kernels of fft2.cu / fft_small.cu, unchanged) serves both, and because V is real
//                h_A(G) = (h(G) + conj(h(-G)))/2, h_B(G) = (h(G) - conj(h(-G)))/(2i).  Half the transforms.
//   non-local  : p(-G) = (-1)^l conj(p(G)), so with the table rows of odd l multiplied by i every projection of a
//                symmetric vector is REAL: <p|psi> = i^(l odd) r, r = 2 sum_half (Pt_r c_r + Pt_i c_i) - (G = 0 term).
//                Both GEMMs become real GEMMs over the interleaved (re, im) doubles of the half sphere
//                (gemm1_kernel<true>, gemm2_kernel<true> in nonlocal.cu): a quarter of the 4-product flops.
//   kinetic    : diagonal on the stored half, in GEMM-2's epilogue as always.
//
// D_ij must not couple projectors of different l-parity (else H does not commute with time reversal and the storage
// is not closed): refused with DFT_ERR_INVALID_ARG.  Nothing here is shared with the CPU checker.
#include <algorithm>

#include "internal.h"

namespace dftb200 {

namespace {

template <typename T>
int up(T **dst, const std::vector<T> &v) {
  *dst = nullptr;
  if (v.empty()) return DFT_OK;
  if (cudaMalloc(dst, v.size() * sizeof(T)) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %zu bytes (Gamma storage)", v.size() * sizeof(T)); return DFT_ERR_ALLOC; }
  DFT_CUDA_CHECK(cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
  return DFT_OK;
}

// f[q][g] = c_{2q}(+-G) (+ conj) + i c_{2q+1}(+-G) (+ conj); grid (ceil(npw / 256), pairs)
__global__ void gamma_pack_kernel(const double2 *__restrict__ psi, double2 *__restrict__ f, const int32_t *__restrict__ f2h,
                                  int npw, int mpw, int nh, int b0, int nband) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x, q = blockIdx.y;
  if (g >= mpw) return;
  double2 out = make_double2(0.0, 0.0);
  if (g < npw) {
    const int t = f2h[g], h = (t > 0 ? t : -t) - 1;
    const int ba = b0 + 2 * q, bb = ba + 1;
    double2 a = psi[(size_t)ba * nh + h];
    double2 b = bb < nband ? psi[(size_t)bb * nh + h] : make_double2(0.0, 0.0);
    if (t < 0) { a.y = -a.y; b.y = -b.y; }
    if (h == 0) { a.y = 0.0; b.y = 0.0; }      // G = 0 is stored first; c(0) is real
    out = make_double2(a.x - b.y, a.y + b.x);
  }
  f[(size_t)q * mpw + g] = out;
}

// hpsi_{2q}(G) = (h(G) + conj(h(-G)))/2, hpsi_{2q+1}(G) = (h(G) - conj(h(-G)))/(2i); grid (ceil(nh / 256), pairs)
__global__ void gamma_unpack_kernel(const double2 *__restrict__ hf, double2 *__restrict__ hpsi, const int32_t *__restrict__ h2f,
                                    const int32_t *__restrict__ h2fneg, int mpw, int nh, int b0, int nband) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x, q = blockIdx.y;
  if (h >= nh) return;
  const double2 u = hf[(size_t)q * mpw + h2f[h]], v = hf[(size_t)q * mpw + h2fneg[h]];
  const int ba = b0 + 2 * q, bb = ba + 1;
  hpsi[(size_t)ba * nh + h] = make_double2(0.5 * (u.x + v.x), 0.5 * (u.y - v.y));
  if (bb < nband) hpsi[(size_t)bb * nh + h] = make_double2(0.5 * (u.y + v.y), -0.5 * (u.x - v.x));
}

}  // namespace

void gamma_free(dft_plan *p) {
  GammaData *G = p->gam;
  if (!G) return;
  cudaFree(G->d_kg); cudaFree(G->d_kin); cudaFree(G->d_h2f); cudaFree(G->d_h2fneg); cudaFree(G->d_f2h); cudaFree(G->d_ptab);
  cudaFree(G->d_p0); cudaFree(G->d_rowpar); cudaFree(G->d_npw); cudaFree((void *)G->d_kinptr); cudaFree(G->d_pack);
  delete G;
  p->gam = nullptr;
}

// D_ij (host, [natom][lmax][lmax]) must vanish between projectors of different l-parity
int gamma_check_dij(const dft_plan *p, const double *dij) {
  for (int a = 0; a < p->natom; a++) {
    const int t = p->typat[a], nl = p->nlmn[t];
    for (int i = 0; i < nl; i++)
      for (int j = 0; j < nl; j++)
        if (((p->lmn_l[t * p->lmax + i] + p->lmn_l[t * p->lmax + j]) & 1) && dij[((size_t)a * p->lmax + i) * p->lmax + j] != 0.0) {
          set_error("Gamma storage: D_ij of atom %d couples projectors %d (l = %d) and %d (l = %d) of different parity; H would not "
                    "commute with time reversal (DESIGN.md reading 26)", a, i, p->lmn_l[t * p->lmax + i], j, p->lmn_l[t * p->lmax + j]);
          return DFT_ERR_INVALID_ARG;
        }
  }
  return DFT_OK;
}

// check_dij: the Gamma STORAGE (dft_apply_h_gamma) needs a D_ij without odd-parity couplings; the tables alone (half
// sphere, maps, rotated projector table) also serve the symmetric-table GEMMs of dft_apply_h at k = 0 (nonlocal.cu), which
// take any D_ij.
int gamma_build(dft_plan *p, bool check_dij) {
  if (check_dij && p->natom > 0 && p->nproj > 0 && p->nkpt == 1) {
    std::vector<double> d((size_t)p->natom * p->lmax * p->lmax);
    DFT_CUDA_CHECK(cudaMemcpy(d.data(), p->d_dij, d.size() * sizeof(double), cudaMemcpyDeviceToHost));
    int rc = gamma_check_dij(p, d.data());
    if (rc) return rc;
  }
  if (p->gam) return DFT_OK;
  if (p->nkpt != 1) { set_error("Gamma storage needs a plan with one k-point (has %d)", p->nkpt); return DFT_ERR_UNSUPPORTED; }
  const KPoint &K = p->kp[0];
  if (K.k[0] != 0.0 || K.k[1] != 0.0 || K.k[2] != 0.0) { set_error("Gamma storage needs k = 0"); return DFT_ERR_UNSUPPORTED; }
  const int npw = K.npw, n1 = p->n[0], n2 = p->n[1], n3 = p->n[2];
  GammaData *G = new GammaData();
  std::vector<int32_t> h2f, h2fneg, f2h(npw, 0);
  // position of a box index in the (ascending) full list
  auto find = [&](int64_t idx) -> int {
    auto it = std::lower_bound(K.h_igfft.begin(), K.h_igfft.end(), (int32_t)idx);
    return (it != K.h_igfft.end() && *it == (int32_t)idx) ? (int)(it - K.h_igfft.begin()) : -1;
  };
  for (int g = 0; g < npw; g++) {
    const int m1 = K.h_kg[3 * g], m2 = K.h_kg[3 * g + 1], m3 = K.h_kg[3 * g + 2];
    const bool keep = m3 > 0 || (m3 == 0 && m2 > 0) || (m3 == 0 && m2 == 0 && m1 >= 0);
    if (!keep) continue;
    const int i1 = ((-m1) % n1 + n1) % n1, i2 = ((-m2) % n2 + n2) % n2, i3 = ((-m3) % n3 + n3) % n3;
    const int gm = find((int64_t)i1 + (int64_t)n1 * (i2 + (int64_t)n2 * i3));
    // the partner must be the plane wave -m itself (not an alias of it): an unpaired Nyquist index m = -n/2 fails here
    if (gm < 0 || K.h_kg[3 * gm] != -m1 || K.h_kg[3 * gm + 1] != -m2 || K.h_kg[3 * gm + 2] != -m3) {
      delete G;
      set_error("Gamma storage: the sphere does not hold -G for G = (%d, %d, %d)", m1, m2, m3);
      return DFT_ERR_UNSUPPORTED;
    }
    const int h = (int)h2f.size();
    h2f.push_back(g); h2fneg.push_back(gm);
    f2h[gm] = -(h + 1);
    f2h[g] = h + 1;                      // after the partner, so that G = 0 (its own partner) is marked as stored
    G->h_kg.push_back(m1); G->h_kg.push_back(m2); G->h_kg.push_back(m3);
    G->h_igfft.push_back(K.h_igfft[g]); G->h_kin.push_back(K.h_kin[g]);
  }
  G->nh = (int)h2f.size();
  p->gam = G;
  if (G->nh == 0) return DFT_OK;
  if (K.h_kg[3 * h2f[0]] != 0 || K.h_kg[3 * h2f[0] + 1] != 0 || K.h_kg[3 * h2f[0] + 2] != 0) {
    gamma_free(p); set_error("Gamma storage: G = 0 is not the first stored plane wave"); return DFT_ERR_UNSUPPORTED;
  }
  int rc;
  std::vector<int32_t> npw1(1, G->nh), rowpar((size_t)p->natom * p->lmax, 0);
  for (int a = 0; a < p->natom; a++)
    for (int i = 0; i < p->nlmn[p->typat[a]]; i++) rowpar[(size_t)a * p->lmax + i] = p->lmn_l[p->typat[a] * p->lmax + i] & 1;
  if ((rc = up(&G->d_kg, G->h_kg)) || (rc = up(&G->d_kin, G->h_kin)) || (rc = up(&G->d_h2f, h2f)) || (rc = up(&G->d_h2fneg, h2fneg)) ||
      (rc = up(&G->d_f2h, f2h)) || (rc = up(&G->d_npw, npw1)) || (rc = up(&G->d_rowpar, rowpar))) { gamma_free(p); return rc; }
  std::vector<const double *> kptr(1, G->d_kin);
  if ((rc = up((const double ***)&G->d_kinptr, kptr))) { gamma_free(p); return rc; }
  if (p->nproj > 0) {
    const size_t tab = (size_t)p->nproj * G->nh * 16;
    if (cudaMalloc(&G->d_ptab, tab + 256) != cudaSuccess || cudaMalloc(&G->d_p0, sizeof(double) * p->nproj) != cudaSuccess) {
      cudaGetLastError(); gamma_free(p); set_error("cannot allocate the Gamma projector table (%zu bytes)", tab); return DFT_ERR_ALLOC;
    }
    DFT_CUDA_CHECK(cudaMemset(G->d_ptab, 0, tab + 256));
    if ((rc = build_projector_table_on(p, G->d_kg, G->nh, G->nh, K.k, G->d_ptab, 1))) { gamma_free(p); return rc; }
    // column G = 0 (real parts): the term that 2 * sum_half counts twice
    DFT_CUDA_CHECK(cudaMemcpy2D(G->d_p0, sizeof(double), G->d_ptab, (size_t)G->nh * 16, sizeof(double), p->nproj, cudaMemcpyDeviceToDevice));
  }
  DFT_CUDA_CHECK(cudaDeviceSynchronize());
  return DFT_OK;
}

// psi, hpsi: [nband][nh] complex (device)
int gamma_apply(dft_plan *p, const double *psi, double *hpsi, int nband, cudaStream_t st, const Recurrence *rec) {
  GammaData *G = p->gam;
  if (!G || !p->gamma_on) { set_error("Gamma storage is not enabled (dft_plan_set_option gamma_real = 1)"); return DFT_ERR_NOT_READY; }
  p->last_launches = 0;
  if (nband == 0 || G->nh == 0) return DFT_OK;
  const bool loc = (p->terms & 2) != 0, kin = (p->terms & 1) != 0, nl = (p->terms & 4) != 0 && p->nproj > 0;
  if (loc && !p->vloc_set) { set_error("dft_apply_h_gamma called before dft_set_vloc"); return DFT_ERR_NOT_READY; }
  // terms this entry point does not carry (a vector potential also breaks the time-reversal symmetry the storage rests on)
  if (p->vecpot_on) { set_error("dft_apply_h_gamma: a vector potential is set (H does not commute with time reversal)"); return DFT_ERR_UNSUPPORTED; }
  if ((p->terms & 8) && p->vtau_set) { set_error("dft_apply_h_gamma: the meta-GGA term is not available in Gamma storage (option terms, bit 3)"); return DFT_ERR_UNSUPPORTED; }
  int rc;
  const int nh = G->nh, mpw = p->mpw, npw = p->kp[0].npw;
  if (loc) {
    const int pairs = (nband + 1) / 2;
    const int pc = pairs < 128 ? pairs : 128;                  // band pairs per round trip (bounds the packed scratch)
    const int64_t need = (int64_t)2 * pc * mpw * 16;
    if (need > G->pack_bytes) {
      if (G->d_pack) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(G->d_pack); G->d_pack = nullptr; G->pack_bytes = 0; }
      if (cudaMalloc(&G->d_pack, need) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes for the packed band pairs", (long long)need); return DFT_ERR_ALLOC; }
      G->pack_bytes = need;
    }
    double2 *f = reinterpret_cast<double2 *>(G->d_pack), *hf = f + (size_t)pc * mpw;
    for (int q0 = 0; q0 < pairs; q0 += pc) {
      const int nq = pairs - q0 < pc ? pairs - q0 : pc;
      phase_begin(p, 9, st);
      gamma_pack_kernel<<<dim3((mpw + 255) / 256, nq), 256, 0, st>>>(reinterpret_cast<const double2 *>(psi), f, G->d_f2h, npw, mpw, nh,
                                                                    2 * q0, nband);
      phase_end(p, 9, st, 1);
      DFT_CUDA_CHECK(cudaGetLastError());
      if ((rc = local_term(p, reinterpret_cast<const double *>(f), reinterpret_cast<double *>(hf), nq, st))) return rc;
      phase_begin(p, 9, st);
      gamma_unpack_kernel<<<dim3((nh + 255) / 256, nq), 256, 0, st>>>(hf, reinterpret_cast<double2 *>(hpsi), G->d_h2f, G->d_h2fneg, mpw,
                                                                     nh, 2 * q0, nband);
      phase_end(p, 9, st, 1);
      DFT_CUDA_CHECK(cudaGetLastError());
    }
  } else {
    phase_begin(p, 4, st);
    if ((rc = zero_fill(hpsi, (int64_t)nband * nh * 2, st))) return rc;
    phase_end(p, 4, st, 1);
  }
  if (kin || nl || rec)
    if ((rc = nonlocal_apply_gamma(p, psi, hpsi, nband, true, kin, nl, st, rec))) return rc;
  return DFT_OK;
}

}  // namespace dftb200
