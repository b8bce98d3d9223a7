// internal.h -- plan structure and the launchers shared by the translation units of libdftb200.
// Nothing here is shared with oracle/ (the CPU checker): every rule is restated from DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <cuda.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/dft.h"

namespace dftb200 {

// ------------------------------------------------------------------------------------------
// error plumbing
// ------------------------------------------------------------------------------------------
void set_error(const char *fmt, ...);
#define DFT_CUDA_CHECK(expr)                                                              \
  do {                                                                                    \
    cudaError_t e__ = (expr);                                                             \
    if (e__ != cudaSuccess) {                                                             \
      ::dftb200::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
      return DFT_ERR_CUDA;                                                                \
    }                                                                                     \
  } while (0)

// ------------------------------------------------------------------------------------------
// FFT schedule of one 1-D length: radices (each in {2,3,4,5,8,9}), product = n
// ------------------------------------------------------------------------------------------
struct FftFactors {
  int n = 0;
  int nfac = 0;
  int radix[12] = {0};
};
bool factorize(int n, FftFactors *f);

// Up to two runs of consecutive box indices along one axis: [lo, lo+nlo) -> base + (x - lo),
// [hi, hi+nhi) -> base + nlo + (x - hi).  The sphere is convex, so the occupied x of a column, the
// occupied y of a plane and the occupied z of the box each have this form (K2).
struct Run {
  int32_t base, lo, nlo, hi, nhi, aux0, aux1, pad;
};

// Per-k-point geometry of the sphere and of the pruned passes (device pointers unless noted)
struct KPoint {
  double k[3];
  int npw = 0;
  // sphere (K1)
  int32_t *kg = nullptr;      // [npw][3]
  int32_t *igfft = nullptr;   // [npw]
  double *kin = nullptr;      // [npw]
  // pruned-FFT geometry derived from kg on the host
  int ncol = 0;               // non-empty (i2,i3) columns, sorted by (i3,i2) = order of first plane wave
  int nplane = 0;             // non-empty i3 planes (s_3)
  int32_t *col_start = nullptr;  // [ncol+1] first plane wave of column c (columns are contiguous runs of the kg list)
  int32_t *col_i2 = nullptr;     // [ncol]
  int32_t *col_plane = nullptr;  // [ncol]  plane ordinal p (0..nplane-1) of the column
  int32_t *pw_i1 = nullptr;      // [npw]   box index along axis 1 of each plane wave
  int32_t *plane_i3 = nullptr;   // [nplane] box index i3 of plane p
  int32_t *plane_col0 = nullptr; // [nplane+1] first column of plane p
  // the same geometry as runs (register-resident FFT path, fft2.cu)
  Run *col_run = nullptr;        // [ncol]   base = first plane wave, runs along x; aux0 = i2, aux1 = plane
  Run *plane_run = nullptr;      // [nplane] base = first column, runs along y; aux0 = i3
  Run zrun = {0, 0, 0, 0, 0, 0, 0, 0};   // base = 0, runs along z (plane ordinals)
  int max_cols_per_plane = 0;    // largest number of non-empty columns in one plane (TMA box height of pass B)
  bool runs_ok = false;          // every occupied set really is <= 2 runs (else the generic path is used)
  // host copies for getters
  std::vector<int32_t> h_kg, h_igfft;
  std::vector<double> h_kin;
};

// Gamma-point real-symmetry storage (gamma.cu; reading 26): the half sphere, its maps to the full sphere and the
// projector table on it (rows of odd l multiplied by i, so that every projection is real)
struct GammaData {
  int nh = 0;                          // stored plane waves = (npw + 1) / 2
  int32_t *d_kg = nullptr;             // [nh][3]
  double *d_kin = nullptr;             // [nh]
  int32_t *d_h2f = nullptr;            // [nh]  position of +G in the full list
  int32_t *d_h2fneg = nullptr;         // [nh]  position of -G in the full list
  int32_t *d_f2h = nullptr;            // [npw] +(h + 1): full entry is stored entry h; -(h + 1): its conjugate
  double *d_ptab = nullptr;            // [nproj][nh] complex
  double *d_p0 = nullptr;              // [nproj] Re of the table's G = 0 column (the term counted twice by 2 sum_half)
  int32_t *d_rowpar = nullptr;         // [natom][lmax] l mod 2 of every projector (D_ij couples equal parity only)
  int32_t *d_npw = nullptr;            // [1] = nh
  const double **d_kinptr = nullptr;   // [1] -> d_kin
  double *d_pack = nullptr; int64_t pack_bytes = 0;   // packed band pairs in / out, [2][pairs][mpw] complex
  std::vector<int32_t> h_kg, h_igfft;
  std::vector<double> h_kin;
};

struct NlMaps;
struct SymMaps;
struct StrassenData;
void nl_maps_free(dft_plan *p);

// timed kernel groups: 0-4 the five FFT passes, 5 GEMM-1, 6 D_ij, 7 GEMM-2, 8 the fused small-box local term (fft_small.cu),
// 9 pack / unpack of band pairs (Gamma storage) and the spin-matrix products of the spinor path
constexpr int NPHASE = 10;
struct PhaseTimer {
  bool on = false;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev[NPHASE];
  std::vector<cudaEvent_t> pool;   // events handed back by dft_plan_phase_ms, reused by later applies
  int64_t launches[NPHASE] = {0};
};

}  // namespace dftb200

struct FacGroup { int frow0, nfrow, blk0, nblk; };   // first FY row / rows, first block / blocks of one group of atom types (projtab.cu)

struct dft_plan {
  // lattice
  double rprimd[9], bm[9], gmet[9];
  double ecut;
  int n[3];
  int64_t nbox;
  int nkpt = 0, mpw = 0;
  std::vector<dftb200::KPoint> kp;
  // atoms / projectors
  int natom = 0, ntypat = 0, lmax = 0, nproj = 0;
  std::vector<int32_t> typat, nlmn, lmn_l, lmn_m, lmn_irad, atom_first;  // lmn_*: [ntypat][lmax]
  std::vector<double> xred;
  std::vector<int32_t> nq; std::vector<double> dq;   // per type
  int nrad_max = 0, nq_max = 0;
  double *d_f = nullptr, *d_f2 = nullptr;            // [ntypat][nrad_max][nq_max]
  int32_t *d_typat = nullptr, *d_nlmn = nullptr, *d_lmn_l = nullptr, *d_lmn_m = nullptr, *d_lmn_irad = nullptr;
  int32_t *d_atom_first = nullptr, *d_nq = nullptr;
  double *d_dq = nullptr, *d_xred = nullptr;
  double *d_dij = nullptr;                           // [natom][lmax][lmax]
  double *d_sij = nullptr;                           // [natom][lmax][lmax] overlap coefficients s_ij (zero until dft_set_sij)
  double *d_kina = nullptr;                          // [nkpt][mpw] 1/2|k+G+A|^2 while a vector potential is set
  const double **d_kinaptr = nullptr;                // [nkpt] device pointers into d_kina
  bool vecpot_on = false;
  double *d_ones = nullptr;                          // [mpw] of 1.0: the unit diagonal of S in GEMM-2's epilogue
  const double **d_oneptr = nullptr;                 // [nkpt] device pointers to d_ones
  double *d_stab = nullptr, *d_fytab = nullptr;      // factorised projectors: structure factors / form factors (proj_mode = 1)
  int32_t *d_blk_atom = nullptr, *d_blk_frow = nullptr, *d_blk_first = nullptr, *d_blk_nl = nullptr;   // projector blocks (<= 8 rows)
  int nblk = 0, nfrow = 0;                           // number of blocks; FY rows of all types
  std::vector<FacGroup> fac_groups;                  // consecutive atom types whose FY rows fit the kernels' shared memory
  int ldf = 0;                                       // row length of d_fytab (mpw rounded up to 8)
  int proj_mode = 0;                                 // 0 = materialised table (GEMMs on P), 1 = factorised P = FY . S
  int fft_c_split = 2;                               // pass C (16-line tiles): two barrier domains per CTA (fft2_c_ring2_kernel): 0 = never, 1 = wherever possible, 2 = where both radices are >= 12
  int gemm2_merge = 1;                               // Strassen path: the seven back-projection products in one launch
  int nl_tiny = 1;                                   // tiny cells: the whole non-local term in one launch (nl_tiny_kernel), 0 = always the GEMM kernels
  bool skip_table_at_create = false;                 // dft_plan_create_opts(proj_mode = 1): never allocate the materialised table
  double *d_ptab = nullptr;                          // [nkpt][nproj][mpw] complex, zero padded beyond npw_k
  int32_t *d_npw = nullptr;                          // [nkpt]
  const double **d_kinptr = nullptr;                 // [nkpt] device pointers to kin of each k-point
  // local potential
  double *d_vloc = nullptr;                          // [n3][n2][n1], pre-scaled by 1/N
  bool vloc_set = false;
  double *d_vtau = nullptr;                          // [n3][n2][n1] v_tau(r)/N (meta-GGA), set by dft_set_vtau
  double *d_qcart = nullptr, *d_qhalf = nullptr;     // [nkpt][3][mpw] Cartesian k+G and half of it
  bool vtau_set = false;
  // FFT
  dftb200::FftFactors fac[3];
  double *d_tw[3] = {nullptr, nullptr, nullptr};     // twiddles exp(+2 pi i j/n_c), [n_c] complex
  // options
  int band_chunk = 0;      // 0 = automatic
  int terms = 15;          // bit 0 kinetic, bit 1 local, bit 2 non-local, bit 3 meta-GGA term (active once dft_set_vtau was called)
  int fft_path = 0;        // 0 = automatic (fused small-box kernel when a band's working set fits one SM's shared memory, else
                           // the register path with the TMA ring for the strided passes), 1 = generic Stockham path only,
                           // 2 = register path without the TMA ring, 3 = fused small-box kernel (error if it does not fit),
                           // 4 = automatic without the small-box kernel
  int splitk = 0;
  int gemm_3m = 1;         // 1 = three real products per complex multiply-add (6 flops), 0 = four (8 flops)
  // workspace
  void *ws_user = nullptr; int64_t ws_user_bytes = 0;
  void *ws_own = nullptr;  int64_t ws_own_bytes = 0;
  // GEMM scratch (plan-owned, sized at first use)
  double *d_part = nullptr; int64_t part_bytes = 0;  // split-K partials
  double *d_cprj = nullptr; int64_t cprj_bytes = 0;  // c' [nkpt][nband][nproj] complex
  // host staging for dft_apply_h_host
  double *d_stage_in = nullptr, *d_stage_out = nullptr; int64_t stage_bytes = 0;
  cudaStream_t host_stream = nullptr, h2d_stream = nullptr, d2h_stream = nullptr;
  int host_groups = 6;     // dft_apply_h_host: band groups whose copies overlap the kernels of their neighbours
  // TMA
  void *encode_fn = nullptr;   // cuTensorMapEncodeTiled
  double *d_wgt = nullptr; int64_t wgt_count = 0;    // device copy of the band weights of dft_accumulate_density
  void *d_geom2 = nullptr;    // device array of per-k-point FFT geometry (fft2.cu, built at first batched call)
  void *d_geom_small = nullptr;   // the same for the fused small-box kernel (fft_small.cu)
  bool small_attr_done = false;
  unsigned small2_attr_mask = 0;  // instantiations of fft_small2.cu whose shared-memory attribute is set on this plan's device
  int32_t *d_dstmap = nullptr;    // [nkpt][mpw] position of every plane wave in the x-line array of fft_small2.cu
  int sm_count = 148;
  int smem_per_sm = 233472, smem_optin = 232448;   // bytes of shared memory per SM / per CTA (opt-in), from the device
  int64_t last_launches = 0;
  bool nl_attr_done = false;   // cudaFuncSetAttribute of the GEMM kernels done on this plan's device
  dftb200::PhaseTimer timer;
  dftb200::SymMaps *sym_maps = nullptr; // the same for the symmetric-table GEMMs at k = 0
  dftb200::NlMaps *nl_maps = nullptr;  // tensor maps of the table-mode GEMMs, kept between calls (nonlocal.cu)
  dftb200::GammaData *gam = nullptr;   // half sphere + rotated table: built by option gamma_real = 1 or by the symmetric-table GEMMs
  bool gamma_on = false;               // option gamma_real = 1 (dft_apply_h_gamma allowed, D_ij parity enforced)
  int gemm_sym = 2;                    // at k = 0 run the projector GEMMs of dft_apply_h as real GEMMs on the half sphere (nonlocal.cu): 0 never, 1 always, 2 = when large enough
  dftb200::StrassenData *strassen = nullptr;   // block tables and scratch of the Strassen level on the real GEMMs (nonlocal_strassen.inc)
  int gemm_strassen = 2;               // 0 never, 1 wherever possible, 2 = automatic (large problems): 7 half-size products per real GEMM instead of 8
  int sym_state = 0;                   // 0 = not tried, 1 = tables ready, -1 = this plan cannot (k != 0, several k-points, unpaired Nyquist index)
  double *d_symx = nullptr; int64_t symx_bytes = 0;   // time-reversal-even/odd halves of the bands, [2 nband][nhalf] complex
  // two-component spinors (spinor.cu): Pauli components of the local potential, spin-dependent D
  double *d_vpauli = nullptr;          // [8][n3][n2][n1]: V0, Vx, Vy, Vz, then V_upup, V_dndn, Re V_updn, Im V_updn, each pre-scaled by 1/N
  int spinor_fused = 1;                // 1: one local application with the 2 x 2 matrix in pass C where the register path serves the box
  double *d_dspin = nullptr;           // [natom][2][2][lmax][lmax] complex
  double *d_spin_tmp = nullptr; int64_t spin_tmp_bytes = 0;   // sigma_mu psi, [nband][2][mpw] complex
  bool vspin_set = false, dspin_set = false, gam_attr_done = false;
};

namespace dftb200 {

// --- sphere.cu (K1) -----------------------------------------------------------------------
void lattice_algebra(const double *a, double *bm, double *gmet, double *det);
// Extents of the sphere over the integer cube |m_j| <= bound_j; returns status.
int sphere_extent(const double *gmet, const double *k, double ecut, const int bound[3], int mmin[3], int mmax[3]);
// Build kg/igfft/kin of one k-point on the device (ascending box index); fills kp.npw and device arrays.
int sphere_build(const double *gmet, const int n[3], double ecut, KPoint *kp);

// --- projtab.cu (S1) ----------------------------------------------------------------------
int build_projector_table(dft_plan *p, int ik, double *maxq_out);
constexpr int FAC_MAX_FROWS = 32;        // FY rows (8 per projector block, summed over atom types) the kernels keep in shared memory
int build_factor_tables(dft_plan *p);   // S [nkpt][natom][mpw] complex and FY [nkpt][ntypat*8][ldf] real (factorised projectors)

// Optional variations of the local application (meta-GGA term): another potential in pass C, a real diagonal factor
// applied to psi in G space while scattering (pass A), another one while gathering (pass A^-1), accumulation onto hpsi.
struct FftExtra {
  const double *vpot = nullptr;   // device [n3][n2][n1], pre-scaled by 1/N; null = the plan's V_loc
  const double *pre = nullptr;    // device [npw]; null = 1
  const double *post = nullptr;   // device [npw]; null = 1
  int accumulate = 0;             // 1: hpsi += result (pad entries untouched) instead of hpsi = result
  const double *vspin = nullptr;  // device [4][n3][n2][n1] = (V_upup, V_dndn, Re V_updn, Im V_updn) / N: the rows are (up, down)
                                  // pairs of two-component spinors and pass C applies the 2 x 2 matrix (register path only)
};
// --- fft.cu (K2) --------------------------------------------------------------------------
int64_t fft_ws_bytes_per_band(const dft_plan *p);
int64_t fft_ws_bytes_per_band_batched(const dft_plan *p);   // per band, all k-points (fft2_apply_batched's layout)
// V_loc psi for `nb` bands of k-point ik: psi/hpsi point at the first band ([nb][mpw] complex)
int fft_apply_vloc(dft_plan *p, int ik, const double *psi, double *hpsi, int nb, void *ws, cudaStream_t st,
                   const FftExtra *extra = nullptr);
int zero_fill(double *hpsi, int64_t ndouble, cudaStream_t st);
// fft2.cu: two-stage register path.  fft2_pair: is n = R1*R2 with both radices available as codelets?
bool fft2_pair(int n, int *r1, int *r2);
// pass: 0 A, 1 B, 2 C, 3 B^-1, 4 A^-1; T1/T2 strides in complex elements per band
int fft2_launch(dft_plan *p, int ik, int pass, const double *psi, double *hpsi, void *T1, void *T2, int64_t t1_band,
                int64_t t2_band, int nb, cudaStream_t st, const FftExtra *extra = nullptr);

// Optional combination applied where H psi is stored (GEMM-2 epilogue): out = sh * (H psi) + sy * psi + sx * xprev.
// One step of a three-term recurrence in H (Chebyshev filter, PAPER.md :458) without extra passes over psi-sized arrays.
struct Recurrence {
  double sh, sy, sx;
  const double *xprev;   // device [nkpt][nband][mpw] complex; read only where sx != 0
};

// several k-points per launch (plain register kernels with blockIdx.y = k-point)
bool fft2_batch_ok(const dft_plan *p);
int fft2_apply_batched(dft_plan *p, const double *psi, double *hpsi, int nb, int nband_total, void *ws, cudaStream_t st);

// rho(r) += sum_b wgt[b] |psi_b(r)|^2 (device wgt [nb]); forward passes A, B and the density kernel
int fft_density_generic(dft_plan *p, int ik, const double *psi, const double *wgt_dev, double *rho, int nb, void *ws, cudaStream_t st,
                        const double *pre);   // fft.cu: any box (generic passes where an axis has no two-radix factorisation)
int fft2_density(dft_plan *p, int ik, const double *psi, const double *wgt_dev, double *rho, int nb, void *ws, cudaStream_t st,
                 const double *pre = nullptr);

// --- fft_small.cu (K2s): the whole local term in one kernel, one CTA per (k-point, band), no scratch in device memory
bool fft_small_ok(const dft_plan *p);
int fft_small_apply(dft_plan *p, int ik0, int nk, const double *psi, double *hpsi, int nb, int nband_total, cudaStream_t st,
                    const FftExtra *extra = nullptr);

int fft_small2_launch(dft_plan *p, void *sb_params, int nk, int nb, cudaStream_t st, bool *handled);   // fft_small2.cu

// --- nonlocal.cu (K3) ---------------------------------------------------------------------
// hpsi (+)= V_nl psi + kin*psi for all k-points; accumulate = hpsi already holds V_loc psi
int nonlocal_apply(dft_plan *p, const double *psi, double *hpsi, int nband, bool accumulate, bool with_kin,
                   bool with_nl, cudaStream_t st, const double *dmat = nullptr, const double *const *diag = nullptr,
                   double *cprj_out = nullptr, const Recurrence *rec = nullptr, double *spsi = nullptr,
                   const double *dspin = nullptr);

// Gamma storage: the same three steps as real GEMMs on the half sphere (psi, hpsi: [nband][nh] complex)
int nonlocal_apply_gamma(dft_plan *p, const double *psi, double *hpsi, int nband, bool accumulate, bool with_kin, bool with_nl,
                         cudaStream_t st, const Recurrence *rec);
// spinors: psi [nband][2][mpw]; dspin = null applies the plan's scalar D_ij to both components
int nonlocal_apply_spinor(dft_plan *p, const double *psi, double *hpsi, int nband, bool accumulate, bool with_kin, bool with_nl,
                          cudaStream_t st);

// --- plan.cu: the local term of all k-points for [nkpt][nband][mpw] blocks (hpsi = V_loc psi, or += with extra->accumulate)
int local_term(dft_plan *p, const double *psi, double *hpsi, int nband, cudaStream_t st, const FftExtra *extra = nullptr);

// --- gamma.cu / spinor.cu ------------------------------------------------------------------------
int gamma_build(dft_plan *p, bool check_dij);
void gamma_free(dft_plan *p);
int gamma_check_dij(const dft_plan *p, const double *dij_host);
int gamma_apply(dft_plan *p, const double *psi, double *hpsi, int nband, cudaStream_t st, const Recurrence *rec = nullptr);
int spinor_apply(dft_plan *p, const double *psi, double *hpsi, int nband, cudaStream_t st);
int spinor_set_vloc(dft_plan *p, const double *v4, cudaStream_t st);
int build_projector_table_on(dft_plan *p, const int32_t *d_kg, int npw, int mpw, const double k[3], double *d_out, int rot_odd);

// --- timing hooks ------------------------------------------------------------------------------
void phase_begin(dft_plan *p, int phase, cudaStream_t st);
void phase_end(dft_plan *p, int phase, cudaStream_t st, int launches);

}  // namespace dftb200
