/* dft.h -- C ABI of libdftb200: the plane-wave Kohn-Sham Hamiltonian applied to a block of bands
 *
 *      H|psi> = 1/2|k+G|^2 psi + FFT^-1[ V_loc(r) . FFT[psi] ] + sum_a sum_ij |p_a,i> D^a_ij <p_a,j|psi>
 *
 * on one NVIDIA B200 (sm_100a), FP64.  The operator is the one the ABINIT 2025 paper offloads in
 * its SCF loop (Sec. V: ":456 applying the Hamiltonian to a set of vectors"; the three
 * terms and their cost at :475; the non-local operator is Eq. 26 at :470; "multiple concurrent
 * Fourier transforms using an array of wave functions" at :436).  The paper prints no interface;
 * the entry points follow BASELINE.json `north_star` (dft_plan_create / dft_set_vloc /
 * dft_apply_h) in the concrete form of SURVEY.md section 8(b).  Conventions the paper is silent
 * on are the numbered "readings" of DESIGN.md section 3.
 *
 * General rules
 *   - every call returns a status code (0 = DFT_OK, negative = error); nothing throws or aborts
 *     across the boundary; on error, output arguments are left untouched and dft_last_error()
 *     holds a message (thread-local).
 *   - reals are double; complex numbers are interleaved (re, im) doubles; sizes are int32/int64.
 *   - "host" / "device" is stated for every pointer.  Host arrays are copied during the call and
 *     may be freed afterwards.  Device arrays stay owned by the caller.
 *   - no CPU fallback exists: without a CUDA device every call that needs one returns DFT_ERR_CUDA.
 *   - a plan may be used from one host thread and one stream at a time.
 */
#ifndef DFT_B200_H
#define DFT_B200_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dft_plan dft_plan; /* opaque; owns its device buffers */

enum {
  DFT_OK = 0,
  DFT_ERR_INVALID_ARG = -1,    /* null pointer, non-positive size, bad l/m/irad, singular lattice ... */
  DFT_ERR_GRID_TOO_SMALL = -2, /* some sphere point violates -floor(n/2) <= m <= floor((n-1)/2)     */
  DFT_ERR_TABLE_RANGE = -3,    /* max |k+G| exceeds (nq-1)*dq of a radial table                    */
  DFT_ERR_ALLOC = -4,          /* host or device allocation failed / workspace too small           */
  DFT_ERR_CUDA = -5,           /* CUDA runtime / driver error (message in dft_last_error)          */
  DFT_ERR_NOT_READY = -6,      /* dft_apply_h before dft_set_vloc                                  */
  DFT_ERR_UNSUPPORTED = -7     /* FFT length with a prime factor > 5, l > 2, ...                   */
};

/* One atom type's non-local projectors (Eq. 26, PAPER.md :470; readings 6-9).  All
 * pointers are HOST memory, copied by dft_plan_create.
 *   projector i (0 <= i < nlmn) has angular momentum l[i] in 0..2, real-harmonic index m[i] in
 *   -l..l and radial function irad[i] in 0..nrad-1.
 *   radial function r is tabulated on the uniform grid q_j = j*dq, j = 0..nq-1 as the cubic-
 *   spline pair f[r*nq + j] (values) and f2[r*nq + j] (second derivatives).                       */
typedef struct {
  int32_t nlmn;
  const int32_t *l, *m, *irad; /* [nlmn]      */
  int32_t nrad, nq;
  double dq;
  const double *f, *f2;        /* [nrad][nq]  */
} dft_proj_table;

/* Build a plan: the G-sphere of every k-point (S_k = {m : 1/2|k+G|^2 <= ecut}, ascending FFT-box
 * index; readings 1-3), the pruned-FFT schedules, and the materialised projector table
 * P[a,i](G) = F(|q|) Y_lm(q^) exp(-2 pi i (k+m).x_a) in device memory ("computed and stored in
 * memory", PAPER.md :479).  All pointer arguments are HOST memory.
 *   rprimd[9]   row i = lattice vector a_i in bohr (row-major)
 *   kpt         [nkpt][3] reduced coordinates; nkpt >= 1 (all k-points are applied in one batch)
 *   ecut        Hartree
 *   ngfft[3]    FFT box n1,n2,n3; each must factor into 2,3,5 and be <= 1024
 *   typat       [natom] type index 0..ntypat-1;   xred [natom][3] reduced positions
 *   tables      [ntypat]
 *   dij         [natom][nlmn_max][nlmn_max] real symmetric, row-major, nlmn_max = max_t nlmn;
 *               entries outside an atom's nlmn are ignored
 * natom may be 0 (no non-local term; tables/dij may then be NULL).
 * On success *out receives the plan.  Synchronises the device.                                   */
int dft_plan_create(dft_plan **out, const double rprimd[9], int32_t nkpt, const double *kpt,
                    double ecut, const int32_t ngfft[3], int32_t natom, const int32_t *typat,
                    const double *xred, int32_t ntypat, const dft_proj_table *tables,
                    const double *dij);

/* dft_plan_create followed by dft_plan_set_option(keys[i], values[i]) for i = 0 .. nopt-1, in that
 * order (keys: HOST array of nopt C strings, values: HOST array of nopt integers; nopt may be 0).
 * One option acts at creation time already: with "proj_mode" = 1 (the paper's "computed
 * on-the-fly" projectors, PAPER.md :477) the materialised [nproj][mpw] table is never allocated
 * nor filled, so a cell whose table does not fit in device memory (19.4 GB at c4, growing with
 * natom^2) can still be planned; the radial-table range check (DFT_ERR_TABLE_RANGE) is done all
 * the same.  Setting "proj_mode" = 0 later builds the table then.  Errors as dft_plan_create and
 * dft_plan_set_option; on any error no plan is returned.                                         */
int dft_plan_create_opts(dft_plan **out, const double rprimd[9], int32_t nkpt, const double *kpt,
                         double ecut, const int32_t ngfft[3], int32_t natom, const int32_t *typat,
                         const double *xred, int32_t ntypat, const dft_proj_table *tables,
                         const double *dij, int32_t nopt, const char *const *keys,
                         const int64_t *values);

/* Sizes.  Any output pointer may be NULL.  npw: HOST [nkpt].  mpw = max_k npw_k is the leading
 * dimension of psi/hpsi.  workspace_bytes_per_band: device scratch dft_apply_h needs per band of
 * a band chunk (see dft_set_workspace).                                                          */
int dft_plan_get_info(const dft_plan *p, int32_t *nkpt, int32_t *npw, int32_t *mpw,
                      int32_t *nproj, int64_t *workspace_bytes_per_band);

/* Copy the index maps of k-point ik to HOST arrays (any may be NULL): kg [npw][3] (integer
 * m1,m2,m3 of each plane wave), igfft [npw] (box index i1 + n1*(i2 + n2*i3), strictly increasing)
 * and kin [npw] = 1/2|k+G|^2.                                                                    */
int dft_plan_get_kg(const dft_plan *p, int32_t ik, int32_t *kg, int32_t *igfft, double *kin);

/* Copy the materialised projector table of k-point ik to a HOST array ptab [nproj][npw] complex
 * (test / inspection aid; the table of the largest cell is 19.4 GB).                             */
int dft_plan_get_projectors(const dft_plan *p, int32_t ik, double *ptab);

/* The same table copied to DEVICE memory ptab_dev [nproj][mpw] complex (rows padded with zeros beyond npw_k),
 * enqueued on `stream`: lets a caller run its own contraction on the identical projectors (bench.py's
 * vendor-library context figure).                                                                  */
int dft_plan_copy_projectors_device(const dft_plan *p, int32_t ik, double *ptab_dev, void *stream);

/* Replace D_ij (PAW: "from self-consistent terms", PAPER.md :473).  HOST [natom][nlmn_max]^2.
 * Synchronises the device first (work enqueued earlier by dft_apply_h on any stream still sees the old values),
 * then copies; later calls see the new ones.                                                     */
int dft_set_dij(dft_plan *p, const double *dij);

/* Set the local potential: V_r is DEVICE memory, [n3][n2][n1] doubles, i1 fastest.  It is copied
 * (pre-scaled by 1/N) on `stream` (a cudaStream_t passed as void*; NULL = default stream); V_r
 * may be reused once that stream has passed the call.                                            */
int dft_set_vloc(dft_plan *p, const double *V_r, void *stream);

/* Optional caller-owned DEVICE scratch (e.g. a torch tensor).  bytes must cover at least one band
 * chunk of one band; dft_apply_h then never allocates.  dev_ptr = NULL returns to plan-owned
 * scratch (allocated lazily, grown on demand).  256-byte alignment required.                     */
int dft_set_workspace(dft_plan *p, void *dev_ptr, int64_t bytes);

/* Scratch sizes for dft_set_workspace (either output may be NULL): *min_bytes = the smallest workspace dft_apply_h can
 * run with (one band of one k-point per launch); *full_bytes = the workspace with which `nband` bands per k-point go
 * through the FFT passes in ONE chunk on the fastest path (for several k-points that is the all-k-points-per-launch
 * path, whose layout is T1 [nkpt][nband][max_k t1] followed by T2 [nkpt][nband][max_k t2]).  Anything in between
 * is used as far as it goes (more, smaller launches).                                              */
int dft_plan_workspace_bytes(const dft_plan *p, int32_t nband, int64_t *min_bytes, int64_t *full_bytes);

/* Options: "band_chunk" (bands per FFT pass launch, > 0), "terms" (bit 0 kinetic, bit 1 local,
 * bit 2 non-local, bit 3 meta-GGA term; default 15), "splitk" (GEMM-1 K splits, 0 = automatic), "proj_mode" (0 = default: projector table materialised in
 * device memory; 1 = factorised projectors FY.S evaluated inside both GEMMs; the table is freed (and rebuilt when the option
 * returns to 0; dft_plan_get_projectors gives DFT_ERR_NOT_READY meanwhile); an atom's projectors are taken in blocks of 8; when the form-factor rows of all types (8
 * per block) exceed 32, consecutive types are served in groups of at most 32 rows, both GEMMs once per group; see also
 * dft_plan_create_opts, which never builds the table), "host_groups" (dft_apply_h_host only: band groups, default 6,
 * whose host<->device copies overlap the kernels of the neighbouring groups), "gemm_3m" (1 = default: three real
 * products per complex multiply-add in the projector GEMMs, 0 = four; same result up to rounding), "fft_path" (0 = automatic:
 * register-resident two-stage transforms where the box length factorises, their strided passes fed by a
 * TMA shared-memory ring, or - when one band's pruned working set fits one SM's shared memory - the whole local term
 * fused in ONE kernel; 1 = generic shared-memory Stockham kernels only; 2 = register-resident transforms without the
 * TMA ring; 3 = the fused small-box kernel (DFT_ERR_UNSUPPORTED if the plan does not fit); 4 = automatic without it;
 * 5 = its run-time-dispatched variant; all compute the same transform), "gemm_sym" (k = 0 only: the projector table is
 * symmetric under G -> -G, so both projector GEMMs of dft_apply_h can run as REAL GEMMs on the half sphere, 4 instead of
 * 6 flops per projector, plane wave and band, same result up to rounding, any D_ij; 0 = never, 1 = wherever possible,
 * 2 = default: when nproj * npw * nband >= 1e8; the first such call builds a second table of half the size),
 * "gemm_strassen" (with gemm_sym active: one level of Strassen's recursion on the two real GEMMs, 7/8 of their flops, same
 * result up to rounding; 0 = never, 1 = wherever nproj is a multiple of 16, 2 = default: for nproj * npw * nband >= 1e10;
 * builds nine block tables of a quarter of the half table each at the first such call),
 * "fft_c_split" (the middle FFT pass with two barrier domains per CTA where its tiles are 16 lines wide: 0 = never, 1 = wherever
 * possible, 2 = default: where both radices of the box length are >= 12, e.g. 180, 192, 225, 256; same results), "nl_tiny" (1 = default: cells with nproj <= 64 and nproj * npw * nband * nkpt <= 1e6 take ONE launch for the whole non-local
 * and kinetic part, one CTA per band, instead of GEMM-1, D_ij, GEMM-2; 0 = always the GEMM kernels),
 * "gamma_real" (1 = enable dft_apply_h_gamma, see there), "spinor_fused" (dft_apply_h_spinor: 1 = default, the 2 x 2 potential
 * multiplied inside the middle FFT pass where the register path serves the box; 0 = four scalar local applications).
 * Unknown key or bad value -> DFT_ERR_INVALID_ARG.  */
int dft_plan_set_option(dft_plan *p, const char *key, int64_t value);

/* hpsi = H psi for nband bands per k-point.  psi and hpsi are DEVICE memory, layout
 * [nkpt][nband][mpw] complex128 (16-byte aligned); entries ipw >= npw_k of psi must be finite and
 * do not influence the result; the same entries of hpsi are written as 0.  hpsi is overwritten;
 * psi is not modified; they must not overlap.  The call only ENQUEUES work on `stream`
 * (cudaStream_t as void*, NULL = default stream) and returns; it performs no host
 * synchronisation and no device->host traffic.  DFT_ERR_NOT_READY if dft_set_vloc was never
 * called (unless the local term is switched off with "terms").                                   */
int dft_apply_h(dft_plan *p, const double *psi, double *hpsi, int32_t nband, void *stream);

/* PAW overlap coefficients s^a_ij, HOST [natom][nlmn_max][nlmn_max] real symmetric (zero after
 * dft_plan_create): "the overlap operator S ... has the same structure" as Eq. 26 (PAPER.md :473).
 * Synchronises the device first, like dft_set_dij.                                                  */
int dft_set_sij(dft_plan *p, const double *sij);

/* spsi = S psi = psi + sum_a sum_ij |p_a,i> s^a_ij <p_a,j|psi> (PAPER.md :473), same layouts, stream and
 * pad-entry rules as dft_apply_h: GEMM-1, s_ij, GEMM-2 with a unit diagonal in its epilogue.        */
int dft_apply_s(dft_plan *p, const double *psi, double *spsi, int32_t nband, void *stream);

/* hpsi = H psi and spsi = S psi in one call, from ONE set of projections <p|psi> (PAPER.md :479-:485: keeping the
 * cprj and reusing them saves non-local operations): the five FFT passes, GEMM-1, then D_ij + GEMM-2 into hpsi and
 * s_ij + GEMM-2 (unit diagonal) into spsi -- three GEMMs instead of the four of dft_apply_h + dft_apply_s.  Arguments
 * and rules of dft_apply_h; spsi like hpsi; the non-local term must be on.                              */
int dft_apply_hs(dft_plan *p, const double *psi, double *hpsi, double *spsi, int32_t nband, void *stream);

/* cprj = <p_a,i|psi_n> (PAPER.md :477 "coefficients c_a,i,n,k ... cprj"): DEVICE output
 * [nkpt][nband][nproj] complex128, projector index fastest, atoms in order, i = 0..nlmn-1 inside an
 * atom.  GEMM-1 and the fixed-order split-K reduction only; enqueues on `stream`.                 */
int dft_get_cprj(dft_plan *p, const double *psi, double *cprj, int32_t nband, void *stream);

/* Density accumulation (Eq. 6, :140: n(r) = sum_nk w_nk |psi_nk(r)|^2; Eq. 3, :110 with
 * w_nk = 2 w_k f_nk):  rho[j] += sum_k sum_n weights[k][n] |psi_nk(r_j)|^2  on the FFT box, with
 * psi_nk(r_j) = sum_G c_nk(G) exp(+2 pi i G.r_j) (the unnormalised G->r transform of dft_apply_h; fold 1/Omega
 * and occupations into the weights).  psi: DEVICE [nkpt][nband][mpw]; weights: HOST [nkpt][nband], copied before
 * the call returns (one synchronisation of `stream`); rho: DEVICE [n3][n2][n1] doubles, i1 fastest, ACCUMULATED into (zero it first).  Runs the
 * scatter + x and y passes of dft_apply_h and the forward half of its z pass, summing over bands in registers
 * (no atomics, fixed order).  Any box the plan accepts is served (generic passes where an axis length has no two-radix
 * factorisation).  */
int dft_accumulate_density(dft_plan *p, const double *psi, const double *weights, double *rho, int32_t nband, void *stream);

/* Kinetic-energy density of the same equation (Eq. 6: tau(r) = 1/2 sum_nk w_nk |grad psi_nk(r)|^2):
 * tau[j] += 1/2 sum_k sum_n weights[k][n] sum_d |FFT[(k+G)_d c_nk](r_j)|^2, (k+G) Cartesian.  Same arguments,
 * layouts and rules as dft_accumulate_density (three density passes with the gradient factor fused into the scatter). */
int dft_accumulate_tau(dft_plan *p, const double *psi, const double *weights, double *tau, int32_t nband, void *stream);

/* Meta-GGA term of the Hamiltonian (Eq. 8, :152: "- 1/2 div( v_tau(r) grad )", v_tau = d f_xc / d tau, Eq. 9):
 * once set, dft_apply_h adds  1/2 sum_{d=x,y,z} (k+G)_d FFT^-1[ v_tau(r) FFT[ (k+G')_d psi ] ]  (three more local
 * applications whose diagonal factors are fused into the scatter and gather passes).  vtau_r: DEVICE
 * [n3][n2][n1] doubles like V_r of dft_set_vloc, copied on `stream`; NULL switches the term off.  Option "terms"
 * bit 3 (value 8) gates it.  Any box the plan accepts is served (the generic FFT passes carry the diagonal factors and
 * the accumulation too).                                                                            */
int dft_set_vtau(dft_plan *p, const double *vtau_r, void *stream);

/* Velocity-gauge vector potential (PAPER.md :340: in RT-TDDFT "the velocity gauge changes only the kinetic
 * term", -i grad -> -i grad + A(t)): while set, the kinetic diagonal of dft_apply_h / dft_chebyshev_filter is
 * 1/2 |k + G + A|^2 with A = a_cart[3] (HOST, Cartesian, atomic units).  The sphere (defined at A = 0) and
 * every other term are unchanged.  NULL or (0,0,0) switches it off.  Synchronises the device.        */
int dft_set_vector_potential(dft_plan *p, const double *a_cart);

/* Chebyshev filter (PAPER.md :458 "Chebyshev filtering algorithm ... filters the spectrum of the Hamiltonian",
 * :489 "mdeg_filter 10"; the paper prints no formula, this is the textbook three-term recurrence):
 *   T_0 = psi,  T_1 = (H - center) T_0 / halfwidth,  T_{j+1} = 2 (H - center) T_j / halfwidth - T_{j-1},
 * psi := T_degree, i.e. the Chebyshev polynomial of the first kind of (H - center)/halfwidth applied to psi
 * (center, halfwidth: centre and half-width of the part of the spectrum to damp, Hartree; halfwidth > 0).
 * psi: DEVICE in/out, layout of dft_apply_h; work: DEVICE scratch of TWO psi-sized arrays
 * (2 * nkpt*nband*mpw complex128, 16-byte aligned), contents undefined afterwards.  `degree` applications
 * of H; the recurrence combination is done where GEMM-2's epilogue stores H T_j (no extra passes).
 * Pad entries ipw >= npw_k of the result are 0.  Enqueues on `stream`, no host synchronisation.     */
int dft_chebyshev_filter(dft_plan *p, double *psi, double *work, int32_t nband, int32_t degree, double center,
                         double halfwidth, void *stream);

/* Gamma-point real-symmetry storage (PAPER.md :407 "time-reversal symmetry"; reading 26).
 * Enabled by dft_plan_set_option(p, "gamma_real", 1) on a plan with ONE k-point k = (0,0,0) whose sphere holds -G for
 * every G; DFT_ERR_UNSUPPORTED otherwise, DFT_ERR_INVALID_ARG if D_ij (now or in a later dft_set_dij) couples
 * projectors of different l-parity (H would not commute with time reversal).  A band whose psi(r) is real has
 * c(-G) = conj(c(G)); only the plane waves with m3 > 0, or m3 = 0 and m2 > 0, or m3 = m2 = 0 and m1 >= 0 are stored, in the
 * order of the full list (ascending box index; G = 0 first), nhalf = (npw + 1)/2 of them.
 * dft_plan_get_kg_gamma: HOST outputs like dft_plan_get_kg for the stored half (any pointer may be NULL).
 * dft_apply_h_gamma: psi, hpsi DEVICE [nband][nhalf] complex128, 16-byte aligned, not aliased; hpsi = restriction of
 * H applied to the symmetric vector (Im psi(0) is ignored, Im hpsi(0) = 0).  Two bands share one complex FFT round
 * trip and both projector GEMMs are REAL GEMMs on the half sphere.  Honours option "terms" (bits 0-2); enqueues on
 * `stream` without host synchronisation (scratch is allocated at the first call of a given size).              */
int dft_plan_get_kg_gamma(const dft_plan *p, int32_t *nhalf, int32_t *kg, int32_t *igfft, double *kin);
int dft_apply_h_gamma(dft_plan *p, const double *psi, double *hpsi, int32_t nband, void *stream);
/* dft_chebyshev_filter in Gamma storage: psi DEVICE in/out [nband][nhalf], work DEVICE 2 * nband * nhalf complex128; the
 * same recurrence with dft_apply_h_gamma as H (for degree >= 1 the result has Im psi(0) = 0).                        */
int dft_chebyshev_filter_gamma(dft_plan *p, double *psi, double *work, int32_t nband, int32_t degree, double center,
                               double halfwidth, void *stream);

/* Two-component spinors (PAPER.md :448 "all types of magnetism": non-collinear magnetism, spin-orbit coupling;
 * SURVEY.md 8(f) row 4; reading 27).  psi = (psi_up, psi_dn): DEVICE [nkpt][nband][2][mpw] complex128.
 *   H = kin (x) 1 + FFT^-1[ V^{ss'}(r) FFT[psi_s'] ] + sum_a sum_ij sum_ss' |p_a,i> D^{a,ss'}_ij <p_a,j|
 * dft_set_vloc_spinor: v4 DEVICE [4][n3][n2][n1] doubles = V_upup, V_dndn, Re V_updn, Im V_updn (V_dnup = conj V_updn),
 * copied on `stream` (pre-scaled by 1/N, as the four fields and as their Pauli components V0, Vx, Vy, Vz).
 * dft_set_dij_spinor: dspin HOST [natom][2][2][lmax][lmax] complex128 (re, im interleaved), Hermitian in
 * ((s,i),(s',j)); NULL returns to the scalar D_ij of dft_set_dij on both components.  Synchronises the device.
 * dft_apply_h_spinor: rules of dft_apply_h; DFT_ERR_NOT_READY before dft_set_vloc_spinor while the local term is on.
 * The GEMMs see 2 nband bands.  The local term is one application with the 2 x 2 matrix multiplied in the middle FFT pass
 * where the five-pass register path serves the box (option "spinor_fused", default 1), else four scalar local
 * applications (V0 psi + sum_mu V_mu sigma_mu psi), which every box the plan accepts can take. */
int dft_set_vloc_spinor(dft_plan *p, const double *v4_dev, void *stream);
int dft_set_dij_spinor(dft_plan *p, const double *dspin_host);
int dft_apply_h_spinor(dft_plan *p, const double *psi, double *hpsi, int32_t nband, void *stream);

/* The local term alone, hpsi = FFT^-1[ V_loc(r) FFT[psi] ] (PAPER.md :475; what dft_apply_h computes with option
 * "terms" = 2), for callers that cannot allocate device memory: code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc.  Arguments, layouts, pad-entry rule and stream semantics of dft_apply_h.  The call
 * performs no cudaMalloc / cudaFree and calls no allocating library routine, whatever the band count: the pass-to-pass
 * scratch of the five FFT passes is a static device array of DFT_NOALLOC_SCRATCH_BYTES inside the library (every GPU that
 * loads the library holds it until the process exits), and the bands go through in chunks that fit it (always the five-pass
 * path, also for boxes where dft_apply_h would take the fused small-box kernel).  DFT_ERR_ALLOC if the scratch of ONE band,
 * (ncol*n1 + nplane*n2*n1) * 16 bytes, exceeds the array (boxes above about 190^3; c4 at 180^3 needs 58.5 MB);
 * DFT_ERR_NOT_READY before dft_set_vloc.  The array is shared by all plans and calls on a GPU and keeps the last call's
 * contents (nothing in it needs to start at zero): calls that overlap on the GPU -- different streams without an event
 * between them -- race on it and give wrong results; calls on one stream are safe.                                  */
#define DFT_NOALLOC_SCRATCH_BYTES (64ll << 20)
int dft_apply_vloc_noalloc(dft_plan *p, const double *psi, double *hpsi, int32_t nband, void *stream);

/* Same, with HOST psi/hpsi (pageable or pinned): copies psi to the device in band blocks, applies
 * H, copies the result back, and returns after the last copy has completed.                      */
int dft_apply_h_host(dft_plan *p, const double *psi_host, double *hpsi_host, int32_t nband);

/* Number of kernel launches the last dft_apply_h / dft_apply_h_host of this plan enqueued.       */
int64_t dft_plan_last_launches(const dft_plan *p);

/* Device time of one named kernel group summed over the last apply is not tracked here; use CUDA
 * events around dft_apply_h, or the bench-only hook below: when `on` != 0 every kernel group of
 * later applies is bracketed by CUDA events on the launching stream; dft_plan_phase_ms then
 * returns (after synchronising) the accumulated milliseconds of phase i and resets it.
 * Phases: 0 fft_A(scatter) 1 fft_B 2 fft_C*V*C^-1 3 fft_B^-1 4 fft_A^-1(gather) 5 gemm1 6 dij
 * 7 gemm2(+kinetic) 8 fused small-box local term 9 pack/unpack (Gamma storage) and sigma products (spinors). */
int dft_plan_set_timing(dft_plan *p, int32_t on);
int dft_plan_phase_ms(dft_plan *p, int32_t phase, double *ms, int64_t *launches);

int dft_plan_destroy(dft_plan *p);

const char *dft_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DFT_B200_H */
