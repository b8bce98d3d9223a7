// nonlocal.cu -- K3: the non-local operator of Eq. 26 (PAPER.md :470) plus the kinetic diagonal,
//
//   (H_nl psi_b)(G) = sum_a sum_ij p_{a,i}(G) D^a_ij sum_G' conj(p_{a,j}(G')) psi_b(G'),
//
// in the BLAS-3 formulation the paper describes for stored projectors (:479 "matrix-matrix
// multiplications"), SURVEY.md 8(a) steps S8-S10:
//
//   GEMM-1  cprj[p][b]  = sum_G conj(P[p][G]) psi[b][G]          M = nproj, N = nband, K = npw   (split-K)
//   D_ij    c'[b][a,i]  = sum_j D^a_ij cprj[a,j][b]              (also reduces the split-K partials, fixed order)
//   GEMM-2  hpsi[b][G]  = (V_loc psi)[b][G] + kin[G] psi[b][G] + sum_p P[p][G] c'[b][p]
//                                                                M = npw, N = nband, K = nproj   (kinetic epilogue)
//
// Both GEMMs run on the FP64 tensor pipe (mma.sync m8n8k4 f64 -> DMMA.8x8x4; sm_100a has no
// tcgen05 FP64 kind) with operands staged by TMA (cp.async.bulk.tensor, 128-byte swizzle) through an
// mbarrier ring filled by one elected thread.  Complex arithmetic is 4 real DMMAs per
// 8x8x4 complex block: the (re, im) halves of a 16-byte element are the A/B fragments of two
// different k-groups, so there is no operand re-packing and no wasted tensor work.
//
// Shared-memory layout of every operand tile: rows of 128 bytes (8 complex numbers), TMA
// SWIZZLE_128B (16-byte chunk c of row r stored at chunk c ^ (r & 7)).  A DMMA k-group takes the
// complex numbers {kg, kg+2, kg+4, kg+6} of a row (kg = 0, 1), which makes every LDS.128 of a
// quarter-warp hit eight distinct chunks (conflict-free).
#include <stdio.h>

#include "internal.h"
#include "ptx.cuh"

namespace dftb200 {

constexpr int NL_BM = 128;        // rows of the M operand per CTA tile
constexpr int NL_BN = 64;         // bands per CTA tile
constexpr int NL_STAGES = 6;
constexpr int NL_PREFETCH = NL_STAGES - 2;   // TMA runs this many slabs ahead of the MMA
constexpr int NL_CONSUMERS = 8;   // warps: 4 (M) x 2 (N), 32 x 32 complex outputs each
// 8 warps = 2 per SM sub-partition, so each thread may hold up to 255 registers (the 64 complex
// accumulators alone are 128); a ninth (producer) warp would put 3 warps on one sub-partition and cap
// the kernel at 168.  Lane 0 of warp 0 therefore also issues the TMA loads, NL_PREFETCH slabs ahead,
// into a stage every warp released two iterations earlier (so it practically never waits).
constexpr int NL_THREADS = NL_CONSUMERS * 32;
// The four-product kernels add a producer warpgroup (warps 8-11, lane 0 of warp 8 issues the TMA loads): with the loads
// issued by a consumer the whole ring was paced by that one warp, and the warps that ran ahead of it starved at the full
// barrier (ncu: 16 % of the samples of the real GEMM-2 of the symmetric-table path; 91.5 % DMMA).  Twelve warps would cap
// every thread at 168 registers, so the producer group gives its registers back (setmaxnreg 24) and the two consumer
// groups take 232 each: 2 x 32 x 232 + 32 x 24 = 15 616 of the 16 384 registers of a sub-partition.
constexpr int NL_THREADS_P = NL_THREADS + 128;
__device__ __forceinline__ void reg_dealloc_producer() { asm volatile("setmaxnreg.dec.sync.aligned.u32 24;"); }
__device__ __forceinline__ void reg_alloc_consumer() { asm volatile("setmaxnreg.inc.sync.aligned.u32 232;"); }
constexpr int NL_STAGE_A = NL_BM * 128;   // 16 KB
constexpr int NL_STAGE_B = NL_BN * 128;   // 8 KB
constexpr int NL_STAGE_BYTES = NL_STAGE_A + NL_STAGE_B;
constexpr int NL_SMEM = NL_STAGES * NL_STAGE_BYTES + 1024 + 256;

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

struct Gemm1Params {
  int nproj, nband, nslab, nsplit, slabs_per_split, tiles_m, tiles_n;
  double2 *part;   // [nkpt][nsplit][nproj][nband]
};
struct Gemm2Params {
  int nproj, nband, mpw, nslab, tiles_n, accumulate, with_kin, with_nl;
  const int32_t *npw;     // [nkpt] device
  const double *const *kin;   // [nkpt] device pointers
  const double2 *psi; double2 *hpsi;   // [nkpt][nband][mpw]
  // optional recurrence combination of the epilogue (Chebyshev filter): out = sh * (H psi) + sy * psi + sx * xprev
  int cheb;
  double sh, sy, sx;
  const double2 *xprev;                // [nkpt][nband][mpw], read only where sx != 0
  int raw;                             // gemm2_kernel<true> only: 1 = an intermediate product (Strassen block): keep Im of row 0
};

// The MMA main loop shared by both GEMMs.  MODE 1: acc += conj(A) B (GEMM-1); MODE 2: acc += A B.
// As/Bs: one stage; A rows are addressed as a_row0 + mb*a_mb_stride bytes (+ row-in-block handled
// by the caller-provided offsets).
// REAL (Gamma-point storage, gamma.cu): MODE 1 keeps only Re(conj(A) B) = A_r B_r + A_i B_i, a REAL GEMM over the
// interleaved (re, im) doubles; MODE 2 takes B as real (its imaginary halves are zero): Re += A_r B_r, Im += A_i B_r.
// Either way two of the four DMMA sets remain.
// MB: 8-row blocks of the M operand per warp (MODE 1 only: 4 = the 128-row tile, 2 / 1 = skinny tiles of 64 / 32 rows for
// systems with few projectors).
template <int MODE, bool REAL = false, int MB = 4>
__device__ __forceinline__ void mma_stage(const unsigned char *As, const unsigned char *Bs, int wm, int wn, int lane,
                                          double (&cre)[4][4][2], double (&cim)[4][4][2]) {
  const int i = lane >> 2, j = lane & 3;
#pragma unroll
  for (int kg = 0; kg < 2; kg++) {
    double ar[4], ai[4], br[4], bi[4];
    if (MODE == 1) {
      // A tile [128 rows p][8 complex g]: row = wm*32 + mb*8 + i, chunk (2j+kg) ^ i
      const unsigned char *a0 = As + (wm * 8 * MB + i) * 128 + (((2 * j + kg) ^ i) << 4);
#pragma unroll
      for (int mb = 0; mb < MB; mb++) {
        double2 v = *reinterpret_cast<const double2 *>(a0 + mb * 8 * 128);
        ar[mb] = v.x; ai[mb] = v.y;
      }
    } else {
      // A tile [16 g-blocks][8 rows p][8 complex g]: block t = wm*4 + mb, row p = 2j+kg, chunk i ^ p
      const int pr = 2 * j + kg;
      const unsigned char *a0 = As + (wm * 4) * 1024 + pr * 128 + ((i ^ pr) << 4);
#pragma unroll
      for (int mb = 0; mb < MB; mb++) {
        double2 v = *reinterpret_cast<const double2 *>(a0 + mb * 1024);
        ar[mb] = v.x; ai[mb] = v.y;
      }
    }
    const unsigned char *b0 = Bs + (wn * 32 + i) * 128 + (((2 * j + kg) ^ i) << 4);
#pragma unroll
    for (int nb = 0; nb < 4; nb++) {
      double2 v = *reinterpret_cast<const double2 *>(b0 + nb * 8 * 128);
      br[nb] = v.x; bi[nb] = v.y;
    }
#pragma unroll
    for (int mb = 0; mb < MB; mb++)
#pragma unroll
      for (int nb = 0; nb < 4; nb++) dmma(cre[mb][nb][0], cre[mb][nb][1], ar[mb], br[nb]);
    if (REAL) {
#pragma unroll
      for (int mb = 0; mb < MB; mb++)
#pragma unroll
        for (int nb = 0; nb < 4; nb++) {
          if (MODE == 1) dmma(cre[mb][nb][0], cre[mb][nb][1], ai[mb], bi[nb]);
          else dmma(cim[mb][nb][0], cim[mb][nb][1], ai[mb], br[nb]);
        }
      continue;
    }
#pragma unroll
    for (int mb = 0; mb < MB; mb++)
#pragma unroll
      for (int nb = 0; nb < 4; nb++) dmma(cim[mb][nb][0], cim[mb][nb][1], ar[mb], bi[nb]);
    if (MODE == 1) {
      // conj(p) psi: re += p_i psi_i, im -= p_i psi_r
#pragma unroll
      for (int mb = 0; mb < MB; mb++)
#pragma unroll
        for (int nb = 0; nb < 4; nb++) dmma(cre[mb][nb][0], cre[mb][nb][1], ai[mb], bi[nb]);
#pragma unroll
      for (int mb = 0; mb < MB; mb++) ai[mb] = -ai[mb];
#pragma unroll
      for (int mb = 0; mb < MB; mb++)
#pragma unroll
        for (int nb = 0; nb < 4; nb++) dmma(cim[mb][nb][0], cim[mb][nb][1], ai[mb], br[nb]);
    } else {
      // p c: im += p_i c_r, re -= p_i c_i
#pragma unroll
      for (int mb = 0; mb < MB; mb++)
#pragma unroll
        for (int nb = 0; nb < 4; nb++) dmma(cim[mb][nb][0], cim[mb][nb][1], ai[mb], br[nb]);
#pragma unroll
      for (int nb = 0; nb < 4; nb++) bi[nb] = -bi[nb];
#pragma unroll
      for (int mb = 0; mb < MB; mb++)
#pragma unroll
        for (int nb = 0; nb < 4; nb++) dmma(cre[mb][nb][0], cre[mb][nb][1], ai[mb], bi[nb]);
    }
  }
}

struct Pipe {
  unsigned char *tiles;
  uint64_t *full, *empty;
};
__device__ __forceinline__ Pipe pipe_setup(unsigned char *smem_raw) {
  Pipe P;
  // 1024-byte alignment (128-byte swizzle atom) by an offset on the __shared__ array itself, so the
  // compiler keeps the shared address space (LDS/STS, not generic LD/ST)
  P.tiles = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  P.full = reinterpret_cast<uint64_t *>(P.tiles + NL_STAGES * NL_STAGE_BYTES);
  P.empty = P.full + NL_STAGES;
  if (threadIdx.x == 0) {
    for (int s = 0; s < NL_STAGES; s++) { mbar_init(&P.full[s], 1); mbar_init(&P.empty[s], NL_CONSUMERS); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  return P;
}

// ---------------------------------------------------------------- GEMM-1: projection (split-K partials)
// grid: (tiles_m*tiles_n, nsplit, nkpt)
template <bool REAL, int MB = 4>
__global__ void __launch_bounds__(NL_THREADS_P, 1)
gemm1_kernel(const __grid_constant__ CUtensorMap mapP, const __grid_constant__ CUtensorMap mapPsi, Gemm1Params Q) {
  constexpr int BM = 32 * MB;            // rows of P per CTA tile (the TMA box of mapP has BM rows)
  extern __shared__ unsigned char smem_raw[];
  Pipe P = pipe_setup(smem_raw);
  const int tile = blockIdx.x, tn = tile % Q.tiles_n, tm = tile / Q.tiles_n;
  const int split = blockIdx.y, ik = blockIdx.z;
  const int s0 = split * Q.slabs_per_split;
  int ns = Q.nslab - s0; if (ns > Q.slabs_per_split) ns = Q.slabs_per_split; if (ns < 0) ns = 0;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  auto issue = [&](int j) {
    int s = j % NL_STAGES;
    if (j >= NL_STAGES) mbar_wait(&P.empty[s], ((j / NL_STAGES) - 1) & 1);
    unsigned char *st = P.tiles + s * NL_STAGE_BYTES;
    mbar_expect_tx(&P.full[s], BM * 128 + NL_STAGE_B);
    tma_load_3d(st, &mapP, &P.full[s], (s0 + j) * 16, tm * BM, ik);
    tma_load_3d(st + NL_STAGE_A, &mapPsi, &P.full[s], (s0 + j) * 16, tn * NL_BN, ik);
  };
  if (warp >= NL_CONSUMERS) {      // the producer group: keeps the whole ring in flight, independent of any consumer's pace
    reg_dealloc_producer();
    if (warp == NL_CONSUMERS && lane == 0)
      for (int j = 0; j < ns; j++) issue(j);
    return;
  }
  reg_alloc_consumer();
  const int wm = warp >> 1, wn = warp & 1;
  double cre[4][4][2], cim[4][4][2];
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int b = 0; b < 4; b++) { cre[a][b][0] = cre[a][b][1] = cim[a][b][0] = cim[a][b][1] = 0.0; }
  for (int it = 0; it < ns; it++) {
    int s = it % NL_STAGES;
    mbar_wait(&P.full[s], (it / NL_STAGES) & 1);
    const unsigned char *st = P.tiles + s * NL_STAGE_BYTES;
    mma_stage<1, REAL, MB>(st, st + NL_STAGE_A, wm, wn, lane, cre, cim);
    __syncwarp();
    if (lane == 0) mbar_arrive(&P.empty[s]);
  }
  // partial[ik][split][p][b] complex (REAL: real); thread holds rows p = lane/4, bands 2*(lane%4)+{0,1} of each 8x8 block
  double2 *out = Q.part + ((size_t)(ik * Q.nsplit + split) * Q.nproj) * Q.nband;
  double *outr = reinterpret_cast<double *>(Q.part) + ((size_t)(ik * Q.nsplit + split) * Q.nproj) * Q.nband;
  const int i = lane >> 2, j = lane & 3;
#pragma unroll
  for (int mb = 0; mb < MB; mb++) {
    int pr = tm * BM + wm * 8 * MB + mb * 8 + i;
    if (pr >= Q.nproj) continue;
#pragma unroll
    for (int nb = 0; nb < 4; nb++) {
      int b = tn * NL_BN + wn * 32 + nb * 8 + 2 * j;
      if (REAL) {
        double *d = outr + (size_t)pr * Q.nband + b;
        if (b < Q.nband) d[0] = cre[mb][nb][0];
        if (b + 1 < Q.nband) d[1] = cre[mb][nb][1];
      } else {
        double2 *d = out + (size_t)pr * Q.nband + b;
        if (b < Q.nband) d[0] = make_double2(cre[mb][nb][0], cim[mb][nb][0]);
        if (b + 1 < Q.nband) d[1] = make_double2(cre[mb][nb][1], cim[mb][nb][1]);
      }
    }
  }
}

// ---------------------------------------------------------------- D_ij + split-K reduction
// c'[ik][b][first_a + i] = sum_j D^a_ij sum_s part[ik][s][first_a + j][b];  one thread per (b, a, ik), b fastest
constexpr int DIJ_MAXL = 16;
// blockDim = (DIJ_BX bands, DIJ_YS): the split-K partials are summed by DIJ_YS groups of threads, group y taking the splits
// y, y + DIJ_YS, ... (with a few dozen splits, one thread per band and 128 bands per CTA most of the chip was idle: 73 us at c1),
// then added up in shared memory in the fixed order y = 0, 1, ...; group 0 applies D.
constexpr int DIJ_YS = 4, DIJ_BX = 32;
__global__ void __launch_bounds__(DIJ_BX * DIJ_YS)
dij_kernel(const double2 *__restrict__ part, double2 *__restrict__ cpr, const double *__restrict__ dij,
           const int32_t *__restrict__ typat, const int32_t *__restrict__ nlmn,
           const int32_t *__restrict__ atom_first, int natom, int lmax, int nproj, int nband, int nsplit) {
  __shared__ double2 red[DIJ_YS - 1][DIJ_MAXL][DIJ_BX];
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int b = blockIdx.x * DIJ_BX + tx, a = blockIdx.y, ik = blockIdx.z;
  const bool live = b < nband;
  int nl = nlmn[typat[a]], first = atom_first[a];
  double2 c[DIJ_MAXL];
  for (int jj = 0; jj < nl; jj++) c[jj] = make_double2(0.0, 0.0);
  // splits outer, projectors inner: the nl loads of one split are independent (fixed summation order per projector)
  if (live)
    for (int s = ty; s < nsplit; s += DIJ_YS) {
      const double2 *src = part + ((size_t)(ik * nsplit + s) * nproj + first) * nband + b;
#pragma unroll 4
      for (int jj = 0; jj < nl; jj++) {
        double2 v = src[(size_t)jj * nband];
        c[jj].x += v.x; c[jj].y += v.y;
      }
    }
  if (ty > 0)
    for (int jj = 0; jj < nl; jj++) red[ty - 1][jj][tx] = c[jj];
  __syncthreads();
  if (ty > 0 || !live) return;
  for (int y = 0; y < DIJ_YS - 1; y++)
    for (int jj = 0; jj < nl; jj++) { const double2 v = red[y][jj][tx]; c[jj].x += v.x; c[jj].y += v.y; }
  double2 *dst = cpr + ((size_t)ik * nband + b) * nproj + first;
  if (!dij) {   // no D: the reduced projections <p|psi> themselves (dft_get_cprj)
    for (int ii = 0; ii < nl; ii++) dst[ii] = c[ii];
    return;
  }
  const double *D = dij + (size_t)a * lmax * lmax;
  for (int ii = 0; ii < nl; ii++) {
    double sr = 0.0, si = 0.0;
    for (int jj = 0; jj < nl; jj++) { double d = D[ii * lmax + jj]; sr += d * c[jj].x; si += d * c[jj].y; }
    dst[ii] = make_double2(sr, si);
  }
}

// Gamma storage (reading 26): the real GEMM-1 gives S_j = sum_half (Pt_r psi_r + Pt_i psi_i) with Pt = i^(l odd) p;
// the projection of the symmetric vector is <p_j|psi> = i^(l_j odd) r_j with r_j = 2 S_j - Pt_r,j(0) Re psi(0) (the G = 0 term
// is its own partner).  D couples projectors of equal l-parity only, so c'_i = i^(l_i odd) sum_j D_ij r_j, stored as the
// real number sum_j D_ij r_j (imaginary half 0) for the real GEMM-2 on the same rotated table.
__global__ void dij_gamma_kernel(const double *__restrict__ part, double2 *__restrict__ cpr, const double *__restrict__ dij,
                                 const int32_t *__restrict__ typat, const int32_t *__restrict__ nlmn,
                                 const int32_t *__restrict__ atom_first, const int32_t *__restrict__ rowpar,
                                 const double *__restrict__ p0, const double2 *__restrict__ psi, int mpw, int lmax, int nproj,
                                 int nband, int nsplit) {
  int b = blockIdx.x * blockDim.x + threadIdx.x, a = blockIdx.y;
  if (b >= nband) return;
  int nl = nlmn[typat[a]], first = atom_first[a];
  const double c0 = psi[(size_t)b * mpw].x;
  double r[DIJ_MAXL];
  for (int jj = 0; jj < nl; jj++) {
    double sr = 0.0;
    for (int s = 0; s < nsplit; s++) sr += part[((size_t)s * nproj + first + jj) * nband + b];
    r[jj] = 2.0 * sr - p0[first + jj] * c0;
  }
  double2 *dst = cpr + (size_t)b * nproj + first;
  const double *D = dij + (size_t)a * lmax * lmax;
  const int32_t *par = rowpar + (size_t)a * lmax;
  for (int ii = 0; ii < nl; ii++) {
    double sr = 0.0;
    for (int jj = 0; jj < nl; jj++)
      if (par[ii] == par[jj]) sr += D[ii * lmax + jj] * r[jj];
    dst[ii] = make_double2(sr, 0.0);
  }
}

// Spinors (reading 27): rows 2 b + s of the projections are the two components of band b;
// c'[2b + s][a,i] = sum_s' sum_j D^{a,s s'}_ij <p_a,j|psi_{b,s'}>, D complex [natom][2][2][lmax][lmax]
__global__ void dij_spinor_kernel(const double2 *__restrict__ part, double2 *__restrict__ cpr, const double2 *__restrict__ dspin,
                                  const int32_t *__restrict__ typat, const int32_t *__restrict__ nlmn,
                                  const int32_t *__restrict__ atom_first, int lmax, int nproj, int nband2, int nsplit) {
  int b = blockIdx.x * blockDim.x + threadIdx.x, a = blockIdx.y, ik = blockIdx.z;
  if (2 * b >= nband2) return;
  int nl = nlmn[typat[a]], first = atom_first[a];
  double2 c[2][DIJ_MAXL];
  for (int sp = 0; sp < 2; sp++)
    for (int jj = 0; jj < nl; jj++) {
      double sr = 0.0, si = 0.0;
      for (int s = 0; s < nsplit; s++) {
        double2 v = part[((size_t)(ik * nsplit + s) * nproj + first + jj) * nband2 + 2 * b + sp];
        sr += v.x; si += v.y;
      }
      c[sp][jj] = make_double2(sr, si);
    }
  for (int sp = 0; sp < 2; sp++) {
    double2 *dst = cpr + ((size_t)ik * nband2 + 2 * b + sp) * nproj + first;
    for (int ii = 0; ii < nl; ii++) {
      double sr = 0.0, si = 0.0;
      for (int s2 = 0; s2 < 2; s2++) {
        const double2 *D = dspin + (((size_t)a * 2 + sp) * 2 + s2) * lmax * lmax + (size_t)ii * lmax;
        for (int jj = 0; jj < nl; jj++) {
          const double2 d = D[jj], v = c[s2][jj];
          sr += d.x * v.x - d.y * v.y; si += d.x * v.y + d.y * v.x;
        }
      }
      dst[ii] = make_double2(sr, si);
    }
  }
}

// ---------------------------------------------------------------- GEMM-2: back-projection + kinetic epilogue
// grid: (tiles_n * tiles_m, 1, nkpt), band tiles fastest so that concurrent CTAs share a slab of P in L2
template <bool REAL>
__device__ __forceinline__ void gemm2_body(const CUtensorMap *mapP, const CUtensorMap *mapC, const Gemm2Params &Q) {
  extern __shared__ unsigned char smem_raw[];
  Pipe P = pipe_setup(smem_raw);
  const int tn = blockIdx.x % Q.tiles_n, tm = blockIdx.x / Q.tiles_n, ik = blockIdx.z;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int ns = Q.with_nl ? Q.nslab : 0;
  auto issue = [&](int j) {
    int s = j % NL_STAGES;
    if (j >= NL_STAGES) mbar_wait(&P.empty[s], ((j / NL_STAGES) - 1) & 1);
    unsigned char *st = P.tiles + s * NL_STAGE_BYTES;
    mbar_expect_tx(&P.full[s], NL_STAGE_BYTES);
    // one box {16 doubles, 8 projector rows, 16 g-blocks}: lands as [g-block][p][8 complex], 128-byte swizzled
    tma_load_4d(st, mapP, &P.full[s], 0, j * 8, tm * (NL_BM / 8), ik);
    tma_load_3d(st + NL_STAGE_A, mapC, &P.full[s], j * 16, tn * NL_BN, ik);
  };
  if (warp >= NL_CONSUMERS) {      // the producer group
    reg_dealloc_producer();
    if (warp == NL_CONSUMERS && lane == 0)
      for (int j = 0; j < ns; j++) issue(j);
    return;
  }
  reg_alloc_consumer();
  const int wm = warp >> 1, wn = warp & 1;
  double cre[4][4][2], cim[4][4][2];
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int b = 0; b < 4; b++) { cre[a][b][0] = cre[a][b][1] = cim[a][b][0] = cim[a][b][1] = 0.0; }
  for (int it = 0; it < ns; it++) {
    int s = it % NL_STAGES;
    mbar_wait(&P.full[s], (it / NL_STAGES) & 1);
    const unsigned char *st = P.tiles + s * NL_STAGE_BYTES;
    mma_stage<2, REAL>(st, st + NL_STAGE_A, wm, wn, lane, cre, cim);
    __syncwarp();
    if (lane == 0) mbar_arrive(&P.empty[s]);
  }
  // epilogue: hpsi[b][g] = (V_loc psi)[b][g] + kin[g] psi[b][g] + acc;  rows g = lane/4, bands 2*(lane%4)+{0,1}
  const int npw = Q.npw[ik];
  const double *kin = Q.kin[ik];
  const double2 *psi = Q.psi + (size_t)ik * Q.nband * Q.mpw;
  double2 *hpsi = Q.hpsi + (size_t)ik * Q.nband * Q.mpw;
  const int i = lane >> 2, j = lane & 3;
#pragma unroll
  for (int mb = 0; mb < 4; mb++) {
    int g = tm * NL_BM + wm * 32 + mb * 8 + i;
    if (g >= npw) continue;
    double kg = Q.with_kin ? kin[g] : 0.0;
#pragma unroll
    for (int nb = 0; nb < 4; nb++) {
#pragma unroll
      for (int e = 0; e < 2; e++) {
        int b = tn * NL_BN + wn * 32 + nb * 8 + 2 * j + e;
        if (b >= Q.nband) continue;
        size_t off = (size_t)b * Q.mpw + g;
        double2 r = make_double2(cre[mb][nb][e], cim[mb][nb][e]);
        if (Q.with_kin) { double2 x = psi[off]; r.x += kg * x.x; r.y += kg * x.y; }
        if (Q.accumulate) { double2 h = hpsi[off]; r.x += h.x; r.y += h.y; }
        if (Q.cheb) {
          double2 y = psi[off], xp = Q.sx != 0.0 ? Q.xprev[(size_t)ik * Q.nband * Q.mpw + off] : make_double2(0.0, 0.0);
          r.x = Q.sh * r.x + Q.sy * y.x + Q.sx * xp.x; r.y = Q.sh * r.y + Q.sy * y.y + Q.sx * xp.y;
        }
        if (REAL && g == 0 && !Q.raw) r.y = 0.0;     // Gamma storage: c(G = 0) is real (reading 26)
        hpsi[off] = r;
      }
    }
  }
}

template <bool REAL>
__global__ void __launch_bounds__(NL_THREADS_P, 1)
gemm2_kernel(const __grid_constant__ CUtensorMap mapP, const __grid_constant__ CUtensorMap mapC, const __grid_constant__ Gemm2Params Q) {
  gemm2_body<REAL>(&mapP, &mapC, Q);
}

// Several independent products of the same shape in ONE launch (the seven back-projections of the Strassen level):
// blockIdx.y picks the product.  Seven launches of 31.2 waves each leave the chip a quarter full for one tile time at the
// end of every launch (0.4 ms of 17.4 at c4, the difference between the 96.8 % DMMA utilisation of GEMM-2 and the 98.2 % of
// GEMM-1, whose split-K factor is chosen for whole waves); one launch of 218.7 waves has one such tail.
constexpr int NL_MAXPROD = 7;
struct Gemm2Multi {
  CUtensorMap mapP[NL_MAXPROD], mapC[NL_MAXPROD];
  double2 *out[NL_MAXPROD];
};
template <bool REAL>
__global__ void __launch_bounds__(NL_THREADS_P, 1)
gemm2_multi_kernel(const __grid_constant__ Gemm2Multi M, const __grid_constant__ Gemm2Params Q0) {
  Gemm2Params Q = Q0;
  Q.psi = M.out[blockIdx.y]; Q.hpsi = M.out[blockIdx.y];
  gemm2_body<REAL>(&M.mapP[blockIdx.y], &M.mapC[blockIdx.y], Q);
}

// ---------------------------------------------------------------- 3M variant of both GEMMs
// A complex product needs only three real products (Gauss / "3M", exact up to rounding order):
//   a b       (GEMM-2):  k1 = (a_r + a_i) b_r,  k2 = a_r (b_i - b_r),  k3 = a_i (b_r + b_i);  Re = k1 - k3,  Im = k1 + k2
//   conj(a) b (GEMM-1):  k1 = (a_r - a_i) b_r,  k2, k3 as above;                              Re = k1 + k3,  Im = k1 + k2
// i.e. three real GEMMs over the same K instead of four: 6 instead of 8 flops per complex multiply-add on
// the FP64 tensor pipe, which is what bounds K3.  The three products need three accumulator sets
// (3 x 128 x 64 doubles per CTA tile = 75 % of the register file), so the CTA has 12 warps in three groups
// of four (one warp of each group per SM sub-partition, 128 accumulator registers per thread):
//   group 0: k1, warp tile 32 (M) x 64 (N): 4 A fragments summed in registers, 8 plain B fragments
//   group 1: k2, warp tile 64 x 32: 8 plain A fragments (re), 4 B fragments (b_i - b_r)
//   group 2: k3, warp tile 64 x 32: 8 plain A fragments (im), 4 B fragments (b_r + b_i)
// so every warp does 12 shared-memory loads, 4 DADDs and 32 DMMAs per k-group: the groups run at the same
// pace (with all the sums in one group that group lagged and the others idled at the ring: 88 % DMMA
// utilisation, profiles/).  The epilogue stages k2 and k3 through the drained tile ring; group 0 combines.
// TMA ring, tile shapes, swizzle and fragment addressing are those of the kernels above.
constexpr int NL3_CONSUMERS = 12;
constexpr int NL3_THREADS = NL3_CONSUMERS * 32;
constexpr int NL3_XS = NL_BN + 2;   // padded row stride (doubles) of the staged k2 / k3 tiles

// GRP 0: acc[mb 0..3][nb 0..7]; GRP 1, 2: acc[mb 0..7][nb 0..3]; flat index (mb * NB + nb) * 2 + e
template <int MODE, int GRP>
__device__ __forceinline__ void mma3_stage(const unsigned char *As, const unsigned char *Bs, int wq, int lane, double (&acc)[64]) {
  constexpr int MB = GRP == 0 ? 4 : 8, NB = GRP == 0 ? 8 : 4;
  const int i = lane >> 2, j = lane & 3;
  const int row0 = GRP == 0 ? wq * 32 : (wq >> 1) * 64, col0 = GRP == 0 ? 0 : (wq & 1) * 32;
#pragma unroll
  for (int kg = 0; kg < 2; kg++) {
    double a[MB], b[NB];
    const unsigned char *a0;
    int astride;
    if (MODE == 1) { a0 = As + (row0 + i) * 128 + (((2 * j + kg) ^ i) << 4); astride = 8 * 128; }
    else { const int pr = 2 * j + kg; a0 = As + (row0 >> 3) * 1024 + pr * 128 + ((i ^ pr) << 4); astride = 1024; }
#pragma unroll
    for (int mb = 0; mb < MB; mb++) {
      if (GRP == 0) {
        double2 v = *reinterpret_cast<const double2 *>(a0 + mb * astride);
        a[mb] = MODE == 1 ? v.x - v.y : v.x + v.y;
      } else if (GRP == 1) a[mb] = *reinterpret_cast<const double *>(a0 + mb * astride);
      else a[mb] = *reinterpret_cast<const double *>(a0 + mb * astride + 8);
    }
    const unsigned char *b0 = Bs + (col0 + i) * 128 + (((2 * j + kg) ^ i) << 4);
#pragma unroll
    for (int nb = 0; nb < NB; nb++) {
      if (GRP == 0) b[nb] = *reinterpret_cast<const double *>(b0 + nb * 8 * 128);
      else {
        double2 v = *reinterpret_cast<const double2 *>(b0 + nb * 8 * 128);
        b[nb] = GRP == 1 ? v.y - v.x : v.x + v.y;
      }
    }
#pragma unroll
    for (int mb = 0; mb < MB; mb++)
#pragma unroll
      for (int nb = 0; nb < NB; nb++) dmma(acc[(mb * NB + nb) * 2], acc[(mb * NB + nb) * 2 + 1], a[mb], b[nb]);
  }
}

__device__ __forceinline__ Pipe pipe_setup3(unsigned char *smem_raw) {
  Pipe P;
  P.tiles = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  P.full = reinterpret_cast<uint64_t *>(P.tiles + NL_STAGES * NL_STAGE_BYTES);
  P.empty = P.full + NL_STAGES;
  if (threadIdx.x == 0) {
    for (int s = 0; s < NL_STAGES; s++) { mbar_init(&P.full[s], 1); mbar_init(&P.empty[s], NL3_CONSUMERS); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  return P;
}

// main loop of one warp of group GRP: waits for slabs, multiplies, releases; the producer lane also issues
template <int MODE, int GRP, typename Issue>
__device__ __forceinline__ void mainloop3(const Pipe &P, int ns, bool producer, int wq, int lane, double (&acc)[64], Issue &issue) {
  for (int it = 0; it < ns; it++) {
    if (producer && it + NL_PREFETCH < ns) issue(it + NL_PREFETCH);
    __syncwarp();
    int s = it % NL_STAGES;
    mbar_wait(&P.full[s], (it / NL_STAGES) & 1);
    const unsigned char *st = P.tiles + s * NL_STAGE_BYTES;
    mma3_stage<MODE, GRP>(st, st + NL_STAGE_A, wq, lane, acc);
    __syncwarp();
    if (lane == 0) mbar_arrive(&P.empty[s]);
  }
}

// k2 (group 1) and k3 (group 2) go through shared memory as [128][NL3_XS] tiles; group 0 combines and hands
// every output (row in tile, column in tile, re, im) of its 32 x 64 warp tile to `emit`
template <int MODE, typename Emit>
__device__ __forceinline__ void combine3(const Pipe &P, int grp, int wq, int lane, double (&acc)[64], Emit &emit) {
  __syncthreads();   // every warp is done with the tile ring (all issued slabs were consumed)
  double *X = reinterpret_cast<double *>(P.tiles);
  const int i = lane >> 2, j = lane & 3;
  if (grp > 0) {
    double *dst = X + (size_t)(grp - 1) * (NL_BM * NL3_XS) + (size_t)((wq >> 1) * 64 + i) * NL3_XS + (wq & 1) * 32 + 2 * j;
#pragma unroll
    for (int mb = 0; mb < 8; mb++)
#pragma unroll
      for (int nb = 0; nb < 4; nb++)
        *reinterpret_cast<double2 *>(dst + (size_t)mb * 8 * NL3_XS + nb * 8) = make_double2(acc[(mb * 4 + nb) * 2], acc[(mb * 4 + nb) * 2 + 1]);
  }
  __syncthreads();
  if (grp == 0) {
    const double *s2 = X + (size_t)(wq * 32 + i) * NL3_XS + 2 * j, *s3 = s2 + NL_BM * NL3_XS;
#pragma unroll
    for (int mb = 0; mb < 4; mb++)
#pragma unroll
      for (int nb = 0; nb < 8; nb++) {
        double2 k2 = *reinterpret_cast<const double2 *>(s2 + (size_t)mb * 8 * NL3_XS + nb * 8);
        double2 k3 = *reinterpret_cast<const double2 *>(s3 + (size_t)mb * 8 * NL3_XS + nb * 8);
        double k1a = acc[(mb * 8 + nb) * 2], k1b = acc[(mb * 8 + nb) * 2 + 1];
        const int r = wq * 32 + mb * 8 + i, c = nb * 8 + 2 * j;
        if (MODE == 1) { emit(r, c, k1a + k3.x, k1a + k2.x); emit(r, c + 1, k1b + k3.y, k1b + k2.y); }
        else { emit(r, c, k1a - k3.x, k1a + k2.x); emit(r, c + 1, k1b - k3.y, k1b + k2.y); }
      }
  }
}

__global__ void __launch_bounds__(NL3_THREADS, 1)
gemm1_3m_kernel(const __grid_constant__ CUtensorMap mapP, const __grid_constant__ CUtensorMap mapPsi, Gemm1Params Q) {
  extern __shared__ unsigned char smem_raw[];
  Pipe P = pipe_setup3(smem_raw);
  const int tile = blockIdx.x, tn = tile % Q.tiles_n, tm = tile / Q.tiles_n;
  const int split = blockIdx.y, ik = blockIdx.z;
  const int s0 = split * Q.slabs_per_split;
  int ns = Q.nslab - s0; if (ns > Q.slabs_per_split) ns = Q.slabs_per_split; if (ns < 0) ns = 0;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, grp = warp >> 2, wq = warp & 3;
  auto issue = [&](int j) {
    int s = j % NL_STAGES;
    if (j >= NL_STAGES) mbar_wait(&P.empty[s], ((j / NL_STAGES) - 1) & 1);
    unsigned char *st = P.tiles + s * NL_STAGE_BYTES;
    mbar_expect_tx(&P.full[s], NL_STAGE_BYTES);
    tma_load_3d(st, &mapP, &P.full[s], (s0 + j) * 16, tm * NL_BM, ik);
    tma_load_3d(st + NL_STAGE_A, &mapPsi, &P.full[s], (s0 + j) * 16, tn * NL_BN, ik);
  };
  const bool producer = (threadIdx.x == 0);
  if (producer)
    for (int j = 0; j < NL_PREFETCH && j < ns; j++) issue(j);
  double acc[64];
#pragma unroll
  for (int q = 0; q < 64; q++) acc[q] = 0.0;
  if (grp == 0) mainloop3<1, 0>(P, ns, producer, wq, lane, acc, issue);
  else if (grp == 1) mainloop3<1, 1>(P, ns, false, wq, lane, acc, issue);
  else mainloop3<1, 2>(P, ns, false, wq, lane, acc, issue);
  double2 *out = Q.part + ((size_t)(ik * Q.nsplit + split) * Q.nproj) * Q.nband;
  auto emit = [&](int r, int c, double re, double im) {
    int pr = tm * NL_BM + r, b = tn * NL_BN + c;
    if (pr < Q.nproj && b < Q.nband) out[(size_t)pr * Q.nband + b] = make_double2(re, im);
  };
  combine3<1>(P, grp, wq, lane, acc, emit);
}

__global__ void __launch_bounds__(NL3_THREADS, 1)
gemm2_3m_kernel(const __grid_constant__ CUtensorMap mapP, const __grid_constant__ CUtensorMap mapC, Gemm2Params Q) {
  extern __shared__ unsigned char smem_raw[];
  Pipe P = pipe_setup3(smem_raw);
  const int tn = blockIdx.x % Q.tiles_n, tm = blockIdx.x / Q.tiles_n, ik = blockIdx.z;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, grp = warp >> 2, wq = warp & 3;
  const int ns = Q.with_nl ? Q.nslab : 0;
  auto issue = [&](int j) {
    int s = j % NL_STAGES;
    if (j >= NL_STAGES) mbar_wait(&P.empty[s], ((j / NL_STAGES) - 1) & 1);
    unsigned char *st = P.tiles + s * NL_STAGE_BYTES;
    mbar_expect_tx(&P.full[s], NL_STAGE_BYTES);
    tma_load_4d(st, &mapP, &P.full[s], 0, j * 8, tm * (NL_BM / 8), ik);
    tma_load_3d(st + NL_STAGE_A, &mapC, &P.full[s], j * 16, tn * NL_BN, ik);
  };
  const bool producer = (threadIdx.x == 0);
  if (producer)
    for (int j = 0; j < NL_PREFETCH && j < ns; j++) issue(j);
  double acc[64];
#pragma unroll
  for (int q = 0; q < 64; q++) acc[q] = 0.0;
  if (grp == 0) mainloop3<2, 0>(P, ns, producer, wq, lane, acc, issue);
  else if (grp == 1) mainloop3<2, 1>(P, ns, false, wq, lane, acc, issue);
  else mainloop3<2, 2>(P, ns, false, wq, lane, acc, issue);
  // group 0 leaves (re, im) of the whole 128 x 64 tile in the k2 / k3 staging tiles; then all 12 warps run the
  // epilogue with g (contiguous in psi / hpsi) along the lanes and their loads batched U at a time
  auto keep = [&](int r, int c, double re, double im) {
    double *X = reinterpret_cast<double *>(P.tiles);
    X[(size_t)r * NL3_XS + c] = re;
    X[(size_t)NL_BM * NL3_XS + (size_t)r * NL3_XS + c] = im;
  };
  combine3<2>(P, grp, wq, lane, acc, keep);
  __syncthreads();
  const double *Xre = reinterpret_cast<const double *>(P.tiles), *Xim = Xre + NL_BM * NL3_XS;
  const int r = threadIdx.x & (NL_BM - 1), c0 = threadIdx.x >> 7;   // 384 threads = 3 columns of 128 rows
  const int g = tm * NL_BM + r;
  const bool gok = g < Q.npw[ik];
  const double kg = (Q.with_kin && gok) ? Q.kin[ik][g] : 0.0;
  const size_t base = (size_t)ik * Q.nband * Q.mpw + g;
  constexpr int U = 6, NQ = (NL_BN + 2) / 3;
#pragma unroll 1
  for (int q0 = 0; q0 < NQ; q0 += U) {
    double2 x[U], h[U], xp[U];
    bool ok[U];
#pragma unroll
    for (int u = 0; u < U; u++) {
      const int c = c0 + 3 * (q0 + u), b = tn * NL_BN + c;
      ok[u] = gok && c < NL_BN && b < Q.nband;
      const size_t off = base + (size_t)b * Q.mpw;
      x[u] = (ok[u] && (Q.with_kin || Q.cheb)) ? Q.psi[off] : make_double2(0.0, 0.0);
      h[u] = (ok[u] && Q.accumulate) ? Q.hpsi[off] : make_double2(0.0, 0.0);
      xp[u] = (ok[u] && Q.cheb && Q.sx != 0.0) ? Q.xprev[off] : make_double2(0.0, 0.0);
    }
#pragma unroll
    for (int u = 0; u < U; u++) {
      const int c = c0 + 3 * (q0 + u), b = tn * NL_BN + c;
      if (ok[u]) {
        double2 v = make_double2(Xre[(size_t)r * NL3_XS + c] + kg * x[u].x + h[u].x, Xim[(size_t)r * NL3_XS + c] + kg * x[u].y + h[u].y);
        if (Q.cheb) {
          v.x = Q.sh * v.x + Q.sy * x[u].x + Q.sx * xp[u].x; v.y = Q.sh * v.y + Q.sy * x[u].y + Q.sx * xp[u].y;
        }
        Q.hpsi[base + (size_t)b * Q.mpw] = v;
      }
    }
  }
}

// ---------------------------------------------------------------- factorised projectors (proj_mode = 1)
// p_{a,i}(G) = FY_{t(a),i}(G) . S_a(G) with FY real and S_a a phase (projtab.cu), the paper's "computed on-the-fly"
// variant (:477).  Neither GEMM then needs the [nproj][npw] table, and because FY is real the contraction over G is a
// REAL x complex product after one complex multiplication per (atom, band, G):
//   GEMM-1:  z_{a,b}(G) = conj(S_a(G)) psi_b(G)                (4 FP64 instructions per thread, shared by the 8 projectors)
//            cprj[a,i,b] = sum_G FY[i,G] z_{a,b}(G)            (2 DMMA per 8 x 8 x 4 block: re and im columns)
// 2 DMMAs + 4 FP64 instructions where the 4-product form needs 4 DMMAs and the Gauss form 3 (+ sums): 40 against 64 /
// 49 pipe clocks per block.  M = 8 of the m8n8k4 shape is the 8 projectors of one atom, so the CTA tile is
// 16 atoms x 64 bands (16 warps, 4 atoms x 16 bands each).
constexpr int FC_BA = 16;                  // atoms per CTA tile
constexpr int FC_OFF_S = NL_BN * 128;      // stage layout: psi tile 8 KB | S tile 2 KB | FY tile <= 1 KB
constexpr int FC_OFF_F = FC_OFF_S + FC_BA * 128;
constexpr int FC_STAGE_BYTES = 12 * 1024;      // FY tile: FAC_MAX_FROWS rows x 8 doubles = 2 KB
constexpr int FC_STAGES = 8;
constexpr int FC_SMEM = FC_STAGES * FC_STAGE_BYTES + 1024 + 256;
constexpr int FC_WARPS = 16;               // 4 (atom groups) x 4 (band groups): four warps per SM sub-partition hide the
constexpr int FC_THREADS = FC_WARPS * 32 + 128;  // DMUL -> DFMA -> DMMA chains of the z = conj(S) psi products; warps 16-19 are the
// producer group (lane 0 of warp 16 issues the TMA loads; a consumer that also issued them paced the ring).  A fifth warp per
// sub-partition would cap every thread at 96 registers, so the producer warps shrink to 24 and the consumers take 112 (the pool is what the CTA got at launch: 640 x 96).
__device__ __forceinline__ void reg_alloc_fac_consumer() { asm volatile("setmaxnreg.inc.sync.aligned.u32 112;"); }

struct Fac1Params {
  int nblk, nfrow, nband, nproj, nslab, nsplit, slabs_per_split, tiles_n;
  const int32_t *blk_atom, *blk_frow, *blk_first, *blk_nl;   // projector blocks of <= 8 rows (projtab.cu)
  double2 *part;   // [nkpt][nsplit][nproj][nband]
};

// grid: (tiles_a * tiles_n, nsplit, nkpt)
__global__ void __launch_bounds__(FC_THREADS, 1)
gemm1_fac_kernel(const __grid_constant__ CUtensorMap mapPsi, const __grid_constant__ CUtensorMap mapS,
                 const __grid_constant__ CUtensorMap mapF, Fac1Params Q) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char *tiles = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint64_t *full = reinterpret_cast<uint64_t *>(tiles + FC_STAGES * FC_STAGE_BYTES), *empty = full + FC_STAGES;
  if (threadIdx.x == 0) {
    for (int s = 0; s < FC_STAGES; s++) { mbar_init(&full[s], 1); mbar_init(&empty[s], FC_WARPS); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int tn = blockIdx.x % Q.tiles_n, ta = blockIdx.x / Q.tiles_n, split = blockIdx.y, ik = blockIdx.z;
  const int s0 = split * Q.slabs_per_split;
  int ns = Q.nslab - s0; if (ns > Q.slabs_per_split) ns = Q.slabs_per_split; if (ns < 0) ns = 0;
  const uint32_t tx = NL_BN * 128 + FC_BA * 128 + 64 * Q.nfrow;
  const int atom0 = __ldg(Q.blk_atom + ta * FC_BA);      // S rows of the tile: 16 atoms from the first block's atom
  auto issue = [&](int j) {
    int s = j % FC_STAGES;
    if (j >= FC_STAGES) mbar_wait(&empty[s], ((j / FC_STAGES) - 1) & 1);
    unsigned char *st = tiles + s * FC_STAGE_BYTES;
    mbar_expect_tx(&full[s], tx);
    tma_load_3d(st, &mapPsi, &full[s], (s0 + j) * 16, tn * NL_BN, ik);
    tma_load_3d(st + FC_OFF_S, &mapS, &full[s], (s0 + j) * 16, atom0, ik);
    tma_load_3d(st + FC_OFF_F, &mapF, &full[s], (s0 + j) * 8, 0, ik);
  };
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, wm = warp >> 2, wn = warp & 3;   // 4 atoms x 16 bands per warp
  if (warp >= FC_WARPS) {
    reg_dealloc_producer();
    if (warp == FC_WARPS && lane == 0)
      for (int j = 0; j < ns; j++) issue(j);
    return;
  }
  reg_alloc_fac_consumer();
  const int i = lane >> 2, j = lane & 3;
  int frow[4], arow[4];   // this lane's FY row (byte offset in the FY tile) and its block's S row, per block of the warp
#pragma unroll
  for (int q = 0; q < 4; q++) {
    const int blk = ta * FC_BA + wm * 4 + q, ok = blk < Q.nblk;
    frow[q] = ((ok ? Q.blk_frow[blk] : 0) + i) * 64;
    arow[q] = ok ? Q.blk_atom[blk] - atom0 : 0;
  }
  double cre[4][2][2], cim[4][2][2];
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int b = 0; b < 2; b++) { cre[a][b][0] = cre[a][b][1] = cim[a][b][0] = cim[a][b][1] = 0.0; }
  for (int it = 0; it < ns; it++) {
    int s = it % FC_STAGES;
    mbar_wait(&full[s], (it / FC_STAGES) & 1);
    const unsigned char *Ps = tiles + s * FC_STAGE_BYTES, *Ss = Ps + FC_OFF_S, *Fs = Ps + FC_OFF_F;
#pragma unroll
    for (int kg = 0; kg < 2; kg++) {
      const int e = 2 * j + kg;   // this lane's G inside the slab (k index of the 8x8x4 block)
      double pr[2], pi[2];
      const unsigned char *b0 = Ps + (wn * 16 + i) * 128 + ((e ^ i) << 4);
#pragma unroll
      for (int nb = 0; nb < 2; nb++) {
        double2 v = *reinterpret_cast<const double2 *>(b0 + nb * 8 * 128);
        pr[nb] = v.x; pi[nb] = v.y;
      }
#pragma unroll
      for (int q = 0; q < 4; q++) {
        const double2 sg = *reinterpret_cast<const double2 *>(Ss + arow[q] * 128 + ((e ^ (arow[q] & 7)) << 4));
        const double fa = *reinterpret_cast<const double *>(Fs + frow[q] + e * 8);
#pragma unroll
        for (int nb = 0; nb < 2; nb++) {
          double zr = sg.x * pr[nb] + sg.y * pi[nb], zi = sg.x * pi[nb] - sg.y * pr[nb];   // conj(S) psi
          dmma(cre[q][nb][0], cre[q][nb][1], fa, zr);
          dmma(cim[q][nb][0], cim[q][nb][1], fa, zi);
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[s]);
  }
  // partial[ik][split][first_blk + i][b]; thread holds projector i of its 4 blocks, bands 2j, 2j+1 of each 8-band block
  double2 *out = Q.part + ((size_t)(ik * Q.nsplit + split) * Q.nproj) * Q.nband;
#pragma unroll
  for (int q = 0; q < 4; q++) {
    const int blk = ta * FC_BA + wm * 4 + q;
    if (blk >= Q.nblk) continue;
    if (i >= Q.blk_nl[blk]) continue;
    double2 *row = out + (size_t)(Q.blk_first[blk] + i) * Q.nband;
#pragma unroll
    for (int nb = 0; nb < 2; nb++) {
      int b = tn * NL_BN + wn * 16 + nb * 8 + 2 * j;
      if (b < Q.nband) row[b] = make_double2(cre[q][nb][0], cim[q][nb][0]);
      if (b + 1 < Q.nband) row[b + 1] = make_double2(cre[q][nb][1], cim[q][nb][1]);
    }
  }
}

//   GEMM-2:  w_{a,b}(G) = sum_i FY[i,G] c'[a,i,b]               (4 DMMA per 8 x 8 block: 2 k-groups of projectors x re/im)
//            hpsi_b(G) += S_a(G) w_{a,b}(G)                     (8 FP64 instructions per thread and block)
// One K-slab = one projector block (an atom's <= 8 rows): its c' tile [64 bands][8 projectors] (TMA, swizzled) and its phases for the tile's 128 G.
// The FY rows of the tile's 128 G (8 per atom type, row stride 132 doubles against bank conflicts) are loaded once.
constexpr int FD_OFF_S = NL_BN * 128;                 // stage: c' tile 8 KB | S_a(G) 2 KB
constexpr int FD_STAGE_BYTES = 10 * 1024;
constexpr int FD_STAGES = 8;
constexpr int FD_FLD = NL_BM + 4;                     // FY row stride in shared memory (doubles)
constexpr int FD_FBYTES = FAC_MAX_FROWS * FD_FLD * 8;  // FY rows of every type for the tile's 128 G
constexpr int FD_SMEM = FD_STAGES * FD_STAGE_BYTES + FD_FBYTES + 1024 + 256;

// grid: (tiles_n * tiles_m, 1, nkpt); Q as in gemm2_kernel, nslab = natom
__global__ void __launch_bounds__(FC_THREADS, 1)
gemm2_fac_kernel(const __grid_constant__ CUtensorMap mapC, const __grid_constant__ CUtensorMap mapS,
                 const __grid_constant__ CUtensorMap mapF, Gemm2Params Q, const int32_t *__restrict__ blk_atom,
                 const int32_t *__restrict__ blk_frow, const int32_t *__restrict__ blk_first, int nfrow) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char *tiles = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  unsigned char *Fs = tiles + FD_STAGES * FD_STAGE_BYTES;
  uint64_t *full = reinterpret_cast<uint64_t *>(Fs + FD_FBYTES), *empty = full + FD_STAGES, *fbar = empty + FD_STAGES;
  if (threadIdx.x == 0) {
    for (int s = 0; s < FD_STAGES; s++) { mbar_init(&full[s], 1); mbar_init(&empty[s], FC_WARPS); }
    mbar_init(fbar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int tn = blockIdx.x % Q.tiles_n, tm = blockIdx.x / Q.tiles_n, ik = blockIdx.z;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, wm = warp >> 2, wn = warp & 3;   // 32 G x 16 bands per warp
  const int i = lane >> 2, j = lane & 3;
  const int ns = Q.with_nl ? Q.nslab : 0;
  auto issue = [&](int a) {
    int s = a % FD_STAGES;
    if (a >= FD_STAGES) mbar_wait(&empty[s], ((a / FD_STAGES) - 1) & 1);
    unsigned char *st = tiles + s * FD_STAGE_BYTES;
    mbar_expect_tx(&full[s], NL_BN * 128 + NL_BM * 16);
    tma_load_3d(st, &mapC, &full[s], 2 * __ldg(blk_first + a), tn * NL_BN, ik);
    tma_load_3d(st + FD_OFF_S, &mapS, &full[s], tm * NL_BM * 2, __ldg(blk_atom + a), ik);
  };
  if (warp >= FC_WARPS) {
    reg_dealloc_producer();
    if (warp == FC_WARPS && lane == 0 && ns > 0) {
      mbar_expect_tx(fbar, (uint32_t)(nfrow * FD_FLD * 8));
      tma_load_3d(Fs, &mapF, fbar, tm * NL_BM, 0, ik);
      for (int a = 0; a < ns; a++) issue(a);
    }
    return;
  }
  reg_alloc_fac_consumer();
  double cre[4][2][2], cim[4][2][2];
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int b = 0; b < 2; b++) { cre[a][b][0] = cre[a][b][1] = cim[a][b][0] = cim[a][b][1] = 0.0; }
  if (ns > 0) mbar_wait(fbar, 0);
  for (int a = 0; a < ns; a++) {
    int s = a % FD_STAGES;
    const int fr0 = __ldg(blk_frow + a);      // first FY row of this block
    mbar_wait(&full[s], (a / FD_STAGES) & 1);
    const unsigned char *Cs = tiles + s * FD_STAGE_BYTES, *Ss = Cs + FD_OFF_S;
    double2 sg[4];
    double fa[4][2];
#pragma unroll
    for (int mb = 0; mb < 4; mb++) {
      const int g = wm * 32 + mb * 8 + i;                                   // G row of this lane inside the tile
      sg[mb] = *reinterpret_cast<const double2 *>(Ss + g * 16);
#pragma unroll
      for (int kgp = 0; kgp < 2; kgp++)                                      // projector 2j + kgp of the atom's type
        fa[mb][kgp] = *reinterpret_cast<const double *>(Fs + ((size_t)((fr0 + 2 * j + kgp) * FD_FLD + g)) * 8);
    }
#pragma unroll
    for (int nb = 0; nb < 2; nb++) {
      double cr[2], ci[2];
      const unsigned char *b0 = Cs + (wn * 16 + nb * 8 + i) * 128;
#pragma unroll
      for (int kgp = 0; kgp < 2; kgp++) {
        double2 v = *reinterpret_cast<const double2 *>(b0 + (((2 * j + kgp) ^ i) << 4));
        cr[kgp] = v.x; ci[kgp] = v.y;
      }
#pragma unroll
      for (int mb = 0; mb < 4; mb++) {
        double wr0 = 0.0, wr1 = 0.0, wi0 = 0.0, wi1 = 0.0;
#pragma unroll
        for (int kgp = 0; kgp < 2; kgp++) {
          dmma(wr0, wr1, fa[mb][kgp], cr[kgp]);
          dmma(wi0, wi1, fa[mb][kgp], ci[kgp]);
        }
        // acc += S_a(G) w: two fused multiply-adds per component (written out so that no separate add is generated)
        cre[mb][nb][0] = fma(-sg[mb].y, wi0, fma(sg[mb].x, wr0, cre[mb][nb][0]));
        cim[mb][nb][0] = fma(sg[mb].y, wr0, fma(sg[mb].x, wi0, cim[mb][nb][0]));
        cre[mb][nb][1] = fma(-sg[mb].y, wi1, fma(sg[mb].x, wr1, cre[mb][nb][1]));
        cim[mb][nb][1] = fma(sg[mb].y, wr1, fma(sg[mb].x, wi1, cim[mb][nb][1]));
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[s]);
  }
  // epilogue as in gemm2_kernel: rows g = lane/4, bands 2*(lane%4)+{0,1}
  const int npw = Q.npw[ik];
  const double *kin = Q.kin[ik];
  const double2 *psi = Q.psi + (size_t)ik * Q.nband * Q.mpw;
  double2 *hpsi = Q.hpsi + (size_t)ik * Q.nband * Q.mpw;
#pragma unroll
  for (int mb = 0; mb < 4; mb++) {
    int g = tm * NL_BM + wm * 32 + mb * 8 + i;
    if (g >= npw) continue;
    double kg = Q.with_kin ? kin[g] : 0.0;
#pragma unroll
    for (int nb = 0; nb < 2; nb++) {
#pragma unroll
      for (int e = 0; e < 2; e++) {
        int b = tn * NL_BN + wn * 16 + nb * 8 + 2 * j + e;
        if (b >= Q.nband) continue;
        size_t off = (size_t)b * Q.mpw + g;
        double2 r = make_double2(cre[mb][nb][e], cim[mb][nb][e]);
        if (Q.with_kin) { double2 x = psi[off]; r.x += kg * x.x; r.y += kg * x.y; }
        if (Q.accumulate) { double2 h = hpsi[off]; r.x += h.x; r.y += h.y; }
        if (Q.cheb) {
          double2 y = psi[off], xp = Q.sx != 0.0 ? Q.xprev[(size_t)ik * Q.nband * Q.mpw + off] : make_double2(0.0, 0.0);
          r.x = Q.sh * r.x + Q.sy * y.x + Q.sx * xp.x; r.y = Q.sh * r.y + Q.sy * y.y + Q.sx * xp.y;
        }
        hpsi[off] = r;
      }
    }
  }
}

// ---------------------------------------------------------------- tiny cells: the whole non-local term in ONE launch
// For a cell with a few projectors and a few hundred plane waves (c0: 16 x 283 x 8 bands) GEMM-1, the D_ij step and GEMM-2
// are three dependent launches of 10-17 us that do 36 000 complex multiply-adds: pure launch latency.  Eq. 26 acts on every
// band by itself, so here one CTA does one band (and k-point) from beginning to end:
//   1. cprj[p] = sum_G conj(P[p][G]) psi[G]: warp w takes the projectors w, w + 8, ...; its lanes stride over G (coalesced
//      rows of the table), fixed-order shuffle reduction;
//   2. c'[i] = sum_j D^a_ij cprj[j] (thread i < nproj, its atom found by a scan of atom_first);
//   3. hpsi[G] (+)= sum_p P[p][G] c'[p] + kin[G] psi[G] (and the recurrence combination), thread per G.
// Plain FP64 FMAs (the DMMA tile shapes would be 7/8 padding here); taken when nproj <= 64 and nproj npw nband nkpt <= 1e6
// (option "nl_tiny" = 0 keeps the GEMM kernels).  Same arithmetic as Eq. 26 in a different summation order.
constexpr int NLT_MAXP = 64, NLT_THREADS = 256;
__global__ void __launch_bounds__(NLT_THREADS)
nl_tiny_kernel(const double2 *__restrict__ ptab, const double2 *__restrict__ psi_all, double2 *__restrict__ hpsi_all,
               const double *__restrict__ dij, const int32_t *__restrict__ typat, const int32_t *__restrict__ nlmn,
               const int32_t *__restrict__ atom_first, const int32_t *__restrict__ npw_k, const double *const *kin_k, int natom,
               int lmax, int nproj, int nband, int mpw, int accumulate, int with_kin, int cheb, double sh, double sy, double sx,
               const double2 *__restrict__ xprev_all) {
  __shared__ double2 cp[NLT_MAXP], cq[NLT_MAXP];
  const int b = blockIdx.x, ik = blockIdx.y, t = threadIdx.x, warp = t >> 5, lane = t & 31;
  const int npw = npw_k[ik];
  const double2 *P = ptab + (size_t)ik * nproj * mpw;
  const size_t row = ((size_t)ik * nband + b) * mpw;
  const double2 *psi = psi_all + row;
  double2 *hpsi = hpsi_all + row;
  for (int p = warp; p < nproj; p += NLT_THREADS / 32) {
    const double2 *pr = P + (size_t)p * mpw;
    double sr = 0.0, si = 0.0;
    for (int g = lane; g < npw; g += 32) {
      const double2 a = pr[g], x = psi[g];
      sr += a.x * x.x + a.y * x.y; si += a.x * x.y - a.y * x.x;       // conj(p) psi
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { sr += __shfl_xor_sync(0xffffffffu, sr, o); si += __shfl_xor_sync(0xffffffffu, si, o); }
    if (lane == 0) cp[p] = make_double2(sr, si);
  }
  __syncthreads();
  if (t < nproj) {
    int a = 0;
    while (a + 1 < natom && atom_first[a + 1] <= t) a++;
    const int first = atom_first[a], nl = nlmn[typat[a]], ii = t - first;
    const double *D = dij + (size_t)a * lmax * lmax + (size_t)ii * lmax;
    double sr = 0.0, si = 0.0;
    for (int jj = 0; jj < nl; jj++) { const double d = D[jj]; sr += d * cp[first + jj].x; si += d * cp[first + jj].y; }
    cq[t] = make_double2(sr, si);
  }
  __syncthreads();
  const double *kin = kin_k[ik];
  for (int g = t; g < npw; g += NLT_THREADS) {
    double rr = 0.0, ri = 0.0;
    for (int p = 0; p < nproj; p++) {
      const double2 a = P[(size_t)p * mpw + g], c = cq[p];
      rr += a.x * c.x - a.y * c.y; ri += a.x * c.y + a.y * c.x;
    }
    const double2 x = psi[g];
    if (with_kin) { const double kg = kin[g]; rr += kg * x.x; ri += kg * x.y; }
    if (accumulate) { const double2 h = hpsi[g]; rr += h.x; ri += h.y; }
    if (cheb) {
      const double2 xp = sx != 0.0 ? xprev_all[row + g] : make_double2(0.0, 0.0);
      rr = sh * rr + sy * x.x + sx * xp.x; ri = sh * ri + sy * x.y + sx * xp.y;
    }
    hpsi[g] = make_double2(rr, ri);
  }
}

// ---------------------------------------------------------------- host side
struct NlMaps {
  CUtensorMap mapP1, mapP2, mapPsi, mapC;
  const void *ptab = nullptr, *psi = nullptr, *cprj = nullptr;
  int bm1 = 0, nband_psi = -1, nband_c = -1;
};
struct SymMaps {
  CUtensorMap mapP1, mapP2, mapX, mapC;
  const void *ptab = nullptr, *x = nullptr, *cprj = nullptr;
  int n2_x = -1, n2_c = -1;
};
void strassen_free(dft_plan *p);
void nl_maps_free(dft_plan *p) { delete p->nl_maps; p->nl_maps = nullptr; delete p->sym_maps; p->sym_maps = nullptr; strassen_free(p); }

typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                             const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 3-D FP64 tensor map over a [d2][d1][d0] array (d0 contiguous doubles), box {16, box1, 1}, 128-byte swizzle
static int make_map(dft_plan *p, CUtensorMap *m, const void *base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t stride1_bytes,
                    uint64_t stride2_bytes, uint32_t box1) {
  cuuint64_t dims[3] = {d0, d1, d2};
  cuuint64_t strides[2] = {stride1_bytes, stride2_bytes};
  cuuint32_t box[3] = {16, box1, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = ((EncodeFn)p->encode_fn)(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void *>(base), dims, strides, box, estr,
                                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_error("cuTensorMapEncodeTiled failed (%d): dims %llu %llu %llu strides %llu %llu box1 %u", (int)r,
              (unsigned long long)d0, (unsigned long long)d1, (unsigned long long)d2, (unsigned long long)stride1_bytes,
              (unsigned long long)stride2_bytes, box1);
    return DFT_ERR_CUDA;
  }
  return DFT_OK;
}

// 3-D FP64 tensor map without swizzle (rows longer than 128 bytes or narrower than a swizzle atom)
static int make_map_plain(dft_plan *p, CUtensorMap *m, const void *base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t stride1_bytes,
                          uint64_t stride2_bytes, uint32_t box0, uint32_t box1) {
  cuuint64_t dims[3] = {d0, d1, d2};
  cuuint64_t strides[2] = {stride1_bytes, stride2_bytes};
  cuuint32_t box[3] = {box0, box1, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = ((EncodeFn)p->encode_fn)(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void *>(base), dims, strides, box, estr,
                                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled (plain map, box %u x %u) failed (%d)", box0, box1, (int)r); return DFT_ERR_CUDA; }
  return DFT_OK;
}

__global__ void kin_only_kernel(const double2 *__restrict__ psi, double2 *__restrict__ hpsi, const double *const *kin,
                                const int32_t *npw, int nband, int mpw, int accumulate, int with_kin, int cheb, double sh,
                                double sy, double sx, const double2 *__restrict__ xprev, int gamma = 0) {
  int ik = blockIdx.z, b = blockIdx.y;
  const double *k = kin[ik];
  int n = npw[ik];
  size_t row = ((size_t)ik * nband + b) * mpw;
  for (int g = blockIdx.x * blockDim.x + threadIdx.x; g < n; g += gridDim.x * blockDim.x) {
    double2 r = make_double2(0.0, 0.0);
    if (with_kin) { double2 x = psi[row + g]; double kg = k[g]; r.x = kg * x.x; r.y = kg * x.y; }
    if (accumulate) { double2 h = hpsi[row + g]; r.x += h.x; r.y += h.y; }
    if (cheb) {
      double2 y = psi[row + g], xp = sx != 0.0 ? xprev[row + g] : make_double2(0.0, 0.0);
      r.x = sh * r.x + sy * y.x + sx * xp.x; r.y = sh * r.y + sy * y.y + sx * xp.y;
    }
    if (gamma && g == 0) r.y = 0.0;
    hpsi[row + g] = r;
  }
}


// choose the number of K splits of GEMM-1: fill the SMs in whole waves, keep >= 32 slabs per split
static int choose_splitk(int tiles, int nslab, int sm_count, int nkpt) {
  int best = 1; double best_eff = 0.0;
  // at least 32 slabs per split when the tiles alone fill the SMs; small problems (latency-bound) may go down to 8
  const int min_slabs = (int64_t)tiles * nkpt >= sm_count ? 32 : (nkpt >= 16 ? 24 : 8);
  for (int s = 1; s <= 64; s++) {
    if (s > 1 && nslab / s < min_slabs) break;
    double units = (double)tiles * s * nkpt;
    double waves = units / sm_count;
    double eff = waves / (double)(int64_t)(waves + 0.999999);
    if (eff > best_eff + 0.01) { best_eff = eff; best = s; }
  }
  return best;
}

// ---------------------------------------------------------------- symmetric-table GEMMs at k = 0
// At k = 0 the projectors obey p(-G) = (-1)^l conj(p(G)) (real F, real Y_lm of parity l, conjugate phases), whatever psi is.
// Any band is psi = psi_A + i psi_B with psi_A, psi_B time-reversal symmetric (c_A(G) = (c(G) + conj(c(-G)))/2,
// c_B(G) = (c(G) - conj(c(-G)))/(2i)), and for a symmetric vector every projection is i^(l odd) times a REAL number obtained
// from the half sphere alone (gamma.cu).  So both GEMMs run as REAL GEMMs over the interleaved (re, im) doubles of the
// half sphere with 2 nband columns -- 4 flops per (projector, plane wave, band) instead of 8 (four products) or 6
// (Gauss): gemm1_kernel<true> / gemm2_kernel<true> on the rotated half table of gamma.cu.  Unlike the Gamma STORAGE this
// needs no symmetry of psi or D_ij: the step between the GEMMs works on the complex z_j = r^A_j + i r^B_j,
//   <p_j|psi> = i^(l_j odd) z_j,   y_i = (-i)^(l_i odd) sum_j D_ij i^(l_j odd) z_j,   (V_nl psi)(+-G) = sum_i Pt_i(G)^(*) y_i,
// i.e. h_A = Pt y_r, h_B = Pt y_i on the half sphere and (V_nl psi)(G) = h_A + i h_B, (V_nl psi)(-G) = conj(h_A) + i conj(h_B).
// Exact up to rounding order, like the Gauss form.
__global__ void sym_split_kernel(const double2 *__restrict__ psi, double2 *__restrict__ X, const int32_t *__restrict__ h2f,
                                 const int32_t *__restrict__ h2fneg, int mpw, int nh) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
  if (h >= nh) return;
  const double2 cp = psi[(size_t)b * mpw + h2f[h]], cm = psi[(size_t)b * mpw + h2fneg[h]];
  X[(size_t)(2 * b) * nh + h] = make_double2(0.5 * (cp.x + cm.x), 0.5 * (cp.y - cm.y));
  X[(size_t)(2 * b + 1) * nh + h] = make_double2(0.5 * (cp.y + cm.y), -0.5 * (cp.x - cm.x));
}

// part [nsplit][nproj][2 nband] real (GEMM-1 partial sums S); psi: the bands (for the G = 0 term); cpr: c' [2 nband][nproj]
// complex with zero imaginary halves (rows 2b, 2b+1 = Re y, Im y), or, when dij is null, cprj_out [nband][nproj] = <p|psi>
__global__ void dij_sym_kernel(const double *__restrict__ part, double2 *__restrict__ cpr, const double *__restrict__ dij,
                               const int32_t *__restrict__ typat, const int32_t *__restrict__ nlmn,
                               const int32_t *__restrict__ atom_first, const int32_t *__restrict__ rowpar,
                               const double *__restrict__ p0, const double2 *__restrict__ psi, int mpw, int lmax, int nproj,
                               int nband, int nsplit, int ldc) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x, a = blockIdx.y;
  if (b >= nband) return;
  const int nl = nlmn[typat[a]], first = atom_first[a], n2 = 2 * nband;
  // c_A(0) = Re psi(0), c_B(0) = Im psi(0); G = 0 has the smallest box index, so it is entry 0 of the band
  const double2 c00 = psi[(size_t)b * mpw];
  const double ca0 = c00.x, cb0 = c00.y;
  const int32_t *par = rowpar + (size_t)a * lmax;
  double2 t[DIJ_MAXL];    // <p_j|psi> = i^(l_j odd) z_j
  for (int jj = 0; jj < nl; jj++) t[jj] = make_double2(0.0, 0.0);
  for (int s = 0; s < nsplit; s++) {
    const double *src = part + ((size_t)s * nproj + first) * n2 + 2 * b;
#pragma unroll 4
    for (int jj = 0; jj < nl; jj++) {
      const double2 v = *reinterpret_cast<const double2 *>(src + (size_t)jj * n2);
      t[jj].x += v.x; t[jj].y += v.y;
    }
  }
  for (int jj = 0; jj < nl; jj++) {
    const double za = 2.0 * t[jj].x - p0[first + jj] * ca0, zb = 2.0 * t[jj].y - p0[first + jj] * cb0;
    t[jj] = par[jj] ? make_double2(-zb, za) : make_double2(za, zb);
  }
  if (!dij) {
    double2 *dst = cpr + (size_t)b * nproj + first;
    for (int ii = 0; ii < nl; ii++) dst[ii] = t[ii];
    return;
  }
  const double *D = dij + (size_t)a * lmax * lmax;
  double2 *da = cpr + (size_t)(2 * b) * ldc + first, *db = da + ldc;      // ldc: row pitch of c' (complex elements)
  for (int ii = 0; ii < nl; ii++) {
    double sr = 0.0, si = 0.0;
    for (int jj = 0; jj < nl; jj++) { const double d = D[ii * lmax + jj]; sr += d * t[jj].x; si += d * t[jj].y; }
    const double yr = par[ii] ? si : sr, yi = par[ii] ? -sr : si;     // y = (-i)^(l_i odd) (sr + i si)
    da[ii] = make_double2(yr, 0.0); db[ii] = make_double2(yi, 0.0);
  }
}

// hpsi[b][g] = (accumulate ? hpsi : 0) + diag[g] psi + h_A(+-G) + i h_B(+-G), then the optional recurrence combination
__global__ void sym_combine_kernel(const double2 *__restrict__ Y, const double2 *__restrict__ psi, double2 *__restrict__ hpsi,
                                   const double *const *kin, const int32_t *__restrict__ f2h, int npw, int mpw, int nh,
                                   int accumulate, int with_kin, int cheb, double sh, double sy, double sx,
                                   const double2 *__restrict__ xprev) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
  if (g >= npw) return;
  const int t = f2h[g], h = (t > 0 ? t : -t) - 1;
  double2 a = Y[(size_t)(2 * b) * nh + h], c = Y[(size_t)(2 * b + 1) * nh + h];
  if (t < 0) { a.y = -a.y; c.y = -c.y; }
  double2 r = make_double2(a.x - c.y, a.y + c.x);
  const size_t off = (size_t)b * mpw + g;
  if (with_kin) { const double2 x = psi[off]; const double kg = kin[0][g]; r.x += kg * x.x; r.y += kg * x.y; }
  if (accumulate) { const double2 hh = hpsi[off]; r.x += hh.x; r.y += hh.y; }
  if (cheb) {
    const double2 y = psi[off], xp = sx != 0.0 ? xprev[off] : make_double2(0.0, 0.0);
    r.x = sh * r.x + sy * y.x + sx * xp.x; r.y = sh * r.y + sy * y.y + sx * xp.y;
  }
  hpsi[off] = r;
}

// Can this plan run the symmetric-table GEMMs?  Builds the half-sphere tables at the first call.
static bool sym_ready(dft_plan *p) {
  if (p->sym_state == 0) {
    p->sym_state = -1;
    if (p->nkpt == 1 && p->nproj > 0 && p->mpw > 0 && p->kp[0].k[0] == 0.0 && p->kp[0].k[1] == 0.0 && p->kp[0].k[2] == 0.0) {
      if (gamma_build(p, false) == DFT_OK && p->gam && p->gam->nh > 0) p->sym_state = 1;
    }
  }
  return p->sym_state == 1;
}

#include "nonlocal_strassen.inc"

static int nonlocal_apply_sym(dft_plan *p, const double *psi, double *hpsi, int nband, bool accumulate, bool with_kin, cudaStream_t st,
                              const double *dmat, const double *const *diag, double *cprj_out, const Recurrence *rec, double *spsi) {
  GammaData *G = p->gam;
  if (!p->gam_attr_done) {
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm1_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm2_multi_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    p->gam_attr_done = true;
  }
  const int nh = G->nh, nproj = p->nproj, mpw = p->mpw, n2 = 2 * nband;
  const double *const *d_kin = diag ? diag : p->d_kinptr;
  if (!dmat) dmat = p->d_dij;
  int rc;
  const int64_t need_x = (int64_t)n2 * nh * 16;
  if (need_x > p->symx_bytes || !p->d_symx) {
    if (p->d_symx) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->d_symx); p->d_symx = nullptr; p->symx_bytes = 0; }
    if (cudaMalloc(&p->d_symx, need_x + 256) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes for the symmetric halves of the bands", (long long)need_x); return DFT_ERR_ALLOC; }
    p->symx_bytes = need_x;
  }
  double2 *X = reinterpret_cast<double2 *>(p->d_symx);
  if (strassen_wanted(p, nband))        // seven half-size products per GEMM instead of eight (nonlocal_strassen.inc)
    return nonlocal_apply_sym_strassen(p, psi, hpsi, nband, accumulate, with_kin, st, dmat, d_kin, cprj_out, rec, spsi, X, false);
  Gemm1Params q1;
  q1.nproj = nproj; q1.nband = n2; q1.nslab = (nh + 7) / 8;
  q1.tiles_m = (nproj + NL_BM - 1) / NL_BM; q1.tiles_n = (n2 + NL_BN - 1) / NL_BN;
  int ns = p->splitk > 0 ? p->splitk : choose_splitk(q1.tiles_m * q1.tiles_n, q1.nslab, p->sm_count, 1);
  if (ns > q1.nslab) ns = q1.nslab;
  q1.slabs_per_split = (q1.nslab + ns - 1) / ns;
  ns = (q1.nslab + q1.slabs_per_split - 1) / q1.slabs_per_split;
  q1.nsplit = ns;
  // row pitch of c': a power-of-two pitch (4096 projectors = 64 KB) makes the 64 rows of a TMA box of GEMM-2 collide in L2
  const int ldc = (nproj % 256 == 0) ? nproj + 8 : nproj;
  const int64_t need_part = (int64_t)ns * nproj * n2 * 8, need_cprj = (int64_t)n2 * ldc * 16;
  if (need_part > p->part_bytes || !p->d_part) {
    if (p->d_part) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->d_part); p->d_part = nullptr; }
    if (cudaMalloc(&p->d_part, need_part) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes of split-K scratch", (long long)need_part); p->part_bytes = 0; return DFT_ERR_ALLOC; }
    p->part_bytes = need_part;
  }
  if (need_cprj > p->cprj_bytes || !p->d_cprj) {
    if (p->d_cprj) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->d_cprj); p->d_cprj = nullptr; }
    if (cudaMalloc(&p->d_cprj, need_cprj) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes for cprj", (long long)need_cprj); p->cprj_bytes = 0; return DFT_ERR_ALLOC; }
    p->cprj_bytes = need_cprj;
  }
  q1.part = reinterpret_cast<double2 *>(p->d_part);
  // tensor maps, kept between calls like those of the complex path
  SymMaps *C = p->sym_maps;
  if (!C) { C = new SymMaps(); p->sym_maps = C; }
  const uint64_t rowb = (uint64_t)nh * 16;
  if (C->ptab != G->d_ptab) {
    if ((rc = make_map(p, &C->mapP1, G->d_ptab, 2 * (uint64_t)nh, nproj, 1, rowb, rowb * nproj, NL_BM))) return rc;
    cuuint64_t dims[4] = {16, (cuuint64_t)nproj, ((cuuint64_t)nh + 7) / 8, 1};
    cuuint64_t strides[3] = {rowb, 128, rowb * nproj};
    cuuint32_t box[4] = {16, 8, NL_BM / 8, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = ((EncodeFn)p->encode_fn)(&C->mapP2, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, G->d_ptab, dims, strides, box, estr,
                                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                          CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled (symmetric GEMM-2 P map) failed (%d)", (int)r); return DFT_ERR_CUDA; }
    C->ptab = G->d_ptab;
  }
  if (C->x != X || C->n2_x != n2) {
    if ((rc = make_map(p, &C->mapX, X, 2 * (uint64_t)nh, n2, 1, rowb, rowb * n2, NL_BN))) return rc;
    C->x = X; C->n2_x = n2;
  }
  if (C->cprj != p->d_cprj || C->n2_c != n2) {
    if ((rc = make_map(p, &C->mapC, p->d_cprj, 2 * (uint64_t)nproj, n2, 1, (uint64_t)ldc * 16, (uint64_t)ldc * 16 * n2, NL_BN))) return rc;
    C->cprj = p->d_cprj; C->n2_c = n2;
  }
  const double2 *cpsi = reinterpret_cast<const double2 *>(psi);
  // ---- halves, GEMM-1 (real)
  phase_begin(p, 9, st);
  sym_split_kernel<<<dim3((nh + 255) / 256, nband), 256, 0, st>>>(cpsi, X, G->d_h2f, G->d_h2fneg, mpw, nh);
  phase_end(p, 9, st, 1);
  phase_begin(p, 5, st);
  gemm1_kernel<true><<<dim3(q1.tiles_m * q1.tiles_n, ns, 1), NL_THREADS_P, NL_SMEM, st>>>(C->mapP1, C->mapX, q1);
  phase_end(p, 5, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  // ---- D_ij (complex step on z = r_A + i r_B)
  phase_begin(p, 6, st);
  dij_sym_kernel<<<dim3((nband + 127) / 128, p->natom, 1), 128, 0, st>>>(
      p->d_part, reinterpret_cast<double2 *>(cprj_out ? cprj_out : p->d_cprj), cprj_out ? nullptr : dmat, p->d_typat, p->d_nlmn,
      p->d_atom_first, G->d_rowpar, G->d_p0, cpsi, mpw, p->lmax, nproj, nband, ns, ldc);
  phase_end(p, 6, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  if (cprj_out) return DFT_OK;
  // ---- GEMM-2 (real) into the halves buffer, then recombination + diagonal + accumulation
  Gemm2Params q2;
  q2.nproj = nproj; q2.nband = n2; q2.mpw = nh; q2.nslab = (nproj + 7) / 8;
  q2.tiles_n = q1.tiles_n; q2.accumulate = 0; q2.with_kin = 0; q2.with_nl = 1;
  q2.npw = G->d_npw; q2.kin = G->d_kinptr; q2.psi = X; q2.hpsi = X;
  q2.cheb = 0; q2.sh = 1.0; q2.sy = 0.0; q2.sx = 0.0; q2.xprev = nullptr; q2.raw = 0;
  const int tiles_m2 = (nh + NL_BM - 1) / NL_BM;
  const dim3 cgrid((mpw + 255) / 256, nband);
  phase_begin(p, 7, st);
  gemm2_kernel<true><<<dim3(q2.tiles_n * tiles_m2, 1, 1), NL_THREADS_P, NL_SMEM, st>>>(C->mapP2, C->mapC, q2);
  phase_end(p, 7, st, 1);
  phase_begin(p, 9, st);
  sym_combine_kernel<<<cgrid, 256, 0, st>>>(X, cpsi, reinterpret_cast<double2 *>(hpsi), d_kin, G->d_f2h, p->kp[0].npw, mpw, nh, accumulate,
                                            with_kin, rec != nullptr, rec ? rec->sh : 1.0, rec ? rec->sy : 0.0, rec ? rec->sx : 0.0,
                                            rec ? reinterpret_cast<const double2 *>(rec->xprev) : nullptr);
  phase_end(p, 9, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  if (spsi) {   // S psi from the same projections (dft_apply_hs): s_ij step, GEMM-2, recombination with a unit diagonal
    phase_begin(p, 6, st);
    dij_sym_kernel<<<dim3((nband + 127) / 128, p->natom, 1), 128, 0, st>>>(
        p->d_part, reinterpret_cast<double2 *>(p->d_cprj), p->d_sij, p->d_typat, p->d_nlmn, p->d_atom_first, G->d_rowpar, G->d_p0, cpsi,
        mpw, p->lmax, nproj, nband, ns, ldc);
    phase_end(p, 6, st, 1);
    phase_begin(p, 7, st);
    gemm2_kernel<true><<<dim3(q2.tiles_n * tiles_m2, 1, 1), NL_THREADS_P, NL_SMEM, st>>>(C->mapP2, C->mapC, q2);
    phase_end(p, 7, st, 1);
    phase_begin(p, 9, st);
    sym_combine_kernel<<<cgrid, 256, 0, st>>>(X, cpsi, reinterpret_cast<double2 *>(spsi), p->d_oneptr, G->d_f2h, p->kp[0].npw, mpw, nh, 0, 1,
                                              0, 1.0, 0.0, 0.0, nullptr);
    phase_end(p, 9, st, 1);
    DFT_CUDA_CHECK(cudaGetLastError());
  }
  return DFT_OK;
}

// dmat: per-atom matrices applied between the GEMMs (null = the plan's D_ij); diag: per-k-point device pointers to the
// diagonal multiplying psi in the epilogue (null = the kinetic energies); cprj_out (device, [nkpt][nband][nproj]
// complex): if given, only GEMM-1 and the split-K reduction run and <p|psi> is written there.
int nonlocal_apply(dft_plan *p, const double *psi, double *hpsi, int nband, bool accumulate, bool with_kin, bool with_nl,
                   cudaStream_t st, const double *dmat, const double *const *diag, double *cprj_out, const Recurrence *rec,
                   double *spsi, const double *dspin) {
  if (p->mpw == 0 || nband == 0) return DFT_OK;
  if (cprj_out && p->nproj == 0) return DFT_OK;
  if (p->nproj == 0) with_nl = false;
  if (!with_nl && !with_kin && accumulate && !rec) return DFT_OK;
  if (!p->nl_attr_done) {   // per plan (= per device), not per process
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm1_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm1_kernel<false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm1_kernel<false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm1_3m_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm2_3m_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm1_fac_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, FC_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm2_fac_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, FD_SMEM));
    p->nl_attr_done = true;
  }
  // k = 0: the projector table is symmetric under G -> -G and both GEMMs run as real GEMMs on the half sphere
  // (option gemm_sym: 1 = wherever possible, 2 = automatic: only where the GEMMs are large enough to pay for the two extra
  // launches, nproj npw nband >= 1e8 complex multiply-adds; tiny cells are launch-bound)
  if (with_nl && (p->gemm_sym == 1 || (p->gemm_sym == 2 && (double)p->nproj * p->mpw * nband >= 1e8)) && p->proj_mode == 0 && !dspin &&
      nband <= 32767 && sym_ready(p))
    return nonlocal_apply_sym(p, psi, hpsi, nband, accumulate, with_kin, st, dmat, diag, cprj_out, rec, spsi);
  const int32_t *d_npw = p->d_npw;
  const double *const *d_kin = diag ? diag : p->d_kinptr;
  if (!dmat) dmat = p->d_dij;
  int rc;
  const double2 *cpsi = reinterpret_cast<const double2 *>(psi);
  double2 *chpsi = reinterpret_cast<double2 *>(hpsi);
  if (with_nl && p->nl_tiny && p->proj_mode == 0 && !cprj_out && !spsi && !dspin && p->nproj <= NLT_MAXP && nband <= 65535 &&
      p->nkpt <= 65535 && (double)p->nproj * p->mpw * nband * p->nkpt <= 1e6) {
    phase_begin(p, 7, st);
    nl_tiny_kernel<<<dim3(nband, p->nkpt), NLT_THREADS, 0, st>>>(
        reinterpret_cast<const double2 *>(p->d_ptab), cpsi, chpsi, dmat, p->d_typat, p->d_nlmn, p->d_atom_first, d_npw, d_kin, p->natom,
        p->lmax, p->nproj, nband, p->mpw, accumulate, with_kin, rec != nullptr, rec ? rec->sh : 1.0, rec ? rec->sy : 0.0,
        rec ? rec->sx : 0.0, rec ? reinterpret_cast<const double2 *>(rec->xprev) : nullptr);
    phase_end(p, 7, st, 1);
    DFT_CUDA_CHECK(cudaGetLastError());
    return DFT_OK;
  }
  if (!with_nl) {
    dim3 grid((p->mpw + 255) / 256 < 64 ? (p->mpw + 255) / 256 : 64, nband, p->nkpt);
    phase_begin(p, 7, st);
    kin_only_kernel<<<grid, 256, 0, st>>>(cpsi, chpsi, d_kin, d_npw, nband, p->mpw, accumulate, with_kin, rec != nullptr,
                                          rec ? rec->sh : 1.0, rec ? rec->sy : 0.0, rec ? rec->sx : 0.0,
                                          rec ? reinterpret_cast<const double2 *>(rec->xprev) : nullptr);
    phase_end(p, 7, st, 1);
    if (spsi) {   // no projectors: S = 1
      phase_begin(p, 7, st);
      kin_only_kernel<<<grid, 256, 0, st>>>(cpsi, reinterpret_cast<double2 *>(spsi), p->d_oneptr, d_npw, nband, p->mpw, 0, 1, 0, 1.0, 0.0,
                                            0.0, nullptr);
      phase_end(p, 7, st, 1);
    }
    DFT_CUDA_CHECK(cudaGetLastError());
    return DFT_OK;
  }
  const int nproj = p->nproj, mpw = p->mpw, nkpt = p->nkpt;
  // ---- GEMM-1
  Gemm1Params q1;
  q1.nproj = nproj; q1.nband = nband;
  q1.nslab = (mpw + 7) / 8;
  const bool fac = p->proj_mode == 1;     // factorised projectors: tiles of 16 atoms instead of 128 table rows
  // few projectors (nproj <= 64): the 4-product GEMM-1 with a 32- or 64-row tile instead of 128 padded rows
  const int skinny_mb = (!fac && nproj <= 32) ? 1 : ((!fac && nproj <= 64) ? 2 : 0);
  const int bm1 = skinny_mb ? 32 * skinny_mb : NL_BM;
  int fac_tiles = 0;                      // tiles of 16 projector blocks, summed over the groups of atom types
  if (fac) for (const FacGroup &G : p->fac_groups) fac_tiles += (G.nblk + FC_BA - 1) / FC_BA;
  q1.tiles_m = fac ? fac_tiles : (nproj + bm1 - 1) / bm1; q1.tiles_n = (nband + NL_BN - 1) / NL_BN;
  int ns = p->splitk > 0 ? p->splitk : choose_splitk(q1.tiles_m * q1.tiles_n, q1.nslab, p->sm_count, nkpt);
  if (ns > q1.nslab) ns = q1.nslab;
  q1.slabs_per_split = (q1.nslab + ns - 1) / ns;
  ns = (q1.nslab + q1.slabs_per_split - 1) / q1.slabs_per_split;
  q1.nsplit = ns;
  int64_t need_part = (int64_t)nkpt * ns * nproj * nband * 16, need_cprj = (int64_t)nkpt * nband * nproj * 16;
  if (need_part > p->part_bytes || !p->d_part) {
    if (p->d_part) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->d_part); p->d_part = nullptr; }
    if (cudaMalloc(&p->d_part, need_part) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes of split-K scratch", (long long)need_part); p->part_bytes = 0; return DFT_ERR_ALLOC; }
    p->part_bytes = need_part;
  }
  if (need_cprj > p->cprj_bytes || !p->d_cprj) {
    if (p->d_cprj) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->d_cprj); p->d_cprj = nullptr; }
    if (cudaMalloc(&p->d_cprj, need_cprj) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes for cprj", (long long)need_cprj); p->cprj_bytes = 0; return DFT_ERR_ALLOC; }
    p->cprj_bytes = need_cprj;
  }
  q1.part = reinterpret_cast<double2 *>(p->d_part);
  // the four tensor maps of the table mode are kept between calls (encoding them costs more host time than launching the
  // kernels of a small cell) and re-encoded only when the pointer or shape they describe changed
  NlMaps *C = p->nl_maps;
  if (!C) { C = new NlMaps(); p->nl_maps = C; }
  CUtensorMap &mapP1 = C->mapP1, &mapPsi = C->mapPsi, &mapP2 = C->mapP2, &mapC = C->mapC;
  uint64_t rowb = (uint64_t)mpw * 16;
  const bool tab_same = !fac && C->ptab == p->d_ptab && C->bm1 == bm1;
  if (!fac && !tab_same && (rc = make_map(p, &mapP1, p->d_ptab, 2 * (uint64_t)mpw, nproj, nkpt, rowb, rowb * nproj, bm1))) return rc;
  if (C->psi != psi || C->nband_psi != nband) {
    if ((rc = make_map(p, &mapPsi, psi, 2 * (uint64_t)mpw, nband, nkpt, rowb, rowb * nband, NL_BN))) return rc;
    C->psi = psi; C->nband_psi = nband;
  }
  // factorised mode: one S map for all atoms and one pair of FY maps per group of atom types (projtab.cu)
  CUtensorMap mapS1, mapS2;
  std::vector<CUtensorMap> mapF1, mapF2;
  const size_t ngrp = fac ? p->fac_groups.size() : 0;
  if (fac) {
    if (!p->d_stab || !p->d_fytab) { set_error("factor tables missing"); return DFT_ERR_NOT_READY; }
    const uint64_t frow = (uint64_t)p->ldf * 8, nfr = (uint64_t)p->nfrow;
    if ((rc = make_map(p, &mapS1, p->d_stab, 2 * (uint64_t)mpw, p->natom, nkpt, rowb, rowb * p->natom, FC_BA))) return rc;
    if ((rc = make_map_plain(p, &mapS2, p->d_stab, 2 * (uint64_t)mpw, p->natom, nkpt, rowb, rowb * p->natom, 2 * NL_BM, 1))) return rc;
    mapF1.resize(ngrp); mapF2.resize(ngrp);
    for (size_t g = 0; g < ngrp; g++) {
      const FacGroup &G = p->fac_groups[g];
      const double *base = p->d_fytab + (size_t)G.frow0 * p->ldf;
      if ((rc = make_map_plain(p, &mapF1[g], base, p->ldf, G.nfrow, nkpt, frow, frow * nfr, 8, (uint32_t)G.nfrow))) return rc;
      if ((rc = make_map_plain(p, &mapF2[g], base, p->ldf, G.nfrow, nkpt, frow, frow * nfr, FD_FLD, (uint32_t)G.nfrow))) return rc;
    }
  }
  if (!fac && !tab_same) {
    // GEMM-2 reads P "M-major": view each table row as [g-block][16 doubles] and put the projector
    // index between them, so ONE box {16, 8 rows, 16 g-blocks} brings a 128 g x 8 p tile in the
    // [g-block][p][8 complex] order the fragments want (16 separate 1 KB boxes starved the MMA loop:
    // profiles/r1_gemm2_tma.md).  The last g-block of a row may run into the next row (or the 256-byte
    // pad after the table); those values only reach output rows g >= npw, which are never stored.
    cuuint64_t dims[4] = {16, (cuuint64_t)nproj, ((cuuint64_t)mpw + 7) / 8, (cuuint64_t)nkpt};
    cuuint64_t strides[3] = {rowb, 128, rowb * nproj};
    cuuint32_t box[4] = {16, 8, NL_BM / 8, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = ((EncodeFn)p->encode_fn)(&mapP2, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, p->d_ptab, dims, strides, box, estr,
                                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                          CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled (GEMM-2 P map) failed (%d)", (int)r); return DFT_ERR_CUDA; }
    C->ptab = p->d_ptab; C->bm1 = bm1;
  }
  if (C->cprj != p->d_cprj || C->nband_c != nband) {
    if ((rc = make_map(p, &mapC, p->d_cprj, 2 * (uint64_t)nproj, nband, nkpt, (uint64_t)nproj * 16, (uint64_t)nproj * 16 * nband, NL_BN))) return rc;
    C->cprj = p->d_cprj; C->nband_c = nband;
  }
  phase_begin(p, 5, st);
  if (fac) {
    for (size_t g = 0; g < ngrp; g++) {     // every group writes its own rows of the partial sums
      const FacGroup &G = p->fac_groups[g];
      Fac1Params f1;
      f1.nblk = G.nblk; f1.nfrow = G.nfrow; f1.nband = nband; f1.nproj = nproj; f1.nslab = q1.nslab; f1.nsplit = q1.nsplit;
      f1.slabs_per_split = q1.slabs_per_split; f1.tiles_n = q1.tiles_n;
      f1.blk_atom = p->d_blk_atom + G.blk0; f1.blk_frow = p->d_blk_frow + G.blk0; f1.blk_first = p->d_blk_first + G.blk0;
      f1.blk_nl = p->d_blk_nl + G.blk0; f1.part = q1.part;
      const int tiles_a = (G.nblk + FC_BA - 1) / FC_BA;
      gemm1_fac_kernel<<<dim3(tiles_a * q1.tiles_n, ns, nkpt), FC_THREADS, FC_SMEM, st>>>(mapPsi, mapS1, mapF1[g], f1);
    }
  } else if (skinny_mb == 1) gemm1_kernel<false, 1><<<dim3(q1.tiles_m * q1.tiles_n, ns, nkpt), NL_THREADS_P, NL_SMEM, st>>>(mapP1, mapPsi, q1);
  else if (skinny_mb == 2) gemm1_kernel<false, 2><<<dim3(q1.tiles_m * q1.tiles_n, ns, nkpt), NL_THREADS_P, NL_SMEM, st>>>(mapP1, mapPsi, q1);
  else if (p->gemm_3m) gemm1_3m_kernel<<<dim3(q1.tiles_m * q1.tiles_n, ns, nkpt), NL3_THREADS, NL_SMEM, st>>>(mapP1, mapPsi, q1);
  else gemm1_kernel<false><<<dim3(q1.tiles_m * q1.tiles_n, ns, nkpt), NL_THREADS_P, NL_SMEM, st>>>(mapP1, mapPsi, q1);
  phase_end(p, 5, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  // ---- D_ij
  phase_begin(p, 6, st);
  if (dspin && !cprj_out)
    dij_spinor_kernel<<<dim3((nband / 2 + 127) / 128, p->natom, nkpt), 128, 0, st>>>(
        q1.part, reinterpret_cast<double2 *>(p->d_cprj), reinterpret_cast<const double2 *>(dspin), p->d_typat, p->d_nlmn,
        p->d_atom_first, p->lmax, nproj, nband, ns);
  else
    dij_kernel<<<dim3((nband + DIJ_BX - 1) / DIJ_BX, p->natom, nkpt), dim3(DIJ_BX, DIJ_YS), 0, st>>>(
        q1.part, reinterpret_cast<double2 *>(cprj_out ? cprj_out : p->d_cprj), cprj_out ? nullptr : dmat, p->d_typat, p->d_nlmn,
        p->d_atom_first, p->natom, p->lmax, nproj, nband, ns);
  phase_end(p, 6, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  if (cprj_out) return DFT_OK;
  // ---- GEMM-2
  Gemm2Params q2;
  q2.nproj = nproj; q2.nband = nband; q2.mpw = mpw; q2.nslab = (nproj + 7) / 8;
  q2.tiles_n = q1.tiles_n; q2.accumulate = accumulate; q2.with_kin = with_kin; q2.with_nl = 1;
  q2.npw = d_npw; q2.kin = d_kin; q2.psi = cpsi; q2.hpsi = chpsi;
  q2.cheb = rec != nullptr; q2.sh = rec ? rec->sh : 1.0; q2.sy = rec ? rec->sy : 0.0; q2.sx = rec ? rec->sx : 0.0;
  q2.xprev = rec ? reinterpret_cast<const double2 *>(rec->xprev) : nullptr; q2.raw = 0;
  int tiles_m2 = (mpw + NL_BM - 1) / NL_BM;
  phase_begin(p, 7, st);
  // factorised GEMM-2, once per group of atom types: the first launch carries the caller's accumulate flag and the kinetic
  // term, the later ones add to its output, and the last one applies the recurrence to the total
  auto launch_gemm2_fac = [&](Gemm2Params q) {
    for (size_t g = 0; g < ngrp; g++) {
      const FacGroup &G = p->fac_groups[g];
      Gemm2Params qg = q;
      qg.nslab = G.nblk;
      if (g > 0) { qg.accumulate = 1; qg.with_kin = 0; }
      if (g + 1 < ngrp) { qg.cheb = 0; }
      gemm2_fac_kernel<<<dim3(q.tiles_n * tiles_m2, 1, nkpt), FC_THREADS, FD_SMEM, st>>>(
          mapC, mapS2, mapF2[g], qg, p->d_blk_atom + G.blk0, p->d_blk_frow + G.blk0, p->d_blk_first + G.blk0, G.nfrow);
    }
  };
  if (fac) launch_gemm2_fac(q2);
  else if (p->gemm_3m) gemm2_3m_kernel<<<dim3(q2.tiles_n * tiles_m2, 1, nkpt), NL3_THREADS, NL_SMEM, st>>>(mapP2, mapC, q2);
  else gemm2_kernel<false><<<dim3(q2.tiles_n * tiles_m2, 1, nkpt), NL_THREADS_P, NL_SMEM, st>>>(mapP2, mapC, q2);
  phase_end(p, 7, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  if (spsi) {
    // second output from the SAME projections (dft_apply_hs): S psi = psi + sum |p> s <p|psi>.  The split-K partials of
    // GEMM-1 are still there; reduce them again with s_ij into c' and back-project with a unit diagonal.
    phase_begin(p, 6, st);
    dij_kernel<<<dim3((nband + DIJ_BX - 1) / DIJ_BX, p->natom, nkpt), dim3(DIJ_BX, DIJ_YS), 0, st>>>(q1.part, reinterpret_cast<double2 *>(p->d_cprj), p->d_sij, p->d_typat,
                                                                          p->d_nlmn, p->d_atom_first, p->natom, p->lmax, nproj, nband, ns);
    phase_end(p, 6, st, 1);
    q2.accumulate = 0; q2.with_kin = 1; q2.kin = p->d_oneptr; q2.hpsi = reinterpret_cast<double2 *>(spsi);
    q2.cheb = 0; q2.sh = 1.0; q2.sy = 0.0; q2.sx = 0.0; q2.xprev = nullptr;
    phase_begin(p, 7, st);
    if (fac) launch_gemm2_fac(q2);
    else if (p->gemm_3m) gemm2_3m_kernel<<<dim3(q2.tiles_n * tiles_m2, 1, nkpt), NL3_THREADS, NL_SMEM, st>>>(mapP2, mapC, q2);
    else gemm2_kernel<false><<<dim3(q2.tiles_n * tiles_m2, 1, nkpt), NL_THREADS_P, NL_SMEM, st>>>(mapP2, mapC, q2);
    phase_end(p, 7, st, 1);
    DFT_CUDA_CHECK(cudaGetLastError());
  }
  return DFT_OK;
}

// ---------------------------------------------------------------- Gamma storage: real GEMMs on the half sphere
int nonlocal_apply_gamma(dft_plan *p, const double *psi, double *hpsi, int nband, bool accumulate, bool with_kin, bool with_nl,
                         cudaStream_t st, const Recurrence *rec) {
  GammaData *G = p->gam;
  if (!G || G->nh == 0 || nband == 0) return DFT_OK;
  if (p->nproj == 0) with_nl = false;
  if (!with_nl && !with_kin && accumulate && !rec) return DFT_OK;
  if (!p->gam_attr_done) {
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm1_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    DFT_CUDA_CHECK(cudaFuncSetAttribute(gemm2_multi_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, NL_SMEM));
    p->gam_attr_done = true;
  }
  const int mpw = G->nh, nproj = p->nproj;
  const double2 *cpsi = reinterpret_cast<const double2 *>(psi);
  double2 *chpsi = reinterpret_cast<double2 *>(hpsi);
  if (!with_nl) {
    dim3 grid((mpw + 255) / 256 < 64 ? (mpw + 255) / 256 : 64, nband, 1);
    phase_begin(p, 7, st);
    kin_only_kernel<<<grid, 256, 0, st>>>(cpsi, chpsi, G->d_kinptr, G->d_npw, nband, mpw, accumulate, with_kin, rec != nullptr,
                                          rec ? rec->sh : 1.0, rec ? rec->sy : 0.0, rec ? rec->sx : 0.0,
                                          rec ? reinterpret_cast<const double2 *>(rec->xprev) : nullptr, 1);
    phase_end(p, 7, st, 1);
    DFT_CUDA_CHECK(cudaGetLastError());
    return DFT_OK;
  }
  int rc;
  if (nband % 2 == 0 && strassen_wanted(p, nband / 2))     // one Strassen level on both real GEMMs (nonlocal_strassen.inc)
    return nonlocal_apply_sym_strassen(p, psi, hpsi, nband, accumulate, with_kin, st, p->d_dij, G->d_kinptr, nullptr, rec, nullptr, cpsi, true);
  Gemm1Params q1;
  q1.nproj = nproj; q1.nband = nband; q1.nslab = (mpw + 7) / 8;
  q1.tiles_m = (nproj + NL_BM - 1) / NL_BM; q1.tiles_n = (nband + NL_BN - 1) / NL_BN;
  int ns = p->splitk > 0 ? p->splitk : choose_splitk(q1.tiles_m * q1.tiles_n, q1.nslab, p->sm_count, 1);
  if (ns > q1.nslab) ns = q1.nslab;
  q1.slabs_per_split = (q1.nslab + ns - 1) / ns;
  ns = (q1.nslab + q1.slabs_per_split - 1) / q1.slabs_per_split;
  q1.nsplit = ns;
  int64_t need_part = (int64_t)ns * nproj * nband * 8, need_cprj = (int64_t)nband * nproj * 16;
  if (need_part > p->part_bytes || !p->d_part) {
    if (p->d_part) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->d_part); p->d_part = nullptr; }
    if (cudaMalloc(&p->d_part, need_part) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes of split-K scratch", (long long)need_part); p->part_bytes = 0; return DFT_ERR_ALLOC; }
    p->part_bytes = need_part;
  }
  if (need_cprj > p->cprj_bytes || !p->d_cprj) {
    if (p->d_cprj) { DFT_CUDA_CHECK(cudaStreamSynchronize(st)); cudaFree(p->d_cprj); p->d_cprj = nullptr; }
    if (cudaMalloc(&p->d_cprj, need_cprj) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %lld bytes for cprj", (long long)need_cprj); p->cprj_bytes = 0; return DFT_ERR_ALLOC; }
    p->cprj_bytes = need_cprj;
  }
  q1.part = reinterpret_cast<double2 *>(p->d_part);
  CUtensorMap mapP1, mapPsi, mapP2, mapC;
  const uint64_t rowb = (uint64_t)mpw * 16;
  if ((rc = make_map(p, &mapP1, G->d_ptab, 2 * (uint64_t)mpw, nproj, 1, rowb, rowb * nproj, NL_BM))) return rc;
  if ((rc = make_map(p, &mapPsi, psi, 2 * (uint64_t)mpw, nband, 1, rowb, rowb * nband, NL_BN))) return rc;
  {
    cuuint64_t dims[4] = {16, (cuuint64_t)nproj, ((cuuint64_t)mpw + 7) / 8, 1};
    cuuint64_t strides[3] = {rowb, 128, rowb * nproj};
    cuuint32_t box[4] = {16, 8, NL_BM / 8, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = ((EncodeFn)p->encode_fn)(&mapP2, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, G->d_ptab, dims, strides, box, estr,
                                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                          CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled (Gamma GEMM-2 P map) failed (%d)", (int)r); return DFT_ERR_CUDA; }
  }
  if ((rc = make_map(p, &mapC, p->d_cprj, 2 * (uint64_t)nproj, nband, 1, (uint64_t)nproj * 16, (uint64_t)nproj * 16 * nband, NL_BN))) return rc;
  phase_begin(p, 5, st);
  gemm1_kernel<true><<<dim3(q1.tiles_m * q1.tiles_n, ns, 1), NL_THREADS_P, NL_SMEM, st>>>(mapP1, mapPsi, q1);
  phase_end(p, 5, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  phase_begin(p, 6, st);
  dij_gamma_kernel<<<dim3((nband + 127) / 128, p->natom, 1), 128, 0, st>>>(
      p->d_part, reinterpret_cast<double2 *>(p->d_cprj), p->d_dij, p->d_typat, p->d_nlmn, p->d_atom_first, G->d_rowpar, G->d_p0,
      cpsi, mpw, p->lmax, nproj, nband, ns);
  phase_end(p, 6, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  Gemm2Params q2;
  q2.nproj = nproj; q2.nband = nband; q2.mpw = mpw; q2.nslab = (nproj + 7) / 8;
  q2.tiles_n = q1.tiles_n; q2.accumulate = accumulate; q2.with_kin = with_kin; q2.with_nl = 1;
  q2.npw = G->d_npw; q2.kin = G->d_kinptr; q2.psi = cpsi; q2.hpsi = chpsi;
  q2.cheb = rec != nullptr; q2.sh = rec ? rec->sh : 1.0; q2.sy = rec ? rec->sy : 0.0; q2.sx = rec ? rec->sx : 0.0;
  q2.xprev = rec ? reinterpret_cast<const double2 *>(rec->xprev) : nullptr; q2.raw = 0;
  const int tiles_m2 = (mpw + NL_BM - 1) / NL_BM;
  phase_begin(p, 7, st);
  gemm2_kernel<true><<<dim3(q2.tiles_n * tiles_m2, 1, 1), NL_THREADS_P, NL_SMEM, st>>>(mapP2, mapC, q2);
  phase_end(p, 7, st, 1);
  DFT_CUDA_CHECK(cudaGetLastError());
  return DFT_OK;
}

int nonlocal_apply_spinor(dft_plan *p, const double *psi, double *hpsi, int nband, bool accumulate, bool with_kin, bool with_nl,
                          cudaStream_t st) {
  // (a vector potential changes the kinetic diagonal of both components alike)
  return nonlocal_apply(p, psi, hpsi, 2 * nband, accumulate, with_kin, with_nl, st, nullptr, p->vecpot_on ? p->d_kinaptr : nullptr, nullptr,
                        nullptr, nullptr, p->dspin_set ? p->d_dspin : nullptr);
}

}  // namespace dftb200
