/* oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU statement of
 *
 *      H|psi> = 1/2|k+G|^2 psi + FFT^-1[ V_loc(r) . FFT[psi] ] + sum_a sum_ij |p_a,i> D^a_ij <p_a,j|psi>
 *
 * (PAPER.md :456 "applying the Hamiltonian to a set of vectors"; :468-:475 Eq. 26 and the three
 * terms kinetic / local-by-FFT / non-local).  The paper prints only Eq. 26; every convention it is
 * silent on follows the numbered "readings" of SURVEY.md section 8(c) (restated in DESIGN.md).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or constant generator with
 * the CUDA library under paper_2507_08578_b200/csrc, and uses no BLAS / FFT library.
 *
 * Every function below is pinned by tests/test_oracle_*.py against closed forms, invariants,
 * brute force or numpy library routines; nothing is "parity unpinned".
 *
 * Layout conventions:
 *   rprimd[9]   row i = lattice vector a_i (bohr), row-major
 *   complex     interleaved (re, im) doubles
 *   V           [n3][n2][n1], i1 fastest;  box index idx = i1 + n1*(i2 + n2*i3)
 *   kg          [npw][3] int32, ascending idx;   psi/hpsi  [nband][ldpsi] complex
 *   per-type projector metadata padded to lmax = max nlmn:  lmn_l/m/irad [ntypat][lmax]
 *   radial tables f, f2: [ntypat][nrad_max][nq_max]; per type nq[t], dq[t]
 *   dij         [natom][lmax][lmax] real symmetric
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* 2*pi^2 and 2*pi rounded to double, written as literals (reading 1: the constant is part of the
 * bit-exact kinetic-energy rule). */
static const double TWO_PI_SQ = 0x1.3bd3cc9be45dep+4;   /* 19.739208802178716 */
static const double TWO_PI    = 0x1.921fb54442d18p+2;   /* 6.283185307179586  */
static const long double PI_L = 3.14159265358979323846264338327950288L;

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * Lattice algebra -- reading 1.  Bm = (A^-1)^T, rows b_i with a_i.b_j = delta_ij (no 2 pi);
 * gmet = Bm Bm^T.  Cofactor formula, operations in exactly the order written (bit-exact rule).
 * ------------------------------------------------------------------------------------------- */
void orc_lattice(const double *a, double *bm, double *gmet) {
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
  for (int i = 0; i < 9; i++) bm[i] = c[i] / det;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++)
      gmet[3 * i + j] = (bm[3 * i] * bm[3 * j] + bm[3 * i + 1] * bm[3 * j + 1]) + bm[3 * i + 2] * bm[3 * j + 2];
}

/* kin(m) = 2 pi^2 (k+m)^T gmet (k+m) = 1/2|k+G|^2 (Hartree).  Fixed order 11,22,33,2*12,2*13,2*23,
 * no FMA contraction (compile with -ffp-contract=off). */
double orc_kin(const double *gmet, const double *k, int m1, int m2, int m3) {
  double t0 = k[0] + (double)m1, t1 = k[1] + (double)m2, t2 = k[2] + (double)m3;
  double s = (t0 * t0) * gmet[0];
  s = s + (t1 * t1) * gmet[4];
  s = s + (t2 * t2) * gmet[8];
  s = s + 2.0 * ((t0 * t1) * gmet[1]);
  s = s + 2.0 * ((t0 * t2) * gmet[2]);
  s = s + 2.0 * ((t1 * t2) * gmet[5]);
  return TWO_PI_SQ * s;
}

static inline int unwrap(int i, int n) { return (i <= (n - 1) / 2) ? i : i - n; }   /* reading 3 */

/* ---------------------------------------------------------------------------------------------
 * Sphere -- readings 1-3 (BASELINE.json: "|k+G|^2/2 <= ecut", inclusive).  Brute force over ALL
 * box points in ascending box index; returns npw.  kg/igfft/kin may be NULL (count only);
 * at most `cap` entries are written.
 * ------------------------------------------------------------------------------------------- */
int64_t orc_sphere(const double *rprimd, const double *k, double ecut, const int32_t *n,
                   int32_t *kg, int32_t *igfft, double *kin, int64_t cap) {
  double bm[9], gmet[9];
  orc_lattice(rprimd, bm, gmet);
  int64_t npw = 0;
  for (int i3 = 0; i3 < n[2]; i3++)
    for (int i2 = 0; i2 < n[1]; i2++)
      for (int i1 = 0; i1 < n[0]; i1++) {
        int m1 = unwrap(i1, n[0]), m2 = unwrap(i2, n[1]), m3 = unwrap(i3, n[2]);
        double e = orc_kin(gmet, k, m1, m2, m3);
        if (e <= ecut) {
          if (npw < cap) {
            if (kg) { kg[3 * npw] = m1; kg[3 * npw + 1] = m2; kg[3 * npw + 2] = m3; }
            if (igfft) igfft[npw] = i1 + n[0] * (i2 + n[1] * i3);
            if (kin) kin[npw] = e;
          }
          npw++;
        }
      }
  return npw;
}

/* Does the whole sphere fit in the box (-floor(n/2) <= m <= floor((n-1)/2))?  Enumerates the
 * integer cube |m_j| <= bound_j with bound_j = ceil(|a_j| sqrt(2 ecut)/(2 pi) + |k_j|) + 1, which
 * contains the sphere because |(k+m)_j| = |a_j . q|/(2 pi) <= |a_j||q|/(2 pi).
 * Returns 1 if it fits, 0 otherwise; mmin/mmax receive the extents of the true sphere. */
int orc_sphere_extent(const double *rprimd, const double *k, double ecut, const int32_t *n,
                      int32_t *mmin, int32_t *mmax) {
  double bm[9], gmet[9];
  orc_lattice(rprimd, bm, gmet);
  int b[3];
  for (int j = 0; j < 3; j++) {
    const double *a = rprimd + 3 * j;
    double len = sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
    b[j] = (int)ceil(len * sqrt(2.0 * ecut) / TWO_PI + fabs(k[j])) + 1;
    mmin[j] = INT32_MAX; mmax[j] = INT32_MIN;
  }
  for (int m3 = -b[2]; m3 <= b[2]; m3++)
    for (int m2 = -b[1]; m2 <= b[1]; m2++)
      for (int m1 = -b[0]; m1 <= b[0]; m1++)
        if (orc_kin(gmet, k, m1, m2, m3) <= ecut) {
          int m[3] = {m1, m2, m3};
          for (int j = 0; j < 3; j++) {
            if (m[j] < mmin[j]) mmin[j] = m[j];
            if (m[j] > mmax[j]) mmax[j] = m[j];
          }
        }
  int fits = 1;
  for (int j = 0; j < 3; j++)
    if (mmin[j] <= mmax[j] && (mmin[j] < -(n[j] / 2) || mmax[j] > (n[j] - 1) / 2)) fits = 0;
  return fits;
}

/* ---------------------------------------------------------------------------------------------
 * Discrete Fourier transforms on the box.  Reading 4: G->r sign +, no scale; r->G sign -, 1/N.
 * T1: naive O(n^2) per line.  T2: textbook recursive mixed-radix Cooley-Tukey (smallest prime
 * factor first, naive DFT for a prime length).  Twiddles exp(sign 2 pi i j/n) from long double.
 * ------------------------------------------------------------------------------------------- */
static void twiddles(int n, int sign, double *w /* [n][2] */) {
  for (int j = 0; j < n; j++) {
    long double ang = 2.0L * PI_L * (long double)j / (long double)n;
    w[2 * j] = (double)cosl(ang);
    w[2 * j + 1] = (double)(sign * sinl(ang));
  }
}

/* out[j] = sum_k in[k] w^(j k), all lengths n, `in` strided by s (in complex elements) */
static void dft_naive(int n, const double *in, int s, double *out, const double *w, int wn) {
  int step = wn / n;  /* w holds the wn-th roots of unity; use every step-th */
  for (int j = 0; j < n; j++) {
    double sr = 0.0, si = 0.0;
    for (int k = 0; k < n; k++) {
      int t = (int)(((int64_t)j * k) % n) * step;
      double ar = in[2 * (size_t)k * s], ai = in[2 * (size_t)k * s + 1];
      sr += ar * w[2 * t] - ai * w[2 * t + 1];
      si += ar * w[2 * t + 1] + ai * w[2 * t];
    }
    out[2 * j] = sr; out[2 * j + 1] = si;
  }
}

static int smallest_factor(int n) {
  for (int p = 2; p * p <= n; p++)
    if (n % p == 0) return p;
  return n;
}

/* Decimation in time: X[k + m q] = sum_r w_n^{r (k + m q)} Y_r[k], Y_r = DFT_m of x[r::p]. */
static void fft_rec(int n, const double *in, int s, double *out, const double *w, int wn, double *tmp) {
  if (n == 1) { out[0] = in[0]; out[1] = in[1]; return; }
  int p = smallest_factor(n);
  if (p == n) { dft_naive(n, in, s, out, w, wn); return; }
  int m = n / p, step = wn / n;
  /* sub-transforms into tmp[r][m]; recursion scratch lives after the p*m block */
  for (int r = 0; r < p; r++) fft_rec(m, in + 2 * (size_t)r * s, s * p, tmp + 2 * (size_t)r * m, w, wn, tmp + 2 * (size_t)n);
  for (int q = 0; q < p; q++)
    for (int k = 0; k < m; k++) {
      int kk = k + m * q;
      double sr = 0.0, si = 0.0;
      for (int r = 0; r < p; r++) {
        int t = (int)(((int64_t)r * kk) % n) * step;
        double yr = tmp[2 * ((size_t)r * m + k)], yi = tmp[2 * ((size_t)r * m + k) + 1];
        sr += yr * w[2 * t] - yi * w[2 * t + 1];
        si += yr * w[2 * t + 1] + yi * w[2 * t];
      }
      out[2 * kk] = sr; out[2 * kk + 1] = si;
    }
}

/* 1-D transform of a contiguous line; method 1 = naive (T1), 2 = own FFT (T2).  Exposed for pins. */
void orc_dft1d(int n, int sign, int method, const double *in, double *out) {
  double *w = (double *)malloc(sizeof(double) * 2 * n);
  double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)n * 34);
  twiddles(n, sign, w);
  if (method == 1) dft_naive(n, in, 1, out, w, n);
  else fft_rec(n, in, 1, out, w, n, tmp);
  free(w); free(tmp);
}

/* In-place 3-D transform of box[n3][n2][n1] (complex), separable, axis by axis. */
void orc_dft3d(const int32_t *n, int sign, int method, double *box) {
  size_t N = (size_t)n[0] * n[1] * n[2];
  size_t stride[3] = {1, (size_t)n[0], (size_t)n[0] * n[1]};
  for (int ax = 0; ax < 3; ax++) {
    int len = n[ax];
    double *w = (double *)malloc(sizeof(double) * 2 * len);
    twiddles(len, sign, w);
    size_t nlines = N / len;
#pragma omp parallel
    {
      double *line = (double *)malloc(sizeof(double) * 2 * len);
      double *res = (double *)malloc(sizeof(double) * 2 * len);
      double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)len * 34);
#pragma omp for schedule(static)
      for (int64_t l = 0; l < (int64_t)nlines; l++) {
        /* line l: all indices except along ax */
        size_t base;
        if (ax == 0) base = (size_t)l * n[0];
        else if (ax == 1) base = ((size_t)l / n[0]) * stride[2] + ((size_t)l % n[0]);
        else base = (size_t)l;
        for (int j = 0; j < len; j++) {
          line[2 * j] = box[2 * (base + j * stride[ax])];
          line[2 * j + 1] = box[2 * (base + j * stride[ax]) + 1];
        }
        if (method == 1) dft_naive(len, line, 1, res, w, len);
        else fft_rec(len, line, 1, res, w, len, tmp);
        for (int j = 0; j < len; j++) {
          box[2 * (base + j * stride[ax])] = res[2 * j];
          box[2 * (base + j * stride[ax]) + 1] = res[2 * j + 1];
        }
      }
      free(line); free(res); free(tmp);
    }
    free(w);
  }
}

/* psi(r_j) = sum_{m in S} c(m) exp(+2 pi i m.j/n): scatter to the box, transform with sign +. */
void orc_g2r(const int32_t *n, int64_t npw, const int32_t *igfft, const double *c, int method, double *box) {
  size_t N = (size_t)n[0] * n[1] * n[2];
  memset(box, 0, sizeof(double) * 2 * N);
  for (int64_t i = 0; i < npw; i++) { box[2 * (size_t)igfft[i]] = c[2 * i]; box[2 * (size_t)igfft[i] + 1] = c[2 * i + 1]; }
  orc_dft3d(n, +1, method, box);
}

/* (H_loc c)(m) = (1/N) sum_j V(r_j) psi(r_j) exp(-2 pi i m.j/n)   -- reading 4, FFT form.
 * One band; `box` is caller scratch of N complex. */
void orc_vloc_apply(const int32_t *n, int64_t npw, const int32_t *igfft, const double *V,
                    const double *c, int method, double *out, double *box) {
  size_t N = (size_t)n[0] * n[1] * n[2];
  orc_g2r(n, npw, igfft, c, method, box);
  for (size_t j = 0; j < N; j++) { box[2 * j] *= V[j]; box[2 * j + 1] *= V[j]; }
  orc_dft3d(n, -1, method, box);
  double inv = 1.0 / (double)N;
  for (int64_t i = 0; i < npw; i++) {
    out[2 * i] = box[2 * (size_t)igfft[i]] * inv;
    out[2 * i + 1] = box[2 * (size_t)igfft[i] + 1] * inv;
  }
}

/* Vt[d] = (1/N) sum_j V(r_j) exp(-2 pi i d.j/n) for every d in the box (naive DFT, T0). */
void orc_vtilde(const int32_t *n, const double *V, double *vt /* N complex */) {
  size_t N = (size_t)n[0] * n[1] * n[2];
  for (size_t j = 0; j < N; j++) { vt[2 * j] = V[j]; vt[2 * j + 1] = 0.0; }
  orc_dft3d(n, -1, 1, vt);
  double inv = 1.0 / (double)N;
  for (size_t j = 0; j < 2 * N; j++) vt[j] *= inv;
}

/* ---------------------------------------------------------------------------------------------
 * Projectors -- Eq. 26 (PAPER.md :470) with readings 6-11:
 *   p_{a,i}(m) = F_{t(a),irad_i}(|q|) . Y_{l_i m_i}(q^) . exp(-2 pi i (k+m).x_a),  q = 2 pi (k+m)^T Bm
 * ------------------------------------------------------------------------------------------- */

/* reading 7: cubic-spline pair (f, f2) on the uniform grid q_j = j dq */
double orc_spline(int nq, double dq, const double *f, const double *f2, double q) {
  int j = (int)floor(q / dq);
  if (j > nq - 2) j = nq - 2;
  if (j < 0) j = 0;
  double A = ((double)(j + 1) * dq - q) / dq, B = 1.0 - A;
  return A * f[j] + B * f[j + 1] + ((A * A * A - A) * f2[j] + (B * B * B - B) * f2[j + 1]) * (dq * dq) / 6.0;
}

/* reading 8: orthonormal real spherical harmonics, no Condon-Shortley sign, m = -l..l.
 * (x,y,z) need not be normalised; q = |(x,y,z)|.  At q = 0: Y_00 as usual, 0 for l > 0. */
double orc_ylm(int l, int m, double x, double y, double z) {
  const double PI = 3.14159265358979323846;
  double q2 = x * x + y * y + z * z, q = sqrt(q2);
  if (l == 0) return 0.5 / sqrt(PI);
  if (q == 0.0) return 0.0;
  if (l == 1) {
    double c = sqrt(3.0 / (4.0 * PI));
    return c * (m == -1 ? y : (m == 0 ? z : x)) / q;
  }
  if (l == 2) {
    double c1 = 0.5 * sqrt(15.0 / PI), c0 = 0.25 * sqrt(5.0 / PI), c2 = 0.25 * sqrt(15.0 / PI);
    switch (m) {
      case -2: return c1 * x * y / q2;
      case -1: return c1 * y * z / q2;
      case 0:  return c0 * (3.0 * z * z - q2) / q2;
      case 1:  return c1 * x * z / q2;
      case 2:  return c2 * (x * x - y * y) / q2;
    }
  }
  return NAN;
}

typedef struct {
  const double *bm, *k;
  int natom; const int32_t *typat; const double *xred;
  int ntypat, lmax; const int32_t *nlmn, *lmn_l, *lmn_m, *lmn_irad;
  int nrad_max, nq_max; const int32_t *nq; const double *dq, *f, *f2;
} projdef;

/* real part F.Y of projector i of type t at plane wave m */
static double proj_fy(const projdef *P, int t, int i, const int32_t *m) {
  double tt[3] = {P->k[0] + (double)m[0], P->k[1] + (double)m[1], P->k[2] + (double)m[2]};
  double q[3];
  for (int c = 0; c < 3; c++) q[c] = TWO_PI * (tt[0] * P->bm[c] + tt[1] * P->bm[3 + c] + tt[2] * P->bm[6 + c]);
  double qn = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2]);
  int ir = P->lmn_irad[t * P->lmax + i];
  size_t off = ((size_t)t * P->nrad_max + ir) * P->nq_max;
  double F = orc_spline(P->nq[t], P->dq[t], P->f + off, P->f2 + off, qn);
  return F * orc_ylm(P->lmn_l[t * P->lmax + i], P->lmn_m[t * P->lmax + i], q[0], q[1], q[2]);
}

/* reading 11: exp(-2 pi i frac((k+m).x_a)) */
static void proj_phase(const projdef *P, int a, const int32_t *m, double *pr, double *pi) {
  const double *x = P->xred + 3 * a;
  double arg = (P->k[0] + (double)m[0]) * x[0] + (P->k[1] + (double)m[1]) * x[1] + (P->k[2] + (double)m[2]) * x[2];
  arg -= floor(arg);
  *pr = cos(TWO_PI * arg);
  *pi = -sin(TWO_PI * arg);
}

static void fill_projdef(projdef *P, const double *bm, const double *k, int natom, const int32_t *typat,
                         const double *xred, int ntypat, int lmax, const int32_t *nlmn, const int32_t *lmn_l,
                         const int32_t *lmn_m, const int32_t *lmn_irad, int nrad_max, int nq_max,
                         const int32_t *nq, const double *dq, const double *f, const double *f2) {
  P->bm = bm; P->k = k; P->natom = natom; P->typat = typat; P->xred = xred; P->ntypat = ntypat; P->lmax = lmax;
  P->nlmn = nlmn; P->lmn_l = lmn_l; P->lmn_m = lmn_m; P->lmn_irad = lmn_irad; P->nrad_max = nrad_max;
  P->nq_max = nq_max; P->nq = nq; P->dq = dq; P->f = f; P->f2 = f2;
}

#define PROJ_ARGS const double *rprimd, const double *k, int natom, const int32_t *typat, const double *xred, \
    int ntypat, int lmax, const int32_t *nlmn, const int32_t *lmn_l, const int32_t *lmn_m,                  \
    const int32_t *lmn_irad, int nrad_max, int nq_max, const int32_t *nq, const double *dq,                 \
    const double *f, const double *f2
#define PROJ_FILL(P, bm) fill_projdef(&(P), bm, k, natom, typat, xred, ntypat, lmax, nlmn, lmn_l, lmn_m, \
                                      lmn_irad, nrad_max, nq_max, nq, dq, f, f2)

/* Materialised table P[nproj][npw] (complex), projector order = atoms in order, i = 0..nlmn-1. */
void orc_projector_table(PROJ_ARGS, int64_t npw, const int32_t *kg, double *ptab) {
  double bm[9], gmet[9]; projdef P;
  orc_lattice(rprimd, bm, gmet); PROJ_FILL(P, bm);
  int64_t row = 0;
  for (int a = 0; a < natom; a++) {
    int t = typat[a];
    for (int i = 0; i < nlmn[t]; i++, row++) {
      double *dst = ptab + 2 * (size_t)row * npw;
#pragma omp parallel for schedule(static)
      for (int64_t g = 0; g < npw; g++) {
        double fy = proj_fy(&P, t, i, kg + 3 * g), pr, pi;
        proj_phase(&P, a, kg + 3 * g, &pr, &pi);
        dst[2 * g] = fy * pr; dst[2 * g + 1] = fy * pi;
      }
    }
  }
}

/* max |k+G| over the list (for the DFT_ERR_TABLE_RANGE check of the boundary) */
double orc_max_q(const double *rprimd, const double *k, int64_t npw, const int32_t *kg) {
  double bm[9], gmet[9], mx = 0.0;
  orc_lattice(rprimd, bm, gmet);
  for (int64_t g = 0; g < npw; g++) {
    double tt[3] = {k[0] + kg[3 * g], k[1] + kg[3 * g + 1], k[2] + kg[3 * g + 2]}, q2 = 0;
    for (int c = 0; c < 3; c++) { double q = TWO_PI * (tt[0] * bm[c] + tt[1] * bm[3 + c] + tt[2] * bm[6 + c]); q2 += q * q; }
    if (sqrt(q2) > mx) mx = sqrt(q2);
  }
  return mx;
}

/* Non-local term, Eq. 26, streamed (the table is never stored):
 *   cprj[a,i,b] = sum_m conj(p_{a,i}(m)) c_b(m);  c'[a,i,b] = sum_j D^a_ij cprj[a,j,b];
 *   out_b(m)   += sum_a sum_i p_{a,i}(m) c'[a,i,b]
 * psi/out: [nband][ld] complex.  cprj_out (optional) receives cprj [nproj][nband] complex. */
void orc_nonlocal_apply(PROJ_ARGS, const double *dij, int64_t npw, const int32_t *kg, int nband, int64_t ld,
                        const double *psi, double *out, double *cprj_out) {
  double bm[9], gmet[9]; projdef P;
  orc_lattice(rprimd, bm, gmet); PROJ_FILL(P, bm);
  int nproj = 0;
  int *first = (int *)malloc(sizeof(int) * (natom + 1));
  for (int a = 0; a < natom; a++) { first[a] = nproj; nproj += nlmn[typat[a]]; }
  first[natom] = nproj;
  double *cp = (double *)calloc((size_t)2 * nproj * nband, sizeof(double));
  double *cd = (double *)calloc((size_t)2 * nproj * nband, sizeof(double));
  /* F.Y does not depend on the atom, only on its type: tabulate fy[t][i][g] once (plain caching of
   * a factor of the definition; the product p = fy * phase is still formed per (a,i,m)). */
  double *fy = (double *)malloc(sizeof(double) * (size_t)ntypat * lmax * npw);
#pragma omp parallel for schedule(static)
  for (int64_t g = 0; g < npw; g++)
    for (int t = 0; t < ntypat; t++)
      for (int i = 0; i < nlmn[t]; i++) fy[((size_t)t * lmax + i) * npw + g] = proj_fy(&P, t, i, kg + 3 * g);
  /* step 1: cprj */
#pragma omp parallel for schedule(dynamic, 1)
  for (int a = 0; a < natom; a++) {
    int t = typat[a];
    for (int64_t g = 0; g < npw; g++) {
      double phr, phi;
      proj_phase(&P, a, kg + 3 * g, &phr, &phi);
      for (int i = 0; i < nlmn[t]; i++) {
        double w = fy[((size_t)t * lmax + i) * npw + g], pr = w * phr, pi = w * phi;
        double *dst = cp + 2 * (size_t)(first[a] + i) * nband;
        for (int b = 0; b < nband; b++) {
          double cr = psi[2 * ((size_t)b * ld + g)], ci = psi[2 * ((size_t)b * ld + g) + 1];
          dst[2 * b] += pr * cr + pi * ci;        /* conj(p) * c */
          dst[2 * b + 1] += pr * ci - pi * cr;
        }
      }
    }
  }
  if (cprj_out) memcpy(cprj_out, cp, sizeof(double) * 2 * (size_t)nproj * nband);
  /* step 2: D_ij (real symmetric, per atom) */
  for (int a = 0; a < natom; a++) {
    int nl = nlmn[typat[a]];
    for (int i = 0; i < nl; i++)
      for (int j = 0; j < nl; j++) {
        double d = dij[((size_t)a * lmax + i) * lmax + j];
        for (int b = 0; b < 2 * nband; b++) cd[2 * (size_t)(first[a] + i) * nband + b] += d * cp[2 * (size_t)(first[a] + j) * nband + b];
      }
  }
  /* step 3: back-projection */
#pragma omp parallel for schedule(static)
  for (int64_t g = 0; g < npw; g++) {
    for (int a = 0; a < natom; a++) {
      int t = typat[a];
      double phr, phi;
      proj_phase(&P, a, kg + 3 * g, &phr, &phi);
      for (int i = 0; i < nlmn[t]; i++) {
        double w = fy[((size_t)t * lmax + i) * npw + g], pr = w * phr, pi = w * phi;
        const double *src = cd + 2 * (size_t)(first[a] + i) * nband;
        for (int b = 0; b < nband; b++) {
          out[2 * ((size_t)b * ld + g)] += pr * src[2 * b] - pi * src[2 * b + 1];
          out[2 * ((size_t)b * ld + g) + 1] += pr * src[2 * b + 1] + pi * src[2 * b];
        }
      }
    }
  }
  free(first); free(cp); free(cd); free(fy);
}

/* ---------------------------------------------------------------------------------------------
 * Whole operator, reading 16:  H psi = kin (.) c + H_loc c + H_nl c, bands independent (:436).
 * terms: bit 0 kinetic, bit 1 local, bit 2 non-local.  method 1 = T1 naive DFT, 2 = T2 own FFT.
 * ------------------------------------------------------------------------------------------- */
void orc_apply_h(PROJ_ARGS, const double *dij, const int32_t *n, const double *V, int64_t npw, const int32_t *kg,
                 const int32_t *igfft, const double *kin, int nband, int64_t ld, const double *psi, double *hpsi,
                 int method, int terms) {
  size_t N = (size_t)n[0] * n[1] * n[2];
  memset(hpsi, 0, sizeof(double) * 2 * (size_t)nband * ld);
  if (terms & 2) {
    double *box = (double *)malloc(sizeof(double) * 2 * N);
    for (int b = 0; b < nband; b++)     /* the 3-D transform itself is OpenMP-parallel over lines */
      orc_vloc_apply(n, npw, igfft, V, psi + 2 * (size_t)b * ld, method, hpsi + 2 * (size_t)b * ld, box);
    free(box);
  }
  if (terms & 1)
    for (int b = 0; b < nband; b++)
      for (int64_t g = 0; g < npw; g++) {
        hpsi[2 * ((size_t)b * ld + g)] += kin[g] * psi[2 * ((size_t)b * ld + g)];
        hpsi[2 * ((size_t)b * ld + g) + 1] += kin[g] * psi[2 * ((size_t)b * ld + g) + 1];
      }
  if (terms & 4)
    orc_nonlocal_apply(rprimd, k, natom, typat, xred, ntypat, lmax, nlmn, lmn_l, lmn_m, lmn_irad, nrad_max, nq_max,
                       nq, dq, f, f2, dij, npw, kg, nband, ld, psi, hpsi, NULL);
}

/* T0: explicit dense H[m][m'] (npw x npw complex, row-major) "in the plane-wave basis":
 *   H = diag(kin) + Vt[(m - m') mod n] + sum_a sum_ij p_{a,i}(m) D^a_ij conj(p_{a,j}(m'))        */
void orc_dense_h(PROJ_ARGS, const double *dij, const int32_t *n, const double *V, int64_t npw, const int32_t *kg,
                 const double *kin, int terms, double *H) {
  size_t N = (size_t)n[0] * n[1] * n[2];
  memset(H, 0, sizeof(double) * 2 * (size_t)npw * npw);
  if (terms & 1) for (int64_t g = 0; g < npw; g++) H[2 * ((size_t)g * npw + g)] += kin[g];
  if (terms & 2) {
    double *vt = (double *)malloc(sizeof(double) * 2 * N);
    orc_vtilde(n, V, vt);
#pragma omp parallel for schedule(static)
    for (int64_t g = 0; g < npw; g++)
      for (int64_t h = 0; h < npw; h++) {
        int d[3];
        for (int c = 0; c < 3; c++) { d[c] = (kg[3 * g + c] - kg[3 * h + c]) % n[c]; if (d[c] < 0) d[c] += n[c]; }
        size_t idx = d[0] + (size_t)n[0] * (d[1] + (size_t)n[1] * d[2]);
        H[2 * ((size_t)g * npw + h)] += vt[2 * idx];
        H[2 * ((size_t)g * npw + h) + 1] += vt[2 * idx + 1];
      }
    free(vt);
  }
  if (terms & 4) {
    int nproj = 0;
    for (int a = 0; a < natom; a++) nproj += nlmn[typat[a]];
    double *pt = (double *)malloc(sizeof(double) * 2 * (size_t)nproj * npw);
    orc_projector_table(rprimd, k, natom, typat, xred, ntypat, lmax, nlmn, lmn_l, lmn_m, lmn_irad, nrad_max, nq_max,
                        nq, dq, f, f2, npw, kg, pt);
    int row0 = 0;
    for (int a = 0; a < natom; a++) {
      int nl = nlmn[typat[a]];
      for (int i = 0; i < nl; i++)
        for (int j = 0; j < nl; j++) {
          double d = dij[((size_t)a * lmax + i) * lmax + j];
          if (d == 0.0) continue;
          const double *pi_ = pt + 2 * (size_t)(row0 + i) * npw, *pj = pt + 2 * (size_t)(row0 + j) * npw;
#pragma omp parallel for schedule(static)
          for (int64_t g = 0; g < npw; g++) {
            double ar = d * pi_[2 * g], ai = d * pi_[2 * g + 1];
            for (int64_t h = 0; h < npw; h++) {
              double br = pj[2 * h], bi = -pj[2 * h + 1];
              H[2 * ((size_t)g * npw + h)] += ar * br - ai * bi;
              H[2 * ((size_t)g * npw + h) + 1] += ar * bi + ai * br;
            }
          }
        }
      row0 += nl;
    }
    free(pt);
  }
}

/* y = H x for a dense row-major complex matrix (plain loops) */
void orc_dense_matvec(int64_t n, const double *H, const double *x, double *y) {
#pragma omp parallel for schedule(static)
  for (int64_t g = 0; g < n; g++) {
    double sr = 0.0, si = 0.0;
    for (int64_t h = 0; h < n; h++) {
      double ar = H[2 * ((size_t)g * n + h)], ai = H[2 * ((size_t)g * n + h) + 1];
      sr += ar * x[2 * h] - ai * x[2 * h + 1];
      si += ar * x[2 * h + 1] + ai * x[2 * h];
    }
    y[2 * g] = sr; y[2 * g + 1] = si;
  }
}
