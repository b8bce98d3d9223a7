// fft_codelets.cuh -- in-register DFT codelets of K2 (the local term, PAPER.md :475 "local part using
// fast Fourier transforms").  Dft<R,S>::run(v) replaces v[0..R) by X[q] = sum_r v[r] w^(q r),
// w = exp(S 2 pi i / R), natural order in and out, everything in registers (all indices are compile-time
// constants after unrolling).  Small radices are written out; composite ones are built from them with the
// prime-factor map (coprime factors, no internal twiddles) or one Cooley-Tukey step (constant twiddles).
// Shared by the generic Stockham path and the two-stage register path of fft.cu.  Nothing here is shared
// with the CPU checker.
#pragma once
#include <cuda_runtime.h>

namespace dftb200 {

#define DFT_HD __host__ __device__ __forceinline__

typedef double2 cplx;
DFT_HD cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
DFT_HD cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
DFT_HD cplx cmul(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
DFT_HD cplx cscale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }
// multiply by S*i
template <int S> DFT_HD cplx mul_si(cplx a) { return S > 0 ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x); }
// a * (c + S i s)
template <int S> DFT_HD cplx cmul_cs(cplx a, double c, double s) {
  return S > 0 ? make_double2(a.x * c - a.y * s, a.y * c + a.x * s) : make_double2(a.x * c + a.y * s, a.y * c - a.x * s);
}

template <int S> DFT_HD void bfly2(cplx &a, cplx &b) {
  cplx t = csub(a, b); a = cadd(a, b); b = t;
}
template <int S> DFT_HD void bfly3(cplx &v0, cplx &v1, cplx &v2) {
  const double H = 0.86602540378443864676;  // sqrt(3)/2
  cplx t = cadd(v1, v2), u = mul_si<S>(cscale(csub(v1, v2), H));
  cplx m = make_double2(v0.x - 0.5 * t.x, v0.y - 0.5 * t.y);
  v0 = cadd(v0, t); v1 = cadd(m, u); v2 = csub(m, u);
}
template <int S> DFT_HD void bfly4(cplx &v0, cplx &v1, cplx &v2, cplx &v3) {
  cplx t0 = cadd(v0, v2), t1 = csub(v0, v2), t2 = cadd(v1, v3), t3 = mul_si<S>(csub(v1, v3));
  v0 = cadd(t0, t2); v2 = csub(t0, t2); v1 = cadd(t1, t3); v3 = csub(t1, t3);
}
template <int S> DFT_HD void bfly5(cplx &v0, cplx &v1, cplx &v2, cplx &v3, cplx &v4) {
  const double C1 = 0.30901699437494742410, C2 = -0.80901699437494742410;  // cos(2pi/5), cos(4pi/5)
  const double S1 = 0.95105651629515357212, S2 = 0.58778525229247312917;   // sin(2pi/5), sin(4pi/5)
  cplx a1 = cadd(v1, v4), a2 = cadd(v2, v3), b1 = csub(v1, v4), b2 = csub(v2, v3);
  cplx m1 = make_double2(v0.x + C1 * a1.x + C2 * a2.x, v0.y + C1 * a1.y + C2 * a2.y);
  cplx m2 = make_double2(v0.x + C2 * a1.x + C1 * a2.x, v0.y + C2 * a1.y + C1 * a2.y);
  cplx u1 = mul_si<S>(make_double2(S1 * b1.x + S2 * b2.x, S1 * b1.y + S2 * b2.y));
  cplx u2 = mul_si<S>(make_double2(S2 * b1.x - S1 * b2.x, S2 * b1.y - S1 * b2.y));
  v0 = cadd(v0, cadd(a1, a2));
  v1 = cadd(m1, u1); v4 = csub(m1, u1);
  v2 = cadd(m2, u2); v3 = csub(m2, u2);
}

template <int R, int S> struct Dft;
template <int S> struct Dft<1, S> { static DFT_HD void run(cplx *) {} };
template <int S> struct Dft<2, S> { static DFT_HD void run(cplx *v) { bfly2<S>(v[0], v[1]); } };
template <int S> struct Dft<3, S> { static DFT_HD void run(cplx *v) { bfly3<S>(v[0], v[1], v[2]); } };
template <int S> struct Dft<4, S> { static DFT_HD void run(cplx *v) { bfly4<S>(v[0], v[1], v[2], v[3]); } };
template <int S> struct Dft<5, S> { static DFT_HD void run(cplx *v) { bfly5<S>(v[0], v[1], v[2], v[3], v[4]); } };
// 8 = 2 x 4 (decimation in time: even/odd halves, then X[q] = E[q] + w8^q O[q], X[q+4] = E[q] - w8^q O[q])
template <int S> struct Dft<8, S> {
  static DFT_HD void run(cplx *v) {
    const double Q = 0.70710678118654752440;
    bfly4<S>(v[0], v[2], v[4], v[6]);   // E[0..3] in v0,v2,v4,v6
    bfly4<S>(v[1], v[3], v[5], v[7]);   // O[0..3] in v1,v3,v5,v7
    cplx o1 = make_double2(Q * (v[3].x - S * v[3].y), Q * (v[3].y + S * v[3].x));       // w8^1 = (1 + S i)/sqrt2
    cplx o2 = mul_si<S>(v[5]);                                                           // w8^2 = S i
    cplx o3 = make_double2(Q * (-v[7].x - S * v[7].y), Q * (-v[7].y + S * v[7].x));     // w8^3 = (-1 + S i)/sqrt2
    cplx e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
    v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
    v[1] = cadd(e1, o1); v[5] = csub(e1, o1);
    v[2] = cadd(e2, o2); v[6] = csub(e2, o2);
    v[3] = cadd(e3, o3); v[7] = csub(e3, o3);
  }
};
// 9 = 3 x 3:  r = 3a + b, q = q1 + 3 q2;  Y_b[q1] = DFT3_a v[3a+b];  X[q1+3q2] = DFT3_b (w9^(b q1) Y_b[q1])
template <int S> struct Dft<9, S> {
  static DFT_HD void run(cplx *v) {
    const double C1 = 0.76604444311897803520, S1 = 0.64278760968653932632;   // cos/sin(2pi/9)
    const double C2 = 0.17364817766693034885, S2 = 0.98480775301220805937;   // cos/sin(4pi/9)
    const double C4 = -0.93969262078590838405, S4 = 0.34202014332566873304;  // cos/sin(8pi/9)
    bfly3<S>(v[0], v[3], v[6]);   // b = 0: Y_0[q1] in v0,v3,v6
    bfly3<S>(v[1], v[4], v[7]);   // b = 1
    bfly3<S>(v[2], v[5], v[8]);   // b = 2
    // twiddles w9^(b q1): (b,q1) = (1,1)->w, (1,2)->w^2, (2,1)->w^2, (2,2)->w^4
    v[4] = cmul_cs<S>(v[4], C1, S1);
    v[7] = cmul_cs<S>(v[7], C2, S2);
    v[5] = cmul_cs<S>(v[5], C2, S2);
    v[8] = cmul_cs<S>(v[8], C4, S4);
    bfly3<S>(v[0], v[1], v[2]);   // q1 = 0: X[0], X[3], X[6]
    bfly3<S>(v[3], v[4], v[5]);   // q1 = 1: X[1], X[4], X[7]
    bfly3<S>(v[6], v[7], v[8]);   // q1 = 2: X[2], X[5], X[8]
    cplx x1 = v[3], x2 = v[6], x3 = v[1], x4 = v[4], x5 = v[7], x6 = v[2], x7 = v[5];
    v[1] = x1; v[2] = x2; v[3] = x3; v[4] = x4; v[5] = x5; v[6] = x6; v[7] = x7;
  }
};
// 16 = 4 x 4, one Cooley-Tukey step: r = 4a + b, q = q1 + 4 q2; Y_b[q1] = DFT4_a v[4a+b]; X[q1+4q2] = DFT4_b (w16^(b q1) Y_b[q1])
template <int S> struct Dft<16, S> {
  static DFT_HD void run(cplx *v) {
    const double C1 = 0.92387953251128675613, S1 = 0.38268343236508977173;   // cos/sin(2pi/16)
    const double Q = 0.70710678118654752440;                                  // cos = sin(4pi/16)
    bfly4<S>(v[0], v[4], v[8], v[12]);    // b = 0: Y_0[q1] in v0,v4,v8,v12
    bfly4<S>(v[1], v[5], v[9], v[13]);    // b = 1
    bfly4<S>(v[2], v[6], v[10], v[14]);   // b = 2
    bfly4<S>(v[3], v[7], v[11], v[15]);   // b = 3
    // Y_b[q1] sits in v[4 q1 + b]; twiddle w16^(b q1)
    v[5] = cmul_cs<S>(v[5], C1, S1);      // (1,1) w^1
    v[9] = cmul_cs<S>(v[9], Q, Q);        // (1,2) w^2
    v[13] = cmul_cs<S>(v[13], S1, C1);    // (1,3) w^3
    v[6] = cmul_cs<S>(v[6], Q, Q);        // (2,1) w^2
    v[10] = mul_si<S>(v[10]);             // (2,2) w^4 = S i
    v[14] = cmul_cs<S>(v[14], -Q, Q);     // (2,3) w^6
    v[7] = cmul_cs<S>(v[7], S1, C1);      // (3,1) w^3
    v[11] = cmul_cs<S>(v[11], -Q, Q);     // (3,2) w^6
    v[15] = cmul_cs<S>(v[15], -C1, -S1);  // (3,3) w^9 = -w^1
    bfly4<S>(v[0], v[1], v[2], v[3]);     // q1 = 0: X[0], X[4], X[8], X[12]
    bfly4<S>(v[4], v[5], v[6], v[7]);     // q1 = 1: X[1], X[5], X[9], X[13]
    bfly4<S>(v[8], v[9], v[10], v[11]);   // q1 = 2
    bfly4<S>(v[12], v[13], v[14], v[15]); // q1 = 3
    // v[4 q1 + q2] holds X[q1 + 4 q2]: transpose the 4 x 4 register block
#define DFT_SWAP(a, b) { cplx t_ = v[a]; v[a] = v[b]; v[b] = t_; }
    DFT_SWAP(1, 4) DFT_SWAP(2, 8) DFT_SWAP(3, 12) DFT_SWAP(6, 9) DFT_SWAP(7, 13) DFT_SWAP(11, 14)
#undef DFT_SWAP
  }
};

// Prime-factor (Good-Thomas) step for coprime N1, N2: input map r = (N2 r1 + N1 r2) mod N, output map
// q = q1 mod N1, q = q2 mod N2 (CRT); X[q] = sum_{r1,r2} v[r] w_N1^(r1 q1) w_N2^(r2 q2), no twiddles.
__host__ __device__ constexpr int dft_inv_mod(int a, int m) {
  int r = 1;
  for (int i = 1; i < m; i++) if ((a * i) % m == 1 % m) r = i;
  return r;
}
template <int N1, int N2, int S> struct Pfa {
  static DFT_HD void run(cplx *v) {
    constexpr int N = N1 * N2;
    constexpr int E1 = N2 * dft_inv_mod(N2 % N1, N1), E2 = N1 * dft_inv_mod(N1 % N2, N2);   // CRT idempotents
    cplx t[N];
#pragma unroll
    for (int r2 = 0; r2 < N2; r2++) {
      cplx a[N1];
#pragma unroll
      for (int r1 = 0; r1 < N1; r1++) a[r1] = v[(N2 * r1 + N1 * r2) % N];
      Dft<N1, S>::run(a);
#pragma unroll
      for (int q1 = 0; q1 < N1; q1++) t[q1 * N2 + r2] = a[q1];
    }
#pragma unroll
    for (int q1 = 0; q1 < N1; q1++) {
      cplx b[N2];
#pragma unroll
      for (int r2 = 0; r2 < N2; r2++) b[r2] = t[q1 * N2 + r2];
      Dft<N2, S>::run(b);
#pragma unroll
      for (int q2 = 0; q2 < N2; q2++) v[(q1 * E1 + q2 * E2) % N] = b[q2];
    }
  }
};
template <int S> struct Dft<6, S> { static DFT_HD void run(cplx *v) { Pfa<2, 3, S>::run(v); } };
template <int S> struct Dft<10, S> { static DFT_HD void run(cplx *v) { Pfa<2, 5, S>::run(v); } };
template <int S> struct Dft<12, S> { static DFT_HD void run(cplx *v) { Pfa<4, 3, S>::run(v); } };
template <int S> struct Dft<15, S> { static DFT_HD void run(cplx *v) { Pfa<3, 5, S>::run(v); } };
template <int S> struct Dft<18, S> { static DFT_HD void run(cplx *v) { Pfa<2, 9, S>::run(v); } };
template <int S> struct Dft<20, S> { static DFT_HD void run(cplx *v) { Pfa<4, 5, S>::run(v); } };
template <int S> struct Dft<24, S> { static DFT_HD void run(cplx *v) { Pfa<3, 8, S>::run(v); } };

}  // namespace dftb200
