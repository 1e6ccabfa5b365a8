// grpic_device.cuh — per-particle device arithmetic of the GRPIC hot path (sm_100a).
//
// Everything here is written from the paper's equations ("P:n" = PAPER.md line n) and from the
// readings listed in DESIGN.md ("R-Sk"); it shares nothing with oracle/.  One source, two
// precisions: T = float (libgrpic_f32.so) or double (libgrpic_f64.so).
//
// All metric quantities are recomputed in registers from (cell, displacement, spin, map constants);
// nothing is tabulated.  Notation follows App. A: Sigma, Delta, A, z, alpha, beta^1,
// h^{ij} ("hu"), h_{ij} ("hd"), code basis of the log-r map A.3 with s1 = dxi*r, s2 = deta.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace grpic {

// ------------------------------------------------------------------------------------------------
// constants of one context, passed by value to every kernel
// ------------------------------------------------------------------------------------------------
template <typename T>
struct Consts {
  int32_t n1, n2, ng, n_iter;
  int32_t ld;        // row length of every grid array: n2 + 2*ng
  int32_t pad_;
  T a, a2;           // spin and its square
  T log_rmin;        // xi at x1 = 0
  T dxi, deta;       // d(xi)/d(x1), d(theta)/d(x2)
  T inv_dxi;         // 1/dxi
  T inv_deta2;       // 1/deta^2
  T th_min, th_max;  // [small_angle, pi - small_angle]
  T sin_min, cos_min;  // sin, cos of th_min
  int32_t early_exit;  // leave a fixed-point loop once the iterate repeats bit for bit (identical result)
  int32_t pad2_;
};

// ------------------------------------------------------------------------------------------------
// scalar helpers: IEEE operators in FP64; hardware approximations (<= 2 ulp) in FP32
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp_(double x) { return 1.0 / x; }
__device__ __forceinline__ double rsqrt_(double x) { return 1.0 / sqrt(x); }
__device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
__device__ __forceinline__ double exp_(double x) { return exp(x); }
__device__ __forceinline__ void sincos_(double x, double* s, double* c) { sincos(x, s, c); }
__device__ __forceinline__ double floor_(double x) { return floor(x); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ double below_one(double) { return 0x1.fffffffffffffp-1; }

__device__ __forceinline__ float rcp_(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsqrt_(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float sqrt_(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float exp_(float x) { return expf(x); }
__device__ __forceinline__ void sincos_(float x, float* s, float* c) { sincosf(x, s, c); }
__device__ __forceinline__ float floor_(float x) { return floorf(x); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float below_one(float) { return 0x1.fffffep-1f; }

// ------------------------------------------------------------------------------------------------
// Coordinate map (r0 = 0, h0 = 0) and the axis regularisation (R-S9).
//
// FP64: the plain formulas, x = i + dx, r = exp(ln r_min + x1*dxi), theta = x2*deta.
// FP32: the same map evaluated so that rounding does not eat the in-cell displacement:
//   - theta is measured from the NEARER axis (theta' = pi - theta on the lower half, exact in the
//     integer part), so that sin(theta) keeps full relative accuracy next to theta = pi;
//   - a midpoint x + h is reached from the stored r, theta' by r*exp(h1*dxi), theta' +- h2*deta,
//     never by re-adding i + dx + h in FP32 (ulp(2048) = 2.4e-4 cells).
// ------------------------------------------------------------------------------------------------
template <typename T>
struct Coord;

template <>
struct Coord<double> {
  double x1, x2;
  __device__ __forceinline__ void init(const Consts<double>&, int i1, double dx1, int i2, double dx2) {
    x1 = (double)i1 + dx1;
    x2 = (double)i2 + dx2;
  }
  // r, sin(theta), cos(theta) at x + (h1, h2)
  __device__ __forceinline__ void at(const Consts<double>& g, double h1, double h2, double& r, double& sth,
                                     double& cth) const {
    r = exp(g.log_rmin + (x1 + h1) * g.dxi);
    double th = (x2 + h2) * g.deta;
    th = fmin(fmax(th, g.th_min), g.th_max);
    sincos(th, &sth, &cth);
  }
};

template <>
struct Coord<float> {
  float r0, thp, s0, c0, sgn;  // r, theta', sin(theta'), cos(theta') at x (theta' unclamped); +1 or -1 (mirrored)
  __device__ __forceinline__ void init(const Consts<float>& g, int i1, float dx1, int i2, float dx2) {
    const float xi = fmaf(dx1, g.dxi, fmaf((float)i1, g.dxi, g.log_rmin));
    r0 = expf(xi);
    if (2 * i2 >= g.n2) {
      thp = ((float)(g.n2 - i2) - dx2) * g.deta;
      sgn = -1.f;
    } else {
      thp = ((float)i2 + dx2) * g.deta;
      sgn = 1.f;
    }
    sincosf(thp, &s0, &c0);
  }
  __device__ __forceinline__ void at(const Consts<float>& g, float h1, float h2, float& r, float& sth,
                                     float& cth) const {
    // r0 * exp(e), |e| = |h1| dxi: 4th-order Taylor (|e|^5/120 < 1e-9 for |e| < 0.04), expf beyond
    const float e = h1 * g.dxi;
    float p = fmaf(e, 1.f / 24.f, 1.f / 6.f);
    p = fmaf(p, e, 0.5f);
    p = fmaf(p, e, 1.f);
    p = fmaf(p, e, 1.f);
    r = (fabsf(e) < 0.04f) ? r0 * p : r0 * expf(e);
    // sin, cos(theta' + d) by angle addition, |d| = |h2| deta: sin d to d^3, cos d to d^4
    // (relative errors d^4/120, d^6/720 < 4e-8 for |d| < 0.045); sincosf beyond
    const float d = sgn * h2 * g.deta;
    const float th = thp + d;
    float s, c;
    if (fabsf(d) < 0.045f) {
      const float d2 = d * d;
      const float sd = fmaf(d * d2, -1.f / 6.f, d);
      const float cd = fmaf(d2, fmaf(d2, 1.f / 24.f, -0.5f), 1.f);
      s = fmaf(s0, cd, c0 * sd);
      c = fmaf(c0, cd, -s0 * sd);
    } else {
      sincosf(th, &s, &c);
    }
    // axis regularisation: theta' clamped to [th_min, th_max]
    if (th < g.th_min) { s = g.sin_min; c = g.cos_min; }
    if (th > g.th_max) { s = g.sin_min; c = -g.cos_min; }
    sth = s;
    cth = sgn * c;
  }
};

// ------------------------------------------------------------------------------------------------
// Metric.  "Lite": what Eq. 29/30 need at a midpoint.
// ------------------------------------------------------------------------------------------------
template <typename T>
struct MetricLite {
  T ia2;   // 1/alpha^2 = 1 + z
  T beta1, hu11, hu22, hu33, hu13;
};

template <typename T>
__device__ __forceinline__ void metric_lite(const Consts<T>& g, T r, T sth, T cth, MetricLite<T>& m) {
  const T r2 = r * r;
  const T s2th = sth * sth;
  const T Sigma = fma_(g.a2 * cth, cth, r2);
  const T Delta = fma_(r, r - T(2), g.a2);
  const T r2a2 = r2 + g.a2;
  const T A = fma_(-(g.a2 * s2th), Delta, r2a2 * r2a2);
  const T Sp2r = fma_(T(2), r, Sigma);          // Sigma (1 + z)
  const T iS = rcp_(Sigma);
  const T iSp2r = rcp_(Sp2r);
  const T is1 = g.inv_dxi * rcp_(r);            // 1/s1
  const T q = iS * is1;
  m.ia2 = Sp2r * iS;
  m.beta1 = (T(2) * r) * (iSp2r * is1);         // z/(1+z)/s1
  m.hu11 = (A * iSp2r) * (q * is1);
  m.hu22 = iS * g.inv_deta2;
  m.hu33 = iS * rcp_(s2th);
  m.hu13 = g.a * q;
}

// 1/u^0 = alpha/gamma at a midpoint (Eq. 20 with footnote 8)
template <typename T>
__device__ __forceinline__ T inv_u0(const MetricLite<T>& m, T u1sq, T u2sq, T u3sq, T u1u3x2, T eps) {
  const T g2 = fma_(m.hu11, u1sq, fma_(m.hu22, u2sq, fma_(m.hu33, u3sq, fma_(m.hu13, u1u3x2, eps))));
  return rsqrt_(g2 * m.ia2);
}

// Full set at x^(n): adds h_ij (for the tetrad) and the twelve derivatives of Eq. 27.
template <typename T>
struct MetricFull {
  T alpha, beta1, hu11, hu22, hu33, hu13;
  T hd22, hd33, hd13;
  T d_alpha[2], d_beta1[2], d_hu11[2], d_hu22[2], d_hu33[2], d_hu13[2];  // [0] = d/dx1, [1] = d/dx2
};

// Derivatives: chain rule on the closed forms above (general rule P:772-778; A.2 list P:814-816;
// the A.3 extras from s1 = dxi*exp(xi) depending on x1; corrections R-S2).
template <typename T>
__device__ __forceinline__ void metric_full(const Consts<T>& g, T r, T sth, T cth, MetricFull<T>& m) {
  const T a = g.a, a2 = g.a2;
  const T r2 = r * r;
  const T s2th = sth * sth;
  const T Sigma = fma_(a2 * cth, cth, r2);
  const T Delta = r2 - T(2) * r + a2;
  const T r2a2 = r2 + a2;
  const T A = r2a2 * r2a2 - a2 * Delta * s2th;
  const T Sp2r = Sigma + T(2) * r;
  const T s1 = g.dxi * r, s2 = g.deta;
  const T iS = rcp_(Sigma), iSp2r = rcp_(Sp2r), is1 = rcp_(s1), is2th = rcp_(s2th);
  const T iS2 = iS * iS;
  const T opz = Sp2r * iS;                       // 1 + z
  m.alpha = sqrt_(Sigma * iSp2r);
  m.beta1 = T(2) * r * iSp2r * is1;
  m.hu11 = A * iS * iSp2r * is1 * is1;
  m.hu22 = iS * g.inv_deta2;
  m.hu33 = iS * is2th;
  m.hu13 = a * iS * is1;
  m.hd22 = s2 * s2 * Sigma;
  m.hd33 = A * s2th * iS;
  m.hd13 = -s1 * a * opz * s2th;

  const T d1S = T(2) * r * s1;
  const T d2S = T(-2) * a2 * sth * cth * s2;
  const T d1D = T(2) * (r - T(1)) * s1;
  const T d1A = T(4) * r * s1 * r2a2 - a2 * s2th * d1D;
  const T d2A = d2S * Delta;                     // -2 a^2 sin cos Delta s2
  const T iP = iS * iSp2r;                       // 1/(Sigma (Sigma + 2r))
  const T iP2s = iP * iP * is1 * is1;
  const T P = Sigma * Sp2r;
  m.d_hu11[0] = (P * d1A - T(2) * A * (r * d1S + Sigma * (d1S + s1))) * iP2s - T(2) * g.dxi * m.hu11;
  m.d_hu11[1] = (P * d2A - T(2) * A * d2S * (r + Sigma)) * iP2s;
  m.d_hu22[0] = -d1S * iS2 * g.inv_deta2;
  m.d_hu22[1] = -d2S * iS2 * g.inv_deta2;
  m.d_hu33[0] = -d1S * iS2 * is2th;
  m.d_hu33[1] = T(-2) * cth * s2 * iS2 * is2th * rcp_(sth) * (Sigma - a2 * s2th);
  m.d_hu13[0] = -a * is1 * d1S * iS2 - g.dxi * m.hu13;
  m.d_hu13[1] = -a * is1 * d2S * iS2;
  const T w = s1 * Sigma - r * d1S;              // Sigma^2/2 * d1 z
  m.d_beta1[0] = T(2) * is1 * w * iSp2r * iSp2r - g.dxi * m.beta1;
  m.d_beta1[1] = T(-2) * is1 * r * d2S * iSp2r * iSp2r;
  const T al3 = m.alpha * m.alpha * m.alpha;
  m.d_alpha[0] = -w * iS2 * al3;
  m.d_alpha[1] = r * d2S * iS2 * al3;
}

// ------------------------------------------------------------------------------------------------
// Tetrad at x^(n): matrix form of P:754 (R-S3).  e[] caches the square roots.
// ------------------------------------------------------------------------------------------------
template <typename T>
struct Tetrad {
  T sq11, isq11;   // sqrt(h^11), 1/sqrt(h^11)
  T sq22, isq22;   // sqrt(h_22), 1/...
  T sq33, isq33;   // sqrt(h_33), 1/...
  T k13;           // h_13 / sqrt(h_33)
  __device__ __forceinline__ void init(const MetricFull<T>& m) {
    isq11 = rsqrt_(m.hu11); sq11 = m.hu11 * isq11;
    isq22 = rsqrt_(m.hd22); sq22 = m.hd22 * isq22;
    isq33 = rsqrt_(m.hd33); sq33 = m.hd33 * isq33;
    k13 = m.hd13 * isq33;
  }
  __device__ __forceinline__ void cntrv_to_tetrad(const T A[3], T Ah[3]) const {
    Ah[0] = A[0] * isq11;
    Ah[1] = sq22 * A[1];
    Ah[2] = k13 * A[0] + sq33 * A[2];
  }
  __device__ __forceinline__ void cov_to_tetrad(const T u[3], T uh[3]) const {
    uh[0] = sq11 * (u[0] - k13 * isq33 * u[2]);
    uh[1] = u[1] * isq22;
    uh[2] = u[2] * isq33;
  }
  __device__ __forceinline__ void tetrad_to_cov(const T uh[3], T u[3]) const {
    u[0] = uh[0] * isq11 + k13 * uh[2];
    u[1] = sq22 * uh[1];
    u[2] = sq33 * uh[2];
  }
};

// Boris rotation over dt/2 in the orthonormal frame (coefficient c = (q/m) alpha dt/4, R-S5).
template <typename T>
__device__ __forceinline__ void boris_half(const T Dh[3], const T Bh[3], T c, T uh[3]) {
  const T um0 = uh[0] + c * Dh[0], um1 = uh[1] + c * Dh[1], um2 = uh[2] + c * Dh[2];
  const T ig = c * rsqrt_(T(1) + um0 * um0 + um1 * um1 + um2 * um2);
  const T t0 = Bh[0] * ig, t1 = Bh[1] * ig, t2 = Bh[2] * ig;
  const T f = T(2) * rcp_(T(1) + t0 * t0 + t1 * t1 + t2 * t2);
  const T s0 = f * t0, s1 = f * t1, s2 = f * t2;
  const T p0 = um0 + (um1 * t2 - um2 * t1);
  const T p1 = um1 + (um2 * t0 - um0 * t2);
  const T p2 = um2 + (um0 * t1 - um1 * t0);
  uh[0] = um0 + (p1 * s2 - p2 * s1) + c * Dh[0];
  uh[1] = um1 + (p2 * s0 - p0 * s2) + c * Dh[1];
  uh[2] = um2 + (p0 * s1 - p1 * s0) + c * Dh[2];
}

// ------------------------------------------------------------------------------------------------
// Field gather (step 2; scheme R-S4): every Yee component is first averaged to the four
// nodes of the particle's cell, then bilinear in (dx1, dx2).  Folded into one weighted sum per
// component: along an axis where the component sits at half-integer positions the three weights are
// {(1-d)/2, 1/2, d/2} on samples {c-1, c, c+1}; where it sits on nodes, {1-d, d} on {c, c+1}.
// `F` is any accessor with  T operator()(int comp, int di, int dj)  returning sample
// (i1 + di, i2 + dj) of component comp (0..5 = D1 D2 D3 B1 B2 B3).
// ------------------------------------------------------------------------------------------------
template <typename T, typename Acc>
__device__ __forceinline__ void interp_fields(const Acc& F, T dx1, T dx2, T D[3], T B[3]) {
  const T n1[2] = {T(1) - dx1, dx1};
  const T n2[2] = {T(1) - dx2, dx2};
  const T h1[3] = {T(0.5) * n1[0], T(0.5), T(0.5) * dx1};
  const T h2[3] = {T(0.5) * n2[0], T(0.5), T(0.5) * dx2};
  T acc;
  // D1(i+1/2, j), B2(i+1/2, j): half-integer along 1, nodes along 2
  acc = T(0);
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int l = 0; l < 2; ++l) acc = fma_(h1[k] * n2[l], F(0, k - 1, l), acc);
  D[0] = acc;
  acc = T(0);
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int l = 0; l < 2; ++l) acc = fma_(h1[k] * n2[l], F(4, k - 1, l), acc);
  B[1] = acc;
  // D2(i, j+1/2), B1(i, j+1/2): nodes along 1, half-integer along 2
  acc = T(0);
#pragma unroll
  for (int k = 0; k < 2; ++k)
#pragma unroll
    for (int l = 0; l < 3; ++l) acc = fma_(n1[k] * h2[l], F(1, k, l - 1), acc);
  D[1] = acc;
  acc = T(0);
#pragma unroll
  for (int k = 0; k < 2; ++k)
#pragma unroll
    for (int l = 0; l < 3; ++l) acc = fma_(n1[k] * h2[l], F(3, k, l - 1), acc);
  B[0] = acc;
  // D3(i, j): nodes
  acc = T(0);
#pragma unroll
  for (int k = 0; k < 2; ++k)
#pragma unroll
    for (int l = 0; l < 2; ++l) acc = fma_(n1[k] * n2[l], F(2, k, l), acc);
  D[2] = acc;
  // B3(i+1/2, j+1/2): half-integer along both
  acc = T(0);
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int l = 0; l < 3; ++l) acc = fma_(h1[k] * h2[l], F(5, k - 1, l - 1), acc);
  B[2] = acc;
}

// ------------------------------------------------------------------------------------------------
// One particle through steps 3-11 and the particle boundary conditions.
// ------------------------------------------------------------------------------------------------
template <typename T>
struct PState {
  int32_t i1, i2;
  T dx1, dx2, u1, u2, u3;
};

// returns: 0 alive, 1 absorbed inside (i1 < 0), 2 absorbed outside (i1 >= n1); `dphidt` = Eq. 30 rate;
// `reflected` tells the caller that the deposited path is not the integrated one.
template <typename T>
__device__ __forceinline__ int push_particle(const Consts<T>& g, PState<T>& p, bool em, const T Dp[3],
                                             const T Bp[3], T qm, T eps, T dt, T& dphidt, bool& reflected) {
  Coord<T> X;
  X.init(g, p.i1, p.dx1, p.i2, p.dx2);
  T u[3] = {p.u1, p.u2, p.u3};
  {
    T r, sth, cth;
    X.at(g, T(0), T(0), r, sth, cth);
    MetricFull<T> m;
    metric_full(g, r, sth, cth, m);

    Tetrad<T> e;
    T Dh[3], Bh[3], uh[3];
    const T c = qm * m.alpha * dt * T(0.25);
    if (em) {
      e.init(m);
      e.cntrv_to_tetrad(Dp, Dh);                         // step 3
      e.cntrv_to_tetrad(Bp, Bh);
      e.cov_to_tetrad(u, uh);
      boris_half(Dh, Bh, c, uh);                         // step 4
      e.tetrad_to_cov(uh, u);                            // step 5
    }
    // step 6, Eq. 26-27: metric frozen at x^(n); exactly n_iter applications, u~(0) = u*
    {
      const T us0 = u[0], us1 = u[1], u3 = u[2];
      // everything that does not change with the iterate (u_3 is fixed)
      const T g2c = eps + m.hu33 * u3 * u3;
      const T f0c = m.d_hu33[0] * u3 * u3, f1c = m.d_hu33[1] * u3 * u3;
      const T h13u3 = T(2) * m.hu13 * u3;
      const T d13u3_0 = T(2) * m.d_hu13[0] * u3, d13u3_1 = T(2) * m.d_hu13[1] * u3;
      T ut0 = us0, ut1 = us1;
      for (int it = 0; it < g.n_iter; ++it) {
        const T ub0 = T(0.5) * (us0 + ut0), ub1 = T(0.5) * (us1 + ut1);
        const T gam2 = g2c + ub0 * (m.hu11 * ub0 + h13u3) + m.hu22 * ub1 * ub1;
        const T igam = rsqrt_(gam2);
        const T gam = gam2 * igam;                        // alpha u^0
        const T hiu0 = T(0.5) * m.alpha * igam;           // 1/(2 u^0)
        const T q0 = f0c + ub0 * (m.d_hu11[0] * ub0 + d13u3_0) + m.d_hu22[0] * ub1 * ub1;
        const T q1 = f1c + ub0 * (m.d_hu11[1] * ub0 + d13u3_1) + m.d_hu22[1] * ub1 * ub1;
        const T nt0 = us0 + dt * (-gam * m.d_alpha[0] + ub0 * m.d_beta1[0] - hiu0 * q0);
        const T nt1 = us1 + dt * (-gam * m.d_alpha[1] + ub0 * m.d_beta1[1] - hiu0 * q1);
        // the map is deterministic: once an iterate repeats bit for bit every later one equals it
        const bool fixed = (nt0 == ut0) && (nt1 == ut1);
        ut0 = nt0;
        ut1 = nt1;
        if (fixed && g.early_exit) break;
      }
      u[0] = ut0;
      u[1] = ut1;
    }
    if (em) {
      e.cov_to_tetrad(u, uh);                            // step 7
      boris_half(Dh, Bh, c, uh);                         // step 8
      e.tetrad_to_cov(uh, u);                            // step 9
    }
  }
  // step 10, Eq. 28-29 in displacement space: del = x~ - x^(n); all coefficients at x^(n) + del/2
  T del1 = T(0), del2 = T(0);
  MetricLite<T> mm;
  T iu0 = T(0);
  const T u1sq = u[0] * u[0], u2sq = u[1] * u[1], u3sq = u[2] * u[2], u1u3x2 = T(2) * u[0] * u[2];
  bool fixed = false;
  for (int it = 0; it < g.n_iter; ++it) {
    T r, sth, cth;
    X.at(g, T(0.5) * del1, T(0.5) * del2, r, sth, cth);
    metric_lite(g, r, sth, cth, mm);
    iu0 = inv_u0(mm, u1sq, u2sq, u3sq, u1u3x2, eps);
    const T n1 = dt * ((mm.hu11 * u[0] + mm.hu13 * u[2]) * iu0 - mm.beta1);
    const T n2 = dt * (mm.hu22 * u[1] * iu0);
    // bit-identical iterate => every later iterate is the same: stopping here IS n_iter iterations
    fixed = (n1 == del1) && (n2 == del2);
    del1 = n1;
    del2 = n2;
    if (fixed && g.early_exit) break;
  }
  // step 11, Eq. 30 at x_m = (x^(n) + x^(n+1))/2.  If the last iterate repeated, the midpoint
  // of the last evaluation is x_m itself and its coefficients are reused; otherwise evaluate there.
  if (!fixed) {
    T r, sth, cth;
    X.at(g, T(0.5) * del1, T(0.5) * del2, r, sth, cth);
    metric_lite(g, r, sth, cth, mm);
    iu0 = inv_u0(mm, u1sq, u2sq, u3sq, u1u3x2, eps);
  }
  dphidt = (mm.hu13 * u[0] + mm.hu33 * u[2]) * iu0;
  // renormalise to (cell, displacement in [0,1))
  T t1 = p.dx1 + del1, t2 = p.dx2 + del2;
  const T f1 = floor_(t1), f2 = floor_(t2);
  int32_t i1 = p.i1 + (int32_t)f1, i2 = p.i2 + (int32_t)f2;
  T dx1 = t1 - f1, dx2 = t2 - f2;
  if (dx1 >= T(1)) { dx1 = T(0); i1 += 1; }
  if (dx2 >= T(1)) { dx2 = T(0); i2 += 1; }
  // axis reflection
  reflected = false;
  if (i2 < 0 || i2 >= g.n2) {
    i2 = (i2 < 0) ? 0 : g.n2 - 1;
    dx2 = T(1) - dx2;
    if (dx2 >= T(1)) dx2 = below_one(T(0));
    u[1] = -u[1];
    reflected = true;
  }
  p.i1 = i1; p.i2 = i2; p.dx1 = dx1; p.dx2 = dx2;
  p.u1 = u[0]; p.u2 = u[1]; p.u3 = u[2];
  // radial removal (P:467 inner ghost zone, P:648 outer absorption)
  return (i1 < 0) ? 1 : ((i1 >= g.n1) ? 2 : 0);
}

// ------------------------------------------------------------------------------------------------
// Deposit (Sec. 3.2, Eq. 32-36; scheme R-S10): first-order shape, two straight segments joined at
// the relay point  x_r = min(min(ia,ib)+1, max(max(ia,ib), (xa+xb)/2))  per axis, positions taken
// relative to node (ia, ja).  Segment s lives in cell (ia,ja) [s=0] or (ib,jb) [s=1].
// J3 = q w (alpha/gamma) u^3 (Eq. 36), half per segment, bilinear on the cell's four nodes.
//
// `v3` = (alpha/gamma)(h^13 u_1 + h^33 u_3) at the midpoint of the deposited path.
// `sink(s, J1lo, J1hi, J2lo, J2hi, J3_00, J3_10, J3_01, J3_11)` receives, for segment s:
//    J1(c1+1/2, c2) += J1lo   J1(c1+1/2, c2+1) += J1hi
//    J2(c1, c2+1/2) += J2lo   J2(c1+1, c2+1/2) += J2hi
//    J3(c1+k, c2+l) += J3_kl
// ------------------------------------------------------------------------------------------------
template <typename T, typename Sink>
__device__ __forceinline__ void deposit_segments(int di, int dj, T xa, T ya, T dx1_new, T dx2_new, T qw_over_dt,
                                                 T qw, T v3, Sink&& sink) {
  const T xb = (T)di + dx1_new, yb = (T)dj + dx2_new;
  const T xr = fmin((T)(di < 0 ? di : 0) + T(1), fmax((T)(di > 0 ? di : 0), T(0.5) * (xa + xb)));
  const T yr = fmin((T)(dj < 0 ? dj : 0) + T(1), fmax((T)(dj > 0 ? dj : 0), T(0.5) * (ya + yb)));
  const T F3 = T(0.5) * qw * v3;
  {
    const T F1 = qw_over_dt * (xr - xa), F2 = qw_over_dt * (yr - ya);
    const T W1 = T(0.5) * (xa + xr), W2 = T(0.5) * (ya + yr);
    const T F3a = F3 * (T(1) - W1), F3b = F3 * W1;
    sink(0, F1 * (T(1) - W2), F1 * W2, F2 * (T(1) - W1), F2 * W1, F3a * (T(1) - W2), F3b * (T(1) - W2), F3a * W2,
         F3b * W2);
  }
  {
    const T F1 = qw_over_dt * (xb - xr), F2 = qw_over_dt * (yb - yr);
    const T W1 = T(0.5) * (xr + xb) - (T)di, W2 = T(0.5) * (yr + yb) - (T)dj;
    const T F3a = F3 * (T(1) - W1), F3b = F3 * W1;
    sink(1, F1 * (T(1) - W2), F1 * W2, F2 * (T(1) - W1), F2 * W1, F3a * (T(1) - W2), F3b * (T(1) - W2), F3a * W2,
         F3b * W2);
  }
}

// out-of-plane velocity of Eq. 36 at the midpoint of the path (ia + (xa+xb)/2, ja + (ya+yb)/2), theta clamped
template <typename T>
__device__ __forceinline__ T v3_at_path_midpoint(const Consts<T>& g, int ia, int ja, T xm, T ym, T u1, T u2, T u3,
                                                 T eps) {
  Coord<T> X;
  X.init(g, ia, xm, ja, ym);
  T r, sth, cth;
  X.at(g, T(0), T(0), r, sth, cth);
  MetricLite<T> mm;
  metric_lite(g, r, sth, cth, mm);
  const T iu0 = inv_u0(mm, u1 * u1, u2 * u2, u3 * u3, T(2) * u1 * u3, eps);
  return (mm.hu13 * u1 + mm.hu33 * u3) * iu0;
}

}  // namespace grpic
