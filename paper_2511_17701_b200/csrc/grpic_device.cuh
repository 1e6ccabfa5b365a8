// grpic_device.cuh — per-particle device arithmetic of the GRPIC hot path (sm_100a).
//
// Everything here is written from the paper's equations ("P:n" = PAPER.md line n) and from the
// readings listed in DESIGN.md ("R-Sk"); it shares nothing with oracle/.  One source, two
// precisions: T = float (libgrpic_f32.so) or double (libgrpic_f64.so).
//
// All metric quantities are recomputed in registers from (cell, displacement, spin, map constants);
// nothing is tabulated.  Notation follows App. A: Sigma, Delta, A, z, alpha, beta^1,
// h^{ij} ("hu"), h_{ij} ("hd"), code basis of the log-r map A.3 with s1 = dxi*r, s2 = deta.
//
// The formulas are the paper's, rearranged so that the two fixed-point loops (Eq. 26-29) execute as few
// instructions as possible:
//   - with s1 = dxi*r the shift is beta^1 = (2/dxi)/(Sigma+2r), and alpha/gamma = Sigma * rsqrt((Sigma+2r) G)
//     with G = Sigma*gamma^2, so 1/Sigma is never formed inside the coordinate loop;
//   - everything that does not change between iterations (u-dependent products, dt factors, the
//     derivative terms that multiply u_3) is folded before the loops.
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
  int32_t ld;          // row length of every grid array: n2 + 2*ng
  int32_t early_exit;  // leave a fixed-point loop once the iterate repeats bit for bit (identical result)
  T a, a2;             // spin and its square
  T log_rmin;          // xi at x1 = 0
  T dxi, deta;         // d(xi)/d(x1), d(theta)/d(x2)
  T inv_dxi;           // 1/dxi
  T inv_deta2;         // 1/deta^2
  T th_min, th_max;    // [small_angle, pi - small_angle]
  T sin_min, cos_min;  // sin, cos of th_min
  T sin_max, cos_max;  // sin, cos of th_max (FP64: the values the plain formula gives at the clamped angle)
  // full A.3 map; both zero in the five BASELINE configs, which then run the specialised Coord<T>
  T r_off;             // radial offset r0: xi = log(r - r0); log_rmin = log(r_min - r0)
  T h0;                // polar stretch: theta = eta + 2 h0 eta (pi - 2 eta)(pi - eta)/pi^2
  // spherical Kerr-Schild map of A.2: r = r_min + x1*dr.  Then dxi = inv_dxi = 1 and rm = dr, so that
  // s1 = dxi*rm = dr everywhere below, and dls1 = d ln(s1)/dx1 = 0 (A.3: dls1 = dxi)
  int32_t r_lin;
  T r_min, dr, dls1;
  // M in units of r_g (1 in the paper's GR runs); M = 0 with a = 0 is the flat kerr_schild_0 metric of A.1.
  // Only the general-map functions read it; Coord<T> / metric_full / eval have M = 1 folded in.
  T mass;
};

// what the metric at a point needs from the coordinate map besides (r, theta)
template <typename T>
struct MapLocal {
  T rm;        // r - r0            (s1 = dxi*rm)
  T s2;        // dtheta/dx2 = deta * dtheta/deta
  T inv_s2sq;  // 1/s2^2
  T dls2;      // d ln(s2)/dx2
};

// ------------------------------------------------------------------------------------------------
// scalar helpers: IEEE operators in FP64; hardware approximations (<= 2 ulp) in FP32
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp_(double x) { return 1.0 / x; }
__device__ __forceinline__ double rsqrt_(double x) { return rsqrt(x); }
__device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
__device__ __forceinline__ double floor_(double x) { return floor(x); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ double abs_(double x) { return fabs(x); }
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
__device__ __forceinline__ float floor_(float x) { return floorf(x); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float abs_(float x) { return fabsf(x); }
__device__ __forceinline__ float below_one(float) { return 0x1.fffffep-1f; }

// Three reciprocals at once.  FP32: three MUFU.RCP.  FP64 has no hardware reciprocal (each 1/x is a Newton sequence of
// ~12 instructions): one division of the product and six multiplications instead.  The products stay far inside the
// FP64 range for the arguments of this file (r, Sigma, Sigma + 2r, sin^2(theta) >= 1e-10).
__device__ __forceinline__ void rcp3_(float a, float b, float c, float& ia, float& ib, float& ic) {
  ia = rcp_(a); ib = rcp_(b); ic = rcp_(c);
}
__device__ __forceinline__ void rcp3_(double a, double b, double c, double& ia, double& ib, double& ic) {
  const double ab = a * b;
  const double inv = 1.0 / (ab * c);
  ic = inv * ab;
  const double ic_c = inv * c;      // 1/(a b)
  ia = ic_c * b;
  ib = ic_c * a;
}

// A kernel parameter copied into a register the compiler cannot rematerialise from the constant bank:
// without this ptxas re-reads loop constants with LDCU + MOV in every iteration of the fixed-point loops.
__device__ __forceinline__ float in_reg(float x) {
  float y;
  asm volatile("mov.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ double in_reg(double x) {
  double y;
  asm volatile("mov.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}
__device__ __forceinline__ int in_reg(int x) {
  int y;
  asm volatile("mov.s32 %0, %1;" : "=r"(y) : "r"(x));
  return y;
}

// exp(e) - 1 ... as 1 + e + ... and sin(d), cos(d) for the small in-step displacements of the midpoint
// iteration.  Truncation errors (relative): FP32 |e| < 0.04: e^5/120 < 1e-9; |d| < 0.045: d^4/120, d^6/720 < 4e-8.
// FP64 |e| < 0.04: e^11/11! < 2e-23; |d| < 0.045: d^12/12!, d^13/13! < 2e-25.
__device__ __forceinline__ float exp_small(float e) {
  float p = fmaf(e, 1.f / 24.f, 1.f / 6.f);
  p = fmaf(p, e, 0.5f);
  p = fmaf(p, e, 1.f);
  return fmaf(p, e, 1.f);
}
__device__ __forceinline__ void sincos_small(float d, float& sd, float& cd) {
  const float d2 = d * d;
  sd = fmaf(d * d2, -1.f / 6.f, d);
  cd = fmaf(d2, fmaf(d2, 1.f / 24.f, -0.5f), 1.f);
}
__device__ __forceinline__ double exp_small(double e) {
  double p = fma(e, 1.0 / 3628800.0, 1.0 / 362880.0);
  p = fma(p, e, 1.0 / 40320.0);
  p = fma(p, e, 1.0 / 5040.0);
  p = fma(p, e, 1.0 / 720.0);
  p = fma(p, e, 1.0 / 120.0);
  p = fma(p, e, 1.0 / 24.0);
  p = fma(p, e, 1.0 / 6.0);
  p = fma(p, e, 0.5);
  p = fma(p, e, 1.0);
  return fma(p, e, 1.0);
}
__device__ __forceinline__ void sincos_small(double d, double& sd, double& cd) {
  const double d2 = d * d;
  double p = fma(d2, -1.0 / 39916800.0, 1.0 / 362880.0);
  p = fma(p, d2, -1.0 / 5040.0);
  p = fma(p, d2, 1.0 / 120.0);
  p = fma(p, d2, -1.0 / 6.0);
  sd = fma(p * d2, d, d);
  double q = fma(d2, -1.0 / 3628800.0, 1.0 / 40320.0);
  q = fma(q, d2, -1.0 / 720.0);
  q = fma(q, d2, 1.0 / 24.0);
  q = fma(q, d2, -0.5);
  cd = fma(q, d2, 1.0);
}
// sin and cos of theta' in [0, pi/2 + a cell]: theta' is folded at pi/4 — the complement pi/2 - theta' is formed
// from the integer cell count, so it is exact to one rounding — and the classic single-precision minimax
// polynomials of the quadrant reduction are evaluated on [0, pi/4 + a cell] (< 1 ulp there).  No range
// reduction, no slow path, no local memory (sincosf carries a Payne-Hanek branch).
__device__ __forceinline__ void sincos_first_quadrant(float cells, float comp_cells, float half_cells, float deta,
                                                      float& s, float& c) {
  const bool hi = cells > 0.5f * half_cells;                 // theta' > pi/4
  const float z = (hi ? comp_cells : cells) * deta;
  const float z2 = z * z;
  float ps = fmaf(z2, -1.9515295891e-4f, 8.3321608736e-3f);
  ps = fmaf(ps, z2, -1.6666654611e-1f);
  const float sz = fmaf(ps * z2, z, z);
  float pc = fmaf(z2, 2.443315711809948e-5f, -1.388731625493765e-3f);
  pc = fmaf(pc, z2, 4.166664568298827e-2f);
  const float cz = fmaf(pc * z2, z2, fmaf(z2, -0.5f, 1.0f));
  s = hi ? cz : sz;
  c = hi ? sz : cz;
}

template <typename T> struct SmallLimits;
template <> struct SmallLimits<float> { static constexpr float e = 0.04f, d = 0.045f; };
template <> struct SmallLimits<double> { static constexpr double e = 0.04, d = 0.045; };

// ------------------------------------------------------------------------------------------------
// Coordinate map (r0 = 0, h0 = 0) and the axis regularisation (R-S9).
//
// r, sin(theta), cos(theta) at x^(n) are evaluated once with the library functions; a midpoint
// x^(n) + h is then reached by r0*exp(h1*dxi) and the angle-addition formulas with short polynomials
// in the small displacement (library functions beyond SmallLimits).
// FP64: theta = (x2 + h2)*deta is formed exactly as the plain formula forms it, so that the
//   ill-conditioned sin(theta) next to theta = pi sees the same rounded angle.
// FP32: theta is measured from the NEARER axis (theta' = pi - theta on the lower half, exact in the
//   integer part) so that sin(theta) keeps full relative accuracy next to theta = pi, and a midpoint is
//   never formed by re-adding i + dx + h in FP32 (ulp(2048) = 2.4e-4 cells).
// ------------------------------------------------------------------------------------------------
template <typename T>
struct Coord;

template <>
struct Coord<double> {
  static constexpr bool kGeneral = false;
  double x2, r0, th0, s0, c0;
  __device__ __forceinline__ void local0(const Consts<double>& g, MapLocal<double>& L) const {
    L.rm = r0; L.s2 = g.deta; L.inv_s2sq = g.inv_deta2; L.dls2 = 0.0;
  }
  __device__ __forceinline__ void init(const Consts<double>& g, int i1, double dx1, int i2, double dx2) {
    const double x1 = (double)i1 + dx1;
    x2 = (double)i2 + dx2;
    r0 = exp(g.log_rmin + x1 * g.dxi);
    th0 = x2 * g.deta;
    sincos(th0, &s0, &c0);
  }
  // r, sin(theta), cos(theta) at x^(n) itself (theta clamped)
  __device__ __forceinline__ void at0(const Consts<double>& g, double& r, double& sth, double& cth) const {
    r = r0; sth = s0; cth = c0;
    if (th0 < g.th_min) { sth = g.sin_min; cth = g.cos_min; }
    if (th0 > g.th_max) { sth = g.sin_max; cth = g.cos_max; }
  }
  __device__ __forceinline__ void at(const Consts<double>& g, double h1, double h2, double& r, double& sth,
                                     double& cth) const {
    const double e = h1 * g.dxi;
    const double th = (x2 + h2) * g.deta;
    const double d = th - th0;
    if (fabs(e) < SmallLimits<double>::e && fabs(d) < SmallLimits<double>::d) {
      r = r0 * exp_small(e);
      double sd, cd;
      sincos_small(d, sd, cd);
      sth = fma(s0, cd, c0 * sd);
      cth = fma(c0, cd, -s0 * sd);
    } else {
      r = r0 * exp(e);
      sincos(th, &sth, &cth);
    }
    if (th < g.th_min) { sth = g.sin_min; cth = g.cos_min; }
    if (th > g.th_max) { sth = g.sin_max; cth = g.cos_max; }
  }
  // Loop form of at(): r and sin(theta) only (Eq. 29 needs no cos), polynomial branch only, loop constants
  // in registers.  Returns false if the displacement is outside SmallLimits (the caller then redoes the
  // loop with at()).  Same arithmetic as the polynomial branch of at().
  struct Fast {
    double hdxi, deta, th_min, th_max, sin_min, sin_max;
    __device__ __forceinline__ void init(const Consts<double>& g, const Coord<double>&) {
      hdxi = in_reg(0.5 * g.dxi); deta = in_reg(g.deta);
      th_min = in_reg(g.th_min); th_max = in_reg(g.th_max);
      sin_min = in_reg(g.sin_min); sin_max = in_reg(g.sin_max);
    }
  };
  __device__ __forceinline__ void at_fast(const Fast& f, double del1, double del2, double& r, double& sth,
                                          double& big) const {
    const double e = del1 * f.hdxi;
    const double th = (x2 + 0.5 * del2) * f.deta;
    const double d = th - th0;
    big = fmax(big, fmax(fabs(e), fabs(d)));
    r = r0 * exp_small(e);
    double sd, cd;
    sincos_small(d, sd, cd);
    sth = fma(s0, cd, c0 * sd);
    if (th < f.th_min) sth = f.sin_min;
    if (th > f.th_max) sth = f.sin_max;
  }
};

template <>
struct Coord<float> {
  static constexpr bool kGeneral = false;
  __device__ __forceinline__ void local0(const Consts<float>& g, MapLocal<float>& L) const {
    L.rm = r0; L.s2 = g.deta; L.inv_s2sq = g.inv_deta2; L.dls2 = 0.f;
  }
  float r0, thp, s0, c0, sgn;  // r, theta', sin(theta'), cos(theta') at x (theta' unclamped); +1 or -1 (mirrored)
  __device__ __forceinline__ void init(const Consts<float>& g, int i1, float dx1, int i2, float dx2) {
    const float xi = fmaf(dx1, g.dxi, fmaf((float)i1, g.dxi, g.log_rmin));
    r0 = expf(xi);
    const bool upper = 2 * i2 >= g.n2;
    const float fc = (float)(upper ? g.n2 - i2 : i2);          // whole cells from the nearer axis
    const float sdx = upper ? -dx2 : dx2;
    sgn = upper ? -1.f : 1.f;
    const float cells = fc + sdx;
    const float half = 0.5f * (float)g.n2;                     // cells in a quadrant
    thp = cells * g.deta;
    sincos_first_quadrant(cells, (half - fc) - sdx, half, g.deta, s0, c0);
  }
  __device__ __forceinline__ void at0(const Consts<float>& g, float& r, float& sth, float& cth) const {
    float s = s0, c = c0;
    if (thp < g.th_min) { s = g.sin_min; c = g.cos_min; }
    if (thp > g.th_max) { s = g.sin_min; c = -g.cos_min; }
    r = r0; sth = s; cth = sgn * c;
  }
  __device__ __forceinline__ void at(const Consts<float>& g, float h1, float h2, float& r, float& sth,
                                     float& cth) const {
    const float e = h1 * g.dxi;
    const float d = (sgn * g.deta) * h2;
    const float th = thp + d;
    float s, c;
    if (fabsf(e) < SmallLimits<float>::e && fabsf(d) < SmallLimits<float>::d) {
      r = r0 * exp_small(e);
      float sd, cd;
      sincos_small(d, sd, cd);
      s = fmaf(s0, cd, c0 * sd);
      c = fmaf(c0, cd, -s0 * sd);
    } else {
      r = r0 * expf(e);
      sincosf(th, &s, &c);
    }
    // axis regularisation: theta' clamped to [th_min, th_max]
    if (th < g.th_min) { s = g.sin_min; c = g.cos_min; }
    if (th > g.th_max) { s = g.sin_min; c = -g.cos_min; }
    sth = s;
    cth = sgn * c;
  }
  // Loop form of at(): r and sin(theta) only, polynomial branch only, loop constants in registers.
  // theta' = thp + d is measured from the nearer axis, so inside SmallLimits it never reaches th_max and
  // only the lower clamp is tested.  Returns false outside SmallLimits (the caller redoes the loop with at()).
  struct Fast {
    float hdxi, hdeta, th_min, sin_min;
    __device__ __forceinline__ void init(const Consts<float>& g, const Coord<float>& X) {
      hdxi = in_reg(0.5f * g.dxi); hdeta = in_reg((0.5f * X.sgn) * g.deta);
      th_min = in_reg(g.th_min); sin_min = in_reg(g.sin_min);
    }
  };
  // `big` accumulates max(|e|, |d|) over the loop: one FMNMX3-style update instead of two compares and selects;
  // the caller tests it once against the smaller of the two SmallLimits (conservative).
  __device__ __forceinline__ void at_fast(const Fast& f, float del1, float del2, float& r, float& sth, float& big) const {
    const float e = del1 * f.hdxi;
    const float d = del2 * f.hdeta;
    big = fmaxf(big, fmaxf(fabsf(e), fabsf(d)));
    r = r0 * exp_small(e);
    float sd, cd;
    sincos_small(d, sd, cd);
    float s = fmaf(s0, cd, c0 * sd);
    if (thp + d < f.th_min) s = f.sin_min;
    sth = s;
  }
};

// ------------------------------------------------------------------------------------------------
// General A.3 map: radial offset r0 and polar stretch h0.  Plain evaluation with the library
// functions at every point (no polynomial shortcuts): this class serves contexts with r0 != 0 or h0 != 0,
// the five BASELINE configs run Coord<T> above.  theta(eta) is symmetric about the equator, so FP32 again
// measures eta from the NEARER axis; FP64 forms x1, x2 and the angle exactly as the plain formulas do.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void sincos_(double x, double& s, double& c) { sincos(x, &s, &c); }
__device__ __forceinline__ void sincos_(float x, float& s, float& c) { sincosf(x, &s, &c); }
__device__ __forceinline__ double exp_(double x) { return exp(x); }
__device__ __forceinline__ float exp_(float x) { return expf(x); }

template <typename T>
struct CoordGen {
  static constexpr bool kGeneral = true;
  static constexpr bool kMirror = sizeof(T) == 4;
  T a1, a2;        // FP64: x1, x2 of x^(n);  FP32: xi and eta' (from the nearer axis) of x^(n)
  T sgn;           // -1 when mirrored onto the axis theta = pi
  T r0, rm0, th0, s0, c0, q0;   // at x^(n): r, r - r_off, theta('), sin, cos, dtheta/deta

  __device__ __forceinline__ static T theta_of(const Consts<T>& g, T eta) {
    if (kMirror) {
      const T x = eta * T(0.31830988618379067154);                     // eta/pi
      return eta * fma_(T(2) * g.h0, (T(1) - T(2) * x) * (T(1) - x), T(1));
    }
    const T pi = T(3.14159265358979323846);                            // FP64: the plain formula, term by term
    return eta + T(2) * g.h0 * eta * (pi - T(2) * eta) * (pi - eta) / (pi * pi);
  }
  __device__ __forceinline__ static T dtheta_deta(const Consts<T>& g, T eta) {
    if (kMirror) {
      const T x = eta * T(0.31830988618379067154);
      return fma_(T(12) * g.h0, x * (x - T(1)), fma_(T(2), g.h0, T(1)));
    }
    const T pi = T(3.14159265358979323846);
    return T(1) + T(2) * g.h0 + T(12) * g.h0 * (eta / pi) * (eta / pi - T(1));
  }
  // (xi, eta or eta') of the point x^(n) + (h1, h2); on the A.2 map "xi" is r itself
  __device__ __forceinline__ void point(const Consts<T>& g, T h1, T h2, T& xi, T& eta) const {
    if (kMirror) {
      xi = fma_(h1, g.r_lin ? g.dr : g.dxi, a1);
      eta = fma_(sgn * g.deta, h2, a2);
    } else {
      xi = g.r_lin ? g.r_min + (a1 + h1) * g.dr : g.log_rmin + (a1 + h1) * g.dxi;
      eta = (a2 + h2) * g.deta;
    }
  }
  // r and r - r_off (A.3) or r and dr (A.2) from the radial coordinate of point()
  __device__ __forceinline__ void radius(const Consts<T>& g, T xi, T& r, T& rm) const {
    if (g.r_lin) { r = xi; rm = g.dr; }
    else { rm = exp_(xi); r = g.r_off + rm; }
  }
  __device__ __forceinline__ void trig(const Consts<T>& g, T eta, T& sth, T& cth) const {
    const T th = theta_of(g, eta);
    T s, c;
    sincos_(th, s, c);
    if (kMirror) {
      if (th < g.th_min) { s = g.sin_min; c = g.cos_min; }
      c = sgn * c;
    } else {
      if (th < g.th_min) { s = g.sin_min; c = g.cos_min; }
      if (th > g.th_max) { s = g.sin_max; c = g.cos_max; }
    }
    sth = s; cth = c;
  }
  __device__ __forceinline__ void init(const Consts<T>& g, int i1, T dx1, int i2, T dx2) {
    sgn = T(1);
    if (kMirror) {
      a1 = g.r_lin ? fma_(dx1, g.dr, fma_((T)i1, g.dr, g.r_min)) : fma_(dx1, g.dxi, fma_((T)i1, g.dxi, g.log_rmin));
      const bool upper = 2 * i2 >= g.n2;
      sgn = upper ? T(-1) : T(1);
      a2 = ((T)(upper ? g.n2 - i2 : i2) + (upper ? -dx2 : dx2)) * g.deta;
    } else {
      a1 = (T)i1 + dx1;
      a2 = (T)i2 + dx2;
    }
    T xi, eta;
    point(g, T(0), T(0), xi, eta);
    radius(g, xi, r0, rm0);
    trig(g, eta, s0, c0);
    q0 = dtheta_deta(g, eta);
    th0 = eta;
  }
  __device__ __forceinline__ void at0(const Consts<T>&, T& r, T& sth, T& cth) const { r = r0; sth = s0; cth = c0; }
  __device__ __forceinline__ void local0(const Consts<T>& g, MapLocal<T>& L) const {
    L.rm = rm0;
    L.s2 = g.deta * q0;
    L.inv_s2sq = g.inv_deta2 * rcp_(q0 * q0);
    const T x = th0 * T(0.31830988618379067154);
    L.dls2 = (sgn * g.deta) * (T(3.8197186342054880585) * g.h0) * (T(2) * x - T(1)) * rcp_(q0);   // 12 h0/pi (2x-1)/q
  }
  struct Fast {
    __device__ __forceinline__ void init(const Consts<T>&, const CoordGen<T>&) {}
  };
  // r, r - r_off, 1/(dtheta/deta)^2 and sin(theta) at the midpoint of the displacement (del1, del2)
  __device__ __forceinline__ void at_mid(const Consts<T>& g, T del1, T del2, T& r, T& rm, T& iq2, T& sth) const {
    T xi, eta, cth;
    point(g, T(0.5) * del1, T(0.5) * del2, xi, eta);
    radius(g, xi, r, rm);
    trig(g, eta, sth, cth);
    const T q = dtheta_deta(g, eta);
    iq2 = rcp_(q * q);
  }
};

// ------------------------------------------------------------------------------------------------
// Midpoint evaluation of Eq. 29/30: everything Eq. 29 needs from the metric at (r, sin theta),
// for a fixed u.  With w1 = u_1/s1, U2 = u_2/s2 (physical-basis covariant components):
//   G = Sigma gamma^2 = eps Sigma + A w1^2/(Sigma+2r) + U2^2 + u_3^2/sin^2 + 2 a w1 u_3      (Eq. 20)
//   1/u^0 = alpha/gamma = Sigma R,   R = rsqrt((Sigma + 2r) G)
//   dx^1/dt = (h^11 u_1 + h^13 u_3)/u^0 - beta^1 = [(A w1/(Sigma+2r) + a u_3)/r * R - 2/(Sigma+2r)]/dxi
//   dx^2/dt = h^22 u_2/u^0 = (u_2/deta^2) R
//   dphi/dt = (h^13 u_1 + h^33 u_3)/u^0 = (a w1 + u_3/sin^2) R
// ------------------------------------------------------------------------------------------------
template <typename T>
struct MidU {           // per-particle constants of the coordinate loop
  T w1c;                // u_1/dxi          (w1 = w1c / r)
  T U2sq;               // (u_2/deta)^2
  T u3, u3sq, au3, c2au3;
  T k1, k2;             // dt/dxi,  dt u_2/deta^2
  T eps, a2;
  __device__ __forceinline__ void init(const Consts<T>& g, T u1, T u2, T u3_, T eps_, T dt) {
    w1c = u1 * g.inv_dxi;
    U2sq = (u2 * u2) * g.inv_deta2;
    u3 = u3_;
    u3sq = u3_ * u3_;
    au3 = g.a * u3_;
    c2au3 = au3 + au3;
    k1 = dt * g.inv_dxi;
    k2 = (dt * u2) * g.inv_deta2;
    eps = eps_;
    a2 = in_reg(g.a2);
  }
};

template <typename T>
struct MidEval {
  T R, w1, is2;
  // returns the two displacement rates times dt
  __device__ __forceinline__ void eval(const Consts<T>& g, const MidU<T>& U, T r, T sth, T& n1, T& n2) {
    const T s2 = sth * sth;
    const T a2s2 = U.a2 * s2;
    const T r2a2 = fma_(r, r, U.a2);
    const T Sigma = r2a2 - a2s2;
    const T Sp2r = fma_(T(2), r, Sigma);
    const T Delta = fma_(r, r - T(2), U.a2);
    const T A = fma_(-a2s2, Delta, r2a2 * r2a2);
    T ir, iSp2r;
    rcp3_(r, Sp2r, s2, ir, iSp2r, is2);
    w1 = U.w1c * ir;
    const T t = (A * iSp2r) * w1;
    T G = fma_(U.eps, Sigma, U.U2sq);
    G = fma_(t, w1, G);
    G = fma_(U.u3sq, is2, G);
    G = fma_(U.c2au3, w1, G);
    R = rsqrt_(Sp2r * G);
    n1 = U.k1 * fma_((t + U.au3) * ir, R, T(-2) * iSp2r);
    n2 = U.k2 * R;
  }
  // General A.3 map: s1 = dxi*(r - r0) and s2 = deta*q with q = dtheta/deta at the midpoint (iq2 = 1/q^2).
  //   beta^1 = 2r/((Sigma+2r) s1),  h^22 = 1/(Sigma s2^2);  the rest as above with 1/r -> 1/(r - r0).
  __device__ __forceinline__ void eval_gen(const Consts<T>& g, const MidU<T>& U, T r, T rm, T iq2, T sth, T& n1,
                                           T& n2) {
    const T s2 = sth * sth;
    const T a2s2 = U.a2 * s2;
    const T r2a2 = fma_(r, r, U.a2);
    const T Sigma = r2a2 - a2s2;
    const T M2 = T(2) * g.mass;
    const T Sp2r = fma_(M2, r, Sigma);
    const T Delta = fma_(r, r - M2, U.a2);
    const T A = fma_(-a2s2, Delta, r2a2 * r2a2);
    T irm, iSp2r;
    rcp3_(rm, Sp2r, s2, irm, iSp2r, is2);
    w1 = U.w1c * irm;
    const T t = (A * iSp2r) * w1;
    T G = fma_(U.eps, Sigma, U.U2sq * iq2);
    G = fma_(t, w1, G);
    G = fma_(U.u3sq, is2, G);
    G = fma_(U.c2au3, w1, G);
    R = rsqrt_(Sp2r * G);
    n1 = U.k1 * fma_((t + U.au3) * irm, R, (-M2 * r) * (irm * iSp2r));
    n2 = (U.k2 * iq2) * R;
  }
  __device__ __forceinline__ T dphidt(const Consts<T>& g, const MidU<T>& U) const {
    return fma_(g.a, w1, U.u3 * is2) * R;
  }
};

// ------------------------------------------------------------------------------------------------
// Full set at x^(n): tetrad coefficients and the Eq. 27 coefficients, with the analytic
// derivatives of App. A (general rule P:772-778; A.2 list P:814-816; the A.3 extras from
// s1 = dxi*exp(xi) depending on x1; corrections R-S2) written in logarithmic form:
//   d h^22 = -h^22 dSigma/Sigma;  d h^33 = -h^33 (dSigma/Sigma + 2 cot(theta) dtheta);
//   d h^13 = -h^13 (dSigma/Sigma + dxi [x1 only]);  d beta^1 = -beta^1 (dSigma + 2 s1 [x1 only])/(Sigma+2r);
//   d alpha = (r dSigma - Sigma dr)/((Sigma+2r)^2 alpha);
//   d h^11 = dA/(Sigma (Sigma+2r) s1^2) - h^11 (dSigma/Sigma + (dSigma + 2 s1 [x1])/(Sigma+2r) + 2 dxi [x1]).
// ------------------------------------------------------------------------------------------------
template <typename T>
struct MetricFull {
  T alpha, hu11, hu22, hu33, hu13;
  T hd22, hd33, hd13;
  T d_alpha[2], d_beta1[2], d_hu11[2], d_hu22[2], d_hu33[2], d_hu13[2];  // [0] = d/dx1, [1] = d/dx2
};

template <typename T>
__device__ __forceinline__ void metric_full(const Consts<T>& g, T r, T sth, T cth, MetricFull<T>& m) {
  const T a = g.a, a2 = g.a2;
  const T r2 = r * r;
  const T s2th = sth * sth;
  const T a2s2 = a2 * s2th;
  const T r2a2 = r2 + a2;
  const T Sigma = fma_(a2 * cth, cth, r2);
  const T Delta = fma_(r, r - T(2), a2);
  const T A = fma_(-a2s2, Delta, r2a2 * r2a2);
  const T Sp2r = fma_(T(2), r, Sigma);
  const T s1 = g.dxi * r;
  T iS, iSp2r, is2th;
  rcp3_(Sigma, Sp2r, s2th, iS, iSp2r, is2th);
  const T is1 = g.inv_dxi * rcp_(r);
  const T al2 = Sigma * iSp2r;                   // alpha^2 = 1/(1+z)
  const T ial = rsqrt_(al2);
  m.alpha = al2 * ial;
  const T beta1 = (T(2) * g.inv_dxi) * iSp2r;
  const T B = (iS * iSp2r) * (is1 * is1);        // 1/(Sigma (Sigma+2r) s1^2)
  m.hu11 = A * B;
  m.hu22 = iS * g.inv_deta2;
  m.hu33 = iS * is2th;
  m.hu13 = (a * iS) * is1;
  m.hd22 = (g.deta * g.deta) * Sigma;
  m.hd33 = (A * s2th) * iS;
  m.hd13 = -(s1 * a) * ((Sp2r * iS) * s2th);

  const T d1S = (T(2) * r) * s1;
  const T d2S = (T(-2) * a2 * g.deta) * (sth * cth);
  const T d1A = (T(4) * r * s1) * r2a2 - a2s2 * ((T(2) * (r - T(1))) * s1);
  const T d2A = d2S * Delta;
  const T l1S = d1S * iS, l2S = d2S * iS;        // d ln Sigma
  const T l1P = (d1S + T(2) * s1) * iSp2r;       // d ln (Sigma + 2r)
  const T l2P = d2S * iSp2r;
  m.d_hu11[0] = fma_(B, d1A, -m.hu11 * (l1S + l1P + T(2) * g.dxi));
  m.d_hu11[1] = fma_(B, d2A, -m.hu11 * (l2S + l2P));
  m.d_hu22[0] = -m.hu22 * l1S;
  m.d_hu22[1] = -m.hu22 * l2S;
  m.d_hu33[0] = -m.hu33 * l1S;
  m.d_hu33[1] = -m.hu33 * fma_((T(2) * g.deta) * cth, rcp_(sth), l2S);
  m.d_hu13[0] = -m.hu13 * (l1S + g.dxi);
  m.d_hu13[1] = -m.hu13 * l2S;
  m.d_beta1[0] = -beta1 * l1P;
  m.d_beta1[1] = -beta1 * l2P;
  const T ka = (iSp2r * iSp2r) * ial;            // 1/((Sigma+2r)^2 alpha)
  m.d_alpha[0] = fma_(r, d1S, -Sigma * s1) * ka;
  m.d_alpha[1] = (r * d2S) * ka;
}

// The same set for the general A.3 map: s1 = dxi (r - r0), s2 = deta dtheta/deta (MapLocal).  Differences:
//   beta^1 = 2r/((Sigma+2r) s1)  ->  d_1 ln beta^1 = s1/r - dxi - d_1 ln(Sigma+2r);
//   h^22 = 1/(Sigma s2^2)        ->  d_2 ln h^22 = -d_2 ln Sigma - 2 d_2 ln s2   (the entry P:842 omits);
//   d_2 Sigma, d_2 A and the cot(theta) term of h^33 carry the local s2.
template <typename T>
__device__ __forceinline__ void metric_full_gen(const Consts<T>& g, const MapLocal<T>& L, T r, T sth, T cth,
                                                MetricFull<T>& m) {
  const T a = g.a, a2 = g.a2, M = g.mass;
  const T r2 = r * r;
  const T s2th = sth * sth;
  const T a2s2 = a2 * s2th;
  const T r2a2 = r2 + a2;
  const T Sigma = fma_(a2 * cth, cth, r2);
  const T Delta = fma_(r, r - T(2) * M, a2);
  const T A = fma_(-a2s2, Delta, r2a2 * r2a2);
  const T Sp2r = fma_(T(2) * M, r, Sigma);
  const T s1 = g.dxi * L.rm;
  const T iS = rcp_(Sigma), iSp2r = rcp_(Sp2r), is2th = rcp_(s2th);
  const T is1 = g.inv_dxi * rcp_(L.rm);
  const T al2 = Sigma * iSp2r;
  const T ial = rsqrt_(al2);
  m.alpha = al2 * ial;
  const T beta1 = ((T(2) * M * r) * iSp2r) * is1;
  const T B = (iS * iSp2r) * (is1 * is1);
  m.hu11 = A * B;
  m.hu22 = iS * L.inv_s2sq;
  m.hu33 = iS * is2th;
  m.hu13 = (a * iS) * is1;
  m.hd22 = (L.s2 * L.s2) * Sigma;
  m.hd33 = (A * s2th) * iS;
  m.hd13 = -(s1 * a) * ((Sp2r * iS) * s2th);

  const T d1S = (T(2) * r) * s1;
  const T d2S = (T(-2) * a2 * L.s2) * (sth * cth);
  const T d1A = (T(4) * r * s1) * r2a2 - a2s2 * ((T(2) * (r - M)) * s1);
  const T d2A = d2S * Delta;
  const T l1S = d1S * iS, l2S = d2S * iS;
  const T l1P = (d1S + T(2) * M * s1) * iSp2r;
  const T l2P = d2S * iSp2r;
  m.d_hu11[0] = fma_(B, d1A, -m.hu11 * (l1S + l1P + T(2) * g.dls1));
  m.d_hu11[1] = fma_(B, d2A, -m.hu11 * (l2S + l2P));
  m.d_hu22[0] = -m.hu22 * l1S;
  m.d_hu22[1] = -m.hu22 * (l2S + T(2) * L.dls2);
  m.d_hu33[0] = -m.hu33 * l1S;
  m.d_hu33[1] = -m.hu33 * fma_((T(2) * L.s2) * cth, rcp_(sth), l2S);
  m.d_hu13[0] = -m.hu13 * (l1S + g.dls1);
  m.d_hu13[1] = -m.hu13 * l2S;
  m.d_beta1[0] = beta1 * (s1 * rcp_(r) - g.dls1 - l1P);
  m.d_beta1[1] = -beta1 * l2P;
  const T ka = (iSp2r * iSp2r) * ial;
  m.d_alpha[0] = (M * fma_(r, d1S, -Sigma * s1)) * ka;
  m.d_alpha[1] = (M * r * d2S) * ka;
}

// ------------------------------------------------------------------------------------------------
// Tetrad at x^(n): matrix form of P:754 (R-S3).
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
    Ah[2] = fma_(k13, A[0], sq33 * A[2]);
  }
  __device__ __forceinline__ void cov_to_tetrad(const T u[3], T uh[3]) const {
    uh[0] = sq11 * fma_(-(k13 * isq33), u[2], u[0]);
    uh[1] = u[1] * isq22;
    uh[2] = u[2] * isq33;
  }
  __device__ __forceinline__ void tetrad_to_cov(const T uh[3], T u[3]) const {
    u[0] = fma_(uh[0], isq11, k13 * uh[2]);
    u[1] = sq22 * uh[1];
    u[2] = sq33 * uh[2];
  }
};

// Boris rotation over dt/2 in the orthonormal frame (coefficient c = (q/m) alpha dt/4, R-S5).
// cD = c*D-hat, cB = c*B-hat.
template <typename T>
__device__ __forceinline__ void boris_half(const T cD[3], const T cB[3], T uh[3]) {
  const T um0 = uh[0] + cD[0], um1 = uh[1] + cD[1], um2 = uh[2] + cD[2];
  const T ig = rsqrt_(fma_(um0, um0, fma_(um1, um1, fma_(um2, um2, T(1)))));
  const T t0 = cB[0] * ig, t1 = cB[1] * ig, t2 = cB[2] * ig;
  const T f = T(2) * rcp_(fma_(t0, t0, fma_(t1, t1, fma_(t2, t2, T(1)))));
  const T s0 = f * t0, s1 = f * t1, s2 = f * t2;
  const T p0 = um0 + fma_(um1, t2, -um2 * t1);
  const T p1 = um1 + fma_(um2, t0, -um0 * t2);
  const T p2 = um2 + fma_(um0, t1, -um1 * t0);
  uh[0] = (um0 + fma_(p1, s2, -p2 * s1)) + cD[0];
  uh[1] = (um1 + fma_(p2, s0, -p0 * s2)) + cD[1];
  uh[2] = (um2 + fma_(p0, s1, -p1 * s0)) + cD[2];
}

// ------------------------------------------------------------------------------------------------
// Field gather (step 2; scheme R-S4): every Yee component is first averaged to the four
// corner nodes of the particle's cell, then bilinear in (dx1, dx2).
//   node value of a component at half-integer positions along axis 1 only (D1, B2): (F(i-1,j) + F(i,j))/2
//   along axis 2 only (D2, B1): (F(i,j-1) + F(i,j))/2;  along both (B3): mean of the four;  D3 sits on nodes.
// `F(comp, di, dj)` returns sample (i1 + di, i2 + dj) of component comp (0..5 = D1 D2 D3 B1 B2 B3).
// The tiled kernel does stage (i) once per tile in shared memory and calls bilinear() only.
// ------------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ T bilinear(T c00, T c10, T c01, T c11, T dx1, T dx2) {
  const T o1 = T(1) - dx1;
  const T lo = fma_(c10, dx1, c00 * o1);
  const T hi = fma_(c11, dx1, c01 * o1);
  return fma_(hi, dx2, lo * (T(1) - dx2));
}

template <typename T, typename Acc>
__device__ __forceinline__ T node_value(const Acc& F, int comp, int kind, int i, int j) {
  switch (kind) {
    case 0: return F(comp, i, j);
    case 1: return T(0.5) * (F(comp, i - 1, j) + F(comp, i, j));
    case 2: return T(0.5) * (F(comp, i, j - 1) + F(comp, i, j));
    default: return T(0.25) * (((F(comp, i - 1, j - 1) + F(comp, i - 1, j)) + F(comp, i, j - 1)) + F(comp, i, j));
  }
}

// staggering kind of each component: 1 = half-integer along x1, 2 = along x2, 3 = both, 0 = on nodes
__device__ __forceinline__ constexpr int yee_kind(int comp) {
  return comp == 0 ? 1 : comp == 1 ? 2 : comp == 2 ? 0 : comp == 3 ? 2 : comp == 4 ? 1 : 3;
}

template <typename T, typename Acc>
__device__ __forceinline__ void interp_fields(const Acc& F, T dx1, T dx2, T D[3], T B[3]) {
  T out[6];
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    const int kind = yee_kind(c);
    const T c00 = node_value<T>(F, c, kind, 0, 0), c10 = node_value<T>(F, c, kind, 1, 0);
    const T c01 = node_value<T>(F, c, kind, 0, 1), c11 = node_value<T>(F, c, kind, 1, 1);
    out[c] = bilinear(c00, c10, c01, c11, dx1, dx2);
  }
  D[0] = out[0]; D[1] = out[1]; D[2] = out[2];
  B[0] = out[3]; B[1] = out[4]; B[2] = out[5];
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
template <typename T, typename CoordT = Coord<T>>
__device__ __forceinline__ int push_particle(const Consts<T>& g, PState<T>& p, bool em, const T Dp[3],
                                             const T Bp[3], T qm, T eps, T dt, T& dphidt, bool& reflected) {
  CoordT X;
  X.init(g, p.i1, p.dx1, p.i2, p.dx2);
  T u[3] = {p.u1, p.u2, p.u3};
  {
    T r, sth, cth;
    X.at0(g, r, sth, cth);
    MetricFull<T> m;
    if constexpr (CoordT::kGeneral) {
      MapLocal<T> L;
      X.local0(g, L);
      metric_full_gen(g, L, r, sth, cth, m);
    } else {
      metric_full(g, r, sth, cth, m);
    }

    Tetrad<T> e;
    T cD[3], cB[3], uh[3];
    if (em) {
      const T c = (qm * T(0.25)) * (m.alpha * dt);
      T Dh[3], Bh[3];
      e.init(m);
      e.cntrv_to_tetrad(Dp, Dh);                         // step 3
      e.cntrv_to_tetrad(Bp, Bh);
#pragma unroll
      for (int k = 0; k < 3; ++k) { cD[k] = c * Dh[k]; cB[k] = c * Bh[k]; }
      e.cov_to_tetrad(u, uh);
      boris_half(cD, cB, uh);                            // step 4
      e.tetrad_to_cov(uh, u);                            // step 5
    }
    // step 6, Eq. 26-27: metric frozen at x^(n); exactly n_iter applications, u~(0) = u*
    {
      const T us0 = u[0], us1 = u[1], u3 = u[2];
      // everything that does not change with the iterate (u_3 is fixed), dt folded in
      const T u3sq = u3 * u3;
      const T g2c = fma_(m.hu33, u3sq, eps);
      const T f0c = m.d_hu33[0] * u3sq, f1c = m.d_hu33[1] * u3sq;
      const T h13u3 = (T(2) * m.hu13) * u3;
      const T d13u3_0 = (T(2) * m.d_hu13[0]) * u3, d13u3_1 = (T(2) * m.d_hu13[1]) * u3;
      const T dta0 = dt * m.d_alpha[0], dta1 = dt * m.d_alpha[1];
      const T dtb0 = dt * m.d_beta1[0], dtb1 = dt * m.d_beta1[1];
      const T hadt = (T(0.5) * m.alpha) * dt;             // dt * alpha/2, so that hadt/gamma = dt/(2 u^0)
      const T hus0 = T(0.5) * us0, hus1 = T(0.5) * us1;
      T ut0 = us0, ut1 = us1;
      const int n_iter_u = in_reg(g.n_iter);
      const bool ee_u = g.early_exit != 0;
      for (int it = 0; it < n_iter_u; ++it) {
        const T ub0 = fma_(T(0.5), ut0, hus0), ub1 = fma_(T(0.5), ut1, hus1);
        const T ub1sq = ub1 * ub1;
        const T gam2 = fma_(ub0, fma_(m.hu11, ub0, h13u3), fma_(m.hu22, ub1sq, g2c));
        const T igam = rsqrt_(gam2);
        const T gam = gam2 * igam;                        // alpha u^0
        const T hiu0 = hadt * igam;                       // dt/(2 u^0)
        const T q0 = fma_(ub0, fma_(m.d_hu11[0], ub0, d13u3_0), fma_(m.d_hu22[0], ub1sq, f0c));
        const T q1 = fma_(ub0, fma_(m.d_hu11[1], ub0, d13u3_1), fma_(m.d_hu22[1], ub1sq, f1c));
        const T nt0 = fma_(-hiu0, q0, fma_(ub0, dtb0, fma_(-gam, dta0, us0)));
        const T nt1 = fma_(-hiu0, q1, fma_(ub0, dtb1, fma_(-gam, dta1, us1)));
        // the map is deterministic: once an iterate repeats bit for bit every later one equals it
        const bool fixed = (nt0 == ut0) & (nt1 == ut1);
        ut0 = nt0;
        ut1 = nt1;
        if (fixed && ee_u) break;
      }
      u[0] = ut0;
      u[1] = ut1;
    }
    if (em) {
      e.cov_to_tetrad(u, uh);                            // step 7
      boris_half(cD, cB, uh);                            // step 8
      e.tetrad_to_cov(uh, u);                            // step 9
    }
  }
  // step 10, Eq. 28-29 in displacement space: del = x~ - x^(n); all coefficients at x^(n) + del/2
  T del1 = T(0), del2 = T(0);
  MidU<T> U;
  U.init(g, u[0], u[1], u[2], eps, dt);
  MidEval<T> E;
  bool fixed = false;
  if constexpr (CoordT::kGeneral) {
    // general A.3 map: plain evaluation of the map at every midpoint
    const int n_iter = in_reg(g.n_iter);
    const bool ee = g.early_exit != 0;
    for (int it = 0; it < n_iter; ++it) {
      T r, rm, iq2, sth, n1, n2;
      X.at_mid(g, del1, del2, r, rm, iq2, sth);
      E.eval_gen(g, U, r, rm, iq2, sth, n1, n2);
      fixed = (n1 == del1) & (n2 == del2);
      del1 = n1;
      del2 = n2;
      if (fixed && ee) break;
    }
    if (!fixed) {
      T r, rm, iq2, sth, n1, n2;
      X.at_mid(g, del1, del2, r, rm, iq2, sth);
      E.eval_gen(g, U, r, rm, iq2, sth, n1, n2);
    }
  } else {
    // fast form: polynomial coordinates, loop constants pinned in registers, no branch but the exit test
    typename Coord<T>::Fast XF;
    XF.init(g, X);
    const int n_iter = in_reg(g.n_iter);
    const bool ee = g.early_exit != 0;
    T big = T(0);
    for (int it = 0; it < n_iter; ++it) {
      T r, sth, n1, n2;
      X.at_fast(XF, del1, del2, r, sth, big);
      E.eval(g, U, r, sth, n1, n2);
      // bit-identical iterate => every later iterate is the same: stopping here IS n_iter iterations
      fixed = (n1 == del1) & (n2 == del2);
      del1 = n1;
      del2 = n2;
      if (fixed && ee) break;
    }
    // step 11, Eq. 30 at x_m = (x^(n) + x^(n+1))/2.  If the last iterate repeated, the midpoint
    // of the last evaluation is x_m itself and its coefficients are reused; otherwise evaluate there.
    if (!fixed) {
      T r, sth, n1, n2;
      X.at_fast(XF, del1, del2, r, sth, big);
      E.eval(g, U, r, sth, n1, n2);
    }
    if (!(big < SmallLimits<T>::e)) {                    // e-limit 0.04 < d-limit 0.045; NaN-safe
      // a displacement left SmallLimits (many cells in one step): redo the loop with the library functions
      del1 = T(0); del2 = T(0);
      for (int it = 0; it < g.n_iter; ++it) {
        T r, sth, cth, n1, n2;
        X.at(g, T(0.5) * del1, T(0.5) * del2, r, sth, cth);
        E.eval(g, U, r, sth, n1, n2);
        del1 = n1;
        del2 = n2;
      }
      T r, sth, cth, n1, n2;
      X.at(g, T(0.5) * del1, T(0.5) * del2, r, sth, cth);
      E.eval(g, U, r, sth, n1, n2);
    }
  }
  dphidt = E.dphidt(g, U);
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
// seg[s][0..7] receives, for segment s with cell (c1, c2):
//    [0] J1(c1+1/2, c2)   [1] J1(c1+1/2, c2+1)   [2] J2(c1, c2+1/2)   [3] J2(c1+1, c2+1/2)
//    [4] J3(c1, c2)       [5] J3(c1+1, c2)       [6] J3(c1, c2+1)     [7] J3(c1+1, c2+1)
// ------------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void deposit_segments(int di, int dj, T xa, T ya, T dx1_new, T dx2_new, T qw_over_dt,
                                                 T qw, T v3, T seg[2][8]) {
  const T xb = (T)di + dx1_new, yb = (T)dj + dx2_new;
  const T xr = fmin((T)(di < 0 ? di : 0) + T(1), fmax((T)(di > 0 ? di : 0), T(0.5) * (xa + xb)));
  const T yr = fmin((T)(dj < 0 ? dj : 0) + T(1), fmax((T)(dj > 0 ? dj : 0), T(0.5) * (ya + yb)));
  const T F3 = T(0.5) * qw * v3;
  {
    const T F1 = qw_over_dt * (xr - xa), F2 = qw_over_dt * (yr - ya);
    const T W1 = T(0.5) * (xa + xr), W2 = T(0.5) * (ya + yr);
    const T F3a = F3 * (T(1) - W1), F3b = F3 * W1;
    seg[0][0] = F1 * (T(1) - W2); seg[0][1] = F1 * W2;
    seg[0][2] = F2 * (T(1) - W1); seg[0][3] = F2 * W1;
    seg[0][4] = F3a * (T(1) - W2); seg[0][5] = F3b * (T(1) - W2);
    seg[0][6] = F3a * W2; seg[0][7] = F3b * W2;
  }
  {
    const T F1 = qw_over_dt * (xb - xr), F2 = qw_over_dt * (yb - yr);
    const T W1 = T(0.5) * (xr + xb) - (T)di, W2 = T(0.5) * (yr + yb) - (T)dj;
    const T F3a = F3 * (T(1) - W1), F3b = F3 * W1;
    seg[1][0] = F1 * (T(1) - W2); seg[1][1] = F1 * W2;
    seg[1][2] = F2 * (T(1) - W1); seg[1][3] = F2 * W1;
    seg[1][4] = F3a * (T(1) - W2); seg[1][5] = F3b * (T(1) - W2);
    seg[1][6] = F3a * W2; seg[1][7] = F3b * W2;
  }
}

// out-of-plane velocity of Eq. 36 at the midpoint of the path (ia + xm, ja + ym), theta clamped
template <typename T, typename CoordT = Coord<T>>
__device__ __forceinline__ T v3_at_path_midpoint(const Consts<T>& g, int ia, int ja, T xm, T ym, T u1, T u2, T u3,
                                                 T eps) {
  CoordT X;
  X.init(g, ia, xm, ja, ym);
  MidU<T> U;
  U.init(g, u1, u2, u3, eps, T(1));
  MidEval<T> E;
  T n1, n2;
  if constexpr (CoordT::kGeneral) {
    T r, rm, iq2, sth;
    X.at_mid(g, T(0), T(0), r, rm, iq2, sth);
    E.eval_gen(g, U, r, rm, iq2, sth, n1, n2);
  } else {
    T r, sth, cth;
    X.at0(g, r, sth, cth);
    E.eval(g, U, r, sth, n1, n2);
  }
  return E.dphidt(g, U);
}

}  // namespace grpic
