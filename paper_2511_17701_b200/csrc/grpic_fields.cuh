// grpic_fields.cuh — field-solver half of the step: auxiliary fields (Eq. 38, 42-44),
// Faraday (Eq. 40) and Ampere (Eq. 41) with the polar-axis form of D^1 (Eq. 45).
//
// Grid kernels, one thread per (row, theta index).  They are HBM/latency-trivial next to the particle step (2M cells
// against 134M particles), so clarity wins: the metric at every Yee location is evaluated inline in FP64 from the map
// parameters in BOTH builds (no tables, no FP32 conditioning problem at the axis) and only the field values have the
// build's precision.  Written from the paper's equations; shares nothing with oracle/.
// Readings (DESIGN.md R-F1..R-F3): every <.> of Eq. 44 (garbled in the text) is the two-point volume-weighted average
// along x1 of Eq. 43, formed with sqrt(h~) = sqrt(h)/sin(theta); B^2, D^3 on the axes are not evolved;
// D^1 on the axes takes +H_3 of the neighbouring half cell at theta = 0 and -H_3 at theta = pi.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace grpic {

struct FieldGeom {
  int32_t n1, n2, ng, ld, rows, r_lin;
  double a, mass, r_off, h0, log_rmin, dxi, deta, r_min, dr;
};

struct FM {
  double alpha, h11, h22, h33, h13, sqh_t, beta1, sth;   // sqh_t = sqrt(h)/sin(theta)
};

__device__ __forceinline__ void field_coords(const FieldGeom& q, double x1, double x2, double& r, double& s1, double& th,
                                             double& s2) {
  if (q.r_lin) {
    r = q.r_min + x1 * q.dr;
    s1 = q.dr;
  } else {
    const double rm = exp(q.log_rmin + x1 * q.dxi);
    r = q.r_off + rm;
    s1 = q.dxi * rm;
  }
  const double pi = 3.14159265358979323846;
  const double eta = x2 * q.deta, x = eta / pi;
  th = eta + 2.0 * q.h0 * eta * (pi - 2.0 * eta) * (pi - eta) / (pi * pi);
  s2 = q.deta * (1.0 + 2.0 * q.h0 + 12.0 * q.h0 * x * (x - 1.0));
}

// metric at the code position (x1, x2), NOT clamped at the axis: sin(theta) is exactly 0 on both axes
__device__ __forceinline__ FM field_metric(const FieldGeom& q, double x1, double x2) {
  double r, s1, th, s2, sth, cth;
  field_coords(q, x1, x2, r, s1, th, s2);
  sincos(th, &sth, &cth);
  if (x2 == 0.0 || x2 == (double)q.n2) sth = 0.0;
  const double s2th = sth * sth, a = q.a;
  const double Sigma = r * r + a * a * cth * cth;
  const double Delta = r * r - 2.0 * q.mass * r + a * a;
  const double A = (r * r + a * a) * (r * r + a * a) - a * a * Delta * s2th;
  const double z = 2.0 * q.mass * r / Sigma;
  FM f;
  f.alpha = 1.0 / sqrt(1.0 + z);
  f.h11 = s1 * s1 * (1.0 + z);
  f.h22 = s2 * s2 * Sigma;
  f.h33 = A * s2th / Sigma;
  f.h13 = -s1 * a * (1.0 + z) * s2th;
  f.sqh_t = s1 * s2 * Sigma / f.alpha;
  f.beta1 = z / (1.0 + z) / s1;
  f.sth = sth;
  return f;
}

__device__ __forceinline__ double field_sqrt_h(const FieldGeom& q, double x1, double x2) {
  const FM f = field_metric(q, x1, x2);
  return f.sqh_t * f.sth;
}

// polar area with a half-cell radius: int_0^{1/2} sqrt(h) dx2
__device__ __forceinline__ double polar_area(const FieldGeom& q, double x1) {
  double r, s1, th, s2;
  field_coords(q, x1, 0.5, r, s1, th, s2);
  const double p = r * r + q.a * q.a;
  return s1 * p * sqrt(1.0 + 2.0 * q.mass * r / p) * (1.0 - cos(th));
}

template <typename T>
struct V3 {
  T* f[3];
};
template <typename T>
struct CV3 {
  const T* f[3];
};

// E_i at the D^i locations and H_i at the B^i locations (Eq. 42).  em = D1 D2 D3 B1 B2 B3; E.f / H.f may hold NULLs.
template <typename T>
__global__ void __launch_bounds__(128) k_aux_fields(const FieldGeom q, const FPtrs<T> em, const V3<T> E, const V3<T> H) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int a1 = blockIdx.y + 1;
  if (j > q.n2 || a1 >= q.rows - 1) return;
  const int64_t o = (int64_t)a1 * q.ld + (j + q.ng);
  const int64_t up = o + q.ld, dn = o - q.ld;
  const double i = (double)(a1 - q.ng), x2 = (double)j;
  const T *D1 = em.f[0], *D2 = em.f[1], *D3 = em.f[2], *B1 = em.f[3], *B2 = em.f[4], *B3 = em.f[5];
  {
    const FM c = field_metric(q, i + 0.5, x2), l = field_metric(q, i, x2), r = field_metric(q, i + 1.0, x2);
    if (E.f[0]) {
      const double avg = (l.sqh_t * l.h13 * (double)D3[o] + r.sqh_t * r.h13 * (double)D3[up]) / (2.0 * c.sqh_t);
      E.f[0][o] = (T)(c.alpha * (c.h11 * (double)D1[o] + avg));
    }
    if (H.f[1]) {
      const double avg = 0.5 * (l.sqh_t * l.sth * l.beta1 * (double)D3[o] + r.sqh_t * r.sth * r.beta1 * (double)D3[up]);
      H.f[1][o] = (T)(c.alpha * c.h22 * (double)B2[o] + avg);
    }
    if (E.f[2]) {
      const FM cl = field_metric(q, i - 0.5, x2);
      const double a13 = (cl.sqh_t * cl.h13 * (double)D1[dn] + c.sqh_t * c.h13 * (double)D1[o]) / (2.0 * l.sqh_t);
      const double ab = 0.5 * (cl.sqh_t * cl.sth * cl.beta1 * (double)B2[dn] + c.sqh_t * c.sth * c.beta1 * (double)B2[o]);
      E.f[2][o] = (T)(l.alpha * (l.h33 * (double)D3[o] + a13) + ab);
    }
  }
  if (j == q.n2) return;
  const FM c = field_metric(q, i, x2 + 0.5), cl = field_metric(q, i - 0.5, x2 + 0.5), cr = field_metric(q, i + 0.5, x2 + 0.5);
  if (E.f[1]) {
    const double ab = 0.5 * (cl.sqh_t * cl.sth * cl.beta1 * (double)B3[dn] + cr.sqh_t * cr.sth * cr.beta1 * (double)B3[o]);
    E.f[1][o] = (T)(c.alpha * c.h22 * (double)D2[o] - ab);
  }
  if (H.f[0]) {
    const double a13 = (cl.sqh_t * cl.h13 * (double)B3[dn] + cr.sqh_t * cr.h13 * (double)B3[o]) / (2.0 * c.sqh_t);
    H.f[0][o] = (T)(c.alpha * (c.h11 * (double)B1[o] + a13));
  }
  if (H.f[2]) {
    const FM r = field_metric(q, i + 1.0, x2 + 0.5);
    const double a13 = (c.sqh_t * c.h13 * (double)B1[o] + r.sqh_t * r.h13 * (double)B1[up]) / (2.0 * cr.sqh_t);
    const double ab = 0.5 * (c.sqh_t * c.sth * c.beta1 * (double)D2[o] + r.sqh_t * r.sth * r.beta1 * (double)D2[up]);
    H.f[2][o] = (T)(cr.alpha * (cr.h33 * (double)B3[o] + a13) - ab);
  }
}

// Eq. 40: B^i -= dt e^{ijk} d_j E_k / sqrt(h)
template <typename T>
__global__ void __launch_bounds__(128) k_faraday(const FieldGeom q, const V3<T> B, const CV3<T> E, double dt) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int a1 = blockIdx.y + 2;
  if (j >= q.n2 || a1 >= q.rows - 2) return;
  const int64_t o = (int64_t)a1 * q.ld + (j + q.ng);
  const double i = (double)(a1 - q.ng);
  const T *E1 = E.f[0], *E2 = E.f[1], *E3 = E.f[2];
  B.f[0][o] = (T)((double)B.f[0][o] - dt * ((double)E3[o + 1] - (double)E3[o]) / field_sqrt_h(q, i, j + 0.5));
  if (j > 0)
    B.f[1][o] = (T)((double)B.f[1][o] + dt * ((double)E3[o + q.ld] - (double)E3[o]) / field_sqrt_h(q, i + 0.5, (double)j));
  B.f[2][o] = (T)((double)B.f[2][o] - dt * (((double)E2[o + q.ld] - (double)E2[o]) - ((double)E1[o + 1] - (double)E1[o])) /
                                          field_sqrt_h(q, i + 0.5, j + 0.5));
}

// Eq. 41 and, on the axes, Eq. 45: D^i += dt (e^{ijk} d_j H_k - kJ J^i)/sqrt(h)
template <typename T>
__global__ void __launch_bounds__(128) k_ampere(const FieldGeom q, const V3<T> D, const CV3<T> H, const CV3<T> J, double kJ,
                                                double dt) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int a1 = blockIdx.y + 2;
  if (j > q.n2 || a1 >= q.rows - 2) return;
  const int64_t o = (int64_t)a1 * q.ld + (j + q.ng);
  const double i = (double)(a1 - q.ng);
  const T *H1 = H.f[0], *H2 = H.f[1], *H3 = H.f[2];
  const double j1 = J.f[0] ? (double)J.f[0][o] : 0.0;
  double d1;
  if (j == 0)
    d1 = ((double)H3[o] - 0.5 * kJ * j1) / polar_area(q, i + 0.5);
  else if (j == q.n2)
    d1 = (-(double)H3[o - 1] - 0.5 * kJ * j1) / polar_area(q, i + 0.5);
  else
    d1 = (((double)H3[o] - (double)H3[o - 1]) - kJ * j1) / field_sqrt_h(q, i + 0.5, (double)j);
  D.f[0][o] = (T)((double)D.f[0][o] + dt * d1);
  if (j == q.n2) return;
  const double j2 = J.f[1] ? (double)J.f[1][o] : 0.0;
  D.f[1][o] = (T)((double)D.f[1][o] + dt * (-((double)H3[o] - (double)H3[o - q.ld]) - kJ * j2) / field_sqrt_h(q, i, j + 0.5));
  if (j > 0) {
    const double j3 = J.f[2] ? (double)J.f[2][o] : 0.0;
    D.f[2][o] = (T)((double)D.f[2][o] + dt * ((((double)H2[o] - (double)H2[o - q.ld]) - ((double)H1[o] - (double)H1[o - 1])) - kJ * j3) /
                                            field_sqrt_h(q, i, (double)j));
  }
}

// Field boundary conditions (Sec. 3.3.3; R-F4): ghost columns beyond the polar axes by reflection
// (r- and phi-components even, theta-components odd), B^2 = D^3 = 0 on the axes, then the constant layer inside the
// horizon: rows i1 in [-ng, n_const] take the values of row n_const + 1.  One thread per (row, column); component
// c = blockIdx.z in the order D1 D2 D3 B1 B2 B3.
template <typename T>
__global__ void __launch_bounds__(128) k_field_bc_axis(const FieldGeom q, const V3<T> D, const V3<T> B, int c0) {
  // c0 = 0 with gridDim.z = 6: all six components; c0 = 3 with gridDim.z = 3: B only (D is not touched)
  const int c = blockIdx.z + c0, a1 = blockIdx.y, t = threadIdx.x + blockIdx.x * blockDim.x;
  if (t >= 2 * q.ng + 2) return;
  T* A = c < 3 ? D.f[c] : B.f[c - 3];
  const bool half = (c == 1 || c == 3 || c == 5);            // sampled at j + 1/2
  const T par = (c == 1 || c == 4) ? T(-1) : T(1);           // theta-components are odd
  T* row = A + (int64_t)a1 * q.ld;
  const int G = q.ng, n2 = q.n2;
  if (t < q.ng) {                                            // ghosts below theta = 0: m = t + 1
    const int m = t + 1;
    row[G - m] = par * row[half ? G + m - 1 : G + m];
  } else if (t < 2 * q.ng) {                                 // ghosts beyond theta = pi
    const int m = t - q.ng + 1;
    const int dst = half ? G + n2 + m - 1 : G + n2 + m;
    if (dst < q.ld) row[dst] = par * row[G + n2 - m];
  } else if (c == 2 || c == 4) {                             // D3, B2 on the axes
    row[t == 2 * q.ng ? G : G + n2] = T(0);
  }
}

template <typename T>
__global__ void __launch_bounds__(128) k_field_bc_layer(const FieldGeom q, const V3<T> D, const V3<T> B, int n_const) {
  const int c = blockIdx.z, a1 = blockIdx.y, a2 = threadIdx.x + blockIdx.x * blockDim.x;
  if (a2 >= q.ld || a1 > q.ng + n_const) return;
  T* A = c < 3 ? D.f[c] : B.f[c - 3];
  A[(int64_t)a1 * q.ld + a2] = A[(int64_t)(q.ng + n_const + 1) * q.ld + a2];
}

// Absorbing layer at the outer radial edge (profile in paper I -> reading R-F6): for r_abs < r the
// field relaxes toward the target, F <- T + s (F - T), s = tanh(4 (r_max - r) / (r_max - r_abs)), s = 0 beyond r_max,
// with r the radius of the component's own Yee location.  One thread per (row, column); blockIdx.z = component.
template <typename T>
__global__ void __launch_bounds__(128) k_field_match(const FieldGeom q, const V3<T> D, const V3<T> B, const CV3<T> D0,
                                                     const CV3<T> B0, double r_abs, double r_max, int row0) {
  const int c = blockIdx.z, a1 = row0 + blockIdx.y, a2 = threadIdx.x + blockIdx.x * blockDim.x;
  if (a2 >= q.ld || a1 >= q.rows) return;
  const bool half = (c == 0 || c == 4 || c == 5);            // D^1, B^2, B^3 sit at i + 1/2
  double r, s1, th, s2;
  field_coords(q, (double)(a1 - q.ng) + (half ? 0.5 : 0.0), 0.0, r, s1, th, s2);
  if (!(r > r_abs)) return;
  double d = (r_max - r) / (r_max - r_abs);
  if (d < 0.0) d = 0.0;
  const double s = tanh(4.0 * d);
  T* A = c < 3 ? D.f[c] : B.f[c - 3];
  const T* tg = c < 3 ? D0.f[c] : B0.f[c - 3];
  const int64_t k = (int64_t)a1 * q.ld + a2;
  const double t = (double)tg[k];
  A[k] = (T)(t + s * ((double)A[k] - t));
}

// One pass of the binomial current filter (reading R-F5): [1 2 1]/4 along x2 then along x1 on the
// component's own Yee lattice, mirror samples with the component's parity beyond the axes (J^1, J^3 even, J^2 odd),
// first and last array row unchanged along x1.  in -> out (different arrays); one thread per (row, theta sample).
template <typename T>
__global__ void __launch_bounds__(128) k_filter_current(const FieldGeom q, const CV3<T> in, const V3<T> out) {
  const int c = blockIdx.z, a1 = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
  const bool half = (c == 1);
  const int ncol = half ? q.n2 : q.n2 + 1;
  if (j >= ncol) return;
  const T par = (c == 1) ? T(-1) : T(1);
  const T* A = in.f[c];
  auto theta_pass = [&](int row) {
    const T* r = A + (int64_t)row * q.ld + q.ng;
    T lo, hi;
    if (j > 0) lo = r[j - 1]; else lo = par * (half ? r[0] : r[1]);
    if (j < ncol - 1) hi = r[j + 1]; else hi = par * (half ? r[q.n2 - 1] : r[q.n2 - 1]);
    return T(0.25) * (lo + T(2) * r[j] + hi);
  };
  const T mid = theta_pass(a1);
  T v = mid;
  if (a1 > 0 && a1 < q.rows - 1) v = T(0.25) * (theta_pass(a1 - 1) + T(2) * mid + theta_pass(a1 + 1));
  out.f[c][(int64_t)a1 * q.ld + q.ng + j] = v;
}

// out = (a + b)/2 over whole arrays (the time averages of Eq. 46 and Eq. 51)
template <typename T>
__global__ void __launch_bounds__(256) k_average(T* out, const T* a, const T* b, int64_t n) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) out[k] = T(0.5) * (a[k] + b[k]);
}

}  // namespace grpic
