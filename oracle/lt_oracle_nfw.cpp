/*
 * lt_oracle_nfw.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow CPU oracle for the deflection map of pseudo-elliptical NFW lenses: the generalisation the paper names at
 * P:385 ("other commonly used parametric lens models like the Navarro-Frenk-White (NFW) profile"; references P:456,
 * P:475-476), SURVEY 8(f) NEXT-4.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it; it shares no code with
 * paper_1902_03252_b200/csrc.
 *
 * What it follows (P:n = /root/reference/PAPER.md line n):
 *   skeleton         : Algorithm 1: translate (l.3-4), rotate by Phi (l.5-6), body, rotate back by -Phi
 *                      (l.10-11), sum (l.13-14).
 *   pseudo-elliptical: the paper's general recipe for any circular deflection |alpha(R)| (eq. 16-20, after
 *                      Golse & Kneib 2002): R = sqrt(a1 x'^2 + a2 y'^2), a1 = 1 - eps, a2 = 1 + eps,
 *                      cos(phi) = sqrt(a1) x'/R, sin(phi) = sqrt(a2) y'/R,
 *                      alpha_1 = |alpha(R)| sqrt(a1) cos(phi), alpha_2 = |alpha(R)| sqrt(a2) sin(phi).
 *                      (For |alpha| = b0 this is Algorithm 1 l.7-9, eq. 21.)
 *   circular body    : NOT in the paper.  Textbook NFW lens (the profile of P:475-476 projected along the line of sight):
 *                      with x = R / rs,
 *                        alpha(x) = 4 kappa_s rs [ ln(x/2) + F(x) ] / x,
 *                        F(x) = arccosh(1/x) / sqrt(1 - x^2)  (x < 1),  1 (x = 1),  arccos(1/x) / sqrt(x^2 - 1)  (x > 1),
 *                      convergence kappa(x) = 2 kappa_s (1 - F(x)) / (x^2 - 1) (kappa(1) = 2 kappa_s / 3), potential
 *                      psi(x) = 2 kappa_s rs^2 [ ln^2(x/2) - arccosh^2(1/x) ] (x < 1), [ ln^2(x/2) + arccos^2(1/x) ] (x > 1)
 *                      (reading R26).  R = 0 contributes 0 (alpha -> 0 like x ln x).
 * Written literally except for F near x = 1 (see nfw_F).  The bracket ln(x/2) + F(x) cancels to O(x^2 ln x) for x << 1: in long double the deflection keeps
 * ~1e-19 * 8 / x absolute accuracy relative to 4 kappa_s rs, i.e. better than 1e-13 of the lens's peak deflection for
 * x > 1e-5; the __float128 instantiation audits that.
 */
#include <cmath>
#include <cstddef>
#include <quadmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
struct lto_nfw_lens {        /* same field order as the [n,6] fp64 array the generators produce */
  double x, y;               /* theta_center */
  double epsilon;            /* pseudo-ellipticity of the potential, eq. 17-18 */
  double angle;              /* Phi, CCW from the theta_1 axis to the semi-major axis, radians */
  double kappa_s;            /* characteristic convergence rho_s rs / Sigma_crit */
  double rs;                 /* scale radius, arcsec */
};
}

namespace {

template <class T> struct M {
  static T sqrt_(T v) { return std::sqrt(v); }
  static T log_(T v) { return std::log(v); }
  static T acosh_(T v) { return std::acosh(v); }
  static T atanh_(T v) { return std::atanh(v); }
  static T atan_(T v) { return std::atan(v); }
  static T sin_(T v) { return std::sin(v); }
  static T cos_(T v) { return std::cos(v); }
};
template <> struct M<__float128> {
  typedef __float128 T;
  static T sqrt_(T v) { return sqrtq(v); }
  static T log_(T v) { return logq(v); }
  static T acosh_(T v) { return acoshq(v); }
  static T atanh_(T v) { return atanhq(v); }
  static T atan_(T v) { return atanq(v); }
  static T sin_(T v) { return sinq(v); }
  static T cos_(T v) { return cosq(v); }
};

/* F(x).  For x >= 1/2, arccosh(1/x) and arccos(1/x) are evaluated through the identities arccosh(1/x) = atanh(sqrt(1 - x^2)) and
 * arccos(1/x) = atan(sqrt(x^2 - 1)) (x > 0): the same numbers, but the literal route through 1/x loses eps/|1 - x| near
 * the scale radius (1.5e-13 of the peak deflection at |1 - x| ~ 1e-7 even in long double), while F itself is smooth
 * there (F = 1 - 2(x-1)/3 + ...).  DESIGN.md reading R27; pinned against the literal formula in 40-digit arithmetic. */
template <class T> T nfw_F(T x) {
  if (x < T(0.5)) return M<T>::acosh_(T(1) / x) / M<T>::sqrt_(T(1) - x * x);      /* literal: well conditioned here */
  if (x < T(1)) { const T s = M<T>::sqrt_((T(1) - x) * (T(1) + x)); return M<T>::atanh_(s) / s; }
  if (x > T(1)) { const T s = M<T>::sqrt_((x - T(1)) * (x + T(1))); return M<T>::atan_(s) / s; }
  return T(1);
}
/* |alpha(R)| of the circular NFW lens */
template <class T> T nfw_alpha(T R, T kappa_s, T rs) {
  const T x = R / rs;
  return T(4) * kappa_s * rs * (M<T>::log_(x / T(2)) + nfw_F<T>(x)) / x;
}

template <class T>
void nfw_pixel(const lto_nfw_lens* L, int n, T t1, T t2, T& G1, T& G2) {
  G1 = T(0); G2 = T(0);
  for (int i = 0; i < n; ++i) {
    const T d1 = t1 - T(L[i].x);                                     /* Alg. 1 l.3 */
    const T d2 = t2 - T(L[i].y);                                     /* l.4 */
    const T c = M<T>::cos_(T(L[i].angle)), s = M<T>::sin_(T(L[i].angle));
    const T x = d1 * c + d2 * s;                                     /* l.5 */
    const T y = d2 * c - d1 * s;                                     /* l.6 */
    const T a1 = T(1) - T(L[i].epsilon), a2 = T(1) + T(L[i].epsilon);
    const T R = M<T>::sqrt_(a1 * x * x + a2 * y * y);                /* eq. 16-18 */
    if (R == T(0)) continue;
    const T a = nfw_alpha<T>(R, T(L[i].kappa_s), T(L[i].rs));
    const T cphi = M<T>::sqrt_(a1) * x / R, sphi = M<T>::sqrt_(a2) * y / R;
    const T g1 = a * M<T>::sqrt_(a1) * cphi;                         /* eq. 20 */
    const T g2 = a * M<T>::sqrt_(a2) * sphi;
    G1 += g1 * c - g2 * s;                                           /* l.10 */
    G2 += g2 * c + g1 * s;                                           /* l.11 */
  }
}

template <class T>
void points_impl(const lto_nfw_lens* L, int n, const double* px, const double* py, long long npts, double* out,
                 int n_threads) {
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 64)
  for (long long p = 0; p < npts; ++p) {
    T G1, G2;
    nfw_pixel<T>(L, n, T(px[p]), T(py[p]), G1, G2);
    out[2 * p + 0] = (double)G1;
    out[2 * p + 1] = (double)G2;
  }
}

template <class T>
void grid_impl(const lto_nfw_lens* L, int n, double x_min, double y_min, double dx, int nx, int ny, double* out,
               int n_threads, int row_stride) {
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic)
  for (int j = 0; j < ny; j += row_stride)
    for (int i = 0; i < nx; ++i) {
      const double t1 = x_min + i * dx, t2 = y_min + j * dx;
      T G1, G2;
      nfw_pixel<T>(L, n, T(t1), T(t2), G1, G2);
      out[2 * ((size_t)j * nx + i) + 0] = (double)G1;
      out[2 * ((size_t)j * nx + i) + 1] = (double)G2;
    }
}

}  // namespace

extern "C" {

/* precision: 0 = long double (reference), 1 = double, 3 = __float128 (audit).  row_stride > 1 computes rows 0, stride,
 * 2*stride, ... only.  Returns 0, or -1 on a bad argument. */
int lt_oracle_nfw_gradient_grid(const lto_nfw_lens* lenses, int n_lens, double x_min, double y_min, double dx, int nx,
                                int ny, int precision, double* out, int n_threads, int row_stride) {
  if ((n_lens > 0 && !lenses) || n_lens < 0 || nx < 1 || ny < 1 || !out || row_stride < 1) return -1;
  switch (precision) {
    case 0: grid_impl<long double>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
    case 1: grid_impl<double>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
    case 3: grid_impl<__float128>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
  }
  return -1;
}

int lt_oracle_nfw_gradient_points(const lto_nfw_lens* lenses, int n_lens, const double* px, const double* py,
                                  long long npts, int precision, double* out, int n_threads) {
  if ((n_lens > 0 && !lenses) || n_lens < 0 || npts < 0 || !out || (npts > 0 && (!px || !py))) return -1;
  switch (precision) {
    case 0: points_impl<long double>(lenses, n_lens, px, py, npts, out, n_threads); return 0;
    case 1: points_impl<double>(lenses, n_lens, px, py, npts, out, n_threads); return 0;
    case 3: points_impl<__float128>(lenses, n_lens, px, py, npts, out, n_threads); return 0;
  }
  return -1;
}

/* potential sum_i psi_i at points (long double), for the pin alpha = grad psi by finite differences */
int lt_oracle_nfw_potential_points(const lto_nfw_lens* L, int n, const double* px, const double* py, long long npts,
                                   double* out) {
  for (long long p = 0; p < npts; ++p) {
    long double psi = 0;
    for (int i = 0; i < n; ++i) {
      const long double c = cosl(L[i].angle), s = sinl(L[i].angle), e = L[i].epsilon;
      const long double d1 = (long double)px[p] - L[i].x, d2 = (long double)py[p] - L[i].y;
      const long double x = d1 * c + d2 * s, y = d2 * c - d1 * s;
      const long double R = sqrtl((1 - e) * x * x + (1 + e) * y * y), X = R / L[i].rs;
      const long double lg = logl(X / 2);
      long double t = 0;
      if (X < 1) { const long double a = acoshl(1 / X); t = lg * lg - a * a; }
      else if (X > 1) { const long double a = acosl(1 / X); t = lg * lg + a * a; }
      else t = lg * lg;
      psi += 2 * L[i].kappa_s * L[i].rs * L[i].rs * t;
    }
    out[p] = (double)psi;
  }
  return 0;
}

/* convergence of ONE circular NFW lens at radius R (for the quadrature pin) */
double lt_oracle_nfw_kappa(double R, double kappa_s, double rs) {
  const long double x = (long double)R / rs;
  if (x == 1) return (double)(2 * (long double)kappa_s / 3);
  return (double)(2 * (long double)kappa_s * (1 - nfw_F<long double>(x)) / (x * x - 1));
}

}  // extern "C"
