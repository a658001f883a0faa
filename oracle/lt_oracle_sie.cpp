/*
 * lt_oracle_sie.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow CPU oracle for the paper's own lens body: Algorithm 1 "Compute grad Psi_eps in each image pixel for a SIE"
 * (arXiv 1902.03252, section 2.3), written out line by line in the paper's order and notation.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code with
 * paper_1902_03252_b200/csrc (own POD struct, own arithmetic).
 *
 * What it follows (P:n = /root/reference/PAPER.md line n):
 *   l.3-4   Delta theta = theta - theta_center
 *   l.5-6   rotate by Phi: x' = D1 cos Phi + D2 sin Phi, y' = D2 cos Phi - D1 sin Phi       (garbled subscripts
 *           read as the primed quantities, reading R3)
 *   l.7     R = sqrt(x'^2 (1 - eps) + y'^2 (1 + eps))                                      (eq. 16-18)
 *   l.8-9   g1 = (1 - eps) b0 x' / R,  g2 = (1 + eps) b0 y' / R                            (eq. 21)
 *   l.10-11 rotate by -Phi: G1 = g1 cos(-Phi) + g2 sin(-Phi), G2 = g2 cos(-Phi) - g1 sin(-Phi)
 *   l.13-14 sum over lenses                                                                (eq. 15)
 *   R = 0 (pixel exactly on a lens centre; the SIS deflection has no direction there): that lens
 *   contributes 0 (reading R5).
 * The potential whose gradient this is: Psi_eps = b0 R (eq. 9-10 P:86-90 with eq. 19): exported for the
 * finite-difference pin alpha = grad psi (eq. 2).
 *
 * Precision: `long double` = reference values (sums rounded to fp64 at the end); `double` = timed CPU baseline (the
 * paper's DP version); `float` = the paper's SP version, "identical up to the change in precision".
 */
#include <cmath>
#include <cstddef>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
struct lto_sie_lens {        /* same field order as the [n,5] fp64 array the generators produce */
  double x, y;               /* theta_center (Alg. 1 Require) */
  double epsilon;            /* pseudo-ellipticity of the potential, eq. 17-18 */
  double angle;              /* Phi, CCW from the theta_1 axis to the semi-major axis, radians */
  double b0;                 /* eq. 22, arcsec */
};
}

namespace {

template <class T>
void sie_pixel(const lto_sie_lens* L, int n, T t1, T t2, T& G1, T& G2) {
  G1 = T(0); G2 = T(0);
  for (int i = 0; i < n; ++i) {
    const T d1 = t1 - T(L[i].x);                                     /* l.3 */
    const T d2 = t2 - T(L[i].y);                                     /* l.4 */
    const T c = std::cos(T(L[i].angle)), s = std::sin(T(L[i].angle));
    const T x = d1 * c + d2 * s;                                     /* l.5 */
    const T y = d2 * c - d1 * s;                                     /* l.6 */
    const T e = T(L[i].epsilon), b0 = T(L[i].b0);
    const T R = std::sqrt(x * x * (T(1) - e) + y * y * (T(1) + e));  /* l.7 */
    if (R == T(0)) continue;                                         /* reading R5 */
    const T g1 = (T(1) - e) * b0 * x / R;                            /* l.8 */
    const T g2 = (T(1) + e) * b0 * y / R;                            /* l.9 */
    const T cm = c, sm = -s;                                         /* cos(-Phi), sin(-Phi) */
    G1 += g1 * cm + g2 * sm;                                         /* l.10 */
    G2 += g2 * cm - g1 * sm;                                         /* l.11 */
  }                                                                  /* l.13-14 */
}

template <class T>
void grid_impl(const lto_sie_lens* L, int n, double x_min, double y_min, double dx, int nx, int ny, double* out,
               int n_threads, int row_stride) {
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic)
  for (int j = 0; j < ny; j += row_stride)
    for (int i = 0; i < nx; ++i) {
      const double t1 = x_min + i * dx, t2 = y_min + j * dx;         /* pixel position in fp64, as the API defines it */
      T G1, G2;
      sie_pixel<T>(L, n, T(t1), T(t2), G1, G2);
      out[2 * ((size_t)j * nx + i) + 0] = (double)G1;
      out[2 * ((size_t)j * nx + i) + 1] = (double)G2;
    }
}

template <class T>
void points_impl(const lto_sie_lens* L, int n, const double* px, const double* py, long long npts, double* out,
                 int n_threads) {
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 64)
  for (long long p = 0; p < npts; ++p) {
    T G1, G2;
    sie_pixel<T>(L, n, T(px[p]), T(py[p]), G1, G2);
    out[2 * p + 0] = (double)G1;
    out[2 * p + 1] = (double)G2;
  }
}

}  // namespace

extern "C" {

/* precision: 0 = long double (reference), 1 = double (timed CPU baseline), 2 = float (the paper's SP version).
 * row_stride > 1 computes rows 0, stride, 2*stride, ... only.  Returns 0, or -1 on a bad argument. */
int lt_oracle_sie_gradient_grid(const lto_sie_lens* lenses, int n_lens, double x_min, double y_min, double dx, int nx,
                                int ny, int precision, double* out, int n_threads, int row_stride) {
  if ((n_lens > 0 && !lenses) || n_lens < 0 || nx < 1 || ny < 1 || !out || row_stride < 1) return -1;
  switch (precision) {
    case 0: grid_impl<long double>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
    case 1: grid_impl<double>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
    case 2: grid_impl<float>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
  }
  return -1;
}

int lt_oracle_sie_gradient_points(const lto_sie_lens* lenses, int n_lens, const double* px, const double* py,
                                  long long npts, int precision, double* out, int n_threads) {
  if ((n_lens > 0 && !lenses) || n_lens < 0 || npts < 0 || !out || (npts > 0 && (!px || !py))) return -1;
  switch (precision) {
    case 0: points_impl<long double>(lenses, n_lens, px, py, npts, out, n_threads); return 0;
    case 1: points_impl<double>(lenses, n_lens, px, py, npts, out, n_threads); return 0;
    case 2: points_impl<float>(lenses, n_lens, px, py, npts, out, n_threads); return 0;
  }
  return -1;
}

/* Psi_eps = sum_i b0_i R_i at points (long double), for the pin alpha = grad psi by finite differences. */
int lt_oracle_sie_potential_points(const lto_sie_lens* L, int n, const double* px, const double* py, long long npts,
                                   double* out) {
  for (long long p = 0; p < npts; ++p) {
    long double psi = 0;
    for (int i = 0; i < n; ++i) {
      const long double c = cosl(L[i].angle), s = sinl(L[i].angle), e = L[i].epsilon;
      const long double d1 = (long double)px[p] - L[i].x, d2 = (long double)py[p] - L[i].y;
      const long double x = d1 * c + d2 * s, y = d2 * c - d1 * s;
      psi += L[i].b0 * sqrtl(x * x * (1 - e) + y * y * (1 + e));
    }
    out[p] = (double)psi;
  }
  return 0;
}

}  // extern "C"
