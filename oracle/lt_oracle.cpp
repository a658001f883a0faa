/*
 * lt_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the deflection-angle (lensing-potential gradient) map of
 * arXiv 1902.03252 with the dPIE/PIEMD lens body named by BASELINE.json:north_star.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code
 * (headers, helpers, constants) with paper_1902_03252_b200/csrc; it defines its own POD lens struct.
 *
 * What it follows (P:n = /root/reference/PAPER.md line n):
 *   skeleton  : Algorithm 1, P:191-226 (section 2.3): for every pixel, for every lens: translate (l.3-4),
 *               rotate by Phi (l.5-6), evaluate the body (l.7-9), rotate back by -Phi (l.10-11), sum (l.13-14,
 *               eq. 15).
 *   body      : NOT in the paper (dPIE is only named at P:385).  BASELINE.json:north_star: "evaluates the
 *               complex-ratio-plus-complex-log PIEMD deflection at the core radius and at the cut radius, takes
 *               their difference scaled by b0*rcut/(rcut-rcore)".  Written out (SURVEY 8(c) "Form C"), in the lens
 *               frame (x, y), for a radius w, with rho^2 = x^2/(1+e)^2 + y^2/(1-e)^2 and q = (1-e)/(1+e):
 *                 I_w = (1-e^2)/(2 i sqrt(e)) * ln[ (q x - i y/q + 2 i sqrt(e) sqrt(w^2+rho^2)) / (x - i y + 2 i w sqrt(e)) ]
 *                 alpha_w = b0 * (Re I_w, Im I_w)
 *                 g = rcut/(rcut-rcore) * (alpha_rcore - alpha_rcut)
 *               whose convergence is kappa = (b0/2) rcut/(rcut-rcore) [1/sqrt(rcore^2+rho^2) - 1/sqrt(rcut^2+rho^2)]
 *               (alpha = grad psi, laplace psi = 2 kappa: eq. 2-4).
 *   circular  : e < 1e-14: north star's closed form
 *               alpha(R) = b0 rcut/(rcut-rcore) [(sqrt(rcore^2+R^2)-rcore) - (sqrt(rcut^2+R^2)-rcut)] / R, along (x,y)/R,
 *               each bracket evaluated as R^2/(sqrt(w^2+R^2)+w) (reading R22: identical value, no cancellation).
 *   mixed rule: section 3.3, eq. 24-28 and the DP centre patches of section 3.2, with the
 *               readings R11-R16 of DESIGN.md (thresholds scaled with the pixel size).
 *
 * One evaluation-point choice is made (reading R21): Form C's numerator and denominator vanish together at
 * the lens-frame point (0, +2 w sqrt(e)) (a removable 0/0).  The dPIE deflection is mirror symmetric about the lens's
 * major axis (alpha_x even, alpha_y odd in y), so the oracle evaluates Form C at (x, -|y|), where both complex numbers
 * lie in the closed upper half plane away from zero, and restores the sign of alpha_y.  tests/test_oracle_pins.py pins
 * that symmetry against the unreflected evaluation, the independent quadrature (oracle/form_q.py) and the
 * __float128 instantiation (which does NOT reflect).
 *
 * Precision: the reference values are the `long double` (x87 80-bit) instantiation, sums rounded to fp64 at the end
 * (reading R7); `double` is the timed CPU baseline; `float` is the paper's "identical up to the change in precision"
 * SP version, used for context only; __float128 audits small samples.
 * Known limit: for 1e-14 <= e < 1e-10 the long-double Form C loses ~eps_ld/sqrt(e) relative accuracy (<= 1e-12);
 * no config goes below e = 1e-6.  For e >= 0.9 and rcut/rcore -> 1 (outside every config) the pin is the __float128
 * instantiation against the density quadrature (tests/test_oracle_pins.py::test_form_q_beyond_the_configs); the long
 * double one loses rcut/(rcut - rcore) times its rounding there.
 */
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#include <quadmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
struct lto_lens {            /* same field order as the [n,7] fp64 array the generators produce */
  double x, y;               /* theta_center (Alg. 1 Require)                             */
  double ellipticity;        /* e, enters rho^2 = x^2/(1+e)^2 + y^2/(1-e)^2 (reading R1)         */
  double angle;              /* Phi, CCW from the theta_1 axis to the major axis, rad    */
  double rcore, rcut, b0;
};
struct lto_mixed_params {    /* readings R11, R14, R15 */
  double m_max;              /* 3.26                              */
  double c28;                /* 0.0104/0.03 (eq. 28 P:321 over Delta x)   */
  double patch_halfwidth_cluster, patch_halfwidth_galaxy;   /* arcsec: 6.0, 0.3 (400/2, 20/2 px at 0.03") */
  double b0_cluster_threshold;                              /* 15 arcsec */
};
}

namespace {

/* ---- thin math shims so that one template serves float / double / long double / __float128 ---- */
template <class T> struct M {
  static T sqrt_(T v) { return std::sqrt(v); }
  static T log_(T v) { return std::log(v); }
  static T atan2_(T a, T b) { return std::atan2(a, b); }
  static T sin_(T v) { return std::sin(v); }
  static T cos_(T v) { return std::cos(v); }
  static T abs_(T v) { return std::fabs(v); }
};
template <> struct M<__float128> {
  typedef __float128 T;
  static T sqrt_(T v) { return sqrtq(v); }
  static T log_(T v) { return logq(v); }
  static T atan2_(T a, T b) { return atan2q(a, b); }
  static T sin_(T v) { return sinq(v); }
  static T cos_(T v) { return cosq(v); }
  static T abs_(T v) { return fabsq(v); }
};

/* complex number without std::complex so that __float128 works too: only what Form C needs. */
template <class T> struct Cx { T re, im; };
template <class T> Cx<T> cdiv(Cx<T> a, Cx<T> b) {          /* textbook a/b = a conj(b) / |b|^2 */
  T d = b.re * b.re + b.im * b.im;
  return Cx<T>{(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d};
}
template <class T> Cx<T> clog(Cx<T> z) {                   /* principal log: ln|z| + i arg z */
  return Cx<T>{M<T>::log_(M<T>::sqrt_(z.re * z.re + z.im * z.im)), M<T>::atan2_(z.im, z.re)};
}

/* PIEMD deflection I_w * b0 at radius w, lens frame, Form C.  reflect: evaluate at (x, -|y|) (reading R21). */
template <class T>
void piemd_form_c(T x, T y, T e, T w, T b0, bool reflect, T& ax, T& ay) {
  T sgn = T(1);
  if (reflect && y > T(0)) { y = -y; sgn = T(-1); }
  const T sqe = M<T>::sqrt_(e);
  const T q = (T(1) - e) / (T(1) + e);
  const T rho2 = x * x / ((T(1) + e) * (T(1) + e)) + y * y / ((T(1) - e) * (T(1) - e));
  const T r = M<T>::sqrt_(w * w + rho2);
  Cx<T> num{q * x, -y / q + T(2) * sqe * r};
  Cx<T> den{x, -y + T(2) * w * sqe};
  Cx<T> L = clog(cdiv(num, den));
  /* (1/i) (a + i b) = b - i a */
  const T K = b0 * (T(1) - e * e) / (T(2) * sqe);
  ax = K * L.im;
  ay = sgn * (-K * L.re);
}

/* one lens, lens frame: dPIE body g (north star). */
template <class T>
void dpie_body(T x, T y, T e, T rcore, T rcut, T b0, bool reflect, T& gx, T& gy) {
  const T scale = rcut / (rcut - rcore);
  if (e < T(1e-14)) {                                     /* circular closed form (north star) */
    const T R2 = x * x + y * y;
    const T R = M<T>::sqrt_(R2);
    if (R == T(0)) { gx = T(0); gy = T(0); return; }      /* reading R5 */
    /* sqrt(w^2+R^2) - w written as R^2 / (sqrt(w^2+R^2) + w): the same number without the cancellation that costs the
     * literal form ulp(w)/R at R << w (reading R22; pinned against the literal form in __float128) */
    const T hc = R2 / (M<T>::sqrt_(rcore * rcore + R2) + rcore), ht = R2 / (M<T>::sqrt_(rcut * rcut + R2) + rcut);
    const T a = b0 * scale * (hc - ht) / R;
    gx = a * x / R; gy = a * y / R;
    return;
  }
  T acx, acy, atx, aty;
  piemd_form_c<T>(x, y, e, rcore, b0, reflect, acx, acy);
  piemd_form_c<T>(x, y, e, rcut, b0, reflect, atx, aty);
  gx = scale * (acx - atx);
  gy = scale * (acy - aty);
}

/* Algorithm 1 for one pixel; sums in T, in lens index order (reading R8). */
template <class T>
void gradient_pixel(const lto_lens* L, int n, T t1, T t2, bool reflect, T& G1, T& G2) {
  G1 = T(0); G2 = T(0);
  for (int k = 0; k < n; ++k) {
    const T d1 = t1 - T(L[k].x);                          /* l.3 */
    const T d2 = t2 - T(L[k].y);                          /* l.4 */
    const T c = M<T>::cos_(T(L[k].angle)), s = M<T>::sin_(T(L[k].angle));
    const T xp = d1 * c + d2 * s;                         /* l.5 */
    const T yp = d2 * c - d1 * s;                         /* l.6 */
    T gx, gy;
    dpie_body<T>(xp, yp, T(L[k].ellipticity), T(L[k].rcore), T(L[k].rcut), T(L[k].b0), reflect, gx, gy); /* l.7-9 */
    G1 += gx * c - gy * s;                                /* l.10 (cos(-Phi), sin(-Phi)) */
    G2 += gy * c + gx * s;                                /* l.11 */
  }                                                       /* l.13-14 */
}

template <class T>
void grid_impl(const lto_lens* L, int n, double x_min, double y_min, double dx, int nx, int ny, double* out,
               int n_threads, int row_stride) {
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic)
  for (int j = 0; j < ny; j += row_stride) {
    for (int i = 0; i < nx; ++i) {
      /* pixel position in fp64 exactly as the API defines it (x_min + i*dx), then widened/narrowed to T */
      const double t1 = x_min + i * dx, t2 = y_min + j * dx;
      T G1, G2;
      gradient_pixel<T>(L, n, T(t1), T(t2), true, G1, G2);
      out[2 * ((size_t)j * nx + i) + 0] = (double)G1;
      out[2 * ((size_t)j * nx + i) + 1] = (double)G2;
    }
  }
}

template <class T>
void points_impl(const lto_lens* L, int n, const double* px, const double* py, long long npts, double* out,
                 int n_threads, bool reflect) {
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 64)
  for (long long p = 0; p < npts; ++p) {
    T G1, G2;
    gradient_pixel<T>(L, n, T(px[p]), T(py[p]), reflect, G1, G2);
    out[2 * p + 0] = (double)G1;
    out[2 * p + 1] = (double)G2;
  }
}

}  // namespace

extern "C" {

/* precision: 0 = long double (reference), 1 = double (timed CPU baseline), 2 = float (paper's SP twin), 3 = __float128.
 * row_stride > 1 computes only rows 0, stride, 2*stride, ... (others untouched) -- the bench's bounded sample.
 * Returns 0, or -1 on a bad argument. */
int lt_oracle_gradient_grid(const lto_lens* lenses, int n_lens, double x_min, double y_min, double dx, int nx, int ny,
                            int precision, double* out, int n_threads, int row_stride) {
  if ((n_lens > 0 && !lenses) || n_lens < 0 || nx < 1 || ny < 1 || !out || row_stride < 1) return -1;
  switch (precision) {
    case 0: grid_impl<long double>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
    case 1: grid_impl<double>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
    case 2: grid_impl<float>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
    case 3: grid_impl<__float128>(lenses, n_lens, x_min, y_min, dx, nx, ny, out, n_threads, row_stride); return 0;
  }
  return -1;
}

/* same at arbitrary points (px[p], py[p]); reflect = 0 switches the reading-R21 mirror evaluation off. */
int lt_oracle_gradient_points(const lto_lens* lenses, int n_lens, const double* px, const double* py, long long npts,
                              int precision, int reflect, double* out, int n_threads) {
  if ((n_lens > 0 && !lenses) || n_lens < 0 || npts < 0 || !out || (npts > 0 && (!px || !py))) return -1;
  switch (precision) {
    case 0: points_impl<long double>(lenses, n_lens, px, py, npts, out, n_threads, reflect != 0); return 0;
    case 1: points_impl<double>(lenses, n_lens, px, py, npts, out, n_threads, reflect != 0); return 0;
    case 2: points_impl<float>(lenses, n_lens, px, py, npts, out, n_threads, reflect != 0); return 0;
    case 3: points_impl<__float128>(lenses, n_lens, px, py, npts, out, n_threads, reflect != 0); return 0;
  }
  return -1;
}

/* convergence kappa of the dPIE sum at points (elementary expression in the header; for the div(alpha) = 2 kappa pin). */
int lt_oracle_kappa_points(const lto_lens* L, int n, const double* px, const double* py, long long npts, double* out) {
  for (long long p = 0; p < npts; ++p) {
    long double k = 0;
    for (int i = 0; i < n; ++i) {
      const long double e = L[i].ellipticity, c = cosl(L[i].angle), s = sinl(L[i].angle);
      const long double d1 = px[p] - L[i].x, d2 = py[p] - L[i].y;
      const long double x = d1 * c + d2 * s, y = d2 * c - d1 * s;
      const long double rho2 = x * x / ((1 + e) * (1 + e)) + y * y / ((1 - e) * (1 - e));
      const long double rc = L[i].rcore, rt = L[i].rcut;
      k += 0.5L * L[i].b0 * rt / (rt - rc) * (1 / sqrtl(rc * rc + rho2) - 1 / sqrtl(rt * rt + rho2));
    }
    out[p] = (double)k;
  }
  return 0;
}

/*
 * Mixed-precision rule (section 3.2-3.3) applied to a given single-precision map `sp` (nx*ny*2 floats).
 * flags[j*nx+i]: bit0 = inside a DP centre patch (R14/R15), bit1 = eq. 25 on delta_1 or delta_2,
 * bit2 = eq. 28 on delta_3 or delta_4.  delta_i per eq. 24 / 27 with the left / lower
 * neighbour, the forward neighbour at i = 0 / j = 0 (R12); the criterion along an axis of extent 1 is skipped.
 * All criterion arithmetic in fp32 (the map's precision; both sides take the decision in the same precision),
 * thresholds dx/m_max and c28*dx rounded to fp32 once.  crit (may be null) receives, per pixel, the four values
 * |dx-delta_1|, |dx-delta_2|, |delta_3|, |delta_4| (fp32) so that a test can exclude near-threshold pixels (R18).
 */
int lt_oracle_mixed_flags(const float* sp, int nx, int ny, double x_min, double y_min, double dx,
                          const lto_lens* L, int n, const lto_mixed_params* mp, uint8_t* flags, float* crit) {
  if (!sp || !flags || !mp || nx < 1 || ny < 1) return -1;
  const float fdx = (float)dx, t25 = (float)(dx / mp->m_max), t28 = (float)(mp->c28 * dx);
  std::memset(flags, 0, (size_t)nx * ny);
  for (int k = 0; k < n; ++k) {                          /* patches: box centred on the pixel nearest the centre */
    const double h = (L[k].b0 >= mp->b0_cluster_threshold) ? mp->patch_halfwidth_cluster : mp->patch_halfwidth_galaxy;
    long long hp = (long long)std::ceil(h / dx); if (hp < 1) hp = 1;
    const long long ic = std::llround((L[k].x - x_min) / dx), jc = std::llround((L[k].y - y_min) / dx);
    const long long i0 = std::max<long long>(ic - hp, 0), i1 = std::min<long long>(ic + hp, nx - 1);
    const long long j0 = std::max<long long>(jc - hp, 0), j1 = std::min<long long>(jc + hp, ny - 1);
    for (long long j = j0; j <= j1; ++j) for (long long i = i0; i <= i1; ++i) flags[j * nx + i] |= 1;
  }
  for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    const size_t p = (size_t)j * nx + i;
    const float a1 = sp[2 * p], a2 = sp[2 * p + 1];
    float c[4] = {INFINITY, INFINITY, 0.f, 0.f};         /* values that never fire */
    if (nx > 1) {                                        /* x-neighbour: delta_1 (comp 1), delta_4 (comp 2) */
      float d1, d4;
      if (i > 0) { d1 = a1 - sp[2 * (p - 1)]; d4 = a2 - sp[2 * (p - 1) + 1]; }
      else       { d1 = sp[2 * (p + 1)] - a1; d4 = sp[2 * (p + 1) + 1] - a2; }
      c[0] = std::fabs(fdx - d1); c[3] = std::fabs(d4);
    }
    if (ny > 1) {                                        /* y-neighbour: delta_2 (comp 2), delta_3 (comp 1) */
      float d2, d3;
      if (j > 0) { d2 = a2 - sp[2 * (p - nx) + 1]; d3 = a1 - sp[2 * (p - nx)]; }
      else       { d2 = sp[2 * (p + nx) + 1] - a2; d3 = sp[2 * (p + nx)] - a1; }
      c[1] = std::fabs(fdx - d2); c[2] = std::fabs(d3);
    }
    if (c[0] < t25 || c[1] < t25) flags[p] |= 2;
    if (c[2] > t28 || c[3] > t28) flags[p] |= 4;
    if (crit) { crit[4 * p] = c[0]; crit[4 * p + 1] = c[1]; crit[4 * p + 2] = c[2]; crit[4 * p + 3] = c[3]; }
  }
  return 0;
}

int lt_oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
