// lt_pack.cuh -- per-lens precompute: raw (xc, yc, e, Phi, rcore, rcut, b0) -> the packed
// constants of lt_math.cuh's LtLens<T> record.  All derivations in fp64; the fp32 record is the fp64 one rounded once.
// P:228 / Fig. 2-3: homogeneous per-parameter data so that every lane reads the same constants;
// cos/sin of Phi are used four times per interaction in Alg. 1 l.5-6, 10-11 and are taken once here.
// Host-compilable like lt_math.cuh.
#pragma once
#include "lt_math.cuh"

struct LtRawLens {  // = lt_lens of include/lt_gradient.h (kept separate so this header needs no C-ABI include)
  double x, y, e, phi, rcore, rcut, b0;
};

// Domain check of the API (include/lt_gradient.h): e in [0,1), 0 < rcore < rcut, everything finite.
LT_HD bool lt_lens_valid(const LtRawLens& r) {
  const bool fin = isfinite(r.x) && isfinite(r.y) && isfinite(r.e) && isfinite(r.phi) && isfinite(r.rcore) &&
                   isfinite(r.rcut) && isfinite(r.b0);
  return fin && r.e >= 0.0 && r.e < 1.0 && r.rcore > 0.0 && r.rcut > r.rcore;
}

// fp64 record.  x0, y0 = lens centre.  (Folding the translation of Alg. 1 l.3-4 into the rotation, X = cx t1 + sx t2 - X0
// with X0 = cx xc + sx yc formed once per lens, saves 1.25 FP64 instructions per interaction and 0.8 % of the fp64 time,
// but X0 carries a rounding of 1e-16 |theta_c|: next to a steep centre -- rcore = 1e-4", central slope b0 / (2 rcore) =
// 5e4 -- that alone is 1.5e-11 of max|alpha| (tests/test_gpu_parity.py: test_fp64_kernel_beyond_the_configs).  Measured,
// not kept: the difference theta - theta_center is formed first, exactly as Alg. 1 states it.)
LT_HD void lt_pack_lens(const LtRawLens& r, LtLens<double>& L) {
  double s, c;
  sincos(r.phi, &s, &c);
  const double e = r.e;
  const double ope = 1.0 + e, ome = 1.0 - e;
  const double q = ome / ope;
  const double q2 = q * q;
  double f = 2.0 * sqrt(e) / ope;            // sqrt(1 - q^2)
  f = f < LT_F_MIN ? LT_F_MIN : f;           // e = 0 stays a regular point (header of lt_math.cuh)
  const double sc = r.rcore * ope, st = r.rcut * ope;
  const double rf = 1.0 / f, qf = q * rf;
  L.cx = qf * c;
  L.sx = qf * s;
  L.cy = rf * c;
  L.sy = rf * s;
  L.x0 = r.x;
  L.y0 = r.y;
  L.Kc = (ome * r.rcore * rf) * (ome * r.rcore * rf);  // q^2 s_c^2 / f^2
  L.dK = (ome * rf) * (ome * rf) * ((r.rcut - r.rcore) * (r.rcut + r.rcore));   // K_t - K_c without cancellation
  L.sc = sc * rf;
  L.st = st * rf;
  L.q2sc = q2 * sc * rf;
  L.q2st = q2 * st * rf;
  L.g = f / q;
  L.f = f;
  const double C = r.b0 * (r.rcut / (r.rcut - r.rcore)) * ome * rf;
  L.Cc = C * c;
  L.Cs = C * s;
}

LT_HD void lt_poison_lens(LtLens<double>& L) {  // invalid parameters: the lens contributes NaN everywhere
  const double n = NAN;
  L.x0 = L.y0 = L.cx = L.sx = L.cy = L.sy = L.Kc = L.dK = L.sc = L.st = L.q2sc = L.q2st = L.g = L.f = L.Cc = L.Cs = n;
}

// fp32 record = fp64 record rounded once, except x0, y0 which the fp32 kernel fills per pixel tile (lens-frame
// coordinates of the tile origin, formed in fp64 and then rounded: DESIGN.md section 5, "fp32 coordinates").
LT_HD void lt_round_lens(const LtLens<double>& D, double dx, LtLens<float>& F) {
  F.x0 = 0.f;
  F.y0 = 0.f;
  F.cx = (float)(dx * D.cx);      // scaled lens-frame steps per pixel
  F.sx = (float)(dx * D.sx);
  F.cy = (float)(dx * D.cy);
  F.sy = (float)(dx * D.sy);
  F.Kc = (float)D.Kc;
  F.dK = (float)D.dK;
  F.sc = (float)D.sc;
  F.st = (float)D.st;
  F.q2sc = (float)D.q2sc;
  F.q2st = (float)D.q2st;
  F.g = (float)D.g;
  F.f = (float)D.f;
  F.Cc = (float)D.Cc;
  F.Cs = (float)D.Cs;
}

// ================================================================================================ SIE
struct LtRawSie {  // = lt_sie_lens of include/lt_gradient.h
  double x, y, e, phi, b0;
};

// Domain of the SIE (eq. 17-18 P:153-160 need 1 -+ eps > 0; the paper assumes eps << 1): |eps| < 1, b0 >= 0
// (eq. 22 P:183 is a square), all finite.
LT_HD bool lt_sie_valid(const LtRawSie& r) {
  const bool fin = isfinite(r.x) && isfinite(r.y) && isfinite(r.e) && isfinite(r.phi) && isfinite(r.b0);
  return fin && r.e > -1.0 && r.e < 1.0 && r.b0 >= 0.0;
}
LT_HD void lt_pack_sie(const LtRawSie& r, LtSieLens<double>& L) {
  double s, c;
  sincos(r.phi, &s, &c);
  const double a1 = 1.0 - r.e, a2 = 1.0 + r.e, b2 = r.b0 * r.b0;
  L.x0 = r.x;
  L.y0 = r.y;
  L.q11 = b2 * fma(a1 * c, c, a2 * s * s);
  L.q12 = b2 * (-2.0 * r.e * c * s);
  L.q22 = b2 * fma(a1 * s, s, a2 * c * c);
  L.pad = 0.0;
}
LT_HD void lt_poison_sie(LtSieLens<double>& L) {
  const double n = NAN;
  L.x0 = L.y0 = L.q11 = L.q12 = L.q22 = L.pad = n;
}
LT_HD void lt_round_sie(const LtSieLens<double>& D, double, LtSieLens<float>& F) {
  F.x0 = 0.f;
  F.y0 = 0.f;
  F.q11 = (float)D.q11;
  F.q12 = (float)D.q12;
  F.q22 = (float)D.q22;
  F.pad = 0.f;
}

// ================================================================================================ NFW
struct LtRawNfw {  // = lt_nfw_lens of include/lt_gradient.h
  double x, y, e, phi, ks, rs;
};
LT_HD bool lt_nfw_valid(const LtRawNfw& r) {
  const bool fin = isfinite(r.x) && isfinite(r.y) && isfinite(r.e) && isfinite(r.phi) && isfinite(r.ks) && isfinite(r.rs);
  return fin && r.e > -1.0 && r.e < 1.0 && r.ks >= 0.0 && r.rs > 0.0;
}
LT_HD void lt_pack_nfw(const LtRawNfw& r, LtNfwLens<double>& L) {
  double s, c;
  sincos(r.phi, &s, &c);
  const double a1 = 1.0 - r.e, a2 = 1.0 + r.e, ir2 = 1.0 / (r.rs * r.rs);
  L.x0 = r.x;
  L.y0 = r.y;
  L.q11 = ir2 * fma(a1 * c, c, a2 * s * s);
  L.q12 = ir2 * (-2.0 * r.e * c * s);
  L.q22 = ir2 * fma(a1 * s, s, a2 * c * c);
  L.amp = 4.0 * r.ks * r.rs * r.rs;
}
LT_HD void lt_poison_nfw(LtNfwLens<double>& L) {
  const double n = NAN;
  L.x0 = L.y0 = L.q11 = L.q12 = L.q22 = L.amp = n;
}
LT_HD void lt_round_nfw(const LtNfwLens<double>& D, double, LtNfwLens<float>& F) {
  F.x0 = 0.f;
  F.y0 = 0.f;
  F.q11 = (float)D.q11;
  F.q12 = (float)D.q12;
  F.q22 = (float)D.q22;
  F.amp = (float)D.amp;
}

// ================================================================================================ lens models
// What the kernels of lt_kernels.cuh are instantiated with: the record types, the per-lens precompute, the products of
// d2 = theta_2 - yc that the pixels of a row share (row) and the per-interaction body given d1 = theta_1 - xc
// (interact_sky).  kSkyFrame32: how the fp32 kernel forms its coordinates (DESIGN.md section 5 / 11): false = lens-frame
// position of the tile centre + in-tile steps along the rotated axes (interact_lens), true = sky-frame offset of the
// tile centre from the lens centre + in-tile steps of dx (interact_sky).
struct LtDpieModel {
  typedef LtRawLens Raw;
  template <class T> struct Rec { typedef LtLens<T> type; };
  template <class T> struct Row { T d2sx, d2cy; };
  static constexpr bool kTables = true;
  static constexpr bool kSkyFrame32 = false;
  static constexpr bool kPacked32 = true;      // the fp32 grid kernel evaluates two pixels per instruction (interact_lens_x2)
  static constexpr bool kConstRecords = true;  // fp64 kernels: records from the constant bank where the call allows it (+3 % at config 3)
  static constexpr int kConstGroup = 1;        // lenses per iteration of the constant-bank loops (lt_kernels.cuh: lt_const_lens_loop)
  static constexpr int kGroup32 = 2;           // lenses per iteration of the packed fp32 grid kernel
#if defined(__CUDACC__)
  static __device__ __forceinline__ void interact_lens_x2(const lt_f2 X, const lt_f2 Y, const LtLens<float>& L,
                                                          const LtTables2& tab, lt_f2& G1, lt_f2& G2) {
    lt_dpie_interact_x2(X, Y, L, tab, G1, G2);
  }
#endif
  static LT_HD bool valid(const Raw& r) { return lt_lens_valid(r); }
  static LT_HD void pack(const Raw& r, LtLens<double>& L) { lt_pack_lens(r, L); }
  static LT_HD void poison(LtLens<double>& L) { lt_poison_lens(L); }
  static LT_HD void round(const LtLens<double>& D, double dx, LtLens<float>& F) { lt_round_lens(D, dx, F); }
  static LT_HD double patch_scale(const Raw& r) { return r.b0; }
  // fp32 record for the plain-coordinate kernel: rotation constants per arcsec instead of per pixel
  static LT_HD void unscale32(const LtLens<double>& D, LtLens<float>& F) {
    F.cx = (float)D.cx; F.sx = (float)D.sx; F.cy = (float)D.cy; F.sy = (float)D.sy;
  }
  template <class T> static LT_HD Row<T> row(const T d2, const LtLens<T>& L) { return Row<T>{d2 * L.sx, d2 * L.cy}; }
  // GRID = called from the fp64 grid kernel (lt_sqrt_h: where a hoisted constant pays)
  template <class T, bool GRID = false>
  static LT_HD void interact_lens(const T X, const T Y, const LtLens<T>& L, const LtTables<T>& tab, T& G1, T& G2) {
    T ax, ay;
    lt_dpie_body<T, GRID>(X, Y, L, tab, ax, ay);
    lt_accumulate<T>(ax, ay, L, G1, G2);
  }
  template <class T, bool GRID = false>
  static LT_HD void interact_sky(const T d1, const Row<T>& r, const LtLens<T>& L, const LtTables<T>& tab, T& G1,
                                 T& G2) {
    const T X = lt_fma(d1, L.cx, r.d2sx);            // Alg. 1 l.5, times q/f
    const T Y = lt_fma(-d1, L.sy, r.d2cy);           // Alg. 1 l.6, times 1/f
    interact_lens<T, GRID>(X, Y, L, tab, G1, G2);
  }
  // the same from the absolute sky coordinates (t1, t2) of the pixel: what the fp64 kernels call
  template <class T> static LT_HD Row<T> row_abs(const T t2, const LtLens<T>& L) { return row<T>(t2 - L.y0, L); }   // l.4
  template <class T, bool GRID = false>
  static LT_HD void interact_abs(const T t1, const Row<T>& r, const LtLens<T>& L, const LtTables<T>& tab, T& G1, T& G2) {
    interact_sky<T, GRID>(t1 - L.x0, r, L, tab, G1, G2);                                                           // l.3
  }
};
struct LtSieModel {
  typedef LtRawSie Raw;
  template <class T> struct Rec { typedef LtSieLens<T> type; };
  static constexpr bool kTables = false;
  static constexpr bool kSkyFrame32 = true;
  static constexpr bool kPacked32 = true;
  // 48-byte records in uniform registers: P and Q lose their third register source (122 -> 114 pipe cycles per four
  // interactions by the count of DESIGN.md section 8); lens by lens the five LDCU at the top of the 66-instruction loop are
  // not hidden (3 % slower than shared memory), eight lenses per iteration are 5 % faster (SIE benchmark 26.8 -> 25.4 ms)
  static constexpr bool kConstRecords = true;
  static constexpr int kConstGroup = 8;
  static constexpr int kGroup32 = 8;
#if defined(__CUDACC__)
  static __device__ __forceinline__ void interact_sky_x2(const lt_f2 d1, const LtSieRow<float>& r, const LtSieLens<float>& L,
                                                         const LtTables2&, lt_f2& G1, lt_f2& G2) {
    lt_sie_interact_x2(d1, r, L, G1, G2);
  }
#endif
  static LT_HD bool valid(const Raw& r) { return lt_sie_valid(r); }
  static LT_HD void pack(const Raw& r, LtSieLens<double>& L) { lt_pack_sie(r, L); }
  static LT_HD void poison(LtSieLens<double>& L) { lt_poison_sie(L); }
  static LT_HD void round(const LtSieLens<double>& D, double dx, LtSieLens<float>& F) { lt_round_sie(D, dx, F); }
  static LT_HD double patch_scale(const Raw& r) { return r.b0; }
  static LT_HD void unscale32(const LtSieLens<double>&, LtSieLens<float>&) {}
  template <class T> static LT_HD LtSieRow<T> row(const T d2, const LtSieLens<T>& L) { return lt_sie_row<T>(d2, L); }
  template <class T>
  static LT_HD void interact_lens(const T, const T, const LtSieLens<T>&, const LtTables<T>&, T&, T&) {}   // unused
  template <class T, bool GRID = false>
  static LT_HD void interact_sky(const T d1, const LtSieRow<T>& r, const LtSieLens<T>& L, const LtTables<T>&, T& G1,
                                 T& G2) {
    lt_sie_interact<T>(d1, r, L, G1, G2);
  }
  template <class T> static LT_HD LtSieRow<T> row_abs(const T t2, const LtSieLens<T>& L) { return row<T>(t2 - L.y0, L); }
  template <class T, bool GRID = false>
  static LT_HD void interact_abs(const T t1, const LtSieRow<T>& r, const LtSieLens<T>& L, const LtTables<T>& tab, T& G1,
                                 T& G2) {
    interact_sky<T, GRID>(t1 - L.x0, r, L, tab, G1, G2);
  }
};
struct LtNfwModel {
  typedef LtRawNfw Raw;
  template <class T> struct Rec { typedef LtNfwLens<T> type; };
  static constexpr bool kTables = true;
  static constexpr bool kSkyFrame32 = true;
  static constexpr bool kPacked32 = false;
  static constexpr bool kConstRecords = false; // measured: -2 % fp64, +0.5 % mixed (profiles/r02_fp64_pipe_diagnostics.md section 13)
  static constexpr int kConstGroup = 1;
  static constexpr int kGroup32 = 1;
  static LT_HD bool valid(const Raw& r) { return lt_nfw_valid(r); }
  static LT_HD void pack(const Raw& r, LtNfwLens<double>& L) { lt_pack_nfw(r, L); }
  static LT_HD void poison(LtNfwLens<double>& L) { lt_poison_nfw(L); }
  static LT_HD void round(const LtNfwLens<double>& D, double dx, LtNfwLens<float>& F) { lt_round_nfw(D, dx, F); }
  static LT_HD double patch_scale(const Raw& r) { return 4.0 * r.ks * r.rs; }
  static LT_HD void unscale32(const LtNfwLens<double>&, LtNfwLens<float>&) {}
  template <class T> static LT_HD LtSieRow<T> row(const T d2, const LtNfwLens<T>& L) {
    return LtSieRow<T>{d2, L.q12 * d2, L.q22 * d2};
  }
  template <class T>
  static LT_HD void interact_lens(const T, const T, const LtNfwLens<T>&, const LtTables<T>&, T&, T&) {}   // unused
  template <class T, bool GRID = false>
  static LT_HD void interact_sky(const T d1, const LtSieRow<T>& r, const LtNfwLens<T>& L, const LtTables<T>& tab, T& G1,
                                 T& G2) {
    lt_nfw_interact<T>(d1, r, L, tab, G1, G2);
  }
  template <class T> static LT_HD LtSieRow<T> row_abs(const T t2, const LtNfwLens<T>& L) { return row<T>(t2 - L.y0, L); }
  template <class T, bool GRID = false>
  static LT_HD void interact_abs(const T t1, const LtSieRow<T>& r, const LtNfwLens<T>& L, const LtTables<T>& tab, T& G1,
                                 T& G2) {
    interact_sky<T, GRID>(t1 - L.x0, r, L, tab, G1, G2);
  }
};
