// lt_chi2.cuh -- the two small steps that close the paper's chi^2 algorithm around the deflection map (section 2.2.2,
// P:140; eq. 11), so that the whole evaluation stays on the device and on one stream:
//   lt_gradient_points (observed images) -> lt_source_barycentres -> lt_gradient_grid -> lt_find_images -> lt_chi2.
// Both are latency-sized (hundreds of images): plain kernels, every fp64 operation written with an explicit
// round-to-nearest intrinsic in the order of the definition, so that the numbers are reproducible bit for bit.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include "lt_images.cuh"

struct LtChi2Result {        // = lt_chi2_result of include/lt_gradient.h (32 bytes)
  double chi2;
  long long n_matched, n_unmatched, reserved;
};

// beta_ij = theta_ij - (D_LS/D_OS) alpha_ij (eq. 13); barycentre_i = (sum_j beta_ij) / n_i, j in catalogue
// order.  One thread per multiple-image system; a system without images gets (nan, nan), which no triangle contains.
__global__ void lt_source_barycentres_kernel(const double2* __restrict__ theta, const double2* __restrict__ alpha,
                                             const int* __restrict__ offsets, int n_systems, double dls_dos,
                                             double2* __restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_systems) return;
  const int a = offsets[i], b = offsets[i + 1];
  if (b <= a) {
    out[i] = make_double2(CUDART_NAN, CUDART_NAN);
    return;
  }
  double s1 = 0.0, s2 = 0.0;
  for (int j = a; j < b; ++j) {
    const double2 t = theta[j], g = alpha[j];
    s1 = __dadd_rn(s1, __dsub_rn(t.x, __dmul_rn(dls_dos, g.x)));
    s2 = __dadd_rn(s2, __dsub_rn(t.y, __dmul_rn(dls_dos, g.y)));
  }
  const double n = (double)(b - a);
  out[i] = make_double2(__ddiv_rn(s1, n), __ddiv_rn(s2, n));
}

// term_ij = |theta_obs,ij - nearest predicted image of system i|^2 / sigma_ij^2 (eq. 11; pairing: reading R28).  One
// thread per observed image; its system is found by bisection in the offsets; the hits are read by all threads alike
// (broadcast loads).  nan = the system has no predicted image.
__global__ void lt_chi2_terms_kernel(const double2* __restrict__ obs, const double* __restrict__ sigma,
                                     const int* __restrict__ offsets, int n_systems, int n_images,
                                     const LtImageHit* __restrict__ hits, const int* __restrict__ n_hits_ptr,
                                     int max_hits, double* __restrict__ terms) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_images) return;
  int lo = 0, hi = n_systems;                       // largest i with offsets[i] <= j (empty systems are skipped over)
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (offsets[mid] <= j) lo = mid; else hi = mid;
  }
  const int n_hits = min(*n_hits_ptr, max_hits);
  const double2 p = obs[j];
  double best = CUDART_INF;
  bool found = false;
  for (int h = 0; h < n_hits; ++h) {
    if (hits[h].source != lo) continue;
    const double dx = __dsub_rn(p.x, hits[h].x), dy = __dsub_rn(p.y, hits[h].y);
    const double d2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
    best = fmin(best, d2);
    found = true;
  }
  const double s = sigma[j];
  terms[j] = found ? __ddiv_rn(best, __dmul_rn(s, s)) : CUDART_NAN;
}

// chi^2 = sum of the terms in catalogue order (one thread: a few hundred additions, and the order is the definition's)
__global__ void lt_chi2_sum_kernel(const double* __restrict__ terms, int n_images, LtChi2Result* __restrict__ res) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  double total = 0.0;
  long long matched = 0, unmatched = 0;
  for (int j = 0; j < n_images; ++j) {
    const double t = terms[j];
    if (t != t) {
      ++unmatched;
    } else {
      total = __dadd_rn(total, t);
      ++matched;
    }
  }
  res->chi2 = total;
  res->n_matched = matched;
  res->n_unmatched = unmatched;
  res->reserved = 0;
}
