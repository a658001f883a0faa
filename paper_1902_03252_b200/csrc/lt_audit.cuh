// lt_audit.cuh -- the paper's accuracy criterion evaluated on the device (calibrating the mixed rule).
//
// Section 3.2: a single precision gradient is accurate enough where its error stays below a quarter of a
// pixel divided by the magnification along the axis, |err_i| <= dx / (4 M_i), with M_i = dx / |dx - delta_i| and
// delta_1, delta_2 the neighbour differences of eq. 24 (eq. 26) -- taken here from the double
// precision map.  The budget of component i is therefore |dx - delta_i| / 4.  Readings R12 (forward neighbour in the
// first column / row; an axis of extent 1 has delta = 0) and R13 (D_LS/D_OS = 1) as in lt_mixed.cuh.
// For every pixel: bit 0 / bit 1 of the violation byte = component 1 / 2 exceeds its budget; counts of violating pixels,
// split by the rule's mask (flagged / missed); the largest |SP - DP| (worse component, arcsec) overall, inside and
// outside the rule's centre patches, and by Chebyshev distance (pixels) to the nearest lens centre in the bins
// [0,1) [1,2) [2,4) ... [64,128) [128,inf) -- the table form of the paper's Fig. 9.
// Every fp64 operation is an explicit round-to-nearest intrinsic in the order of the definition, so the results can be
// compared bit for bit with a plain CPU evaluation (oracle/calibrate_ref.py, which shares no code with this file).
#pragma once
#include "lt_kernels.cuh"

#define LT_AUDIT_BINS 9
#define LT_AUDIT_CHUNK 512              // lens centres staged in shared memory at a time

struct LtAuditResult {                  // = lt_audit_result of include/lt_gradient.h
  long long n_pixels, n_violating, n_violating_flagged, n_violating_missed, n_flagged;
  double max_err, max_err_in_patch, max_err_outside_patch;
  double max_err_by_distance[LT_AUDIT_BINS];
  double implied_m_max, implied_m_max_outside_patch;       // filled on the host by lt_rule_audit_result
};

// max of non-negative doubles through their bit patterns (which order like the values)
__device__ __forceinline__ void lt_atomic_max_nonneg(double* addr, double v) {
  atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

__global__ void __launch_bounds__(256)
lt_rule_audit_kernel(const float2* __restrict__ sp, const double2* __restrict__ dp, double x_min, double y_min, double dx,
                     int nx, int ny, const double* __restrict__ centres, int n_centres,
                     const unsigned char* __restrict__ flags, unsigned char* __restrict__ violation,
                     LtAuditResult* __restrict__ res) {
  __shared__ double2 s_c[LT_AUDIT_CHUNK];                  // centres in pixel units: ((xc - x_min) / dx, (yc - y_min) / dx)
  __shared__ double s_max[3 + LT_AUDIT_BINS];
  __shared__ unsigned long long s_cnt[4];
  if (threadIdx.x < 3 + LT_AUDIT_BINS) s_max[threadIdx.x] = 0.0;
  if (threadIdx.x < 4) s_cnt[threadIdx.x] = 0ull;
  __syncthreads();
  const size_t n_pix = (size_t)nx * ny;
  // whole CTAs iterate together (the centre chunks are staged cooperatively)
  for (size_t base = (size_t)blockIdx.x * blockDim.x; base < n_pix; base += (size_t)gridDim.x * blockDim.x) {
    const size_t p = base + threadIdx.x;
    const bool live = p < n_pix;
    const size_t q = live ? p : n_pix - 1;
    const int j = (int)(q / (size_t)nx), i = (int)(q - (size_t)j * nx);
    double best = INFINITY;                                // Chebyshev distance to the nearest centre, pixels
    for (int c0 = 0; c0 < n_centres; c0 += LT_AUDIT_CHUNK) {
      const int cnt = min(LT_AUDIT_CHUNK, n_centres - c0);
      __syncthreads();
      for (int k = threadIdx.x; k < cnt; k += blockDim.x)
        s_c[k] = make_double2(__ddiv_rn(__dsub_rn(centres[3 * (c0 + k)], x_min), dx),
                              __ddiv_rn(__dsub_rn(centres[3 * (c0 + k) + 1], y_min), dx));
      __syncthreads();
      for (int k = 0; k < cnt; ++k) {
        const double da = fabs(__dsub_rn((double)i, s_c[k].x)), db = fabs(__dsub_rn((double)j, s_c[k].y));
        best = fmin(best, fmax(da, db));
      }
    }
    if (live) {
      const double2 a = dp[p];
      const float2 s = sp[p];
      const double e1 = fabs(__dsub_rn((double)s.x, a.x)), e2 = fabs(__dsub_rn((double)s.y, a.y));
      double d1 = 0.0, d2 = 0.0;                           // eq. 24 on the DP map (R12 at the first column / row)
      if (nx > 1) d1 = i > 0 ? __dsub_rn(a.x, dp[p - 1].x) : __dsub_rn(dp[p + 1].x, a.x);
      if (ny > 1) d2 = j > 0 ? __dsub_rn(a.y, dp[p - nx].y) : __dsub_rn(dp[p + nx].y, a.y);
      const double s1 = fabs(__dsub_rn(dx, d1)), s2 = fabs(__dsub_rn(dx, d2));     // eq. 26: |dx - delta_i|
      const unsigned char v = (unsigned char)((e1 > __dmul_rn(0.25, s1) ? 1 : 0) | (e2 > __dmul_rn(0.25, s2) ? 2 : 0));
      if (violation) violation[p] = v;
      const unsigned char f = flags ? flags[p] : (unsigned char)0;
      const double err = fmax(e1, e2);
      if (v) {
        atomicAdd(&s_cnt[0], 1ull);
        atomicAdd(&s_cnt[f ? 1 : 2], 1ull);
      }
      if (f) atomicAdd(&s_cnt[3], 1ull);
      if (err > 0.0) {                                     // NaN and zero change nothing
        lt_atomic_max_nonneg(&s_max[0], err);
        lt_atomic_max_nonneg(&s_max[(f & 1) ? 1 : 2], err);
        int bin = LT_AUDIT_BINS - 1;                       // edges 0 1 2 4 8 16 32 64 128
        if (best < 1.0) bin = 0;
        else if (best < 2.0) bin = 1;
        else if (best < 4.0) bin = 2;
        else if (best < 8.0) bin = 3;
        else if (best < 16.0) bin = 4;
        else if (best < 32.0) bin = 5;
        else if (best < 64.0) bin = 6;
        else if (best < 128.0) bin = 7;
        lt_atomic_max_nonneg(&s_max[3 + bin], err);
      }
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (s_cnt[0]) atomicAdd(reinterpret_cast<unsigned long long*>(&res->n_violating), s_cnt[0]);
    if (s_cnt[1]) atomicAdd(reinterpret_cast<unsigned long long*>(&res->n_violating_flagged), s_cnt[1]);
    if (s_cnt[2]) atomicAdd(reinterpret_cast<unsigned long long*>(&res->n_violating_missed), s_cnt[2]);
    if (s_cnt[3]) atomicAdd(reinterpret_cast<unsigned long long*>(&res->n_flagged), s_cnt[3]);
    if (blockIdx.x == 0) res->n_pixels = (long long)n_pix;
  }
  if (threadIdx.x < 3 + LT_AUDIT_BINS && s_max[threadIdx.x] > 0.0) {
    double* dst = threadIdx.x == 0 ? &res->max_err : threadIdx.x == 1 ? &res->max_err_in_patch
                : threadIdx.x == 2 ? &res->max_err_outside_patch : &res->max_err_by_distance[threadIdx.x - 3];
    lt_atomic_max_nonneg(dst, s_max[threadIdx.x]);
  }
}
