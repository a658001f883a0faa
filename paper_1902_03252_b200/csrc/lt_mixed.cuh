// lt_mixed.cuh -- the paper's mixed-precision rule on the device: DP centre patches (section 3.2,
// P:284) and the critical-line criteria of section 3.3 (eq. 24-28) evaluated on the single
// precision map, with the readings R11-R16 of DESIGN.md (thresholds scale with the pixel size; forward neighbour at
// i = 0 / j = 0; a criterion along an axis of extent 1 is skipped; one DP pass over patch OR criteria).
// Flag byte per pixel: bit0 = inside a centre patch, bit1 = eq. 25 on delta_1 or delta_2, bit2 = eq. 28 on delta_3
// or delta_4.  All criterion arithmetic is fp32 with separately rounded operations (the file is built with
// --fmad=false), thresholds rounded to fp32 once on the host.
#pragma once
#include "lt_kernels.cuh"

struct LtCentre { double x, y, scale; };            // lt_mixed_rule: a lens as the rule sees it (centre, deflection scale)
struct LtCentreModel {
  typedef LtCentre Raw;
  static __host__ __device__ double patch_scale(const Raw& r) { return r.scale; }
};

struct LtMixedDev {          // host-prepared constants of the rule
  float fdx;                 // (float)dx
  float t25;                 // (float)(dx / m_max)
  float t28;                 // (float)(c28 * dx)
  double h_cluster, h_galaxy, b0_cluster;
};

// a8, part 1: one CTA per lens marks its DP patch: the box of half-width hp = max(1, ceil(h/dx)) pixels centred on the
// pixel nearest the lens centre, clipped to the grid (R14); h by lens class (b0 >= threshold: cluster-scale, R15).
// Overlapping patches write the same value, so plain stores are race-free in effect.
template <class M>
__global__ void lt_patch_kernel(const typename M::Raw* __restrict__ raw, int n_lens, double x_min, double y_min, double dx,
                                int nx, int ny, LtMixedDev mp, unsigned char* __restrict__ flags) {
  lt_grid_dependency_wait();      // launched as a programmatic dependent (lt_kernels.cuh); keeps the chain of waits whole
  const int k = blockIdx.x;
  if (k >= n_lens) return;
  const double xc = raw[k].x, yc = raw[k].y, b0 = M::patch_scale(raw[k]);   // the lens's deflection scale (R15)
  if (!(isfinite(xc) && isfinite(yc))) return;
  const double h = (b0 >= mp.b0_cluster) ? mp.h_cluster : mp.h_galaxy;
  long long hp = (long long)ceil(h / dx);
  if (hp < 1) hp = 1;
  // centres far outside the grid: clamp before the integer conversion (the box is then empty after clipping)
  const double fi = fmin(fmax((xc - x_min) / dx, -4.0e9), 4.0e9), fj = fmin(fmax((yc - y_min) / dx, -4.0e9), 4.0e9);
  const long long ic = llround(fi), jc = llround(fj);
  const long long i0 = max(ic - hp, 0LL), i1 = min(ic + hp, (long long)nx - 1);
  const long long j0 = max(jc - hp, 0LL), j1 = min(jc + hp, (long long)ny - 1);
  if (i1 < i0 || j1 < j0) return;
  const long long w = i1 - i0 + 1, n = w * (j1 - j0 + 1);
  for (long long t = threadIdx.x; t < n; t += blockDim.x) {
    const long long jj = t / w, ii = t - jj * w;
    flags[(size_t)(j0 + jj) * nx + (size_t)(i0 + ii)] = 1;
  }
}

// a8, part 2: criteria on the fp32 map, merge with the patch bit (the fp32 kernel has already written the widened fp32
// values into the fp64 output, R17),
// append flagged pixels to the compact list (CTA-aggregated atomic; the order of the list is irrelevant because
// every pixel is recomputed independently), count.
__global__ void __launch_bounds__(256)
lt_flag_kernel(const float2* __restrict__ sp, int nx, int ny, LtMixedDev mp, unsigned char* __restrict__ flags,
               unsigned int* __restrict__ list, LtWsHeader* __restrict__ hdr) {
  lt_grid_dependency_wait();
  const size_t n_pix = (size_t)nx * ny;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const unsigned lane = threadIdx.x & 31;
  unsigned long long c_patch = 0, c25 = 0, c28 = 0;
  // whole CTAs iterate together (the trip count is rounded up to a multiple of 256 pixels) so that the ballots see a full
  // mask and the barriers below are reached by every thread
  __shared__ unsigned int warp_cnt[8], warp_base[8];
  const unsigned wrp = threadIdx.x >> 5;
  const size_t n_round = (n_pix + 255) / 256 * 256;
  for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n_round; p += stride) {
    const bool live = p < n_pix;
    unsigned char f = 0;
    if (live) {
      const int j = (int)(p / (size_t)nx), i = (int)(p - (size_t)j * nx);
      const float2 a = sp[p];
      float c0 = INFINITY, c1 = INFINITY, c2 = 0.f, c3 = 0.f;     // values that never fire
      if (nx > 1) {                                               // x neighbour: delta_1 (eq. 24), delta_4 (eq. 27)
        float d1, d4;
        if (i > 0) {
          const float2 b = sp[p - 1];
          d1 = a.x - b.x;
          d4 = a.y - b.y;
        } else {
          const float2 b = sp[p + 1];
          d1 = b.x - a.x;
          d4 = b.y - a.y;
        }
        c0 = fabsf(mp.fdx - d1);
        c3 = fabsf(d4);
      }
      if (ny > 1) {                                               // y neighbour: delta_2 (eq. 24), delta_3 (eq. 27)
        float d2, d3;
        if (j > 0) {
          const float2 b = sp[p - nx];
          d2 = a.y - b.y;
          d3 = a.x - b.x;
        } else {
          const float2 b = sp[p + nx];
          d2 = b.y - a.y;
          d3 = b.x - a.x;
        }
        c1 = fabsf(mp.fdx - d2);
        c2 = fabsf(d3);
      }
      f = flags[p] & 1;
      if (c0 < mp.t25 || c1 < mp.t25) f |= 2;                     // eq. 25
      if (c2 > mp.t28 || c3 > mp.t28) f |= 4;                     // eq. 28
      flags[p] = f;
      c_patch += f & 1;
      c25 += (f >> 1) & 1;
      c28 += (f >> 2) & 1;
    }
    // append: one atomic per CTA and iteration (the eight warps' counts are scanned in shared memory)
    const unsigned m = __ballot_sync(0xffffffffu, f != 0);
    if (lane == 0) warp_cnt[wrp] = (unsigned int)__popc(m);
    __syncthreads();
    if (threadIdx.x == 0) {
      unsigned int tot = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) { warp_base[w] = tot; tot += warp_cnt[w]; }
      const unsigned int cta_base = tot ? atomicAdd(&hdr->list_count, tot) : 0u;
#pragma unroll
      for (int w = 0; w < 8; ++w) warp_base[w] += cta_base;
    }
    __syncthreads();
    if (f != 0) list[warp_base[wrp] + __popc(m & ((1u << lane) - 1u))] = (unsigned int)p;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    c_patch += __shfl_xor_sync(0xffffffffu, c_patch, o);
    c25 += __shfl_xor_sync(0xffffffffu, c25, o);
    c28 += __shfl_xor_sync(0xffffffffu, c28, o);
  }
  if (lane == 0) {
    if (c_patch) atomicAdd(&hdr->n_patch, c_patch);
    if (c25) atomicAdd(&hdr->n_eq25, c25);
    if (c28) atomicAdd(&hdr->n_eq28, c28);
  }
}
