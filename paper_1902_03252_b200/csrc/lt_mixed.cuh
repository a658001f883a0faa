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

#define LT_PATCH_SPLIT 8
struct LtMixedDev {          // host-prepared constants of the rule
  float fdx;                 // (float)dx
  float t25;                 // (float)(dx / m_max)
  float t28;                 // (float)(c28 * dx)
  double h_cluster, h_galaxy, b0_cluster;
};

// a8, part 1: LT_PATCH_SPLIT CTAs per lens mark its DP patch: the box of half-width hp = max(1, ceil(h/dx)) pixels centred on the
// pixel nearest the lens centre, clipped to the grid (R14); h by lens class (b0 >= threshold: cluster-scale, R15).
// Overlapping patches write the same value, so plain stores are race-free in effect.
template <class M>
__global__ void lt_patch_kernel(const typename M::Raw* __restrict__ raw, int n_lens, double x_min, double y_min, double dx,
                                int nx, int ny, LtMixedDev mp, unsigned char* __restrict__ flags) {
  lt_grid_dependency_wait();      // launched as a programmatic dependent (lt_kernels.cuh); keeps the chain of waits whole
  const int k = blockIdx.x / LT_PATCH_SPLIT, part = blockIdx.x % LT_PATCH_SPLIT;     // grid: n_lens * LT_PATCH_SPLIT CTAs
  if (k >= n_lens) return;
  // one thread reads the lens (the catalogue may sit in pinned host memory: lt_gradient_grid_host), the CTA shares it
  __shared__ double s_lens[3];
  if (threadIdx.x == 0) {
    const typename M::Raw r = raw[k];
    s_lens[0] = r.x;
    s_lens[1] = r.y;
    s_lens[2] = M::patch_scale(r);                                            // the lens's deflection scale (R15)
  }
  __syncthreads();
  const double xc = s_lens[0], yc = s_lens[1], b0 = s_lens[2];
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
  // LT_PATCH_SPLIT CTAs share a lens: a cluster-scale patch is 160 000 pixels at the paper's scale, a galaxy-scale one 441
  for (long long t = (long long)part * blockDim.x + threadIdx.x; t < n; t += (long long)blockDim.x * LT_PATCH_SPLIT) {
    const long long jj = t / w, ii = t - jj * w;
    flags[(size_t)(j0 + jj) * nx + (size_t)(i0 + ii)] = 1;
  }
}

// a8, part 2: criteria on the fp32 map, merged with the patch bit (the fp32 kernel has already written the widened fp32
// values into the fp64 output, R17), flag byte written back, counts.
// A CTA takes LT_FLAG_PPI * 256 consecutive pixels per iteration, LT_FLAG_PPI per thread (256 apart, so every load is
// coalesced): the loads of the four pixels and their neighbours are in flight together.
// a8, part 3 (lt_quad_list_kernel): the flagged pixels are handed to the fp64 pass as a compact list of QUADS -- four
// neighbouring pixels of one row, i = 4 iq .. 4 iq + 3, listed when any of them is flagged.  The fp64 pass recomputes all
// four (they share the row terms of every lens exactly as the four pixels of a thread do in the grid kernel) and
// stores the flagged ones only.  Flagged pixels come in runs (patches are boxes, the critical-line bands are many pixels
// wide): on the SIE benchmark the listed quads hold 1.005 x the flagged pixels.
#define LT_FLAG_PPI 4
struct LtFlagLoads { float2 a, bx, by; unsigned char f0; bool fwd_x, fwd_y; };
// the loads of one pixel, branch-free so that those of the LT_FLAG_PPI pixels of a thread are issued back to back:
// x neighbour i - 1 (i + 1 at i = 0, R12), y neighbour j - 1 (j + 1 at j = 0); an axis of extent 1 reads the pixel itself
__device__ __forceinline__ LtFlagLoads lt_flag_load(const float2* __restrict__ sp, unsigned int p, int nx, int ny,
                                                    const unsigned char* __restrict__ flags) {
  const unsigned int j = p / (unsigned int)nx, i = p - j * (unsigned int)nx;     // n_pix < 2^32 (the list holds 32-bit indices)
  LtFlagLoads v;
  v.fwd_x = i == 0;
  v.fwd_y = j == 0;
  const size_t qx = nx > 1 ? (v.fwd_x ? (size_t)p + 1 : (size_t)p - 1) : (size_t)p;
  const size_t qy = ny > 1 ? (v.fwd_y ? (size_t)p + (size_t)nx : (size_t)p - (size_t)nx) : (size_t)p;
  v.a = sp[p];
  v.bx = sp[qx];
  v.by = sp[qy];
  v.f0 = flags[p];
  return v;
}
__device__ __forceinline__ unsigned char lt_flag_decide(const LtFlagLoads& v, int nx, int ny, const LtMixedDev& mp) {
  float c0 = INFINITY, c1 = INFINITY, c2 = 0.f, c3 = 0.f;     // values that never fire
  if (nx > 1) {                                               // x neighbour: delta_1 (eq. 24), delta_4 (eq. 27)
    const float d1 = v.fwd_x ? v.bx.x - v.a.x : v.a.x - v.bx.x;
    const float d4 = v.fwd_x ? v.bx.y - v.a.y : v.a.y - v.bx.y;
    c0 = fabsf(mp.fdx - d1);
    c3 = fabsf(d4);
  }
  if (ny > 1) {                                               // y neighbour: delta_2 (eq. 24), delta_3 (eq. 27)
    const float d2 = v.fwd_y ? v.by.y - v.a.y : v.a.y - v.by.y;
    const float d3 = v.fwd_y ? v.by.x - v.a.x : v.a.x - v.by.x;
    c1 = fabsf(mp.fdx - d2);
    c2 = fabsf(d3);
  }
  unsigned char f = v.f0 & 1;
  if (c0 < mp.t25 || c1 < mp.t25) f |= 2;                     // eq. 25
  if (c2 > mp.t28 || c3 > mp.t28) f |= 4;                     // eq. 28
  return f;
}

__global__ void __launch_bounds__(256)
lt_flag_kernel(const float2* __restrict__ sp, int nx, int ny, LtMixedDev mp, unsigned char* __restrict__ flags,
               LtWsHeader* __restrict__ hdr) {
  lt_grid_dependency_wait();
  const size_t n_pix = (size_t)nx * ny;
  constexpr size_t TILE = (size_t)LT_FLAG_PPI * 256;
  const unsigned lane = threadIdx.x & 31;
  unsigned long long c_any = 0, c_patch = 0, c25 = 0, c28 = 0;
  for (size_t base = (size_t)blockIdx.x * TILE; base < n_pix; base += (size_t)gridDim.x * TILE) {
    LtFlagLoads v[LT_FLAG_PPI];
#pragma unroll
    for (int k = 0; k < LT_FLAG_PPI; ++k) {
      const size_t p = base + (size_t)k * 256 + threadIdx.x;
      v[k] = lt_flag_load(sp, (unsigned int)(p < n_pix ? p : n_pix - 1), nx, ny, flags);   // past the end: a valid pixel, unused
    }
#pragma unroll
    for (int k = 0; k < LT_FLAG_PPI; ++k) {
      const size_t p = base + (size_t)k * 256 + threadIdx.x;
      if (p < n_pix) {
        const unsigned char f = lt_flag_decide(v[k], nx, ny, mp);
        flags[p] = f;
        c_any += f != 0;
        c_patch += f & 1;
        c25 += (f >> 1) & 1;
        c28 += (f >> 2) & 1;
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    c_any += __shfl_xor_sync(0xffffffffu, c_any, o);
    c_patch += __shfl_xor_sync(0xffffffffu, c_patch, o);
    c25 += __shfl_xor_sync(0xffffffffu, c25, o);
    c28 += __shfl_xor_sync(0xffffffffu, c28, o);
  }
  if (lane == 0) {
    if (c_any) atomicAdd(&hdr->n_flagged, c_any);
    if (c_patch) atomicAdd(&hdr->n_patch, c_patch);
    if (c25) atomicAdd(&hdr->n_eq25, c25);
    if (c28) atomicAdd(&hdr->n_eq28, c28);
  }
}

// a8, part 3: compact list of the quads (j, iq) -> j * quads_per_row + iq that hold a flagged pixel.  A CTA takes
// LT_QUADS_PER_THREAD * 256 consecutive quads per iteration, LT_QUADS_PER_THREAD per thread (256 apart: coalesced, all
// loads in flight together), and appends with ONE atomic per CTA and iteration (a warp scans the 32 segment counts) --
// where nearly every quad is listed, an atomic per warp is a queue on one address (config 3: 131 000 of them, 92 us).
// The order of the list is irrelevant because every quad is recomputed independently.  Flag bytes are read with one
// 32-bit load where the quad is 4-byte aligned and inside the row.
#define LT_QUADS_PER_THREAD 4
__device__ __forceinline__ bool lt_quad_any(const unsigned char* __restrict__ flags, size_t q, size_t n_quads, int nx,
                                            int quads_per_row) {
  if (q >= n_quads) return false;
  const size_t j = q / (size_t)quads_per_row;
  const int i0 = (int)(q - j * (size_t)quads_per_row) * 4;
  const size_t p = j * (size_t)nx + (size_t)i0;
  if (i0 + 3 < nx && (p & 3) == 0) return *reinterpret_cast<const unsigned int*>(flags + p) != 0u;
  bool any = false;
  for (int k = 0; k < 4; ++k)
    if (i0 + k < nx) any = any || flags[p + k] != 0;
  return any;
}
__global__ void __launch_bounds__(256)
lt_quad_list_kernel(const unsigned char* __restrict__ flags, int nx, int ny, int quads_per_row,
                    unsigned int* __restrict__ list, LtWsHeader* __restrict__ hdr) {
  lt_grid_dependency_wait();
  const unsigned lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  const size_t n_quads = (size_t)quads_per_row * ny;
  constexpr size_t TILE = (size_t)LT_QUADS_PER_THREAD * 256;
  __shared__ unsigned int seg_base[LT_QUADS_PER_THREAD * 8];          // segment s = k * 8 + warp: 32 quads of sub-tile k
  static_assert(LT_QUADS_PER_THREAD * 8 == 32, "one segment per lane of warp 0");
  // whole CTAs iterate together so that the ballots see a full mask and the barriers are reached by every thread
  for (size_t base = (size_t)blockIdx.x * TILE; base < n_quads; base += (size_t)gridDim.x * TILE) {
    bool any[LT_QUADS_PER_THREAD];
    unsigned m[LT_QUADS_PER_THREAD];
#pragma unroll
    for (int k = 0; k < LT_QUADS_PER_THREAD; ++k)
      any[k] = lt_quad_any(flags, base + (size_t)k * 256 + threadIdx.x, n_quads, nx, quads_per_row);
#pragma unroll
    for (int k = 0; k < LT_QUADS_PER_THREAD; ++k) {
      m[k] = __ballot_sync(0xffffffffu, any[k]);
      if (lane == 0) seg_base[k * 8 + wrp] = (unsigned int)__popc(m[k]);
    }
    __syncthreads();
    if (wrp == 0) {
      const unsigned int cnt = seg_base[lane];
      unsigned int incl = cnt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned int v = __shfl_up_sync(0xffffffffu, incl, o);
        if ((int)lane >= o) incl += v;
      }
      unsigned int cta_base = 0;
      if (lane == 31 && incl) cta_base = atomicAdd(&hdr->list_count, incl);
      cta_base = __shfl_sync(0xffffffffu, cta_base, 31);
      seg_base[lane] = cta_base + incl - cnt;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < LT_QUADS_PER_THREAD; ++k)
      if (any[k])
        list[seg_base[k * 8 + wrp] + __popc(m[k] & ((1u << lane) - 1u))] = (unsigned int)(base + (size_t)k * 256 + threadIdx.x);
    __syncthreads();                                          // seg_base is rewritten by the next iteration
  }
}
