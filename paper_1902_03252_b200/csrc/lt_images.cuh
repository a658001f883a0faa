// lt_images.cuh -- the consumer of the deflection map described in the paper's section 2.2.2 and Fig. 1,
// lens every image-plane triangle into the source plane (eq. 13) and report the triangles
// whose source-plane image contains a given source point ("barycenter"), i.e. the predicted multiple images.
//
// Readings (R23-R25): a pixel is the cell between four neighbouring nodes of the map, cut along the diagonal
// from node (i+1, j) to node (i, j+1) into T0 = [(i,j), (i+1,j), (i,j+1)] and T1 = [(i+1,j+1), (i,j+1), (i+1,j)]; triangles
// are closed (a point on a shared edge is reported by both neighbours), zero-area source triangles contain nothing; the
// predicted image position is the image-plane point with the same barycentric coordinates.
//
// Mapping: a WARP owns a strip of 32 node columns (31 cell columns; neighbouring strips share one node column) and
// walks down a block of rows.  Every node of the map is loaded ONCE (16 B, one coalesced 512-byte row segment per warp
// and row) and lensed once: beta = theta - (D_LS/D_OS) gradPsi in fp64, rounded to fp32 for the culling.  A cell's four
// corners are the lane's own node, its right neighbour's (one shuffle) and the same two of the previous row (kept in
// registers).  Rows are taken four at a time: four loads in flight per lane, and the conservative source-plane bounding
// box of the warp's 4 x 31 cells is reduced over the lanes once per group.  The sources are staged in shared memory once
// per CTA with their coordinates rounded down / up to fp32.  Culling is hierarchical and conservative: 32 sources at a
// time are tested, one per lane, against the warp's box; the survivors (usually none) against the conservatively rounded
// fp32 box of each of the lane's four cells; only on a hit are the cell's corners re-read (L1/L2) and the exact fp64 edge
// functions evaluated.
// All fp64 products and differences are written with explicit round-to-nearest intrinsics in the order of the
// definition, so that the inside / outside decision is the same bit for bit wherever it is evaluated.
#pragma once
#include <cuda_runtime.h>

struct LtImageHit {          // = lt_image_hit of include/lt_gradient.h (32 bytes)
  int source, cell, triangle, reserved;
  double x, y;
};

#define LT_SRC_CHUNK 256

// one source point in shared memory: the exact coordinates and, separately (one broadcast LDS.128 per source in the
// hot loop), the coordinates rounded down / up to fp32 for the conservative bounding-box test
struct LtSrcBox { float x_rd, x_ru, y_rd, y_ru; };

__device__ __forceinline__ double lt_cross(double ux, double uy, double vx, double vy) {
  return __dsub_rn(__dmul_rn(ux, vy), __dmul_rn(uy, vx));
}

// exact test of one triangle (A, B, C in the source plane; tA, tB, tC the image-plane nodes) against source P
__device__ __forceinline__ void lt_test_triangle(double Ax, double Ay, double Bx, double By, double Cx, double Cy,
                                                 double tAx, double tAy, double tBx, double tBy, double tCx, double tCy,
                                                 double Px, double Py, int source, int cell, int triangle,
                                                 LtImageHit* __restrict__ hits, int max_hits, int* __restrict__ n_hits) {
  const double e0 = lt_cross(__dsub_rn(Bx, Ax), __dsub_rn(By, Ay), __dsub_rn(Px, Ax), __dsub_rn(Py, Ay));
  const double e1 = lt_cross(__dsub_rn(Cx, Bx), __dsub_rn(Cy, By), __dsub_rn(Px, Bx), __dsub_rn(Py, By));
  const double e2 = lt_cross(__dsub_rn(Ax, Cx), __dsub_rn(Ay, Cy), __dsub_rn(Px, Cx), __dsub_rn(Py, Cy));
  const double area = __dadd_rn(__dadd_rn(e0, e1), e2);
  const bool inside = ((e0 >= 0.0 && e1 >= 0.0 && e2 >= 0.0) || (e0 <= 0.0 && e1 <= 0.0 && e2 <= 0.0)) && area != 0.0;
  if (!inside) return;
  const int slot = atomicAdd(n_hits, 1);
  if (slot >= max_hits) return;                       // counted, not stored: the caller sees *n_hits > max_hits
  const double wA = __ddiv_rn(e1, area), wB = __ddiv_rn(e2, area), wC = __ddiv_rn(e0, area);
  LtImageHit h;
  h.source = source;
  h.cell = cell;
  h.triangle = triangle;
  h.reserved = 0;
  h.x = __dadd_rn(__dadd_rn(__dmul_rn(wA, tAx), __dmul_rn(wB, tBx)), __dmul_rn(wC, tCx));
  h.y = __dadd_rn(__dadd_rn(__dmul_rn(wA, tAy), __dmul_rn(wB, tBy)), __dmul_rn(wC, tCy));
  hits[slot] = h;
}

#ifndef LT_FI_ROWS
#define LT_FI_ROWS 4            // rows per group
#endif
#ifndef LT_FI_BLOCK_ROWS
#define LT_FI_BLOCK_ROWS 64     // cell rows per work item (one more node row is read to start it: 1.6 % of the traffic)
#endif
#ifndef LT_FI_MINB
#define LT_FI_MINB 2
#endif
#define LT_FI_STRIP 31          // cell columns per strip

// source-plane image of node (i, j), eq. 13: exactly the operations of the API's definition, so that the hot path (which
// keeps only the fp32 rounding) and the exact path (which re-reads the node) agree bit for bit
__device__ __forceinline__ double2 lt_node_beta(const double2 g, int i, int j, double x_min, double y_min, double dx,
                                                double dls_dos, double& t1, double& t2) {
  t1 = __dadd_rn(x_min, __dmul_rn((double)i, dx));
  t2 = __dadd_rn(y_min, __dmul_rn((double)j, dx));
  return make_double2(__dsub_rn(t1, __dmul_rn(dls_dos, g.x)), __dsub_rn(t2, __dmul_rn(dls_dos, g.y)));
}

// the exact fp64 test of both triangles of cell (i, j) against source k (rare: only after the fp32 boxes overlap)
__device__ __forceinline__ void lt_cell_exact(const double2* __restrict__ grad, int i, int j, int nx, double x_min, double y_min,
                                           double dx, double dls_dos, double Px, double Py, int source,
                                           LtImageHit* __restrict__ hits, int max_hits, int* __restrict__ n_hits) {
  const size_t p = (size_t)j * nx + i;
  double t1a, t1b, t2a, t2b, u1, u2;        // (the two outputs of lt_node_beta must not alias)
  const double2 b00 = lt_node_beta(__ldg(grad + p), i, j, x_min, y_min, dx, dls_dos, t1a, t2a);
  const double2 b10 = lt_node_beta(__ldg(grad + p + 1), i + 1, j, x_min, y_min, dx, dls_dos, t1b, u2);
  const double2 b01 = lt_node_beta(__ldg(grad + p + nx), i, j + 1, x_min, y_min, dx, dls_dos, u1, t2b);
  const double2 b11 = lt_node_beta(__ldg(grad + p + nx + 1), i + 1, j + 1, x_min, y_min, dx, dls_dos, u1, u2);
  const int cell = j * nx + i;
  lt_test_triangle(b00.x, b00.y, b10.x, b10.y, b01.x, b01.y, t1a, t2a, t1b, t2a, t1a, t2b, Px, Py, source, cell, 0, hits,
                   max_hits, n_hits);
  lt_test_triangle(b11.x, b11.y, b01.x, b01.y, b10.x, b10.y, t1b, t2b, t1a, t2b, t1b, t2a, Px, Py, source, cell, 1, hits,
                   max_hits, n_hits);
}

__global__ void __launch_bounds__(256, LT_FI_MINB)
lt_find_images_kernel(const double2* __restrict__ grad, double x_min, double y_min, double dx, int nx, int ny,
                      double dls_dos, const double2* __restrict__ sources, int n_sources, int n_strips, int n_items,
                      LtImageHit* __restrict__ hits, int max_hits, int* __restrict__ n_hits) {
  __shared__ LtSrcBox box[LT_SRC_CHUNK];
  __shared__ double2 src[LT_SRC_CHUNK];
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5, warps = blockDim.x >> 5;
  for (int base = 0; base < n_sources; base += LT_SRC_CHUNK) {            // usually one chunk: the map is walked once
    const int cnt = min(LT_SRC_CHUNK, n_sources - base);
    __syncthreads();
    for (int k = threadIdx.x; k < LT_SRC_CHUNK; k += blockDim.x) {
      if (k < cnt) {
        const double2 s = sources[base + k];
        src[k] = s;
        box[k] = LtSrcBox{__double2float_rd(s.x), __double2float_ru(s.x), __double2float_rd(s.y), __double2float_ru(s.y)};
      } else {
        box[k] = LtSrcBox{0.f, -INFINITY, 0.f, -INFINITY};                // x_ru = -inf: fails against every box
      }
    }
    __syncthreads();
    for (int item = blockIdx.x * warps + wrp; item < n_items; item += gridDim.x * warps) {
      const int rb = item / n_strips, strip = item - rb * n_strips;
      const int i = strip * LT_FI_STRIP + lane;
      const int j_begin = rb * LT_FI_BLOCK_ROWS, j_end = min(j_begin + LT_FI_BLOCK_ROWS, ny - 1);   // cell rows [j_begin, j_end)
      const bool node_ok = i < nx;
      const bool cell_col_ok = lane < LT_FI_STRIP && i < nx - 1;
      const double2* col = grad + (node_ok ? i : nx - 1);
      double t1, t2;
      // node row j_begin: the "previous row" of the first cell row
      double2 b = lt_node_beta(__ldg(col + (size_t)j_begin * nx), i, j_begin, x_min, y_min, dx, dls_dos, t1, t2);
      float pfx = (float)b.x, pfy = (float)b.y;
      float prx = __shfl_down_sync(0xffffffffu, pfx, 1), pry = __shfl_down_sync(0xffffffffu, pfy, 1);
      double2 g[LT_FI_ROWS], g_next[LT_FI_ROWS];
#pragma unroll
      for (int r = 0; r < LT_FI_ROWS; ++r)                                 // node rows j_begin + 1 .. + 4, clamped to the map
        g_next[r] = __ldg(col + (size_t)min(j_begin + r + 1, ny - 1) * nx);
      for (int j0 = j_begin; j0 < j_end; j0 += LT_FI_ROWS) {
#pragma unroll
        for (int r = 0; r < LT_FI_ROWS; ++r) {
          g[r] = g_next[r];
          // the rows of the NEXT group are requested before this group is worked on: the kernel is bound by the latency
          // of a row segment, not by arithmetic (past the block's end the clamped row is loaded and dropped)
          g_next[r] = __ldg(col + (size_t)min(j0 + LT_FI_ROWS + r + 1, ny - 1) * nx);
        }
        float lo_x[LT_FI_ROWS], hi_x[LT_FI_ROWS], lo_y[LT_FI_ROWS], hi_y[LT_FI_ROWS];
        float wlo_x = INFINITY, whi_x = -INFINITY, wlo_y = INFINITY, whi_y = -INFINITY;
#pragma unroll
        for (int r = 0; r < LT_FI_ROWS; ++r) {
          b = lt_node_beta(g[r], i, j0 + r + 1, x_min, y_min, dx, dls_dos, t1, t2);
          const float fx = (float)b.x, fy = (float)b.y;
          const float rx = __shfl_down_sync(0xffffffffu, fx, 1), ry = __shfl_down_sync(0xffffffffu, fy, 1);
          // conservative fp32 bounding box of cell (i, j0 + r): corners rounded to nearest (error <= 2^-24 |v|), min / max
          // on the FP32 pipe, then widened by 2^-23 |v| plus a constant below every coordinate of interest
          float ax = fminf(fminf(pfx, prx), fminf(fx, rx)), bx = fmaxf(fmaxf(pfx, prx), fmaxf(fx, rx));
          float ay = fminf(fminf(pfy, pry), fminf(fy, ry)), by = fmaxf(fmaxf(pfy, pry), fmaxf(fy, ry));
          ax -= fmaf(fabsf(ax), 1.1920929e-7f, 1e-30f);
          bx += fmaf(fabsf(bx), 1.1920929e-7f, 1e-30f);
          ay -= fmaf(fabsf(ay), 1.1920929e-7f, 1e-30f);
          by += fmaf(fabsf(by), 1.1920929e-7f, 1e-30f);
          const bool ok = cell_col_ok && j0 + r < j_end;
          lo_x[r] = ok ? ax : 1.f;                                        // dead cells keep a box that no source can hit
          hi_x[r] = ok ? bx : -1.f;
          lo_y[r] = ok ? ay : 1.f;
          hi_y[r] = ok ? by : -1.f;
          if (ok) {
            wlo_x = fminf(wlo_x, ax);
            whi_x = fmaxf(whi_x, bx);
            wlo_y = fminf(wlo_y, ay);
            whi_y = fmaxf(whi_y, by);
          }
          pfx = fx; pfy = fy; prx = rx; pry = ry;
        }
        // the lane's own box (its four cells), then the bounding box of the warp's 4 x 31 cells
        const float llo_x = wlo_x, lhi_x = whi_x, llo_y = wlo_y, lhi_y = whi_y;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          wlo_x = fminf(wlo_x, __shfl_xor_sync(0xffffffffu, wlo_x, o));
          whi_x = fmaxf(whi_x, __shfl_xor_sync(0xffffffffu, whi_x, o));
          wlo_y = fminf(wlo_y, __shfl_xor_sync(0xffffffffu, wlo_y, o));
          whi_y = fmaxf(whi_y, __shfl_xor_sync(0xffffffffu, whi_y, o));
        }
        // warp-level culling: 32 sources at a time, one per lane, against the warp's box; survivors per cell
        for (int k0 = 0; k0 < cnt; k0 += 32) {
          const LtSrcBox bw = box[k0 + lane];        // entries beyond cnt are boxes nothing can hit
          unsigned m = __ballot_sync(0xffffffffu, (bw.x_ru >= wlo_x) & (bw.x_rd <= whi_x) & (bw.y_ru >= wlo_y) & (bw.y_rd <= whi_y));
          while (m) {
            const int k = k0 + __ffs(m) - 1;
            m &= m - 1;
            const LtSrcBox sb = box[k];
            // most survivors of the warp's box are in no lane's box: one vote instead of four cell tests per lane
            if (!__any_sync(0xffffffffu, (sb.x_ru >= llo_x) & (sb.x_rd <= lhi_x) & (sb.y_ru >= llo_y) & (sb.y_rd <= lhi_y))) continue;
            unsigned cells = 0;        // the lane's cells whose box the source can be in
#pragma unroll
            for (int r = 0; r < LT_FI_ROWS; ++r)
              // conservative: P in [lo, hi] in exact arithmetic implies this test passes
              if ((sb.x_ru >= lo_x[r]) & (sb.x_rd <= hi_x[r]) & (sb.y_ru >= lo_y[r]) & (sb.y_rd <= hi_y[r])) cells |= 1u << r;
            while (cells) {
              const int r = __ffs(cells) - 1;
              cells &= cells - 1;
              lt_cell_exact(grad, i, j0 + r, nx, x_min, y_min, dx, dls_dos, src[k].x, src[k].y, base + k, hits, max_hits,
                            n_hits);
            }
          }
        }
      }
    }
  }
}
