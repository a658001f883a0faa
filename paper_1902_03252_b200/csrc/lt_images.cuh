// lt_images.cuh -- the consumer of the deflection map described in the paper's section 2.2.2 and Fig. 1,
// lens every image-plane triangle into the source plane (eq. 13) and report the triangles
// whose source-plane image contains a given source point ("barycenter"), i.e. the predicted multiple images.
//
// Readings (R23-R25): a pixel is the cell between four neighbouring nodes of the map, cut along the diagonal
// from node (i+1, j) to node (i, j+1) into T0 = [(i,j), (i+1,j), (i,j+1)] and T1 = [(i+1,j+1), (i,j+1), (i+1,j)]; triangles
// are closed (a point on a shared edge is reported by both neighbours), zero-area source triangles contain nothing; the
// predicted image position is the image-plane point with the same barycentric coordinates.
//
// One thread per cell, a CTA = 32 x 8 cells, persistent grid over the tiles.  The four corner deflections are read once
// per cell (neighbouring threads and rows hit L1/L2: 16 B of DRAM traffic per node), beta = theta - (D_LS/D_OS) gradPsi is
// formed in registers.  The sources are staged in shared memory once per CTA with their coordinates rounded down / up to
// fp32.  Culling is hierarchical and conservative: 32 sources at a time are tested, one per lane, against the bounding
// box of the warp's 32 cells; the survivors (usually none) against the cell's own conservatively rounded fp32 box --
// four compares on the FP32 pipe -- and only on a hit the exact fp64 edge functions are evaluated.  (Staging the tile's
// nodes in shared memory instead was measured slower: two barriers per 256-cell tile cost more than the re-reads.)
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

__global__ void __launch_bounds__(256, 4)
lt_find_images_kernel(const double2* __restrict__ grad, double x_min, double y_min, double dx, int nx, int ny,
                      double dls_dos, const double2* __restrict__ sources, int n_sources, int tiles_x, int n_tiles,
                      LtImageHit* __restrict__ hits, int max_hits, int* __restrict__ n_hits) {
  __shared__ LtSrcBox box[LT_SRC_CHUNK];
  __shared__ double2 src[LT_SRC_CHUNK];
  const int lx = threadIdx.x & 31, ly = threadIdx.x >> 5, lane = lx;
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int ty = tile / tiles_x, tx = tile - ty * tiles_x;
    const int i = tx * 32 + lx, j = ty * 8 + ly;
    const bool live = i < nx - 1 && j < ny - 1;
    // image-plane nodes and their source-plane images (eq. 13); dead threads keep a box that no source can hit
    double t1a = 0, t1b = 0, t2a = 0, t2b = 0;
    double b00x = 0, b00y = 0, b10x = 0, b10y = 0, b01x = 0, b01y = 0, b11x = 0, b11y = 0;
    float lo_x = 1.f, hi_x = -1.f, lo_y = 1.f, hi_y = -1.f;
    if (live) {
      t1a = __dadd_rn(x_min, __dmul_rn((double)i, dx));
      t1b = __dadd_rn(x_min, __dmul_rn((double)(i + 1), dx));
      t2a = __dadd_rn(y_min, __dmul_rn((double)j, dx));
      t2b = __dadd_rn(y_min, __dmul_rn((double)(j + 1), dx));
      const size_t p = (size_t)j * nx + i;
      const double2 g00 = __ldg(grad + p), g10 = __ldg(grad + p + 1), g01 = __ldg(grad + p + nx),
                    g11 = __ldg(grad + p + nx + 1);
      b00x = __dsub_rn(t1a, __dmul_rn(dls_dos, g00.x)); b00y = __dsub_rn(t2a, __dmul_rn(dls_dos, g00.y));
      b10x = __dsub_rn(t1b, __dmul_rn(dls_dos, g10.x)); b10y = __dsub_rn(t2a, __dmul_rn(dls_dos, g10.y));
      b01x = __dsub_rn(t1a, __dmul_rn(dls_dos, g01.x)); b01y = __dsub_rn(t2b, __dmul_rn(dls_dos, g01.y));
      b11x = __dsub_rn(t1b, __dmul_rn(dls_dos, g11.x)); b11y = __dsub_rn(t2b, __dmul_rn(dls_dos, g11.y));
      // conservative fp32 bounding box: corners rounded to nearest (error <= 2^-24 |v|), min / max on the FP32 pipe, then
      // widened by 2^-23 |v| plus a constant below every coordinate of interest
      const float f00x = (float)b00x, f10x = (float)b10x, f01x = (float)b01x, f11x = (float)b11x;
      const float f00y = (float)b00y, f10y = (float)b10y, f01y = (float)b01y, f11y = (float)b11y;
      lo_x = fminf(fminf(f00x, f10x), fminf(f01x, f11x));
      hi_x = fmaxf(fmaxf(f00x, f10x), fmaxf(f01x, f11x));
      lo_y = fminf(fminf(f00y, f10y), fminf(f01y, f11y));
      hi_y = fmaxf(fmaxf(f00y, f10y), fmaxf(f01y, f11y));
      lo_x -= fmaf(fabsf(lo_x), 1.1920929e-7f, 1e-30f);
      hi_x += fmaf(fabsf(hi_x), 1.1920929e-7f, 1e-30f);
      lo_y -= fmaf(fabsf(lo_y), 1.1920929e-7f, 1e-30f);
      hi_y += fmaf(fabsf(hi_y), 1.1920929e-7f, 1e-30f);
    }
    // bounding box of the warp's 32 cells (dead lanes carry an empty box: +-1 swapped, widened here to +-inf)
    float wlo_x = live ? lo_x : INFINITY, whi_x = live ? hi_x : -INFINITY, wlo_y = live ? lo_y : INFINITY,
          whi_y = live ? hi_y : -INFINITY;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      wlo_x = fminf(wlo_x, __shfl_xor_sync(0xffffffffu, wlo_x, o));
      whi_x = fmaxf(whi_x, __shfl_xor_sync(0xffffffffu, whi_x, o));
      wlo_y = fminf(wlo_y, __shfl_xor_sync(0xffffffffu, wlo_y, o));
      whi_y = fmaxf(whi_y, __shfl_xor_sync(0xffffffffu, whi_y, o));
    }
    for (int base = 0; base < n_sources; base += LT_SRC_CHUNK) {
      const int cnt = min(LT_SRC_CHUNK, n_sources - base);
      if (n_sources > LT_SRC_CHUNK || tile == (int)blockIdx.x) {      // a single chunk is staged once per CTA
        __syncthreads();
        for (int k = threadIdx.x; k < LT_SRC_CHUNK; k += blockDim.x) {
          if (k < cnt) {
            const double2 s = sources[base + k];
            src[k] = s;
            box[k] = LtSrcBox{__double2float_rd(s.x), __double2float_ru(s.x), __double2float_rd(s.y), __double2float_ru(s.y)};
          } else {
            box[k] = LtSrcBox{0.f, -INFINITY, 0.f, -INFINITY};   // x_ru = -inf: fails against every box
          }
        }
        __syncthreads();
      }
      // warp-level culling: the 32 cells of a warp (one row segment) share a source-plane bounding box; 32 sources at a
      // time are tested against it, one per lane, and only the survivors (usually none or one) are tested per cell
      for (int k0 = 0; k0 < cnt; k0 += 32) {
        const LtSrcBox bw = box[k0 + lane];        // entries beyond cnt are boxes nothing can hit
        unsigned m = __ballot_sync(0xffffffffu, (bw.x_ru >= wlo_x) & (bw.x_rd <= whi_x) & (bw.y_ru >= wlo_y) & (bw.y_rd <= whi_y));
        while (m) {
          const int k = k0 + __ffs(m) - 1;
          m &= m - 1;
          const LtSrcBox b = box[k];
          // conservative: P in [lo, hi] in exact arithmetic implies this test passes
          if ((b.x_ru >= lo_x) & (b.x_rd <= hi_x) & (b.y_ru >= lo_y) & (b.y_rd <= hi_y)) {
            const double Px = src[k].x, Py = src[k].y;
            const int cell = j * nx + i;
            lt_test_triangle(b00x, b00y, b10x, b10y, b01x, b01y, t1a, t2a, t1b, t2a, t1a, t2b, Px, Py, base + k, cell,
                             0, hits, max_hits, n_hits);
            lt_test_triangle(b11x, b11y, b01x, b01y, b10x, b10y, t1b, t2b, t1a, t2b, t1b, t2a, Px, Py, base + k, cell,
                             1, hits, max_hits, n_hits);
          }
        }
      }
    }
  }
}
