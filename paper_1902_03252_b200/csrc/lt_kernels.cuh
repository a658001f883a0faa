// lt_kernels.cuh -- device kernels of the gradient-map path: per-lens precompute, the fp64 and
// fp32 grid kernels, the fp64 quad kernel of the mixed-precision recompute (a9) and the kernels of lt_gradient_points.
//
// Mapping: data parallelism over pixels only.  A CTA owns tiles of TILE_W x TILE_H
// pixels (a warp = one row segment, each thread PPT pixels strided by 32 in x so that every store instruction of a
// warp is one contiguous 512 B / 256 B line), walks the lens catalogue staged in shared memory in chunks (every lane
// reads the same record: broadcast LDS.128, no bank conflicts), keeps the 2*PPT accumulators in registers for the whole
// lens loop (Alg. 1 l.13-14) and stores each pixel once.  The grid is persistent: min(#tiles, CTAs/SM * #SM) CTAs
// stride over the tiles [tile_begin, tile_end) of the row-major tile order, so a catalogue that fits one chunk is
// staged once per CTA (fp64).  The host (lt_api.cu) gives each launch a whole number of waves and hands the ragged
// rest to the next smaller pixels-per-thread variant.
#pragma once
#include <cuda_runtime.h>
#include "lt_pack.cuh"

#ifndef LT_WARPS_PER_CTA
#define LT_WARPS_PER_CTA 8
#endif
#define LT_THREADS (32 * LT_WARPS_PER_CTA)
#define LT_TILE_H LT_WARPS_PER_CTA
#define LT_PRECOMPUTE_THREADS 128
#define LT_TABLE_BLOCKS ((LT_TABLE_ENTRIES + LT_PRECOMPUTE_THREADS - 1) / LT_PRECOMPUTE_THREADS)

// Domain check: precompute block b stores max over its invalid lenses of (n_lens - k), 0 = all valid, in slot b of an
// int array that follows the header (plain stores: nothing has to be zeroed before the kernel runs).
#define LT_BAD_SLOTS 512            // LT_MAX_LENSES / LT_PRECOMPUTE_THREADS

struct LtWsHeader {                 // first 256 bytes of the workspace; (re)initialised by the precompute kernel
  int bad_blocks;                   // number of slots of the bad-code array written by this call
  int n_lens;
  unsigned int list_count;          // number of quads appended to the recompute list (mixed)
  unsigned int pad0;
  unsigned long long n_patch, n_eq25, n_eq28;
  unsigned long long n_flagged;     // flagged pixels (patch OR eq. 25 OR eq. 28)
  unsigned long long pad1[26];
};
static_assert(sizeof(LtWsHeader) == 256, "workspace header is 256 bytes");

// Programmatic dependent launch (sm_90+): the grid kernels are launched with the programmatic-stream-serialization
// attribute (lt_api.cu), so their CTAs may be dispatched while the kernel before them in the stream is still running.
// lt_grid_dependency_wait() returns once that kernel has completed and its writes are visible; lt_launch_dependents()
// lets the kernel after this one start its dispatch.  Both are no-ops in a launch without the attribute.
__device__ __forceinline__ void lt_grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void lt_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ------------------------------------------------------------------------------------------------ a1: precompute
template <class M>
__global__ void lt_precompute_kernel(const typename M::Raw* __restrict__ raw, int n_lens, double dx,
                                     typename M::template Rec<double>::type* __restrict__ l64,
                                     typename M::template Rec<float>::type* __restrict__ l32,
                                     LtTables<double>* __restrict__ t64, LtTables<float>* __restrict__ t32,
                                     LtWsHeader* __restrict__ hdr, int* __restrict__ bad) {
  // the last LT_TABLE_BLOCKS blocks write the range-reduction tables (lt_math.cuh), one entry per thread, next to the
  // blocks that pack the lenses: the kernel is one dependent chain per thread, so its duration is the longest chain
  lt_launch_dependents();
  const int lens_blocks = (int)gridDim.x - (M::kTables ? LT_TABLE_BLOCKS : 0);
  if ((int)blockIdx.x >= lens_blocks) {
    const int e = ((int)blockIdx.x - lens_blocks) * (int)blockDim.x + (int)threadIdx.x;
    if (e < LT_TABLE_ENTRIES) lt_fill_table_entry(e, *t64, *t32);
    return;
  }
  __shared__ int block_bad;
  if (threadIdx.x == 0) block_bad = 0;
  __syncthreads();
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k == 0) {                       // the header of this call (the mixed-mode kernels add to the counters later)
    hdr->bad_blocks = lens_blocks;
    hdr->n_lens = n_lens;
    hdr->list_count = 0;
    hdr->n_patch = 0;
    hdr->n_eq25 = 0;
    hdr->n_eq28 = 0;
    hdr->n_flagged = 0;
  }
  if (k < n_lens) {
    const typename M::Raw r = raw[k];
    typename M::template Rec<double>::type D;
    if (M::valid(r)) {
      M::pack(r, D);
    } else {
      M::poison(D);
      atomicMax(&block_bad, n_lens - k);
    }
    typename M::template Rec<float>::type F;
    M::round(D, dx, F);
    l64[k] = D;
    l32[k] = F;
  }
  __syncthreads();
  if (threadIdx.x == 0) bad[blockIdx.x] = block_bad;
}

// cooperative copy of `count` 16-byte words global -> shared
__device__ __forceinline__ void lt_copy16(void* dst, const void* src, int count) {
  uint4* d = reinterpret_cast<uint4*>(dst);
  const uint4* s = reinterpret_cast<const uint4*>(src);
  for (int w = threadIdx.x; w < count; w += blockDim.x) d[w] = s[w];
}

template <bool C, class A, class B> struct LtSelect { typedef A type; };
template <class A, class B> struct LtSelect<false, A, B> { typedef B type; };
// global (tau, phi) entries -> the shared structure-of-arrays copy the packed fp32 body reads (lt_math.cuh)
__device__ __forceinline__ void lt_stage_tables2(LtTables2* dst, const LtTables<float>* __restrict__ src) {
  for (int k = threadIdx.x; k < 2 * LT_ATAN_B + 1; k += blockDim.x) {
    dst->at_tau[k] = src->at[k][0];
    dst->at_phi[k] = src->at[k][1];
  }
  for (int k = threadIdx.x; k < 2 * LT_ATANH_B + 1; k += blockDim.x) {
    dst->ah_tau[k] = src->ah[k][0];
    dst->ah_K[k] = src->ah[k][1];
  }
}

// ------------------------------------------------------------------------------------------------ fp64 grid kernel
// a2 pixel coordinate (x_min + i*dx, product and sum rounded separately, exactly as the API states it), a3-a6 per
// lens (the model's interact_sky), a7 one double2 store per pixel.
template <class M, int PPT, int MINB>
__global__ void __launch_bounds__(LT_THREADS, MINB)
lt_grad_f64_kernel(const typename M::template Rec<double>::type* __restrict__ lens,
                   const LtTables<double>* __restrict__ tables, int n_lens,
                   int chunk, double x_min, double y_min, double dx, int nx, int ny, int tiles_x, int tile_begin,
                   int tile_end, double2* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char lt_smem[];
  typedef typename M::template Rec<double>::type Rec;
  __shared__ LtTables<double> tab;
  Rec* sl = reinterpret_cast<Rec*>(lt_smem);
  lt_grid_dependency_wait();
  if (M::kTables) lt_copy16(&tab, tables, (int)(sizeof(tab) / 16));
  __syncthreads();
  constexpr int TILE_W = 32 * PPT;
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  const bool single = n_lens <= chunk;
  if (single) {
    lt_copy16(sl, lens, n_lens * (int)(sizeof(Rec) / 16));
    __syncthreads();
  }
  for (int tile = tile_begin + blockIdx.x; tile < tile_end; tile += gridDim.x) {
    const int ty = tile / tiles_x, tx = tile - ty * tiles_x;
    const int j = ty * LT_TILE_H + wrp;
    const int i0 = tx * TILE_W + lane;
    const double t2 = __dadd_rn(y_min, __dmul_rn((double)j, dx));
    double t1[PPT], G1[PPT], G2[PPT];
#pragma unroll
    for (int p = 0; p < PPT; ++p) {
      t1[p] = __dadd_rn(x_min, __dmul_rn((double)(i0 + 32 * p), dx));
      G1[p] = 0.0;
      G2[p] = 0.0;
    }
    for (int base = 0; base < n_lens; base += chunk) {
      const int cnt = min(chunk, n_lens - base);
      if (!single) {
        __syncthreads();
        lt_copy16(sl, lens + base, cnt * (int)(sizeof(Rec) / 16));
        __syncthreads();
      }
#pragma unroll 1
      for (int k = 0; k < cnt; ++k) {
        const Rec L = sl[k];
        const auto row = M::template row_abs<double>(t2, L);        // Alg. 1 l.4 and what the pixels of the row share
#pragma unroll
        for (int p = 0; p < PPT; ++p) M::template interact_abs<double, true>(t1[p], row, L, tab, G1[p], G2[p]);  // l.3, l.5-14
      }
    }
    if (j < ny) {
#pragma unroll
      for (int p = 0; p < PPT; ++p) {
        const int i = i0 + 32 * p;
        if (i < nx) out[(size_t)j * nx + i] = make_double2(G1[p], G2[p]);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ fp64 grid kernel, records in the constant bank
// The same loop with the lens records held in __constant__ memory: a record is read with LDCU.128 into UNIFORM registers
// (every lane of every warp reads the same record anyway) and the FP64 instructions take those as operands directly,
// instead of eight broadcast LDS.128 into 32 vector registers per lens.  Same operations in the same order: identical
// bits; 3.6 % faster (profiles/r02_fp64_pipe_diagnostics.md).  __constant__ memory is per-module state, so the host side
// (lt_api.cu: ConstSlot) copies at most LT_CONST_SLOT_BYTES of records into the slot per launch, orders the slot's users
// across streams with an event, and launches once per slot-load: `acc` != null continues the sums that the launch before
// left there (the partial sum of the lenses so far, exactly the value the one-launch loop carries in registers); `acc` may
// be `out` itself or a device staging buffer when `out` is pinned host memory (only the last launch writes that).
// 4 pixels per thread only; the ragged rest of a grid keeps the shared-memory kernels above.
#define LT_CONST_SLOT_BYTES 57344
__constant__ double2 lt_const_slot[LT_CONST_SLOT_BYTES / 16];

// The lens loop of the constant-bank kernels for four pixels of a row: M::kConstGroup lenses per iteration.  The records
// of a group are all requested at its top (LDCU into uniform registers: no vector register is spent on them), so a short
// loop body -- the SIE's 66 instructions per lens -- does not wait for its record at every lens; the dPIE body is long
// enough alone and is not grouped (grouped, its loop outgrows the instruction cache: config 2 +7 % at 8 per group).
template <class M>
__device__ __forceinline__ void lt_const_lens_loop(const typename M::template Rec<double>::type* cl, int n_lens, double t2,
                                                   const double (&t1)[4], const LtTables<double>& tab, double (&G1)[4],
                                                   double (&G2)[4]) {
  typedef typename M::template Rec<double>::type Rec;
  constexpr int GROUP = M::kConstGroup;
  int k = 0;
  if constexpr (GROUP > 1) {
#pragma unroll 1
    for (; k + GROUP <= n_lens; k += GROUP) {
#pragma unroll
      for (int u = 0; u < GROUP; ++u) {
        const Rec& L = cl[k + u];
        const auto row = M::template row_abs<double>(t2, L);
#pragma unroll
        for (int p = 0; p < 4; ++p) M::template interact_abs<double, true>(t1[p], row, L, tab, G1[p], G2[p]);
      }
    }
  }
#pragma unroll 1
  for (; k < n_lens; ++k) {
    const Rec& L = cl[k];
    const auto row = M::template row_abs<double>(t2, L);
#pragma unroll
    for (int p = 0; p < 4; ++p) M::template interact_abs<double, true>(t1[p], row, L, tab, G1[p], G2[p]);
  }
}

// INPLACE: `acc` is a flag and the partial sums are read from `out` itself (device output); else `acc` is the buffer they
// are read from (null: start from zero) -- two instantiations because the in-place form compiles to the faster loop
template <class M, bool INPLACE>
__global__ void __launch_bounds__(LT_THREADS, 2)
lt_grad_f64_const_kernel(const LtTables<double>* __restrict__ tables, int n_lens,
                         typename LtSelect<INPLACE, int, const double2*>::type acc, double x_min, double y_min, double dx,
                         int nx, int ny, int tiles_x, int tile_begin, int tile_end, double2* __restrict__ out) {
  typedef typename M::template Rec<double>::type Rec;
  __shared__ LtTables<double> tab;
  lt_grid_dependency_wait();
  if (M::kTables) lt_copy16(&tab, tables, (int)(sizeof(tab) / 16));
  __syncthreads();
  constexpr int PPT = 4, TILE_W = 32 * PPT;
  const Rec* cl = reinterpret_cast<const Rec*>(lt_const_slot);
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  for (int tile = tile_begin + blockIdx.x; tile < tile_end; tile += gridDim.x) {
    const int ty = tile / tiles_x, tx = tile - ty * tiles_x;
    const int j = ty * LT_TILE_H + wrp;
    const int i0 = tx * TILE_W + lane;
    const double t2 = __dadd_rn(y_min, __dmul_rn((double)j, dx));
    double t1[PPT], G1[PPT], G2[PPT];
#pragma unroll
    for (int p = 0; p < PPT; ++p) {
      const int i = i0 + 32 * p;
      t1[p] = __dadd_rn(x_min, __dmul_rn((double)i, dx));
      G1[p] = 0.0;
      G2[p] = 0.0;
      if (acc && j < ny && i < nx) {
        double2 g;
        if constexpr (INPLACE) g = out[(size_t)j * nx + i];
        else g = acc[(size_t)j * nx + i];
        G1[p] = g.x;
        G2[p] = g.y;
      }
    }
    lt_const_lens_loop<M>(cl, n_lens, t2, t1, tab, G1, G2);
    if (j < ny) {
#pragma unroll
      for (int p = 0; p < PPT; ++p) {
        const int i = i0 + 32 * p;
        if (i < nx) out[(size_t)j * nx + i] = make_double2(G1[p], G2[p]);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ fp32 grid kernel
// Same mapping.  Coordinates: for every tile and lens the lens-frame position of the TILE CENTRE
// is formed in fp64 from the fp64 catalogue while the chunk is staged (a few fp64 operations per lens per tile, i.e.
// per 256*PPT interactions) and rounded to fp32; each pixel adds its small in-tile offset in fp32:
//   x' = X0 + il*(dx cos) + jl*(dx sin),  y' = Y0 + jl*(dx cos) - il*(dx sin)      (Alg. 1 l.3-6 merged)
// so the fp32 rounding of the coordinate is relative to the tile size, not to |theta| (the |theta_c|/|dtheta| term of
// (A.65)).  All per-interaction arithmetic is FP32.
template <class M, int PPT, int MINB, bool WIDE>
__global__ void __launch_bounds__(LT_THREADS, MINB)
lt_grad_f32_kernel(const typename M::template Rec<double>::type* __restrict__ lens64,
                   const typename M::template Rec<float>::type* __restrict__ lens32,
                   const LtTables<float>* __restrict__ tables, int n_lens, int chunk, double x_min, double y_min,
                   double dx, int nx, int ny, int tiles_x, int tile_begin, int tile_end, float2* __restrict__ out,
                   double2* __restrict__ out_wide) {
  extern __shared__ __align__(16) unsigned char lt_smem[];
  typedef typename M::template Rec<float>::type Rec;
  typedef typename M::template Rec<double>::type Rec64;
  constexpr int TILE_W = 32 * PPT;
  constexpr bool PACK = M::kPacked32 && (PPT % 2 == 0);
  __shared__ typename LtSelect<PACK, LtTables2, LtTables<float>>::type tab;
  Rec* sl = reinterpret_cast<Rec*>(lt_smem);
  lt_grid_dependency_wait();
  // the tables become visible with the first __syncthreads of the chunk loop
  if constexpr (PACK) {
    if (M::kTables) lt_stage_tables2(reinterpret_cast<LtTables2*>(&tab), tables);
  } else if (M::kTables) {
    lt_copy16(&tab, tables, (int)(sizeof(tab) / 16));
  }
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  // in-tile offsets from the tile centre, in pixels (exact in fp32)
  const float fdx = (float)dx;
  const float jl = (float)wrp - 0.5f * (float)(LT_TILE_H - 1);
  float il[PPT];
#pragma unroll
  for (int p = 0; p < PPT; ++p) il[p] = (float)(lane + 32 * p) - 0.5f * (float)(TILE_W - 1);
  for (int tile = tile_begin + blockIdx.x; tile < tile_end; tile += gridDim.x) {
    const int ty = tile / tiles_x, tx = tile - ty * tiles_x;
    const int j = ty * LT_TILE_H + wrp;
    const int i0 = tx * TILE_W + lane;
    // tile centre in the sky frame, fp64
    const double cx = x_min + ((double)(tx * TILE_W) + 0.5 * (double)(TILE_W - 1)) * dx;
    const double cy = y_min + ((double)(ty * LT_TILE_H) + 0.5 * (double)(LT_TILE_H - 1)) * dx;
    float G1[PPT], G2[PPT];
    lt_f2 H1[(PPT + 1) / 2], H2[(PPT + 1) / 2];      // PACK: the accumulators of pixel pairs (2p, 2p + 1)
#pragma unroll
    for (int p = 0; p < PPT; ++p) {
      G1[p] = 0.f;
      G2[p] = 0.f;
      H1[p / 2] = lt2(0.f);
      H2[p / 2] = lt2(0.f);
    }
    for (int base = 0; base < n_lens; base += chunk) {
      const int cnt = min(chunk, n_lens - base);
      __syncthreads();
      for (int k = threadIdx.x; k < cnt; k += LT_THREADS) {
        Rec F = lens32[base + k];
        const Rec64& D = lens64[base + k];
        if constexpr (M::kSkyFrame32) {             // sky-frame offset of the tile centre from the lens centre
          F.x0 = (float)(cx - D.x0);
          F.y0 = (float)(cy - D.y0);
        } else {                                    // (scaled) lens-frame position of the tile centre
          const double d1 = cx - D.x0, d2 = cy - D.y0;
          F.x0 = (float)fma(d1, D.cx, d2 * D.sx);
          F.y0 = (float)fma(-d1, D.sy, d2 * D.cy);
        }
        sl[k] = F;
      }
      __syncthreads();
      int k = 0;
      // M::kGroup32 lenses per iteration (packed kernels): the records of a group are requested from shared memory together,
      // so the loop does not wait for a record at every lens -- the SIE body is 27 instructions per lens and four pixels
      // (8 per group: SIE benchmark 10.7 -> 9.3 ms; dPIE, 156 instructions, 2 per group: -1.2 %).  Lens order and operations
      // per lens are those of the loop below: identical bits.
      if constexpr (PACK && M::kGroup32 > 1) {
        constexpr int GROUP = M::kGroup32;
#pragma unroll 1
        for (; k + GROUP <= cnt; k += GROUP) {
          Rec Lg[GROUP];
#pragma unroll
          for (int u = 0; u < GROUP; ++u) Lg[u] = sl[k + u];
#pragma unroll
          for (int u = 0; u < GROUP; ++u) {
            if constexpr (M::kSkyFrame32) {
              const float d2 = fmaf(jl, fdx, Lg[u].y0);
              const auto row = M::template row<float>(d2, Lg[u]);
#pragma unroll
              for (int p = 0; p < PPT; p += 2)
                M::interact_sky_x2(lt2_fma(lt2(il[p], il[p + 1]), lt2(fdx), lt2(Lg[u].x0)), row, Lg[u], tab, H1[p / 2], H2[p / 2]);
            } else {
              const float xr = fmaf(jl, Lg[u].sx, Lg[u].x0);
              const float yr = fmaf(jl, Lg[u].cy, Lg[u].y0);
#pragma unroll
              for (int p = 0; p < PPT; p += 2) {
                const lt_f2 il2 = lt2(il[p], il[p + 1]);
                const lt_f2 x = lt2_fma(il2, lt2(Lg[u].cx), lt2(xr));
                const lt_f2 y = lt2_fma(lt2_neg(il2), lt2(Lg[u].sy), lt2(yr));
                M::interact_lens_x2(x, y, Lg[u], tab, H1[p / 2], H2[p / 2]);
              }
            }
          }
        }
      }
#pragma unroll 1
      for (; k < cnt; ++k) {
        const Rec L = sl[k];
        if constexpr (M::kSkyFrame32 && PACK) {       // two pixels of the thread per instruction (lt_math.cuh)
          const float d2 = fmaf(jl, fdx, L.y0);
          const auto row = M::template row<float>(d2, L);
#pragma unroll
          for (int p = 0; p < PPT; p += 2)
            M::interact_sky_x2(lt2_fma(lt2(il[p], il[p + 1]), lt2(fdx), lt2(L.x0)), row, L, tab, H1[p / 2], H2[p / 2]);
        } else if constexpr (M::kSkyFrame32) {
          const float d2 = fmaf(jl, fdx, L.y0);
          const auto row = M::template row<float>(d2, L);
#pragma unroll
          for (int p = 0; p < PPT; ++p)
            M::template interact_sky<float>(fmaf(il[p], fdx, L.x0), row, L, tab, G1[p], G2[p]);   // Alg. 1 l.3-14
        } else if constexpr (PACK) {                  // two pixels of the thread per instruction (lt_math.cuh)
          const float xr = fmaf(jl, L.sx, L.x0);
          const float yr = fmaf(jl, L.cy, L.y0);
#pragma unroll
          for (int p = 0; p < PPT; p += 2) {
            const lt_f2 il2 = lt2(il[p], il[p + 1]);
            const lt_f2 x = lt2_fma(il2, lt2(L.cx), lt2(xr));
            const lt_f2 y = lt2_fma(lt2_neg(il2), lt2(L.sy), lt2(yr));
            M::interact_lens_x2(x, y, L, tab, H1[p / 2], H2[p / 2]);   // Alg. 1 l.7-14
          }
        } else {
          const float xr = fmaf(jl, L.sx, L.x0);
          const float yr = fmaf(jl, L.cy, L.y0);
#pragma unroll
          for (int p = 0; p < PPT; ++p) {
            const float x = fmaf(il[p], L.cx, xr);
            const float y = fmaf(-il[p], L.sy, yr);
            M::template interact_lens<float>(x, y, L, tab, G1[p], G2[p]);   // Alg. 1 l.7-14
          }
        }
      }
    }
    if constexpr (PACK) {
#pragma unroll
      for (int p = 0; p < PPT; ++p) {
        G1[p] = (p & 1) ? H1[p / 2].y : H1[p / 2].x;
        G2[p] = (p & 1) ? H2[p / 2].y : H2[p / 2].x;
      }
    }
    if (j < ny) {
#pragma unroll
      for (int p = 0; p < PPT; ++p) {
        const int i = i0 + 32 * p;
        if (i < nx) {
          out[(size_t)j * nx + i] = make_float2(G1[p], G2[p]);
          // mixed mode (R17): the widened value goes straight to the fp64 output; the fp64 pass overwrites flagged pixels
          if (WIDE) out_wide[(size_t)j * nx + i] = make_double2((double)G1[p], (double)G2[p]);
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ fp32, plain coordinates
// The paper's own SP version: "identical [to the DP version] up to the change in precision", i.e. Algorithm 1
// with theta, theta_center and their difference (l.3-4) all in fp32 -- no tile centre formed in fp64.  Not the product's
// fp32 mode: it exists so that the error that the tile-centre scheme removes can be measured (the |theta_c| / |dtheta|
// term of (A.65), the reason for the paper's DP patches around the lens centres; Fig. 9).
// Selected by lt_set_tuning (single_launch bit 4).  One pixel per thread, scalar arithmetic, no claim on speed.
template <class M, bool WIDE>
__global__ void __launch_bounds__(LT_THREADS)
lt_grad_f32_plain_kernel(const typename M::Raw* __restrict__ raw, const typename M::template Rec<double>::type* __restrict__ lens64,
                         const typename M::template Rec<float>::type* __restrict__ lens32,
                         const LtTables<float>* __restrict__ tables, int n_lens, int chunk, double x_min, double y_min,
                         double dx, int nx, int ny, float2* __restrict__ out, double2* __restrict__ out_wide) {
  extern __shared__ __align__(16) unsigned char lt_smem[];
  typedef typename M::template Rec<float>::type Rec;
  __shared__ LtTables<float> tab;
  Rec* sl = reinterpret_cast<Rec*>(lt_smem);
  lt_grid_dependency_wait();
  if (M::kTables) lt_copy16(&tab, tables, (int)(sizeof(tab) / 16));
  const float fx = (float)x_min, fy = (float)y_min, fdx = (float)dx;
  const size_t n_pix = (size_t)nx * ny;
  for (size_t base = (size_t)blockIdx.x * LT_THREADS; base < n_pix; base += (size_t)gridDim.x * LT_THREADS) {
    const size_t p = base + threadIdx.x;
    const size_t q = p < n_pix ? p : n_pix - 1;
    const int j = (int)(q / (size_t)nx), i = (int)(q - (size_t)j * nx);
    const float t1 = __fadd_rn(fx, __fmul_rn((float)i, fdx));      // a2 in fp32
    const float t2 = __fadd_rn(fy, __fmul_rn((float)j, fdx));
    float G1 = 0.f, G2 = 0.f;
    for (int b0 = 0; b0 < n_lens; b0 += chunk) {
      const int cnt = min(chunk, n_lens - b0);
      __syncthreads();
      for (int k = threadIdx.x; k < cnt; k += LT_THREADS) {
        Rec F = lens32[b0 + k];
        M::unscale32(lens64[b0 + k], F);                           // the rotation constants without the pixel size
        F.x0 = (float)raw[b0 + k].x;                               // theta_center rounded to fp32
        F.y0 = (float)raw[b0 + k].y;
        sl[k] = F;
      }
      __syncthreads();
#pragma unroll 1
      for (int k = 0; k < cnt; ++k) {
        const Rec L = sl[k];
        const float d2 = __fsub_rn(t2, L.y0);                      // Alg. 1 l.4 in fp32
        M::template interact_sky<float>(__fsub_rn(t1, L.x0), M::template row<float>(d2, L), L, tab, G1, G2);   // l.3, l.5-14
      }
    }
    if (p < n_pix) {
      out[p] = make_float2(G1, G2);
      if (WIDE) out_wide[p] = make_double2((double)G1, (double)G2);
    }
  }
}

// ------------------------------------------------------------------------------------------------ fp64 point-list kernel
// lt_gradient_points with more than a few thousand points: the gradient at an array of arbitrary points, one thread per
// point.  Uses the same interact_abs in the same lens order as the fp64 grid kernel: for a point that is a grid node,
// identical bits.  Groups of 4 * 256 points, 4 per thread (256 apart, so the reads stay coalesced); a rest of at most one
// 256-point group per CTA after the whole waves runs one point per thread.
template <class M, int PPT>
__device__ __forceinline__ void lt_points_group(const typename M::template Rec<double>::type* __restrict__ lens,
                                                const typename M::template Rec<double>::type* sl,
                                                const LtTables<double>& tab, int n_lens, int chunk, bool single,
                                                const double2* __restrict__ points, long long first, long long total,
                                                double2* __restrict__ out) {
  double t1[PPT], t2[PPT], G1[PPT], G2[PPT];
  bool live[PPT];
#pragma unroll
  for (int p = 0; p < PPT; ++p) {
    const long long t = first + (long long)p * LT_THREADS + threadIdx.x;
    live[p] = t < total;
    t1[p] = 0.0; t2[p] = 0.0; G1[p] = 0.0; G2[p] = 0.0;
    if (live[p]) {
      const double2 pt = points[t];
      t1[p] = pt.x;
      t2[p] = pt.y;
    }
  }
  for (int base = 0; base < n_lens; base += chunk) {
    const int cnt = min(chunk, n_lens - base);
    if (!single) {
      __syncthreads();
      lt_copy16(const_cast<typename M::template Rec<double>::type*>(sl), lens + base,
                cnt * (int)(sizeof(typename M::template Rec<double>::type) / 16));
      __syncthreads();
    }
#pragma unroll 1
    for (int k = 0; k < cnt; ++k) {
      const typename M::template Rec<double>::type L = sl[k];
#pragma unroll
      for (int p = 0; p < PPT; ++p)
        M::template interact_abs<double>(t1[p], M::template row_abs<double>(t2[p], L), L, tab, G1[p], G2[p]);
    }
  }
#pragma unroll
  for (int p = 0; p < PPT; ++p)
    if (live[p]) out[first + (long long)p * LT_THREADS + threadIdx.x] = make_double2(G1[p], G2[p]);
}

template <class M>
__global__ void __launch_bounds__(LT_THREADS, 2)
lt_grad_points_f64_kernel(const typename M::template Rec<double>::type* __restrict__ lens, const LtTables<double>* __restrict__ tables,
                          int n_lens, int chunk, const double2* __restrict__ points, long long n_points,
                          double2* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char lt_smem[];
  typedef typename M::template Rec<double>::type Rec;
  __shared__ LtTables<double> tab;
  Rec* sl = reinterpret_cast<Rec*>(lt_smem);
  lt_grid_dependency_wait();
  if (M::kTables) lt_copy16(&tab, tables, (int)(sizeof(tab) / 16));
  __syncthreads();
  const long long total = n_points;
  const bool single = n_lens <= chunk;
  if (single) {
    lt_copy16(sl, lens, n_lens * (int)(sizeof(Rec) / 16));
    __syncthreads();
  }
  constexpr int WIDE = 4;
  const long long per_wave = (long long)gridDim.x * (WIDE * LT_THREADS);
  long long n_wide = total / per_wave * gridDim.x;                  // groups of WIDE * 256 points: whole waves
  long long rest0 = n_wide * (WIDE * LT_THREADS);
  if (total - rest0 > (long long)gridDim.x * LT_THREADS) {          // more than one narrow group per CTA left:
    n_wide = (total + WIDE * LT_THREADS - 1) / (WIDE * LT_THREADS); // a ragged wide wave is cheaper than narrow rounds
    rest0 = total;
  }
  for (long long g = blockIdx.x; g < n_wide; g += gridDim.x)
    lt_points_group<M, WIDE>(lens, sl, tab, n_lens, chunk, single, points, g * (WIDE * LT_THREADS), total, out);
  const long long n_rest = (total - rest0 + LT_THREADS - 1) / LT_THREADS;   // <= gridDim.x
  for (long long g = blockIdx.x; g < n_rest; g += gridDim.x)
    lt_points_group<M, 1>(lens, sl, tab, n_lens, chunk, single, points, rest0 + g * LT_THREADS, total, out);
}

// ------------------------------------------------------------------------------------------------ fp64 quad kernel (a9)
// The fp64 pass of the mixed mode.  Work list: the quads of lt_quad_list_kernel (lt_mixed.cuh), count read from the
// workspace header on the device (no host round trip).  A thread owns one quad = four neighbouring pixels of a row, so
// its lens loop is the grid kernel's: one row term per lens shared by four interact_abs calls, same operations in the
// same order -- identical bits for identical pixels at the grid kernel's instruction count (the per-point kernel
// above forms the row terms once per pixel).  All four pixels are recomputed, the flagged ones are stored.
template <class M>
__global__ void __launch_bounds__(LT_THREADS, 2)
lt_grad_quads_f64_kernel(const typename M::template Rec<double>::type* __restrict__ lens,
                         const LtTables<double>* __restrict__ tables, int n_lens, int chunk, double x_min, double y_min,
                         double dx, int nx, int quads_per_row, const unsigned int* __restrict__ list,
                         const LtWsHeader* __restrict__ hdr, const unsigned char* __restrict__ flags,
                         double2* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char lt_smem[];
  typedef typename M::template Rec<double>::type Rec;
  __shared__ LtTables<double> tab;
  Rec* sl = reinterpret_cast<Rec*>(lt_smem);
  lt_grid_dependency_wait();
  if (M::kTables) lt_copy16(&tab, tables, (int)(sizeof(tab) / 16));
  __syncthreads();
  const long long total = (long long)hdr->list_count;
  const bool single = n_lens <= chunk;
  if (single) {
    lt_copy16(sl, lens, n_lens * (int)(sizeof(Rec) / 16));
    __syncthreads();
  }
  // whole CTAs iterate together (the lens chunks are staged cooperatively)
  for (long long first = (long long)blockIdx.x * LT_THREADS; first < total; first += (long long)gridDim.x * LT_THREADS) {
    const long long g = first + threadIdx.x;
    const bool live = g < total;
    const unsigned int q = live ? list[g] : 0u;
    const int j = (int)(q / (unsigned int)quads_per_row);
    const int i0 = (int)(q - (unsigned int)j * (unsigned int)quads_per_row) * 4;
    const size_t p0 = (size_t)j * nx + (size_t)i0;
    const double t2 = __dadd_rn(y_min, __dmul_rn((double)j, dx));
    double t1[4], G1[4], G2[4];
    bool keep[4];
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      t1[p] = __dadd_rn(x_min, __dmul_rn((double)(i0 + p), dx));
      G1[p] = 0.0;
      G2[p] = 0.0;
      keep[p] = live && i0 + p < nx && flags[p0 + p] != 0;
    }
    for (int base = 0; base < n_lens; base += chunk) {
      const int cnt = min(chunk, n_lens - base);
      if (!single) {
        __syncthreads();
        lt_copy16(sl, lens + base, cnt * (int)(sizeof(Rec) / 16));
        __syncthreads();
      }
#pragma unroll 1
      for (int k = 0; k < cnt; ++k) {
        const Rec L = sl[k];
        const auto row = M::template row_abs<double>(t2, L);
#pragma unroll
        for (int p = 0; p < 4; ++p) M::template interact_abs<double, true>(t1[p], row, L, tab, G1[p], G2[p]);
      }
    }
#pragma unroll
    for (int p = 0; p < 4; ++p)
      if (keep[p]) out[p0 + p] = make_double2(G1[p], G2[p]);
  }
}

// the quad kernel with the records in the constant bank (see lt_grad_f64_const_kernel): `acc` != null continues the
// sums of the flagged pixels that the launch before stored there
template <class M, bool INPLACE>
__global__ void __launch_bounds__(LT_THREADS, 2)
lt_grad_quads_f64_const_kernel(const LtTables<double>* __restrict__ tables, int n_lens,
                               typename LtSelect<INPLACE, int, const double2*>::type acc, double x_min, double y_min, double dx,
                               int nx, int quads_per_row, const unsigned int* __restrict__ list,
                               const LtWsHeader* __restrict__ hdr, const unsigned char* __restrict__ flags,
                               double2* __restrict__ out) {
  typedef typename M::template Rec<double>::type Rec;
  __shared__ LtTables<double> tab;
  lt_grid_dependency_wait();
  if (M::kTables) lt_copy16(&tab, tables, (int)(sizeof(tab) / 16));
  __syncthreads();
  const Rec* cl = reinterpret_cast<const Rec*>(lt_const_slot);
  const long long total = (long long)hdr->list_count;
  for (long long g = (long long)blockIdx.x * LT_THREADS + threadIdx.x; g < total; g += (long long)gridDim.x * LT_THREADS) {
    const unsigned int q = list[g];
    const int j = (int)(q / (unsigned int)quads_per_row);
    const int i0 = (int)(q - (unsigned int)j * (unsigned int)quads_per_row) * 4;
    const size_t p0 = (size_t)j * nx + (size_t)i0;
    const double t2 = __dadd_rn(y_min, __dmul_rn((double)j, dx));
    double t1[4], G1[4], G2[4];
    bool keep[4];
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      t1[p] = __dadd_rn(x_min, __dmul_rn((double)(i0 + p), dx));
      G1[p] = 0.0;
      G2[p] = 0.0;
      keep[p] = i0 + p < nx && flags[p0 + p] != 0;
      if (acc && keep[p]) {
        double2 v;
        if constexpr (INPLACE) v = out[p0 + p];
        else v = acc[p0 + p];
        G1[p] = v.x;
        G2[p] = v.y;
      }
    }
    lt_const_lens_loop<M>(cl, n_lens, t2, t1, tab, G1, G2);
#pragma unroll
    for (int p = 0; p < 4; ++p)
      if (keep[p]) out[p0 + p] = make_double2(G1[p], G2[p]);
  }
}

// ------------------------------------------------------------------------------------------------ short point lists
// The observed image positions of the chi^2 algorithm (step 1: "lens the observed images to the source plane"):
// a few hundred points against the whole catalogue.  One thread per point would leave the machine empty and run the N
// interactions of a point as one dependent chain, so here a warp owns a point: lane l sums the lenses l, l + 32, ... in
// catalogue order (two at a time, for two independent chains per lane) and the 32 partial sums are combined by a
// fixed butterfly.  Every term is the grid kernel's, bit for bit; the order of the sum is not, so the result differs
// from the grid kernel's by the rounding of the additions only.  The records are read from global memory (L1/L2: the
// catalogue is a few hundred KB at most), one record per lane.
#define LT_SPLIT_THREADS 128
template <class M>
__global__ void __launch_bounds__(LT_SPLIT_THREADS)
lt_grad_points_split_kernel(const typename M::template Rec<double>::type* __restrict__ lens,
                            const LtTables<double>* __restrict__ tables, int n_lens,
                            const double2* __restrict__ points, long long n_points, double2* __restrict__ out) {
  typedef typename M::template Rec<double>::type Rec;
  __shared__ LtTables<double> tab;
  lt_grid_dependency_wait();
  if (M::kTables) lt_copy16(&tab, tables, (int)(sizeof(tab) / 16));
  __syncthreads();
  const int lane = threadIdx.x & 31;
  constexpr int WARPS = LT_SPLIT_THREADS / 32;
  for (long long p = (long long)blockIdx.x * WARPS + (threadIdx.x >> 5); p < n_points; p += (long long)gridDim.x * WARPS) {
    const double2 pt = points[p];
    double A1 = 0.0, A2 = 0.0, B1 = 0.0, B2 = 0.0;
    int k = lane;
#pragma unroll 1
    for (; k + 32 < n_lens; k += 64) {
      const Rec La = lens[k], Lb = lens[k + 32];
      M::template interact_abs<double>(pt.x, M::template row_abs<double>(pt.y, La), La, tab, A1, A2);
      M::template interact_abs<double>(pt.x, M::template row_abs<double>(pt.y, Lb), Lb, tab, B1, B2);
    }
    if (k < n_lens) {
      const Rec La = lens[k];
      M::template interact_abs<double>(pt.x, M::template row_abs<double>(pt.y, La), La, tab, A1, A2);
    }
    double G1 = __dadd_rn(A1, B1), G2 = __dadd_rn(A2, B2);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      G1 = __dadd_rn(G1, __shfl_xor_sync(0xffffffffu, G1, o));
      G2 = __dadd_rn(G2, __shfl_xor_sync(0xffffffffu, G2, o));
    }
    if (lane == 0) out[p] = make_double2(G1, G2);
  }
}
