// lt_api.cu -- C ABI of liblt_gradient.so (include/lt_gradient.h): argument checks, workspace carving, launches.
// No torch types, no allocation, no synchronisation except where the header says so.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <string.h>

#include <atomic>
#include <map>
#include <mutex>
#include <tuple>
#include <utility>

#include "../../include/lt_gradient.h"
#include "lt_mixed.cuh"
#include "lt_images.cuh"
#include "lt_chi2.cuh"
#include "lt_audit.cuh"

static_assert(sizeof(lt_lens) == sizeof(LtRawLens), "lt_lens and LtRawLens must have the same layout");
static_assert(sizeof(lt_image_hit) == sizeof(LtImageHit) && sizeof(LtImageHit) == 32, "lt_image_hit layout");
static_assert(sizeof(lt_nfw_lens) == sizeof(LtRawNfw), "lt_nfw_lens and LtRawNfw must have the same layout");
static_assert(sizeof(lt_sie_lens) == sizeof(LtRawSie), "lt_sie_lens and LtRawSie must have the same layout");
static_assert(sizeof(LtSieLens<double>) == 48 && sizeof(LtSieLens<float>) == 32, "SIE record sizes");
template <class M> struct Rec64 { typedef typename M::template Rec<double>::type type; };
template <class M> struct Rec32 { typedef typename M::template Rec<float>::type type; };
static_assert(sizeof(LtLens<double>) == 128 && sizeof(LtLens<float>) == 64, "lens record sizes");
static_assert(LT_MAX_LENSES <= LT_BAD_SLOTS * LT_PRECOMPUTE_THREADS, "one bad-code slot per precompute block");

namespace {

thread_local int g_last_cuda_error = 0;

// lt_set_tuning's knobs: process-wide, each one an atomic int read with relaxed loads on the launch path, so a call
// that races lt_set_tuning sees every knob either old or new (the knobs are independent of one another)
struct Tuning {
  std::atomic<int> ppt64{0}, ppt32{0}, chunk64{0}, chunk32{0}, ctas_per_sm{0}, single_launch{0}, staged_host_output{0},
      points_per_thread{0}, no_dependent_launch{0}, plain_sp{0}, no_const_records{0};
};
Tuning g_tuning;
thread_local cudaEvent_t g_ev_start = nullptr, g_ev_stop = nullptr;   // lt_set_kernel_events
thread_local int g_launches = 0;                                      // kernels launched by the last entry-point call

constexpr int kDefaultChunk64 = 256;   // 32 KB of fp64 records per CTA
constexpr int kDefaultChunk32 = 1024;  // 64 KB of fp32 records per CTA
constexpr size_t kAlign = 256;
constexpr long long kSplitMaxPoints = 4096;   // lt_gradient_points: lists up to this length run one warp per point (measured crossover ~6000)

inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Layout {   // byte offsets into the workspace
  size_t header, bad, tab64, tab32, lens64, lens32, flags, sp, list, total;
};

Layout make_layout(int n_lens, long long n_pix, bool mixed) {   // dPIE record sizes (the larger) serve both models
  Layout L;
  size_t o = 0;
  L.header = o; o += sizeof(LtWsHeader);
  L.bad = o;    o += LT_BAD_SLOTS * sizeof(int);   /* directly behind the header: lt_last_status reads both in one copy */
  L.tab64 = o;  o += align_up(sizeof(LtTables<double>));
  L.tab32 = o;  o += align_up(sizeof(LtTables<float>));
  L.lens64 = o; o += align_up((size_t)n_lens * sizeof(LtLens<double>));
  L.lens32 = o; o += align_up((size_t)n_lens * sizeof(LtLens<float>));
  L.flags = o;  if (mixed) o += align_up((size_t)n_pix);
  L.sp = o;     if (mixed) o += align_up((size_t)n_pix * sizeof(float2));
  L.list = o;   if (mixed) o += align_up((size_t)n_pix * sizeof(unsigned int));
  L.total = o;
  return L;
}

bool sizes_ok(int n_lens, int nx, int ny) {
  if (n_lens < 0 || n_lens > LT_MAX_LENSES || nx < 1 || ny < 1) return false;
  return (long long)nx * (long long)ny < (1LL << 31);
}

int cuda_fail(cudaError_t e) {
  g_last_cuda_error = (int)e;
  return LT_ERR_CUDA;
}
#define LT_CUDA(call)                                   \
  do {                                                  \
    cudaError_t e_ = (call);                            \
    if (e_ != cudaSuccess) return cuda_fail(e_);        \
  } while (0)

struct DeviceInfo {
  int device = -1, sms = 0;
  size_t smem_optin = 0;
};
int device_info(DeviceInfo& d) {
  static thread_local DeviceInfo cache;
  int dev = 0;
  LT_CUDA(cudaGetDevice(&dev));
  if (cache.device != dev) {
    int sms = 0, smem = 0;
    LT_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    LT_CUDA(cudaDeviceGetAttribute(&smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    cache.device = dev;
    cache.sms = sms;
    cache.smem_optin = (size_t)smem;
  }
  d = cache;
  return LT_OK;
}

// Per-kernel facts, cached for the life of the process in maps that never evict (one entry per kernel instantiation and
// device; one per (kernel, device, dynamic shared memory) for the occupancy): the runtime queries cost microseconds on a
// path that launches sub-millisecond kernels.  The first use of a kernel opts it in ONCE to the largest dynamic shared
// memory it can ever be given (the device's opt-in limit minus the kernel's own static shared memory), so the attribute
// is never lowered and a launch from another host thread with a larger chunk cannot fail on it.
struct KernelInfo {
  size_t static_smem = 0, max_dynamic = 0;
};
std::mutex g_kernel_mu;
template <class K>
int kernel_info(K kernel, const DeviceInfo& d, KernelInfo& out) {
  static std::map<std::pair<const void*, int>, KernelInfo> cache;
  const std::pair<const void*, int> key(reinterpret_cast<const void*>(kernel), d.device);
  std::lock_guard<std::mutex> lock(g_kernel_mu);
  auto it = cache.find(key);
  if (it == cache.end()) {
    cudaFuncAttributes fa;
    LT_CUDA(cudaFuncGetAttributes(&fa, kernel));
    KernelInfo ki;
    ki.static_smem = fa.sharedSizeBytes;
    ki.max_dynamic = d.smem_optin > ki.static_smem ? d.smem_optin - ki.static_smem : 0;
    LT_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ki.max_dynamic));
    it = cache.emplace(key, ki).first;
  }
  out = it->second;
  return LT_OK;
}

// resident CTAs of `kernel` (CTAs of `threads` threads) on the whole device with `smem` bytes of dynamic shared memory
template <class K>
int resident_ctas(K kernel, size_t smem, const DeviceInfo& d, long long& resident, int threads = LT_THREADS) {
  KernelInfo ki;
  const int rc = kernel_info(kernel, d, ki);
  if (rc != LT_OK) return rc;
  if (smem > ki.max_dynamic) return cuda_fail(cudaErrorLaunchOutOfResources);
  static std::map<std::tuple<const void*, int, size_t>, int> cache;
  const std::tuple<const void*, int, size_t> key(reinterpret_cast<const void*>(kernel), d.device, smem);
  int occ = 0;
  {
    std::lock_guard<std::mutex> lock(g_kernel_mu);
    auto it = cache.find(key);
    if (it != cache.end()) occ = it->second;
  }
  if (occ == 0) {
    LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem));
    if (occ < 1) return cuda_fail(cudaErrorLaunchOutOfResources);
    std::lock_guard<std::mutex> lock(g_kernel_mu);
    cache[key] = occ;
  }
  const int cap = g_tuning.ctas_per_sm;
  if (cap > 0 && cap < occ) occ = cap;
  resident = (long long)occ * d.sms;
  return LT_OK;
}

// persistent grid: min(#work groups, resident CTAs)
template <class K>
int grid_for(K kernel, size_t smem, long long n_work, const DeviceInfo& d, int& grid, int threads = LT_THREADS) {
  long long g = 0;
  const int rc = resident_ctas(kernel, smem, d, g, threads);
  if (rc != LT_OK) return rc;
  if (g > n_work) g = n_work;
  if (g < 1) g = 1;
  grid = (int)g;
  return LT_OK;
}

// lenses per shared-memory chunk: the wanted number, clamped to the catalogue and to what fits beside the kernel's own
// static shared memory (the range-reduction tables) under the device's opt-in limit
template <class K>
int pick_chunk(K kernel, int n_lens, int wanted, size_t rec_bytes, const DeviceInfo& d, int& chunk) {
  KernelInfo ki;
  const int rc = kernel_info(kernel, d, ki);
  if (rc != LT_OK) return rc;
  chunk = wanted;
  const int max_chunk = (int)(ki.max_dynamic / rec_bytes);
  if (chunk > max_chunk) chunk = max_chunk;
  if (chunk > n_lens) chunk = n_lens;
  if (chunk < 1) chunk = 1;
  return LT_OK;
}

// pixels per thread: the largest of the candidates that still gives every SM about two tiles
int pick_ppt(int wanted, int max_ppt, int nx, int ny, const DeviceInfo& d) {
  if (wanted == 1 || wanted == 2 || wanted == 4) return wanted <= max_ppt ? wanted : max_ppt;
  int ppt = max_ppt;
  while (ppt > 1) {
    const long long tiles = (long long)((nx + 32 * ppt - 1) / (32 * ppt)) * ((ny + LT_TILE_H - 1) / LT_TILE_H);
    if (tiles >= 2LL * d.sms) break;
    ppt >>= 1;
  }
  return ppt;
}

// records the measurement-hook events around the dominant kernel's launch
struct KernelEvents {
  cudaStream_t st;
  bool on;
  explicit KernelEvents(cudaStream_t s, bool enable = true) : st(s), on(enable && g_ev_start && g_ev_stop) {
    if (on) cudaEventRecord(g_ev_start, st);
  }
  ~KernelEvents() {
    if (on) cudaEventRecord(g_ev_stop, st);
  }
};

// Launch of a grid kernel as a programmatic dependent of the kernel before it in the stream (lt_kernels.cuh: the
// kernel waits for that kernel itself before it reads anything).  lt_set_tuning's single_launch bit 3 switches the
// attribute off.
template <class... KArgs, class... Args>
cudaError_t launch_dependent(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)block);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = g_tuning.no_dependent_launch ? 0 : 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

struct GridArgs {
  int n_lens;
  double x_min, y_min, dx;
  int nx, ny;
  double2* staging = nullptr;   // device buffer of nx*ny double2 the host entry points own: where a map that goes straight
                                // into pinned host memory keeps its partial sums between launches (constant-bank records)
};

// Launch plan shared by the fp64 and fp32 grid kernels.  All tiles cost the same, so a persistent grid of R resident CTAs
// over n tiles runs ceil(n/R) waves and the last one may be nearly empty (config 1: 1024 tiles of 128 x 8 pixels on
// 296 CTAs = 3.46 waves).  Each launch therefore gets a whole number of waves of the row-major tile order and the
// ragged rest is handed to the next smaller pixels-per-thread variant (half the tile width, more resident CTAs), whose
// waves are proportionally shorter.  fn(ppt, tiles_x, begin, end, resident_or_null): query (resident != null) or launch.
template <class Fn>
int launch_waves(int ppt, const GridArgs& a, Fn fn) {
  const long long tiles_y = (a.ny + LT_TILE_H - 1) / LT_TILE_H;
  long long begin = 0;
  for (;;) {
    const int tiles_x = (a.nx + 32 * ppt - 1) / (32 * ppt);
    const long long n_tiles = tiles_x * tiles_y;
    long long end = n_tiles;
    if (ppt > 1 && !g_tuning.single_launch) {
      long long resident = 0;
      const int rc = fn(ppt, tiles_x, 0, 0, &resident);
      if (rc != LT_OK) return rc;
      const long long rest = n_tiles - begin;
      if (rest % resident != 0) end = begin + rest / resident * resident;
    }
    if (end > begin) {
      const int rc = fn(ppt, tiles_x, begin, end, nullptr);
      if (rc != LT_OK) return rc;
    }
    if (end == n_tiles) return LT_OK;
    const long long ty = end / tiles_x, tx = end % tiles_x;     // first tile of the rest, in the finer tiling
    ppt >>= 1;
    begin = ty * ((a.nx + 32 * ppt - 1) / (32 * ppt)) + 2 * tx;
  }
}

template <class M, int PPT, int MINB>
int launch_f64_ppt(const typename Rec64<M>::type* l64, const LtTables<double>* t64, const GridArgs& a, double2* out,
                   const DeviceInfo& d, cudaStream_t st, int tiles_x, long long begin, long long end, long long* resident) {
  int chunk = 1, grid = 1;
  const int wanted = g_tuning.chunk64;
  int rc = pick_chunk(lt_grad_f64_kernel<M, PPT, MINB>, a.n_lens, wanted > 0 ? wanted : kDefaultChunk64,
                      sizeof(typename Rec64<M>::type), d, chunk);
  if (rc != LT_OK) return rc;
  const size_t smem = (size_t)chunk * sizeof(typename Rec64<M>::type);
  if (resident) return resident_ctas(lt_grad_f64_kernel<M, PPT, MINB>, smem, d, *resident);
  rc = grid_for(lt_grad_f64_kernel<M, PPT, MINB>, smem, end - begin, d, grid);
  if (rc != LT_OK) return rc;
  LT_CUDA(launch_dependent(lt_grad_f64_kernel<M, PPT, MINB>, grid, LT_THREADS, smem, st, l64, t64, a.n_lens, chunk, a.x_min,
                           a.y_min, a.dx, a.nx, a.ny, tiles_x, (int)begin, (int)end, out));
  ++g_launches;
  return LT_OK;
}
// ---- lens records in the constant bank (lt_kernels.cuh: lt_grad_f64_const_kernel) --------------------------------------
// One slot of __constant__ memory per device (= per context: the library is one module).  Whoever launches a kernel that
// reads the slot holds `mu` while it enqueues: [wait for the slot's last reader if that was another stream] copy the
// records in (device to device, stream-ordered), launch, record `ev`.  Nothing blocks the host; two streams that both use
// the slot are ordered on it (two maps at once would not overlap anyway: each fills the GPU).
struct ConstSlot {
  std::mutex mu;
  cudaEvent_t ev = nullptr;
  cudaStream_t last = nullptr;
  bool used = false;
};
ConstSlot g_const_slot[64];

// May this call use the slot?  Not while the stream is being captured into a graph (a replay could not be ordered against
// other users of the slot), not when lt_set_tuning switched it off, not beyond 64 devices.  A catalogue that needs several
// slot-loads is accumulated over launches: in `out` if that is device memory, else in the caller's device staging buffer
// with only the last launch writing to `out` (a map that goes straight into pinned host memory crosses PCIe once).
bool const_records_ok(cudaStream_t st, const DeviceInfo& d, const void* out, const void* staging, int n_lens,
                      size_t rec_bytes) {
  if (g_tuning.no_const_records || d.device < 0 || d.device >= 64 || n_lens < 1) return false;
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
    (void)cudaGetLastError();
    return false;
  }
  if ((size_t)n_lens * rec_bytes > LT_CONST_SLOT_BYTES && !staging) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, out) != cudaSuccess || at.type != cudaMemoryTypeDevice) {
      (void)cudaGetLastError();
      return false;
    }
  }
  return true;
}

// fn(cnt, acc, dst): enqueue the kernel for the `cnt` records now in the slot, continuing the sums in `acc` (null: start
// from zero) and storing to `dst`
template <class Rec, class Fn>
int with_const_records(const Rec* d_records, int n_lens, const DeviceInfo& d, cudaStream_t st, double2* out, double2* staging,
                       Fn fn) {
  ConstSlot& slot = g_const_slot[d.device];
  std::lock_guard<std::mutex> lock(slot.mu);
  if (!slot.ev) LT_CUDA(cudaEventCreateWithFlags(&slot.ev, cudaEventDisableTiming));
  if (slot.used && slot.last != st) LT_CUDA(cudaStreamWaitEvent(st, slot.ev, 0));
  const int per = (int)(LT_CONST_SLOT_BYTES / sizeof(Rec));
  int rc = LT_OK;
  for (int base = 0; base < n_lens && rc == LT_OK; base += per) {
    const int cnt = n_lens - base < per ? n_lens - base : per;
    LT_CUDA(cudaMemcpyToSymbolAsync(lt_const_slot, d_records + base, (size_t)cnt * sizeof(Rec), 0, cudaMemcpyDeviceToDevice, st));
    // partial sums live in `between` (the staging buffer if there is one, else `out` itself); the last launch stores to `out`
    double2* between = staging ? staging : out;
    const bool last = base + cnt >= n_lens;
    rc = fn(cnt, base > 0 ? (const double2*)between : (const double2*)nullptr, last ? out : between);
  }
  LT_CUDA(cudaEventRecord(slot.ev, st));     // also after a failed launch: the copies are in the stream
  slot.last = st;
  slot.used = true;
  return rc;
}

// the 4-pixel main launch over tiles [begin, end) with the records in the constant bank
template <class M>
int launch_f64_const(const typename Rec64<M>::type* l64, const LtTables<double>* t64, const GridArgs& a, double2* out,
                     const DeviceInfo& d, cudaStream_t st, int tiles_x, long long begin, long long end, long long* resident) {
  if (resident) return resident_ctas(lt_grad_f64_const_kernel<M, true>, 0, d, *resident);
  int grid = 1;
  const int rc = grid_for(lt_grad_f64_const_kernel<M, true>, 0, end - begin, d, grid);
  if (rc != LT_OK) return rc;
  long long r2 = 0;   // (opts the second instantiation in; same resources)
  if (a.staging) {
    const int rc2 = resident_ctas(lt_grad_f64_const_kernel<M, false>, 0, d, r2);
    if (rc2 != LT_OK) return rc2;
  }
  return with_const_records(l64, a.n_lens, d, st, out, a.staging, [&](int cnt, const double2* acc, double2* dst) -> int {
    if (a.staging)      // partial sums in the staging buffer, the last launch stores to `out` (pinned host memory)
      LT_CUDA(launch_dependent(lt_grad_f64_const_kernel<M, false>, grid, LT_THREADS, 0, st, t64, cnt, acc, a.x_min, a.y_min,
                               a.dx, a.nx, a.ny, tiles_x, (int)begin, (int)end, dst));
    else                // in place
      LT_CUDA(launch_dependent(lt_grad_f64_const_kernel<M, true>, grid, LT_THREADS, 0, st, t64, cnt, acc ? 1 : 0, a.x_min,
                               a.y_min, a.dx, a.nx, a.ny, tiles_x, (int)begin, (int)end, dst));
    ++g_launches;
    return LT_OK;
  });
}

template <class M>
int launch_f64(const typename Rec64<M>::type* l64, const LtTables<double>* t64, const GridArgs& a, double2* out,
               const DeviceInfo& d, cudaStream_t st, bool hook = true) {
  // 4 pixels per thread (4 independent chains, lens record loaded once per 4 interactions) at <= 128 registers, two
  // CTAs per SM; fewer pixels per thread for the ragged rest and for grids too small to give every SM two tiles
  // The 4-pixel launch reads its records from the constant bank where it may (const_records_ok); the ragged rest and
  // small grids keep the shared-memory kernels (they loop over the whole catalogue in one launch, on tiles of their own).
  KernelEvents ke(st, hook);
  const bool cb = M::kConstRecords && const_records_ok(st, d, out, a.staging, a.n_lens, sizeof(typename Rec64<M>::type));
  return launch_waves(pick_ppt(g_tuning.ppt64, 4, a.nx, a.ny, d), a,
                      [&](int ppt, int tiles_x, long long b, long long e, long long* resident) {
                        switch (ppt) {
                          case 1: return launch_f64_ppt<M, 1, 4>(l64, t64, a, out, d, st, tiles_x, b, e, resident);
                          case 2: return launch_f64_ppt<M, 2, 3>(l64, t64, a, out, d, st, tiles_x, b, e, resident);
                          default:
                            if constexpr (M::kConstRecords) {
                              if (cb) return launch_f64_const<M>(l64, t64, a, out, d, st, tiles_x, b, e, resident);
                            }
                            return launch_f64_ppt<M, 4, 2>(l64, t64, a, out, d, st, tiles_x, b, e, resident);
                        }
                      });
}

template <class M, int PPT, int MINB, bool WIDE>
int launch_f32_ppt(const typename Rec64<M>::type* l64, const typename Rec32<M>::type* l32, const LtTables<float>* t32,
                   const GridArgs& a, float2* out, double2* out_wide, const DeviceInfo& d, cudaStream_t st,
                   int tiles_x, long long begin, long long end, long long* resident) {
  int chunk = 1, grid = 1;
  const int wanted = g_tuning.chunk32;
  int rc = pick_chunk(lt_grad_f32_kernel<M, PPT, MINB, WIDE>, a.n_lens, wanted > 0 ? wanted : kDefaultChunk32,
                      sizeof(typename Rec32<M>::type), d, chunk);
  if (rc != LT_OK) return rc;
  const size_t smem = (size_t)chunk * sizeof(typename Rec32<M>::type);
  if (resident) return resident_ctas(lt_grad_f32_kernel<M, PPT, MINB, WIDE>, smem, d, *resident);
  rc = grid_for(lt_grad_f32_kernel<M, PPT, MINB, WIDE>, smem, end - begin, d, grid);
  if (rc != LT_OK) return rc;
  LT_CUDA(launch_dependent(lt_grad_f32_kernel<M, PPT, MINB, WIDE>, grid, LT_THREADS, smem, st, l64, l32, t32, a.n_lens, chunk,
                           a.x_min, a.y_min, a.dx, a.nx, a.ny, tiles_x, (int)begin, (int)end, out, out_wide));
  ++g_launches;
  return LT_OK;
}
template <class M>
int launch_f32(const typename Rec64<M>::type* l64, const typename Rec32<M>::type* l32, const LtTables<float>* t32,
               const GridArgs& a,
               float2* out, const DeviceInfo& d, cudaStream_t st, bool hook = true, double2* out_wide = nullptr) {
  // 4 pixels per thread at <= 80 registers (3 CTAs per SM): with a tighter register budget the compiler reloads the
  // constants inside the loop and the kernel, which is bound by issue slots, loses 10 %
  KernelEvents ke(st, hook);
  return launch_waves(pick_ppt(g_tuning.ppt32, 4, a.nx, a.ny, d), a,
                      [&](int ppt, int tiles_x, long long b, long long e, long long* resident) {
                        if (out_wide) {      // mixed mode: the kernel variant that also stores the widened value
                          switch (ppt) {
                            case 1: return launch_f32_ppt<M, 1, 6, true>(l64, l32, t32, a, out, out_wide, d, st, tiles_x, b, e, resident);
                            case 2: return launch_f32_ppt<M, 2, 4, true>(l64, l32, t32, a, out, out_wide, d, st, tiles_x, b, e, resident);
                            default: return launch_f32_ppt<M, 4, 3, true>(l64, l32, t32, a, out, out_wide, d, st, tiles_x, b, e, resident);
                          }
                        }
                        switch (ppt) {
                          case 1: return launch_f32_ppt<M, 1, 6, false>(l64, l32, t32, a, out, out_wide, d, st, tiles_x, b, e, resident);
                          case 2: return launch_f32_ppt<M, 2, 4, false>(l64, l32, t32, a, out, out_wide, d, st, tiles_x, b, e, resident);
                          default: return launch_f32_ppt<M, 4, 3, false>(l64, l32, t32, a, out, out_wide, d, st, tiles_x, b, e, resident);
                        }
                      });
}

// the paper's plain SP version (lt_kernels.cuh): measurement variant selected by lt_set_tuning
template <class M>
int launch_f32_plain(const void* d_raw, const typename Rec64<M>::type* l64, const typename Rec32<M>::type* l32,
                     const LtTables<float>* t32, const GridArgs& a, float2* out, double2* out_wide, const DeviceInfo& d,
                     cudaStream_t st) {
  int chunk = 1, grid = 1;
  const long long n_pix = (long long)a.nx * a.ny;
  auto go = [&](auto kernel) -> int {
    int rc = pick_chunk(kernel, a.n_lens, kDefaultChunk32, sizeof(typename Rec32<M>::type), d, chunk);
    if (rc != LT_OK) return rc;
    const size_t smem = (size_t)chunk * sizeof(typename Rec32<M>::type);
    rc = grid_for(kernel, smem, (n_pix + LT_THREADS - 1) / LT_THREADS, d, grid);
    if (rc != LT_OK) return rc;
    LT_CUDA(launch_dependent(kernel, grid, LT_THREADS, smem, st, reinterpret_cast<const typename M::Raw*>(d_raw), l64, l32, t32,
                             a.n_lens, chunk, a.x_min, a.y_min, a.dx, a.nx, a.ny, out, out_wide));
    ++g_launches;
    return LT_OK;
  };
  return out_wide ? go(lt_grad_f32_plain_kernel<M, true>) : go(lt_grad_f32_plain_kernel<M, false>);
}

// a9: the fp64 pass of the mixed mode over the quad list (count known on the device only: the grid is sized for the
// worst case, all quads listed, and CTAs beyond the count leave at once)
template <class M>
int launch_quads(const typename Rec64<M>::type* l64, const LtTables<double>* t64, const GridArgs& a, int quads_per_row,
                 const unsigned int* list, const LtWsHeader* hdr, const unsigned char* flags, double2* out,
                 const DeviceInfo& d, cudaStream_t st) {
  const long long n_quads_all = (long long)quads_per_row * a.ny;
  if constexpr (M::kConstRecords) {
    if (const_records_ok(st, d, out, a.staging, a.n_lens, sizeof(typename Rec64<M>::type))) {
      int grid_c = 1;
      const int rc_c = grid_for(lt_grad_quads_f64_const_kernel<M, true>, 0, (n_quads_all + LT_THREADS - 1) / LT_THREADS, d, grid_c);
      if (rc_c != LT_OK) return rc_c;
      long long r2 = 0;
      if (a.staging) {
        const int rc2 = resident_ctas(lt_grad_quads_f64_const_kernel<M, false>, 0, d, r2);
        if (rc2 != LT_OK) return rc2;
      }
      KernelEvents ke(st);
      return with_const_records(l64, a.n_lens, d, st, out, a.staging, [&](int cnt, const double2* acc, double2* dst) -> int {
        if (a.staging)
          LT_CUDA(launch_dependent(lt_grad_quads_f64_const_kernel<M, false>, grid_c, LT_THREADS, 0, st, t64, cnt, acc, a.x_min,
                                   a.y_min, a.dx, a.nx, quads_per_row, list, hdr, flags, dst));
        else
          LT_CUDA(launch_dependent(lt_grad_quads_f64_const_kernel<M, true>, grid_c, LT_THREADS, 0, st, t64, cnt, acc ? 1 : 0,
                                   a.x_min, a.y_min, a.dx, a.nx, quads_per_row, list, hdr, flags, dst));
        ++g_launches;
        return LT_OK;
      });
    }
  }
  int chunk = 1, grid = 1;
  const int wanted = g_tuning.chunk64;
  int rc = pick_chunk(lt_grad_quads_f64_kernel<M>, a.n_lens, wanted > 0 ? wanted : kDefaultChunk64,
                      sizeof(typename Rec64<M>::type), d, chunk);
  if (rc != LT_OK) return rc;
  const size_t smem = (size_t)chunk * sizeof(typename Rec64<M>::type);
  const long long n_quads = (long long)quads_per_row * a.ny;
  rc = grid_for(lt_grad_quads_f64_kernel<M>, smem, (n_quads + LT_THREADS - 1) / LT_THREADS, d, grid);
  if (rc != LT_OK) return rc;
  KernelEvents ke(st);
  LT_CUDA(launch_dependent(lt_grad_quads_f64_kernel<M>, grid, LT_THREADS, smem, st, l64, t64, a.n_lens, chunk, a.x_min,
                           a.y_min, a.dx, a.nx, quads_per_row, list, hdr, flags, out));
  ++g_launches;
  return LT_OK;
}

template <class M>
int launch_points(const typename Rec64<M>::type* l64, const LtTables<double>* t64, int n_lens, const double2* points,
                  long long n_points, double2* out, const DeviceInfo& d, cudaStream_t st) {
  int chunk = 1, grid = 1;
  const int wanted = g_tuning.chunk64;
  int rc = pick_chunk(lt_grad_points_f64_kernel<M>, n_lens, wanted > 0 ? wanted : kDefaultChunk64,
                      sizeof(typename Rec64<M>::type), d, chunk);
  if (rc != LT_OK) return rc;
  const size_t smem = (size_t)chunk * sizeof(typename Rec64<M>::type);
  rc = grid_for(lt_grad_points_f64_kernel<M>, smem, (n_points + LT_THREADS - 1) / LT_THREADS, d, grid);
  if (rc != LT_OK) return rc;
  LT_CUDA(launch_dependent(lt_grad_points_f64_kernel<M>, grid, LT_THREADS, smem, st, l64, t64, n_lens, chunk, points,
                           n_points, out));
  ++g_launches;
  return LT_OK;
}

int check_mixed(const lt_mixed_params& m) {
  const bool ok = isfinite(m.m_max) && m.m_max > 0 && isfinite(m.c28) && m.c28 >= 0 &&
                  isfinite(m.patch_halfwidth_cluster) && m.patch_halfwidth_cluster >= 0 &&
                  isfinite(m.patch_halfwidth_galaxy) && m.patch_halfwidth_galaxy >= 0 &&
                  !isnan(m.b0_cluster_threshold);
  return ok ? LT_OK : LT_ERR_BAD_MIXED_PARAMS;
}

template <class M>
int precompute(const void* d_lenses, int n_lens, double dx, unsigned char* ws, const Layout& L, cudaStream_t st) {
  const int blocks = (n_lens > 0 ? (n_lens + LT_PRECOMPUTE_THREADS - 1) / LT_PRECOMPUTE_THREADS : 1) +
                     (M::kTables ? LT_TABLE_BLOCKS : 0);
  lt_precompute_kernel<M><<<blocks, LT_PRECOMPUTE_THREADS, 0, st>>>(reinterpret_cast<const typename M::Raw*>(d_lenses), n_lens, dx,
                                               reinterpret_cast<typename Rec64<M>::type*>(ws + L.lens64),
                                               reinterpret_cast<typename Rec32<M>::type*>(ws + L.lens32),
                                               reinterpret_cast<LtTables<double>*>(ws + L.tab64),
                                               reinterpret_cast<LtTables<float>*>(ws + L.tab32),
                                               reinterpret_cast<LtWsHeader*>(ws + L.header),
                                               reinterpret_cast<int*>(ws + L.bad));
  LT_CUDA(cudaGetLastError());
  ++g_launches;
  return LT_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ peak probes
// Dependent-free FMA chains (8 independent accumulators per thread) to confirm the FP64 / FP32 pipe peaks in the same
// run as the bench (peak convention of the paper's Table 1: 2 ops x clock x lanes).
__device__ double lt_probe_sink64;
__device__ float lt_probe_sink32;

template <class T>
__global__ void __launch_bounds__(256) lt_probe_kernel(int iters, T seed) {
  T a0 = seed + (T)threadIdx.x, a1 = a0 + (T)1, a2 = a0 + (T)2, a3 = a0 + (T)3, a4 = a0 + (T)4, a5 = a0 + (T)5,
    a6 = a0 + (T)6, a7 = a0 + (T)7;
  const T m = (T)0.999999, c = (T)1e-6;
  for (int it = 0; it < iters; ++it) {
    a0 = lt_fma(a0, m, c); a1 = lt_fma(a1, m, c); a2 = lt_fma(a2, m, c); a3 = lt_fma(a3, m, c);
    a4 = lt_fma(a4, m, c); a5 = lt_fma(a5, m, c); a6 = lt_fma(a6, m, c); a7 = lt_fma(a7, m, c);
  }
  const T s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (s == (T)-12345.678) {   // never true: keeps the chains alive without a store on the timed path
    if (sizeof(T) == 8) lt_probe_sink64 = (double)s; else lt_probe_sink32 = (float)s;
  }
}

// the same with packed pairs (FFMA2): two results per instruction; which = 2 of lt_peak_probe
__global__ void __launch_bounds__(256) lt_probe_kernel_x2(int iters, float seed) {
  float2 a[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = make_float2(seed + (float)threadIdx.x + (float)i, seed - (float)i);
  const float2 m = make_float2(0.999999f, 0.999999f), c = make_float2(1e-6f, 1e-6f);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = __ffma2_rn(a[i], m, c);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i].x + a[i].y;
  if (s == -12345.678f) lt_probe_sink32 = s;
}

// Register-file read rate (which = 3, 4 of lt_peak_probe): the same chains with THREE distinct register sources per
// instruction, a[i] = fma(a[i], b[i], c[i]).  On B200 an FP64 (or packed FP32) instruction whose sources are three distinct
// 64-bit register pairs holds its pipe for 3 cycles instead of 2 -- the register file delivers two 32-bit source reads per
// lane and cycle -- which is what the kernels of lt_math.cuh are written around.
template <class T2, class T>
__global__ void __launch_bounds__(256) lt_probe_kernel_3src(int iters, T seed) {
  T2 a[8], b[8], c[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const T l = (T)(threadIdx.x + 1);          // every operand differs from lane to lane: nothing moves to uniform registers
    a[i] = T2{seed + l + (T)i, seed - l - (T)i};
    b[i] = T2{(T)0.999999 + (T)1e-9 * (l + (T)i), (T)0.999998 + (T)1e-9 * (l - (T)i)};
    c[i] = T2{(T)1e-6 * (l + (T)(2 * i)), (T)2e-6 * (l + (T)(3 * i))};
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if constexpr (sizeof(T) == 8) { a[i].x = fma(a[i].x, b[i].x, c[i].x); a[i].y = fma(a[i].y, b[i].y, c[i].y); }
      else a[i] = __ffma2_rn(a[i], b[i], c[i]);
    }
  }
  T s = (T)0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i].x + a[i].y;
  if (s == (T)-12345.678) {
    if (sizeof(T) == 8) lt_probe_sink64 = (double)s; else lt_probe_sink32 = (float)s;
  }
}

// ------------------------------------------------------------------------------------------------ entry points, per lens model
namespace {

template <class M>
int gradient_grid_impl(const void* d_lenses, int n_lens, double x_min, double y_min, double dx, int nx, int ny,
                     lt_precision mode, const lt_mixed_params* mixed_or_null, void* d_out_grad, void* d_workspace,
                     size_t workspace_bytes, void* cuda_stream, void* d_staging = nullptr) {
  if (!sizes_ok(n_lens, nx, ny)) return LT_ERR_BAD_SIZE;
  if (mode != LT_FP64 && mode != LT_FP32 && mode != LT_MIXED) return LT_ERR_BAD_MODE;
  if (!d_out_grad || !d_workspace || (n_lens > 0 && !d_lenses)) return LT_ERR_NULL_POINTER;
  if (!(isfinite(x_min) && isfinite(y_min) && isfinite(dx)) || !(dx > 0.0)) return LT_ERR_BAD_GRID;
  if (((uintptr_t)d_out_grad & 15) || ((uintptr_t)d_workspace & 15)) return LT_ERR_MISALIGNED;
  const long long n_pix = (long long)nx * ny;
  const Layout L = make_layout(n_lens, n_pix, mode == LT_MIXED);
  if (workspace_bytes < L.total) return LT_ERR_WORKSPACE_TOO_SMALL;
  lt_mixed_params mp;
  lt_mixed_defaults(&mp);
  if (mode == LT_MIXED && mixed_or_null) {
    mp = *mixed_or_null;
    const int rc = check_mixed(mp);
    if (rc != LT_OK) return rc;
  }
  DeviceInfo dev;
  int rc = device_info(dev);
  if (rc != LT_OK) return rc;
  g_launches = 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  unsigned char* ws = (unsigned char*)d_workspace;
  LtWsHeader* hdr = reinterpret_cast<LtWsHeader*>(ws + L.header);
  const typename Rec64<M>::type* l64 = reinterpret_cast<const typename Rec64<M>::type*>(ws + L.lens64);
  const typename Rec32<M>::type* l32 = reinterpret_cast<const typename Rec32<M>::type*>(ws + L.lens32);
  const LtTables<double>* t64 = reinterpret_cast<const LtTables<double>*>(ws + L.tab64);
  const LtTables<float>* t32 = reinterpret_cast<const LtTables<float>*>(ws + L.tab32);
  GridArgs a{n_lens, x_min, y_min, dx, nx, ny};
  if (mode != LT_FP32) a.staging = reinterpret_cast<double2*>(d_staging);

  if (mode == LT_MIXED)   /* the flag map is cleared before the first kernel so that the kernels follow one another */
    LT_CUDA(cudaMemsetAsync(ws + L.flags, 0, (size_t)n_pix, st));
  {
    // measurement hook (lt_set_kernel_events): in the fp64 and fp32 modes the pair of events brackets the precompute
    // kernel too -- the grid kernel is its programmatic dependent, an event between the two would serialise them
    KernelEvents ke(st, mode != LT_MIXED);
    rc = precompute<M>(d_lenses, n_lens, dx, ws, L, st);                                   /* a1 */
    if (rc != LT_OK) return rc;
    if (mode == LT_FP64) return launch_f64<M>(l64, t64, a, (double2*)d_out_grad, dev, st, /*hook=*/false);   /* a2-a7 */
    if (mode == LT_FP32) {
      if (g_tuning.plain_sp) return launch_f32_plain<M>(d_lenses, l64, l32, t32, a, (float2*)d_out_grad, nullptr, dev, st);
      return launch_f32<M>(l64, l32, t32, a, (float2*)d_out_grad, dev, st, /*hook=*/false);
    }
  }

  /* LT_MIXED: single precision everywhere, flag, double precision on the flagged pixels */
  unsigned char* flags = ws + L.flags;
  float2* sp = reinterpret_cast<float2*>(ws + L.sp);
  unsigned int* list = reinterpret_cast<unsigned int*>(ws + L.list);
  LtMixedDev md;
  md.fdx = (float)dx;
  md.t25 = (float)(dx / mp.m_max);
  md.t28 = (float)(mp.c28 * dx);
  md.h_cluster = mp.patch_halfwidth_cluster;
  md.h_galaxy = mp.patch_halfwidth_galaxy;
  md.b0_cluster = mp.b0_cluster_threshold;
  if (n_lens > 0) {
    LT_CUDA(launch_dependent(lt_patch_kernel<M>, n_lens * LT_PATCH_SPLIT, 256, 0, st, reinterpret_cast<const typename M::Raw*>(d_lenses), n_lens,
                             x_min, y_min, dx, nx, ny, md, flags));
    ++g_launches;
  }
  rc = g_tuning.plain_sp ? launch_f32_plain<M>(d_lenses, l64, l32, t32, a, sp, (double2*)d_out_grad, dev, st)
                         : launch_f32<M>(l64, l32, t32, a, sp, dev, st, /*hook=*/false, (double2*)d_out_grad);
  if (rc != LT_OK) return rc;
  {
    long long blocks = (n_pix + LT_FLAG_PPI * 256 - 1) / (LT_FLAG_PPI * 256);
    const long long cap = (long long)dev.sms * 8;
    if (blocks > cap) blocks = cap;
    LT_CUDA(launch_dependent(lt_flag_kernel, (int)blocks, 256, 0, st, sp, nx, ny, md, flags, hdr));   /* a8 */
    ++g_launches;
  }
  const int quads_per_row = (nx + 3) / 4;
  {
    long long blocks = ((long long)quads_per_row * ny + LT_QUADS_PER_THREAD * 256 - 1) / (LT_QUADS_PER_THREAD * 256);
    const long long cap = (long long)dev.sms * 8;
    if (blocks > cap) blocks = cap;
    LT_CUDA(launch_dependent(lt_quad_list_kernel, (int)blocks, 256, 0, st, (const unsigned char*)flags, nx, ny, quads_per_row,
                             list, hdr));
    ++g_launches;
  }
  return launch_quads<M>(l64, t64, a, quads_per_row, list, hdr, flags, (double2*)d_out_grad, dev, st);        /* a9 */
}

template <class M>
int gradient_points_impl(const void* d_lenses, int n_lens, const double* d_points, long long n_points,
                       double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!sizes_ok(n_lens, 1, 1) || n_points < 0) return LT_ERR_BAD_SIZE;
  if (!d_workspace || (n_lens > 0 && !d_lenses) || (n_points > 0 && (!d_points || !d_out))) return LT_ERR_NULL_POINTER;
  if (((uintptr_t)d_out & 15) || ((uintptr_t)d_points & 15) || ((uintptr_t)d_workspace & 15)) return LT_ERR_MISALIGNED;
  const Layout L = make_layout(n_lens, 1, false);
  if (workspace_bytes < L.total) return LT_ERR_WORKSPACE_TOO_SMALL;
  DeviceInfo dev;
  int rc = device_info(dev);
  if (rc != LT_OK) return rc;
  g_launches = 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  unsigned char* ws = (unsigned char*)d_workspace;
  rc = precompute<M>(d_lenses, n_lens, 1.0, ws, L, st);
  if (rc != LT_OK || n_points == 0) return rc;
  const GridArgs a{n_lens, 0.0, 0.0, 1.0, 1, 1};
  if (n_points <= kSplitMaxPoints && !g_tuning.points_per_thread) {   /* short list: one warp per point */
    int grid = 1;
    constexpr int per_cta = LT_SPLIT_THREADS / 32;
    rc = grid_for(lt_grad_points_split_kernel<M>, 0, (n_points + per_cta - 1) / per_cta, dev, grid, LT_SPLIT_THREADS);
    if (rc != LT_OK) return rc;
    LT_CUDA(launch_dependent(lt_grad_points_split_kernel<M>, grid, LT_SPLIT_THREADS, 0, st,
                             reinterpret_cast<const typename Rec64<M>::type*>(ws + L.lens64),
                             reinterpret_cast<const LtTables<double>*>(ws + L.tab64), n_lens,
                             reinterpret_cast<const double2*>(d_points), n_points, reinterpret_cast<double2*>(d_out)));
    ++g_launches;
    return LT_OK;
  }
  return launch_points<M>(reinterpret_cast<const typename Rec64<M>::type*>(ws + L.lens64),
                          reinterpret_cast<const LtTables<double>*>(ws + L.tab64), n_lens,
                          reinterpret_cast<const double2*>(d_points), n_points, reinterpret_cast<double2*>(d_out), dev, st);
}

template <class M>
int gradient_grid_host_impl(const void* h_lenses, int n_lens, double x_min, double y_min, double dx, int nx, int ny,
                          lt_precision mode, const lt_mixed_params* mixed_or_null, void* h_out_grad,
                          void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!sizes_ok(n_lens, nx, ny)) return LT_ERR_BAD_SIZE;
  if (mode != LT_FP64 && mode != LT_FP32 && mode != LT_MIXED) return LT_ERR_BAD_MODE;
  if (!h_out_grad || !d_workspace || (n_lens > 0 && !h_lenses)) return LT_ERR_NULL_POINTER;
  if ((uintptr_t)d_workspace & 15) return LT_ERR_MISALIGNED;
  if (workspace_bytes < lt_host_workspace_bytes(n_lens, nx, ny, mode)) return LT_ERR_WORKSPACE_TOO_SMALL;
  const size_t w = align_up(lt_workspace_bytes(n_lens, nx, ny, mode));
  const size_t lens_bytes = (size_t)n_lens * sizeof(typename M::Raw);
  const size_t elem = (mode == LT_FP32) ? sizeof(float2) : sizeof(double2);
  unsigned char* ws = (unsigned char*)d_workspace;
  void* d_lenses = ws + w;
  void* d_out = ws + w + align_up(lens_bytes);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // A pinned catalogue (a few KB) is read by the precompute kernel straight from host memory: one PCIe read instead of
  // a copy-engine operation in front of the first kernel.  Pageable catalogues are copied.
  const void* d_cat = d_lenses;
  bool cat_direct = false;
  if (n_lens > 0 && !g_tuning.staged_host_output) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, h_lenses) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer) {
      d_cat = at.devicePointer;
      cat_direct = true;
    } else {
      (void)cudaGetLastError();
    }
  }
  if (n_lens > 0 && !cat_direct) LT_CUDA(cudaMemcpyAsync(d_lenses, h_lenses, lens_bytes, cudaMemcpyHostToDevice, st));
  // A pinned (page-locked, hence device-mapped under UVA) output buffer is written by the gradient kernel itself: its
  // warp-wide 512 B / 256 B stores go straight over PCIe while the kernel computes, instead of a device-to-host copy of
  // the whole map after it (in LT_MIXED the fp32 pass stores the widened value of every pixel and the fp64 pass
  // overwrites the flagged ones, both while computing).  Not for pageable memory.
  void* d_direct = nullptr;
  if (!g_tuning.staged_host_output) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, h_out_grad) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer &&
        ((uintptr_t)at.devicePointer & 15) == 0)
      d_direct = at.devicePointer;
    else
      (void)cudaGetLastError();
  }
  const int rc = gradient_grid_impl<M>(d_cat, n_lens, x_min, y_min, dx, nx, ny, mode, mixed_or_null,
                                       d_direct ? d_direct : d_out, ws, w, st, d_direct ? d_out : nullptr);
  if (rc != LT_OK) return rc;
  if (!d_direct) LT_CUDA(cudaMemcpyAsync(h_out_grad, d_out, (size_t)nx * ny * elem, cudaMemcpyDeviceToHost, st));
  return LT_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ C ABI
extern "C" {

int lt_version(void) { return LT_VERSION; }

const char* lt_error_string(int code) {
  switch (code) {
    case LT_OK: return "ok";
    case LT_ERR_NULL_POINTER: return "null pointer";
    case LT_ERR_BAD_SIZE: return "bad size (n_lens, nx, ny or n_points out of range)";
    case LT_ERR_BAD_GRID: return "bad grid (dx <= 0 or non-finite x_min / y_min / dx)";
    case LT_ERR_BAD_MODE: return "unknown precision mode";
    case LT_ERR_WORKSPACE_TOO_SMALL: return "workspace too small (see lt_workspace_bytes)";
    case LT_ERR_MISALIGNED: return "buffer not 16-byte aligned";
    case LT_ERR_BAD_MIXED_PARAMS: return "bad mixed-rule parameters";
    case LT_ERR_CUDA: return "CUDA runtime error (see lt_last_cuda_error)";
    case LT_ERR_BAD_LENS_PARAMS: return "lens parameters outside the domain (e in [0,1), 0 < rcore < rcut, finite)";
    case LT_ERR_NOALLOC_TOO_LARGE: return "catalogue larger than the built-in scratch of lt_gradient_grid_noalloc (LT_NOALLOC_MAX_LENSES)";
  }
  return "unknown error code";
}

int lt_last_cuda_error(void) { return g_last_cuda_error; }

void lt_mixed_defaults(lt_mixed_params* out) {
  if (!out) return;
  out->m_max = 3.26;
  out->c28 = 0.0104 / 0.03;                /* eq. 28 P:321 over the paper's pixel size P:301 */
  out->patch_halfwidth_cluster = 6.0;      /* 400/2 px * 0.03" */
  out->patch_halfwidth_galaxy = 0.3;       /*  20/2 px * 0.03" */
  out->b0_cluster_threshold = 15.0;        /* R15 */
}

int lt_last_launch_count(void) { return g_launches; }

int lt_set_tuning(int ppt64, int ppt32, int chunk64, int chunk32, int ctas_per_sm, int single_launch) {
  if (ppt64 < 0 || ppt32 < 0 || chunk64 < 0 || chunk32 < 0 || ctas_per_sm < 0 || single_launch < 0) return LT_ERR_BAD_SIZE;
  g_tuning.single_launch = single_launch & 1;
  g_tuning.staged_host_output = (single_launch >> 1) & 1;
  g_tuning.points_per_thread = (single_launch >> 2) & 1;
  g_tuning.no_dependent_launch = (single_launch >> 3) & 1;
  g_tuning.plain_sp = (single_launch >> 4) & 1;
  g_tuning.no_const_records = (single_launch >> 5) & 1;
  g_tuning.ppt64 = ppt64;
  g_tuning.ppt32 = ppt32;
  g_tuning.chunk64 = chunk64;
  g_tuning.chunk32 = chunk32;
  g_tuning.ctas_per_sm = ctas_per_sm;
  return LT_OK;
}

int lt_set_kernel_events(void* ev_start, void* ev_stop) {
  if ((ev_start == nullptr) != (ev_stop == nullptr)) return LT_ERR_NULL_POINTER;
  g_ev_start = (cudaEvent_t)ev_start;
  g_ev_stop = (cudaEvent_t)ev_stop;
  return LT_OK;
}

size_t lt_workspace_bytes(int n_lens, int nx, int ny, lt_precision mode) {
  if (!sizes_ok(n_lens, nx, ny)) return 0;
  if (mode != LT_FP64 && mode != LT_FP32 && mode != LT_MIXED) return 0;
  return make_layout(n_lens, (long long)nx * ny, mode == LT_MIXED).total;
}

size_t lt_host_workspace_bytes(int n_lens, int nx, int ny, lt_precision mode) {
  const size_t w = lt_workspace_bytes(n_lens, nx, ny, mode);
  if (w == 0) return 0;
  const size_t elem = (mode == LT_FP32) ? sizeof(float2) : sizeof(double2);
  return align_up(w) + align_up((size_t)n_lens * sizeof(lt_lens)) + align_up((size_t)nx * ny * elem);
}

int lt_gradient_grid(const lt_lens* d_lenses, int n_lens, double x_min, double y_min, double dx, int nx, int ny,
                     lt_precision mode, const lt_mixed_params* mixed_or_null, void* d_out_grad, void* d_workspace,
                     size_t workspace_bytes, void* cuda_stream) {
  return gradient_grid_impl<LtDpieModel>(d_lenses, n_lens, x_min, y_min, dx, nx, ny, mode, mixed_or_null, d_out_grad,
                                         d_workspace, workspace_bytes, cuda_stream);
}
int lt_gradient_grid_sie(const lt_sie_lens* d_lenses, int n_lens, double x_min, double y_min, double dx, int nx, int ny,
                         lt_precision mode, const lt_mixed_params* mixed_or_null, void* d_out_grad, void* d_workspace,
                         size_t workspace_bytes, void* cuda_stream) {
  return gradient_grid_impl<LtSieModel>(d_lenses, n_lens, x_min, y_min, dx, nx, ny, mode, mixed_or_null, d_out_grad,
                                        d_workspace, workspace_bytes, cuda_stream);
}

int lt_gradient_grid_nfw(const lt_nfw_lens* d_lenses, int n_lens, double x_min, double y_min, double dx, int nx, int ny,
                         lt_precision mode, const lt_mixed_params* mixed_or_null, void* d_out_grad, void* d_workspace,
                         size_t workspace_bytes, void* cuda_stream) {
  return gradient_grid_impl<LtNfwModel>(d_lenses, n_lens, x_min, y_min, dx, nx, ny, mode, mixed_or_null, d_out_grad,
                                        d_workspace, workspace_bytes, cuda_stream);
}
int lt_gradient_points_nfw(const lt_nfw_lens* d_lenses, int n_lens, const double* d_points, long long n_points,
                           double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  return gradient_points_impl<LtNfwModel>(d_lenses, n_lens, d_points, n_points, d_out, d_workspace, workspace_bytes,
                                          cuda_stream);
}
int lt_gradient_grid_nfw_host(const lt_nfw_lens* h_lenses, int n_lens, double x_min, double y_min, double dx, int nx,
                              int ny, lt_precision mode, const lt_mixed_params* mixed_or_null, void* h_out_grad,
                              void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  return gradient_grid_host_impl<LtNfwModel>(h_lenses, n_lens, x_min, y_min, dx, nx, ny, mode, mixed_or_null,
                                             h_out_grad, d_workspace, workspace_bytes, cuda_stream);
}

int lt_gradient_points(const lt_lens* d_lenses, int n_lens, const double* d_points, long long n_points,
                       double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  return gradient_points_impl<LtDpieModel>(d_lenses, n_lens, d_points, n_points, d_out, d_workspace, workspace_bytes,
                                           cuda_stream);
}
int lt_gradient_points_sie(const lt_sie_lens* d_lenses, int n_lens, const double* d_points, long long n_points,
                           double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  return gradient_points_impl<LtSieModel>(d_lenses, n_lens, d_points, n_points, d_out, d_workspace, workspace_bytes,
                                          cuda_stream);
}

int lt_gradient_grid_host(const lt_lens* h_lenses, int n_lens, double x_min, double y_min, double dx, int nx, int ny,
                          lt_precision mode, const lt_mixed_params* mixed_or_null, void* h_out_grad,
                          void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  return gradient_grid_host_impl<LtDpieModel>(h_lenses, n_lens, x_min, y_min, dx, nx, ny, mode, mixed_or_null,
                                              h_out_grad, d_workspace, workspace_bytes, cuda_stream);
}
int lt_gradient_grid_sie_host(const lt_sie_lens* h_lenses, int n_lens, double x_min, double y_min, double dx, int nx,
                              int ny, lt_precision mode, const lt_mixed_params* mixed_or_null, void* h_out_grad,
                              void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  return gradient_grid_host_impl<LtSieModel>(h_lenses, n_lens, x_min, y_min, dx, nx, ny, mode, mixed_or_null,
                                             h_out_grad, d_workspace, workspace_bytes, cuda_stream);
}

int lt_mixed_rule(const float* d_sp_map, double x_min, double y_min, double dx, int nx, int ny, const double* d_centres,
                  int n_centres, const lt_mixed_params* mixed_or_null, unsigned char* d_flags, void* d_workspace,
                  size_t workspace_bytes, void* cuda_stream) {
  if (!sizes_ok(n_centres, nx, ny)) return LT_ERR_BAD_SIZE;
  if (!d_sp_map || !d_flags || !d_workspace || (n_centres > 0 && !d_centres)) return LT_ERR_NULL_POINTER;
  if (!(isfinite(x_min) && isfinite(y_min) && isfinite(dx)) || !(dx > 0.0)) return LT_ERR_BAD_GRID;
  if (((uintptr_t)d_sp_map & 7) || ((uintptr_t)d_workspace & 15)) return LT_ERR_MISALIGNED;
  const long long n_pix = (long long)nx * ny;
  const Layout L = make_layout(0, n_pix, true);
  if (workspace_bytes < L.total) return LT_ERR_WORKSPACE_TOO_SMALL;
  lt_mixed_params mp;
  lt_mixed_defaults(&mp);
  if (mixed_or_null) {
    mp = *mixed_or_null;
    const int rc = check_mixed(mp);
    if (rc != LT_OK) return rc;
  }
  DeviceInfo dev;
  const int rc = device_info(dev);
  if (rc != LT_OK) return rc;
  g_launches = 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  unsigned char* ws = (unsigned char*)d_workspace;
  LT_CUDA(cudaMemsetAsync(ws + L.header, 0, sizeof(LtWsHeader), st));
  LT_CUDA(cudaMemsetAsync(d_flags, 0, (size_t)n_pix, st));
  LtMixedDev md;
  md.fdx = (float)dx;
  md.t25 = (float)(dx / mp.m_max);
  md.t28 = (float)(mp.c28 * dx);
  md.h_cluster = mp.patch_halfwidth_cluster;
  md.h_galaxy = mp.patch_halfwidth_galaxy;
  md.b0_cluster = mp.b0_cluster_threshold;
  if (n_centres > 0) {
    lt_patch_kernel<LtCentreModel><<<n_centres * LT_PATCH_SPLIT, 256, 0, st>>>(reinterpret_cast<const LtCentre*>(d_centres), n_centres,
                                                              x_min, y_min, dx, nx, ny, md, d_flags);
    LT_CUDA(cudaGetLastError());
    ++g_launches;
  }
  long long blocks = (n_pix + LT_FLAG_PPI * 256 - 1) / (LT_FLAG_PPI * 256);
  const long long cap = (long long)dev.sms * 8;
  if (blocks > cap) blocks = cap;
  lt_flag_kernel<<<(int)blocks, 256, 0, st>>>(reinterpret_cast<const float2*>(d_sp_map), nx, ny, md, d_flags,
                                              reinterpret_cast<LtWsHeader*>(ws + L.header));
  LT_CUDA(cudaGetLastError());
  ++g_launches;
  return LT_OK;
}

int lt_find_images(const double* d_grad, double x_min, double y_min, double dx, int nx, int ny, double dls_dos,
                   const double* d_sources, int n_sources, lt_image_hit* d_hits, int max_hits, int* d_n_hits,
                   void* cuda_stream) {
  if (nx < 2 || ny < 2 || (long long)nx * ny >= (1LL << 31) || n_sources < 0 || n_sources > LT_MAX_SOURCES ||
      max_hits < 0)
    return LT_ERR_BAD_SIZE;
  if (!d_grad || !d_n_hits || (n_sources > 0 && !d_sources) || (max_hits > 0 && !d_hits)) return LT_ERR_NULL_POINTER;
  if (!(isfinite(x_min) && isfinite(y_min) && isfinite(dx) && isfinite(dls_dos)) || !(dx > 0.0)) return LT_ERR_BAD_GRID;
  if (((uintptr_t)d_grad & 15) || ((uintptr_t)d_sources & 15) || ((uintptr_t)d_hits & 7)) return LT_ERR_MISALIGNED;
  DeviceInfo dev;
  const int rc = device_info(dev);
  if (rc != LT_OK) return rc;
  g_launches = 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LT_CUDA(cudaMemsetAsync(d_n_hits, 0, sizeof(int), st));
  if (n_sources == 0) return LT_OK;
  const int n_strips = (nx - 1 + LT_FI_STRIP - 1) / LT_FI_STRIP, n_row_blocks = (ny - 1 + LT_FI_BLOCK_ROWS - 1) / LT_FI_BLOCK_ROWS;
  const long long n_items = (long long)n_strips * n_row_blocks;            // one warp each
  int grid = 1;
  const int rc2 = grid_for(lt_find_images_kernel, 0, (n_items + 7) / 8, dev, grid, 256);
  if (rc2 != LT_OK) return rc2;
  KernelEvents ke(st);
  lt_find_images_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const double2*>(d_grad), x_min, y_min, dx, nx, ny,
                                              dls_dos, reinterpret_cast<const double2*>(d_sources), n_sources,
                                              n_strips, (int)n_items, reinterpret_cast<LtImageHit*>(d_hits), max_hits,
                                              d_n_hits);
  LT_CUDA(cudaGetLastError());
  ++g_launches;
  return LT_OK;
}

int lt_source_barycentres(const double* d_theta, const double* d_alpha, const int* d_offsets, int n_systems,
                          double dls_dos, double* d_barycentres, void* cuda_stream) {
  if (n_systems < 0 || n_systems > LT_MAX_SOURCES) return LT_ERR_BAD_SIZE;
  if (n_systems == 0) return LT_OK;
  if (!d_theta || !d_alpha || !d_offsets || !d_barycentres) return LT_ERR_NULL_POINTER;
  if (!isfinite(dls_dos)) return LT_ERR_BAD_GRID;
  if (((uintptr_t)d_theta & 15) || ((uintptr_t)d_alpha & 15) || ((uintptr_t)d_barycentres & 15) || ((uintptr_t)d_offsets & 3))
    return LT_ERR_MISALIGNED;
  g_launches = 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  lt_source_barycentres_kernel<<<(n_systems + 127) / 128, 128, 0, st>>>(
      reinterpret_cast<const double2*>(d_theta), reinterpret_cast<const double2*>(d_alpha), d_offsets, n_systems, dls_dos,
      reinterpret_cast<double2*>(d_barycentres));
  LT_CUDA(cudaGetLastError());
  ++g_launches;
  return LT_OK;
}

int lt_chi2(const double* d_theta_obs, const double* d_sigma, const int* d_offsets, int n_systems, int n_images,
            const lt_image_hit* d_hits, const int* d_n_hits, int max_hits, double* d_terms, lt_chi2_result* d_result,
            void* cuda_stream) {
  static_assert(sizeof(lt_chi2_result) == sizeof(LtChi2Result) && sizeof(lt_chi2_result) == 32, "lt_chi2_result layout");
  if (n_systems < 0 || n_systems > LT_MAX_SOURCES || n_images < 0 || n_images > (1 << 24) || max_hits < 0)
    return LT_ERR_BAD_SIZE;
  if (!d_result || !d_n_hits || (max_hits > 0 && !d_hits) ||
      (n_images > 0 && (!d_theta_obs || !d_sigma || !d_offsets || !d_terms)))
    return LT_ERR_NULL_POINTER;
  if (n_images > 0 && n_systems == 0) return LT_ERR_BAD_SIZE;
  if (((uintptr_t)d_theta_obs & 15) || ((uintptr_t)d_sigma & 7) || ((uintptr_t)d_terms & 7) || ((uintptr_t)d_hits & 7) ||
      ((uintptr_t)d_result & 7) || ((uintptr_t)d_offsets & 3))
    return LT_ERR_MISALIGNED;
  g_launches = 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (n_images > 0) {
    lt_chi2_terms_kernel<<<(n_images + 127) / 128, 128, 0, st>>>(
        reinterpret_cast<const double2*>(d_theta_obs), d_sigma, d_offsets, n_systems, n_images,
        reinterpret_cast<const LtImageHit*>(d_hits), d_n_hits, max_hits, d_terms);
    LT_CUDA(cudaGetLastError());
    ++g_launches;
  }
  lt_chi2_sum_kernel<<<1, 32, 0, st>>>(d_terms, n_images, reinterpret_cast<LtChi2Result*>(d_result));
  LT_CUDA(cudaGetLastError());
  ++g_launches;
  return LT_OK;
}

int lt_last_status(const void* d_workspace, void* cuda_stream, int* bad_lens_or_null) {
  if (!d_workspace) return LT_ERR_NULL_POINTER;
  struct { LtWsHeader h; int bad[LT_BAD_SLOTS]; } w;   /* make_layout: the slots follow the header */
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LT_CUDA(cudaMemcpyAsync(&w, d_workspace, sizeof(w), cudaMemcpyDeviceToHost, st));
  LT_CUDA(cudaStreamSynchronize(st));
  int bad_code = 0;
  for (int b = 0; b < w.h.bad_blocks && b < LT_BAD_SLOTS; ++b) bad_code = w.bad[b] > bad_code ? w.bad[b] : bad_code;
  if (bad_lens_or_null) *bad_lens_or_null = bad_code > 0 ? w.h.n_lens - bad_code : -1;
  return bad_code > 0 ? LT_ERR_BAD_LENS_PARAMS : LT_OK;
}

int lt_mixed_last_stats(const void* d_workspace, void* cuda_stream, lt_mixed_stats* out) {
  if (!d_workspace || !out) return LT_ERR_NULL_POINTER;
  LtWsHeader h;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LT_CUDA(cudaMemcpyAsync(&h, d_workspace, sizeof(h), cudaMemcpyDeviceToHost, st));
  LT_CUDA(cudaStreamSynchronize(st));
  out->n_pixels = -1;          /* not recorded in the header: the caller knows nx*ny */
  out->n_flagged = (long long)h.n_flagged;
  out->n_patch = (long long)h.n_patch;
  out->n_eq25 = (long long)h.n_eq25;
  out->n_eq28 = (long long)h.n_eq28;
  return LT_OK;
}

int lt_mixed_last_flags(const void* d_workspace, int n_lens, int nx, int ny, unsigned char* d_flags_out,
                        void* cuda_stream) {
  if (!d_workspace || !d_flags_out) return LT_ERR_NULL_POINTER;
  if (!sizes_ok(n_lens, nx, ny)) return LT_ERR_BAD_SIZE;
  const Layout L = make_layout(n_lens, (long long)nx * ny, true);
  LT_CUDA(cudaMemcpyAsync(d_flags_out, (const unsigned char*)d_workspace + L.flags, (size_t)nx * ny,
                          cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
  return LT_OK;
}

int lt_mixed_last_sp_map(const void* d_workspace, int n_lens, int nx, int ny, float* d_sp_out, void* cuda_stream) {
  if (!d_workspace || !d_sp_out) return LT_ERR_NULL_POINTER;
  if (!sizes_ok(n_lens, nx, ny)) return LT_ERR_BAD_SIZE;
  const Layout L = make_layout(n_lens, (long long)nx * ny, true);
  LT_CUDA(cudaMemcpyAsync(d_sp_out, (const unsigned char*)d_workspace + L.sp, (size_t)nx * ny * sizeof(float2),
                          cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
  return LT_OK;
}

int lt_rule_audit(const float* d_sp_map, const double* d_dp_map, double x_min, double y_min, double dx, int nx, int ny,
                  const double* d_centres, int n_centres, const unsigned char* d_flags, unsigned char* d_violation,
                  lt_audit_result* d_result, void* cuda_stream) {
  static_assert(sizeof(lt_audit_result) == sizeof(LtAuditResult), "lt_audit_result layout");
  if (!sizes_ok(0, nx, ny) || n_centres < 0) return LT_ERR_BAD_SIZE;
  if (!d_sp_map || !d_dp_map || !d_result || (n_centres > 0 && !d_centres)) return LT_ERR_NULL_POINTER;
  if (!(isfinite(x_min) && isfinite(y_min) && isfinite(dx)) || !(dx > 0.0)) return LT_ERR_BAD_GRID;
  if (((uintptr_t)d_sp_map & 7) || ((uintptr_t)d_dp_map & 15) || ((uintptr_t)d_result & 7) || ((uintptr_t)d_centres & 7))
    return LT_ERR_MISALIGNED;
  DeviceInfo dev;
  const int rc = device_info(dev);
  if (rc != LT_OK) return rc;
  g_launches = 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LT_CUDA(cudaMemsetAsync(d_result, 0, sizeof(lt_audit_result), st));
  const long long n_pix = (long long)nx * ny;
  long long blocks = (n_pix + 255) / 256;
  if (blocks > (long long)dev.sms * 8) blocks = (long long)dev.sms * 8;
  lt_rule_audit_kernel<<<(int)blocks, 256, 0, st>>>(reinterpret_cast<const float2*>(d_sp_map),
                                                    reinterpret_cast<const double2*>(d_dp_map), x_min, y_min, dx, nx, ny,
                                                    d_centres, n_centres, d_flags, d_violation,
                                                    reinterpret_cast<LtAuditResult*>(d_result));
  LT_CUDA(cudaGetLastError());
  ++g_launches;
  return LT_OK;
}

int lt_rule_audit_result(const lt_audit_result* d_result, double dx, void* cuda_stream, lt_audit_result* h_out) {
  if (!d_result || !h_out) return LT_ERR_NULL_POINTER;
  if (!(dx > 0.0)) return LT_ERR_BAD_GRID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LT_CUDA(cudaMemcpyAsync(h_out, d_result, sizeof(lt_audit_result), cudaMemcpyDeviceToHost, st));
  LT_CUDA(cudaStreamSynchronize(st));
  h_out->implied_m_max = dx / 4.0 / h_out->max_err;
  h_out->implied_m_max_outside_patch = dx / 4.0 / h_out->max_err_outside_patch;
  return LT_OK;
}

// ------------------------------------------------------------------------------------------------ no-allocation entry point
// For callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc): lt_gradient_grid for LT_FP64 / LT_FP32 with the workspace -- the scratch the precompute kernel
// writes (header, domain-check slots, range-reduction tables, packed fp64 / fp32 records) and the grid kernels read --
// in a file-scope device array instead of a caller-allocated buffer.  LT_NOALLOC_SCRATCH_BYTES (800 KiB) per GPU that
// loads the library, held until exit.  In host code `lt_noalloc_scratch` is a host-side stand-in, not a device address:
// its device address is taken once per device with cudaGetSymbolAddress (that device current) and passed to the kernels.
static __device__ __align__(256) unsigned char lt_noalloc_scratch[LT_NOALLOC_SCRATCH_BYTES];

namespace {
std::mutex g_noalloc_mu;
void* g_noalloc_ptr[64] = {};

// device address of the scratch array on the current device (set up on first use, per device)
int noalloc_scratch(const DeviceInfo& d, unsigned char** out) {
  if (d.device < 0 || d.device >= 64) return LT_ERR_BAD_SIZE;
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[d.device]) {
    void* p = nullptr;
    LT_CUDA(cudaGetSymbolAddress(&p, lt_noalloc_scratch));
    if (!p) return cuda_fail(cudaErrorInvalidSymbol);
    g_noalloc_ptr[d.device] = p;
  }
  *out = (unsigned char*)g_noalloc_ptr[d.device];
  return LT_OK;
}
}  // namespace

int lt_gradient_grid_noalloc(const lt_lens* d_lenses, int n_lens, double x_min, double y_min, double dx, int nx, int ny,
                             lt_precision mode, void* d_out_grad, void* cuda_stream) {
  typedef LtDpieModel M;
  if (!sizes_ok(n_lens, nx, ny)) return LT_ERR_BAD_SIZE;
  if (mode != LT_FP64 && mode != LT_FP32) return LT_ERR_BAD_MODE;      /* mixed scratch grows with the map: not here */
  if (n_lens > LT_NOALLOC_MAX_LENSES) return LT_ERR_NOALLOC_TOO_LARGE;
  if (!d_out_grad || (n_lens > 0 && !d_lenses)) return LT_ERR_NULL_POINTER;
  if (!(isfinite(x_min) && isfinite(y_min) && isfinite(dx)) || !(dx > 0.0)) return LT_ERR_BAD_GRID;
  if ((uintptr_t)d_out_grad & 15) return LT_ERR_MISALIGNED;
  const Layout L = make_layout(n_lens, (long long)nx * ny, false);
  if (L.total > (size_t)LT_NOALLOC_SCRATCH_BYTES) return LT_ERR_NOALLOC_TOO_LARGE;
  DeviceInfo dev;
  int rc = device_info(dev);
  if (rc != LT_OK) return rc;
  unsigned char* ws = nullptr;
  rc = noalloc_scratch(dev, &ws);
  if (rc != LT_OK) return rc;
  g_launches = 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const Rec64<M>::type* l64 = reinterpret_cast<const Rec64<M>::type*>(ws + L.lens64);
  const Rec32<M>::type* l32 = reinterpret_cast<const Rec32<M>::type*>(ws + L.lens32);
  const LtTables<double>* t64 = reinterpret_cast<const LtTables<double>*>(ws + L.tab64);
  const LtTables<float>* t32 = reinterpret_cast<const LtTables<float>*>(ws + L.tab32);
  const GridArgs a{n_lens, x_min, y_min, dx, nx, ny};
  /* Nothing of the last call's contents is read before it is rewritten: the precompute kernel initialises the header and
   * the domain-check slots of this call with plain stores and writes every record and table entry the grid kernels read. */
  rc = precompute<M>(d_lenses, n_lens, dx, ws, L, st);                                       /* a1 */
  if (rc != LT_OK) return rc;
  if (mode == LT_FP32) return launch_f32<M>(l64, l32, t32, a, (float2*)d_out_grad, dev, st, /*hook=*/false);
  /* fp64: the shared-memory grid kernels at every pixels-per-thread (the constant-bank variant of lt_gradient_grid
   * creates an event on its first use; same operations in the same order, identical bits) */
  return launch_waves(pick_ppt(g_tuning.ppt64, 4, a.nx, a.ny, dev), a,
                      [&](int ppt, int tiles_x, long long b, long long e, long long* resident) {
                        switch (ppt) {
                          case 1: return launch_f64_ppt<M, 1, 4>(l64, t64, a, (double2*)d_out_grad, dev, st, tiles_x, b, e, resident);
                          case 2: return launch_f64_ppt<M, 2, 3>(l64, t64, a, (double2*)d_out_grad, dev, st, tiles_x, b, e, resident);
                          default: return launch_f64_ppt<M, 4, 2>(l64, t64, a, (double2*)d_out_grad, dev, st, tiles_x, b, e, resident);
                        }
                      });
}

int lt_noalloc_last_status(void* cuda_stream, int* bad_lens_or_null) {
  DeviceInfo dev;
  int rc = device_info(dev);
  if (rc != LT_OK) return rc;
  unsigned char* ws = nullptr;
  rc = noalloc_scratch(dev, &ws);
  if (rc != LT_OK) return rc;
  return lt_last_status(ws, cuda_stream, bad_lens_or_null);
}

int lt_peak_probe(int which, int iters, double* flops_out, void* cuda_stream) {
  if (!flops_out) return LT_ERR_NULL_POINTER;
  if (which < 0 || which > 4 || iters < 1) return LT_ERR_BAD_SIZE;
  DeviceInfo dev;
  const int rc = device_info(dev);
  if (rc != LT_OK) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaEvent_t e0, e1;
  LT_CUDA(cudaEventCreate(&e0));
  LT_CUDA(cudaEventCreate(&e1));
  const int grid = dev.sms * 8;
  for (int rep = 0; rep < 2; ++rep) {      /* first pass warms up */
    LT_CUDA(cudaEventRecord(e0, st));
    if (which == 0) lt_probe_kernel<double><<<grid, 256, 0, st>>>(iters, 1.0);
    else if (which == 1) lt_probe_kernel<float><<<grid, 256, 0, st>>>(iters, 1.0f);
    else if (which == 2) lt_probe_kernel_x2<<<grid, 256, 0, st>>>(iters, 1.0f);
    else if (which == 3) lt_probe_kernel_3src<double2, double><<<grid, 256, 0, st>>>(iters, 1.0);
    else lt_probe_kernel_3src<float2, float><<<grid, 256, 0, st>>>(iters, 1.0f);
    LT_CUDA(cudaGetLastError());
    LT_CUDA(cudaEventRecord(e1, st));
    LT_CUDA(cudaEventSynchronize(e1));
  }
  float ms = 0.f;
  LT_CUDA(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *flops_out = (which >= 2 ? 2.0 : 1.0) * 2.0 * 8.0 * (double)iters * 256.0 * (double)grid / ((double)ms * 1e-3);
  return LT_OK;
}

}  // extern "C"
