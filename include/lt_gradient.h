/*
 * lt_gradient.h -- C ABI of liblt_gradient.so: the lensing-potential gradient (deflection-angle) map of
 * arXiv 1902.03252 on a regular pixel grid, summed over N dPIE/PIEMD lenses, on one B200 (sm_100a).
 *
 * Operation (P:n = PAPER.md line n):
 *   For every pixel theta = (x_min + i*dx, y_min + j*dx), 0 <= i < nx, 0 <= j < ny:
 *     gradPsi(theta) = sum_k Rot(+Phi_k) g_k( Rot(-Phi_k) (theta - theta_center,k) )
 *   -- Algorithm 1, P:191-226 (translate l.3-4, rotate l.5-6, body l.7-9, rotate back l.10-11, sum l.13-14;
 *   superposition eq. 14-15).  The per-lens body g_k is the dPIE deflection named by
 *   BASELINE.json:north_star (the paper's own body is the SIE, eq. 21; dPIE is named at P:385):
 *   PIEMD deflection at rcore minus PIEMD deflection at rcut, times b0*rcut/(rcut-rcore), i.e. the gradient of the
 *   potential whose convergence is kappa = (b0/2) rcut/(rcut-rcore) [1/sqrt(rcore^2+rho^2) - 1/sqrt(rcut^2+rho^2)],
 *   rho^2 = x'^2/(1+e)^2 + y'^2/(1-e)^2 in the lens frame (alpha = grad psi, laplace psi = 2 kappa: eq. 2-4).
 *   Mixed precision: section 3.2-3.3 and section 4: single precision everywhere, then double
 *   precision inside centre patches and wherever the critical-line criteria eq. 25 / eq. 28
 *   on the neighbour differences eq. 24 / 27 fire.  Thresholds scale with dx (R11-R16).
 *
 * Conventions
 *   - All pointers named d_* are DEVICE pointers (cudaMalloc / torch CUDA tensors); h_* are HOST pointers.
 *   - Ownership: the caller owns every buffer.  The library never allocates or frees device memory, never
 *     synchronises the stream (except the calls marked "synchronises"), and enqueues all work on `cuda_stream`
 *     (a cudaStream_t passed as void*; NULL = the legacy default stream).
 *   - Output layout: d_out_grad[2*(j*nx+i) + c], c = 0 -> dPsi/dtheta_1, c = 1 -> dPsi/dtheta_2; x (i) fastest.
 *     Element type: double for LT_FP64 and LT_MIXED (reading R17), float for LT_FP32.  Must be 16-byte aligned.
 *   - Lens parameters are fp64 in all modes; the per-lens precompute kernel derives the fp32 copies.
 *   - Errors: every int-returning entry point returns LT_OK (0) or a negative lt_status; nothing throws or aborts.
 *     Parameter-domain violations (e outside [0,1), rcore <= 0, rcut <= rcore, non-finite) are detected on the
 *     device by the precompute kernel: the offending lens contributes NaN and lt_last_status() reports it.
 *   - n_lens == 0 gives a zero map.  Limits: 0 <= n_lens <= LT_MAX_LENSES, 1 <= nx, ny, nx*ny < 2^31.
 */
#ifndef LT_GRADIENT_H
#define LT_GRADIENT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LT_VERSION 100
#define LT_MAX_LENSES 65536
#define LT_MAX_SOURCES 65536

typedef struct {              /* one dPIE lens; fp64; lengths in arcsec, angle in radians                         */
  double x, y;                /* centre theta_center (Alg. 1 Require)                                      */
  double ellipticity;         /* e in [0,1): enters rho^2 = x'^2/(1+e)^2 + y'^2/(1-e)^2 (reading R1)              */
  double angle;               /* Phi: counter-clockwise angle from the theta_1 axis to the major axis     */
  double rcore, rcut;         /* 0 < rcore < rcut                                                                 */
  double b0;                  /* deflection scale (eq. 22 P:183 for its SIS meaning)                              */
} lt_lens;

typedef struct {              /* one SIE lens: the paper's own body, Algorithm 1; fp64                */
  double x, y;                /* centre theta_center (Alg. 1 Require)                                      */
  double epsilon;             /* pseudo-ellipticity of the potential, eq. 17-18; |epsilon| < 1        */
  double angle;               /* Phi: counter-clockwise angle from the theta_1 axis to the semi-major axis */
  double b0;                  /* eq. 22, arcsec                                                           */
} lt_sie_lens;

typedef struct {              /* one pseudo-elliptical NFW lens (named by the paper at P:385); fp64                 */
  double x, y;                /* centre theta_center                                                               */
  double epsilon;             /* pseudo-ellipticity of the potential, eq. 17-18; |epsilon| < 1        */
  double angle;               /* Phi: counter-clockwise angle from the theta_1 axis to the semi-major axis */
  double kappa_s;             /* characteristic convergence rho_s rs / Sigma_crit, >= 0                           */
  double rs;                  /* scale radius, arcsec, > 0                                                        */
} lt_nfw_lens;

typedef enum { LT_FP64 = 0, LT_FP32 = 1, LT_MIXED = 2 } lt_precision;

typedef enum {
  LT_OK = 0,
  LT_ERR_NULL_POINTER = -1,
  LT_ERR_BAD_SIZE = -2,        /* n_lens < 0 or > LT_MAX_LENSES, nx/ny < 1, nx*ny >= 2^31                        */
  LT_ERR_BAD_GRID = -3,        /* dx <= 0 or non-finite x_min / y_min / dx                                       */
  LT_ERR_BAD_MODE = -4,
  LT_ERR_WORKSPACE_TOO_SMALL = -5,
  LT_ERR_MISALIGNED = -6,      /* d_out_grad or d_workspace not 16-byte aligned                                  */
  LT_ERR_BAD_MIXED_PARAMS = -7,
  LT_ERR_CUDA = -8,            /* a launch or runtime call failed; lt_last_cuda_error() has the cudaError_t      */
  LT_ERR_BAD_LENS_PARAMS = -9, /* reported by lt_last_status only (device-side domain check)                     */
  LT_ERR_NOALLOC_TOO_LARGE = -10 /* lt_gradient_grid_noalloc: n_lens > LT_NOALLOC_MAX_LENSES                       */
} lt_status;

typedef struct {               /* mixed-rule constants; lt_mixed_defaults() gives the paper's values             */
  double m_max;                /* 3.26: eq. 25 fires when |dx - delta_{1,2}| < dx/m_max (R11)            */
  double c28;                  /* 0.0104/0.03 (eq. 28): fires when |delta_{3,4}| > c28*dx (R11)           */
  double patch_halfwidth_cluster;   /* 6.0 arcsec = 400/2 px * 0.03" (R14)                                */
  double patch_halfwidth_galaxy;    /* 0.3 arcsec =  20/2 px * 0.03"                                             */
  double b0_cluster_threshold;      /* lenses with b0 >= this are cluster-scale (15 arcsec, R15)                 */
} lt_mixed_params;

typedef struct {               /* one predicted image found by lt_find_images (32 bytes)                            */
  int source;                  /* index into d_sources                                                              */
  int cell;                    /* j*nx + i of the cell's lower-left node (i, j)                                     */
  int triangle;                /* 0: nodes (i,j), (i+1,j), (i,j+1);  1: nodes (i+1,j+1), (i,j+1), (i+1,j)           */
  int reserved;
  double x, y;                 /* image-plane position with the barycentric coordinates of the source point        */
} lt_image_hit;

typedef struct {               /* written by lt_chi2 (device memory, 32 bytes)                                    */
  double chi2;                 /* eq. 11 over the observed images that have a predicted counterpart               */
  long long n_matched;         /* observed images with a term in the sum                                          */
  long long n_unmatched;       /* observed images whose system has no predicted image (left out of the sum)       */
  long long reserved;
} lt_chi2_result;

typedef struct {               /* filled by lt_mixed_last_stats */
  long long n_pixels;          /* -1: not recorded (the caller knows nx*ny)                                      */
  long long n_flagged;         /* pixels that carry double precision values = patch OR eq.25 OR eq.28             */
  long long n_patch, n_eq25, n_eq28;   /* pixels with the respective bit set (not exclusive)                     */
} lt_mixed_stats;

int lt_version(void);
const char* lt_error_string(int code);
int lt_last_cuda_error(void);                      /* cudaError_t of the last LT_ERR_CUDA on this thread        */
void lt_mixed_defaults(lt_mixed_params* out);

/* Bytes of device scratch lt_gradient_grid needs for these sizes (monotone in every argument).  0 on bad sizes. */
size_t lt_workspace_bytes(int n_lens, int nx, int ny, lt_precision mode);

/*
 * The hot path.  Enqueues on cuda_stream: the per-lens precompute kernel, the gradient kernel
 * (a2-a7) in the requested precision and, for LT_MIXED, the patch/flag/compaction kernels (a8) and the fp64
 * recompute of the flagged pixels (a9; done in row quads -- four neighbouring pixels of a row that hold a flagged pixel are
 * recomputed together, only the flagged ones are stored).  Asynchronous; returns after the launches.
 *   d_lenses       device, n_lens lt_lens structs (= a contiguous [n_lens,7] fp64 array); read only
 *   mixed_or_null  host pointer; NULL = lt_mixed_defaults; ignored unless mode == LT_MIXED
 *   d_out_grad     device, nx*ny*2 elements (type per mode, see above); fully overwritten
 *   d_workspace    device, >= lt_workspace_bytes(...) bytes, 16-byte aligned; contents undefined afterwards except
 *                  what the *_last_* calls below read.  One workspace must not be shared by concurrent calls.
 */
int lt_gradient_grid(const lt_lens* d_lenses, int n_lens,
                     double x_min, double y_min, double dx, int nx, int ny,
                     lt_precision mode, const lt_mixed_params* mixed_or_null,
                     void* d_out_grad, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The same hot path with the paper's own lens body, the SIE of Algorithm 1: per lens
 *   x' = D1 cos Phi + D2 sin Phi, y' = D2 cos Phi - D1 sin Phi (l.5-6), R = sqrt(x'^2 (1-eps) + y'^2 (1+eps)) (l.7),
 *   g = b0 ((1-eps) x', (1+eps) y') / R (l.8-9, eq. 21), rotated back by -Phi (l.10-11) and summed (l.13-14).
 * A pixel exactly on a lens centre (R = 0) receives nothing from that lens (reading R5).  Arguments, modes, output
 * layout, workspace (lt_workspace_bytes / lt_host_workspace_bytes of the same sizes serve both lens models), status
 * and mixed-rule calls exactly as for lt_gradient_grid; the mixed rule's constants are the paper's own at dx = 0.03".
 * Domain: |epsilon| < 1, everything finite (checked on the device like the dPIE parameters).
 */
int lt_gradient_grid_sie(const lt_sie_lens* d_lenses, int n_lens,
                         double x_min, double y_min, double dx, int nx, int ny,
                         lt_precision mode, const lt_mixed_params* mixed_or_null,
                         void* d_out_grad, void* d_workspace, size_t workspace_bytes, void* cuda_stream);
int lt_gradient_points_sie(const lt_sie_lens* d_lenses, int n_lens, const double* d_points, long long n_points,
                           double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream);
int lt_gradient_grid_sie_host(const lt_sie_lens* h_lenses, int n_lens,
                              double x_min, double y_min, double dx, int nx, int ny,
                              lt_precision mode, const lt_mixed_params* mixed_or_null,
                              void* h_out_grad, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The same hot path for pseudo-elliptical NFW lenses, the generalisation the paper names at P:385:
 * the paper's recipe for any circular profile, eq. 16-20: R = sqrt(x'^2 (1-eps) + y'^2 (1+eps)),
 * g = |alpha(R)| ((1-eps) x', (1+eps) y') / R, with the circular NFW deflection (x = R/rs)
 *   |alpha(R)| = 4 kappa_s rs [ln(x/2) + F(x)] / x,  F = arccosh(1/x)/sqrt(1-x^2) (x<1), 1 (x=1), arccos(1/x)/sqrt(x^2-1) (x>1),
 * rotated back and summed as in Algorithm 1.  A pixel exactly on a centre receives nothing from that lens.  Arguments,
 * modes, workspace, status and mixed-rule calls exactly as for lt_gradient_grid (the rule's cluster / galaxy classes use
 * the scale 4 kappa_s rs in place of b0).  Domain: |epsilon| < 1, kappa_s >= 0, rs > 0, everything finite.
 */
int lt_gradient_grid_nfw(const lt_nfw_lens* d_lenses, int n_lens,
                         double x_min, double y_min, double dx, int nx, int ny,
                         lt_precision mode, const lt_mixed_params* mixed_or_null,
                         void* d_out_grad, void* d_workspace, size_t workspace_bytes, void* cuda_stream);
int lt_gradient_points_nfw(const lt_nfw_lens* d_lenses, int n_lens, const double* d_points, long long n_points,
                           double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream);
int lt_gradient_grid_nfw_host(const lt_nfw_lens* h_lenses, int n_lens,
                              double x_min, double y_min, double dx, int nx, int ny,
                              lt_precision mode, const lt_mixed_params* mixed_or_null,
                              void* h_out_grad, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Gradient at an arbitrary list of points (the per-lens arithmetic of a3-a6 exposed; used for sampled parity at full size and for
 * image positions).  d_points: n_points*2 doubles (theta_1, theta_2 interleaved); d_out: n_points*2 doubles.
 * fp64 only.  Same workspace rule with nx = ny = 1.  Lists of more than 4096 points run one thread per point and return,
 * for a point that is a grid node, the bits of lt_gradient_grid's LT_FP64 map.  Shorter lists (the image positions of
 * the chi^2 algorithm) run one warp per point, the lenses dealt to the lanes: the same terms, added in another
 * order, so the result differs from the grid kernel's by the rounding of the sum (a few ulp of the largest term);
 * it does not depend on the length of the list below that limit.  lt_set_tuning's single_launch bit 2 forces the
 * thread-per-point kernel for every length.
 */
int lt_gradient_points(const lt_lens* d_lenses, int n_lens, const double* d_points, long long n_points,
                       double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The same call with HOST buffers (the end-to-end path of bench.py's `e2e` figure): enqueues, on cuda_stream, the
 * host->device copy of the n_lens lens structs from h_lenses, lt_gradient_grid, and the device->host copy of the
 * whole map into h_out_grad (nx*ny*2 elements, type per mode).  Asynchronous with respect to the host only if both
 * host buffers are pinned; the caller synchronises cuda_stream before reading h_out_grad.  If h_out_grad is pinned
 * (cudaHostAlloc / cudaHostRegister, 16-byte aligned) the kernels store the map into it directly over PCIe while they
 * compute (LT_MIXED: every pixel by the fp32 pass, flagged pixels again by the fp64 pass), and no separate
 * device-to-host copy is enqueued.  The device staging
 * buffers for the catalogue and the map are carved from d_workspace, which must hold
 * lt_host_workspace_bytes(n_lens, nx, ny, mode) bytes (>= lt_workspace_bytes; 0 on bad sizes).
 */
size_t lt_host_workspace_bytes(int n_lens, int nx, int ny, lt_precision mode);
int lt_gradient_grid_host(const lt_lens* h_lenses, int n_lens,
                          double x_min, double y_min, double dx, int nx, int ny,
                          lt_precision mode, const lt_mixed_params* mixed_or_null,
                          void* h_out_grad, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The mixed rule alone (section 3.2-3.3, eq. 24-28, patches P:284) applied to a single
 * precision map the CALLER supplies: d_sp_map = nx*ny*2 floats (layout as the LT_FP32 output), d_centres = n_centres * 3
 * doubles (x, y, deflection scale: b0, resp. 4 kappa_s rs) for the centre patches, d_flags = nx*ny bytes out (bit0 patch,
 * bit1 eq. 25, bit2 eq. 28).  lt_gradient_grid in LT_MIXED mode runs exactly these kernels on its own fp32 map; this
 * entry point exists so that the rule can be checked against its definition on any map.  d_workspace needs
 * lt_workspace_bytes(0, nx, ny, LT_MIXED) bytes; lt_mixed_last_stats works on it afterwards.  Asynchronous.
 */
int lt_mixed_rule(const float* d_sp_map, double x_min, double y_min, double dx, int nx, int ny,
                  const double* d_centres, int n_centres, const lt_mixed_params* mixed_or_null,
                  unsigned char* d_flags, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The consumer of the map in the paper's chi^2 algorithm (section 2.2.2, Fig. 1): every
 * pixel -- the cell between four neighbouring nodes of the fp64 map d_grad ([ny, nx, 2], the output of lt_gradient_grid in
 * LT_FP64 or LT_MIXED mode on the same grid) -- is cut into two triangles, each triangle is lensed into the source plane
 * with beta = theta - dls_dos * gradPsi (eq. 13), and every (source point, triangle) pair whose source-plane
 * triangle contains the point is appended to d_hits: a predicted multiple image, with its image-plane position by
 * barycentric interpolation.  Triangles are closed (a point on a shared edge is reported by both neighbours); zero-area
 * triangles contain nothing.  The inside test is exact fp64 arithmetic in a fixed order: the set of hits is reproducible
 * bit for bit, their order in d_hits is not.
 *   d_sources  device, n_sources * 2 doubles (beta_1, beta_2), 16-byte aligned; 0 <= n_sources <= LT_MAX_SOURCES
 *   d_hits     device, max_hits records; d_n_hits: device int, set to the number of hits FOUND (zeroed first); if it
 *              exceeds max_hits the surplus was counted but not stored.
 * Asynchronous on cuda_stream; needs nx, ny >= 2.
 */
int lt_find_images(const double* d_grad, double x_min, double y_min, double dx, int nx, int ny, double dls_dos,
                   const double* d_sources, int n_sources, lt_image_hit* d_hits, int max_hits, int* d_n_hits,
                   void* cuda_stream);

/*
 * The two small steps that close the chi^2 algorithm around the map (section 2.2.2; eq. 11), so that one
 * evaluation of the goodness of fit is a sequence of calls on one stream without a host round trip:
 *   lt_gradient_points (deflection alpha at the observed images) -> lt_source_barycentres -> lt_gradient_grid ->
 *   lt_find_images (sources = the barycentres) -> lt_chi2.
 * The observed images of system i are rows d_offsets[i] .. d_offsets[i+1]-1 (n_systems+1 ascending ints, d_offsets[0] = 0,
 * d_offsets[n_systems] = n_images) of d_theta / d_alpha / d_theta_obs ([n_images, 2] doubles, 16-byte aligned) and of
 * d_sigma ([n_images] doubles, > 0).  All pointers are device pointers; both calls are asynchronous on cuda_stream.
 *
 * lt_source_barycentres: beta_ij = theta_ij - dls_dos * alpha_ij (eq. 13; product and difference rounded
 * separately), d_barycentres[i] = (sum over j, in catalogue order, of beta_ij) / n_i ([n_systems, 2] doubles); a system
 * without images gets (nan, nan), which lt_find_images finds in no triangle.  One D_LS/D_OS per call: systems at another
 * source redshift go through their own sequence of calls.
 *
 * lt_chi2: d_terms[j] = |theta_obs_j - x_j|^2 / sigma_j^2 with x_j the predicted image (d_hits / d_n_hits / max_hits as
 * lt_find_images left them; hit.source = system index) of the image's own system nearest to it -- the paper does not say
 * how predicted and observed images are paired (reading R28) -- or nan if that system has no predicted image;
 * d_result->chi2 = the sum of the non-nan terms in catalogue order (eq. 11), with the counts of both kinds.  What a model
 * that loses images should cost is the caller's decision (R28).  Every operation is a correctly rounded fp64 operation in
 * the order written here: the result is reproducible bit for bit.
 * Errors: LT_ERR_BAD_SIZE (negative counts, n_systems > LT_MAX_SOURCES, n_images > 2^24, images without systems),
 * LT_ERR_NULL_POINTER, LT_ERR_MISALIGNED, LT_ERR_BAD_GRID (dls_dos not finite), LT_ERR_CUDA.
 */
int lt_source_barycentres(const double* d_theta, const double* d_alpha, const int* d_offsets, int n_systems,
                          double dls_dos, double* d_barycentres, void* cuda_stream);
int lt_chi2(const double* d_theta_obs, const double* d_sigma, const int* d_offsets, int n_systems, int n_images,
            const lt_image_hit* d_hits, const int* d_n_hits, int max_hits, double* d_terms, lt_chi2_result* d_result,
            void* cuda_stream);

/*
 * Launch-configuration knobs (process-wide; 0 = the library's default).  ppt64 / ppt32: pixels per thread of the
 * fp64 (1, 2, 4) and fp32 (1, 2, 4) grid kernels; chunk64 / chunk32: lens records staged in shared memory at a time;
 * ctas_per_sm: cap on resident CTAs per SM of the persistent grids; single_launch: bit 0 = one launch of the chosen
 * variant over the whole grid instead of whole waves plus a finer-grained rest, bit 1 = the host
 * entry points always stage the map in device memory and copy it, even into a pinned buffer, bit 2 = lt_gradient_points
 * runs one thread per point whatever the length of the list, bit 3 = the grid kernels are launched without the
 * programmatic-dependent-launch attribute, bit 4 = LT_FP32 and the first step of LT_MIXED run the
 * paper's plain SP version, "identical up to the change in precision": pixel coordinates, lens centres and
 * their difference in fp32, instead of the tile-centre coordinates of DESIGN.md section 5 -- a measurement variant
 * for the calibration of the mixed rule (what the centre patches of P:284 are for), not a mode; bit 5 = the fp64 kernels
 * stage the lens records in shared memory always, instead of reading them from the constant bank where the call allows it
 * (DESIGN.md section 6).  Results do not depend on
 * any of the others except that the fp32 tile centre moves with the pixels per thread of the launch
 * that owns the pixel.  Returns LT_ERR_BAD_SIZE on a negative value.
 * Thread safety: the knobs are independent atomics; a launch racing this call sees each knob either old or new.  They
 * are measurement and test hooks, not per-call state: set them before the threads that launch are started.
 */
int lt_set_tuning(int ppt64, int ppt32, int chunk64, int chunk32, int ctas_per_sm, int single_launch);

/* Number of kernels of this library the last lt_gradient_grid / lt_gradient_grid_host / lt_gradient_points call on this
 * host thread enqueued (memsets and copies not counted): bench.py's `gpu_launches`. */
int lt_last_launch_count(void);

/*
 * Measurement hook for bench.py's roofline figure: two cudaEvent_t (as void*; both NULL switches the hook off) that the
 * NEXT calls of lt_gradient_grid on this host thread record on cuda_stream immediately before and after the launch of
 * the dominant kernel (fp64 / fp32 grid kernel; for LT_MIXED the fp64 recompute kernel), so that its duration can be
 * taken on the launching stream without a profiler.  In LT_FP64 and LT_FP32 mode the pair also brackets the precompute
 * kernel (a few microseconds): the grid kernel is launched as its programmatic dependent and an event between the two
 * would serialise them, so the duration reported is an upper bound of the grid kernels' own.  Returns LT_ERR_NULL_POINTER if exactly one is NULL.
 */
int lt_set_kernel_events(void* ev_start, void* ev_stop);

/* After a call on this workspace: LT_OK or LT_ERR_BAD_LENS_PARAMS (first offending lens index in *bad_lens_or_null).
 * Synchronises cuda_stream. */
int lt_last_status(const void* d_workspace, void* cuda_stream, int* bad_lens_or_null);

/* After an LT_MIXED call on this workspace: counts of flagged pixels.  Synchronises cuda_stream. */
int lt_mixed_last_stats(const void* d_workspace, void* cuda_stream, lt_mixed_stats* out);

/* After an LT_MIXED call: copies the per-pixel flag byte map (bit0 patch, bit1 eq.25, bit2 eq.28; nx*ny bytes)
 * kept in the workspace into d_flags_out (device).  Asynchronous on cuda_stream. */
int lt_mixed_last_flags(const void* d_workspace, int n_lens, int nx, int ny, unsigned char* d_flags_out,
                        void* cuda_stream);

/* After an LT_MIXED call: copies the single precision map of its first step ("first, we compute the gradient in SP
 * for every pixel"; nx*ny*2 floats, layout of the output) kept in the workspace into d_sp_out (device).  This is the map
 * eq. 24-28 were evaluated on, so the flag map of lt_mixed_last_flags is a function of it and of the lens
 * centres alone.  Asynchronous on cuda_stream. */
int lt_mixed_last_sp_map(const void* d_workspace, int n_lens, int nx, int ny, float* d_sp_out, void* cuda_stream);

/*
 * The paper's accuracy criterion on a pair of maps (section 3.2): a single precision gradient is accurate
 * enough where |err_i| <= dx / (4 M_i), M_i = dx / |dx - delta_i| the magnification along axis i (eq. 24, 26, P:298-310;
 * delta_i from the DOUBLE precision map; forward neighbour in the first column / row, delta = 0 along an axis of extent 1).
 * This is the measurement behind the constants of the mixed rule (M_max = (dx/4) / E_SP = 3.26 for the paper's SIE error
 * model), which "has to be computed for each model independently": SURVEY 8(f) NEXT-2.
 *   d_sp_map      nx*ny*2 floats  (e.g. lt_mixed_last_sp_map, or an LT_FP32 map)
 *   d_dp_map      nx*ny*2 doubles (an LT_FP64 map of the same grid)
 *   d_centres     n_centres * 3 doubles (x, y, unused) or NULL: lens centres for the error-by-distance table
 *   d_flags       nx*ny bytes, the rule's mask (lt_mixed_last_flags: bit 0 = centre patch) or NULL
 *   d_violation   nx*ny bytes out or NULL: bit 0 / bit 1 = component 1 / 2 exceeds its budget
 *   d_result      one lt_audit_result in DEVICE memory (8-byte aligned), zeroed and filled by the call
 * Asynchronous on cuda_stream; read the result with lt_rule_audit_result.  max_err_by_distance[k]: largest |SP - DP|
 * (worse component, arcsec) among the pixels whose Chebyshev distance in pixels to the nearest centre lies in
 * [0,1) [1,2) [2,4) [4,8) [8,16) [16,32) [32,64) [64,128) [128,inf): the table form of Fig. 9; 0 = empty bin.
 */
#define LT_AUDIT_BINS 9
typedef struct {
  long long n_pixels, n_violating, n_violating_flagged, n_violating_missed, n_flagged;
  double max_err, max_err_in_patch, max_err_outside_patch;    /* arcsec; patch = bit 0 of d_flags */
  double max_err_by_distance[LT_AUDIT_BINS];
  double implied_m_max, implied_m_max_outside_patch;          /* (dx/4) / max_err...: filled by lt_rule_audit_result */
} lt_audit_result;
int lt_rule_audit(const float* d_sp_map, const double* d_dp_map, double x_min, double y_min, double dx, int nx, int ny,
                  const double* d_centres, int n_centres, const unsigned char* d_flags, unsigned char* d_violation,
                  lt_audit_result* d_result, void* cuda_stream);
/* Copies the result of lt_rule_audit to the host (synchronises cuda_stream) and fills the two implied_m_max fields
 * (M_max = (dx / 4) / E_SP; inf when the error is 0). */
int lt_rule_audit_result(const lt_audit_result* d_result, double dx, void* cuda_stream, lt_audit_result* h_out);

/* lt_gradient_grid without any allocation, by the library or by the caller: the deflection map of dPIE lenses (the same
 * operation as lt_gradient_grid: Algorithm 1, with the dPIE body of BASELINE.json's north star) for
 * mode = LT_FP64 or LT_FP32, with the workspace -- the scratch that the per-lens precompute kernel writes and the grid
 * kernels read -- held in a device array built into the library (LT_NOALLOC_SCRATCH_BYTES = 800 KiB of device memory on
 * every GPU that loads the library, until the process exits).  For callers that cannot call cudaMalloc: code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it.  The call itself makes no cudaMalloc / cudaFree and calls
 * no allocating library routine; it enqueues the precompute kernel and the shared-memory grid kernels on cuda_stream and
 * returns (asynchronous, like lt_gradient_grid).
 *   d_lenses   device, [n_lens] lt_lens, caller-owned, read only; 0 <= n_lens <= LT_NOALLOC_MAX_LENSES (4096).
 *   d_out_grad device, [ny][nx][2] double (LT_FP64) or float (LT_FP32), 16-byte aligned, caller-owned, every element
 *              written.  Grid arguments as for lt_gradient_grid.
 * Results: LT_FP32 bit-identical to lt_gradient_grid; LT_FP64 the same operations in the same order as lt_gradient_grid
 * (identical bits; the records come from shared memory instead of the constant bank).
 * Sharing: every call on a device uses the SAME array.  It keeps the last call's contents; nothing in it has to start at
 * zero (the precompute kernel rewrites the header, the domain-check slots, the tables and every record the call reads).
 * Two calls that overlap on the GPU (different streams, or different host threads) RACE on it: order them on one stream
 * or with events.  lt_noalloc_last_status reports the domain check of the LAST call on the current device.
 * Errors: LT_ERR_NOALLOC_TOO_LARGE (n_lens > LT_NOALLOC_MAX_LENSES: use lt_gradient_grid with a workspace),
 * LT_ERR_BAD_MODE (LT_MIXED: its scratch grows with the map), LT_ERR_BAD_SIZE, LT_ERR_NULL_POINTER, LT_ERR_BAD_GRID,
 * LT_ERR_MISALIGNED, LT_ERR_CUDA -- all argument errors before any CUDA call. */
#define LT_NOALLOC_MAX_LENSES 4096
#define LT_NOALLOC_SCRATCH_BYTES 819200
int lt_gradient_grid_noalloc(const lt_lens* d_lenses, int n_lens, double x_min, double y_min, double dx, int nx, int ny,
                             lt_precision mode, void* d_out_grad, void* cuda_stream);
/* lt_last_status for the built-in scratch of the current device (synchronises cuda_stream). */
int lt_noalloc_last_status(void* cuda_stream, int* bad_lens_or_null);

/* FMA-chain microbenchmarks used by bench.py to confirm the FP64 / FP32 peaks on the device in the same run
 * (SURVEY 8(d)): runs `iters` dependent-free FMAs per thread on a full grid; returns achieved FLOP/s in *flops_out
 * (2 flops per FMA).  Synchronises.  which: 0 = fp64, 1 = fp32, 2 = fp32 in packed pairs (FFMA2: two FMAs per
 * instruction -- the same FLOP/s as which = 1 where the FP32 pipe takes a packed instruction for two cycles, which is
 * what this chip does: packing saves issue slots, not pipe cycles); 3 = fp64 and 4 = packed fp32
 * with THREE distinct register-pair sources per instruction (a = fma(a, b, c), all in registers): 2/3 of the rate of
 * which = 0 / 2 on B200, whose register file delivers two 32-bit source reads per lane and cycle -- the reason the kernels
 * keep constants in uniform registers / immediates and avoid three-register FMAs. */
int lt_peak_probe(int which, int iters, double* flops_out, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* LT_GRADIENT_H */
