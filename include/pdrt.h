/*
 * pdrt.h — C ABI of the B200-native PyDoseRT dose hot path (libpdrt.so).
 *
 * The library computes, entirely in hand-written CUDA kernels for sm_100a, the forward and
 * backward dose computation of arxiv 2512.18863 ("A physics-informed, plug-and-play dose engine
 * for gradient-based radiotherapy treatment planning", /root/reference/PAPER.md) from delivery
 * parameters:
 *
 *   S1  aperture -> fluence map          PAPER.md:103-119, Eq. 4 (+ transmission, penumbra,
 *                                        head scatter, off-axis)
 *   S2  radiological depth               PAPER.md:135-143, Eq. 7 (central-axis ray per gantry angle)
 *   S4  depth-dependent lateral kernels
 *   S3  divergent projection             PAPER.md:123-133, Eq. 5-6
 *   S5  per-slice 2-D convolution        PAPER.md:151-158, Eq. 8
 *   S6  beam -> patient resampling and MU-weighted accumulation   PAPER.md:160-168, Eq. 9
 *   S7-S10  the exact transposes of S6, S5, S3, S1 that map dL/dDose to dL/d(leaf, jaw, MU)
 *           (PAPER.md:33-35, :67; depth and kernels carry no gradient, :143, :149)
 *
 * Where the paper is silent the readings G1-G22 of DESIGN.md §3 apply (geometry conventions,
 * kernel form, sampling rules).  Units: millimetres and degrees.  All arithmetic on the dose path
 * is float32 (float64 only in the ray marcher's positions and prefix sum).
 *
 * Conventions
 *   Patient grid: nx*ny*nz voxels, memory [z][y][x] (x fastest), centre of voxel (i,j,k) at
 *     (ox + i*sx, oy + j*sy, oz + k*sz).
 *   Gantry angle phi: u^ = (cos phi, sin phi, 0), w^ = (-sin phi, cos phi, 0), v^ = (0,0,1);
 *     the source sits at iso - SID*w^ (phi = 0: beam travels +y; phi = 90: source on the +x side).
 *   Beam grid: Nu x Nv x Nw with Nv = nz, dv = sz (beam v-slices are patient z-slices),
 *     u_i = (i - (Nu-1)/2) du,  w_k = beam_wmin + k dw,  v_j = oz + j sz - iso_z.
 *   Fluence map: flu_nu x flu_nv pixels, memory [v][u], pixel centres
 *     uf_a = (a - (flu_nu-1)/2) flu_du,  vf_b = (b - (flu_nv-1)/2) flu_dv  at the isocentre plane.
 *   Leaves: [n_cp][2][n_pairs], bank 0 = left edge l_i, bank 1 = right edge r_i (along u, mm at
 *     the isocentre plane); leaf pair i shadows v in [leaf_bounds_mm[i], leaf_bounds_mm[i+1]].
 *   Jaws: [n_cp][4] = x1, x2 (along u), y1, y2 (along v).
 *
 * Ownership and execution
 *   The caller owns every buffer it passes.  pdrt_create copies the density volume and all tables
 *   (they may be freed on return).  Pointers named *_dev are device pointers on the engine's
 *   device; pointers named *_host are host pointers (pinned memory makes the copies asynchronous).
 *   Outputs are caller-allocated and fully overwritten.  Scratch memory is engine-owned, grown
 *   lazily to the largest n_cp seen.  pdrt_dose / pdrt_dose_backward enqueue work on `cuda_stream`
 *   (a cudaStream_t, may be NULL for the default stream) and return without synchronising;
 *   the *_host variants copy in, run, copy out and synchronise the stream before returning.
 *   An engine must not be used from two threads at once.
 *
 * Errors
 *   Every function returning int returns PDRT_OK (0) or a negative code; pdrt_last_error gives
 *   the message of the last failure on that engine (or of the last failed pdrt_create when the
 *   engine argument is NULL).  Nothing aborts or throws across this boundary.  Device-resident
 *   parameters are not validated: l_i > r_i is a closed pair by Eq. 4's max(0, .); a control point
 *   whose jaws are inverted or NaN is a closed field (dose contribution and gradients exactly 0);
 *   NaN or infinite leaf positions and MU are not detected (NaN MU gives NaN dose; results are
 *   otherwise unspecified but every access stays in bounds).  There is no CPU fallback: without
 *   a CUDA device pdrt_create fails with PDRT_ECUDA.
 */
#ifndef PDRT_H
#define PDRT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define PDRT_API __attribute__((visibility("default")))
#else
#define PDRT_API
#endif

#define PDRT_OK       0
#define PDRT_EINVAL  (-1)   /* null pointer, non-positive size, even/out-of-range kernel size, bad table */
#define PDRT_ENOMEM  (-2)   /* host or device allocation failed                                        */
#define PDRT_ECUDA   (-3)   /* CUDA runtime error (message from cudaGetErrorString)                    */

typedef struct pdrt_engine pdrt_engine;   /* opaque */

/* Patient dose / density grid (CT volume as relative electron density). */
typedef struct {
    int32_t nx, ny, nz;      /* voxels                                   */
    float   sx, sy, sz;      /* spacing [mm]                             */
    float   ox, oy, oz;      /* centre of voxel (0,0,0) [mm]             */
    float   iso[3];          /* isocentre [mm], patient frame            */
} pdrt_grid;

/* "Beam-model tables": the machine-specific coefficients of PAPER.md:119, :176.  All pointers are
 * HOST pointers, read during pdrt_create only. */
typedef struct {
    float   sid_mm;                      /* source-isocentre distance (1000)                              */
    int32_t n_pairs;                     /* MLC leaf pairs                                                */
    const float *leaf_bounds_mm;         /* n_pairs+1 leaf boundaries along v, strictly ascending         */
    int32_t flu_nu, flu_nv;              /* fluence map pixels                                            */
    float   flu_du, flu_dv;              /* fluence pixel size [mm]                                       */
    float   tau;                         /* MLC transmission (~0.002)                       */
    float   fwhm_mlc_mm, fwhm_jaw_mm;    /* source penumbra FWHM along u / along v; 0 = off */
    int32_t n_hs;                        /* head-scatter Gaussians; 0 = off                */
    const float *hs_amp, *hs_sigma_mm;   /* n_hs amplitudes and sigmas                                    */
    int32_t n_oar; float oar_dr_mm;      /* radial off-axis table; n_oar = 0 = off         */
    const float *oar;                    /* n_oar factors at r = n * oar_dr_mm, clamped at the last entry */
    int32_t n_z; float dz_mm;            /* kernel parameters tabulated at radiological depth z = n * dz  */
    const float *kA, *ka, *kB, *kb;      /* n_z each: K(r;z) = (A e^{-a r} + B e^{-b r}) / r */
    int32_t kernel_size;                 /* lateral kernel size in beam-grid pixels: odd, 3..255          */
    float   cal;                         /* global dose scale (PAPER.md:178 energy scaling factor)        */
    int32_t beam_nu, beam_nw;            /* beam grid; beam_nu == 0 selects the default grid as a whole:  */
    float   beam_du, beam_dw, beam_wmin; /*   Nu = nx, Nw = ny, du = dw = sx, wmin = -(Nw-1)/2 * dw       */
    float   ray_step_mm;                 /* ray-march step; 0 => 0.5 * min(sx, sy, sz)                    */
    int32_t depth_mode;                  /* PDRT_DEPTH_AXIS (0, the paper's mode) or PDRT_DEPTH_FAN       */
} pdrt_beam_model;

/* Radiological-depth modes.  PDRT_DEPTH_AXIS: one ray per gantry angle through the isocentre (the paper's
 * mode and the default).  PDRT_DEPTH_FAN (reading G24): additionally one diverging ray
 * per fluence-map pixel, depth counted per unit axial distance; the projected fluence is weighted by
 * T(z_ray)/T(z_axis), T(z) = 2 pi (A/a + B/b)(z) the plane integral of the kernel, interpolated between the rays; the
 * lateral kernel stays per slice.  Identical to the paper's mode where the medium is homogeneous across the beam. */
#define PDRT_DEPTH_AXIS 0
#define PDRT_DEPTH_FAN  1

/* Resolved sizes of an engine (after defaults). */
typedef struct {
    int32_t nx, ny, nz;
    int32_t beam_nu, beam_nv, beam_nw;
    float   beam_du, beam_dv, beam_dw, beam_wmin;
    int32_t flu_nu, flu_nv, n_pairs;
    int32_t kernel_size;                 /* as requested                                      */
    int32_t kernel_size_compiled;        /* compiled conv variant of one pass (single pass: >= kernel_size) */
    float   ray_step_mm;
    int32_t ray_samples;                 /* samples per central-axis ray                      */
    int32_t sm_count;
    uint64_t scratch_bytes;              /* device scratch currently held                     */
    int32_t kernel_passes;               /* conv passes per slice: 1, or NB^2 sub-kernels for kernel sizes above 75 */
} pdrt_info;

/* Work counters of the most recent pdrt_dose / pdrt_dose_backward (device-counted from the actual
 * fluence support of that call).  Reading them synchronises the call's stream. */
typedef struct {
    int32_t  n_cp;
    int64_t  conv_items;        /* (control point, slice, chunk) work items of the conv kernel    */
    int64_t  support_voxels;    /* sum over CPs and slices of |S_k| (possibly non-zero Phi_vol)   */
    int64_t  footprint_voxels;  /* sum over CPs and slices of |F_k| = |S_k (+) k x k|             */
    int64_t  region_voxels;     /* voxels of the compact per-CP beam-frame regions (materialised) */
    int64_t  conv_macs;         /* multiply-adds the conv kernel executed (counted by the kernel; the row-symmetric kernel shares
                                   each row correlation between two output rows, so this can be below k^2 per output)          */
    int32_t  kernel_size, kernel_size_compiled;
    int64_t  fan_rays;          /* PDRT_DEPTH_FAN: diverging rays traced (sum over control points), else 0  */
    int32_t  ray_samples;       /* samples per ray (upper bound: samples outside the grid are skipped)     */
    int32_t  conv_symmetric;    /* that call's convolution kernel: 0 output-stationary (k_conv), 1 row-symmetric (k_conv_sym),
                                   2 row- and column-symmetric (k_conv_fold)                                                   */
} pdrt_work;

/* pdrt_create: grid geometry, density volume [nz][ny][nx] (host OR device pointer; copied) and
 * beam-model tables.  Builds the pencil-kernel table W_tab[n_z][k][k] on the host in float64 by
 * 8x8 midpoint sub-sampling of K over each pixel (G4) and uploads it as float32.
 * Uses the current CUDA device. */
PDRT_API int pdrt_create(const pdrt_grid *grid, const float *density, const pdrt_beam_model *model,
                pdrt_engine **out);
PDRT_API void pdrt_destroy(pdrt_engine *engine);

/* Message of the last failure; valid until the next call on that engine. */
PDRT_API const char *pdrt_last_error(const pdrt_engine *engine);

/* Rebuilds W_tab for another lateral kernel size (odd, 3..255; the paper's operating point is 55, and its
 * sensitivity study goes to 225, Table 4); used by the kernel-size sweep
 * (Table 4).  Synchronises the device. */
PDRT_API int pdrt_set_kernel_size(pdrt_engine *engine, int32_t kernel_size);

/* Switches the radiological-depth mode (PDRT_DEPTH_AXIS / PDRT_DEPTH_FAN) for subsequent calls. */
PDRT_API int pdrt_set_depth_mode(pdrt_engine *engine, int32_t depth_mode);

/* Collimator rotation (reading G25).  coll_deg [n_cp] (host or device
 * pointer; copied on `cuda_stream`) are per-control-point collimator angles for subsequent pdrt_dose / pdrt_dose_backward
 * calls with the same n_cp: the aperture point (uf, vf) appears at R(phi_c)(uf, vf) in the beam frame (counter-clockwise in
 * the (u, v) plane); the fluence map is resampled (bilinear, zero outside) on its own grid after the rotation and before
 * the projection.  n_cp = 0 removes the angles (the default: no rotation).  No gradient w.r.t. the angle is returned. */
PDRT_API int pdrt_set_collimator(pdrt_engine *engine, int32_t n_cp, const float *coll_deg, void *cuda_stream);

PDRT_API int pdrt_get_info(const pdrt_engine *engine, pdrt_info *info);
PDRT_API int pdrt_get_work(pdrt_engine *engine, pdrt_work *work);

/* Per-stage device timing.  With profiling enabled every stage's kernel launches are bracketed by CUDA
 * events on the call's stream; pdrt_get_stage_ms synchronises that stream and returns, for the most recent
 * call, the milliseconds and the number of kernel launches of each stage (launches are counted even with
 * profiling off; ms are then zero). */
enum {
    PDRT_STAGE_FLUENCE = 0,      /* S1  k_fluence (+ control-point descriptors)        */
    PDRT_STAGE_DEPTH = 1,        /* S2  k_depth                                       */
    PDRT_STAGE_SCAN = 2,         /*     k_scan_items (work-item prefix, counters)     */
    PDRT_STAGE_CONV = 3,         /* S4+S5  k_conv<K,false>                            */
    PDRT_STAGE_GATHER = 4,       /* S6  k_gather_dose                                 */
    PDRT_STAGE_RESAMPLE_ADJ = 5, /* S7  k_resample_adjoint                            */
    PDRT_STAGE_CONV_ADJ = 6,     /* S8  k_conv<K,true>                                */
    PDRT_STAGE_PROJECT_ADJ = 7,  /* S9  k_project_adjoint                             */
    PDRT_STAGE_FLUENCE_ADJ = 8,  /* S10 k_fluence_adjoint                             */
    PDRT_STAGE_PROJECT = 9,      /* S3  k_project                                     */
    PDRT_STAGE_TRANSPOSE = 10,   /*     k_transpose_g (dL/dDose with z fastest)       */
    PDRT_N_STAGES = 11
};
PDRT_API int pdrt_set_profiling(pdrt_engine *engine, int32_t enable);
PDRT_API int pdrt_get_stage_ms(pdrt_engine *engine, float *ms /*[PDRT_N_STAGES]*/, int32_t *launches /*[PDRT_N_STAGES]*/);

/* Forward (S1-S6, Eq. 4-9):  dose = cal * sum_b MU_b * R_b[ (P Phi_b) (*) K(z_rad) ].
 *   leaves_dev [n_cp][2][n_pairs], jaws_dev [n_cp][4], gantry_deg_dev [n_cp], mu_dev [n_cp],
 *   dose_dev [nz][ny][nx] overwritten.  n_cp >= 1. */
PDRT_API int pdrt_dose(pdrt_engine *engine, int32_t n_cp,
              const float *leaves_dev, const float *jaws_dev,
              const float *gantry_deg_dev, const float *mu_dev,
              float *dose_dev, void *cuda_stream);

/* Backward (S7-S10): from dL_ddose_dev [nz][ny][nx] to d_leaves_dev [n_cp][2][n_pairs],
 * d_jaws_dev [n_cp][4], d_mu_dev [n_cp], all overwritten.  Stateless: takes the parameters again
 * and recomputes the fluence maps and depths.  Subgradient convention at the kinks of Eq. 4:
 * DESIGN.md G9.  No gradient w.r.t. gantry angle, density or tables. */
PDRT_API int pdrt_dose_backward(pdrt_engine *engine, int32_t n_cp,
                       const float *leaves_dev, const float *jaws_dev,
                       const float *gantry_deg_dev, const float *mu_dev,
                       const float *dL_ddose_dev,
                       float *d_leaves_dev, float *d_jaws_dev, float *d_mu_dev,
                       void *cuda_stream);

/* The same two calls with HOST buffers: host->device copies of the parameters (and dL/dDose),
 * the kernels, the device->host copy of the result, and a stream synchronise.  The four parameter arrays are packed into a
 * pinned block of the engine when the call is made (the caller's arrays may be reused at once) and travel as ONE copy; the
 * three gradient arrays come back as one copy and are unpacked on the host before the call returns.  The two volumes move on
 * copy streams of the engine: the backward call's parameters and dL/dDose are uploaded there, so they do not wait for
 * work still queued on `cuda_stream` (e.g. the forward pass of the same step). */
PDRT_API int pdrt_dose_host(pdrt_engine *engine, int32_t n_cp,
                   const float *leaves_host, const float *jaws_host,
                   const float *gantry_deg_host, const float *mu_host,
                   float *dose_host, void *cuda_stream);
/* pdrt_dose_host without the final wait: the parameters are uploaded, the kernels run and the dose travels to dose_host
 * (pinned memory) on a copy stream of the engine; pdrt_host_wait blocks until it has arrived.  Between the two the caller may
 * issue further calls (e.g. pdrt_dose_backward_host for a dL/dDose it already has): the download overlaps with them.
 * All host buffers of the call must stay valid until pdrt_host_wait (or the next synchronising call on the stream) returns. */
PDRT_API int pdrt_dose_host_async(pdrt_engine *engine, int32_t n_cp,
                   const float *leaves_host, const float *jaws_host,
                   const float *gantry_deg_host, const float *mu_host,
                   float *dose_host, void *cuda_stream);
PDRT_API int pdrt_host_wait(pdrt_engine *engine);
PDRT_API int pdrt_dose_backward_host(pdrt_engine *engine, int32_t n_cp,
                            const float *leaves_host, const float *jaws_host,
                            const float *gantry_deg_host, const float *mu_host,
                            const float *dL_ddose_host,
                            float *d_leaves_host, float *d_jaws_host, float *d_mu_host,
                            void *cuda_stream);

/* Stage taps for parity tests (device pointers, outputs overwritten; they run the same kernels
 * as pdrt_dose / pdrt_dose_backward and copy an intermediate out):
 *   pdrt_stage_fluence   S1: fluence maps (as they enter the projection: after the collimator rotation, if any)
 *                                                    phimap_dev [n_cp][flu_nv][flu_nu]
 *   pdrt_stage_depth     S2: radiological depths     zrad_dev   [n_cp][beam_nw]
 *   pdrt_stage_beam_dose S3-S5: beam-frame dose D_b of ONE control point, dense
 *                                                    db_dev     [beam_nw][beam_nv][beam_nu]
 *   pdrt_stage_grad_fluence S7-S9: dL/dPhimap per control point (zero outside the fluence
 *                        support of that control point) gphimap_dev [n_cp][flu_nv][flu_nu]
 *   pdrt_stage_fan_factor (PDRT_DEPTH_FAN) depth factor at the ray nodes, dense
 *                                                    factor_dev [n_cp][beam_nw][flu_nv][flu_nu], 0 outside the rays traced
 *                                                    (the fluence support bbox grown by one pixel)                          */
PDRT_API int pdrt_stage_fluence(pdrt_engine *engine, int32_t n_cp, const float *leaves_dev, const float *jaws_dev,
                       float *phimap_dev, void *cuda_stream);
PDRT_API int pdrt_stage_fan_factor(pdrt_engine *engine, int32_t n_cp, const float *leaves_dev, const float *jaws_dev,
                          const float *gantry_deg_dev, float *factor_dev, void *cuda_stream);
PDRT_API int pdrt_stage_depth(pdrt_engine *engine, int32_t n_cp, const float *gantry_deg_dev,
                     float *zrad_dev, void *cuda_stream);
PDRT_API int pdrt_stage_beam_dose(pdrt_engine *engine, const float *leaves_dev, const float *jaws_dev,
                         const float *gantry_deg_dev, float *db_dev, void *cuda_stream);
PDRT_API int pdrt_stage_grad_fluence(pdrt_engine *engine, int32_t n_cp, const float *leaves_dev, const float *jaws_dev,
                            const float *gantry_deg_dev, const float *dL_ddose_dev,
                            float *gphimap_dev, void *cuda_stream);

/* ------------------------------------------------------------------------------------------------------------------
 * Planning-loop steps: with these a whole optimisation iteration
 *     theta^ = pdrt_validate(theta);  jaws = pdrt_track_jaws(theta^);  D = pdrt_dose(theta^);  (L, g) = pdrt_objective(D);
 *     g^ = pdrt_dose_backward(theta^, g);  g_theta = pdrt_validate_backward(theta, g^);  theta = pdrt_plan_step(theta, g_theta)
 * runs on the device without leaving the library (and can be captured in a CUDA graph: none of the calls synchronises).
 * All pointers are device pointers unless named *_host; all calls are asynchronous on `cuda_stream`. */

/* Limits of the hardware-constrained projection, PAPER.md:83-101 (BeamValidationLayer). */
typedef struct {
    float leaf_w_min;        /* minimum opening of a leaf pair, w >= w_min (Eq. 1)            */
    float leaf_F;            /* half field width: pair centre clamped to [-F, F]              */
    float jaw_w_min;         /* minimum opening of a jaw pair                                 */
    float jaw_Fx, jaw_Fy;    /* centre range of the (x1,x2) and of the (y1,y2) jaw pair       */
    float mu_eps;            /* minimum MU per control point (Eq. 3; pdrt_mu_epsilon)         */
} pdrt_limits;

/* Eq. 3: eps = D_min * delta_phi / phidot_max — minimum dose rate [MU/s] times control-point spacing
 * [deg] over maximum gantry speed [deg/s].  Host arithmetic. */
PDRT_API float pdrt_mu_epsilon(float dose_rate_min, float delta_phi_deg, float gantry_speed_max);

/* Eq. 1-2 on every leaf pair and on the two jaw pairs, and MU >= mu_eps: c = (p_a + p_b)/2, w = p_b - p_a, w >= w_min,
 * c clamped to [-F, F], p_a^ = c - w/2, p_b^ = c + w/2.  Shapes as in pdrt_dose; outputs may alias the inputs. */
PDRT_API int pdrt_validate(pdrt_engine *engine, int32_t n_cp, const pdrt_limits *limits,
                           const float *leaves_dev, const float *jaws_dev, const float *mu_dev,
                           float *leaves_out_dev, float *jaws_out_dev, float *mu_out_dev, void *cuda_stream);

/* Transposed Jacobian of pdrt_validate at the RAW parameters ("preserve gradients"): maps gradients w.r.t.
 * the projected parameters (what pdrt_dose_backward returns) to gradients w.r.t. the raw ones.  The map is piecewise
 * linear; a clamp passes the gradient where its input lies inside the closed interval (reading G23). */
PDRT_API int pdrt_validate_backward(pdrt_engine *engine, int32_t n_cp, const pdrt_limits *limits,
                                    const float *leaves_dev, const float *jaws_dev, const float *mu_dev,
                                    const float *g_leaves_hat_dev, const float *g_jaws_hat_dev, const float *g_mu_hat_dev,
                                    float *g_leaves_dev, float *g_jaws_dev, float *g_mu_dev, void *cuda_stream);

/* Weighted-sum objective and its dose gradient (Eq. 10 for power = 1; power = 2 is the quadratic
 * objective of BASELINE.json's c4/c5):  L = sum_s lambda_s sum_{x in s} |D(x) - p_s|^power.  structure_bits_dev
 * [nz][ny][nx] uint32: bit s set when the voxel belongs to structure s (structures may overlap), n_struct <= 32;
 * lambda_host / presc_host: n_struct weights and prescriptions (0 for organs at risk).  Writes dL_ddose_dev [nz][ny][nx]
 * and the loss (float64, device).  power 1: sign(0) = 0. */
PDRT_API int pdrt_objective(pdrt_engine *engine, const float *dose_dev, const uint32_t *structure_bits_dev, int32_t n_struct,
                            const float *lambda_host, const float *presc_host, int32_t power,
                            float *dL_ddose_dev, double *loss_dev, void *cuda_stream);

/* pdrt_objective for callers that cannot allocate device memory (code under CUDA stream capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments, same result (dL/dDose bit-identical; the loss differs by float64
 * rounding order only and does not depend on the GPU's SM count), but the call makes no cudaMalloc / cudaFree and uses no
 * engine scratch.  Its scratch (8192 float64 block partials and a ticket, 64.25 KiB) is a static __device__ array of the
 * library: every GPU that loads libpdrt.so holds it until the process exits.  Limits and rules:
 *   - the dose grid may have at most PDRT_NOALLOC_MAX_VOXELS voxels; a larger grid is rejected with PDRT_EINVAL and a
 *     message naming both numbers (use pdrt_objective there);
 *   - all calls on one GPU — of every engine and every stream — share the array: calls that overlap on the GPU race
 *     (wrong loss).  Order them on one stream or with events.  What must start at zero (the ticket) is cleared by
 *     the call itself on `cuda_stream`, so a call does not depend on what the previous one left;
 *   - the first call on a device resolves the array's device address (cudaGetSymbolAddress; no allocation): make one call
 *     before stream capture begins.  One kernel launch and one 256-byte memset node per call, no synchronisation. */
#define PDRT_NOALLOC_MAX_VOXELS (1 << 25)   /* 33 554 432 voxels, e.g. 512 x 512 x 128 */
PDRT_API int pdrt_objective_noalloc(pdrt_engine *engine, const float *dose_dev, const uint32_t *structure_bits_dev, int32_t n_struct,
                                    const float *lambda_host, const float *presc_host, int32_t power,
                                    float *dL_ddose_dev, double *loss_dev, void *cuda_stream);

/* Jaws tracking the aperture (BASELINE.json configs[4]): over the leaf pairs open by more than open_gap_mm (all pairs when
 * none is) x1 = min l - margin, x2 = max r + margin, y1 / y2 = the leaf boundaries that enclose them.  jaws_dev [n_cp][4]. */
PDRT_API int pdrt_track_jaws(pdrt_engine *engine, int32_t n_cp, const float *leaves_dev, float margin_mm, float open_gap_mm,
                             float *jaws_dev, void *cuda_stream);

/* Normalised-gradient step of the c5 planning loop: leaves -= step_leaf * g / max|g| over all leaf edges
 * of the arc, mu -= step_mu * g / max|g|; a group with an identically zero gradient does not move.  In place. */
PDRT_API int pdrt_plan_step(pdrt_engine *engine, int32_t n_cp, float step_leaf_mm, float step_mu,
                            const float *g_leaves_dev, const float *g_mu_dev, float *leaves_dev, float *mu_dev, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PDRT_H */
