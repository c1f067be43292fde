/* mcx.h -- C ABI of libmcx_b200.so: the data-parallel hot path of McXtrace-style X-ray ray tracing
 * (arxiv 2410.08747) as hand-written sm_100a CUDA kernels.
 *
 * What the library computes.  "Rays are generated at the source component and sequentially propagated through
 * the list of X-ray components" (section 1); each ray is independent and carries the
 * particle state of PAPER.md:92-98 (here: position, direction, energy, weight); monitors are histogram arrays
 * updated atomically.  The paper prints no physics formulas; every formula follows the reading
 * in DESIGN.md ("Readings", steps 1-15 of SURVEY.md 8(c)).  BASELINE.json:north_star names the three primary
 * entry points: mcx_instrument_create, mcx_trace, mcx_tally_read.
 *
 * Conventions.  Units: metres, keV, 1/m, radians.  A pose maps lab to component coordinates,
 * r_local = rot * (r_lab - origin), rot row-major, rows = local axes in lab coordinates (the paper's
 * "AT (...) RELATIVE" placement, given as an absolute rigid transform).  The ray between components
 * is held in lab coordinates.  Component 0 of a chain must be a source.
 *
 * Memory.  Pointers marked HOST are read during mcx_instrument_create only and may be freed afterwards.
 * Pointers marked DEVICE must stay valid (and, for inputs, unchanged) until mcx_instrument_destroy.  The library
 * never allocates device memory: everything it keeps on the device lives in the caller's `workspace`.
 *
 * Streams.  `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All calls enqueue
 * work on it and return without synchronising; the caller synchronises before reading outputs.
 *
 * Errors.  Every call returns an mcx_status; mcx_last_error() gives a thread-local message for the last failure.
 * Argument and range errors are found synchronously at create.  A sticky CUDA error is reported by the next call
 * as MCX_ERR_CUDA.  Errors of the asynchronous trace itself surface the same way: if a ray overflowed its per-ray
 * scratch capacity (MCX_ERR_CAPACITY below), every later call on the handle that finds the overflowing trace finished
 * on the device -- mcx_trace*, mcx_tally_read*, mcx_counters_read -- still does its work and returns MCX_ERR_CAPACITY,
 * until mcx_tally_reset; mcx_trace_status synchronises the stream first and is therefore definitive.
 * A handle must be used from one host thread at a time; distinct handles are independent.
 */
#ifndef MCX_H_
#define MCX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mcx_instrument mcx_instrument; /* opaque, host side */

typedef enum {
  MCX_OK = 0,
  MCX_ERR_INVALID_ARG = 1, /* null pointer, bad enum, chain not starting with a source, ... */
  MCX_ERR_UNSUPPORTED = 2, /* a limit of this build exceeded (see MCX_MAX_*) */
  MCX_ERR_RANGE = 3,       /* a table that is not strictly increasing / positive, an empty grid or bin range */
  MCX_ERR_WORKSPACE = 4,   /* workspace too small or misaligned (needs 256-byte alignment) */
  MCX_ERR_CUDA = 5,        /* a CUDA runtime call failed */
  MCX_ERR_CAPACITY = 6     /* during a trace some ray produced more interval end points in one solids group than the
                              per-ray scratch holds (2 per primitive + 8 per mesh, at least 16, at most 48: e.g. a ray
                              through the apex of a fan of more triangles than that).  Such rays are dropped as
                              MCX_FATE_DEGENERATE and counted in the capacity_overflows counter; the tallies hold
                              every other ray. */
} mcx_status;

enum { MCX_MAX_COMPONENTS = 16, MCX_MAX_DETECTORS = 8, MCX_MAX_MATERIALS = 32, MCX_MAX_SOLIDS = 16, MCX_MAX_LENSES = 256,
       MCX_MAX_SCATTER_ORDER = 1 << 20 };

typedef enum {
  MCX_SOURCE = 0,          /* step 3 (point / flat / Gaussian emitters) */
  MCX_SLIT_RECT = 1,       /* step 6 */
  MCX_SLIT_CIRC = 2,       /* step 6 */
  MCX_SOLIDS = 3,          /* steps 8-10: primitives and closed triangle meshes, Beer-Lambert */
  MCX_VOXELS = 4,          /* step 11: uint8 material-ID volume, exact traversal */
  MCX_MIRROR_ELLIPTIC = 5, /* step 12 (optics category) */
  MCX_CRYSTAL_BRAGG = 6,   /* step 13 */
  MCX_DETECTOR = 7,        /* step 14: PSD / E / EPSD / L monitors */
  MCX_LENS_PARAB = 8       /* step 16: compound refractive lens, a stack of double-sided parabolic lenses (PAPER.md:134,
                              138, 153: where the paper's focusing instrument spends its time) */
} mcx_kind;

typedef enum { MCX_POS_POINT = 0, MCX_POS_DISK = 1, MCX_POS_GAUSS = 2 } mcx_pos_mode;
typedef enum { MCX_DIR_TARGET = 0, MCX_DIR_GAUSS = 1 } mcx_dir_mode;
typedef enum { MCX_E_MONO = 0, MCX_E_UNIFORM = 1, MCX_E_SPECTRUM = 2 } mcx_energy_mode;
typedef enum { MCX_BOX = 0, MCX_CYLINDER = 1, MCX_SPHERE = 2, MCX_MESH = 3 } mcx_shape;
typedef enum { MCX_DET_ENERGY = 0, MCX_DET_WAVELENGTH = 1 } mcx_det_mode;

/* Fate of a ray (mcx_ray_fate.fate): >= 0 means "absorbed by the component with that chain index". */
enum { MCX_FATE_DETECTED = -1, MCX_FATE_MISSED = -2, MCX_FATE_DEGENERATE = -3 };

typedef struct mcx_pose {
  double rot[9];    /* row-major 3x3, orthonormal */
  double origin[3]; /* lab position of the component origin */
} mcx_pose;

/* mu(E) table of one material (step 7: log-log interpolation, end segments extrapolate).
 * n_points == 0: vacuum (mu = 0).  Otherwise n_points >= 2, energy strictly increasing, mu > 0. */
typedef struct mcx_material {
  int64_t n_points;
  const double* energy_keV; /* HOST [n_points] */
  const double* mu_per_m;   /* HOST [n_points], total attenuation coefficient */
  const double* mu_scatter_per_m; /* HOST [n_points] or NULL: the part of mu that scatters (step 17), 0 < mu_s <= mu,
                               interpolated like mu; NULL = the material only attenuates */
} mcx_material;

/* One solid of a MCX_SOLIDS group (step 8).  Its pose is absolute (lab), like a component's. */
typedef struct mcx_solid {
  int32_t shape;    /* mcx_shape */
  int32_t material; /* index into the materials array */
  int32_t priority; /* the highest priority owns an overlap; equal priorities: the earlier solid wins */
  int32_t reserved;
  mcx_pose pose;
  double dims[3];          /* BOX: half extents x,y,z.  CYLINDER (axis = local y): radius, half height.  SPHERE: radius */
  int64_t n_vertices;      /* MESH only */
  int64_t n_triangles;     /* MESH only; closed, outward-wound */
  const double* vertices;  /* HOST [n_vertices][3], solid-local frame */
  const int32_t* triangles;/* HOST [n_triangles][3] */
} mcx_solid;

typedef struct mcx_source_params {
  int32_t pos_mode, dir_mode, energy_mode, reserved;
  double radius;             /* POS_DISK */
  double sigma_x, sigma_y;   /* POS_GAUSS */
  double target_w, target_h, target_dist; /* DIR_TARGET: uniform in area on a rectangle at z = target_dist */
  double div_x, div_y;       /* DIR_GAUSS: sigma of the direction tangents */
  double e0;                 /* E_MONO / E_UNIFORM centre */
  double de_rel;             /* E_UNIFORM: E = e0 (1 + de_rel (2u - 1)) */
  double spec_emin, spec_emax; /* E_SPECTRUM: bins of equal width over [emin, emax] */
  int64_t spec_n;
  const double* spectrum;    /* HOST [spec_n], non-negative bin weights */
} mcx_source_params;

typedef struct mcx_slit_params {
  double xw, yh;  /* SLIT_RECT full widths */
  double radius;  /* SLIT_CIRC */
} mcx_slit_params;

typedef struct mcx_solids_params {
  int64_t n_solids;         /* <= MCX_MAX_SOLIDS */
  const mcx_solid* solids;  /* HOST [n_solids] */
  int64_t scatter_order;    /* step 17, as in mcx_voxels_params */
} mcx_solids_params;

typedef struct mcx_voxels_params {
  double h;                 /* voxel edge; the component origin is the outer corner of voxel (0,0,0) */
  int64_t nx, ny, nz;
  const uint8_t* ids;       /* DEVICE [nz][ny][nx], x fastest; values index the materials array (a value >=
                               n_materials is not a material and is traced as material 0, vacuum).
                               Read once by create (copied into the workspace in the traversal layout). */
  int64_t scatter_order;    /* step 17 (a step updates the ray's weight "and direction"): at most this
                               many elastic scattering events per ray in the sample, 0..MCX_MAX_SCATTER_ORDER; 0 =
                               Beer-Lambert attenuation only.  Leg k draws the scattering optical depth to its event,
                               -ln(u), and the Thomson-distributed angle (1 + cos^2) from slots 2k, 2k+1 of this component's
                               Philox stream; up to the event and on a leg that leaves without one the weight is
                               attenuated by mu - mu_s, after the last allowed event by mu. */
} mcx_voxels_params;

typedef struct mcx_mirror_params {
  double p, q, theta;       /* source distance, image distance, grazing angle at the pole */
  double length, width;     /* along the local z (tangential) and x (sagittal) axes; local y = surface normal */
  double theta_min, theta_max, e_min, e_max; /* uniform reflectivity grid */
  int64_t n_theta, n_e;
  const double* reflectivity; /* HOST [n_theta][n_e] */
} mcx_mirror_params;

typedef struct mcx_crystal_params {
  double length, width;     /* along local z and x; the reflecting surface is the plane y = 0, normal +y */
  double d_hkl;             /* Angstrom */
  double zeta;              /* relative Darwin width: w_D = zeta tan(theta_B) */
  double delta0;            /* refraction offset of the curve centre, radians */
  double g, kappa;          /* step 13b, Darwin-Prins curve of an absorbing crystal: g = Im(chi_0) / Re(chi_h) >= 0,
                               kappa = Im(chi_h) / Re(chi_h); eta_c = (eta + i g) / (1 + i kappa), R = |eta_c - sqrt(eta_c^2 - 1)|^2
                               on the branch with R <= 1.  0, 0: the non-absorbing Darwin curve of step 13 */
} mcx_crystal_params;

/* Step 16.  Lens frame: z = axis of the stack, origin at its centre.  Lens i = 0..n_lenses-1 is centred at
 * z_i = (i - (n_lenses-1)/2) pitch; it is material between the paraboloids z = z_i -+ (web/2 + rho^2 / (2 radius)).  At each
 * of the 2 n_lenses surfaces, in order: intersection, aperture test rho <= aperture (outside: absorbed), Snell's law with
 * n = 1 - delta(E) (total reflection or a ray running backwards: absorbed).  Beer-Lambert with mu(E) of `material` over
 * the summed chords inside the lenses.  Needs web/2 + aperture^2 / (2 radius) <= pitch/2 (the lenses do not overlap). */
typedef struct mcx_lens_params {
  double radius;            /* apex radius of curvature of the paraboloids */
  double web;               /* thickness of a lens on the axis */
  double pitch;             /* lens-to-lens distance */
  double aperture;          /* radius of the circular opening */
  int64_t n_lenses;         /* <= MCX_MAX_LENSES */
  int64_t material;         /* index into the materials array: mu(E) of the lens material */
  int64_t n_delta;          /* points of the delta(E) table, >= 2 */
  const double* delta_energy_keV; /* HOST [n_delta], strictly increasing */
  const double* delta;      /* HOST [n_delta], > 0; log-log interpolated like mu(E) (step 7) */
} mcx_lens_params;

typedef struct mcx_detector_params {
  double xmin, xmax, ymin, ymax, emin, emax; /* half-open bins */
  int64_t nx, ny, ne;
  int64_t mode;             /* mcx_det_mode.  MCX_DET_WAVELENGTH (an L_monitor): the third axis bins
                               lambda = hc / E in Angstrom over [emin, emax) read as wavelengths (step 14b) */
} mcx_detector_params;

typedef struct mcx_component {
  int32_t kind; /* mcx_kind */
  int32_t reserved;
  mcx_pose pose;
  union {
    mcx_source_params source;
    mcx_slit_params slit;
    mcx_solids_params solids;
    mcx_voxels_params voxels;
    mcx_mirror_params mirror;
    mcx_crystal_params crystal;
    mcx_detector_params detector;
    mcx_lens_params lens;
  } u;
} mcx_component;

/* Per-ray record written by mcx_trace_dump (per-ray branch parity). */
typedef struct mcx_ray_fate {
  int32_t fate;  /* MCX_FATE_* or the chain index of the absorbing component */
  int32_t reserved;
  int64_t bin;   /* bin in the last detector if fate == MCX_FATE_DETECTED, else -1 */
  double p;      /* final weight */
} mcx_ray_fate;

/* Number of int64 counters mcx_counters_read writes: [0, n_components) absorbed per component, then
 * detected, missed, degenerate, capacity_overflows. */
#define MCX_N_COUNTERS(n_components) ((n_components) + 4)

/* Bytes of device workspace mcx_instrument_create needs for this instrument (tables, BVH, re-laid voxel volume,
 * tally records, counters).  Reads only sizes, never the HOST/DEVICE arrays. */
mcx_status mcx_instrument_workspace_size(const mcx_component* components, int n_components,
                                         const mcx_material* materials, int n_materials, size_t* bytes_out);

/* Builds the device image of an instrument in `workspace` (DEVICE, caller-owned, 256-byte aligned, at least
 * mcx_instrument_workspace_size bytes): ln-tables of mu(E), spectrum CDFs, mirror constants, a BVH per mesh,
 * the voxel volume in its traversal layout; zeroes tallies and counters.  HOST inputs are consumed before return. */
mcx_status mcx_instrument_create(const mcx_component* components, int n_components,
                                 const mcx_material* materials, int n_materials,
                                 void* workspace, size_t workspace_bytes, void* cuda_stream,
                                 mcx_instrument** out);

/* Traces rays with indices [0, n_rays) (mcx_trace) or [first_ray, first_ray + n_rays) (mcx_trace_range).
 * Ray i draws from Philox4x32-10 with key = seed and counter = (i lo, i hi, slot, component index), so a ray is
 * a pure function of (instrument, seed, i).  Tallies and counters ACCUMULATE over calls; weights are not divided
 * by n_rays. */
mcx_status mcx_trace(mcx_instrument* inst, uint64_t n_rays, uint64_t seed, void* cuda_stream);
mcx_status mcx_trace_range(mcx_instrument* inst, uint64_t first_ray, uint64_t n_rays, uint64_t seed,
                           void* cuda_stream);

/* Lane scheduling.  Results do not depend on it beyond the summation order of the tallies:
 * a ray is a pure function of (instrument, seed, ray index) whatever order rays are traced in.
 *   MCX_EXEC_DIRECT  rays are traced in index order, 32 consecutive indices per warp;
 *   MCX_EXEC_SORTED  each chunk of <= 2^26 ray indices is first bucketed by the cell of a grid over the source's
 *                    direction draw (count, scan, scatter; 4 bytes of workspace per ray of a chunk), so that a warp
 *                    traces rays aimed at the same spot (coherent voxel / BVH / primitive walks);
 *   MCX_EXEC_AUTO    (default) SORTED where the source aims at a target rectangle and the instrument has a mesh, a
 *                    voxel volume or a group of two or more solids, DIRECT otherwise.
 * In either order, a chain that starts with slits, mirrors or crystals is traced through those first and only the
 * survivors, compacted warp by warp, through the whole chain (absorber gate); same results. */
typedef enum { MCX_EXEC_AUTO = 0, MCX_EXEC_DIRECT = 1, MCX_EXEC_SORTED = 2 } mcx_exec_mode;
mcx_status mcx_instrument_set_exec(mcx_instrument* inst, int mode);

/* Tuning of the lane scheduling, for sweeps and tests; 0 in a field = keep the library's choice.  Results never depend
 * on it beyond the summation order of the tallies.
 *   chunk_log2      rays per sorted chunk = 2^chunk_log2, 14..26 (default 26: the workspace always holds the order
 *                   buffer of a 2^26 chunk, 256 MiB, whatever is set here);
 *   sort_grid_bits  bits per axis of the bucket grid of MCX_EXEC_SORTED, 1..11 (default: by chunk length, at most 9
 *                   for instruments of analytic solids only, else 10);
 *   absorber_gate   1 = on (default), 2 = off;
 *   tally_mode      how a detected ray reaches its tally record (step 14), an mcx_tally_mode:
 *                   MCX_TALLY_GLOBAL  three reductions (u64 count, two fp64 sums) per detected ray into its record;
 *                   MCX_TALLY_WARP    warp-aggregated: lanes of a warp in the same bin are summed first, one leader
 *                                     per distinct bin issues the reductions;
 *                   MCX_TALLY_BLOCK   warp-aggregated into a block-private shared-memory cache of tally records
 *                                     (2048 direct-mapped slots; chains without solids or voxels only, MCX_TALLY_WARP
 *                                     elsewhere), flushed to the records once per block and launch; only detectors
 *                                     whose bins fit (together at most 1024, smallest first) go through the cache;
 *                   MCX_TALLY_AUTO (0 here = keep) is the library's choice from measurement:
 *                   MCX_TALLY_BLOCK where some detector fits the cache, MCX_TALLY_GLOBAL otherwise.
 *                   N is the same integer in every mode; p and p2 differ in summation order only.
 *   staged_walk     1 = on (default), 2 = off.  On, a chain of slits, voxel volumes and detectors whose first scattering
 *                   volume (scatter_order > 0) is walked by a kernel of its own, in which a lane takes
 *                   the next ray when its ray leaves the sample: per chunk of <= 2^22 rays, the components before the
 *                   volume, the volume, the components after it (80 bytes of workspace per ray of a chunk between
 *                   them, and one more byte per cell for a volume of at most 16 materials and 96 Mi cells, whose
 *                   walk then reads one-byte cells that stay in L2).  Off, or for any other chain: the whole chain in one launch.  Same results
 *                   ray for ray, to the rounding of two compilations of the same expressions;
 *   walk_batch_setup, walk_batch_settle   1..32: how many lanes of a warp of that kernel must wait for the set-up of a
 *                   leg / for the end of a run of equal voxels before the warp turns to them (defaults 16, 12). */
typedef enum { MCX_TALLY_AUTO = 0, MCX_TALLY_GLOBAL = 1, MCX_TALLY_WARP = 2, MCX_TALLY_BLOCK = 3 } mcx_tally_mode;
typedef struct mcx_tuning {
  int32_t chunk_log2, sort_grid_bits, absorber_gate, tally_mode, staged_walk, walk_batch_setup, walk_batch_settle;
} mcx_tuning;
mcx_status mcx_instrument_set_tuning(mcx_instrument* inst, const mcx_tuning* tuning);
/* The settings in effect: chunk_log2; sort_grid_bits (0 = chosen per chunk length); absorber_gate 1 / 2; tally_mode =
 * the mode the next trace will use (never MCX_TALLY_AUTO); staged_walk 1 = the next trace will be staged, 2 = not. */
mcx_status mcx_instrument_get_tuning(const mcx_instrument* inst, mcx_tuning* tuning_out);

/* Finalises detector `detector` (ordinal among MCX_DETECTOR components): writes N (ray counts), p (sum of
 * weights) and p2 (sum of squared weights) for all bins, bin = (iy * nx + ix) * ne + ie.
 * N, p, p2: DEVICE [n_bins]; n_bins must equal nx*ny*ne. */
mcx_status mcx_tally_read(mcx_instrument* inst, int detector, uint64_t* N, double* p, double* p2, size_t n_bins,
                          void* cuda_stream);

/* Same, with HOST output arrays (pinned memory if the copy is to be asynchronous): finalises into a staging area of
 * the workspace and enqueues three device-to-host copies on the stream.  This is the end-to-end read a caller
 * without device buffers uses (the paper's "update host"). */
mcx_status mcx_tally_read_host(mcx_instrument* inst, int detector, uint64_t* N, double* p, double* p2, size_t n_bins,
                               void* cuda_stream);

/* Bytes mcx_instrument_create copied from the host to the device for this handle (instrument image and tables; the
 * voxel volume is the caller's own upload). */
uint64_t mcx_upload_bytes(const mcx_instrument* inst);

/* Moves component `component` (a slit, voxel volume, mirror, crystal, lens or detector; not the source, not a solids
 * group, whose solids carry their own poses) to a new pose for the traces enqueued after this call: the line-by-line scan
 * of PAPER.md:190 ("550 lines per projection") translates the sample between traces.  Tallies are kept (read and reset
 * them per line as needed).  The pose is read before the call returns.  A voxel volume keeps the memory layout chosen at
 * create (fastest axis = the one most aligned with source -> volume); a pose that would change that choice is refused
 * with MCX_ERR_UNSUPPORTED. */
mcx_status mcx_instrument_set_pose(mcx_instrument* inst, int component, const mcx_pose* pose, void* cuda_stream);

/* Contrast-to-noise ratio of PAPER.md:257 Eq. (1) per energy bin of one detector's finalised tallies, and its
 * least-squares line above e_fit_min.  N, p, p2: DEVICE [ny*nx*ne] as written by mcx_tally_read.
 * region_mat, region_ref: HOST int32[4] = pixel rectangles x0, x1, y0, y1 (half-open, inside the detector, non-empty).
 * I_region = mean over its pixels of p; sigma_region^2 = sum over its pixels of sigma_bin^2 / n_pixels^2 with
 * sigma_bin^2 = N/(N-1) |p2 - (p/N)^2| for N > 1 and sigma_bin = p for N <= 1;
 * cnr_out[e] = |I_mat - I_ref| / sqrt(sigma_mat^2 + sigma_ref^2) (0 where the noise is 0): DEVICE [ne].
 * fit_out: DEVICE [2] = intercept, slope of the least-squares line through (bin-centre energy, cnr) over the bins with
 * centre >= e_fit_min (0, 0 with fewer than two such bins); emin, emax: the detector's energy range.  Asynchronous. */
mcx_status mcx_cnr(const uint64_t* N, const double* p, const double* p2, int64_t nx, int64_t ny, int64_t ne,
                   const int32_t* region_mat, const int32_t* region_ref, double emin, double emax, double e_fit_min,
                   double* cnr_out, double* fit_out, void* cuda_stream);

/* mcx_cnr for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): finalises detector `detector` of `inst` and computes the same cnr_out[ne] and fit_out[2] as
 * mcx_tally_read followed by mcx_cnr (Eq. (1), :268; emin, emax are the detector's own), with the
 * intermediate arrays (N, p, p2, the CNR per bin) in a file-scope device array of the library instead of buffers of the
 * caller's: 24 * MCX_CNR_STATIC_MAX_BINS + 8 * (MCX_CNR_STATIC_MAX_NE + 2) bytes (6 MiB) on every GPU that loads the
 * library, held until exit.  Calls no cudaMalloc, cudaFree or allocating library routine.
 * cnr_out [ne], fit_out [2]: HOST (pinned memory if the copy is to be asynchronous) or DEVICE memory, the caller's.
 * region_mat, region_ref: HOST int32[4] as for mcx_cnr.
 * Limits: a detector with more than MCX_CNR_STATIC_MAX_BINS bins or MCX_CNR_STATIC_MAX_NE energy bins is refused with
 * MCX_ERR_UNSUPPORTED (use mcx_tally_read + mcx_cnr with buffers of your own).
 * All calls on a device share the one array, and it keeps the last call's contents (every call overwrites what it reads,
 * nothing needs clearing): calls whose work overlaps on the GPU -- two streams without an ordering between them --
 * race on it and return garbage; calls on one stream, or ordered by events, are safe.  Asynchronous. */
enum { MCX_CNR_STATIC_MAX_BINS = 1 << 18, MCX_CNR_STATIC_MAX_NE = 4096 };
mcx_status mcx_cnr_static(mcx_instrument* inst, int detector, const int32_t* region_mat, const int32_t* region_ref,
                          double e_fit_min, double* cnr_out, double* fit_out, void* cuda_stream);

/* Zeroes all tallies and counters. */
mcx_status mcx_tally_reset(mcx_instrument* inst, void* cuda_stream);

/* Copies the MCX_N_COUNTERS(n_components) ray-accounting counters to `counters` (DEVICE [n]).  Their sum over
 * absorbed + detected + missed + degenerate equals the number of rays traced since the last reset. */
mcx_status mcx_counters_read(mcx_instrument* inst, uint64_t* counters, int n, void* cuda_stream);

/* Waits for everything enqueued on `cuda_stream` and reports what the traces since the last mcx_tally_reset did:
 * MCX_OK, MCX_ERR_CAPACITY (mcx_last_error gives the number of rays dropped) or MCX_ERR_CUDA (an asynchronous fault).
 * The one call that synchronises. */
mcx_status mcx_trace_status(mcx_instrument* inst, void* cuda_stream);

/* Traces rays [first_ray, first_ray + n_rays) and writes one record per ray to `out` (DEVICE [n_rays]) instead of
 * tallying: tallies and counters are left untouched.  For parity tests. */
mcx_status mcx_trace_dump(mcx_instrument* inst, uint64_t first_ray, uint64_t n_rays, uint64_t seed,
                          mcx_ray_fate* out, void* cuda_stream);

/* Number of kernel launches this handle has enqueued so far (create, trace, read, reset). */
uint64_t mcx_launch_count(const mcx_instrument* inst);

/* Device-time split of the traces, for the measurement of SURVEY.md 8(d).  With timing on (on != 0), every chunk of a
 * trace records CUDA events on the launching stream before its ray sort, between the sort and trace_kernel, and after
 * trace_kernel (at most 4096 chunks between two reads; later ones go untimed).  mcx_timing_read waits for the last of
 * them and gives the sums since the previous read: milliseconds in the sort kernels, milliseconds in trace_kernel, and
 * the number of trace_kernel launches timed (all HOST pointers, each may be NULL); then it forgets them.  A staged trace
 * (mcx_tuning.staged_walk) has three launches per chunk between the last two events -- trace_kernel, scatter_walk_kernel,
 * trace_kernel -- and counts all three. */
mcx_status mcx_instrument_set_timing(mcx_instrument* inst, int on);
mcx_status mcx_timing_read(mcx_instrument* inst, double* sort_ms, double* trace_ms, int64_t* n_trace_launches);

/* Sustained-FP64 probe used for the ALU roofline: enqueues a kernel in which every thread of a
 * (n_blocks x 256) grid runs n_iters x 8 dependent-chain-free DFMAs; `sink` is DEVICE [n_blocks*256] doubles.
 * Lane-ops performed = n_blocks * 256 * n_iters * 8. */
mcx_status mcx_probe_dfma(double* sink, int n_blocks, int64_t n_iters, void* cuda_stream);

/* Tally-reduction probe for the atomics roofline ("measure random red.add.f64 rate"): every thread of a
 * (n_blocks x 256) grid does n_iters rounds of the three reductions of a detected ray (u64 count, two fp64 sums)
 * into one pseudo-random 32-byte record of `table` (DEVICE, n_records * 32 bytes, n_records a power of two; contents
 * are garbage afterwards).  Records updated = n_blocks * 256 * n_iters. */
mcx_status mcx_probe_tally(void* table, uint64_t n_records, int n_blocks, int64_t n_iters, void* cuda_stream);

/* Memory-side probes for the rooflines of the mesh and voxel paths ("measure L2 sector
 * peak").  Both read `table` (DEVICE, n_bytes, a power of two >= 4096; contents irrelevant for mcx_probe_l2, overwritten
 * with a pointer chain by mcx_probe_latency) and write one value per thread to `sink` (DEVICE [n_blocks * 256] uint32).
 *   mcx_probe_l2       every thread does n_iters independent loads of one pseudo-random aligned 32-byte sector (the
 *                      size of a BVH node; read through L1 with ld.global.nc as the walk does) --
 *                      sectors read = n_blocks * 256 * n_iters;
 *   mcx_probe_latency  every thread chases a dependent chain of n_iters 8-byte loads through a random cyclic
 *                      permutation of the table's 32-byte sectors -- loads in flight per thread = 1;
 *                      n_blocks x 256 threads (use 1 block of 32 for the unloaded latency). */
mcx_status mcx_probe_l2(const void* table, uint64_t n_bytes, uint32_t* sink, int n_blocks, int64_t n_iters, void* cuda_stream);
mcx_status mcx_probe_latency(void* table, uint64_t n_bytes, uint32_t* sink, int n_blocks, int n_threads, int64_t n_iters,
                             void* cuda_stream);

void mcx_instrument_destroy(mcx_instrument* inst);

const char* mcx_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MCX_H_ */
