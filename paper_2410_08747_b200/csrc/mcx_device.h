// mcx_device.h -- device-side image of an instrument (what mcx_instrument_create packs into the workspace) and
// the host-side launch interface between mcx_host.cu and mcx_kernels.cu.  Product code: shares nothing with
// oracle/.  Step numbers refer to DESIGN.md "Readings".
#ifndef MCX_DEVICE_H_
#define MCX_DEVICE_H_

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/mcx.h"

namespace mcx {

struct DPose {
  double R[9];
  double T[3];
  int identity, pad;  // R is exactly the identity matrix
};

// mu(E) of one material as ln-tables (step 7); slope[j] = (lnMu[j+1]-lnMu[j]) / (lnE[j+1]-lnE[j]).
struct DMaterial {
  int n;  // 0 = vacuum
  int pad;
  const double* E;
  const double* lnE;
  const double* lnMu;
  const double* slope;
  double inv_dlnE;  // (n-1) / (lnE[n-1]-lnE[0]): first guess of the segment, verified against E[]
  const double* lnMuS;   // step 17: ln of the scattering part of mu on the same grid, and its slopes; null = does not scatter
  const double* slopeS;
};

struct DSource {
  int pos_mode, dir_mode, e_mode, spec_n;
  double radius, sigma_x, sigma_y;
  double target_w, target_h, target_dist, div_x, div_y;
  double e0, de_rel, spec_emin, spec_bin_w;
  const double* cdf;  // [spec_n + 1] running sum of the spectrum
  const int* guide;   // [kSpecGuide + 1]: guide[k] <= the bin holding v = (k / kSpecGuide) cdf[spec_n] (starts the search)
};
enum { kSpecGuide = 2048 };

struct DSlit {
  double half_x, half_y, radius2;
};

// BVH2 node, 32 bytes.  The tree over a mesh is a COMPLETE binary tree of depth D = ceil(log2(n_triangles)), stored in
// heap order with node i at slot i + 1 (children 2i+1, 2i+2 share one 64-byte line), leaves all at level D, leaf
// number p = i - (2^D - 1) holding triangle slot p (slots without a triangle, and subtrees without one, have count 0
// and are never entered).  Nothing needs a pointer: the walk keeps (i, level) and one bit per level for "the right
// sibling is still to be visited", so it needs no stack either.  Boxes are fp32, rounded outward and padded; they only
// select candidate triangles, the exact fp64 triangle test decides.
struct BvhNode {
  float lo[3];
  int count;   // triangles below this node
  float hi[3];
  int unused;
};

struct DSolid {
  int shape, material, priority, depth;  // depth: D of a mesh's BVH
  DPose pose;
  double dims[3];
  double bound2;                  // primitives: (radius of the bounding sphere about the solid's origin, plus 1e-9)^2;
                                  // meshes: the beam limit of the warp-cooperative walk (a length)
  double ctr[3], radius;          // meshes: bounding sphere of the mesh's (padded) box, solid-local
  double unused[2];
  const BvhNode* nodes;
  const double* tris;  // [2^D][9] vertices by leaf number (zeros where a leaf holds no triangle)
};

// The solids of a group are stored in ascending order of precedence (priority, then earlier-listed first among
// equals, step 10): where several overlap, the one with the highest index owns the segment.
struct DSolids {
  int n_solids, n_mesh;
  const DSolid* solids;
  int scatter_order, pad;  // step 17: direction changes allowed per ray in this group; 0 = attenuation only
};

// Voxel volume in traversal layout: kVoxelCellBytes per cell, {material ID, run, radius, 0}, where run = how many cells
// FOLLOWING this one along the fast axis in the beam's direction (run_dir) hold the same ID (capped at 255), and radius =
// the Chebyshev radius of the largest cube of cells around it that holds its ID throughout (capped; mcx_kernels.cu).  Cells are addressed as
// ((i[a2]+1) * (n[a1]+2) + i[a1]+1) * pitch + i[fast]+1, with a one-cell guard border of ID kVoxelGuard all around.
enum { kVoxelCellBytes = 4 };
struct DVoxels {
  double h, inv_h;
  int n[3];       // nx, ny, nz
  int fast;       // axis stored fastest in the traversal layout
  int a1, a2;     // the other two axes
  int pitch;      // cells per row: n[fast] + 2 rounded up to a multiple of 16
  unsigned slab;  // cells per slab: (n[a1] + 2) * pitch
  unsigned mg_pitch, sh_pitch, mg_slab, sh_slab;  // x / pitch, x / slab by multiplication (fast_div in mcx_kernels.cu)
  int run_dir;    // +1 / -1: the direction along the fast axis the runs are counted in (source -> volume)
  int scatter_order;  // step 17: direction changes allowed per ray in the volume; 0 = attenuation only
  const uint8_t* ids;  // cell k at ids[4 k] (ID), ids[4 k + 1] (run), ids[4 k + 2] (radius)
  // Scattering volumes of at most 16 materials: the same cells once more, one byte each: ID in the low four bits, a code
  // of the radius in the high four (codes 0..14 = radius 0..6, 8, 10, 12, 16, 24, 32, 64, 128, rounded down; 0xF0 = guard cell).
  // What scatter_walk_kernel reads: a quarter of the bytes, so that much more of the volume stays in L2.  Null: not built.
  const uint8_t* cmap;
};

struct DMirror {
  double a, b, inv_a2, inv_b2;
  double Z0, Y0, nZ, nY, tZ, tY;
  double half_length, half_width;
  double theta_min, theta_max, e_min, e_max;
  double st, se;  // grid cells per unit: (n_theta - 1) / (theta_max - theta_min), (n_e - 1) / (e_max - e_min)
  int n_theta, n_e;
  const double* table;
};

struct DCrystal {
  double half_length, half_width, d_hkl, zeta, delta0;
  double g, kappa;  // step 13b (Darwin-Prins); 0, 0 = Darwin
};

// Step 16: a stack of double-sided parabolic lenses.  delta(E) is kept as the same ln-tables as mu(E).
struct DLens {
  double inv_R, half_inv_R;  // 1 / R, 1 / (2 R)
  double half_web, pitch, ra2;
  int n_lenses, material;
  DMaterial delta;
};

struct DDetector {
  double xmin, xmax, ymin, ymax, emin, emax;
  double sx, sy, se;  // bins per unit: nx / (xmax - xmin), ...
  int nx, ny, ne, index;
  uint64_t n_bins;
  int mode, pad;  // mcx_det_mode
};

struct DComponent {
  int kind;
  int pad;
  DPose pose;
  union {
    DSource source;
    DSlit slit;
    DSolids solids;
    DVoxels voxels;
    DMirror mirror;
    DCrystal crystal;
    DDetector detector;
    DLens lens;
  } u;
};

// One tally record = one 32-byte sector: a detected ray touches exactly one sector.
struct TallyBin {
  unsigned long long N;
  double P;
  double P2;
  unsigned long long pad;
};

enum { CNT_DETECTED = 0, CNT_MISSED = 1, CNT_DEGENERATE = 2, CNT_OVERFLOW = 3 };

struct alignas(16) DInstrument {
  int n_comps, n_mats, n_dets, features;
  DComponent comps[MCX_MAX_COMPONENTS];
  DMaterial mats[MCX_MAX_MATERIALS];
  TallyBin* tallies[MCX_MAX_DETECTORS];
  unsigned long long* counters;  // [n_comps + 4]
};

static_assert(sizeof(DInstrument) % 16 == 0, "copied to shared memory as int4");
static_assert(sizeof(TallyBin) == 32, "one tally record per 32-byte sector");

// feature bits: select the kernel instantiation (code for absent component kinds is compiled out)
enum { F_SOLIDS = 1, F_MESH = 2, F_VOXELS = 4, F_OPTICS = 8, F_PRIM = 16, F_LENS = 32, F_SCATTER = 64, F_ALL = 127 };  // F_SOLIDS: a solids group; F_PRIM / F_MESH: what it holds

struct PoolRay;

// One trace launch: rays first + offset(q) for positions q in [0, n); offset(q) = order[q] if order != null, else q.
struct TraceArgs {
  uint64_t first, n, seed;
  int n_comps, n_mats, n_solids;  // sizes of the instrument: components, materials, solids of all groups together
  unsigned tile;           // positions per work ticket (set by launch_trace)
  int gate_max;            // components 1..gate_max are slits / mirrors / crystals: candidates for the absorber gate; 0 = off
  int cap_endpoints;       // interval endpoints per ray and solids group held in shared memory (a multiple of 8)
  const uint32_t* order;   // detector-tile order of the chunk (launch_sort), or null
  mcx_ray_fate* dump;      // per-ray records indexed by ray offset, or null = tally
  unsigned int* ticket;    // [2] work-tile ticket and departure count, zero between launches
  unsigned int* gate_known;  // the absorber gate an earlier launch on this instrument settled on, plus 1 (0 = not yet)
  unsigned int* host_flag;   // mapped pinned host word: receives epoch + 1 when a ray overflowed its scratch capacity
  unsigned int epoch;        // number of mcx_tally_reset calls on the handle so far
  int tally_mode;            // mcx_tally_mode (never MCX_TALLY_AUTO here)
  int tally_cache_log2;      // MCX_TALLY_BLOCK: log2 of the slots of the block-private cache (32 bytes each); 0 = none
  unsigned tally_cache_dets; // MCX_TALLY_BLOCK: bit d = detector d's updates go through the cache (its bins fit in it)
  // Staged tracing of a chain with a scattering voxel sample: 0 = the whole chain in one launch;
  // 1 = components 1 .. stage_comp - 1, survivors to the pool; 2 = positions are pool records, components stage_comp + 1 ..
  int stage;
  int stage_comp;
  PoolRay* pool;             // [1 << kPoolCapacityLog2]
  unsigned int* pool_count;  // [4]: records in the pool, next record to hand out, departures of the walk kernel, spare
};

// One ray between the stages of a staged trace: written by stage 1, walked in place by scatter_walk_kernel, read by stage 2.
struct alignas(16) PoolRay {
  double r[3], d[3], E, p;
  uint64_t offset;  // of the ray in the call (ray index - first)
  uint64_t pad;
};
static_assert(sizeof(PoolRay) == 80, "five 16-byte words");
enum { kPoolCapacityLog2 = 22 };  // records (336 MB); a staged chunk holds at most this many rays

// The walk stage: every record of the pool through component `comp` (a scattering voxel volume).
struct WalkArgs {
  uint64_t first, seed;
  int comp, n_mats;
  int compact;                    // walk the one-byte cells (DVoxels::cmap)
  int batch_setup, batch_settle;  // lanes that must wait for a leg set-up / a run end before the warp turns to them
  PoolRay* pool;
  unsigned int* pool_count;
};

// sizes of the sort workspace
enum { MCX_SORT_MAX_G = 11, MCX_SORT_MAX_BUCKETS = 1 << 22, MCX_SORT_MAX_SCAN_BLOCKS = 2048 };

// ---- launch interface (defined in mcx_kernels.cu) ----
cudaError_t launch_trace(const DInstrument* d_inst, int features, int n_mats, const TraceArgs& args, cudaStream_t stream);  // args.cap_endpoints sizes the shared memory
cudaError_t launch_scatter_walk(const DInstrument* d_inst, const WalkArgs& args, uint64_t n_max, cudaStream_t stream);
cudaError_t launch_sort(uint64_t first, uint32_t n, uint64_t seed, int g, unsigned int* cnt, unsigned int* bsum,
                        uint32_t* order, cudaStream_t stream);
cudaError_t launch_tally_read(const TallyBin* bins, uint64_t n_bins, unsigned long long* N, double* p, double* p2,
                              cudaStream_t stream);
cudaError_t launch_voxel_relayout(const uint8_t* src, uint8_t* dst, int nx, int ny, int nz, int fast, int a1, int a2,
                                  int pitch, int run_dir, int n_mats, cudaStream_t stream);
cudaError_t launch_cnr(const unsigned long long* N, const double* p, const double* p2, int nx, int ny, int ne, const int* region_mat,
                       const int* region_ref, double emin, double emax, double e_fit_min, double* cnr_out, double* fit_out,
                       cudaStream_t stream);
cudaError_t launch_cnr_static(const TallyBin* bins, uint64_t n_bins, int nx, int ny, int ne, const int* region_mat, const int* region_ref,
                              double emin, double emax, double e_fit_min, double* cnr_out, double* fit_out, cudaStream_t stream);
cudaError_t launch_voxel_radius(uint8_t* cells, uint8_t* scratch, uint8_t* cmap, int d0, int d1, int d2, cudaStream_t stream);
cudaError_t launch_probe_dfma(double* sink, int n_blocks, long long n_iters, cudaStream_t stream);
cudaError_t launch_probe_tally(void* table, unsigned long long n_records, int n_blocks, long long n_iters, cudaStream_t stream);
cudaError_t launch_probe_l2(const void* table, unsigned long long n_bytes, uint32_t* sink, int n_blocks, long long n_iters,
                            cudaStream_t stream);
cudaError_t launch_probe_latency(void* table, unsigned long long n_bytes, uint32_t* sink, int n_blocks, int n_threads,
                                 long long n_iters, cudaStream_t stream);

}  // namespace mcx
#endif
