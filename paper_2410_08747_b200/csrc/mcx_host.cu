// mcx_host.cu -- the C ABI of include/mcx.h: validation, host-side precomputation (ln-tables, spectrum CDFs,
// mirror constants, BVH build), packing of the device image into the caller's workspace, and kernel launches.
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <new>
#include <vector>

#include "mcx_device.h"

using namespace mcx;

struct mcx_instrument {
  DInstrument host_image;            // what sits at workspace offset 0
  unsigned char* workspace = nullptr;
  size_t workspace_bytes = 0;
  size_t zero_begin = 0, zero_end = 0;  // tallies + counters
  size_t off_staging = 0;
  size_t upload_bytes = 0;              // host -> device bytes moved by create
  int n_comps = 0, n_mats = 0, n_dets = 0, features = 0;
  int cap_endpoints = 16;               // interval endpoints per ray and solids group (shared memory of the trace kernel)
  int n_solids_total = 0;               // solids of all groups together (staged in shared memory by the trace kernel)
  int gate_max = 0;                     // leading slits / mirrors / crystals of the chain (TraceArgs::gate_max)
  bool sort_pays = false;               // AUTO lane scheduling: detector-tile order
  uint64_t det_bins[MCX_MAX_DETECTORS] = {};
  mcx_pose source_pose;                 // for mcx_instrument_set_pose on a voxel volume (layout check)
  mcx_voxels_params voxel_params[MCX_MAX_COMPONENTS];  // sizes of the voxel components (same purpose)
  uint64_t launches = 0;
  // lane scheduling (row a13)
  int exec_mode = MCX_EXEC_AUTO;
  size_t off_ticket = 0, off_gate = 0, off_sort_cnt = 0, off_sort_bsum = 0, off_order = 0;
  uint64_t chunk_rays = 0;  // rays per sorted chunk (<= kChunkCapacity, the order buffer in the workspace)
  int sort_grid_bits = 0;   // 0 = by chunk length (sort_bits)
  bool gate_enabled = true;
  int tally_mode = MCX_TALLY_AUTO;
  // staged trace: the scattering voxel volume the walk stage takes, 0 = none (one launch per chunk)
  int stage_comp = 0;
  bool staged_enabled = true;
  int walk_batch_setup = 16, walk_batch_settle = 12;  // WalkArgs (measured: DESIGN.md 5.4)
  size_t off_pool = 0, off_pool_count = 0;
  // MCX_ERR_CAPACITY: a mapped pinned host word the trace kernel writes (epoch + 1) when a ray overflows its scratch
  unsigned int* host_flag = nullptr;
  unsigned int epoch = 0;   // resets so far: an overflow of an earlier epoch is forgotten
  // mcx_instrument_set_timing: events around the sort and trace_kernel of every chunk (three per chunk, reused)
  bool timing = false;
  std::vector<cudaEvent_t> events;  // pool, 3 per timed chunk
  size_t events_used = 0;
  int64_t timed_launches = 0;  // trace_kernel / scatter_walk_kernel launches between the events recorded so far
  ~mcx_instrument() {
    if (host_flag) cudaFreeHost(host_flag);
    for (cudaEvent_t e : events) cudaEventDestroy(e);
  }
};

namespace {

thread_local char g_err[512] = "";

mcx_status fail(mcx_status s, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return s;
}

mcx_status cuda_fail(cudaError_t e, const char* what) {
  return fail(MCX_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

constexpr size_t kAlign = 256;
size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

// Bump allocator over the workspace.  The same sequence of reserve() calls is made by the size query and by
// create, so both arrive at the same offsets.
struct Arena {
  size_t top = 0;
  size_t reserve(size_t bytes) {
    const size_t off = top;
    top = align_up(top + bytes);
    return off;
  }
};

bool pose_ok(const mcx_pose& P) {
  for (int k = 0; k < 9; ++k) if (!std::isfinite(P.rot[k])) return false;
  for (int k = 0; k < 3; ++k) if (!std::isfinite(P.origin[k])) return false;
  return true;
}

void copy_pose(DPose* d, const mcx_pose& s) {
  std::memcpy(d->R, s.rot, sizeof(d->R));
  std::memcpy(d->T, s.origin, sizeof(d->T));
  d->identity = 1;
  for (int k = 0; k < 9; ++k)
    if (s.rot[k] != ((k % 4 == 0) ? 1.0 : 0.0)) d->identity = 0;
  d->pad = 0;
}

// ---------------------------------------------------------------------------------------------------------
// BVH over one mesh: a complete binary tree in heap order (BvhNode), built top-down by splitting the triangles of a
// node at the median of their centroids along the widest axis, the left child taking the larger half.  Node boxes
// are stored in fp32 rounded outward and padded by 2^-16 of the mesh scale, far above the fp32 rounding of the box
// walk (<= a few 2^-24 of the scale), so the walk never loses a triangle the exact fp64 test would hit.
// ---------------------------------------------------------------------------------------------------------
struct TriRef {
  double c[3], lo[3], hi[3];
  int idx;
};

float round_down(double x) {
  float f = (float)x;
  if ((double)f > x) f = std::nextafterf(f, -std::numeric_limits<float>::infinity());
  return f;
}
float round_up(double x) {
  float f = (float)x;
  if ((double)f < x) f = std::nextafterf(f, std::numeric_limits<float>::infinity());
  return f;
}

int bvh_depth(int64_t n_tris) {
  int d = 0;
  while (((int64_t)1 << d) < n_tris) ++d;
  return d;
}
size_t bvh_node_bound(int64_t n_tris) { return (size_t)2 << bvh_depth(n_tris); }  // slots: node i at slot i + 1
size_t bvh_leaf_count(int64_t n_tris) { return (size_t)1 << bvh_depth(n_tris); }

struct BvhBuilder {
  std::vector<TriRef>& refs;
  std::vector<BvhNode>& slots;  // zero-initialised: count 0 everywhere
  std::vector<int>& leaf_tri;   // triangle (index into the caller's array) of every leaf, -1 = none
  double pad;
  int depth;
  void build(int64_t i, int begin, int end, int level) {
    const int count = end - begin;
    if (count == 0) return;
    BvhNode& N = slots[(size_t)i + 1];
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    double clo[3] = {1e300, 1e300, 1e300}, chi[3] = {-1e300, -1e300, -1e300};
    for (int k = begin; k < end; ++k)
      for (int a = 0; a < 3; ++a) {
        lo[a] = std::min(lo[a], refs[k].lo[a]); hi[a] = std::max(hi[a], refs[k].hi[a]);
        clo[a] = std::min(clo[a], refs[k].c[a]); chi[a] = std::max(chi[a], refs[k].c[a]);
      }
    for (int a = 0; a < 3; ++a) {
      N.lo[a] = round_down(lo[a] - pad);
      N.hi[a] = round_up(hi[a] + pad);
    }
    N.count = count;
    if (level == depth) {  // count == 1: 2^(depth - level) bounds the triangles of a node
      leaf_tri[(size_t)(i - (((int64_t)1 << depth) - 1))] = refs[begin].idx;
      return;
    }
    int axis = 0;
    if (chi[1] - clo[1] > chi[axis] - clo[axis]) axis = 1;
    if (chi[2] - clo[2] > chi[axis] - clo[axis]) axis = 2;
    const int mid = begin + (count + 1) / 2;
    if (mid < end)
      std::nth_element(refs.begin() + begin, refs.begin() + mid, refs.begin() + end,
                       [axis](const TriRef& x, const TriRef& y) { return x.c[axis] < y.c[axis]; });
    build(2 * i + 1, begin, mid, level + 1);
    build(2 * i + 2, mid, end, level + 1);
  }
};

// Rays per sorted chunk.  The more rays a chunk holds the closer together the 32 rays of a warp land (the bucket grid
// is capped at 2^10 x 2^10 cells, so past 2^24 rays the buckets only get fuller and a warp spans less of one): c4
// gains 6 % from 2^24 to 2^26 and 1 % more at 2^28; the order buffer (4 B per ray, 256 MiB) is streamed once each
// way.  mcx_instrument_set_tuning can shorten the chunks (tests, sweeps); the workspace always holds a full one.
constexpr int kChunkLog2Max = 26, kChunkLog2Min = 14;
constexpr uint64_t kChunkCapacity = (uint64_t)1 << kChunkLog2Max;
constexpr uint64_t kSortMinRays = 1u << 14;  // shorter chunks are traced in index order

// Bits per axis of the bucket grid: at least 64 rays per bucket, at most 2^10 x 2^10 cells (a finer grid measured no
// gain on c3 / c4), and 2^9 x 2^9 where the instrument has only analytic solids: there coherence of the branches is
// all the order buys, and the coarser grid keeps the scatter's write fronts L2-resident (c1: 7 % faster than 2^10).
int sort_bits(uint64_t n, int features, int forced) {
  if (forced) return forced;
  const int g_max = (features & (F_MESH | F_VOXELS)) ? 10 : 9;
  int g = 1;
  while (g < g_max && ((uint64_t)64 << (2 * (g + 1))) <= n) ++g;
  return g;
}

// sizes and offsets of everything in the workspace
struct Plan {
  size_t off_inst = 0;
  size_t blob_begin = 0, blob_end = 0;  // tables, built on the host
  size_t off_voxels[MCX_MAX_COMPONENTS];
  size_t off_vox_scratch[MCX_MAX_COMPONENTS];
  size_t off_cmap[MCX_MAX_COMPONENTS];  // 0 = none
  size_t off_tally[MCX_MAX_DETECTORS];
  size_t off_counters = 0;
  size_t zero_begin = 0, zero_end = 0;
  size_t off_staging = 0;  // N, p, p2 of the largest detector, for mcx_tally_read_host
  size_t off_ticket = 0, off_gate = 0, off_sort_cnt = 0, off_sort_bsum = 0, off_order = 0;
  size_t off_pool = 0, off_pool_count = 0;
  int stage_comp = 0;
  size_t total = 0;
  // blob offsets
  size_t off_mat[MCX_MAX_MATERIALS];      // 4 arrays of n doubles each
  size_t off_cdf[MCX_MAX_COMPONENTS];
  size_t off_guide[MCX_MAX_COMPONENTS];
  size_t off_table[MCX_MAX_COMPONENTS];
  size_t off_solids[MCX_MAX_COMPONENTS];  // DSolid array
  size_t off_nodes[MCX_MAX_COMPONENTS][MCX_MAX_SOLIDS];
  size_t off_tris[MCX_MAX_COMPONENTS][MCX_MAX_SOLIDS];
};

// traversal layout of a voxel volume: one guard cell on every side, rows padded to 16 bytes
int voxel_pitch(int64_t n_fast) { return (int)((n_fast + 2 + 15) / 16 * 16); }
size_t voxel_bytes(int64_t n_fast, int64_t n_1, int64_t n_2) { return (size_t)kVoxelCellBytes * (size_t)(n_2 + 2) * (size_t)(n_1 + 2) * (size_t)voxel_pitch(n_fast); }
// The walk issues the loads of the slab after the one it is looking at; past a guard cell these reach at most one step
// along every axis further.  That much of the workspace on either side of the volume belongs to the volume.
size_t voxel_pad(int64_t n_fast, int64_t n_1) { return align_up((size_t)kVoxelCellBytes * ((size_t)(n_1 + 3) * (size_t)voxel_pitch(n_fast) + 16)); }

// n / d == (t + ((n - t) >> 1)) >> sh with t = mulhi(m, n), for every 32-bit n and d >= 2 (Granlund & Montgomery 1994,
// "Division by invariant integers using multiplication", the 33-bit multiplier case)
void fast_div_constants(unsigned d, unsigned* m, unsigned* sh) {
  unsigned L = 0;
  while (((uint64_t)1 << L) < d) ++L;  // ceil(log2 d) >= 1
  *m = (unsigned)((((uint64_t)1 << 32) * (((uint64_t)1 << L) - d)) / d + 1);
  *sh = L - 1;
}

// chooses the axis stored fastest: the voxel axis most aligned with the line from the source to the volume centre
void voxel_axes(const mcx_component& src, const mcx_component& vox, int* fast, int* a1, int* a2, int* run_dir) {
  const mcx_voxels_params& V = vox.u.voxels;
  const double half[3] = {0.5 * V.nx * V.h, 0.5 * V.ny * V.h, 0.5 * V.nz * V.h};
  // volume centre in lab coordinates: origin + R^T half
  double dirl[3];
  for (int a = 0; a < 3; ++a) {
    double c = vox.pose.origin[a];
    for (int k = 0; k < 3; ++k) c += vox.pose.rot[3 * k + a] * half[k];
    dirl[a] = c - src.pose.origin[a];
  }
  double best = -1.0;
  *fast = 2;
  *run_dir = 1;
  for (int k = 0; k < 3; ++k) {
    const double comp = vox.pose.rot[3 * k] * dirl[0] + vox.pose.rot[3 * k + 1] * dirl[1] + vox.pose.rot[3 * k + 2] * dirl[2];
    if (std::fabs(comp) > best) { best = std::fabs(comp); *fast = k; *run_dir = comp < 0.0 ? -1 : 1; }
  }
  *a1 = (*fast + 1) % 3;
  *a2 = (*fast + 2) % 3;
  if (*a1 > *a2) std::swap(*a1, *a2);
}

// Staged trace: where the chain holds a scattering voxel volume and nothing else that needs scratch
// or optics code (the kernel instantiation F_VOXELS | F_SCATTER), the first such volume is walked by a kernel of its
// own between the part of the chain before it and the part after it.  Returns its component index, 0 = not staged.
int staged_component(const mcx_component* comps, int n_comps) {
  int first = 0;
  for (int c = 1; c < n_comps; ++c) {
    const int k = comps[c].kind;
    if (k == MCX_SOLIDS || k == MCX_MIRROR_ELLIPTIC || k == MCX_CRYSTAL_BRAGG || k == MCX_LENS_PARAB) return 0;
    if (k == MCX_VOXELS && comps[c].u.voxels.scatter_order > 0 && first == 0) first = c;
  }
  return first;
}

mcx_status make_plan(const mcx_component* comps, int n_comps, const mcx_material* mats, int n_mats, Plan* P) {
  if (!comps || n_comps < 1) return fail(MCX_ERR_INVALID_ARG, "no components");
  if (n_comps > MCX_MAX_COMPONENTS) return fail(MCX_ERR_UNSUPPORTED, "more than %d components", MCX_MAX_COMPONENTS);
  if (n_mats < 0 || n_mats > MCX_MAX_MATERIALS) return fail(MCX_ERR_UNSUPPORTED, "more than %d materials", MCX_MAX_MATERIALS);
  if (n_mats > 0 && !mats) return fail(MCX_ERR_INVALID_ARG, "materials is null");
  if (comps[0].kind != MCX_SOURCE) return fail(MCX_ERR_INVALID_ARG, "component 0 must be a source");
  Arena A;
  P->off_inst = A.reserve(sizeof(DInstrument));
  P->blob_begin = A.top;
  for (int m = 0; m < n_mats; ++m) {
    if (mats[m].n_points < 0 || mats[m].n_points == 1) return fail(MCX_ERR_INVALID_ARG, "material %d: n_points must be 0 or >= 2", m);
    P->off_mat[m] = A.reserve((size_t)mats[m].n_points * (mats[m].mu_scatter_per_m ? 6 : 4) * sizeof(double));
  }
  int n_dets = 0;
  for (int c = 0; c < n_comps; ++c) {
    const mcx_component& C = comps[c];
    if (c > 0 && C.kind == MCX_SOURCE) return fail(MCX_ERR_INVALID_ARG, "component %d: only component 0 may be a source", c);
    if (!pose_ok(C.pose)) return fail(MCX_ERR_INVALID_ARG, "component %d: pose is not finite", c);
    switch (C.kind) {
      case MCX_SOURCE:
        if (C.u.source.energy_mode == MCX_E_SPECTRUM) {
          if (C.u.source.spec_n < 1) return fail(MCX_ERR_INVALID_ARG, "source: empty spectrum");
          P->off_cdf[c] = A.reserve((size_t)(C.u.source.spec_n + 1) * sizeof(double));
          P->off_guide[c] = A.reserve((size_t)(kSpecGuide + 1) * sizeof(int));
        }
        break;
      case MCX_SLIT_RECT: case MCX_SLIT_CIRC: case MCX_CRYSTAL_BRAGG: break;
      case MCX_LENS_PARAB:
        if (C.u.lens.n_delta < 2) return fail(MCX_ERR_INVALID_ARG, "component %d: the delta(E) table needs >= 2 points", c);
        P->off_table[c] = A.reserve((size_t)C.u.lens.n_delta * 4 * sizeof(double));
        break;
      case MCX_SOLIDS: {
        const mcx_solids_params& G = C.u.solids;
        if (G.n_solids < 0 || G.n_solids > MCX_MAX_SOLIDS) return fail(MCX_ERR_UNSUPPORTED, "component %d: more than %d solids", c, MCX_MAX_SOLIDS);
        if (G.n_solids > 0 && !G.solids) return fail(MCX_ERR_INVALID_ARG, "component %d: solids is null", c);
        P->off_solids[c] = A.reserve((size_t)std::max<int64_t>(G.n_solids, 1) * sizeof(DSolid));
        for (int64_t s = 0; s < G.n_solids; ++s)
          if (G.solids[s].shape == MCX_MESH) {
            if (G.solids[s].n_triangles < 1 || G.solids[s].n_vertices < 3) return fail(MCX_ERR_INVALID_ARG, "component %d solid %d: empty mesh", c, (int)s);
            P->off_nodes[c][s] = A.reserve(bvh_node_bound(G.solids[s].n_triangles) * sizeof(BvhNode));
            P->off_tris[c][s] = A.reserve(bvh_leaf_count(G.solids[s].n_triangles) * 9 * sizeof(double));
          }
        break;
      }
      case MCX_VOXELS: break;  // below, outside the blob
      case MCX_MIRROR_ELLIPTIC:
        if (C.u.mirror.n_theta < 2 || C.u.mirror.n_e < 2) return fail(MCX_ERR_INVALID_ARG, "component %d: reflectivity grid needs >= 2x2 points", c);
        P->off_table[c] = A.reserve((size_t)C.u.mirror.n_theta * C.u.mirror.n_e * sizeof(double));
        break;
      case MCX_DETECTOR:
        if (n_dets >= MCX_MAX_DETECTORS) return fail(MCX_ERR_UNSUPPORTED, "more than %d detectors", MCX_MAX_DETECTORS);
        if (C.u.detector.nx < 1 || C.u.detector.ny < 1 || C.u.detector.ne < 1) return fail(MCX_ERR_INVALID_ARG, "component %d: empty detector", c);
        ++n_dets;
        break;
      default: return fail(MCX_ERR_INVALID_ARG, "component %d: unknown kind %d", c, C.kind);
    }
  }
  P->blob_end = A.top;
  for (int c = 0; c < n_comps; ++c)
    if (comps[c].kind == MCX_VOXELS) {
      const mcx_voxels_params& V = comps[c].u.voxels;
      if (V.nx < 1 || V.ny < 1 || V.nz < 1 || V.nx > 4096 || V.ny > 4096 || V.nz > 4096 || !(V.h > 0.0))
        return fail(MCX_ERR_INVALID_ARG, "component %d: bad voxel grid", c);
      int f, a1, a2;
      int run_dir;
      voxel_axes(comps[0], comps[c], &f, &a1, &a2, &run_dir);
      const int64_t n[3] = {V.nx, V.ny, V.nz};
      if (voxel_bytes(n[f], n[a1], n[a2]) + 2 * voxel_pad(n[f], n[a1]) > 0xFFFFFFFFull)
        return fail(MCX_ERR_UNSUPPORTED, "component %d: voxel volume above 2^30 cells (the walk uses 32-bit byte offsets, 4 bytes per cell)", c);
      // twice the size: create shifts the volume past a 4 GiB address boundary if it would straddle one
      P->off_voxels[c] = A.reserve(2 * voxel_bytes(n[f], n[a1], n[a2]) + 4 * voxel_pad(n[f], n[a1]));
      // two scratch arrays of one byte per cell for the radius transform at create
      P->off_vox_scratch[c] = A.reserve(voxel_bytes(n[f], n[a1], n[a2]) / kVoxelCellBytes * 2);
      // The one-byte cells of a scattering volume (DVoxels::cmap: four bits of ID), placed by the same rule as the volume.
      // Built where they fit in L2 (126 MB on B200) with room to spare: there the walk stage runs out of L2 instead of DRAM
      // (c8, 66 MB: +16 %); a larger volume misses either way and does better with the exact radii and the runs of the
      // four-byte cells (c9, 134 MB: -2 %).
      P->off_cmap[c] = (V.scatter_order > 0 && n_mats <= 16 && voxel_bytes(n[f], n[a1], n[a2]) / kVoxelCellBytes <= ((size_t)96 << 20))
                           ? A.reserve((2 * voxel_bytes(n[f], n[a1], n[a2]) + 4 * voxel_pad(n[f], n[a1])) / kVoxelCellBytes + 2 * kAlign)
                           : 0;
    }
  P->zero_begin = A.top;
  int d = 0;
  for (int c = 0; c < n_comps; ++c)
    if (comps[c].kind == MCX_DETECTOR) {
      const mcx_detector_params& D = comps[c].u.detector;
      P->off_tally[d++] = A.reserve((size_t)D.nx * D.ny * D.ne * sizeof(TallyBin));
    }
  P->off_counters = A.reserve((size_t)MCX_N_COUNTERS(n_comps) * sizeof(unsigned long long));
  P->off_ticket = A.reserve(2 * sizeof(unsigned int));
  P->zero_end = A.top;
  P->off_gate = A.reserve(sizeof(unsigned int));  // zeroed by create only: survives mcx_tally_reset
  size_t max_bins = 0;
  for (int c = 0; c < n_comps; ++c)
    if (comps[c].kind == MCX_DETECTOR)
      max_bins = std::max(max_bins, (size_t)comps[c].u.detector.nx * comps[c].u.detector.ny * comps[c].u.detector.ne);
  P->off_staging = A.reserve(max_bins * 24);
  P->off_sort_cnt = A.reserve((size_t)MCX_SORT_MAX_BUCKETS * sizeof(unsigned int));
  P->off_sort_bsum = A.reserve((size_t)MCX_SORT_MAX_SCAN_BLOCKS * sizeof(unsigned int));
  P->off_order = A.reserve((size_t)kChunkCapacity * sizeof(uint32_t));
  P->stage_comp = staged_component(comps, n_comps);
  if (P->stage_comp > 0) {
    P->off_pool_count = A.reserve(4 * sizeof(unsigned int));
    P->off_pool = A.reserve(((size_t)1 << kPoolCapacityLog2) * sizeof(PoolRay));
  }
  P->total = A.top;
  return MCX_OK;
}

mcx_status check_sticky() {
  const cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) return cuda_fail(e, "earlier CUDA error");
  return MCX_OK;
}

// include/mcx.h "Errors": has a trace of the current reset epoch, finished on the device, overflowed a per-ray capacity?
bool capacity_overflowed(const mcx_instrument* H) {
  return H->host_flag && *reinterpret_cast<volatile unsigned int*>(H->host_flag) == H->epoch + 1u;
}
mcx_status capacity_status(const mcx_instrument* H) {
  if (!capacity_overflowed(H)) return MCX_OK;
  return fail(MCX_ERR_CAPACITY, "rays overflowed the per-ray end-point capacity (%d) of a solids group and were dropped as "
              "degenerate; mcx_trace_status / mcx_counters_read give the count", H->cap_endpoints);
}

}  // namespace

extern "C" {

const char* mcx_last_error(void) { return g_err; }

mcx_status mcx_instrument_workspace_size(const mcx_component* components, int n_components, const mcx_material* materials,
                                         int n_materials, size_t* bytes_out) {
  if (!bytes_out) return fail(MCX_ERR_INVALID_ARG, "bytes_out is null");
  Plan P;
  const mcx_status s = make_plan(components, n_components, materials, n_materials, &P);
  if (s != MCX_OK) return s;
  *bytes_out = P.total;
  return MCX_OK;
}

mcx_status mcx_instrument_create(const mcx_component* components, int n_components, const mcx_material* materials,
                                 int n_materials, void* workspace, size_t workspace_bytes, void* cuda_stream,
                                 mcx_instrument** out) {
  if (!out) return fail(MCX_ERR_INVALID_ARG, "out is null");
  *out = nullptr;
  Plan P;
  mcx_status st = make_plan(components, n_components, materials, n_materials, &P);
  if (st != MCX_OK) return st;
  if (!workspace || ((uintptr_t)workspace % kAlign) != 0) return fail(MCX_ERR_WORKSPACE, "workspace is null or not 256-byte aligned");
  if (workspace_bytes < P.total) return fail(MCX_ERR_WORKSPACE, "workspace has %zu bytes, %zu needed", workspace_bytes, P.total);
  if ((st = check_sticky()) != MCX_OK) return st;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  unsigned char* ws = (unsigned char*)workspace;

  mcx_instrument* H = new (std::nothrow) mcx_instrument();
  if (!H) return fail(MCX_ERR_INVALID_ARG, "out of host memory");
  H->workspace = ws;
  H->workspace_bytes = workspace_bytes;
  H->n_comps = n_components;
  H->n_mats = n_materials;
  H->zero_begin = P.zero_begin;
  H->zero_end = P.zero_end;
  H->off_staging = P.off_staging;
  H->off_ticket = P.off_ticket;
  H->off_gate = P.off_gate;
  H->off_sort_cnt = P.off_sort_cnt;
  H->off_sort_bsum = P.off_sort_bsum;
  H->off_order = P.off_order;
  H->off_pool = P.off_pool;
  H->off_pool_count = P.off_pool_count;
  H->stage_comp = P.stage_comp;
  H->chunk_rays = kChunkCapacity;
  // host copy of the table section; consumed by the upload below (a copy from pageable memory has been staged when
  // cudaMemcpyAsync returns), so it lives only as long as this call
  std::vector<unsigned char> blob_storage(P.blob_end - P.blob_begin, 0);
  unsigned char* blob = blob_storage.data();
  auto host_ptr = [&](size_t off) { return blob + (off - P.blob_begin); };
  auto dev_ptr = [&](size_t off) { return ws + off; };
  DInstrument& I = H->host_image;
  std::memset(&I, 0, sizeof(I));
  I.n_comps = n_components;
  I.n_mats = n_materials;
  int features = 0, cap_endpoints = 16;  // a ray through a mesh vertex makes one hit per triangle around it, on both sides

#define MCX_BAIL(status, ...) do { const mcx_status s_ = fail(status, __VA_ARGS__); delete H; return s_; } while (0)

  // ---- materials: ln-tables (step 7) ----
  for (int m = 0; m < n_materials; ++m) {
    const mcx_material& M = materials[m];
    DMaterial& D = I.mats[m];
    D.n = (int)M.n_points;
    if (M.n_points == 0) continue;
    if (!M.energy_keV || !M.mu_per_m) MCX_BAIL(MCX_ERR_INVALID_ARG, "material %d: null table", m);
    const size_t n = (size_t)M.n_points;
    double* E = (double*)host_ptr(P.off_mat[m]);
    double* lnE = E + n;
    double* lnMu = lnE + n;
    double* slope = lnMu + n;
    for (size_t j = 0; j < n; ++j) {
      if (!(M.energy_keV[j] > 0.0) || !(M.mu_per_m[j] > 0.0)) MCX_BAIL(MCX_ERR_RANGE, "material %d: non-positive table entry %zu", m, j);
      if (j > 0 && !(M.energy_keV[j] > M.energy_keV[j - 1])) MCX_BAIL(MCX_ERR_RANGE, "material %d: energies not increasing at %zu", m, j);
      E[j] = M.energy_keV[j];
      lnE[j] = std::log(M.energy_keV[j]);
      lnMu[j] = std::log(M.mu_per_m[j]);
    }
    for (size_t j = 0; j + 1 < n; ++j) slope[j] = (lnMu[j + 1] - lnMu[j]) / (lnE[j + 1] - lnE[j]);
    slope[n - 1] = 0.0;
    D.E = (const double*)dev_ptr(P.off_mat[m]);
    D.lnE = D.E + n;
    D.lnMu = D.lnE + n;
    D.slope = D.lnMu + n;
    D.inv_dlnE = (double)(n - 1) / (lnE[n - 1] - lnE[0]);
    if (M.mu_scatter_per_m) {  // step 17: the scattering part, same grid
      double* lnS = slope + n;
      double* slopeS = lnS + n;
      for (size_t j = 0; j < n; ++j) {
        if (!(M.mu_scatter_per_m[j] > 0.0) || !(M.mu_scatter_per_m[j] <= M.mu_per_m[j]))
          MCX_BAIL(MCX_ERR_RANGE, "material %d: mu_scatter must be in (0, mu] (entry %zu)", m, j);
        lnS[j] = std::log(M.mu_scatter_per_m[j]);
      }
      for (size_t j = 0; j + 1 < n; ++j) slopeS[j] = (lnS[j + 1] - lnS[j]) / (lnE[j + 1] - lnE[j]);
      slopeS[n - 1] = 0.0;
      D.lnMuS = D.slope + n;
      D.slopeS = D.lnMuS + n;
    }
  }

  int n_dets = 0;
  for (int c = 0; c < n_components; ++c) {
    const mcx_component& C = components[c];
    DComponent& D = I.comps[c];
    D.kind = C.kind;
    copy_pose(&D.pose, C.pose);
    switch (C.kind) {
      case MCX_SOURCE: {
        const mcx_source_params& S = C.u.source;
        DSource& d = D.u.source;
        if (S.pos_mode < 0 || S.pos_mode > 2 || S.dir_mode < 0 || S.dir_mode > 1 || S.energy_mode < 0 || S.energy_mode > 2)
          MCX_BAIL(MCX_ERR_INVALID_ARG, "source: bad mode");
        d.pos_mode = S.pos_mode; d.dir_mode = S.dir_mode; d.e_mode = S.energy_mode;
        d.radius = S.radius; d.sigma_x = S.sigma_x; d.sigma_y = S.sigma_y;
        d.target_w = S.target_w; d.target_h = S.target_h; d.target_dist = S.target_dist;
        d.div_x = S.div_x; d.div_y = S.div_y; d.e0 = S.e0; d.de_rel = S.de_rel;
        if (S.energy_mode == MCX_E_SPECTRUM) {
          if (!S.spectrum) MCX_BAIL(MCX_ERR_INVALID_ARG, "source: spectrum is null");
          if (!(S.spec_emax > S.spec_emin)) MCX_BAIL(MCX_ERR_RANGE, "source: empty spectrum range");
          double* cdf = (double*)host_ptr(P.off_cdf[c]);
          cdf[0] = 0.0;
          for (int64_t j = 0; j < S.spec_n; ++j) {  // plain running sum (step 3)
            if (!(S.spectrum[j] >= 0.0)) MCX_BAIL(MCX_ERR_RANGE, "source: negative spectrum bin %lld", (long long)j);
            cdf[j + 1] = cdf[j] + S.spectrum[j];
          }
          if (!(cdf[S.spec_n] > 0.0)) MCX_BAIL(MCX_ERR_RANGE, "source: spectrum sums to zero");
          d.spec_n = (int)S.spec_n;
          d.spec_emin = S.spec_emin;
          d.spec_bin_w = (S.spec_emax - S.spec_emin) / (double)S.spec_n;
          d.cdf = (const double*)dev_ptr(P.off_cdf[c]);
          // guide table: where the inverse-CDF search of step 3 may start for v in [k, k+1) / kSpecGuide of the total
          // (one bin below the exact answer for the lower edge; the kernel verifies its bracket and falls back to
          // the whole table, so the table only has to be nearly right)
          int* guide = (int*)host_ptr(P.off_guide[c]);
          int64_t j = 0;
          for (int k = 0; k <= kSpecGuide; ++k) {
            const double v = ((double)k / (double)kSpecGuide) * cdf[S.spec_n];
            while (j + 1 < S.spec_n && cdf[j + 1] <= v) ++j;
            guide[k] = (int)std::max<int64_t>(j - 1, 0);
          }
          d.guide = (const int*)dev_ptr(P.off_guide[c]);
        }
        break;
      }
      case MCX_SLIT_RECT:
        D.u.slit.half_x = 0.5 * C.u.slit.xw;
        D.u.slit.half_y = 0.5 * C.u.slit.yh;
        break;
      case MCX_SLIT_CIRC:
        D.u.slit.radius2 = C.u.slit.radius * C.u.slit.radius;
        break;
      case MCX_SOLIDS: {
        features |= F_SOLIDS;
        const mcx_solids_params& G = C.u.solids;
        DSolid* hs = (DSolid*)host_ptr(P.off_solids[c]);
        D.u.solids.n_solids = (int)G.n_solids;
        D.u.solids.solids = (const DSolid*)dev_ptr(P.off_solids[c]);
        if (G.scatter_order < 0 || G.scatter_order > MCX_MAX_SCATTER_ORDER) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: bad scatter_order", c);
        D.u.solids.scatter_order = (int)G.scatter_order;
        if (G.scatter_order > 0) features |= F_SCATTER;
        // device order = ascending precedence: by priority, among equals the LATER-listed first (step 10: the earlier
        // solid wins a tie), so that the owner of an overlap is the solid with the highest device index
        int pos[MCX_MAX_SOLIDS];
        {
          int order[MCX_MAX_SOLIDS];
          for (int k = 0; k < (int)G.n_solids; ++k) order[k] = k;
          std::sort(order, order + G.n_solids, [&](int x, int y) {
            if (G.solids[x].priority != G.solids[y].priority) return G.solids[x].priority < G.solids[y].priority;
            return x > y;
          });
          for (int k = 0; k < (int)G.n_solids; ++k) pos[order[k]] = k;
        }
        int n_prim = 0, n_mesh = 0;
        for (int64_t s = 0; s < G.n_solids; ++s) (G.solids[s].shape == MCX_MESH ? n_mesh : n_prim)++;
        cap_endpoints = std::max(cap_endpoints, std::min(48, (2 * n_prim + 8 * n_mesh + 7) / 8 * 8));
        for (int64_t s = 0; s < G.n_solids; ++s) {
          const mcx_solid& S = G.solids[s];
          DSolid& d = hs[pos[s]];
          if (S.shape < 0 || S.shape > 3) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d solid %d: bad shape", c, (int)s);
          if (S.material < 0 || S.material >= n_materials) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d solid %d: material out of range", c, (int)s);
          if (!pose_ok(S.pose)) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d solid %d: pose is not finite", c, (int)s);
          d.shape = S.shape; d.material = S.material; d.priority = S.priority;
          copy_pose(&d.pose, S.pose);
          for (int k = 0; k < 3; ++k) d.dims[k] = S.dims[k];
          {  // bounding sphere about the solid's origin: box half-diagonal, sphere radius, cylinder (radius, half height)
            const double r2 = S.shape == MCX_BOX ? S.dims[0] * S.dims[0] + S.dims[1] * S.dims[1] + S.dims[2] * S.dims[2]
                            : S.shape == MCX_SPHERE ? S.dims[0] * S.dims[0] : S.dims[0] * S.dims[0] + S.dims[1] * S.dims[1];
            d.bound2 = r2 * (1.0 + 2e-9);
          }
          if (S.shape != MCX_MESH) { features |= F_PRIM; continue; }
          features |= F_MESH;
          D.u.solids.n_mesh++;
          if (!S.vertices || !S.triangles) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d solid %d: null mesh arrays", c, (int)s);
          const int nt = (int)S.n_triangles;
          std::vector<TriRef> refs((size_t)nt);
          double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
          for (int t = 0; t < nt; ++t) {
            TriRef& r = refs[t];
            r.idx = t;
            for (int a = 0; a < 3; ++a) { r.lo[a] = 1e300; r.hi[a] = -1e300; r.c[a] = 0.0; }
            for (int v = 0; v < 3; ++v) {
              const int32_t vi = S.triangles[3 * (size_t)t + v];
              if (vi < 0 || vi >= S.n_vertices) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d solid %d: vertex index out of range", c, (int)s);
              for (int a = 0; a < 3; ++a) {
                const double x = S.vertices[3 * (size_t)vi + a];
                r.lo[a] = std::min(r.lo[a], x); r.hi[a] = std::max(r.hi[a], x); r.c[a] += x / 3.0;
              }
            }
            for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], r.lo[a]); hi[a] = std::max(hi[a], r.hi[a]); }
          }
          double scale = 0.0;
          for (int a = 0; a < 3; ++a) scale = std::max(scale, std::max(std::fabs(lo[a]), std::fabs(hi[a])));
          const double pad = scale * (1.0 / 65536.0);
          if ((size_t)nt >= ((size_t)1 << 27)) MCX_BAIL(MCX_ERR_UNSUPPORTED, "component %d solid %d: more than 2^27 triangles", c, (int)s);
          std::vector<BvhNode> slots(bvh_node_bound(nt), BvhNode{});
          std::vector<int> leaf_tri(bvh_leaf_count(nt), -1);
          BvhBuilder B{refs, slots, leaf_tri, pad, bvh_depth(nt)};
          B.build(0, 0, nt, 0);
          std::memcpy(host_ptr(P.off_nodes[c][s]), slots.data(), slots.size() * sizeof(BvhNode));
          double* tri = (double*)host_ptr(P.off_tris[c][s]);  // zero-filled blob: leaves without a triangle stay zero
          for (size_t leaf = 0; leaf < leaf_tri.size(); ++leaf)
            if (leaf_tri[leaf] >= 0)
              for (int v = 0; v < 3; ++v)
                for (int a = 0; a < 3; ++a)
                  tri[9 * leaf + 3 * v + a] = S.vertices[3 * (size_t)S.triangles[3 * (size_t)leaf_tri[leaf] + v] + a];
          {  // bounding sphere of the padded box (participation test and parameter range of the mesh walk)
            double r2 = 0.0;
            for (int a = 0; a < 3; ++a) {
              d.ctr[a] = 0.5 * (lo[a] + hi[a]);
              const double half = 0.5 * (hi[a] - lo[a]) + pad;
              r2 += half * half;
            }
            d.radius = std::sqrt(r2) * (1.0 + 1e-12);
          }
          {  // beam limit of the warp-cooperative walk (mesh_endpoints_beam): the rays of a warp may lie apart by up to
             // half the mean extent of a triangle's box; wider beams collect too many candidates to pay
            double sum = 0.0;
            for (int t = 0; t < nt; ++t) {
              double ext = 0.0;
              for (int a = 0; a < 3; ++a) ext = std::max(ext, refs[t].hi[a] - refs[t].lo[a]);
              sum += ext;
            }
            d.bound2 = 0.5 * sum / (double)nt;
          }
          d.depth = bvh_depth(nt);
          d.nodes = (const BvhNode*)dev_ptr(P.off_nodes[c][s]);
          d.tris = (const double*)dev_ptr(P.off_tris[c][s]);
        }
        break;
      }
      case MCX_VOXELS: {
        features |= F_VOXELS;
        const mcx_voxels_params& V = C.u.voxels;
        if (!V.ids) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: ids is null", c);
        if (n_materials < 1) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: a voxel volume needs a materials array (ID 0 = materials[0])", c);
        DVoxels& d = D.u.voxels;
        if (V.scatter_order < 0 || V.scatter_order > MCX_MAX_SCATTER_ORDER) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: bad scatter_order", c);
        d.scatter_order = (int)V.scatter_order;
        if (V.scatter_order > 0) features |= F_SCATTER;
        d.h = V.h;
        d.inv_h = 1.0 / V.h;
        d.n[0] = (int)V.nx; d.n[1] = (int)V.ny; d.n[2] = (int)V.nz;
        voxel_axes(components[0], C, &d.fast, &d.a1, &d.a2, &d.run_dir);
        d.pitch = voxel_pitch(d.n[d.fast]);
        d.slab = (unsigned)(d.n[d.a1] + 2) * (unsigned)d.pitch;
        fast_div_constants((unsigned)d.pitch, &d.mg_pitch, &d.sh_pitch);
        fast_div_constants(d.slab, &d.mg_slab, &d.sh_slab);
        {  // keep [ids - pad, ids + bytes + pad) inside one 4 GiB window of the address space (32-bit stepping in the walk)
          const size_t bytes = voxel_bytes(d.n[d.fast], d.n[d.a1], d.n[d.a2]);
          const size_t pad = voxel_pad(d.n[d.fast], d.n[d.a1]);
          uintptr_t p0 = (uintptr_t)dev_ptr(P.off_voxels[c]) + pad;
          if (((p0 - pad) >> 32) != ((p0 + bytes + pad - 1) >> 32)) p0 = ((((p0 + bytes + pad - 1) >> 32)) << 32) + pad;
          d.ids = (const uint8_t*)p0;
        }
        const cudaError_t e = launch_voxel_relayout(V.ids, (uint8_t*)d.ids, d.n[0], d.n[1], d.n[2], d.fast,
                                                    d.a1, d.a2, d.pitch, d.run_dir, n_materials, stream);
        if (e != cudaSuccess) { const mcx_status s_ = cuda_fail(e, "voxel relayout"); delete H; return s_; }
        H->launches += 2;
        d.cmap = nullptr;
        if (P.off_cmap[c]) {  // one byte per cell, inside one 4 GiB window like the volume
          const size_t bytes = voxel_bytes(d.n[d.fast], d.n[d.a1], d.n[d.a2]) / kVoxelCellBytes;
          const size_t pad = voxel_pad(d.n[d.fast], d.n[d.a1]) / kVoxelCellBytes + kAlign;
          uintptr_t p0 = (uintptr_t)dev_ptr(P.off_cmap[c]) + pad;
          if (((p0 - pad) >> 32) != ((p0 + bytes + pad - 1) >> 32)) p0 = ((((p0 + bytes + pad - 1) >> 32)) << 32) + pad;
          d.cmap = (const uint8_t*)p0;
        }
        {  // the cube radii beside the runs (and the compact cells)
          const cudaError_t e2 = launch_voxel_radius((uint8_t*)d.ids, (uint8_t*)dev_ptr(P.off_vox_scratch[c]), (uint8_t*)d.cmap, d.pitch,
                                                     d.n[d.a1] + 2, d.n[d.a2] + 2, stream);
          if (e2 != cudaSuccess) { const mcx_status s_ = cuda_fail(e2, "voxel radius transform"); delete H; return s_; }
          H->launches += 9;  // boundary, seven doubling passes, store
        }
        break;
      }
      case MCX_MIRROR_ELLIPTIC: {
        features |= F_OPTICS;
        const mcx_mirror_params& M = C.u.mirror;
        DMirror& d = D.u.mirror;
        if (!M.reflectivity) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: reflectivity is null", c);
        if (!(M.p > 0.0) || !(M.q > 0.0) || !(M.theta > 0.0)) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: p, q, theta must be positive", c);
        if (!(M.theta_max > M.theta_min) || !(M.e_max > M.e_min)) MCX_BAIL(MCX_ERR_RANGE, "component %d: empty reflectivity grid", c);
        // step 12: ellipse with foci at the source and image points, pole at distance p from the first focus
        d.a = 0.5 * (M.p + M.q);
        d.b = std::sqrt(M.p * M.q) * std::sin(M.theta);
        d.inv_a2 = 1.0 / (d.a * d.a);
        d.inv_b2 = 1.0 / (d.b * d.b);
        const double cfoc = std::sqrt(d.a * d.a - d.b * d.b);
        d.Z0 = (M.p - d.a) * d.a / cfoc;
        d.Y0 = -d.b * std::sqrt(1.0 - (d.Z0 * d.Z0) / (d.a * d.a));
        const double gZ = d.Z0 / (d.a * d.a), gY = d.Y0 / (d.b * d.b);
        const double gn = std::sqrt(gZ * gZ + gY * gY);
        d.nZ = -gZ / gn; d.nY = -gY / gn;
        d.tZ = d.nY; d.tY = -d.nZ;
        d.half_length = 0.5 * M.length; d.half_width = 0.5 * M.width;
        d.theta_min = M.theta_min; d.theta_max = M.theta_max; d.e_min = M.e_min; d.e_max = M.e_max;
        d.n_theta = (int)M.n_theta; d.n_e = (int)M.n_e;
        d.st = (double)(d.n_theta - 1) / (M.theta_max - M.theta_min);
        d.se = (double)(d.n_e - 1) / (M.e_max - M.e_min);
        std::memcpy(host_ptr(P.off_table[c]), M.reflectivity, (size_t)M.n_theta * M.n_e * sizeof(double));
        d.table = (const double*)dev_ptr(P.off_table[c]);
        break;
      }
      case MCX_CRYSTAL_BRAGG: {
        features |= F_OPTICS;
        const mcx_crystal_params& X = C.u.crystal;
        if (!(X.d_hkl > 0.0) || !(X.zeta > 0.0)) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: d_hkl and zeta must be positive", c);
        D.u.crystal.half_length = 0.5 * X.length; D.u.crystal.half_width = 0.5 * X.width;
        D.u.crystal.d_hkl = X.d_hkl; D.u.crystal.zeta = X.zeta; D.u.crystal.delta0 = X.delta0;
        if (!(X.g >= 0.0) || !std::isfinite(X.kappa)) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: g must be >= 0 and kappa finite", c);
        D.u.crystal.g = X.g; D.u.crystal.kappa = X.kappa;
        break;
      }
      case MCX_LENS_PARAB: {
        features |= F_LENS;
        const mcx_lens_params& L = C.u.lens;
        DLens& d = D.u.lens;
        if (!(L.radius > 0.0) || !(L.web >= 0.0) || !(L.pitch > 0.0) || !(L.aperture > 0.0))
          MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: radius, pitch, aperture must be positive, web non-negative", c);
        if (L.n_lenses < 1 || L.n_lenses > MCX_MAX_LENSES) MCX_BAIL(MCX_ERR_UNSUPPORTED, "component %d: 1..%d lenses", c, MCX_MAX_LENSES);
        if (L.material < 0 || L.material >= n_materials) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: lens material out of range", c);
        if (0.5 * L.web + L.aperture * L.aperture / (2.0 * L.radius) > 0.5 * L.pitch * (1.0 + 1e-12))
          MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: lenses overlap (web/2 + aperture^2 / (2 radius) > pitch/2)", c);
        if (!L.delta_energy_keV || !L.delta) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: null delta table", c);
        d.inv_R = 1.0 / L.radius; d.half_inv_R = 1.0 / (2.0 * L.radius);
        d.half_web = 0.5 * L.web; d.pitch = L.pitch; d.ra2 = L.aperture * L.aperture;
        d.n_lenses = (int)L.n_lenses; d.material = (int)L.material;
        const size_t n = (size_t)L.n_delta;
        double* E = (double*)host_ptr(P.off_table[c]);
        double* lnE = E + n;
        double* lnD = lnE + n;
        double* slope = lnD + n;
        for (size_t j = 0; j < n; ++j) {
          if (!(L.delta_energy_keV[j] > 0.0) || !(L.delta[j] > 0.0)) MCX_BAIL(MCX_ERR_RANGE, "component %d: non-positive delta table entry %zu", c, j);
          if (j > 0 && !(L.delta_energy_keV[j] > L.delta_energy_keV[j - 1])) MCX_BAIL(MCX_ERR_RANGE, "component %d: delta energies not increasing at %zu", c, j);
          E[j] = L.delta_energy_keV[j];
          lnE[j] = std::log(L.delta_energy_keV[j]);
          lnD[j] = std::log(L.delta[j]);
        }
        for (size_t j = 0; j + 1 < n; ++j) slope[j] = (lnD[j + 1] - lnD[j]) / (lnE[j + 1] - lnE[j]);
        slope[n - 1] = 0.0;
        d.delta.n = (int)n;
        d.delta.E = (const double*)dev_ptr(P.off_table[c]);
        d.delta.lnE = d.delta.E + n;
        d.delta.lnMu = d.delta.lnE + n;
        d.delta.slope = d.delta.lnMu + n;
        d.delta.inv_dlnE = (double)(n - 1) / (lnE[n - 1] - lnE[0]);
        break;
      }
      case MCX_DETECTOR: {
        const mcx_detector_params& T = C.u.detector;
        if (!(T.xmax > T.xmin) || !(T.ymax > T.ymin) || !(T.emax > T.emin)) MCX_BAIL(MCX_ERR_RANGE, "component %d: empty detector range", c);
        DDetector& d = D.u.detector;
        d.xmin = T.xmin; d.xmax = T.xmax; d.ymin = T.ymin; d.ymax = T.ymax; d.emin = T.emin; d.emax = T.emax;
        if (T.mode != MCX_DET_ENERGY && T.mode != MCX_DET_WAVELENGTH) MCX_BAIL(MCX_ERR_INVALID_ARG, "component %d: bad detector mode", c);
        d.mode = (int)T.mode;
        d.nx = (int)T.nx; d.ny = (int)T.ny; d.ne = (int)T.ne; d.index = n_dets;
        d.sx = (double)T.nx / (T.xmax - T.xmin); d.sy = (double)T.ny / (T.ymax - T.ymin); d.se = (double)T.ne / (T.emax - T.emin);
        d.n_bins = (uint64_t)T.nx * T.ny * T.ne;
        H->det_bins[n_dets] = d.n_bins;
        I.tallies[n_dets] = (TallyBin*)dev_ptr(P.off_tally[n_dets]);
        ++n_dets;
        break;
      }
    }
  }
#undef MCX_BAIL
  // voxel IDs must index the materials array; the kernel sizes its per-thread mu[] by n_materials
  I.n_dets = n_dets;
  I.features = features;
  I.counters = (unsigned long long*)dev_ptr(P.off_counters);
  H->n_dets = n_dets;
  H->features = features;
  H->source_pose = components[0].pose;
  for (int c = 0; c < n_components; ++c)
    if (components[c].kind == MCX_VOXELS) H->voxel_params[c] = components[c].u.voxels;
  H->cap_endpoints = cap_endpoints;
  for (int c = 0; c < n_components; ++c)
    if (components[c].kind == MCX_SOLIDS) H->n_solids_total += (int)components[c].u.solids.n_solids;
  for (int c = 1; c + 1 < n_components; ++c) {
      const int k = components[c].kind;
    if (k != MCX_SLIT_RECT && k != MCX_SLIT_CIRC && k != MCX_MIRROR_ELLIPTIC && k != MCX_CRYSTAL_BRAGG) break;
    H->gate_max = c;
  }
  {  // Detector-tile order needs a source whose slot-1 draw is a target point (step 3) and pays where neighbouring rays
     // share work: voxels, meshes, groups of several solids (measured: c1 1.4x, c3 5x, c4 3x; c0 and c2 nothing)
    bool shared_work = (features & (F_MESH | F_VOXELS)) != 0;
    for (int c = 0; c < n_components; ++c)
      if (components[c].kind == MCX_SOLIDS && components[c].u.solids.n_solids >= 2) shared_work = true;
    H->sort_pays = components[0].u.source.dir_mode == MCX_DIR_TARGET && shared_work;
  }

  cudaError_t e = cudaHostAlloc((void**)&H->host_flag, 64, cudaHostAllocMapped | cudaHostAllocPortable);
  if (e != cudaSuccess) { H->host_flag = nullptr; const mcx_status s_ = cuda_fail(e, "pinned status word"); delete H; return s_; }
  *H->host_flag = 0u;
  e = cudaMemcpyAsync(ws + P.off_inst, &H->host_image, sizeof(DInstrument), cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess && !blob_storage.empty())
    e = cudaMemcpyAsync(ws + P.blob_begin, blob_storage.data(), blob_storage.size(), cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(ws + P.zero_begin, 0, P.zero_end - P.zero_begin, stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(ws + P.off_gate, 0, sizeof(unsigned int), stream);
  if (e == cudaSuccess && P.stage_comp > 0) e = cudaMemsetAsync(ws + P.off_pool_count, 0, 4 * sizeof(unsigned int), stream);
  if (e != cudaSuccess) { const mcx_status s_ = cuda_fail(e, "upload of the instrument image"); delete H; return s_; }
  H->upload_bytes = sizeof(DInstrument) + blob_storage.size();
  *out = H;
  return MCX_OK;
}

}  // extern "C"

namespace {

// Rows a13: which order the rays of a call are traced in.  AUTO = detector-tile order where neighbouring rays share
// work (mcx_instrument_create decides, see sort_pays), index order otherwise (DESIGN.md 6 "What round 1 measured").
bool use_sorted(const mcx_instrument* H) {
  if (H->exec_mode == MCX_EXEC_SORTED) return true;
  if (H->exec_mode == MCX_EXEC_DIRECT) return false;
  return H->sort_pays;
}

constexpr size_t kMaxTimedChunks = 4096;
constexpr int kTallyCacheLog2 = 11;  // MCX_TALLY_BLOCK: 2048 slots of 32 bytes per block

// MCX_TALLY_BLOCK: the detectors whose bins all fit in half the cache go through it (smallest first, while they fit
// together); a detector with more bins would only evict those and takes the global path.
unsigned tally_cache_dets(const mcx_instrument* H) {
  unsigned mask = 0u;
  uint64_t used = 0;
  const uint64_t room = ((uint64_t)1 << kTallyCacheLog2) / 2;
  for (;;) {
    int best = -1;
    for (int d = 0; d < H->n_dets; ++d)
      if (!((mask >> d) & 1u) && (best < 0 || H->det_bins[d] < H->det_bins[best])) best = d;
    if (best < 0 || used + H->det_bins[best] > room) break;
    mask |= 1u << best;
    used += H->det_bins[best];
  }
  return mask;
}

// Step 14 update path (include/mcx.h, mcx_tally_mode).  AUTO (measured): per-ray reductions into the
// records, except where a detector has so few bins that every block can keep a private copy of all of them in shared
// memory (an L_monitor or E_monitor: all rays into ~100 bins; there same-address reductions serialise in
// L2 and the private copy is 11x faster); warp aggregation alone never paid.
int tally_mode_of(const mcx_instrument* H) {
  int mode = H->tally_mode;
  if (mode == MCX_TALLY_AUTO)
    mode = (!(H->features & (F_SOLIDS | F_VOXELS)) && tally_cache_dets(H) != 0u) ? MCX_TALLY_BLOCK : MCX_TALLY_GLOBAL;
  if (mode == MCX_TALLY_BLOCK && (H->features & (F_SOLIDS | F_VOXELS))) mode = MCX_TALLY_WARP;  // no room beside their scratch
  return mode;
}

bool is_staged(const mcx_instrument* H) { return H->stage_comp > 0 && H->staged_enabled && H->features == (F_VOXELS | F_SCATTER); }

// Traces rays [first, first + n) chunk by chunk; dump == nullptr tallies.
mcx_status run_trace(mcx_instrument* H, uint64_t first, uint64_t n, uint64_t seed, mcx_ray_fate* dump, cudaStream_t stream) {
  const bool sorted = use_sorted(H);
  const bool staged = is_staged(H);
  uint64_t cap = sorted ? H->chunk_rays : ((uint64_t)1 << 32);
  if (staged) {  // a chunk's survivors must fit the pool; chunks of equal length
    cap = std::min(cap, (uint64_t)1 << kPoolCapacityLog2);
    const uint64_t n_chunks = (n + cap - 1) / cap;
    if (n_chunks > 1) cap = std::min(cap, ((n + n_chunks - 1) / n_chunks + 31) / 32 * 32);
  }
  unsigned char* ws = H->workspace;
  for (uint64_t base = 0; base < n; base += cap) {
    const uint64_t m = std::min(cap, n - base);
    TraceArgs A;
    A.stage = 0;
    A.stage_comp = H->stage_comp;
    A.pool = (PoolRay*)(ws + H->off_pool);
    A.pool_count = (unsigned int*)(ws + H->off_pool_count);
    A.first = first + base;
    A.n = m;
    A.seed = seed;
    A.n_comps = H->n_comps;
    A.n_mats = H->n_mats;
    A.n_solids = H->n_solids_total;
    A.cap_endpoints = H->cap_endpoints;
    A.gate_max = H->gate_enabled ? H->gate_max : 0;
    A.host_flag = H->host_flag;
    A.epoch = H->epoch;
    A.tally_mode = tally_mode_of(H);
    A.tally_cache_log2 = A.tally_mode == MCX_TALLY_BLOCK ? kTallyCacheLog2 : 0;
    A.tally_cache_dets = tally_cache_dets(H);
    A.order = nullptr;
    A.dump = dump ? dump + base : nullptr;
    A.ticket = (unsigned int*)(ws + H->off_ticket);
    A.gate_known = (unsigned int*)(ws + H->off_gate);
    cudaEvent_t* tev = nullptr;  // mcx_instrument_set_timing: before the sort, after it, after trace_kernel
    if (H->timing && !dump && H->events_used + 3 <= kMaxTimedChunks * 3) {
      while (H->events.size() < H->events_used + 3) {
        cudaEvent_t ev;
        if (cudaEventCreate(&ev) != cudaSuccess) return cuda_fail(cudaGetLastError(), "event create");
        H->events.push_back(ev);
      }
      tev = H->events.data() + H->events_used;
      H->events_used += 3;
      H->timed_launches += staged ? 3 : 1;
      cudaEventRecord(tev[0], stream);
    }
    if (sorted && m >= kSortMinRays) {
      const int g = sort_bits(m, H->features, H->sort_grid_bits);
      unsigned int* cnt = (unsigned int*)(ws + H->off_sort_cnt);
      cudaError_t e = cudaMemsetAsync(cnt, 0, sizeof(unsigned int) << (2 * g), stream);
      if (e == cudaSuccess)
        e = launch_sort(A.first, (uint32_t)m, seed, g, cnt, (unsigned int*)(ws + H->off_sort_bsum), (uint32_t*)(ws + H->off_order), stream);
      if (e != cudaSuccess) return cuda_fail(e, "ray sort launch");
      H->launches += 3;
      A.order = (const uint32_t*)(ws + H->off_order);
    }
    if (tev) cudaEventRecord(tev[1], stream);
    if (staged) {
      // before the sample | the sample, every lane busy (scatter_walk_kernel) | after the sample
      cudaError_t e = cudaMemsetAsync(A.pool_count, 0, sizeof(unsigned int), stream);
      if (e != cudaSuccess) return cuda_fail(e, "pool reset");
      A.stage = 1;
      e = launch_trace((const DInstrument*)ws, H->features, H->n_mats, A, stream);
      if (e != cudaSuccess) return cuda_fail(e, "trace launch (stage 1)");
      WalkArgs Wk;
      Wk.first = A.first;
      Wk.seed = seed;
      Wk.comp = H->stage_comp;
      Wk.n_mats = H->n_mats;
      Wk.compact = H->host_image.comps[H->stage_comp].u.voxels.cmap != nullptr;
      Wk.batch_setup = H->walk_batch_setup;
      Wk.batch_settle = H->walk_batch_settle;
      Wk.pool = A.pool;
      Wk.pool_count = A.pool_count;
      e = launch_scatter_walk((const DInstrument*)ws, Wk, m, stream);
      if (e != cudaSuccess) return cuda_fail(e, "scatter walk launch");
      A.stage = 2;
      A.order = nullptr;
      e = launch_trace((const DInstrument*)ws, H->features, H->n_mats, A, stream);
      if (e != cudaSuccess) return cuda_fail(e, "trace launch (stage 2)");
      H->launches += 3;
    } else {
      const cudaError_t e = launch_trace((const DInstrument*)ws, H->features, H->n_mats, A, stream);
      if (e != cudaSuccess) return cuda_fail(e, "trace launch");
      H->launches++;
    }
    if (tev) cudaEventRecord(tev[2], stream);
  }
  return MCX_OK;
}

}  // namespace

extern "C" {

mcx_status mcx_instrument_set_exec(mcx_instrument* inst, int mode) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  if (mode != MCX_EXEC_AUTO && mode != MCX_EXEC_DIRECT && mode != MCX_EXEC_SORTED) return fail(MCX_ERR_INVALID_ARG, "bad exec mode %d", mode);
  inst->exec_mode = mode;
  return MCX_OK;
}

mcx_status mcx_trace_range(mcx_instrument* inst, uint64_t first_ray, uint64_t n_rays, uint64_t seed, void* cuda_stream) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  mcx_status st = check_sticky();
  if (st != MCX_OK) return st;
  st = run_trace(inst, first_ray, n_rays, seed, nullptr, (cudaStream_t)cuda_stream);
  return st != MCX_OK ? st : capacity_status(inst);
}

mcx_status mcx_trace(mcx_instrument* inst, uint64_t n_rays, uint64_t seed, void* cuda_stream) {
  return mcx_trace_range(inst, 0, n_rays, seed, cuda_stream);
}

mcx_status mcx_trace_dump(mcx_instrument* inst, uint64_t first_ray, uint64_t n_rays, uint64_t seed, mcx_ray_fate* out,
                          void* cuda_stream) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  if (!out && n_rays) return fail(MCX_ERR_INVALID_ARG, "out is null");
  mcx_status st = check_sticky();
  if (st != MCX_OK) return st;
  if (n_rays == 0) return MCX_OK;
  return run_trace(inst, first_ray, n_rays, seed, out, (cudaStream_t)cuda_stream);
}

mcx_status mcx_tally_read(mcx_instrument* inst, int detector, uint64_t* N, double* p, double* p2, size_t n_bins,
                          void* cuda_stream) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  if (detector < 0 || detector >= inst->n_dets) return fail(MCX_ERR_INVALID_ARG, "detector %d out of range (%d detectors)", detector, inst->n_dets);
  if (!N || !p || !p2) return fail(MCX_ERR_INVALID_ARG, "null output array");
  if ((uint64_t)n_bins != inst->det_bins[detector]) return fail(MCX_ERR_INVALID_ARG, "n_bins is %zu, detector has %llu", n_bins, (unsigned long long)inst->det_bins[detector]);
  mcx_status st = check_sticky();
  if (st != MCX_OK) return st;
  const cudaError_t e = launch_tally_read(inst->host_image.tallies[detector], n_bins, (unsigned long long*)N, p, p2, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "tally_read launch");
  inst->launches++;
  return capacity_status(inst);
}

mcx_status mcx_tally_read_host(mcx_instrument* inst, int detector, uint64_t* N, double* p, double* p2, size_t n_bins,
                               void* cuda_stream) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  if (detector < 0 || detector >= inst->n_dets) return fail(MCX_ERR_INVALID_ARG, "detector %d out of range (%d detectors)", detector, inst->n_dets);
  if (!N || !p || !p2) return fail(MCX_ERR_INVALID_ARG, "null output array");
  if ((uint64_t)n_bins != inst->det_bins[detector]) return fail(MCX_ERR_INVALID_ARG, "n_bins is %zu, detector has %llu", n_bins, (unsigned long long)inst->det_bins[detector]);
  unsigned long long* dN = (unsigned long long*)(inst->workspace + inst->off_staging);
  double* dP = (double*)(dN + n_bins);
  double* dP2 = dP + n_bins;
  const mcx_status st = mcx_tally_read(inst, detector, (uint64_t*)dN, dP, dP2, n_bins, cuda_stream);
  if (st != MCX_OK && st != MCX_ERR_CAPACITY) return st;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaMemcpyAsync(N, dN, n_bins * sizeof(uint64_t), cudaMemcpyDeviceToHost, stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(p, dP, n_bins * sizeof(double), cudaMemcpyDeviceToHost, stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(p2, dP2, n_bins * sizeof(double), cudaMemcpyDeviceToHost, stream);
  if (e != cudaSuccess) return cuda_fail(e, "tally copy to the host");
  return st;
}

mcx_status mcx_instrument_set_pose(mcx_instrument* inst, int component, const mcx_pose* pose, void* cuda_stream) {
  if (!inst || !pose) return fail(MCX_ERR_INVALID_ARG, "null argument");
  if (component < 1 || component >= inst->n_comps) return fail(MCX_ERR_INVALID_ARG, "component %d out of range (1..%d)", component, inst->n_comps - 1);
  if (!pose_ok(*pose)) return fail(MCX_ERR_INVALID_ARG, "pose is not finite");
  DComponent& D = inst->host_image.comps[component];
  if (D.kind == MCX_SOLIDS) return fail(MCX_ERR_UNSUPPORTED, "component %d is a solids group: its solids carry their own poses", component);
  if (D.kind == MCX_VOXELS) {  // the traversal layout was chosen at create from the old pose
    mcx_component src, vox;
    std::memset(&src, 0, sizeof(src));
    std::memset(&vox, 0, sizeof(vox));
    src.pose = inst->source_pose;
    vox.pose = *pose;
    vox.u.voxels = inst->voxel_params[component];
    int fast, a1, a2, run_dir;
    voxel_axes(src, vox, &fast, &a1, &a2, &run_dir);
    if (fast != D.u.voxels.fast || run_dir != D.u.voxels.run_dir)
      return fail(MCX_ERR_UNSUPPORTED, "component %d: the new pose would change the voxel layout (fast axis %d -> %d); create a new instrument",
                  component, D.u.voxels.fast, fast);
  }
  mcx_status st = check_sticky();
  if (st != MCX_OK) return st;
  copy_pose(&D.pose, *pose);
  // host_image outlives the copy: pageable memory is staged before cudaMemcpyAsync returns
  const size_t off = (size_t)((const unsigned char*)&D.pose - (const unsigned char*)&inst->host_image);
  const cudaError_t e = cudaMemcpyAsync(inst->workspace + off, &D.pose, sizeof(DPose), cudaMemcpyHostToDevice, (cudaStream_t)cuda_stream);  // (rotation, origin and the identity flag)
  if (e != cudaSuccess) return cuda_fail(e, "pose upload");
  return MCX_OK;
}

mcx_status mcx_cnr(const uint64_t* N, const double* p, const double* p2, int64_t nx, int64_t ny, int64_t ne, const int32_t* region_mat,
                   const int32_t* region_ref, double emin, double emax, double e_fit_min, double* cnr_out, double* fit_out,
                   void* cuda_stream) {
  if (!N || !p || !p2 || !region_mat || !region_ref || !cnr_out || !fit_out) return fail(MCX_ERR_INVALID_ARG, "null argument");
  if (nx < 1 || ny < 1 || ne < 1 || nx > (1 << 20) || ny > (1 << 20) || ne > (1 << 20)) return fail(MCX_ERR_INVALID_ARG, "bad detector shape");
  if (!(emax > emin)) return fail(MCX_ERR_RANGE, "empty energy range");
  for (const int32_t* r : {region_mat, region_ref})
    if (r[0] < 0 || r[1] > nx || r[0] >= r[1] || r[2] < 0 || r[3] > ny || r[2] >= r[3])
      return fail(MCX_ERR_INVALID_ARG, "region (%d, %d, %d, %d) is empty or outside the %lld x %lld detector", r[0], r[1], r[2], r[3], (long long)nx, (long long)ny);
  mcx_status st = check_sticky();
  if (st != MCX_OK) return st;
  const cudaError_t e = launch_cnr((const unsigned long long*)N, p, p2, (int)nx, (int)ny, (int)ne, region_mat, region_ref, emin, emax,
                                   e_fit_min, cnr_out, fit_out, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "cnr launch");
  return MCX_OK;
}

mcx_status mcx_cnr_static(mcx_instrument* inst, int detector, const int32_t* region_mat, const int32_t* region_ref, double e_fit_min,
                          double* cnr_out, double* fit_out, void* cuda_stream) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  if (detector < 0 || detector >= inst->n_dets) return fail(MCX_ERR_INVALID_ARG, "detector %d out of range (%d detectors)", detector, inst->n_dets);
  if (!region_mat || !region_ref || !cnr_out || !fit_out) return fail(MCX_ERR_INVALID_ARG, "null argument");
  const DDetector* D = nullptr;
  for (int c = 0; c < inst->n_comps; ++c)
    if (inst->host_image.comps[c].kind == MCX_DETECTOR && inst->host_image.comps[c].u.detector.index == detector) D = &inst->host_image.comps[c].u.detector;
  if (!D) return fail(MCX_ERR_INVALID_ARG, "detector %d not found", detector);
  const uint64_t n_bins = inst->det_bins[detector];
  if (n_bins > (uint64_t)MCX_CNR_STATIC_MAX_BINS || D->ne > MCX_CNR_STATIC_MAX_NE)
    return fail(MCX_ERR_UNSUPPORTED, "detector %d has %llu bins, %d energy bins: above the %d bins / %d energy bins the static scratch of "
                "mcx_cnr_static holds (use mcx_tally_read + mcx_cnr)", detector, (unsigned long long)n_bins, D->ne, (int)MCX_CNR_STATIC_MAX_BINS,
                (int)MCX_CNR_STATIC_MAX_NE);
  for (const int32_t* r : {region_mat, region_ref})
    if (r[0] < 0 || r[1] > D->nx || r[0] >= r[1] || r[2] < 0 || r[3] > D->ny || r[2] >= r[3])
      return fail(MCX_ERR_INVALID_ARG, "region (%d, %d, %d, %d) is empty or outside the %d x %d detector", r[0], r[1], r[2], r[3], D->nx, D->ny);
  mcx_status st = check_sticky();
  if (st != MCX_OK) return st;
  const cudaError_t e = launch_cnr_static(inst->host_image.tallies[detector], n_bins, D->nx, D->ny, D->ne, region_mat, region_ref, D->emin,
                                          D->emax, e_fit_min, cnr_out, fit_out, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "static cnr launch");
  inst->launches += 3;
  return capacity_status(inst);
}

uint64_t mcx_upload_bytes(const mcx_instrument* inst) { return inst ? (uint64_t)inst->upload_bytes : 0; }

mcx_status mcx_tally_reset(mcx_instrument* inst, void* cuda_stream) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  mcx_status st = check_sticky();
  if (st != MCX_OK) return st;
  const cudaError_t e = cudaMemsetAsync(inst->workspace + inst->zero_begin, 0, inst->zero_end - inst->zero_begin, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "tally reset");
  inst->epoch++;  // an overflow reported by a trace enqueued before this reset no longer counts
  return MCX_OK;
}

mcx_status mcx_counters_read(mcx_instrument* inst, uint64_t* counters, int n, void* cuda_stream) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  if (!counters || n != MCX_N_COUNTERS(inst->n_comps)) return fail(MCX_ERR_INVALID_ARG, "counters must hold %d values", MCX_N_COUNTERS(inst->n_comps));
  mcx_status st = check_sticky();
  if (st != MCX_OK) return st;
  const cudaError_t e = cudaMemcpyAsync(counters, inst->host_image.counters, (size_t)n * sizeof(uint64_t), cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "counters copy");
  return capacity_status(inst);
}

mcx_status mcx_trace_status(mcx_instrument* inst, void* cuda_stream) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  cudaError_t e = cudaStreamSynchronize((cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "stream synchronize");
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e, "asynchronous CUDA error");
  if (!capacity_overflowed(inst)) return MCX_OK;
  unsigned long long dropped = 0;
  e = cudaMemcpy(&dropped, inst->host_image.counters + inst->n_comps + CNT_OVERFLOW, sizeof(dropped), cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) return cuda_fail(e, "overflow counter copy");
  return fail(MCX_ERR_CAPACITY, "%llu rays overflowed the per-ray end-point capacity (%d) of a solids group and were dropped as degenerate",
              dropped, inst->cap_endpoints);
}

mcx_status mcx_instrument_set_tuning(mcx_instrument* inst, const mcx_tuning* t) {
  if (!inst || !t) return fail(MCX_ERR_INVALID_ARG, "null argument");
  if (t->chunk_log2 != 0 && (t->chunk_log2 < kChunkLog2Min || t->chunk_log2 > kChunkLog2Max))
    return fail(MCX_ERR_INVALID_ARG, "chunk_log2 %d outside %d..%d", t->chunk_log2, kChunkLog2Min, kChunkLog2Max);
  if (t->sort_grid_bits < 0 || t->sort_grid_bits > MCX_SORT_MAX_G) return fail(MCX_ERR_INVALID_ARG, "sort_grid_bits %d outside 1..%d", t->sort_grid_bits, MCX_SORT_MAX_G);
  if (t->absorber_gate < 0 || t->absorber_gate > 2) return fail(MCX_ERR_INVALID_ARG, "absorber_gate must be 0, 1 or 2");
  if (t->tally_mode < 0 || t->tally_mode > MCX_TALLY_BLOCK) return fail(MCX_ERR_INVALID_ARG, "tally_mode must be an mcx_tally_mode");
  if (t->staged_walk < 0 || t->staged_walk > 2) return fail(MCX_ERR_INVALID_ARG, "staged_walk must be 0, 1 or 2");
  if (t->walk_batch_setup < 0 || t->walk_batch_setup > 32 || t->walk_batch_settle < 0 || t->walk_batch_settle > 32)
    return fail(MCX_ERR_INVALID_ARG, "walk_batch_setup and walk_batch_settle must be 0 (keep) or 1..32");
  if (t->chunk_log2) inst->chunk_rays = (uint64_t)1 << t->chunk_log2;
  if (t->sort_grid_bits) inst->sort_grid_bits = t->sort_grid_bits;
  if (t->absorber_gate) inst->gate_enabled = t->absorber_gate == 1;
  if (t->tally_mode) inst->tally_mode = t->tally_mode;
  if (t->staged_walk) inst->staged_enabled = t->staged_walk == 1;
  if (t->walk_batch_setup) inst->walk_batch_setup = t->walk_batch_setup;
  if (t->walk_batch_settle) inst->walk_batch_settle = t->walk_batch_settle;
  return MCX_OK;
}

mcx_status mcx_instrument_get_tuning(const mcx_instrument* inst, mcx_tuning* t) {
  if (!inst || !t) return fail(MCX_ERR_INVALID_ARG, "null argument");
  int log2 = 0;
  while (((uint64_t)1 << log2) < inst->chunk_rays) ++log2;
  t->chunk_log2 = log2;
  t->sort_grid_bits = inst->sort_grid_bits;
  t->absorber_gate = inst->gate_enabled ? 1 : 2;
  t->tally_mode = tally_mode_of(inst);
  t->staged_walk = is_staged(inst) ? 1 : 2;
  t->walk_batch_setup = inst->walk_batch_setup;
  t->walk_batch_settle = inst->walk_batch_settle;
  return MCX_OK;
}

uint64_t mcx_launch_count(const mcx_instrument* inst) { return inst ? inst->launches : 0; }

mcx_status mcx_instrument_set_timing(mcx_instrument* inst, int on) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  inst->timing = on != 0;
  return MCX_OK;
}

mcx_status mcx_timing_read(mcx_instrument* inst, double* sort_ms, double* trace_ms, int64_t* n_trace_launches) {
  if (!inst) return fail(MCX_ERR_INVALID_ARG, "inst is null");
  double s_ms = 0.0, t_ms = 0.0;
  const size_t n = inst->events_used / 3;
  if (n > 0) {
    cudaError_t e = cudaEventSynchronize(inst->events[3 * n - 1]);
    if (e != cudaSuccess) return cuda_fail(e, "event synchronize");
    for (size_t k = 0; k < n; ++k) {
      float a = 0.0f, b = 0.0f;
      e = cudaEventElapsedTime(&a, inst->events[3 * k], inst->events[3 * k + 1]);
      if (e == cudaSuccess) e = cudaEventElapsedTime(&b, inst->events[3 * k + 1], inst->events[3 * k + 2]);
      if (e != cudaSuccess) return cuda_fail(e, "event elapsed time");
      s_ms += a;
      t_ms += b;
    }
  }
  inst->events_used = 0;
  if (sort_ms) *sort_ms = s_ms;
  if (trace_ms) *trace_ms = t_ms;
  if (n_trace_launches) *n_trace_launches = inst->timed_launches;
  inst->timed_launches = 0;
  return MCX_OK;
}

mcx_status mcx_probe_dfma(double* sink, int n_blocks, int64_t n_iters, void* cuda_stream) {
  if (!sink || n_blocks < 1 || n_iters < 0) return fail(MCX_ERR_INVALID_ARG, "bad probe arguments");
  const cudaError_t e = launch_probe_dfma(sink, n_blocks, (long long)n_iters, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "probe launch");
  return MCX_OK;
}

mcx_status mcx_probe_tally(void* table, uint64_t n_records, int n_blocks, int64_t n_iters, void* cuda_stream) {
  if (!table || n_records == 0 || (n_records & (n_records - 1)) != 0 || n_blocks < 1 || n_iters < 0)
    return fail(MCX_ERR_INVALID_ARG, "bad probe arguments (n_records must be a power of two)");
  const cudaError_t e = launch_probe_tally(table, n_records, n_blocks, (long long)n_iters, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "probe launch");
  return MCX_OK;
}

mcx_status mcx_probe_l2(const void* table, uint64_t n_bytes, uint32_t* sink, int n_blocks, int64_t n_iters, void* cuda_stream) {
  if (!table || !sink || n_bytes < 4096 || (n_bytes & (n_bytes - 1)) != 0 || n_blocks < 1 || n_iters < 0)
    return fail(MCX_ERR_INVALID_ARG, "bad probe arguments (n_bytes must be a power of two >= 4096)");
  const cudaError_t e = launch_probe_l2(table, n_bytes, sink, n_blocks, (long long)n_iters, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "probe launch");
  return MCX_OK;
}

mcx_status mcx_probe_latency(void* table, uint64_t n_bytes, uint32_t* sink, int n_blocks, int n_threads, int64_t n_iters,
                             void* cuda_stream) {
  if (!table || !sink || n_bytes < 4096 || (n_bytes & (n_bytes - 1)) != 0 || n_blocks < 1 || n_threads < 1 || n_threads > 256 || n_iters < 0)
    return fail(MCX_ERR_INVALID_ARG, "bad probe arguments (n_bytes must be a power of two >= 4096, n_threads <= 256)");
  const cudaError_t e = launch_probe_latency(table, n_bytes, sink, n_blocks, n_threads, (long long)n_iters, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return cuda_fail(e, "probe launch");
  return MCX_OK;
}

void mcx_instrument_destroy(mcx_instrument* inst) { delete inst; }

}  // extern "C"
