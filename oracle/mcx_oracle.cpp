// oracle/mcx_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded fp64 CPU tracer of the hot path named by BASELINE.json:north_star
// (arxiv 2410.08747, "Accelerated ray-tracing simulations using McXtrace"): rays sampled at a source and
// passed sequentially through a component chain ("rays are generated at the source component
// and sequentially propagated through the list of X-ray components"), then tallied into monitor arrays
// (PAPER.md:85, 106).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this file's library.  It shares NO code, header, table or helper with the CUDA path under
// paper_2410_08747_b200/csrc/ and neither includes the other.
//
// The paper is a performance paper and prints none of the physics formulas; every formula here follows the
// reading recorded in SURVEY.md section 8(c) (steps 1..15, readings R1..R27) and DESIGN.md "Readings".
// Each function cites the step it follows.  Nothing is blocked, fused or reordered beyond that text.
//
// Build:  g++ -O2 -ffp-contract=off -std=c++17 -shared -fPIC  (no FMA contraction, glibc libm; reading R20)
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known answers, u01 end points, slab exp(-mu L),
// slit acceptance 0.16, weight conservation, ray accounting, power-law mu(E), sphere/box/cylinder chords,
// cube-mesh == box (random rays, and rays exactly through face diagonals, edges and vertices: duplicate-hit
// collapse; rays grazing an edge or vertex: enter-before-exit tie order; open and inward-wound meshes: the
// DEGENERATE return), icosphere vs analytic sphere (levels 5 and 6), grid accelerator == brute force, no degenerate
// ray in 1e6 through closed meshes, voxel closed forms and the paper's fixed-step marching as a
// convergence cross-check, ellipse focal property, bilinear exactness, Darwin closed forms, detector binning, the
// fate rule of chains with several monitors against plane geometry written out in numpy; compound refractive lens:
// thin-lens deflection 2 N delta x / R, thick-stack focal length R / (2 N delta) + L / 6, plane-parallel slab
// displacement by Snell's law, on-axis transmission exp(-mu N d), parabolic thickness profile, reversibility;
// Darwin-Prins: g = kappa = 0 limit, closed form at eta = 0, numpy complex arithmetic; wavelength bins: lambda = hc / E;
// scattering (step 17): K = 0 and mu_s = 0 reduce to steps 10 / 11 bit for bit, Thomson inverse CDF and moments, unit
// orthogonal frames, exp(-mu_s L) unscattered fraction, event depth = -ln(u) / mu_s replayed from the draws, weight 1 in a
// purely scattering medium, a fine-step marching of the same draws (the paper's own stepping) on a small volume.
// Whole-config tallies of c1..c4 have no closed form: "parity unpinned" beyond those part-wise pins
// (SURVEY.md 8(c) last row).
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

const double kInf = std::numeric_limits<double>::infinity();
const double kPi = 3.14159265358979323846;
const double kHC_keV_A = 12.398419843;  // h*c in keV*Angstrom (SURVEY 8(c) conventions)

// ---------------------------------------------------------------------------------------------------
// Interface structs (the oracle's own; the CUDA library has a different, unrelated ABI in include/mcx.h)
// ---------------------------------------------------------------------------------------------------
enum Kind { K_SOURCE = 0, K_SLIT_RECT = 1, K_SLIT_CIRC = 2, K_SOLIDS = 3, K_VOXELS = 4, K_MIRROR = 5,
            K_CRYSTAL = 6, K_DETECTOR = 7, K_LENS = 8 };
enum DetMode { DET_ENERGY = 0, DET_WAVELENGTH = 1 };  // what the third detector axis bins (step 14 / 14b)
enum PosMode { POS_POINT = 0, POS_DISK = 1, POS_GAUSS = 2 };
enum DirMode { DIR_TARGET = 0, DIR_GAUSS = 1 };
enum EMode { E_MONO = 0, E_UNIFORM = 1, E_SPECTRUM = 2 };
enum Shape { S_BOX = 0, S_CYL = 1, S_SPHERE = 2, S_MESH = 3 };
enum Fate { F_DETECTED = -1, F_MISSED = -2, F_DEGENERATE = -3 };  // >= 0: absorbed at that component

}  // namespace

extern "C" {

struct OrcMaterial {  // n == 0: vacuum, mu == 0 (step 7)
  int64_t n;
  const double* E;     // keV, strictly increasing
  const double* mu;    // 1/m, total attenuation
  const double* mu_s;  // 1/m, the part of mu that scatters (step 17); null = none
};

struct OrcSolid {
  int32_t shape, material, priority, pad;
  double R[9], T[3];  // pose: r_local = R (r_lab - T)
  double hx, hy, hz;  // box half extents
  double radius;      // cylinder / sphere
  double half_height; // cylinder, axis = local y (R13)
  int64_t n_verts, n_tris;
  const double* verts;  // [n_verts][3], solid-local frame
  const int32_t* tris;  // [n_tris][3], outward-wound
};

struct OrcComponent {
  int32_t kind, pos_mode, dir_mode, e_mode;
  double R[9], T[3];
  // source (step 3)
  double radius, sigma_x, sigma_y;
  double target_w, target_h, target_dist, div_x, div_y;
  double E0, dE_rel, spec_Emin, spec_Emax;
  int64_t spec_n;
  const double* spectrum;
  // slit (step 6)
  double xw, yh, slit_radius;
  // solids (steps 8-10)
  int64_t n_solids;
  const OrcSolid* solids;
  // voxels (step 11)
  double vox_h;
  int64_t vnx, vny, vnz;
  const uint8_t* vox_ids;  // [iz][iy][ix], x fastest
  // mirror (step 12)
  double mir_p, mir_q, mir_theta, mir_length, mir_width;
  double tab_theta_min, tab_theta_max, tab_E_min, tab_E_max;
  int64_t tab_n_theta, tab_n_E;
  const double* tab_R;  // [n_theta][n_E]
  // crystal (step 13)
  double xtal_length, xtal_width, xtal_d, xtal_zeta, xtal_delta0;
  // detector (step 14)
  double det_xmin, det_xmax, det_ymin, det_ymax, det_Emin, det_Emax;
  int64_t det_nx, det_ny, det_nE;
  // ---- SURVEY.md 8(f) rows ----
  int64_t det_mode;       // DetMode (step 14b): DET_WAVELENGTH bins lambda = hc / E [Angstrom] over [det_Emin, det_Emax]
  // Darwin-Prins crystal (step 13b): absorption ratios g = Im(chi_0) / |chi_h|', kappa = Im(chi_h) / Re(chi_h); 0, 0 = Darwin
  double xtal_g, xtal_kappa;
  // compound refractive lens (step 16)
  double lens_R, lens_d, lens_pitch, lens_ra;  // apex radius of curvature, web thickness, lens-to-lens pitch, aperture radius
  int64_t lens_N, lens_material;               // number of double-sided lenses; material index of mu(E)
  int64_t lens_nd;                             // points of the delta(E) table (refractive index n = 1 - delta)
  const double* lens_dE;                       // keV, strictly increasing
  const double* lens_delta;                    // > 0, log-log interpolated like mu(E) (step 7)
  // scattering in samples (step 17): at most this many direction changes per ray in this component; 0 = attenuation only
  int64_t scatter_order;
};

struct OrcRayFate {
  int32_t fate;  // Fate, or index of the absorbing component
  int32_t pad;
  int64_t bin;   // bin in the last detector hit, -1 if none
  double p;      // final weight
};

}  // extern "C"

namespace {

// ---------------------------------------------------------------------------------------------------
// Step 1: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  PAPER.md:91 only says the RNG was
// "reimplemented for the GPU"; north_star fixes Philox4x32-10 keyed by (seed, ray index).
// ---------------------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    const uint64_t prod0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t prod1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
    const uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Step 2 (reading R5, corrected in DESIGN.md): 52 random bits, centred in their cell, so the value is exact
// in fp64 and lies in [2^-53, 1 - 2^-53]: never 0 or 1.
double u01(uint32_t wa, uint32_t wb) {
  const uint64_t x = ((uint64_t)wa << 32) | wb;
  return ((double)(x >> 12) + 0.5) * (1.0 / 4503599627370496.0);  // 2^-52
}

// Slot-addressed draws (step 1): counter = (i lo, i hi, slot, component index), key = (seed lo, seed hi).
void draw2(uint64_t seed, uint64_t i, uint32_t slot, uint32_t comp, double* ua, double* ub) {
  const uint32_t ctr[4] = {(uint32_t)i, (uint32_t)(i >> 32), slot, comp};
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  *ua = u01(w[0], w[1]);
  *ub = u01(w[2], w[3]);
}

// Step 2: Box-Muller, both values used.
void gauss_pair(double ua, double ub, double* g0, double* g1) {
  const double rad = std::sqrt(-2.0 * std::log(ua));
  const double ang = 2.0 * kPi * ub;
  *g0 = rad * std::cos(ang);
  *g1 = rad * std::sin(ang);
}

// ---------------------------------------------------------------------------------------------------
// small vector helpers
// ---------------------------------------------------------------------------------------------------
struct V3 { double x, y, z; };
V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
// Step 4: r' = R (r - T), d' = R d;   inverse: r = R^T r' + T.
V3 rot(const double R[9], V3 v) {
  return {R[0] * v.x + R[1] * v.y + R[2] * v.z, R[3] * v.x + R[4] * v.y + R[5] * v.z,
          R[6] * v.x + R[7] * v.y + R[8] * v.z};
}
V3 rotT(const double R[9], V3 v) {
  return {R[0] * v.x + R[3] * v.y + R[6] * v.z, R[1] * v.x + R[4] * v.y + R[7] * v.z,
          R[2] * v.x + R[5] * v.y + R[8] * v.z};
}
V3 to_local_pos(const double R[9], const double T[3], V3 r) { return rot(R, r - V3{T[0], T[1], T[2]}); }
V3 to_lab_pos(const double R[9], const double T[3], V3 r) { return rotT(R, r) + V3{T[0], T[1], T[2]}; }

// ---------------------------------------------------------------------------------------------------
// Step 7: mu(E) by log-log interpolation; end segments extrapolate (R11).
// ---------------------------------------------------------------------------------------------------
struct MuTable {
  std::vector<double> E, lnE, lnMu;
  std::vector<double> lnMuS;  // ln of the scattering part (step 17); empty = the material does not scatter
};

double mu_of_E(const MuTable& m, double E) {
  const int64_t n = (int64_t)m.E.size();
  if (n == 0) return 0.0;  // vacuum
  // j = index with E_j <= E < E_{j+1}, clamped to [0, n-2]
  int64_t j = (int64_t)(std::upper_bound(m.E.begin(), m.E.end(), E) - m.E.begin()) - 1;
  if (j < 0) j = 0;
  if (j > n - 2) j = n - 2;
  const double lnE = std::log(E);
  const double slope = (m.lnMu[j + 1] - m.lnMu[j]) / (m.lnE[j + 1] - m.lnE[j]);
  return std::exp(m.lnMu[j] + (lnE - m.lnE[j]) * slope);
}

// Step 17: the scattering part of mu(E), the same log-log interpolation on the same grid; 0 without a table.
double mu_s_of_E(const MuTable& m, double E) {
  if (m.lnMuS.empty()) return 0.0;
  MuTable t;
  t.E = m.E; t.lnE = m.lnE; t.lnMu = m.lnMuS;
  return mu_of_E(t, E);
}

// ---------------------------------------------------------------------------------------------------
// Step 8: inside-intervals of the ray parameter for the convex primitives.  Ray (o, d) is in the solid's
// own frame; d is unit so t is metres.  Returns false if there is no interval of positive length.
// ---------------------------------------------------------------------------------------------------
bool slab_axis(double o, double d, double lo, double hi, double* tmin, double* tmax) {
  if (d == 0.0) return (o > lo && o < hi);
  double t1 = (lo - o) / d, t2 = (hi - o) / d;
  if (t1 > t2) std::swap(t1, t2);
  if (t1 > *tmin) *tmin = t1;
  if (t2 < *tmax) *tmax = t2;
  return true;
}

bool box_interval(V3 o, V3 d, double hx, double hy, double hz, double* tin, double* tout) {
  double tmin = -kInf, tmax = kInf;
  if (!slab_axis(o.x, d.x, -hx, hx, &tmin, &tmax)) return false;
  if (!slab_axis(o.y, d.y, -hy, hy, &tmin, &tmax)) return false;
  if (!slab_axis(o.z, d.z, -hz, hz, &tmin, &tmax)) return false;
  if (!(tmin < tmax)) return false;
  *tin = tmin; *tout = tmax;
  return true;
}

bool sphere_interval(V3 o, V3 d, double radius, double* tin, double* tout) {
  const double b = dot(o, d);
  const double c = dot(o, o) - radius * radius;
  const double disc = b * b - c;
  if (!(disc > 0.0)) return false;
  const double s = std::sqrt(disc);
  *tin = -b - s; *tout = -b + s;
  return true;
}

// finite cylinder, axis = local y (R13): infinite-cylinder quadratic in (x,z) intersected with the y-slab
bool cylinder_interval(V3 o, V3 d, double radius, double half_height, double* tin, double* tout) {
  double tmin = -kInf, tmax = kInf;
  const double a = d.x * d.x + d.z * d.z;
  const double c = o.x * o.x + o.z * o.z - radius * radius;
  if (a == 0.0) {
    if (!(c < 0.0)) return false;
  } else {
    const double b = o.x * d.x + o.z * d.z;
    const double disc = b * b - a * c;
    if (!(disc > 0.0)) return false;
    const double s = std::sqrt(disc);
    tmin = (-b - s) / a; tmax = (-b + s) / a;
  }
  if (!slab_axis(o.y, d.y, -half_height, half_height, &tmin, &tmax)) return false;
  if (!(tmin < tmax)) return false;
  *tin = tmin; *tout = tmax;
  return true;
}

// ---------------------------------------------------------------------------------------------------
// Step 9: watertight ray/triangle test (Woop, Benthin, Wald 2013) in fp64.  Edge functions are plain
// products and differences (no FMA), so a shared edge gives exactly negated values in its two triangles.
// Returns 0 = miss, +1 = entering (d.n_geo < 0), -1 = exiting.
// ---------------------------------------------------------------------------------------------------
int ray_triangle(const double o[3], const double d[3], const double* v0, const double* v1, const double* v2,
                 double* t_out) {
  int kz = 0;
  if (std::fabs(d[1]) > std::fabs(d[kz])) kz = 1;
  if (std::fabs(d[2]) > std::fabs(d[kz])) kz = 2;
  int kx = (kz + 1) % 3, ky = (kx + 1) % 3;
  if (d[kz] < 0.0) std::swap(kx, ky);
  const double Sx = d[kx] / d[kz], Sy = d[ky] / d[kz], Sz = 1.0 / d[kz];
  const double A[3] = {v0[0] - o[0], v0[1] - o[1], v0[2] - o[2]};
  const double B[3] = {v1[0] - o[0], v1[1] - o[1], v1[2] - o[2]};
  const double C[3] = {v2[0] - o[0], v2[1] - o[1], v2[2] - o[2]};
  const double Ax = A[kx] - Sx * A[kz], Ay = A[ky] - Sy * A[kz];
  const double Bx = B[kx] - Sx * B[kz], By = B[ky] - Sy * B[kz];
  const double Cx = C[kx] - Sx * C[kz], Cy = C[ky] - Sy * C[kz];
  const double U = Cx * By - Cy * Bx;
  const double V = Ax * Cy - Ay * Cx;
  const double W = Bx * Ay - By * Ax;
  if ((U < 0.0 || V < 0.0 || W < 0.0) && (U > 0.0 || V > 0.0 || W > 0.0)) return 0;
  const double det = U + V + W;
  if (det == 0.0) return 0;
  const double Az = Sz * A[kz], Bz = Sz * B[kz], Cz = Sz * C[kz];
  *t_out = (U * Az + V * Bz + W * Cz) / det;
  return det > 0.0 ? +1 : -1;
}

struct Hit { double t; int orient; };

// The oracle's own accelerator (R26): a uniform grid over the mesh AABB holding, per cell, the triangles
// whose AABB overlaps the cell.  A ray visits the cells its line crosses; every candidate is tested with the
// same ray_triangle as brute force, and each triangle at most once, so the hit set is identical to brute
// force by construction (pinned in tests/test_oracle_solids.py).
struct MeshGrid {
  double lo[3], cell[3];
  int n[3];
  std::vector<int32_t> start, items;  // CSR
};

struct MeshPrep {
  const OrcSolid* s;
  bool has_grid = false;
  MeshGrid g;
  mutable std::vector<uint32_t> stamp;  // per triangle: id of the last ray that tested it
  mutable uint32_t stamp_id = 0;
};

int grid_resolution(int64_t n_tris) {
  const int res = (int)std::ceil(std::cbrt((double)n_tris));
  return std::max(1, std::min(res, 128));
}

void build_mesh_grid(MeshPrep* mp, int res) {
  const OrcSolid& s = *mp->s;
  MeshGrid& g = mp->g;
  double lo[3] = {kInf, kInf, kInf}, hi[3] = {-kInf, -kInf, -kInf};
  for (int64_t v = 0; v < s.n_verts; ++v)
    for (int a = 0; a < 3; ++a) {
      lo[a] = std::min(lo[a], s.verts[3 * v + a]);
      hi[a] = std::max(hi[a], s.verts[3 * v + a]);
    }
  for (int a = 0; a < 3; ++a) {
    const double pad = 1e-9 * (hi[a] - lo[a]) + 1e-12;
    g.lo[a] = lo[a] - pad;
    g.n[a] = res;
    g.cell[a] = ((hi[a] + pad) - g.lo[a]) / res;
  }
  const int64_t ncell = (int64_t)res * res * res;
  std::vector<int32_t> count(ncell + 1, 0);
  auto cell_range = [&](int64_t tri, int a, int* c0, int* c1) {
    double tlo = kInf, thi = -kInf;
    for (int k = 0; k < 3; ++k) {
      const double x = s.verts[3 * (int64_t)s.tris[3 * tri + k] + a];
      tlo = std::min(tlo, x); thi = std::max(thi, x);
    }
    // the triangle's box is grown by `slack` (far above any rounding in the cell walk below, far below a
    // cell): candidates are a superset of the cells the triangle touches, the exact test decides
    const double slack = 1e-6 * g.cell[a];
    *c0 = std::min(res - 1, std::max(0, (int)std::floor((tlo - slack - g.lo[a]) / g.cell[a])));
    *c1 = std::max(0, std::min(res - 1, (int)std::floor((thi + slack - g.lo[a]) / g.cell[a])));
  };
  for (int pass = 0; pass < 2; ++pass) {
    for (int64_t tri = 0; tri < s.n_tris; ++tri) {
      int x0, x1, y0, y1, z0, z1;
      cell_range(tri, 0, &x0, &x1); cell_range(tri, 1, &y0, &y1); cell_range(tri, 2, &z0, &z1);
      for (int z = z0; z <= z1; ++z)
        for (int y = y0; y <= y1; ++y)
          for (int x = x0; x <= x1; ++x) {
            const int64_t c = ((int64_t)z * res + y) * res + x;
            if (pass == 0) count[c + 1]++;
            else g.items[g.start[c] + count[c]++] = (int32_t)tri;
          }
    }
    if (pass == 0) {
      g.start.assign(ncell + 1, 0);
      for (int64_t c = 0; c < ncell; ++c) g.start[c + 1] = g.start[c] + count[c + 1];
      g.items.resize(g.start[ncell]);
      std::fill(count.begin(), count.end(), 0);
    }
  }
  mp->stamp.assign(s.n_tris, 0u);
  mp->stamp_id = 0;
  mp->has_grid = true;
}

// all hits of the full line (t in R) with one mesh, in the mesh's local frame
void mesh_hits(const MeshPrep& mp, V3 o, V3 d, bool use_grid, std::vector<Hit>* hits, uint64_t* n_tests) {
  const OrcSolid& s = *mp.s;
  const double oo[3] = {o.x, o.y, o.z}, dd[3] = {d.x, d.y, d.z};
  hits->clear();
  auto test = [&](int64_t tri) {
    double t;
    const int r = ray_triangle(oo, dd, s.verts + 3 * (int64_t)s.tris[3 * tri], s.verts + 3 * (int64_t)s.tris[3 * tri + 1],
                               s.verts + 3 * (int64_t)s.tris[3 * tri + 2], &t);
    ++*n_tests;
    if (r != 0) hits->push_back({t, r});
  };
  if (!use_grid || !mp.has_grid) {
    for (int64_t tri = 0; tri < s.n_tris; ++tri) test(tri);
    return;
  }
  const MeshGrid& g = mp.g;
  // clip the line to the grid box
  double tmin = -kInf, tmax = kInf;
  for (int a = 0; a < 3; ++a) {
    const double lo = g.lo[a], hi = g.lo[a] + g.cell[a] * g.n[a];
    if (!slab_axis(oo[a], dd[a], lo, hi, &tmin, &tmax)) return;
  }
  if (!(tmin < tmax)) return;
  // walk the cells the line crosses and test every triangle listed in a visited cell, each once per ray
  if (++mp.stamp_id == 0) { std::fill(mp.stamp.begin(), mp.stamp.end(), 0u); mp.stamp_id = 1; }
  int idx[3], step[3];
  double tMax[3], tDelta[3];
  for (int a = 0; a < 3; ++a) {
    const double q = oo[a] + tmin * dd[a];
    idx[a] = std::min(g.n[a] - 1, std::max(0, (int)std::floor((q - g.lo[a]) / g.cell[a])));
    if (dd[a] > 0.0) { step[a] = 1; tMax[a] = (g.lo[a] + (idx[a] + 1) * g.cell[a] - oo[a]) / dd[a]; tDelta[a] = g.cell[a] / dd[a]; }
    else if (dd[a] < 0.0) { step[a] = -1; tMax[a] = (g.lo[a] + idx[a] * g.cell[a] - oo[a]) / dd[a]; tDelta[a] = -g.cell[a] / dd[a]; }
    else { step[a] = 0; tMax[a] = kInf; tDelta[a] = kInf; }
  }
  while (true) {
    // the triangle lists carry slack, so rounding in this walk cannot lose a candidate
    const int64_t c = ((int64_t)idx[2] * g.n[1] + idx[1]) * g.n[0] + idx[0];
    for (int32_t k = g.start[c]; k < g.start[c + 1]; ++k) {
      const int32_t tri = g.items[k];
      if (mp.stamp[tri] != mp.stamp_id) { mp.stamp[tri] = mp.stamp_id; test(tri); }
    }
    int a = 0;
    if (tMax[1] < tMax[a]) a = 1;
    if (tMax[2] < tMax[a]) a = 2;
    if (tMax[a] > tmax) break;
    idx[a] += step[a];
    if (idx[a] < 0 || idx[a] >= g.n[a]) break;
    tMax[a] += tDelta[a];
  }
}

struct Interval { double a, b; int solid; };

// Step 9 (second half): sort hits, collapse consecutive same-orientation hits (shared edge / vertex
// duplicates), pair enter/exit.  Returns false if the sequence is not enter,exit,enter,exit,...
bool hits_to_intervals(std::vector<Hit>* hits, int solid, std::vector<Interval>* out) {
  std::stable_sort(hits->begin(), hits->end(), [](const Hit& x, const Hit& y) {
    if (x.t != y.t) return x.t < y.t;
    return x.orient > y.orient;  // equal t: enter first
  });
  std::vector<Hit> seq;
  for (const Hit& h : *hits)
    if (seq.empty() || seq.back().orient != h.orient) seq.push_back(h);
  if (seq.empty()) return true;
  if (seq.size() % 2 != 0 || seq.front().orient != +1) return false;
  for (size_t k = 0; k < seq.size(); k += 2) out->push_back({seq[k].t, seq[k + 1].t, solid});
  return true;
}

// ---------------------------------------------------------------------------------------------------
// Step 12 helpers: elliptic-cylinder mirror constants (computed once per component)
// ---------------------------------------------------------------------------------------------------
struct MirrorPrep {
  double a, b;       // semi-axes
  double Z0, Y0;     // pole in the ellipse's principal frame (Z, Y)
  double nZ, nY;     // inward unit normal at the pole (mirror-frame y axis)
  double tZ, tY;     // unit tangent at the pole (mirror-frame z axis), tZ > 0
};

MirrorPrep mirror_prep(double p, double q, double theta) {
  MirrorPrep m;
  m.a = 0.5 * (p + q);
  m.b = std::sqrt(p * q) * std::sin(theta);
  const double c = std::sqrt(m.a * m.a - m.b * m.b);
  m.Z0 = (p - m.a) * m.a / c;  // |P F1| = a + (c/a) Z0 = p, F1 = (-c, 0)
  m.Y0 = -m.b * std::sqrt(1.0 - (m.Z0 * m.Z0) / (m.a * m.a));
  const double gZ = m.Z0 / (m.a * m.a), gY = m.Y0 / (m.b * m.b);  // grad F / 2
  const double gn = std::sqrt(gZ * gZ + gY * gY);
  m.nZ = -gZ / gn; m.nY = -gY / gn;  // inward
  m.tZ = m.nY; m.tY = -m.nZ;         // n rotated by -90 degrees
  return m;
}

// ---------------------------------------------------------------------------------------------------
// prepared instrument
// ---------------------------------------------------------------------------------------------------
struct Prepared {
  const OrcComponent* comps;
  int n_comps;
  std::vector<MuTable> mats;
  std::vector<std::vector<double>> cdf;          // per component (sources with a spectrum)
  std::vector<std::vector<MeshPrep>> meshes;     // per component, per solid
  std::vector<MirrorPrep> mirrors;               // per component
  std::vector<int> det_index;                    // per component: detector ordinal or -1
  std::vector<MuTable> lens_delta;               // per component: delta(E) of a lens as ln-tables
  bool use_grid;
};

void prepare(Prepared* P, const OrcComponent* comps, int n_comps, const OrcMaterial* mats, int n_mats, int mesh_accel) {
  P->comps = comps; P->n_comps = n_comps; P->use_grid = mesh_accel != 0;
  P->mats.resize(n_mats);
  for (int m = 0; m < n_mats; ++m) {
    MuTable& t = P->mats[m];
    for (int64_t j = 0; j < mats[m].n; ++j) {
      t.E.push_back(mats[m].E[j]);
      t.lnE.push_back(std::log(mats[m].E[j]));
      t.lnMu.push_back(std::log(mats[m].mu[j]));
      if (mats[m].mu_s) t.lnMuS.push_back(std::log(mats[m].mu_s[j]));
    }
  }
  P->cdf.resize(n_comps); P->meshes.resize(n_comps); P->mirrors.resize(n_comps); P->det_index.assign(n_comps, -1);
  P->lens_delta.resize(n_comps);
  int ndet = 0;
  for (int c = 0; c < n_comps; ++c) {
    const OrcComponent& k = comps[c];
    if (k.kind == K_SOURCE && k.e_mode == E_SPECTRUM) {
      // step 3: C[j] = sum_{m<j} S[m], plain running sum
      std::vector<double>& C = P->cdf[c];
      C.assign(k.spec_n + 1, 0.0);
      for (int64_t j = 0; j < k.spec_n; ++j) C[j + 1] = C[j] + k.spectrum[j];
    }
    if (k.kind == K_SOLIDS) {
      P->meshes[c].resize(k.n_solids);
      for (int64_t s = 0; s < k.n_solids; ++s) {
        P->meshes[c][s].s = &k.solids[s];
        if (k.solids[s].shape == S_MESH && P->use_grid) {
          build_mesh_grid(&P->meshes[c][s], grid_resolution(k.solids[s].n_tris));
        }
      }
    }
    if (k.kind == K_MIRROR) P->mirrors[c] = mirror_prep(k.mir_p, k.mir_q, k.mir_theta);
    if (k.kind == K_DETECTOR) P->det_index[c] = ndet++;
    if (k.kind == K_LENS) {
      MuTable& t = P->lens_delta[c];
      for (int64_t j = 0; j < k.lens_nd; ++j) {
        t.E.push_back(k.lens_dE[j]);
        t.lnE.push_back(std::log(k.lens_dE[j]));
        t.lnMu.push_back(std::log(k.lens_delta[j]));
      }
    }
  }
}

struct Work { uint64_t voxel_steps = 0, solid_tests = 0, tri_tests = 0, segments = 0; };

// Step 13: symmetric Bragg, thick non-absorbing crystal (Darwin curve), cancellation-free tail.
double darwin_R(double eta) {
  const double ae = std::fabs(eta);
  if (ae <= 1.0) return 1.0;
  const double s = ae + std::sqrt(ae * ae - 1.0);
  return 1.0 / (s * s);
}

// Step 13b (reading in DESIGN.md): Darwin-Prins curve of a thick ABSORBING crystal in symmetric
// Bragg geometry (Zachariasen 1945, eq. 3.192 in reduced form): with the complex deviation parameter
//   eta_c = (eta + i g) / (1 + i kappa),   g = Im(chi_0) / Re(chi_h) >= 0,  kappa = Im(chi_h) / Re(chi_h),
// the reflectivity is R = |eta_c - s|^2, s = the square root of eta_c^2 - 1 for which |eta_c - s| <= 1.  Because
// (eta_c - s)(eta_c + s) = 1 this is R = 1 / |eta_c + s|^2 with s the root whose inner product with eta_c is
// non-negative: no cancellation.  g = kappa = 0 is the Darwin curve of step 13 (and is evaluated by darwin_R).
double darwin_prins_R(double eta, double g, double kappa) {
  if (g == 0.0 && kappa == 0.0) return darwin_R(eta);
  const std::complex<double> ec = std::complex<double>(eta, g) / std::complex<double>(1.0, kappa);
  std::complex<double> s = std::sqrt(ec * ec - 1.0);
  if (ec.real() * s.real() + ec.imag() * s.imag() < 0.0) s = -s;
  return 1.0 / std::norm(ec + s);
}

// Step 12: bilinear R(theta, E) on a uniform grid; theta above range is handled by the caller.
double bilinear_R(const OrcComponent& k, double theta, double E) {
  const int64_t nt = k.tab_n_theta, nE = k.tab_n_E;
  double ft = (theta - k.tab_theta_min) / (k.tab_theta_max - k.tab_theta_min) * (double)(nt - 1);
  double fe = (E - k.tab_E_min) / (k.tab_E_max - k.tab_E_min) * (double)(nE - 1);
  if (ft < 0.0) ft = 0.0;
  if (ft > (double)(nt - 1)) ft = (double)(nt - 1);
  if (fe < 0.0) fe = 0.0;
  if (fe > (double)(nE - 1)) fe = (double)(nE - 1);
  int64_t it = (int64_t)std::floor(ft), ie = (int64_t)std::floor(fe);
  if (it > nt - 2) it = nt - 2;
  if (ie > nE - 2) ie = nE - 2;
  const double wt = ft - (double)it, we = fe - (double)ie;
  const double r00 = k.tab_R[it * nE + ie], r01 = k.tab_R[it * nE + ie + 1];
  const double r10 = k.tab_R[(it + 1) * nE + ie], r11 = k.tab_R[(it + 1) * nE + ie + 1];
  return (1.0 - wt) * ((1.0 - we) * r00 + we * r01) + wt * ((1.0 - we) * r10 + we * r11);
}

struct Ray { V3 r, d; double E, p; };

// ---------------------------------------------------------------------------------------------------
// the components, one function each.  Return true if the ray continues.
// ---------------------------------------------------------------------------------------------------

// Step 3.  Slot 0 -> position, slot 1 -> direction, slot 2 -> energy.
void source_sample(const Prepared& P, int c, uint64_t seed, uint64_t i, Ray* ray) {
  const OrcComponent& k = P.comps[c];
  double ua, ub, uc, ud, ue, uf;
  V3 r{0.0, 0.0, 0.0}, d{0.0, 0.0, 1.0};
  if (k.pos_mode == POS_DISK) {
    draw2(seed, i, 0, (uint32_t)c, &ua, &ub);
    const double rad = k.radius * std::sqrt(ua), ang = 2.0 * kPi * ub;
    r = {rad * std::cos(ang), rad * std::sin(ang), 0.0};
  } else if (k.pos_mode == POS_GAUSS) {
    draw2(seed, i, 0, (uint32_t)c, &ua, &ub);
    double g0, g1;
    gauss_pair(ua, ub, &g0, &g1);
    r = {k.sigma_x * g0, k.sigma_y * g1, 0.0};
  }
  draw2(seed, i, 1, (uint32_t)c, &uc, &ud);
  if (k.dir_mode == DIR_TARGET) {  // uniform in area on the target rectangle, no solid-angle weight (R6)
    const V3 target{(uc - 0.5) * k.target_w, (ud - 0.5) * k.target_h, k.target_dist};
    const V3 v = target - r;
    d = (1.0 / std::sqrt(dot(v, v))) * v;
  } else {  // Gaussian tangents, then normalise (R7)
    double g0, g1;
    gauss_pair(uc, ud, &g0, &g1);
    const V3 v{k.div_x * g0, k.div_y * g1, 1.0};
    d = (1.0 / std::sqrt(dot(v, v))) * v;
  }
  double E = k.E0;
  if (k.e_mode == E_UNIFORM) {
    draw2(seed, i, 2, (uint32_t)c, &ue, &uf);
    E = k.E0 * (1.0 + k.dE_rel * (2.0 * ue - 1.0));
  } else if (k.e_mode == E_SPECTRUM) {  // inverse CDF, p = 1 (R9)
    draw2(seed, i, 2, (uint32_t)c, &ue, &uf);
    const std::vector<double>& C = P.cdf[c];
    const int64_t n = k.spec_n;
    const double v = ue * C[n];
    int64_t j = (int64_t)(std::upper_bound(C.begin(), C.end(), v) - C.begin()) - 1;  // largest j with C[j] <= v
    if (j > n - 1) j = n - 1;
    if (j < 0) j = 0;
    const double dE = (k.spec_Emax - k.spec_Emin) / (double)n;
    E = k.spec_Emin + ((double)j + (v - C[j]) / (C[j + 1] - C[j])) * dE;
  }
  ray->r = to_lab_pos(k.R, k.T, r);
  ray->d = rotT(k.R, d);
  ray->E = E;
  ray->p = 1.0;
}

// Step 5: propagate to the plane z' = 0 of the component frame.
bool plane_hit(const OrcComponent& k, const Ray& ray, V3* hit, V3* dloc) {
  const V3 o = to_local_pos(k.R, k.T, ray.r);
  const V3 d = rot(k.R, ray.d);
  if (!(d.z > 0.0)) return false;
  const double t = -o.z / d.z;
  if (t < 0.0) return false;
  *hit = o + t * d;
  *dloc = d;
  return true;
}

// Step 6.  The slit only tests; the lab-frame ray is left as it is (its line does not change).
bool slit(const OrcComponent& k, const Ray& ray) {
  V3 h, d;
  if (!plane_hit(k, ray, &h, &d)) return false;
  if (k.kind == K_SLIT_RECT) return std::fabs(h.x) <= 0.5 * k.xw && std::fabs(h.y) <= 0.5 * k.yh;
  return h.x * h.x + h.y * h.y <= k.slit_radius * k.slit_radius;
}

struct Seg { double ta, tb; int material; };  // a stretch of the ray inside one material

// Step 17 (a step updates "the ray's attenuation (Monte Carlo weight) and direction
// (wavevector)"; reading in DESIGN.md).  Elastic scattering with the Thomson angular distribution
// dsigma/dOmega ~ 1 + cos^2(theta): cos(theta) by inversion of its distribution function
// F(x) = 1/2 + (3/8)(x + x^3/3), i.e. the real root of x^3 + 3x - (8u - 4) = 0, x = w - 1/w with
// w = cbrt(q + sqrt(q^2 + 1)), q = 4u - 2 (Cardano); azimuth phi = 2 pi u'.  The new direction is
// cos(theta) d + sin(theta) (cos(phi) e1 + sin(phi) e2), e1 = (d x a) / |d x a| with a the coordinate axis along which
// |d| is smallest (ties: the lowest axis), e2 = d x e1; normalised once more.
V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }

V3 scatter_direction(V3 d, double u_mu, double u_phi) {
  const double q = 4.0 * u_mu - 2.0;
  const double w = std::cbrt(q + std::sqrt(q * q + 1.0));
  const double ct = w - 1.0 / w;
  const double st = std::sqrt(std::max(0.0, 1.0 - ct * ct));
  const double phi = 2.0 * kPi * u_phi;
  V3 a{1.0, 0.0, 0.0};
  double m = std::fabs(d.x);
  if (std::fabs(d.y) < m) { a = {0.0, 1.0, 0.0}; m = std::fabs(d.y); }
  if (std::fabs(d.z) < m) { a = {0.0, 0.0, 1.0}; }
  V3 e1 = cross(d, a);
  e1 = (1.0 / std::sqrt(dot(e1, e1))) * e1;
  const V3 e2 = cross(d, e1);
  const V3 v = ct * d + st * (std::cos(phi) * e1 + std::sin(phi) * e2);
  return (1.0 / std::sqrt(dot(v, v))) * v;
}

// Step 17: the walk of one ray through a sample with up to K direction changes.  `segments(o, d, &segs)` gives the
// stretches of the half-line o + t d, t >= 0, inside materials, in order (1 = ok, 0 = degenerate).  Leg k < K draws
// (u_f, u_mu) from slot 2k and u_phi from slot 2k + 1 of this component (step 1): the scattering optical depth to the next
// event is -ln(u_f); walking the stretches, the event lies where the running sum of mu_s * length reaches it.  Up to
// there, and on a leg that leaves the sample without an event, the weight is attenuated by what does not scatter,
// mu - mu_s; once the K events are used up a further scattering counts as a loss and the full mu attenuates.  K = 0 or
// mu_s = 0 is Beer-Lambert as in steps 10 and 11.  *o, *d: the ray, updated at every event; *tau: the optical depth of
// the weight, accumulated over all legs.
template <class SegFn>
int scatter_walk(const Prepared& P, int c, int64_t K, uint64_t seed, uint64_t i, double E, V3* o, V3* d, SegFn segments,
                 double* tau, int* n_events) {
  std::vector<Seg> segs;
  int64_t k = 0;
  for (;;) {
    segs.clear();
    if (!segments(*o, *d, &segs)) return 0;
    double tau_s = kInf, u_mu = 0.0;
    if (k < K) {
      double u_f;
      draw2(seed, i, (uint32_t)(2 * k), (uint32_t)c, &u_f, &u_mu);
      tau_s = -std::log(u_f);
    }
    double cum = 0.0;
    bool event = false;
    for (const Seg& sg : segs) {
      const double len = sg.tb - sg.ta;
      const double mt = mu_of_E(P.mats[sg.material], E);
      const double ms = k < K ? mu_s_of_E(P.mats[sg.material], E) : 0.0;
      if (k < K && ms > 0.0 && cum + ms * len >= tau_s) {
        const double l = (tau_s - cum) / ms;
        *tau += (mt - ms) * l;
        double u_phi, unused;
        draw2(seed, i, (uint32_t)(2 * k + 1), (uint32_t)c, &u_phi, &unused);
        *o = *o + (sg.ta + l) * (*d);
        *d = scatter_direction(*d, u_mu, u_phi);
        ++k;
        event = true;
        break;
      }
      cum += ms * len;
      *tau += (mt - ms) * len;
    }
    if (!event) break;
  }
  *n_events = (int)k;
  return 1;
}

// Steps 8-10 up to the elementary segments of the half-line r + t d, t >= 0, and their owners.  1 = ok, 0 = degenerate.
int solid_segments(const Prepared& P, int c, V3 r, V3 dl, Work* w, std::vector<Seg>* segs) {
  const OrcComponent& k = P.comps[c];
  std::vector<Interval> iv;
  std::vector<Hit> hits;
  for (int64_t s = 0; s < k.n_solids; ++s) {
    const OrcSolid& S = k.solids[s];
    const V3 o = to_local_pos(S.R, S.T, r);
    const V3 d = rot(S.R, dl);
    double a, b;
    bool hit = false;
    w->solid_tests++;
    if (S.shape == S_BOX) hit = box_interval(o, d, S.hx, S.hy, S.hz, &a, &b);
    else if (S.shape == S_CYL) hit = cylinder_interval(o, d, S.radius, S.half_height, &a, &b);
    else if (S.shape == S_SPHERE) hit = sphere_interval(o, d, S.radius, &a, &b);
    else {
      mesh_hits(P.meshes[c][s], o, d, P.use_grid, &hits, &w->tri_tests);
      if (!hits_to_intervals(&hits, (int)s, &iv)) return 0;
      continue;
    }
    if (hit) iv.push_back({a, b, (int)s});
  }
  // clip to t >= 0 (step 8)
  std::vector<Interval> cl;
  for (Interval x : iv) {
    if (x.a < 0.0) x.a = 0.0;
    if (x.b > x.a) cl.push_back(x);
  }
  if (cl.empty()) return 1;
  // step 10: all endpoints sorted; classify each elementary segment by its midpoint
  std::vector<double> ts;
  for (const Interval& x : cl) { ts.push_back(x.a); ts.push_back(x.b); }
  std::sort(ts.begin(), ts.end());
  for (size_t m = 0; m + 1 < ts.size(); ++m) {
    const double ta = ts[m], tb = ts[m + 1];
    if (!(tb > ta)) continue;
    const double mid = 0.5 * (ta + tb);
    int owner = -1, best = std::numeric_limits<int>::min();
    for (const Interval& x : cl)
      if (x.a <= mid && mid <= x.b) {
        const int pr = k.solids[x.solid].priority;
        if (owner < 0 || pr > best) { owner = x.solid; best = pr; }
      }
    if (owner < 0) continue;  // vacuum gap
    w->segments++;
    segs->push_back({ta, tb, k.solids[owner].material});
  }
  return 1;
}

// Steps 8-10 (and 17 where the group scatters).  Returns 1 = continue, 0 = degenerate.
int solids(const Prepared& P, int c, Ray* ray, Work* w, uint64_t seed, uint64_t i) {
  const OrcComponent& k = P.comps[c];
  if (k.scatter_order > 0) {
    double tau = 0.0;
    int n_events = 0;
    V3 o = ray->r, d = ray->d;
    auto segments = [&](V3 oo, V3 dd, std::vector<Seg>* segs) { return solid_segments(P, c, oo, dd, w, segs); };
    if (!scatter_walk(P, c, k.scatter_order, seed, i, ray->E, &o, &d, segments, &tau, &n_events)) return 0;
    ray->p *= std::exp(-tau);
    if (n_events > 0) { ray->r = o; ray->d = d; }
    return 1;
  }
  std::vector<Seg> segs;
  if (!solid_segments(P, c, ray->r, ray->d, w, &segs)) return 0;
  if (segs.empty()) return 1;
  double tau = 0.0;
  for (const Seg& sg : segs) tau += mu_of_E(P.mats[sg.material], ray->E) * (sg.tb - sg.ta);
  ray->p *= std::exp(-tau);
  return 1;
}

// Step 11: exact traversal of the voxel grid (Amanatides & Woo 1987), R15/R16.
void voxels(const Prepared& P, int c, Ray* ray, Work* w) {
  const OrcComponent& k = P.comps[c];
  const V3 ol = to_local_pos(k.R, k.T, ray->r);
  const V3 dl = rot(k.R, ray->d);
  const double o[3] = {ol.x, ol.y, ol.z}, d[3] = {dl.x, dl.y, dl.z};
  const int64_t n[3] = {k.vnx, k.vny, k.vnz};
  const double h = k.vox_h;
  double t0 = -kInf, t1 = kInf;
  for (int a = 0; a < 3; ++a)
    if (!slab_axis(o[a], d[a], 0.0, (double)n[a] * h, &t0, &t1)) return;
  if (t0 < 0.0) t0 = 0.0;
  if (!(t0 < t1)) return;
  int64_t idx[3];
  int step[3];
  for (int a = 0; a < 3; ++a) {
    const double q = o[a] + t0 * d[a];
    int64_t v = (int64_t)std::floor(q / h);
    idx[a] = std::min(n[a] - 1, std::max((int64_t)0, v));
    step[a] = d[a] > 0.0 ? 1 : (d[a] < 0.0 ? -1 : 0);
  }
  // parameter of the next face along axis a, recomputed from the integer index (no drift)
  auto next_face = [&](int a) {
    if (step[a] == 0) return kInf;
    const double face = (double)(idx[a] + (step[a] > 0 ? 1 : 0)) * h;
    return (face - o[a]) / d[a];
  };
  // per-ray mu of every material once (step 7)
  std::vector<double> mu(P.mats.size());
  for (size_t m = 0; m < P.mats.size(); ++m) mu[m] = mu_of_E(P.mats[m], ray->E);
  double tau = 0.0, tcur = t0;
  while (true) {
    const double tx = next_face(0), ty = next_face(1), tz = next_face(2);
    int a = 0;
    double tn = tx;
    if (ty < tn) { tn = ty; a = 1; }
    if (tz < tn) { tn = tz; a = 2; }
    const bool last = !(tn < t1);
    if (last) tn = t1;
    const uint8_t id = k.vox_ids[(idx[2] * n[1] + idx[1]) * n[0] + idx[0]];
    w->voxel_steps++;
    if (tn > tcur) { tau += mu[id] * (tn - tcur); tcur = tn; }
    if (last) break;
    idx[a] += step[a];
    if (idx[a] < 0 || idx[a] >= n[a]) break;
  }
  ray->p *= std::exp(-tau);
}

// Step 11 as a list: the voxels the half-line o + t d, t >= 0, crosses (volume frame), one stretch per voxel visited
// with positive length, in the order and with the face parameters of voxels() above.
int voxel_segments(const OrcComponent& k, V3 ol, V3 dl, Work* w, std::vector<Seg>* segs) {
  const double o[3] = {ol.x, ol.y, ol.z}, d[3] = {dl.x, dl.y, dl.z};
  const int64_t n[3] = {k.vnx, k.vny, k.vnz};
  const double h = k.vox_h;
  double t0 = -kInf, t1 = kInf;
  for (int a = 0; a < 3; ++a)
    if (!slab_axis(o[a], d[a], 0.0, (double)n[a] * h, &t0, &t1)) return 1;
  if (t0 < 0.0) t0 = 0.0;
  if (!(t0 < t1)) return 1;
  int64_t idx[3];
  int step[3];
  for (int a = 0; a < 3; ++a) {
    const double q = o[a] + t0 * d[a];
    int64_t v = (int64_t)std::floor(q / h);
    idx[a] = std::min(n[a] - 1, std::max((int64_t)0, v));
    step[a] = d[a] > 0.0 ? 1 : (d[a] < 0.0 ? -1 : 0);
  }
  auto next_face = [&](int a) {
    if (step[a] == 0) return kInf;
    const double face = (double)(idx[a] + (step[a] > 0 ? 1 : 0)) * h;
    return (face - o[a]) / d[a];
  };
  double tcur = t0;
  while (true) {
    const double tx = next_face(0), ty = next_face(1), tz = next_face(2);
    int a = 0;
    double tn = tx;
    if (ty < tn) { tn = ty; a = 1; }
    if (tz < tn) { tn = tz; a = 2; }
    const bool last = !(tn < t1);
    if (last) tn = t1;
    const uint8_t id = k.vox_ids[(idx[2] * n[1] + idx[1]) * n[0] + idx[0]];
    w->voxel_steps++;
    if (tn > tcur) { segs->push_back({tcur, tn, (int)id}); tcur = tn; }
    if (last) break;
    idx[a] += step[a];
    if (idx[a] < 0 || idx[a] >= n[a]) break;
  }
  return 1;
}

// Steps 11 + 17: a voxel volume that scatters (scatter_order > 0).  The walk runs in the volume's frame.
void voxels_scatter(const Prepared& P, int c, Ray* ray, Work* w, uint64_t seed, uint64_t i) {
  const OrcComponent& k = P.comps[c];
  V3 o = to_local_pos(k.R, k.T, ray->r), d = rot(k.R, ray->d);
  double tau = 0.0;
  int n_events = 0;
  auto segments = [&](V3 oo, V3 dd, std::vector<Seg>* segs) { return voxel_segments(k, oo, dd, w, segs); };
  scatter_walk(P, c, k.scatter_order, seed, i, ray->E, &o, &d, segments, &tau, &n_events);
  ray->p *= std::exp(-tau);
  if (n_events > 0) {
    ray->r = to_lab_pos(k.R, k.T, o);
    ray->d = rotT(k.R, d);
  }
}

// Step 12.  Returns true if reflected.
bool mirror(const Prepared& P, int c, Ray* ray) {
  const OrcComponent& k = P.comps[c];
  const MirrorPrep& m = P.mirrors[c];
  const V3 o = to_local_pos(k.R, k.T, ray->r);
  const V3 d = rot(k.R, ray->d);
  // mirror frame (x sagittal, y normal, z tangential) -> ellipse principal frame (Z, Y)
  const double oZ = m.Z0 + o.z * m.tZ + o.y * m.nZ, oY = m.Y0 + o.z * m.tY + o.y * m.nY;
  const double dZ = d.z * m.tZ + d.y * m.nZ, dY = d.z * m.tY + d.y * m.nY;
  const double ia2 = 1.0 / (m.a * m.a), ib2 = 1.0 / (m.b * m.b);
  const double A = dZ * dZ * ia2 + dY * dY * ib2;
  const double B = oZ * dZ * ia2 + oY * dY * ib2;
  const double C = oZ * oZ * ia2 + oY * oY * ib2 - 1.0;
  if (A == 0.0) return false;
  const double disc = B * B - A * C;
  if (!(disc >= 0.0)) return false;
  // stable roots of A t^2 + 2 B t + C = 0
  const double qq = -(B + (B >= 0.0 ? 1.0 : -1.0) * std::sqrt(disc));
  double ta = qq / A, tb = (qq != 0.0) ? C / qq : ta;
  if (ta > tb) std::swap(ta, tb);
  const double cand[2] = {ta, tb};
  for (int r = 0; r < 2; ++r) {
    const double t = cand[r];
    if (!(t > 0.0)) continue;
    const V3 h = o + t * d;
    if (std::fabs(h.z) > 0.5 * k.mir_length || std::fabs(h.x) > 0.5 * k.mir_width) continue;
    // the arc near the pole only (the far side of the ellipse also satisfies the quadratic)
    const double hZ = m.Z0 + h.z * m.tZ + h.y * m.nZ, hY = m.Y0 + h.z * m.tY + h.y * m.nY;
    if (!(hY < 0.0)) continue;
    const double gZ = hZ * ia2, gY = hY * ib2;
    const double gn = std::sqrt(gZ * gZ + gY * gY);
    const double nZ = -gZ / gn, nY = -gY / gn;  // inward normal in (Z, Y)
    // back to the mirror frame: components along t (z) and n0 (y)
    const V3 nrm{0.0, nZ * m.nZ + nY * m.nY, nZ * m.tZ + nY * m.tY};
    const double dn = dot(d, nrm);
    if (!(dn < 0.0)) return false;
    const double theta = std::asin(-dn);
    if (theta > k.tab_theta_max) return false;
    ray->p *= bilinear_R(k, theta, ray->E);
    const V3 dr = d - (2.0 * dn) * nrm;
    ray->r = to_lab_pos(k.R, k.T, h);
    ray->d = rotT(k.R, dr);
    return true;
  }
  return false;
}

// Step 13.  Crystal frame: surface = plane y' = 0, normal +y', z' along the length.
bool crystal(const OrcComponent& k, Ray* ray) {
  const V3 o = to_local_pos(k.R, k.T, ray->r);
  const V3 d = rot(k.R, ray->d);
  if (!(d.y < 0.0)) return false;
  const double t = -o.y / d.y;
  if (!(t > 0.0)) return false;
  const V3 h = o + t * d;
  if (std::fabs(h.z) > 0.5 * k.xtal_length || std::fabs(h.x) > 0.5 * k.xtal_width) return false;
  const double theta = std::asin(-d.y);
  const double lambda = kHC_keV_A / ray->E;
  const double s = lambda / (2.0 * k.xtal_d);
  if (!(s < 1.0)) return false;
  const double thetaB = std::asin(s);
  const double wD = k.xtal_zeta * std::tan(thetaB);
  const double eta = (theta - thetaB - k.xtal_delta0) / (0.5 * wD);
  ray->p *= darwin_prins_R(eta, k.xtal_g, k.xtal_kappa);
  const V3 dr{d.x, -d.y, d.z};
  ray->r = to_lab_pos(k.R, k.T, V3{h.x, 0.0, h.z});
  ray->d = rotT(k.R, dr);
  return true;
}

// Step 16 ("a stack of sixteen double-sided parabolic beryllium lenses",
// where problem 2 spends its time).  Lens frame: z = axis of the stack, origin at its centre.  Lens i = 0..N-1 is centred
// at z_i = (i - (N-1)/2) pitch and is material between two paraboloids of revolution, apex radius R, web thickness d:
//   front surface  z = z_i - d/2 - rho^2 / (2R)   (the ray enters the material),
//   back surface   z = z_i + d/2 + rho^2 / (2R)   (the ray leaves it),        rho^2 = x^2 + y^2.
// The ray meets the 2N surfaces in order.  At each: intersection (the root of the quadratic that tends to the plane
// intersection as R -> inf, in its cancellation-free form), aperture test rho <= r_a (outside: absorbed by the holder),
// Snell's law in vector form with n = 1 - delta(E) inside the material.  With m = n_before / n_after, c = d.nrm > 0
// (nrm = unit normal along +z) and c_t = sqrt(1 - m^2 (1 - c^2)):  d' = m d + (c_t - m c) nrm, where
// c_t - m c = (1 - m)(1 + m) / (c_t + m c) and 1 - m is formed from delta directly (entering: -delta / (1 - delta),
// leaving: delta), so the deflection, of relative size delta ~ 1e-6, carries no cancellation.  Total reflection or a
// ray running backwards: absorbed.  Beer-Lambert with mu(E) of the lens material over the summed path inside the N lenses.
bool lens(const Prepared& P, int c, Ray* ray) {
  const OrcComponent& k = P.comps[c];
  V3 o = to_local_pos(k.R, k.T, ray->r);
  V3 d = rot(k.R, ray->d);
  const double delta = mu_of_E(P.lens_delta[c], ray->E);  // the same log-log interpolation as mu(E), step 7
  const double n_in = 1.0 - delta;
  double path = 0.0;
  for (int64_t surf = 0; surf < 2 * k.lens_N; ++surf) {
    const int64_t i = surf / 2;
    const bool entering = (surf % 2) == 0;
    const double zc = ((double)i - 0.5 * (double)(k.lens_N - 1)) * k.lens_pitch;
    const double sgn = entering ? -1.0 : 1.0;
    const double z0 = zc + sgn * 0.5 * k.lens_d;
    // F(r) = z - z0 - sgn rho^2 / (2R) = 0 along o + t d:  a t^2 + b t + cc = 0
    const double a = -sgn * (d.x * d.x + d.y * d.y) / (2.0 * k.lens_R);
    const double b = d.z - sgn * (o.x * d.x + o.y * d.y) / k.lens_R;
    const double cc = o.z - z0 - sgn * (o.x * o.x + o.y * o.y) / (2.0 * k.lens_R);
    if (!(b > 0.0)) return false;
    const double disc = b * b - 4.0 * a * cc;
    if (!(disc >= 0.0)) return false;
    const double t = -2.0 * cc / (b + std::sqrt(disc));
    if (t < 0.0) return false;
    const V3 h = o + t * d;
    if (h.x * h.x + h.y * h.y > k.lens_ra * k.lens_ra) return false;
    if (!entering) path += t;  // d is unit: t is the length of the chord inside lens i
    // unit normal along +z: grad F = (-sgn x / R, -sgn y / R, 1)
    const V3 gr{-sgn * h.x / k.lens_R, -sgn * h.y / k.lens_R, 1.0};
    const V3 nrm = (1.0 / std::sqrt(dot(gr, gr))) * gr;
    const double cs = dot(d, nrm);
    if (!(cs > 0.0)) return false;
    const double m = entering ? 1.0 / n_in : n_in;
    const double one_minus_m = entering ? -delta / n_in : delta;
    const double under = 1.0 - m * m * (1.0 - cs * cs);
    if (!(under > 0.0)) return false;  // total reflection
    const double ct = std::sqrt(under);
    const double coef = one_minus_m * (1.0 + m) / (ct + m * cs);
    d = m * d + coef * nrm;
    o = h;
  }
  ray->p *= std::exp(-mu_of_E(P.mats[k.lens_material], ray->E) * path);
  ray->r = to_lab_pos(k.R, k.T, o);
  ray->d = rotT(k.R, d);
  return true;
}

// Step 14.  Returns the bin or -1.
int64_t detector_bin(const OrcComponent& k, const Ray& ray) {
  V3 h, d;
  if (!plane_hit(k, ray, &h, &d)) return -1;
  const double fx = (h.x - k.det_xmin) / (k.det_xmax - k.det_xmin) * (double)k.det_nx;
  const double fy = (h.y - k.det_ymin) / (k.det_ymax - k.det_ymin) * (double)k.det_ny;
  // step 14b: an L_monitor bins the wavelength lambda = hc / E [Angstrom] instead of the energy
  const double q = k.det_mode == DET_WAVELENGTH ? kHC_keV_A / ray.E : ray.E;
  const double fe = (q - k.det_Emin) / (k.det_Emax - k.det_Emin) * (double)k.det_nE;
  const double ix = std::floor(fx), iy = std::floor(fy), ie = std::floor(fe);
  if (!(ix >= 0.0 && ix < (double)k.det_nx)) return -1;
  if (!(iy >= 0.0 && iy < (double)k.det_ny)) return -1;
  if (!(ie >= 0.0 && ie < (double)k.det_nE)) return -1;
  return ((int64_t)iy * k.det_nx + (int64_t)ix) * k.det_nE + (int64_t)ie;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
// C entry points (called from oracle/oracle.py through ctypes)
// ---------------------------------------------------------------------------------------------------
extern "C" {

// Trace rays [first, first+n).  Tallies accumulate (R2): N[det][bin] += 1, P += p, P2 += p*p.
// absorbed: [n_comps]; fates: [3] = detected, missed, degenerate; dump: nullable [n]; work: nullable [4].
int orc_trace(const OrcComponent* comps, int n_comps, const OrcMaterial* mats, int n_mats, uint64_t first,
              uint64_t n, uint64_t seed, uint64_t** N, double** Pw, double** P2, uint64_t* absorbed,
              uint64_t* fates, OrcRayFate* dump, uint64_t* work, int mesh_accel) {
  if (n_comps < 1 || comps[0].kind != K_SOURCE) return 1;
  Prepared P;
  prepare(&P, comps, n_comps, mats, n_mats, mesh_accel);
  Work w;
  for (uint64_t q = 0; q < n; ++q) {
    const uint64_t i = first + q;
    Ray ray;
    source_sample(P, 0, seed, i, &ray);
    int fate = F_MISSED;
    int64_t bin = -1;
    for (int c = 1; c < n_comps; ++c) {
      const OrcComponent& k = comps[c];
      bool alive = true;
      switch (k.kind) {
        case K_SLIT_RECT: case K_SLIT_CIRC: alive = slit(k, ray); break;
        case K_SOLIDS:
          if (!solids(P, c, &ray, &w, seed, i)) { fate = F_DEGENERATE; alive = false; }
          break;
        case K_VOXELS:
          if (k.scatter_order > 0) voxels_scatter(P, c, &ray, &w, seed, i);
          else voxels(P, c, &ray, &w);
          break;
        case K_MIRROR: alive = mirror(P, c, &ray); break;
        case K_CRYSTAL: alive = crystal(k, &ray); break;
        case K_LENS: alive = lens(P, c, &ray); break;
        case K_DETECTOR: {
          const int64_t b = detector_bin(k, ray);
          if (b >= 0) {
            const int det = P.det_index[c];
            N[det][b] += 1; Pw[det][b] += ray.p; P2[det][b] += ray.p * ray.p;
            bin = b;
            fate = F_DETECTED;
          } else {
            fate = F_MISSED;  // a detector that is missed leaves the ray going (monitors do not absorb)
          }
          break;
        }
        default: return 2;
      }
      if (!alive) {
        if (fate != F_DEGENERATE) fate = c;
        break;
      }
      // fate of a ray that ends the chain = what the LAST component said (DETECTED / MISSED)
      if (k.kind != K_DETECTOR) fate = F_MISSED;
    }
    if (fate >= 0) absorbed[fate]++;
    else fates[-fate - 1]++;
    if (dump) dump[q] = OrcRayFate{fate, 0, fate == F_DETECTED ? bin : -1, ray.p};
  }
  if (work) { work[0] += w.voxel_steps; work[1] += w.solid_tests; work[2] += w.tri_tests; work[3] += w.segments; }
  return 0;
}

// ---- single-purpose wrappers so tests can pin each part on its own ----
void orc_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
double orc_u01(uint32_t wa, uint32_t wb) { return u01(wa, wb); }
void orc_draw2(uint64_t seed, uint64_t i, uint32_t slot, uint32_t comp, double* ua, double* ub) { draw2(seed, i, slot, comp, ua, ub); }
void orc_gauss_pair(double ua, double ub, double* g) { gauss_pair(ua, ub, &g[0], &g[1]); }

double orc_mu(const double* E, const double* mu, int64_t n, double Eq) {
  MuTable t;
  for (int64_t j = 0; j < n; ++j) { t.E.push_back(E[j]); t.lnE.push_back(std::log(E[j])); t.lnMu.push_back(std::log(mu[j])); }
  return mu_of_E(t, Eq);
}

// source sample of ray i for component list index 0 -> out[8] = r, d, E, p
void orc_source(const OrcComponent* comp, uint64_t seed, uint64_t i, double* out) {
  Prepared P;
  prepare(&P, comp, 1, nullptr, 0, 0);
  Ray ray;
  source_sample(P, 0, seed, i, &ray);
  out[0] = ray.r.x; out[1] = ray.r.y; out[2] = ray.r.z; out[3] = ray.d.x; out[4] = ray.d.y; out[5] = ray.d.z;
  out[6] = ray.E; out[7] = ray.p;
}

// primitive interval in the solid's own frame: returns 1 and ab[2] on a hit
int orc_primitive_interval(int shape, const double* o, const double* d, const double* dims, double* ab) {
  const V3 oo{o[0], o[1], o[2]}, dd{d[0], d[1], d[2]};
  bool hit = false;
  if (shape == S_BOX) hit = box_interval(oo, dd, dims[0], dims[1], dims[2], &ab[0], &ab[1]);
  else if (shape == S_CYL) hit = cylinder_interval(oo, dd, dims[0], dims[1], &ab[0], &ab[1]);
  else if (shape == S_SPHERE) hit = sphere_interval(oo, dd, dims[0], &ab[0], &ab[1]);
  return hit ? 1 : 0;
}

int orc_ray_triangle(const double* o, const double* d, const double* v0, const double* v1, const double* v2, double* t) {
  return ray_triangle(o, d, v0, v1, v2, t);
}

// all hits of the line with one mesh (solid-local frame).  Returns the number of hits written (<= cap),
// sorted by t; orient +1 enter / -1 exit.
int64_t orc_mesh_hits(const OrcSolid* solid, const double* o, const double* d, int use_grid, double* t, int32_t* orient,
                      int64_t cap, uint64_t* n_tests) {
  MeshPrep mp;
  mp.s = solid;
  if (use_grid) build_mesh_grid(&mp, grid_resolution(solid->n_tris));
  std::vector<Hit> hits;
  uint64_t tests = 0;
  mesh_hits(mp, V3{o[0], o[1], o[2]}, V3{d[0], d[1], d[2]}, use_grid != 0, &hits, &tests);
  std::sort(hits.begin(), hits.end(), [](const Hit& a, const Hit& b) { return a.t < b.t; });
  if (n_tests) *n_tests = tests;
  const int64_t m = std::min<int64_t>(cap, (int64_t)hits.size());
  for (int64_t k = 0; k < m; ++k) { t[k] = hits[k].t; orient[k] = hits[k].orient; }
  return (int64_t)hits.size();
}

// apply one non-source component to a given ray state: io[8] = r, d, E, p (lab frame).
// Returns 1 = continues, 0 = absorbed, -3 = degenerate.  For a detector, *bin receives the bin (or -1).
// (a scattering sample draws from the stream of ray index `ray_index` under `seed`, as component 1)
int orc_apply_seeded(const OrcComponent* comp, const OrcMaterial* mats, int n_mats, double* io, int64_t* bin, int mesh_accel,
                     uint64_t seed, uint64_t ray_index);
int orc_apply(const OrcComponent* comp, const OrcMaterial* mats, int n_mats, double* io, int64_t* bin, int mesh_accel) {
  return orc_apply_seeded(comp, mats, n_mats, io, bin, mesh_accel, 1, 0);
}
int orc_apply_seeded(const OrcComponent* comp, const OrcMaterial* mats, int n_mats, double* io, int64_t* bin, int mesh_accel,
                     uint64_t seed, uint64_t ray_index) {
  // the component is placed at chain index 1 behind a dummy slot so Prepared indexing matches
  OrcComponent two[2];
  std::memset(&two[0], 0, sizeof(OrcComponent));
  two[0].kind = K_SLIT_RECT;  // never executed
  two[1] = *comp;
  Prepared P;
  prepare(&P, two, 2, mats, n_mats, mesh_accel);
  Ray ray{V3{io[0], io[1], io[2]}, V3{io[3], io[4], io[5]}, io[6], io[7]};
  Work w;
  int rc = 1;
  if (bin) *bin = -1;
  switch (comp->kind) {
    case K_SLIT_RECT: case K_SLIT_CIRC: rc = slit(two[1], ray) ? 1 : 0; break;
    case K_SOLIDS: rc = solids(P, 1, &ray, &w, seed, ray_index) ? 1 : -3; break;
    case K_VOXELS:
      if (comp->scatter_order > 0) voxels_scatter(P, 1, &ray, &w, seed, ray_index);
      else voxels(P, 1, &ray, &w);
      break;
    case K_MIRROR: rc = mirror(P, 1, &ray) ? 1 : 0; break;
    case K_CRYSTAL: rc = crystal(two[1], &ray) ? 1 : 0; break;
    case K_LENS: rc = lens(P, 1, &ray) ? 1 : 0; break;
    case K_DETECTOR: { const int64_t b = detector_bin(two[1], ray); if (bin) *bin = b; break; }
    default: rc = -100;
  }
  io[0] = ray.r.x; io[1] = ray.r.y; io[2] = ray.r.z; io[3] = ray.d.x; io[4] = ray.d.y; io[5] = ray.d.z;
  io[6] = ray.E; io[7] = ray.p;
  return rc;
}

void orc_scatter_direction(const double* d, double u_mu, double u_phi, double* out) {
  const V3 v = scatter_direction(V3{d[0], d[1], d[2]}, u_mu, u_phi);
  out[0] = v.x; out[1] = v.y; out[2] = v.z;
}
double orc_darwin(double eta) { return darwin_R(eta); }
double orc_darwin_prins(double eta, double g, double kappa) { return darwin_prins_R(eta, g, kappa); }
double orc_bilinear(const OrcComponent* comp, double theta, double E) { return bilinear_R(*comp, theta, E); }
// mirror constants out[8] = a, b, Z0, Y0, nZ, nY, tZ, tY
void orc_mirror_prep(double p, double q, double theta, double* out) {
  const MirrorPrep m = mirror_prep(p, q, theta);
  out[0] = m.a; out[1] = m.b; out[2] = m.Z0; out[3] = m.Y0; out[4] = m.nZ; out[5] = m.nY; out[6] = m.tZ; out[7] = m.tY;
}

int64_t orc_sizeof_component(void) { return (int64_t)sizeof(OrcComponent); }
int64_t orc_sizeof_solid(void) { return (int64_t)sizeof(OrcSolid); }

}  // extern "C"
