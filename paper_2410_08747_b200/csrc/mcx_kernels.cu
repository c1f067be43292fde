// mcx_kernels.cu -- the ray-tracing megakernel and its helper kernels, hand-written for sm_100a.
//
// One thread traces one ray at a time through the whole component chain with its state (r, d, E, p) in fp64
// registers; a grid of 148 x k resident blocks pulls tiles of ray positions from a ticket counter.
// Step numbers are those of DESIGN.md "Readings".  This file shares no code with oracle/.
#include <math_constants.h>

#include <atomic>
#include <cstdio>

#include "mcx_device.h"

namespace mcx {

namespace {

constexpr int kBlock = 256;
constexpr unsigned kVoxelGuard = 255u;  // ID of the guard cells around the voxel volume (material IDs are < MCX_MAX_MATERIALS)

// What a block keeps of the instrument in shared memory: only the components and materials the instrument has (the
// arrays of DInstrument are sized for the limits of the ABI; every kilobyte of shared memory a block does not take is L1
// for the BVH and the voxel rows -- 512 bytes more per block cost the mesh config 12 %).
struct SInst {
  int n_comps, n_mats;
  const DComponent* comps;       // shared memory [n_comps]
  const DMaterial* mats;         // shared memory [n_mats]
  TallyBin* const* tallies;      // shared memory [MCX_MAX_DETECTORS]
  unsigned long long* counters;  // global
};

// ------------------------------------------------------------------------------------------------------------
// Step 1: Philox4x32-10 (Salmon et al., SC'11); key = seed, counter = (i lo, i hi, slot, component).
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                              uint32_t (&out)[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Step 2: the top 52 bits of (wa:wb), centred in their cell: u = (m + 1/2) 2^-52, exact in fp64.
// Built as [1 + m 2^-52] - [1 - 2^-53]; both the operand and the difference are exactly representable.
__device__ __forceinline__ double u01(uint32_t wa, uint32_t wb) {
  const double one_plus = __hiloint2double(0x3FF00000 | (int)(wa >> 12), (int)((wa << 20) | (wb >> 12)));
  return one_plus - 0.99999999999999988897769753748434595763683319091796875;  // 1 - 2^-53
}

__device__ __forceinline__ void draw2(uint64_t seed, uint64_t i, uint32_t slot, uint32_t comp, double& ua, double& ub) {
  uint32_t w[4];
  philox4x32_10((uint32_t)i, (uint32_t)(i >> 32), slot, comp, (uint32_t)seed, (uint32_t)(seed >> 32), w);
  ua = u01(w[0], w[1]);
  ub = u01(w[2], w[3]);
}

// 1 / x and sqrt(x) for the hot loops: the hardware's 20-bit seeds (MUFU.RCP64H / RSQ64H) and two Newton
// steps (2^-20 -> 2^-40 -> 2^-80) in explicit fmas -- within an ulp or two of the correctly rounded results of `/` and sqrt(), whose IEEE sequences cost
// about 25 and 30 instructions each (the lens spent 35 % of its instructions in two such lines).  For normal, finite,
// positive x (rcp: any sign); fast_sqrt returns 0 below 1e-280 (the callers have excluded negative arguments).  Used in the lens and the mirror: in the other
// kernels (source sampling, primitives, voxel set-up) the same substitution measured 0 to -4 %.
// (Measured on 1.6e9 random arguments over 120 binades: fast_rcp and fast_sqrt equal `/` and sqrt() bit for bit,
// fast_rsqrt is within 2.7e-16 of 1 / sqrt().)
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}
__device__ __forceinline__ double fast_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double h = 0.5 * x;
  double e = fma(-h * y, y, 0.5);
  y = fma(y, e, y);
  e = fma(-h * y, y, 0.5);
  return fma(y, e, y);
}
__device__ __forceinline__ double fast_sqrt(double x) {
  if (x < 1e-280) return 0.0;  // zero and what the seed would flush to zero: an absolute error below 1e-140
  const double y = fast_rsqrt(x);
  const double s = x * y;
  return fma(fma(-s, s, x), 0.5 * y, s);  // one more correction on the product
}

// Box-Muller, both values used (step 2)
__device__ __forceinline__ void gauss_pair(double ua, double ub, double& g0, double& g1) {
  const double rad = sqrt(-2.0 * log(ua));
  double s, c;
  sincospi(2.0 * ub, &s, &c);  // sin / cos of 2 pi u without the argument reduction of a general angle (within an ulp or two of both libraries' values of the rounded 2 pi u, like sincos itself)
  g0 = rad * c;
  g1 = rad * s;
}

struct Vec3 {
  double x, y, z;
};
__device__ __forceinline__ Vec3 operator+(Vec3 a, Vec3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ Vec3 operator-(Vec3 a, Vec3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ Vec3 operator*(double s, Vec3 a) { return {s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ double dot(Vec3 a, Vec3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }

// Step 4: into a component frame and back
// (a pose whose rotation is the identity -- most components of an in-line instrument -- skips the nine products: x * 1 +
// y * 0 + z * 0 is x exactly)
__device__ __forceinline__ Vec3 rotate(const DPose& P, Vec3 v) {
  if (P.identity) return v;
  const double* R = P.R;
  return {R[0] * v.x + R[1] * v.y + R[2] * v.z, R[3] * v.x + R[4] * v.y + R[5] * v.z, R[6] * v.x + R[7] * v.y + R[8] * v.z};
}
__device__ __forceinline__ Vec3 rotate_back(const DPose& P, Vec3 v) {
  if (P.identity) return v;
  const double* R = P.R;
  return {R[0] * v.x + R[3] * v.y + R[6] * v.z, R[1] * v.x + R[4] * v.y + R[7] * v.z, R[2] * v.x + R[5] * v.y + R[8] * v.z};
}
__device__ __forceinline__ Vec3 to_local(const DPose& P, Vec3 r) { return rotate(P, r - Vec3{P.T[0], P.T[1], P.T[2]}); }
__device__ __forceinline__ Vec3 to_lab(const DPose& P, Vec3 r) { return rotate_back(P, r) + Vec3{P.T[0], P.T[1], P.T[2]}; }

struct Ray {
  Vec3 r, d;
  double E, p;
};

// ------------------------------------------------------------------------------------------------------------
// Step 3: source.  Slot 0 -> position, slot 1 -> direction, slot 2 -> energy.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void sample_source(const DComponent& C, uint64_t seed, uint64_t i, Ray& ray) {
  const DSource& S = C.u.source;
  Vec3 r{0.0, 0.0, 0.0}, d;
  double ua, ub;
  if (S.pos_mode == MCX_POS_DISK) {
    draw2(seed, i, 0u, 0u, ua, ub);
    const double rad = S.radius * sqrt(ua);
    double s, c;
    sincospi(2.0 * ub, &s, &c);
    r = {rad * c, rad * s, 0.0};
  } else if (S.pos_mode == MCX_POS_GAUSS) {
    draw2(seed, i, 0u, 0u, ua, ub);
    double g0, g1;
    gauss_pair(ua, ub, g0, g1);
    r = {S.sigma_x * g0, S.sigma_y * g1, 0.0};
  }
  draw2(seed, i, 1u, 0u, ua, ub);
  Vec3 v;
  if (S.dir_mode == MCX_DIR_TARGET) {  // uniform in area on the target rectangle, no solid-angle weight
    v = Vec3{(ua - 0.5) * S.target_w, (ub - 0.5) * S.target_h, S.target_dist} - r;
  } else {  // Gaussian tangents, then normalise
    double g0, g1;
    gauss_pair(ua, ub, g0, g1);
    v = {S.div_x * g0, S.div_y * g1, 1.0};
  }
  d = (1.0 / sqrt(dot(v, v))) * v;
  double E = S.e0;
  if (S.e_mode == MCX_E_UNIFORM) {
    draw2(seed, i, 2u, 0u, ua, ub);
    E = S.e0 * (1.0 + S.de_rel * (2.0 * ua - 1.0));
  } else if (S.e_mode == MCX_E_SPECTRUM) {  // inverse CDF, weight stays 1
    draw2(seed, i, 2u, 0u, ua, ub);
    const double* __restrict__ cdf = S.cdf;
    const int n = S.spec_n;
    const double v01 = ua * cdf[n];
    // largest j in [0, n-1] with cdf[j] <= v01: bisection with the invariant cdf[lo] <= v01 < cdf[hi] (or hi = n),
    // started from the guide table's bracket where that bracket holds (it nearly always does: ~2 steps instead of 11)
    const int k = (int)(ua * (double)kSpecGuide);
    int lo = S.guide[k], hi = min(S.guide[k + 1] + 3, n);
    if (!(cdf[lo] <= v01)) lo = 0;
    if (hi < n && cdf[hi] <= v01) hi = n;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (cdf[mid] <= v01) lo = mid; else hi = mid;
    }
    const double c0 = cdf[lo], c1 = cdf[lo + 1];
    E = S.spec_emin + ((double)lo + (v01 - c0) / (c1 - c0)) * S.spec_bin_w;
  }
  ray.r = to_lab(C.pose, r);
  ray.d = rotate_back(C.pose, d);
  ray.E = E;
  ray.p = 1.0;
}

// Step 5: intersection with the plane z' = 0 of a component frame
__device__ __forceinline__ bool plane_hit(const DPose& P, const Ray& ray, Vec3& hit) {
  const Vec3 o = to_local(P, ray.r);
  const Vec3 d = rotate(P, ray.d);
  if (!(d.z > 0.0)) return false;
  const double t = -o.z / d.z;
  if (t < 0.0) return false;
  hit = o + t * d;
  return true;
}

// Step 14: bin index or -1
__device__ __forceinline__ long long detector_bin(const DComponent& C, const Ray& ray) {
  const DDetector& D = C.u.detector;
  Vec3 h;
  if (!plane_hit(C.pose, ray, h)) return -1;
  // (x - x_min) / (x_max - x_min) * nx with the quotient nx / (x_max - x_min) formed once at create: differs from the
  // oracle's order of operations by 2 ulp, i.e. only for a ray within 1e-15 of a bin edge
  const double fx = floor((h.x - D.xmin) * D.sx);
  const double fy = floor((h.y - D.ymin) * D.sy);
  // step 14b: an L_monitor bins lambda = hc / E [Angstrom]
  const double q = D.mode == MCX_DET_WAVELENGTH ? 12.398419843 / ray.E : ray.E;
  const double fe = floor((q - D.emin) * D.se);
  if (!(fx >= 0.0 && fx < (double)D.nx)) return -1;
  if (!(fy >= 0.0 && fy < (double)D.ny)) return -1;
  if (!(fe >= 0.0 && fe < (double)D.ne)) return -1;
  return ((long long)fy * D.nx + (long long)fx) * D.ne + (long long)fe;
}

// ------------------------------------------------------------------------------------------------------------
// Step 7: mu(E) by log-log interpolation.  lnE = log(E) is computed once per ray by the caller.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double mu_of(const DMaterial& M, double E, double lnE) {
  const int n = M.n;
  if (n == 0) return 0.0;
  const double* __restrict__ Eg = M.E;
  // segment j with Eg[j] <= E < Eg[j+1], clamped to [0, n-2]: guess from a uniform-in-lnE grid, then verify
  int j = (int)((lnE - M.lnE[0]) * M.inv_dlnE);
  j = max(0, min(j, n - 2));
  if (Eg[j] <= E && (j == n - 2 || E < Eg[j + 1])) {
    // guess was right
  } else if (Eg[j] > E) {
    if (j >= 2 && Eg[j - 1] <= E) {
      j = j - 1;
    } else if (j >= 1) {
      int lo = 0, hi = j;  // answer in [lo, hi): largest k with Eg[k] <= E, or 0
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (Eg[mid] <= E) lo = mid; else hi = mid;
      }
      j = lo;
    }
  } else {  // E >= Eg[j+1], j < n-2
    if (j + 2 <= n - 2 && E < Eg[j + 2]) {
      j = j + 1;
    } else {
      int lo = j + 1, hi = n - 1;  // largest k in [j+1, n-2] with Eg[k] <= E
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (Eg[mid] <= E) lo = mid; else hi = mid;
      }
      j = lo;
    }
  }
  return exp(M.lnMu[j] + (lnE - M.lnE[j]) * M.slope[j]);
}

// ------------------------------------------------------------------------------------------------------------
// Step 8: inside-interval of the ray parameter for the convex primitives, in the solid's own frame.
// ------------------------------------------------------------------------------------------------------------
// slab of one axis with 1/d supplied (one division per axis and solid instead of two; one more rounding per plane)
__device__ __forceinline__ bool clip_axis_inv(double o, double d, double inv, double lo, double hi, double& tmin, double& tmax) {
  if (d == 0.0) return o > lo && o < hi;
  const double ta = (lo - o) * inv, tb = (hi - o) * inv;
  tmin = fmax(tmin, fmin(ta, tb));
  tmax = fmin(tmax, fmax(ta, tb));
  return true;
}

__device__ __forceinline__ bool primitive_interval(const DSolid& S, Vec3 o, Vec3 d, double& tin, double& tout) {
  double tmin = -CUDART_INF, tmax = CUDART_INF;
  if (S.shape == MCX_BOX) {
    if (!clip_axis_inv(o.x, d.x, 1.0 / d.x, -S.dims[0], S.dims[0], tmin, tmax)) return false;
    if (!clip_axis_inv(o.y, d.y, 1.0 / d.y, -S.dims[1], S.dims[1], tmin, tmax)) return false;
    if (!clip_axis_inv(o.z, d.z, 1.0 / d.z, -S.dims[2], S.dims[2], tmin, tmax)) return false;
  } else if (S.shape == MCX_SPHERE) {
    const double b = dot(o, d);
    const double c = dot(o, o) - S.dims[0] * S.dims[0];
    const double disc = b * b - c;
    if (!(disc > 0.0)) return false;
    const double s = sqrt(disc);
    tmin = -b - s;
    tmax = -b + s;
  } else {  // finite cylinder, axis = local y
    const double a = d.x * d.x + d.z * d.z;
    const double c = o.x * o.x + o.z * o.z - S.dims[0] * S.dims[0];
    if (a == 0.0) {
      if (!(c < 0.0)) return false;
    } else {
      const double b = o.x * d.x + o.z * d.z;
      const double disc = b * b - a * c;
      if (!(disc > 0.0)) return false;
      const double s = sqrt(disc), inv_a = 1.0 / a;
      tmin = (-b - s) * inv_a;
      tmax = (-b + s) * inv_a;
    }
    if (!clip_axis_inv(o.y, d.y, 1.0 / d.y, -S.dims[1], S.dims[1], tmin, tmax)) return false;
  }
  if (!(tmin < tmax)) return false;
  tin = tmin;
  tout = tmax;
  return true;
}

// ------------------------------------------------------------------------------------------------------------
// Step 9: watertight ray/triangle test (Woop, Benthin, Wald 2013) in fp64.  The shear constants depend on the ray
// only.  Every product and difference of the edge functions is rounded separately (__dmul_rn/__dsub_rn are never
// contracted to FMA), so an edge shared by two triangles gives exactly negated values in both.
// ------------------------------------------------------------------------------------------------------------
struct Shear {
  int kx, ky, kz;
  double Sx, Sy, Sz;
  double ox, oy, oz;  // the ray origin's components kx, ky, kz
};

__device__ __forceinline__ double pick(Vec3 v, int k) { return k == 0 ? v.x : (k == 1 ? v.y : v.z); }

__device__ __forceinline__ Shear make_shear(Vec3 o, Vec3 d) {
  Shear s;
  s.kz = 0;
  double m = fabs(d.x);
  if (fabs(d.y) > m) { s.kz = 1; m = fabs(d.y); }
  if (fabs(d.z) > m) { s.kz = 2; }
  s.kx = s.kz == 2 ? 0 : s.kz + 1;
  s.ky = s.kx == 2 ? 0 : s.kx + 1;
  const double dz = pick(d, s.kz);
  if (dz < 0.0) { const int t = s.kx; s.kx = s.ky; s.ky = t; }
  // the same constants serve every triangle of the ray, which is all watertightness needs; as products with 1/d_kz
  // they are within an ulp of the quotients
  s.Sz = 1.0 / dz;
  s.Sx = pick(d, s.kx) * s.Sz;
  s.Sy = pick(d, s.ky) * s.Sz;
  s.ox = pick(o, s.kx); s.oy = pick(o, s.ky); s.oz = pick(o, s.kz);
  return s;
}

// returns 0 = miss, +1 = entering, -1 = exiting.  The vertex components are fetched in the ray's own axis order
// (kx, ky, kz), which saves permuting them in registers.
__device__ __forceinline__ int ray_triangle(const Shear& s, const double* __restrict__ tri, double& t_out) {
  const double Akx = tri[s.kx] - s.ox, Aky = tri[s.ky] - s.oy, Akz = tri[s.kz] - s.oz;
  const double Bkx = tri[3 + s.kx] - s.ox, Bky = tri[3 + s.ky] - s.oy, Bkz = tri[3 + s.kz] - s.oz;
  const double Ckx = tri[6 + s.kx] - s.ox, Cky = tri[6 + s.ky] - s.oy, Ckz = tri[6 + s.kz] - s.oz;
  const double Ax = __dsub_rn(Akx, __dmul_rn(s.Sx, Akz)), Ay = __dsub_rn(Aky, __dmul_rn(s.Sy, Akz));
  const double Bx = __dsub_rn(Bkx, __dmul_rn(s.Sx, Bkz)), By = __dsub_rn(Bky, __dmul_rn(s.Sy, Bkz));
  const double Cx = __dsub_rn(Ckx, __dmul_rn(s.Sx, Ckz)), Cy = __dsub_rn(Cky, __dmul_rn(s.Sy, Ckz));
  const double U = __dsub_rn(__dmul_rn(Cx, By), __dmul_rn(Cy, Bx));
  const double V = __dsub_rn(__dmul_rn(Ax, Cy), __dmul_rn(Ay, Cx));
  const double W = __dsub_rn(__dmul_rn(Bx, Ay), __dmul_rn(By, Ax));
  if ((U < 0.0 || V < 0.0 || W < 0.0) && (U > 0.0 || V > 0.0 || W > 0.0)) return 0;
  const double det = __dadd_rn(__dadd_rn(U, V), W);
  if (det == 0.0) return 0;
  const double Az = __dmul_rn(s.Sz, Akz), Bz = __dmul_rn(s.Sz, Bkz), Cz = __dmul_rn(s.Sz, Ckz);
  const double num = __dadd_rn(__dadd_rn(__dmul_rn(U, Az), __dmul_rn(V, Bz)), __dmul_rn(W, Cz));
  t_out = num / det;
  return det > 0.0 ? 1 : -1;
}

// ------------------------------------------------------------------------------------------------------------
// Steps 8-10 work on one list of interval END POINTS per ray and solids group, held in shared memory (element k of
// thread tid at [k * kBlock + tid]: conflict-free, dynamically indexable, no local memory): the parameter t and a tag
// byte = index of the solid in the group (device order = ascending precedence, DSolids) | 0x80 for an exit.
// ------------------------------------------------------------------------------------------------------------
struct Endpoints {
  double* t;
  unsigned char* tag;
  int cap;
};
constexpr unsigned char kTagExit = 0x80;
constexpr int kTriQueue = 16;  // candidate triangles per thread between two rounds of exact tests

__device__ __forceinline__ bool ep_push(const Endpoints& E, int& n, double t, unsigned tag) {
  if (n >= E.cap) return false;
  E.t[n * kBlock] = t;
  E.tag[n * kBlock] = (unsigned char)tag;
  ++n;
  return true;
}

// insertion sort of E[begin, end) by t; exits_last: among equal t an entry comes before an exit (step 9)
__device__ __forceinline__ void ep_sort(const Endpoints& E, int begin, int end, bool exits_last) {
  for (int a = begin + 1; a < end; ++a) {
    const double t = E.t[a * kBlock];
    const unsigned tag = E.tag[a * kBlock];
    int b = a - 1;
    while (b >= begin) {
      const double tb = E.t[b * kBlock];
      const unsigned tagb = E.tag[b * kBlock];
      if (!(tb > t || (exits_last && tb == t && (tagb & kTagExit) > (tag & kTagExit)))) break;
      E.t[(b + 1) * kBlock] = tb;
      E.tag[(b + 1) * kBlock] = (unsigned char)tagb;
      --b;
    }
    E.t[(b + 1) * kBlock] = t;
    E.tag[(b + 1) * kBlock] = (unsigned char)tag;
  }
}

// Step 9, second half, on the raw hits E[begin, ne) of one mesh: sort by t (enter before exit on ties), collapse
// consecutive same-orientation hits (shared-edge / vertex duplicates), check the enter / exit alternation, clip to t >= 0.
// Returns 1 = ok, 0 = degenerate sequence.
__device__ __forceinline__ int mesh_finish(const Endpoints& E, int begin, int& ne, unsigned solid) {
  if (ne == begin) return 1;
  ep_sort(E, begin, ne, true);
  // collapse consecutive same-orientation hits (shared-edge duplicates); what is left must alternate enter, exit, ...
  int m = begin;
  for (int a = begin; a < ne; ++a) {
    const unsigned tag = E.tag[a * kBlock];
    if (m == begin || E.tag[(m - 1) * kBlock] != tag) {
      E.t[m * kBlock] = E.t[a * kBlock];
      E.tag[m * kBlock] = (unsigned char)tag;
      ++m;
    }
  }
  if (((m - begin) & 1) || (E.tag[begin * kBlock] & kTagExit)) { ne = begin; return 0; }
  // clip the pairs to t >= 0 and drop the empty ones
  int w = begin;
  for (int a = begin; a < m; a += 2) {
    const double ta = fmax(E.t[a * kBlock], 0.0), tb = E.t[(a + 1) * kBlock];
    if (tb > ta) {
      E.t[w * kBlock] = ta; E.tag[w * kBlock] = (unsigned char)solid;
      E.t[(w + 1) * kBlock] = tb; E.tag[(w + 1) * kBlock] = (unsigned char)(solid | kTagExit);
      w += 2;
    }
  }
  ne = w;
  return 1;
}


// ------------------------------------------------------------------------------------------------------------
// Step 9 for one mesh and one WARP of rays: all crossings of every lane's full line with the mesh, appended to the lane's
// end-point list as sorted, duplicate-collapsed, paired end points clipped to t >= 0.  Must be called by all 32 lanes
// (`active` = this lane has a live ray).  Returns per lane 1 = ok, 0 = degenerate sequence, -1 = capacity overflow, or,
// for the whole warp, 2 = the beam walk met more nodes than its stack holds, nothing was appended: call again with
// coherent = false.
//
// The BVH (a complete binary tree in heap order, BvhNode) only yields CANDIDATE triangles; the exact fp64 watertight
// test of the lane's own ray decides, so a lane's hit set is what brute force gives it.  Two walks produce candidates:
//
//  beam walk (coherent warps: detector-tile order, where a warp's rays are aimed at one spot, far
//    closer together than a triangle is wide).  The warp walks ONE beam instead of 32 lines: the line of its first
//    participating lane (the leader), with every node box inflated by delta = the largest distance, per axis, of any
//    participating lane's line from the leader's at equal parameter inside the mesh's bounding sphere.  If lane l's
//    line meets a node box at parameter t, the leader's point at t lies within delta of that point, i.e. inside the
//    inflated box: the leader's line meets every inflated box whose original any lane's line meets, so the candidate set
//    is a superset of every lane's.  A step expands one pending node by up to five levels at once -- lane l tests
//    descendant l, 32 boxes of 32 bytes read as one coalesced kilobyte -- so a root-to-leaf path of c3's depth-17 tree
//    is 4 dependent loads instead of 17, and the node sectors are read once per warp instead of once per lane (c3 is
//    bound by L2 sector traffic and dependent-load latency, profiles/r02_README.md).  Hit descendants go on a stack
//    (inner nodes) or the candidate list (leaves), both warp-shared;
//
//  lane walk (any warp; also where the beam is too wide to pay, or its stack would overflow).  Every lane walks its
//    own line: at node i of `level`, already known to be hit, both children are tested at once (one 64-byte line); bit
//    `level` of `trail` says the right child was hit too and waits while the left subtree is walked; going back up
//    needs no memory (the ancestor of i at level m is ((i + 1) >> (level - m)) - 1).  Leaves go into the lane's queue.
//
// Both use the warp's triangle-queue words in shared memory (kTriQueue words per thread): the lane walk as per-lane
// queues, the beam walk as warp-shared lists.  The exact tests, the sort and the pairing exist once, behind both.
// ------------------------------------------------------------------------------------------------------------
constexpr int kBeamStack = 64, kBeamCand = 64;  // warp-shared words: rows 0-1 and rows 2-3 of the warp's triangle queues
static_assert(kBeamStack + kBeamCand <= 32 * kTriQueue, "the beam lists live in the warp's triangle-queue words");

__device__ __forceinline__ int mesh_endpoints_warp(const DSolid& S, unsigned solid, bool active, Vec3 o, Vec3 d, const Endpoints& E,
                                                   int& ne, unsigned* __restrict__ queue, bool coherent) {
  const unsigned full = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  unsigned* __restrict__ wq = queue - lane;  // word j of the warp's list space at wq[(j >> 5) * kBlock + (j & 31)]
#define MCX_WQ(j) wq[((j) >> 5) * kBlock + ((j) & 31)]
  // Does this lane's line pass the mesh at all?  Bounding sphere of the mesh box (DSolid::ctr, radius): the line's closest approach to the centre is at parameter tc.
  const Vec3 ctr{S.ctr[0], S.ctr[1], S.ctr[2]};
  const double rad = S.radius;
  const double tc = dot(ctr - o, d);
  bool part = false;
  if (active) {
    const Vec3 q = (o + tc * d) - ctr;
    part = dot(q, q) <= rad * rad;
  }
  const unsigned pmask = __ballot_sync(full, part);
  if (pmask == 0u) return 1;
  const int leader = __ffs(pmask) - 1;
  bool beam = coherent;
  float ex = 0.0f, ey = 0.0f, ez = 0.0f;
  if (beam) {
    // delta per axis: |p_l(t) - p_0(t)| is convex in t, so its maximum over the lane's stretch [tc - rad, tc + rad]
    // inside the sphere is at an end
    const Vec3 lo{__shfl_sync(full, o.x, leader), __shfl_sync(full, o.y, leader), __shfl_sync(full, o.z, leader)};
    const Vec3 ld{__shfl_sync(full, d.x, leader), __shfl_sync(full, d.y, leader), __shfl_sync(full, d.z, leader)};
    if (part) {
      const double ta = tc - rad, tb = tc + rad;
      const Vec3 a = (o + ta * d) - (lo + ta * ld), b = (o + tb * d) - (lo + tb * ld);
      ex = __double2float_ru(fmax(fabs(a.x), fabs(b.x)));
      ey = __double2float_ru(fmax(fabs(a.y), fabs(b.y)));
      ez = __double2float_ru(fmax(fabs(a.z), fabs(b.z)));
    }
    // non-negative floats order like their bit patterns
    ex = __uint_as_float(__reduce_max_sync(full, __float_as_uint(ex)));
    ey = __uint_as_float(__reduce_max_sync(full, __float_as_uint(ey)));
    ez = __uint_as_float(__reduce_max_sync(full, __float_as_uint(ez)));
    beam = fmaxf(fmaxf(ex, ey), ez) <= (float)S.bound2;  // (bound2 of a mesh = its beam limit)
    // the deviations were rounded up; 2^-20 of them more covers the roundings of the folded constants below
    ex *= 1.000001f; ey *= 1.000001f; ez *= 1.000001f;
  }
  if (!beam) ex = ey = ez = 0.0f;  // the lane walk tests the boxes as they are
  const Shear sh = make_shear(o, d);
  const int begin = ne, depth = S.depth, leaf_base = (1 << depth) - 1;
  const int k_first = depth - 5 * ((depth - 1) / 5);  // levels of the beam's first step, 1..5 (the others take 5)
  const float4* __restrict__ nodes = reinterpret_cast<const float4*>(S.nodes);
  const double* __restrict__ tris = S.tris;
  bool overflow = false;
  {
    // The line the boxes are tested against -- the leader's (beam walk) or the lane's own -- in fp32, re-origined just
    // before the mesh so that rounding errors scale with the mesh size, not with the distance to the source.
    const int src = beam ? leader : lane;
    const Vec3 so{__shfl_sync(full, o.x, src), __shfl_sync(full, o.y, src), __shfl_sync(full, o.z, src)};
    const Vec3 sd{__shfl_sync(full, d.x, src), __shfl_sync(full, d.y, src), __shfl_sync(full, d.z, src)};
    const Vec3 le = so + (__shfl_sync(full, tc, src) - rad) * sd;
    // 1/d in fp32, held to +-1e30 so that the products below stay finite (a line parallel to a pair of planes gets huge
    // parameters of the right signs instead of infinities)
    const float big = 1.0e30f;
    const float ix = sd.x != 0.0 ? fminf(fmaxf(1.0f / (float)sd.x, -big), big) : big;
    const float iy = sd.y != 0.0 ? fminf(fmaxf(1.0f / (float)sd.y, -big), big) : big;
    const float iz = sd.z != 0.0 ? fminf(fmaxf(1.0f / (float)sd.z, -big), big) : big;
    // (x -+ e - o) / d as one fused multiply-add per plane: x * (1/d) + (-o/d -+ e/d).  Its rounding error is below
    // 2^-21 of the mesh scale times |1/d| (1/d itself is within 2^-22 of the exact reciprocal), the boxes are padded by
    // 2^-16 of the scale (times |1/d| in t): the test stays conservative.
    const float bx = -(float)le.x * ix, by = -(float)le.y * iy, bz = -(float)le.z * iz;
    const float bxl = bx - ex * ix, bxh = bx + ex * ix, byl = by - ey * iy, byh = by + ey * iy, bzl = bz - ez * iz, bzh = bz + ez * iz;
    // beam walk state (warp-uniform)
    int sn = 0, cn = 0, node = 0;
    bool walking_w = depth > 0;
    if (beam && depth == 0) {  // a single triangle
      if (lane == 0) MCX_WQ(kBeamStack) = 0u;
      __syncwarp();
      cn = 1;
    }
    // lane walk state
    int i = 0, level = 0;
    unsigned trail = 0u;
    bool walking_l = part;
    for (;;) {
      int n_c = 0;  // candidates this lane tests in this round
      if (beam) {
        while (walking_w) {
          const int lv = 31 - __clz(node + 1), k = lv == 0 ? k_first : 5;
          const bool leaf_step = lv + k == depth;
          if (leaf_step && cn > kBeamCand - 32) break;  // make room in the candidate list first
          const int child = ((node + 1) << k) - 1 + lane;
          bool hit = false;
          if (lane < (1 << k)) {
            const float4 a = __ldg(nodes + 2 * (child + 1)), b = __ldg(nodes + 2 * (child + 1) + 1);
            const float x0 = fmaf(a.x, ix, bxl), x1 = fmaf(b.x, ix, bxh);
            const float y0 = fmaf(a.y, iy, byl), y1 = fmaf(b.y, iy, byh);
            const float z0 = fmaf(a.z, iz, bzl), z1 = fmaf(b.z, iz, bzh);
            const float n0 = fmaxf(fmaxf(fminf(x0, x1), fminf(y0, y1)), fminf(z0, z1));
            const float f0 = fminf(fminf(fmaxf(x0, x1), fmaxf(y0, y1)), fmaxf(z0, z1));
            hit = n0 <= f0 && __float_as_int(a.w) != 0;
          }
          const unsigned hits = __ballot_sync(full, hit);
          if (hits) {
            const int nh = __popc(hits), rank = __popc(hits & ((1u << lane) - 1u));
            if (leaf_step) {
              if (hit) MCX_WQ(kBeamStack + cn + rank) = (unsigned)(child - leaf_base);
              cn += nh;
            } else {
              if (sn + nh > kBeamStack) { ne = begin; return 2; }  // (warp-uniform)
              if (hit) MCX_WQ(sn + rank) = (unsigned)child;
              sn += nh;
            }
            __syncwarp();
          }
          if (sn == 0) { walking_w = false; break; }
          node = (int)MCX_WQ(sn - 1);
          --sn;
        }
        n_c = cn;
      } else {
        while (walking_l && n_c < kTriQueue) {
          if (level == depth) {  // a leaf whose box the line hits: queue its triangle
            queue[n_c * kBlock] = (unsigned)(i - leaf_base);
            ++n_c;
          } else {
            const float4* pair = nodes + 2 * (2 * i + 2);  // children 2i+1, 2i+2 sit in slots 2i+2, 2i+3
            const float4 a0 = __ldg(pair), b0 = __ldg(pair + 1), a1 = __ldg(pair + 2), b1 = __ldg(pair + 3);
            // slab tests of the full line against the padded fp32 boxes (no t range: the line is tested, as in step 9)
            // (bxl = bxh here: no inflation)
            const float x00 = fmaf(a0.x, ix, bxl), x01 = fmaf(b0.x, ix, bxh), x10 = fmaf(a1.x, ix, bxl), x11 = fmaf(b1.x, ix, bxh);
            const float y00 = fmaf(a0.y, iy, byl), y01 = fmaf(b0.y, iy, byh), y10 = fmaf(a1.y, iy, byl), y11 = fmaf(b1.y, iy, byh);
            const float z00 = fmaf(a0.z, iz, bzl), z01 = fmaf(b0.z, iz, bzh), z10 = fmaf(a1.z, iz, bzl), z11 = fmaf(b1.z, iz, bzh);
            const float n0 = fmaxf(fmaxf(fminf(x00, x01), fminf(y00, y01)), fminf(z00, z01));
            const float f0 = fminf(fminf(fmaxf(x00, x01), fmaxf(y00, y01)), fmaxf(z00, z01));
            const float n1 = fmaxf(fmaxf(fminf(x10, x11), fminf(y10, y11)), fminf(z10, z11));
            const float f1 = fminf(fminf(fmaxf(x10, x11), fmaxf(y10, y11)), fmaxf(z10, z11));
            const bool hit0 = n0 <= f0 && __float_as_int(a0.w) != 0, hit1 = n1 <= f1 && __float_as_int(a1.w) != 0;
            if (hit0) {
              if (hit1) trail |= 1u << level;
              i = 2 * i + 1;
              ++level;
              continue;
            }
            if (hit1) {
              i = 2 * i + 2;
              ++level;
              continue;
            }
          }
          // to the deepest right sibling still to be visited, or done
          if (trail == 0u) { walking_l = false; break; }
          const int l = 31 - __clz(trail);
          trail ^= 1u << l;
          i = ((i + 1) >> (level - (l + 1)));  // = (left child at level l + 1) + 1 = its right sibling
          level = l + 1;
        }
      }
      // the exact test of the lane's own ray on the candidates (beam walk: the warp's list, uniform loads)
      for (int k = 0; k < n_c; ++k) {
        const unsigned leaf = beam ? MCX_WQ(kBeamStack + k) : queue[k * kBlock];
        if (part) {
          double t;
          const int r = ray_triangle(sh, tris + 9 * (size_t)leaf, t);
          if (r != 0 && !ep_push(E, ne, t, solid | (r < 0 ? kTagExit : 0u))) overflow = true;
        }
      }
      if (beam) {
        __syncwarp();
        cn = 0;
        if (!walking_w) break;
      } else if (!walking_l) {
        break;
      }
    }
  }
#undef MCX_WQ
  __syncwarp();
  if (overflow) return -1;
  if (!part) return 1;
  return mesh_finish(E, begin, ne, solid);
}

// Steps 8-10 for one solids group.  Returns 1 = continue, 0 = degenerate, -1 = capacity overflow.
// With meshes (MESH) the function must be called by all 32 lanes of the warp, `active` saying which have a live ray;
// `coherent` = the warp's rays are neighbours (detector-tile order), so the beam walk of the meshes is tried first.
// PRIM = some group of the instrument holds a box, cylinder or sphere.
template <bool MESH, bool PRIM>
__device__ __forceinline__ int trace_solids(const SInst& I, const DComponent& C, Ray& ray, const Endpoints& E,
                                            unsigned* __restrict__ queue, bool active, bool coherent) {
  const DSolids& G = C.u.solids;
  int ne = 0, status = 1;
  for (int s = 0; s < G.n_solids; ++s) {
    const DSolid& S = G.solids[s];
    if (MESH && S.shape == MCX_MESH) {  // warp-uniform branch
      const bool act = active && status == 1;
      int rc;
      for (bool coh = coherent;; coh = false) {  // (a second round only if the beam walk gives up: rc 2, warp-uniform)
        Vec3 o{0.0, 0.0, 0.0}, d{0.0, 0.0, 1.0};
        if (act) { o = to_local(S.pose, ray.r); d = rotate(S.pose, ray.d); }
        rc = mesh_endpoints_warp(S, (unsigned)s, act, o, d, E, ne, queue, coh);
        if (rc != 2) break;
      }
      if (act && rc != 1) status = rc;
      continue;
    }
    if (!PRIM || !(active && status == 1)) continue;
    if (!MESH) {  // (the mesh kernels run at the register limit and do without)
      // the line misses the solid's bounding sphere, by more than the rounding of this test (1e-9 of the radius^2 in
      // bound2, 1e-14 of the squared distance for the cancellation): no interval, no need for the solid's frame
      const Vec3 oc = Vec3{S.pose.T[0], S.pose.T[1], S.pose.T[2]} - ray.r;
      const double along = dot(oc, ray.d), oc2 = dot(oc, oc);
      if (oc2 - along * along > S.bound2 + 1e-14 * oc2) continue;
    }
    const Vec3 o = to_local(S.pose, ray.r);
    const Vec3 d = rotate(S.pose, ray.d);
    double a, b;
    if (primitive_interval(S, o, d, a, b)) {  // clip to t >= 0, drop if empty
      a = fmax(a, 0.0);
      if (b > a) {
        if (!ep_push(E, ne, a, (unsigned)s)) status = -1;
        if (!ep_push(E, ne, b, (unsigned)s | kTagExit)) status = -1;
      }
    }
  }
  if (!active || status != 1) return status;
  if (ne == 0) return 1;
  // Step 10.  Between two consecutive end points the set of solids the ray is inside of is constant, so sweeping the
  // sorted end points with that set as a bit mask classifies every elementary segment exactly as its midpoint would;
  // the owner is the solid of highest precedence in the set = the highest bit (DSolids).  Equal end points only
  // make zero-length segments, whatever their order.
  ep_sort(E, 0, ne, false);
  const double lnE = log(ray.E);
  double tau = 0.0, t_prev = 0.0, last_mu = 0.0;
  int last_mat = -1;
  unsigned inside = 0u;
  for (int k = 0; k < ne; ++k) {
    const double t = E.t[k * kBlock];
    const unsigned tag = E.tag[k * kBlock];
    if (inside != 0u && t > t_prev) {
      const int mat = G.solids[31 - __clz(inside)].material;
      if (mat != last_mat) { last_mu = mu_of(I.mats[mat], ray.E, lnE); last_mat = mat; }
      tau += last_mu * (t - t_prev);
    }
    t_prev = t;
    const unsigned bit = 1u << (tag & 31u);
    inside = (tag & kTagExit) ? (inside & ~bit) : (inside | bit);
  }
  ray.p *= exp(-tau);
  return 1;
}

// ------------------------------------------------------------------------------------------------------------
// Step 17: scattering in samples (a step updates the ray's weight "and direction").  Elastic, Thomson
// angular distribution: cos(theta) is the real root of x^3 + 3x = 8u - 4 (inverse of F(x) = 1/2 + (3/8)(x + x^3/3)),
// x = w - 1/w with w = cbrt(q + sqrt(q^2 + 1)), q = 4u - 2; azimuth 2 pi u'.  New direction = cos(theta) d +
// sin(theta)(cos(phi) e1 + sin(phi) e2), e1 = (d x a)/|d x a| with a the coordinate axis along which |d| is smallest
// (ties: the lowest axis), e2 = d x e1; normalised once more.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ Vec3 cross(Vec3 a, Vec3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }

__device__ __noinline__ Vec3 scatter_direction(Vec3 d, double u_mu, double u_phi) {
  const double q = 4.0 * u_mu - 2.0;
  const double w = cbrt(q + sqrt(q * q + 1.0));
  const double ct = w - 1.0 / w;
  const double st = sqrt(fmax(0.0, 1.0 - ct * ct));
  double sp, cp;
  sincos(2.0 * CUDART_PI * u_phi, &sp, &cp);
  Vec3 a{1.0, 0.0, 0.0};
  double m = fabs(d.x);
  if (fabs(d.y) < m) { a = {0.0, 1.0, 0.0}; m = fabs(d.y); }
  if (fabs(d.z) < m) { a = {0.0, 0.0, 1.0}; }
  Vec3 e1 = cross(d, a);
  e1 = (1.0 / sqrt(dot(e1, e1))) * e1;
  const Vec3 e2 = cross(d, e1);
  const Vec3 v = ct * d + st * (cp * e1 + sp * e2);
  return (1.0 / sqrt(dot(v, v))) * v;
}

// the scattering part of mu(E): same grid, same interpolation (step 7); 0 for a material without the table
__device__ __forceinline__ double mu_s_of(const DMaterial& M, double E, double lnE) {
  if (M.lnMuS == nullptr) return 0.0;
  DMaterial S = M;
  S.lnMu = M.lnMuS;
  S.slope = M.slopeS;
  return mu_of(S, E, lnE);
}

// Step 17 state of one ray inside one sample
struct Scat {
  double tau_s;    // scattering optical depth at which the next event lies (leg k < K)
  double cum;      // running sum of mu_s * length on this leg
  double s_pre;    // sum of mu_s * length over everything walked while events were left: tau = sum mu L - s_pre
  double t_event;  // parameter of the event on this leg
  int k, K;        // events so far, events allowed
  unsigned have_ms;  // (voxels) bit m: the ray's mu_s of material m is in shared memory
  bool event;
};

// Steps 8-10 (and 17 where the group scatters) for one solids group.  Returns 1 = continue, 0 = degenerate, -1 = capacity
// overflow.  Must be called by all 32 lanes of the warp, `active` saying which have a live ray (the mesh walk is
// warp-cooperative, and the legs of step 17 are walked by the warp together); `coherent` = the warp's rays are neighbours
// (detector-tile order), so the beam walk of the meshes is tried first.  PRIM = some group of the instrument holds a box,
// cylinder or sphere.  SCAT: a ray walks leg after leg, each from its last scattering event, while events are left.
template <bool MESH, bool PRIM, bool SCAT>
__device__ __forceinline__ int trace_solids_legs(const SInst& I, const DComponent& C, int comp, Ray& ray, uint64_t seed, uint64_t ray_index,
                                            const Endpoints& E, unsigned* __restrict__ queue, bool active, bool coherent) {
  const DSolids& G = C.u.solids;
  int status = 1;
  double tau = 0.0, lnE = 0.0;
  Scat S;
  S.k = 0; S.K = SCAT ? G.scatter_order : 0; S.cum = 0.0; S.tau_s = 0.0; S.s_pre = 0.0; S.t_event = 0.0; S.have_ms = 0u; S.event = false;
  bool more = active;  // this lane has a leg to walk
  for (int leg = 0;; ++leg) {
    if (SCAT && leg > 0 && !__any_sync(0xffffffffu, more)) break;
    const bool walk = more && status == 1;
    int ne = 0;
    for (int s = 0; s < G.n_solids; ++s) {
      const DSolid& Sd = G.solids[s];
      if (MESH && Sd.shape == MCX_MESH) {  // warp-uniform branch
        const bool act = walk && status == 1;
        int rc;
        for (bool coh = coherent && leg == 0;; coh = false) {  // (a second round only if the beam walk gives up: rc 2, warp-uniform)
          Vec3 o{0.0, 0.0, 0.0}, d{0.0, 0.0, 1.0};
          if (act) { o = to_local(Sd.pose, ray.r); d = rotate(Sd.pose, ray.d); }
          rc = mesh_endpoints_warp(Sd, (unsigned)s, act, o, d, E, ne, queue, coh);
          if (rc != 2) break;
        }
        if (act && rc != 1) status = rc;
        continue;
      }
      if (!PRIM || !(walk && status == 1)) continue;
      if (!MESH) {  // (the mesh kernels run at the register limit and do without)
        // the line misses the solid's bounding sphere, by more than the rounding of this test (1e-9 of the radius^2 in
        // bound2, 1e-14 of the squared distance for the cancellation): no interval, no need for the solid's frame
        const Vec3 oc = Vec3{Sd.pose.T[0], Sd.pose.T[1], Sd.pose.T[2]} - ray.r;
        const double along = dot(oc, ray.d), oc2 = dot(oc, oc);
        if (oc2 - along * along > Sd.bound2 + 1e-14 * oc2) continue;
      }
      const Vec3 o = to_local(Sd.pose, ray.r);
      const Vec3 d = rotate(Sd.pose, ray.d);
      double a, b;
      if (primitive_interval(Sd, o, d, a, b)) {  // clip to t >= 0, drop if empty
        a = fmax(a, 0.0);
        if (b > a) {
          if (!ep_push(E, ne, a, (unsigned)s)) status = -1;
          if (!ep_push(E, ne, b, (unsigned)s | kTagExit)) status = -1;
        }
      }
    }
    more = false;
    if (walk && status == 1 && ne > 0) {
      // Step 10.  Between two consecutive end points the set of solids the ray is inside of is constant, so sweeping the
      // sorted end points with that set as a bit mask classifies every elementary segment exactly as its midpoint would;
      // the owner is the solid of highest precedence in the set = the highest bit (DSolids).  Equal end points only
      // make zero-length segments, whatever their order.
      ep_sort(E, 0, ne, false);
      if (leg == 0) lnE = log(ray.E);
      double u_mu = 0.0;
      if (SCAT && S.k < S.K) {  // step 17: where on this leg the next event lies, in scattering optical depth
        double u_f;
        draw2(seed, ray_index, (uint32_t)(2 * S.k), (uint32_t)comp, u_f, u_mu);
        S.tau_s = -log(u_f);
        S.cum = 0.0;
      }
      double t_prev = 0.0, last_mu = 0.0, last_ms = 0.0;
      int last_mat = -1;
      unsigned inside = 0u;
      for (int k = 0; k < ne; ++k) {
        const double t = E.t[k * kBlock];
        const unsigned tag = E.tag[k * kBlock];
        if (inside != 0u && t > t_prev) {
          const int mat = G.solids[31 - __clz(inside)].material;
          if (mat != last_mat) {
            last_mu = mu_of(I.mats[mat], ray.E, lnE);
            if (SCAT) last_ms = mu_s_of(I.mats[mat], ray.E, lnE);
            last_mat = mat;
          }
          const double len = t - t_prev;
          if (SCAT && S.k < S.K) {
            if (last_ms > 0.0 && S.cum + last_ms * len >= S.tau_s) {
              const double l = (S.tau_s - S.cum) / last_ms;
              tau += (last_mu - last_ms) * l;
              double u_phi, unused;
              draw2(seed, ray_index, (uint32_t)(2 * S.k + 1), (uint32_t)comp, u_phi, unused);
              ray.r = ray.r + (t_prev + l) * ray.d;
              ray.d = scatter_direction(ray.d, u_mu, u_phi);
              ++S.k;
              more = true;  // walk the next leg from here
              break;
            }
            S.cum += last_ms * len;
            tau += (last_mu - last_ms) * len;
          } else {
            tau += last_mu * len;
          }
        }
        t_prev = t;
        const unsigned bit = 1u << (tag & 31u);
        inside = (tag & kTagExit) ? (inside & ~bit) : (inside | bit);
      }
    }
    if (!SCAT) break;
  }
  if (!active || status != 1) return status;
  ray.p *= exp(-tau);
  return 1;
}

// ------------------------------------------------------------------------------------------------------------
// Step 11: exact traversal of the voxel grid (Amanatides & Woo 1987).  tau = sum over the voxels crossed of
// mu[id] * length; PAPER.md:186-188 names this loop ("steps reach into the thousands") as where the EDXCT time goes.
//
// The volume sits in the workspace in traversal layout with a one-voxel guard border of kVoxelGuard on every side
// (DVoxels), so the walk needs no bounds arithmetic: a step adds a constant to the voxel address, and stepping onto a
// guard cell ends the walk.
//
// The walk is organised by slabs of the ray's own dominant axis w (|d_w| >= |d_u|, |d_v|; in c4 w is the beam axis =
// the axis stored fastest, and 512 of the ~553 faces a ray crosses are w faces).  Per slab the ray crosses one w face
// and at most one face of each lateral axis, because the lateral coordinate, in voxels, advances by a = |d_u / d_w|
// <= 1 per slab.  That coordinate is carried as a 64-bit binary fraction: "does the ray cross a u face in this slab"
// is the carry of one 64-bit integer add, exact (no rounding accumulates over the slabs; the only rounding is that of
// a itself and of the starting fraction, ~1e-13 voxel, which can reorder two crossings closer than that, i.e. move a
// zero-length visit).  A slab therefore costs two add-with-carry pairs, two byte loads (the voxel after the lateral
// step, if any, and the voxel after the w face) and two compares, all on the integer pipe and free of branches as
// long as the material does not change; no face parameter is tracked.
//
// Attenuation.  Face parameters are needed only where a RUN of equal IDs ends.  There t is computed from the integer
// index of the face, (face - o) / d, the formula of step 11 itself, and the run's length is added to the path length
// of its material (len_s, shared memory, element m at len_s[m * kBlock]).  tau = sum_m mu_m(E) * len_m is formed at
// the end over the materials the ray touched, so mu(E) (a table search and an exp each, step 7) is evaluated only for
// those -- a ray of c4 meets 3-6 of the 16.  Same real number as summing mu[id] * length voxel by voxel; only the
// rounding order differs.
// ------------------------------------------------------------------------------------------------------------
// 64-bit x += a, returns the carry (0 or 1)
__device__ __forceinline__ unsigned add_carry(unsigned& lo, unsigned& hi, unsigned alo, unsigned ahi) {
  unsigned c;
  asm("add.cc.u32 %0, %0, %3;\n\taddc.cc.u32 %1, %1, %4;\n\taddc.u32 %2, 0, 0;" : "+r"(lo), "+r"(hi), "=r"(c) : "r"(alo), "r"(ahi));
  return c;
}

// one voxel ID through the read-only path, zero-extended into a 32-bit register
__device__ __forceinline__ unsigned ld_voxel(unsigned long long addr) {
  unsigned v;
  asm("ld.global.nc.u8 %0, [%1];" : "=r"(v) : "l"(addr));
  return v;
}

// one cell {ID, run, radius, 0} of the voxel volume as ID | run << 8 | radius << 16
__device__ __forceinline__ unsigned ld_cell(unsigned long long addr) {
  unsigned v;
  asm("ld.global.nc.u32 %0, [%1];" : "=r"(v) : "l"(addr));
  return v;
}

// n / d for any 32-bit n by multiplication (Granlund & Montgomery 1994): m, sh precomputed by mcx_instrument_create
__device__ __forceinline__ unsigned fast_div(unsigned n, unsigned m, unsigned sh) {
  const unsigned t = __umulhi(m, n);
  return (t + ((n - t) >> 1)) >> sh;
}

// x in [0, 1) -> floor(x 2^64); exact (x 2^64 has at most 53 significant bits)
__device__ __forceinline__ unsigned long long frac64(double x) { return __double2ull_rz(x * 18446744073709551616.0); }

// Per-ray values the walk needs only where a run of equal IDs ends live in shared memory, not in registers
// (cold_s, element k at cold_s[k * kBlock]): o and 1/d of the axes w, u, v, and the exit parameter t1.
enum { VC_O = 0, VC_INVD = 1, VC_T1 = 6, VC_WFACE = 7, VC_COUNT = 8 };

// One axis of the walk at set-up time
struct VoxAxis {
  double o, d;      // ray origin and direction component in the volume frame
  double inv_d;     // 1 / d (the walk's set-up divides once per axis and multiplies from there on)
  int idx;          // entry voxel index
  int dir;          // +1, -1, 0
  unsigned slot;    // 0, 1, 2: position of this axis in the traversal layout (fast, a1, a2)
  unsigned stride;  // address step (bytes) per voxel along this axis
};

__device__ __forceinline__ VoxAxis vox_axis(const DVoxels& V, Vec3 o, Vec3 d, Vec3 inv_d, int g, double t0, unsigned cell_bytes) {
  VoxAxis A;
  A.o = pick(o, g);
  A.d = pick(d, g);
  A.inv_d = pick(inv_d, g);
  const int n = V.n[g];
  A.idx = min(n - 1, max(0, (int)floor((A.o + t0 * A.d) * V.inv_h)));
  A.dir = A.d > 0.0 ? 1 : (A.d < 0.0 ? -1 : 0);
  A.slot = g == V.fast ? 0u : (g == V.a1 ? 1u : 2u);
  A.stride = cell_bytes * (A.slot == 0u ? 1u : (A.slot == 1u ? (unsigned)V.pitch : V.slab));  // bytes
  return A;
}

// Lateral coordinate at the first w face ahead (parameter t_w0), in voxels from the entry voxel's near face in the
// direction of travel: in [0, 2); >= 1 means the lateral face is crossed within the first (partial) slab (c0 = 1).
// f = its fraction, a = |d / d_w| <= 1 = advance per slab, both as 64-bit binary fractions.
__device__ __forceinline__ void lateral_init(const VoxAxis& A, double inv_dw, double t_w0, double inv_h, unsigned long long& f,
                                             unsigned long long& a, unsigned& c0) {
  double pos = 0.0, adv = 0.0;
  if (A.dir != 0) {
    const double y = (A.o + t_w0 * A.d) * inv_h;
    pos = A.dir > 0 ? y - (double)A.idx : (double)(A.idx + 1) - y;
    pos = fmin(fmax(pos, 0.0), 1.9999999999999998);
    adv = fabs(A.d * inv_dw);
  }
  c0 = pos >= 1.0 ? 1u : 0u;
  f = frac64(pos - (double)c0);
  a = adv >= 1.0 ? 0xFFFFFFFFFFFFFFFFull : frac64(adv);
}

// The walk of one ray through the volume, leg by leg: a leg is the half-line ol + t dl, t >= 0, in the volume's frame,
// from where it enters the grid to where it leaves it or (SCAT, step 17) to the scattering event.  setup() starts a leg,
// step() does one slab and a skip and says when the leg is over.  Path lengths go to len_s / touched, which accumulate
// over the legs.  (Everything is inlined; the members live in registers.)
// CELL = bytes per cell: kVoxelCellBytes, or 1 = the compact cells of a scattering volume (DVoxels::cmap; walk stage only:
// setup / probe / settle / advance).
#define MCX_VOXEL_AT(lo32) id_at(lo32)
constexpr unsigned kCompactGuard = 16u;  // what id_of_compact makes of a guard cell
// compact cell -> ID (0..15), guard (0xF0) -> 16
__device__ __forceinline__ unsigned id_of_compact(unsigned v) { return (v & 15u) | (((v + 16u) >> 4) & 16u); }
// radius code -> radius: 0..6, 8, 10, 12, 16, 24, 32, 64, 128 (code 15 = guard: unused)
__device__ __forceinline__ unsigned radius_of_code(unsigned c) {
  return (unsigned)((c < 8u ? 0x0806050403020100ull : 0x0080402018100c0aull) >> (8u * (c & 7u))) & 0xffu;
}
template <bool SCAT, int CELL = kVoxelCellBytes>
struct VoxWalk {
  const SInst& I;
  const DVoxels& V;
  double E, lnE;
  double* len_s;
  double* cold_s;
  double* mus_s;
  unsigned& touched;
  Scat& S;
  unsigned ful, fuh, fvl, fvh, aul, auh, avl, avh, so_u, so_v, so_w, meta, inv_u, inv_v;
  unsigned cur, w_crossed, cu, cv, lo;
  unsigned long long base, hi;
  double t_run;
  static constexpr unsigned kGuard = CELL == 1 ? kCompactGuard : kVoxelGuard;
  __device__ __forceinline__ unsigned id_at(unsigned lo32) const {
    const unsigned v = ld_voxel(hi | lo32);
    return CELL == 1 ? id_of_compact(v) : v;
  }

  // false: the half-line misses the grid
  __device__ __forceinline__ bool setup(Vec3 ol, Vec3 dl) {
    const double h = V.h;
    unsigned cu0, cv0, lo_start;
    S.event = false;
    const Vec3 inv_d{1.0 / dl.x, 1.0 / dl.y, 1.0 / dl.z};  // the only divisions of the set-up (+-inf where d = 0: unused)
    double t0 = -CUDART_INF, t1 = CUDART_INF;
    auto clip = [&](double o, double d, double inv, double top) {  // slab [0, top] of one axis, as clip_axis
      if (d == 0.0) return o > 0.0 && o < top;
      const double ta = -o * inv, tb = (top - o) * inv;
      t0 = fmax(t0, fmin(ta, tb));
      t1 = fmin(t1, fmax(ta, tb));
      return true;
    };
    if (!clip(ol.x, dl.x, inv_d.x, (double)V.n[0] * h)) return false;
    if (!clip(ol.y, dl.y, inv_d.y, (double)V.n[1] * h)) return false;
    if (!clip(ol.z, dl.z, inv_d.z, (double)V.n[2] * h)) return false;
    if (t0 < 0.0) t0 = 0.0;
    if (!(t0 < t1)) return false;
    // the ray's dominant axis w and the two lateral axes u < v
    int gw = 0;
    {
      double m = fabs(dl.x);
      if (fabs(dl.y) > m) { gw = 1; m = fabs(dl.y); }
      if (fabs(dl.z) > m) gw = 2;
    }
    const int gu = gw == 0 ? 1 : 0, gv = gw == 2 ? 1 : 2;
    const VoxAxis W = vox_axis(V, ol, dl, inv_d, gw, t0, CELL), U = vox_axis(V, ol, dl, inv_d, gu, t0, CELL), X = vox_axis(V, ol, dl, inv_d, gv, t0, CELL);
    const double t_w0 = ((double)(W.idx + (W.dir > 0 ? 1 : 0)) * h - W.o) * W.inv_d;  // first w face ahead
    unsigned long long fu, au, fv, av;
    lateral_init(U, W.inv_d, t_w0, V.inv_h, fu, au, cu0);
    lateral_init(X, W.inv_d, t_w0, V.inv_h, fv, av, cv0);
    ful = (unsigned)fu; fuh = (unsigned)(fu >> 32); aul = (unsigned)au; auh = (unsigned)(au >> 32);
    fvl = (unsigned)fv; fvh = (unsigned)(fv >> 32); avl = (unsigned)av; avh = (unsigned)(av >> 32);
    so_w = (unsigned)W.dir * W.stride; so_u = (unsigned)U.dir * U.stride; so_v = (unsigned)X.dir * X.stride;
    // axis k (0 = w, 1 = u, 2 = v): layout slot in bits 2k, 2k+1; "travels in the + direction" in bit 6 + k
    meta = W.slot | (U.slot << 2) | (X.slot << 4) | (W.dir > 0 ? 64u : 0u) | (U.dir > 0 ? 128u : 0u) | (X.dir > 0 ? 256u : 0u);
    cold_s[(VC_O + 0) * kBlock] = W.o; cold_s[(VC_INVD + 0) * kBlock] = W.inv_d;
    cold_s[(VC_O + 2) * kBlock] = U.o; cold_s[(VC_INVD + 2) * kBlock] = U.inv_d;
    cold_s[(VC_O + 4) * kBlock] = X.o; cold_s[(VC_INVD + 4) * kBlock] = X.inv_d;
    cold_s[VC_T1 * kBlock] = t1;
    // index of the first w face ahead and the walk's direction along w, as one 8-byte slot
    cold_s[VC_WFACE * kBlock] = __hiloint2double(W.dir, W.idx + (W.dir > 0 ? 1 : 0));
    {  // skipping (see the loop below): only along the fast axis in the direction the runs were counted in
      const bool can_skip = CELL == kVoxelCellBytes && W.slot == 0u && W.dir == V.run_dir;  // (compact cells carry no runs)
      // inv <= 2^32 / (a_hi + 1): float quotient less a relative 1e-6 (its own error is 2^-22)
      inv_u = can_skip ? __float2uint_rz(__fdividef(4294967296.0f, (float)auh + 1.0f) * 0.999999f) : 0u;
      inv_v = can_skip ? __float2uint_rz(__fdividef(4294967296.0f, (float)avh + 1.0f) * 0.999999f) : 0u;
    }
    lo_start = (unsigned)(W.idx + 1) * W.stride + (unsigned)(U.idx + 1) * U.stride + (unsigned)(X.idx + 1) * X.stride;
    t_run = t0;
    // The volume does not straddle a 4 GiB address boundary (mcx_instrument_create places it so): the walk keeps the
    // low address word only and a step is one 32-bit add.
    base = (unsigned long long)(CELL == 1 ? V.cmap : V.ids);
    hi = base & 0xFFFFFFFF00000000ull;
    lo_start += (unsigned)base;
    cur = MCX_VOXEL_AT(lo_start);
    w_crossed = 0u;
    cu = cu0; cv = cv0; lo = lo_start;
    return true;
  }
  // (touched: bit m = len_s[m] holds this ray's path length in material m)
  // The run of `cur` ends where the ray enters the voxel at address `at` through a face of axis k: the index of that
  // voxel along the axis comes back out of the address (a guard cell gives -1 or n, i.e. the outer face of the grid),
  // and the face parameter is (face - o) / d as in step 11 (as a product with 1/d, one more rounding).
  // (For w faces, most of them, the index is simply counted: w_crossed faces lie behind the current slab.)
  __device__ __forceinline__ bool close_run(unsigned at, unsigned k, unsigned id) {
    const double h = V.h;
    int face;
    if (k == 0u) {
      const double wf = cold_s[VC_WFACE * kBlock];
      face = __double2loint(wf) + __double2hiint(wf) * (int)w_crossed;
    } else {
      const unsigned off = (at - (unsigned)base) / (unsigned)CELL;  // cell index
      const unsigned q2 = fast_div(off, V.mg_slab, V.sh_slab), r = off - q2 * V.slab;
      const unsigned q1 = fast_div(r, V.mg_pitch, V.sh_pitch), q0 = r - q1 * (unsigned)V.pitch;
      const unsigned slot = (meta >> (2u * k)) & 3u;
      face = (int)(slot == 0u ? q0 : (slot == 1u ? q1 : q2)) - (int)((meta >> (6u + k)) & 1u);  // index - 1 + (dir > 0 ? 0 : 1)
    }
    const double tf = ((double)face * h - cold_s[(VC_O + 2 * k) * kBlock]) * cold_s[(VC_INVD + 2 * k) * kBlock];
    const double tn = fmin(tf, cold_s[VC_T1 * kBlock]);
    double len = tn - t_run;
    bool ev = false;
    if (SCAT && S.k < S.K) {  // step 17: does the event fall inside this run?
      const DMaterial& M = I.mats[cur];
      double ms = 0.0;
      if (M.lnMuS != nullptr) {
        if (!((S.have_ms >> cur) & 1u)) { mus_s[cur * kBlock] = mu_s_of(M, E, lnE); S.have_ms |= 1u << cur; }
        ms = mus_s[cur * kBlock];
      }
      if (ms > 0.0 && S.cum + ms * len >= S.tau_s) {
        len = (S.tau_s - S.cum) / ms;
        S.t_event = t_run + len;
        ev = true;
      } else {
        S.cum += ms * len;
      }
    }
    const double prev = (touched >> cur) & 1u ? len_s[cur * kBlock] : 0.0;
    len_s[cur * kBlock] = prev + len;
    touched |= 1u << cur;
    t_run = tn;
    cur = id;
    return ev;
  }
  // One iteration = one slab, then a skip.
  //  Slab: the lateral step (if any; the same cell again if cu = cv = 0) and the w face that ends the slab: cell b at
  //  lo_b, then cell c at lo_c.  If both lateral faces are crossed in one slab (rare) lo_b is the diagonal neighbour
  //  and the slow path visits the cell in between first.
  //  Skip: standing in cell c (same ID as the run), the ray may cross s more w faces without looking at anything if
  //  the next s cells of the row hold the same ID (the cell's run) and no lateral face comes in those s slabs, i.e.
  //  s additions of a leave the fraction below 1: s <= (2^64 - 1 - f) / a, taken conservatively from the high words
  //  as mulhi(~f_hi, inv) with inv <= 2^32 / (a_hi + 1).  Then f += s a exactly and the address moves s cells on.
  //  inv = 0 (no skipping) unless the ray runs along the fast axis in the direction the runs were counted in.
  __device__ __forceinline__ bool settle_slab(unsigned cuA, unsigned cvA, unsigned lo_bA, unsigned lo_cA, unsigned idbA, unsigned idcA) {
    unsigned k_lat = cuA ? 1u : 2u, k_first = 0u, lo_a = 0u, ida = cur;
    if (cuA & cvA) {
      // The face crossed first is the one with more of the slab left after it: f / a, f the fraction after this
      // slab's add (ties: u).  Compared as f_u a_v >= f_v a_u on the high 64 bits of the products.
      const unsigned long long au = ((unsigned long long)auh << 32) | aul, av = ((unsigned long long)avh << 32) | avl;
      const unsigned long long fu = ((unsigned long long)fuh << 32) | ful, fv = ((unsigned long long)fvh << 32) | fvl;
      const bool u_first = __umul64hi(fu, av) >= __umul64hi(fv, au);
      k_first = u_first ? 1u : 2u;
      k_lat = u_first ? 2u : 1u;
      lo_a = lo_bA - (u_first ? so_v : so_u);
      ida = MCX_VOXEL_AT(lo_a);
    }
    if (ida != cur) {  // the cell in between the two lateral faces of a double step
      if (close_run(lo_a, k_first, ida)) { S.event = true; return true; }
      if (ida == kVoxelGuard) return true;
    }
    if (idbA != cur) {
      if (close_run(lo_bA, k_lat, idbA)) { S.event = true; return true; }
      if (idbA == kVoxelGuard) return true;
    }
    if (idcA != cur) {
      if (close_run(lo_cA, 0u, idcA)) { S.event = true; return true; }
      if (idcA == kVoxelGuard) return true;
    }
    return false;
  }
  // The same slab in three parts, for the walk stage (scatter_walk_kernel), where the lanes of a warp are on unrelated
  // paths and the long, rare part -- the end of a run -- is worth waiting for company with:  probe() looks at the slab's
  // cells and says whether a run ends in it; settle() closes the runs (true = the leg is over); advance() skips on.
  unsigned p_idb, p_cell;  // what probe() saw
  __device__ __forceinline__ unsigned id_of_cell(unsigned cell) const { return CELL == 1 ? id_of_compact(cell) : (cell & 0xffu); }
  __device__ __forceinline__ bool probe() {
    const unsigned lo_b = lo + cu * so_u + cv * so_v;
    p_idb = (cu | cv) ? MCX_VOXEL_AT(lo_b) : cur;  // (no lateral step: b is the cell the ray stands in)
    p_cell = CELL == 1 ? ld_voxel(hi | (lo_b + so_w)) : ld_cell(hi | (lo_b + so_w));
    return p_idb != cur || id_of_cell(p_cell) != cur || (cu & cv) != 0u;
  }
  // The crossings of the slab in the order the ray meets them -- the cell between the two lateral faces of a double
  // step (a), the lateral neighbour (b), the cell behind the w face (c) -- closed one per round by ONE copy of
  // close_run, so that the lanes of a warp that settle together run it together (most have one crossing).  Same
  // arithmetic in the same order as settle_slab.
  __device__ __forceinline__ bool settle() {
    const unsigned lo_b = lo + cu * so_u + cv * so_v, lo_c = lo_b + so_w, idb = p_idb, idc = id_of_cell(p_cell);
    unsigned k_lat = cu ? 1u : 2u, k_first = 0u, lo_a = 0u, ida = cur;
    if (cu & cv) {
      const unsigned long long au = ((unsigned long long)auh << 32) | aul, av = ((unsigned long long)avh << 32) | avl;
      const unsigned long long fu = ((unsigned long long)fuh << 32) | ful, fv = ((unsigned long long)fvh << 32) | fvl;
      const bool u_first = __umul64hi(fu, av) >= __umul64hi(fv, au);
      k_first = u_first ? 1u : 2u;
      k_lat = u_first ? 2u : 1u;
      lo_a = lo_b - (u_first ? so_v : so_u);
      ida = MCX_VOXEL_AT(lo_a);
    }
    // which of a, b, c the ray enters through a face between different IDs: each against the cell before it
    unsigned todo = (ida != cur ? 1u : 0u) | (idb != ida ? 2u : 0u) | (idc != idb ? 4u : 0u);
#pragma unroll 1
    while (todo) {
      const unsigned crossing = (unsigned)__ffs((int)todo) - 1u;
      todo &= todo - 1u;
      const unsigned id = crossing == 0u ? ida : (crossing == 1u ? idb : idc);
      if (close_run(crossing == 0u ? lo_a : (crossing == 1u ? lo_b : lo_c), crossing == 0u ? k_first : (crossing == 1u ? k_lat : 0u), id)) {
        S.event = true;
        return true;
      }
      if (id == kGuard) return true;
    }
    return false;
  }
  __device__ __forceinline__ void advance() {  // the skip of step(), from what probe() saw
    const unsigned lo_c = lo + cu * so_u + cv * so_v + so_w;
    unsigned s;
    if (CELL == 1) {  // the cube radius only
      const unsigned R = radius_of_code(p_cell >> 4);
      s = R > 0u ? R - 1u : 0u;
    } else {
      const unsigned run = (p_cell >> 8) & 0xffu, R = (p_cell >> 16) & 0xffu;
      const unsigned s_run = min(min(run, __umulhi(~fuh, inv_u)), __umulhi(~fvh, inv_v));
      s = max(s_run, R > 0u ? R - 1u : 0u);
    }
    const unsigned long long tu = (unsigned long long)s * aul + ful, tv = (unsigned long long)s * avl + fvl;
    const unsigned long long tu1 = (unsigned long long)s * auh + fuh + (tu >> 32), tv1 = (unsigned long long)s * avh + fvh + (tv >> 32);
    ful = (unsigned)tu; fuh = (unsigned)tu1;
    fvl = (unsigned)tv; fvh = (unsigned)tv1;
    lo = lo_c + s * so_w + (unsigned)(tu1 >> 32) * so_u + (unsigned)(tv1 >> 32) * so_v;
    w_crossed += s + 1u;
    cu = add_carry(ful, fuh, aul, auh);
    cv = add_carry(fvl, fvh, avl, avh);
  }
  // one slab and a skip; true = the leg is over (the ray left the grid, or S.event)
  __device__ __forceinline__ bool step() {
    const unsigned lo_b = lo + cu * so_u + cv * so_v, lo_c = lo_b + so_w;
    const unsigned idb = MCX_VOXEL_AT(lo_b);
    const unsigned cell_c = ld_cell(hi | lo_c);
    const unsigned idc = cell_c & 0xffu;
    if (idb != cur || idc != cur || (cu & cv) != 0u) {
      if (settle_slab(cu, cv, lo_b, lo_c, idb, idc)) return true;
    }
    // Skip.  Standing in cell c (same ID as the run), the ray may cross s more w faces without looking at anything
    //  (a) if the next s cells of the row hold the same ID (the cell's RUN; rays along the fast axis in the direction the
    //      runs were counted in, inv != 0) and no lateral face comes in those s slabs: s <= (2^64 - 1 - f) / a, taken
    //      conservatively from the high words as mulhi(~f_hi, inv) with inv <= 2^32 / (a_hi + 1); or
    //  (b) if s = R - 1, R the cell's RADIUS: the cube of cells within Chebyshev distance R of c holds c's ID throughout
    //      (voxel_boundary_kernel), and in s slabs the ray crosses at most s a + 1 <= R faces of either lateral axis, so
    //      every cell on the way lies in the cube -- in any direction, with whatever lateral faces come.
    // The larger of the two.  f += s a exactly; what that carries out of the 64-bit fraction is the number of lateral
    // faces crossed (none in case (a)), and the address moves by as many lateral strides.
    {
      const unsigned run = (cell_c >> 8) & 0xffu, R = (cell_c >> 16) & 0xffu;
      const unsigned s_run = min(min(run, __umulhi(~fuh, inv_u)), __umulhi(~fvh, inv_v));
      const unsigned s = max(s_run, R > 0u ? R - 1u : 0u);
      const unsigned long long tu = (unsigned long long)s * aul + ful, tv = (unsigned long long)s * avl + fvl;
      const unsigned long long tu1 = (unsigned long long)s * auh + fuh + (tu >> 32), tv1 = (unsigned long long)s * avh + fvh + (tv >> 32);
      ful = (unsigned)tu; fuh = (unsigned)tu1;
      fvl = (unsigned)tv; fvh = (unsigned)tv1;
      lo = lo_c + s * so_w + (unsigned)(tu1 >> 32) * so_u + (unsigned)(tv1 >> 32) * so_v;
      w_crossed += s + 1u;
    }
    cu = add_carry(ful, fuh, aul, auh);
    cv = add_carry(fvl, fvh, avl, avh);
    return false;
  }
};
#undef MCX_VOXEL_AT


// Step 11 (and 17 where the volume scatters): the legs of one ray, then tau = sum over the touched materials of
// mu_m(E) * len_m (step 7 evaluated for those only) - what the scattering took of it while events were left.
template <bool SCAT>
__device__ __forceinline__ void trace_voxels(const SInst& I, const DComponent& C, int comp, Ray& ray, uint64_t seed, uint64_t i,
                                             double* len_s, double* cold_s, double* mus_s, unsigned lanes) {
  const DVoxels& V = C.u.voxels;
  Vec3 ol = to_local(C.pose, ray.r), dl = rotate(C.pose, ray.d);
  unsigned touched = 0u;
  Scat S;
  S.k = 0; S.K = SCAT ? V.scatter_order : 0; S.s_pre = 0.0; S.cum = 0.0; S.tau_s = 0.0; S.t_event = 0.0; S.have_ms = 0u; S.event = false;
  const double lnE_early = SCAT ? log(ray.E) : 0.0;  // (without scattering ln E is not needed, nor kept in a register, during the walk)
  VoxWalk<SCAT> walk{I, V, ray.E, lnE_early, len_s, cold_s, mus_s, touched, S};
  if (!SCAT) {
    if (walk.setup(ol, dl))
      while (!walk.step()) {}
  } else {
    // The lanes of the warp that are in this volume (`lanes`) stay in ONE loop, whose iteration is warp-uniformly either
    // one slab for the lanes that are walking, or -- when nobody walks any more, or kBatch lanes are waiting -- the end of
    // a leg (the scattering event) and the set-up of the next one for all the lanes whose leg is over.  So the long
    // set-up and event code runs with many lanes at a time, and a lane whose leg ends early waits for company instead of
    // stalling 31 walkers.  (Left to themselves, lanes that re-enter a walk loop after an event never rejoin those
    // still in it: a first version with a loop per leg and no barrier ran with 1.4 of 32 lanes active.)
    enum { kPending, kWalking, kDone };
    constexpr int kBatch = 8;
    int state = kPending;
    bool first_leg = true;
    double u_mu = 0.0;
    for (;;) {
      const unsigned pending = __ballot_sync(lanes, state == kPending), walking = __ballot_sync(lanes, state == kWalking);
      if ((pending | walking) == 0u) break;
      if (walking == 0u || __popc(pending) >= kBatch) {
        if (state == kPending) {
          bool go_on = true;
          if (!first_leg) {  // how the last leg ended
            if (!S.event) {
              if (S.k < S.K) S.s_pre += S.cum;
              state = kDone;
              go_on = false;
            } else {
              S.s_pre += S.tau_s;
              double u_phi, unused;
              draw2(seed, i, (uint32_t)(2 * S.k + 1), (uint32_t)comp, u_phi, unused);
              ol = ol + S.t_event * dl;
              dl = scatter_direction(dl, u_mu, u_phi);
              ++S.k;
            }
          }
          if (go_on) {
            first_leg = false;
            if (S.k < S.K) {
              double u_f;
              draw2(seed, i, (uint32_t)(2 * S.k), (uint32_t)comp, u_f, u_mu);
              S.tau_s = -log(u_f);
              S.cum = 0.0;
            }
            if (walk.setup(ol, dl)) state = kWalking;  // (a half-line that misses the grid: leg over at once, no event)
          }
        }
      } else if (state == kWalking) {
        if (walk.step()) state = kPending;
      }
    }
  }
  const double lnE = SCAT ? lnE_early : log(ray.E);
  double tau = 0.0;
  while (touched) {
    const int m = __ffs(touched) - 1;
    touched &= touched - 1u;
    tau += mu_of(I.mats[m], ray.E, lnE) * len_s[m * kBlock];
  }
  if (SCAT) tau -= S.s_pre;
  ray.p *= exp(-tau);
  if (SCAT && S.k > 0) {
    ray.r = to_lab(C.pose, ol);
    ray.d = rotate_back(C.pose, dl);
  }
}

// ------------------------------------------------------------------------------------------------------------
// Steps 11 + 17 as a stage of their own: every ray of the pool through one scattering voxel volume.
// Inside trace_kernel the 32 rays of a warp enter the sample together and the warp leaves when its last ray does; with
// 1 to K + 1 legs per ray of very different lengths, 9 of 32 lanes work on average.  Here a lane whose ray has left the
// sample takes the next ray of the pool, so all lanes walk until the pool is empty.  Same arithmetic, ray for ray, as
// trace_voxels<true>.  The loop is warp-uniform; an iteration is one of
//   - one slab (probe + skip) for the lanes that are walking;
//   - the ends of runs (close_run: path lengths, the scattering depth, the event) for the lanes whose slab holds one,
//     once nobody walks or batch_settle lanes wait for it;
//   - the end of a leg (the scattering event, or the ray's weight back into its record and the next ray of the pool)
//     and the set-up of the next leg, once nobody else has work or batch_setup lanes wait for it.
// ------------------------------------------------------------------------------------------------------------
constexpr unsigned kWalkRange = 256u;  // consecutive records a warp takes from the pool at a time
constexpr int kWalkBlocks = 2;

template <int CELL>
__global__ void __launch_bounds__(kBlock, kWalkBlocks) scatter_walk_kernel(const DInstrument* __restrict__ g_inst, WalkArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n_mats = A.n_mats;
  double* len_s = reinterpret_cast<double*>(smem_raw) + threadIdx.x;
  double* cold_s = len_s + (size_t)n_mats * kBlock;
  double* mus_s = cold_s + (size_t)VC_COUNT * kBlock;
  DComponent* s_comp = reinterpret_cast<DComponent*>(smem_raw + (size_t)(2 * n_mats + VC_COUNT) * kBlock * sizeof(double));
  DMaterial* s_mats = reinterpret_cast<DMaterial*>(s_comp + 1);
  {
    const unsigned long long* src = reinterpret_cast<const unsigned long long*>(g_inst->comps + A.comp);
    unsigned long long* dst = reinterpret_cast<unsigned long long*>(s_comp);
    for (int k = threadIdx.x; k < (int)(sizeof(DComponent) / 8); k += kBlock) dst[k] = src[k];
    src = reinterpret_cast<const unsigned long long*>(g_inst->mats);
    dst = reinterpret_cast<unsigned long long*>(s_mats);
    for (int k = threadIdx.x; k < n_mats * (int)(sizeof(DMaterial) / 8); k += kBlock) dst[k] = src[k];
  }
  __syncthreads();
  const SInst I{1, n_mats, s_comp, s_mats, nullptr, nullptr};
  const DComponent& C = *s_comp;
  const DVoxels& V = C.u.voxels;
  const int lane = threadIdx.x & 31;
  const unsigned lanes_below = (1u << lane) - 1u;
  const unsigned count = A.pool_count[0];
  const uint64_t seed = A.seed;
  const uint32_t comp = (uint32_t)A.comp;
  const int batch_setup = A.batch_setup, batch_settle = A.batch_settle;

  enum { kFetch, kPending, kWalking, kSettle, kDone };
  int state = kFetch;
  unsigned r_next = 0u, r_end = 0u;  // the warp's range of records (warp-uniform)
  bool exhausted = false;            // the pool has no further range (warp-uniform)
  unsigned rec = 0u;                 // this lane's record
  uint64_t ray_index = 0;
  double p = 0.0, u_mu = 0.0;
  bool first_leg = true;
  Vec3 ol{0.0, 0.0, 0.0}, dl{0.0, 0.0, 1.0};
  unsigned touched = 0u;
  Scat S;
  S.k = 0; S.K = V.scatter_order; S.s_pre = 0.0; S.cum = 0.0; S.tau_s = 0.0; S.t_event = 0.0; S.have_ms = 0u; S.event = false;
  VoxWalk<true, CELL> walk{I, V, 1.0, 0.0, len_s, cold_s, mus_s, touched, S};
  for (;;) {
    const unsigned waiting = __ballot_sync(0xffffffffu, state == kPending || state == kFetch);
    const unsigned walking = __ballot_sync(0xffffffffu, state == kWalking);
    const unsigned settling = __ballot_sync(0xffffffffu, state == kSettle);
    if ((waiting | walking | settling) == 0u) break;
    if (settling != 0u && (walking == 0u || __popc(settling) >= batch_settle)) {
      // the runs that end in the slabs these lanes stand in; a leg that ends there (event, or out of the grid) waits for
      // its set-up below, the others walk on
      if (state == kSettle) {
        if (walk.settle()) {
          state = kPending;
        } else {
          walk.advance();
          state = kWalking;
        }
      }
    } else if (waiting != 0u && ((walking | settling) == 0u || __popc(waiting) >= batch_setup)) {
      if (state == kPending && !first_leg) {  // how the last leg ended
        if (!S.event) {  // the ray has left the sample: its weight, and where it goes, back into its record
          if (S.k < S.K) S.s_pre += S.cum;
          double tau = 0.0;
          while (touched) {
            const int m = __ffs(touched) - 1;
            touched &= touched - 1u;
            tau += mu_of(I.mats[m], walk.E, walk.lnE) * len_s[m * kBlock];
          }
          tau -= S.s_pre;
          PoolRay& R = A.pool[rec];
          R.p = p * exp(-tau);
          if (S.k > 0) {
            const Vec3 r = to_lab(C.pose, ol), d = rotate_back(C.pose, dl);
            R.r[0] = r.x; R.r[1] = r.y; R.r[2] = r.z;
            R.d[0] = d.x; R.d[1] = d.y; R.d[2] = d.z;
          }
          state = kFetch;
        } else {
          S.s_pre += S.tau_s;
          double u_phi, unused;
          draw2(seed, ray_index, (uint32_t)(2 * S.k + 1), comp, u_phi, unused);
          ol = ol + S.t_event * dl;
          dl = scatter_direction(dl, u_mu, u_phi);
          ++S.k;
        }
      }
      {  // the next rays of the pool for the lanes without one
        const unsigned want = __ballot_sync(0xffffffffu, state == kFetch);
        if (want) {
          if (r_next == r_end && !exhausted) {
            unsigned t = 0u;
            if (lane == 0) t = atomicAdd(A.pool_count + 1, kWalkRange);
            t = __shfl_sync(0xffffffffu, t, 0);
            exhausted = t >= count;
            r_next = exhausted ? 0u : t;
            r_end = exhausted ? 0u : min(t + kWalkRange, count);
          }
          const unsigned avail = r_end - r_next, rank = __popc(want & lanes_below);
          if (state == kFetch) {
            if (rank < avail) {
              rec = r_next + rank;
              const PoolRay& R = A.pool[rec];
              ol = to_local(C.pose, Vec3{R.r[0], R.r[1], R.r[2]});
              dl = rotate(C.pose, Vec3{R.d[0], R.d[1], R.d[2]});
              walk.E = R.E;
              walk.lnE = log(R.E);
              p = R.p;
              ray_index = A.first + R.offset;
              touched = 0u;
              S.k = 0; S.s_pre = 0.0; S.cum = 0.0; S.tau_s = 0.0; S.t_event = 0.0; S.have_ms = 0u; S.event = false;
              first_leg = true;
              state = kPending;
            } else if (exhausted) {
              state = kDone;
            }
          }
          r_next += min(avail, (unsigned)__popc(want));
        }
      }
      if (state == kPending) {  // the next leg
        first_leg = false;
        if (S.k < S.K) {
          double u_f;
          draw2(seed, ray_index, (uint32_t)(2 * S.k), comp, u_f, u_mu);
          S.tau_s = -log(u_f);
          S.cum = 0.0;
        }
        if (walk.setup(ol, dl)) state = kWalking;  // (a half-line that misses the grid: leg over at once, no event)
        else S.event = false;
      }
    } else if (state == kWalking) {
      if (walk.probe()) state = kSettle;
      else walk.advance();
    }
  }
  // The last block to leave re-arms the pool's hand-out counter for the next chunk (the record count itself is cleared by
  // the host side before stage 1; stage 2 reads it after this kernel, on the same stream).  The barrier: every warp of the
  // block has taken its last range by then -- without it a late warp of another block could find the counter at zero
  // again and walk the pool a second time.
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    if (atomicAdd(A.pool_count + 2, 1u) == gridDim.x - 1) {
      A.pool_count[1] = 0u;
      A.pool_count[2] = 0u;
    }
  }
}

// ------------------------------------------------------------------------------------------------------------
// Step 12: elliptic-cylinder mirror.  Mirror frame: origin at the pole, z tangential, y = surface normal,
// x sagittal.  Returns true if reflected.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double reflectivity(const DMirror& M, double theta, double E) {
  const int nt = M.n_theta, ne = M.n_e;
  double ft = (theta - M.theta_min) * M.st;  // (grid cells per unit, from mcx_instrument_create: no division here)
  double fe = (E - M.e_min) * M.se;
  ft = fmin(fmax(ft, 0.0), (double)(nt - 1));
  fe = fmin(fmax(fe, 0.0), (double)(ne - 1));
  const int it = min((int)floor(ft), nt - 2), ie = min((int)floor(fe), ne - 2);
  const double wt = ft - (double)it, we = fe - (double)ie;
  const double* __restrict__ row0 = M.table + (size_t)it * ne + ie;
  const double* __restrict__ row1 = row0 + ne;
  const double r00 = row0[0], r01 = row0[1], r10 = row1[0], r11 = row1[1];
  return (1.0 - wt) * ((1.0 - we) * r00 + we * r01) + wt * ((1.0 - we) * r10 + we * r11);
}

__device__ __forceinline__ bool trace_mirror(const DComponent& C, Ray& ray) {
  const DMirror& M = C.u.mirror;
  const Vec3 o = to_local(C.pose, ray.r);
  const Vec3 d = rotate(C.pose, ray.d);
  // into the ellipse's principal frame (Z, Y)
  const double oZ = M.Z0 + o.z * M.tZ + o.y * M.nZ, oY = M.Y0 + o.z * M.tY + o.y * M.nY;
  const double dZ = d.z * M.tZ + d.y * M.nZ, dY = d.z * M.tY + d.y * M.nY;
  const double A = dZ * dZ * M.inv_a2 + dY * dY * M.inv_b2;
  const double B = oZ * dZ * M.inv_a2 + oY * dY * M.inv_b2;
  const double Cc = oZ * oZ * M.inv_a2 + oY * oY * M.inv_b2 - 1.0;
  if (A == 0.0) return false;
  const double disc = B * B - A * Cc;
  if (!(disc >= 0.0)) return false;
  const double qq = -(B + (B >= 0.0 ? 1.0 : -1.0) * fast_sqrt(disc));  // stable roots of A t^2 + 2 B t + C = 0
  double ta = qq / A, tb = (qq != 0.0) ? Cc / qq : ta;
  if (ta > tb) { const double t = ta; ta = tb; tb = t; }
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const double t = r == 0 ? ta : tb;
    if (!(t > 0.0)) continue;
    const Vec3 hp = o + t * d;
    if (fabs(hp.z) > M.half_length || fabs(hp.x) > M.half_width) continue;
    const double hZ = M.Z0 + hp.z * M.tZ + hp.y * M.nZ, hY = M.Y0 + hp.z * M.tY + hp.y * M.nY;
    if (!(hY < 0.0)) continue;  // the arc near the pole only
    const double gZ = hZ * M.inv_a2, gY = hY * M.inv_b2;
    const double ign = fast_rcp(fast_sqrt(gZ * gZ + gY * gY));  // (on the ellipse the gradient is far from zero)
    const double nZ = -gZ * ign, nY = -gY * ign;  // inward normal in (Z, Y)
    const Vec3 nrm{0.0, nZ * M.nZ + nY * M.nY, nZ * M.tZ + nY * M.tY};
    const double dn = dot(d, nrm);
    if (!(dn < 0.0)) return false;
    const double theta = asin(-dn);
    if (theta > M.theta_max) return false;
    ray.p *= reflectivity(M, theta, ray.E);
    const Vec3 dr = d - (2.0 * dn) * nrm;
    ray.r = to_lab(C.pose, hp);
    ray.d = rotate_back(C.pose, dr);
    return true;
  }
  return false;
}

// Step 13b: Darwin-Prins curve of an absorbing crystal.  eta_c = (eta + i g) / (1 + i kappa); R = 1 / |eta_c + s|^2 with s
// the square root of eta_c^2 - 1 whose inner product with eta_c is non-negative (then |eta_c + s| >= 1: no cancellation).
__device__ __forceinline__ double darwin_prins(double eta, double g, double kappa) {
  // (eta + i g) / (1 + i kappa) by the plain formula: |kappa| is small, nothing over- or underflows
  const double den = 1.0 + kappa * kappa;
  const double er = (eta + g * kappa) / den, ei = (g - eta * kappa) / den;
  // w = eta_c^2 - 1
  const double wr = er * er - ei * ei - 1.0, wi = 2.0 * er * ei;
  // principal square root of w: sr = sqrt((|w| + wr) / 2) without cancellation, si = wi / (2 sr) (or the mirrored form)
  const double mod = hypot(wr, wi);
  double sr, si;
  if (mod == 0.0) {
    sr = 0.0; si = 0.0;
  } else if (wr >= 0.0) {
    sr = sqrt(0.5 * (mod + wr));
    si = wi / (2.0 * sr);
  } else {
    const double t = sqrt(0.5 * (mod - wr));
    sr = fabs(wi) / (2.0 * t);
    si = wi < 0.0 ? -t : t;
  }
  if (er * sr + ei * si < 0.0) { sr = -sr; si = -si; }
  const double ar = er + sr, ai = ei + si;
  return 1.0 / (ar * ar + ai * ai);
}

// Step 16: compound refractive lens, DLens.  The ray meets the 2 N paraboloids in order; at each:
// the root of the intersection quadratic that tends to the plane intersection as R -> inf, in its cancellation-free form;
// aperture test; Snell's law in vector form, d' = m d + (c_t - m c) nrm with c_t - m c = (1 - m)(1 + m) / (c_t + m c) and
// 1 - m formed from delta directly, so the deflection (relative size delta ~ 1e-6) carries no cancellation.
__device__ __forceinline__ bool trace_lens(const SInst& I, const DComponent& C, Ray& ray) {
  const DLens& L = C.u.lens;
  Vec3 o = to_local(C.pose, ray.r);
  Vec3 d = rotate(C.pose, ray.d);
  const double lnE = log(ray.E);
  const double delta = mu_of(L.delta, ray.E, lnE);
  const double n_in = 1.0 - delta;
  const double m_in = 1.0 / n_in, omm_in = -delta / n_in;  // entering: m = 1 / n, 1 - m = -delta / n
  double path = 0.0;
  const int n_surf = 2 * L.n_lenses;
  const double mid = 0.5 * (double)(L.n_lenses - 1);
  for (int surf = 0; surf < n_surf; ++surf) {
    const bool entering = (surf & 1) == 0;
    const double zc = ((double)(surf >> 1) - mid) * L.pitch;
    const double sgn = entering ? -1.0 : 1.0;
    const double z0 = zc + sgn * L.half_web;
    const double a = -sgn * (d.x * d.x + d.y * d.y) * L.half_inv_R;
    const double b = d.z - sgn * (o.x * d.x + o.y * d.y) * L.inv_R;
    const double cc = o.z - z0 - sgn * (o.x * o.x + o.y * o.y) * L.half_inv_R;
    if (!(b > 0.0)) return false;
    const double disc = b * b - 4.0 * a * cc;
    if (!(disc >= 0.0)) return false;
    const double t = -2.0 * cc * fast_rcp(b + fast_sqrt(disc));
    if (t < 0.0) return false;
    const Vec3 h = o + t * d;
    if (h.x * h.x + h.y * h.y > L.ra2) return false;
    if (!entering) path += t;
    // Snell's law with the UNNORMALISED normal G = grad F = (-sgn x / R, -sgn y / R, 1): with g2 = |G|^2, D = d.G = c |G| and
    // Ct = c_t |G| = sqrt(g2 - m^2 (g2 - D^2)), the refracted direction m d + (c_t - m c) G / |G| is
    // m d + [(1 - m)(1 + m) / (Ct + m D)] G: one square root and one division per surface instead of two and two (the same
    // real number as step 16's form with the unit normal; only the rounding differs).
    const double gx = -sgn * h.x * L.inv_R, gy = -sgn * h.y * L.inv_R;
    const double g2 = gx * gx + gy * gy + 1.0;
    const double D = d.x * gx + d.y * gy + d.z;
    if (!(D > 0.0)) return false;
    const double m = entering ? m_in : n_in;
    const double one_minus_m = entering ? omm_in : delta;
    const double under = g2 - m * m * (g2 - D * D);
    if (!(under > 0.0)) return false;  // total reflection
    const double coef = one_minus_m * (1.0 + m) * fast_rcp(fast_sqrt(under) + m * D);
    d = Vec3{m * d.x + coef * gx, m * d.y + coef * gy, m * d.z + coef};
    o = h;
  }
  ray.p *= exp(-mu_of(I.mats[L.material], ray.E, lnE) * path);
  ray.r = to_lab(C.pose, o);
  ray.d = rotate_back(C.pose, d);
  return true;
}

// Step 13: symmetric Bragg reflection off a thick non-absorbing crystal (Darwin curve).
__device__ __forceinline__ bool trace_crystal(const DComponent& C, Ray& ray) {
  const DCrystal& X = C.u.crystal;
  const Vec3 o = to_local(C.pose, ray.r);
  const Vec3 d = rotate(C.pose, ray.d);
  if (!(d.y < 0.0)) return false;
  const double t = -o.y / d.y;
  if (!(t > 0.0)) return false;
  const Vec3 hp = o + t * d;
  if (fabs(hp.z) > X.half_length || fabs(hp.x) > X.half_width) return false;
  const double theta = asin(-d.y);
  const double lambda = 12.398419843 / ray.E;  // h c in keV Angstrom
  const double s = lambda / (2.0 * X.d_hkl);
  if (!(s < 1.0)) return false;
  const double theta_b = asin(s);
  const double w_d = X.zeta * tan(theta_b);
  const double eta_s = (theta - theta_b - X.delta0) / (0.5 * w_d);
  if (X.g != 0.0 || X.kappa != 0.0) {
    ray.p *= darwin_prins(eta_s, X.g, X.kappa);
  } else {
    const double eta = fabs(eta_s);
    if (eta > 1.0) {
      const double g = eta + sqrt(eta * eta - 1.0);
      ray.p *= 1.0 / (g * g);
    }
  }
  ray.r = to_lab(C.pose, Vec3{hp.x, 0.0, hp.z});
  ray.d = rotate_back(C.pose, Vec3{d.x, -d.y, d.z});
  return true;
}

// ------------------------------------------------------------------------------------------------------------
// Detector-tile ordering of a chunk of rays (row a13).  A ray's direction is fixed by its slot-1
// draw (ua, ub) (step 3), and draws are slot-addressed (step 1), so rays may be traced in any order.  The three
// kernels below bucket the ray offsets of a chunk by the cell of a 2^g x 2^g grid over (ua, ub) their slot-1 draw
// falls in (count -> scan -> scatter); trace_kernel then gives each warp 32 consecutive entries = rays aimed at
// (nearly) the same spot, which walk the same voxel rows / BVH nodes / primitives in lockstep.
// Cell order: 8 x 8 blocks of cells are contiguous, so a tile of consecutive positions is compact in 2-D.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t sort_key(uint64_t seed, uint64_t i, int g) {
  uint32_t w[4];
  philox4x32_10((uint32_t)i, (uint32_t)(i >> 32), 1u, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), w);
  const uint32_t kx = w[0] >> (32 - g), ky = w[2] >> (32 - g);  // top g bits of ua and ub (step 2)
  if (g >= 3) return ((((ky >> 3) << (g - 3)) | (kx >> 3)) << 6) | ((ky & 7u) << 3) | (kx & 7u);
  return (ky << g) | kx;
}

__global__ void __launch_bounds__(256) sort_count_kernel(uint64_t first, uint32_t n, uint64_t seed, int g,
                                                         unsigned int* __restrict__ cnt) {
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < n; q += stride) atomicAdd(&cnt[sort_key(seed, first + q, g)], 1u);
}

// In-place exclusive scan of cnt within blocks of kScanBlock entries; bsum[b] = total of block b.
constexpr int kScanBlock = 2048;
__global__ void __launch_bounds__(256) sort_scan_kernel(unsigned int* __restrict__ cnt, uint32_t n_buckets,
                                                        unsigned int* __restrict__ bsum) {
  __shared__ unsigned int s_w[8];
  const uint32_t base = blockIdx.x * kScanBlock + threadIdx.x * 8;
  unsigned int v[8], tot = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const unsigned int x = base + k < n_buckets ? cnt[base + k] : 0u;
    v[k] = tot;
    tot += x;
  }
  unsigned int inc = tot;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const unsigned int y = __shfl_up_sync(0xffffffffu, inc, d);
    if ((threadIdx.x & 31) >= d) inc += y;
  }
  if ((threadIdx.x & 31) == 31) s_w[threadIdx.x >> 5] = inc;
  __syncthreads();
  unsigned int off = 0;
  for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) off += s_w[w];
  const unsigned int excl = off + inc - tot;
#pragma unroll
  for (int k = 0; k < 8; ++k)
    if (base + k < n_buckets) cnt[base + k] = excl + v[k];
  if (threadIdx.x == 255) bsum[blockIdx.x] = off + inc;
}

constexpr int kMaxScanBlocks = MCX_SORT_MAX_SCAN_BLOCKS;  // 2^22 buckets / kScanBlock
__global__ void __launch_bounds__(256) sort_scatter_kernel(uint64_t first, uint32_t n, uint64_t seed, int g,
                                                           unsigned int* __restrict__ cnt, const unsigned int* __restrict__ bsum,
                                                           int n_scan_blocks, uint32_t* __restrict__ order) {
  __shared__ unsigned int s_pre[kMaxScanBlocks];
  __shared__ unsigned int s_w[8];
  {  // exclusive scan of the block totals, kMaxScanBlocks / 256 consecutive ones per thread
    constexpr int kPer = kMaxScanBlocks / 256;
    const int t = threadIdx.x;
    unsigned int v[kPer], tot = 0;
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
      v[k] = tot;
      tot += kPer * t + k < n_scan_blocks ? bsum[kPer * t + k] : 0u;
    }
    unsigned int inc = tot;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const unsigned int y = __shfl_up_sync(0xffffffffu, inc, d);
      if ((t & 31) >= d) inc += y;
    }
    if ((t & 31) == 31) s_w[t >> 5] = inc;
    __syncthreads();
    unsigned int off = 0;
    for (int w = 0; w < (t >> 5); ++w) off += s_w[w];
    const unsigned int excl = off + inc - tot;
#pragma unroll
    for (int k = 0; k < kPer; ++k) s_pre[kPer * t + k] = excl + v[k];
    __syncthreads();
  }
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < n; q += stride) {
    const uint32_t key = sort_key(seed, first + q, g);
    const uint32_t pos = s_pre[key / kScanBlock] + atomicAdd(&cnt[key], 1u);
    order[pos] = q;
  }
}

// ------------------------------------------------------------------------------------------------------------
// Step 14, the tally update (row a12; monitor arrays updated atomically).  Three ways, chosen per
// launch (TraceArgs::tally_mode, mcx_tuning.tally_mode; DESIGN.md 5.5 has the measurements that pick the default):
//   TALLY_GLOBAL   every detected ray issues its own three reductions (u64 count, two fp64 sums) into its 32-byte record;
//   TALLY_WARP     warp-aggregated: the lanes of a warp that hit the same bin are found with match.any, their weights
//                  are summed with a shuffle butterfly, and one leader per distinct bin issues the three reductions;
//   TALLY_BLOCK    as TALLY_WARP, but the leader adds into a block-private cache in shared memory (a direct-mapped
//                  table of 2^k records keyed by detector and bin, claimed with a compare-and-swap); bins whose slot is
//                  taken by another bin go to global memory as before.  The block flushes its cache with one set of
//                  reductions per occupied slot when it has no work left: the "privatised per block, then reduced"
//                  scheme north_star names, for detectors whose illuminated bins fit (c0: 32 x 32 pixels).
// All three add the same integers; the fp64 sums differ in summation order only.
// ------------------------------------------------------------------------------------------------------------
struct TallyCache {
  unsigned long long* key;  // [2^log2] 0 = empty, else ((detector + 1) << 48) | bin; then N, P, P2 arrays of the same length
  int log2;                 // 0 = no cache
  unsigned dets;            // bit d: detector d goes through the cache (its bins fit; TraceArgs::tally_cache_dets)
};

__device__ __forceinline__ void tally_global(TallyBin* rec, unsigned long long cnt, double sp, double sp2) {
  atomicAdd(&rec->N, cnt);
  atomicAdd(&rec->P, sp);
  atomicAdd(&rec->P2, sp2);
}

// The aggregating paths (TALLY_WARP, TALLY_BLOCK).  Must be called by all 32 lanes; `on` = this lane has a ray to tally
// into bin `bin` of detector `det` with weight p.  Kept out of line: the default path (tally_add below) must not pay
// registers for it (the optics kernel sits at the edge of two resident blocks).
__device__ __noinline__ void tally_add_aggregated(TallyBin* const* tallies, int mode, unsigned long long* cache_key, int cache_log2,
                                                  unsigned det, bool on, long long bin, double p) {
  const unsigned full = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const unsigned m = __ballot_sync(full, on);
  if (m == 0u) return;
  if (cache_log2 > 0) {
    // Block cache: unless many of the warp's rays share one bin, every lane adds for itself -- the butterfly sums below
    // cost more than the few same-address retries in shared memory (measured on an L_monitor of n bins under a flat
    // spectrum: 8 bins 3.5 ms against 3.6, 128 bins 2.4 against 3.3; 1 bin 12.5 against 2.5: there the sums win).  The
    // test: how many lanes share the first ray's bin (a flat distribution over >= 8 bins gives about 32 / n).
    const long long b0 = __shfl_sync(full, bin, __ffs(m) - 1);
    if (__popc(__ballot_sync(full, on && bin == b0)) < 8) {
      if (on) {
        const unsigned long long k = ((unsigned long long)(det + 1u) << 48) | (unsigned long long)bin;
        const unsigned h = (unsigned)((k * 0x9E3779B97F4A7C15ull) >> (64 - cache_log2));
        const unsigned long long prev = atomicCAS(&cache_key[h], 0ull, k);
        if (prev == 0ull || prev == k) {
          const size_t n = (size_t)1 << cache_log2;
          atomicAdd(&cache_key[n + h], 1ull);
          atomicAdd(reinterpret_cast<double*>(&cache_key[2 * n + h]), p);
          atomicAdd(reinterpret_cast<double*>(&cache_key[3 * n + h]), p * p);
        } else {
          tally_global(tallies[det] + bin, 1ull, p, p * p);
        }
      }
      return;
    }
  }
  unsigned grp = 0u;
  if (on) grp = __match_any_sync(m, (unsigned long long)bin);
  const bool lead = on && (__ffs(grp) - 1) == lane;
  const unsigned cnt = (unsigned)__popc(grp);
  double sp = p, sp2 = p * p;
  // groups of more than one lane (rare unless a warp's rays share pixel AND energy bin): butterfly sums, group by group
  for (unsigned todo = __ballot_sync(full, lead && cnt > 1u); todo; todo &= todo - 1u) {
    const int l = __ffs(todo) - 1;
    const unsigned g = __shfl_sync(full, grp, l);
    const bool in = (g >> lane) & 1u;
    double a = in ? p : 0.0, b = in ? p * p : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a += __shfl_xor_sync(full, a, o);
      b += __shfl_xor_sync(full, b, o);
    }
    if (lane == l) { sp = a; sp2 = b; }
  }
  if (!lead) return;
  if (cache_log2 > 0) {
    const unsigned long long k = ((unsigned long long)(det + 1u) << 48) | (unsigned long long)bin;
    const unsigned h = (unsigned)((k * 0x9E3779B97F4A7C15ull) >> (64 - cache_log2));
    const unsigned long long prev = atomicCAS(&cache_key[h], 0ull, k);
    if (prev == 0ull || prev == k) {
      const size_t n = (size_t)1 << cache_log2;
      atomicAdd(&cache_key[n + h], (unsigned long long)cnt);
      atomicAdd(reinterpret_cast<double*>(&cache_key[2 * n + h]), sp);
      atomicAdd(reinterpret_cast<double*>(&cache_key[3 * n + h]), sp2);
      return;
    }
  }
  tally_global(tallies[det] + bin, (unsigned long long)cnt, sp, sp2);
}

// Step 14 for one warp and one detector (all 32 lanes call it).
__device__ __forceinline__ void tally_add(const SInst& I, int mode, const TallyCache& tc, unsigned det, bool on, long long bin,
                                          double p) {
  if (mode == MCX_TALLY_GLOBAL) {
    if (on) tally_global(I.tallies[det] + bin, 1ull, p, p * p);
  } else {
    tally_add_aggregated(I.tallies, mode, tc.key, (mode == MCX_TALLY_BLOCK && ((tc.dets >> det) & 1u)) ? tc.log2 : 0, det, on, bin, p);
  }
}

// the block's cache goes to global memory: one set of reductions per occupied slot (all threads of the block)
__device__ __forceinline__ void tally_flush(const SInst& I, const TallyCache& tc) {
  if (tc.log2 == 0) return;
  const int n = 1 << tc.log2;
  for (int h = threadIdx.x; h < n; h += kBlock) {
    const unsigned long long k = tc.key[h];
    if (k == 0ull) continue;
    const unsigned det = (unsigned)(k >> 48) - 1u;
    const unsigned long long bin = k & 0xFFFFFFFFFFFFull;
    tally_global(I.tallies[det] + bin, tc.key[n + h], __longlong_as_double((long long)tc.key[2 * n + h]),
                 __longlong_as_double((long long)tc.key[3 * n + h]));
  }
}

// ------------------------------------------------------------------------------------------------------------
// The megakernel.  FEAT selects which component kinds are compiled in; DUMP writes per-ray fates instead of
// tallying; GATE compiles in the absorber gate.  Shared memory: the instrument image, per-block ray-accounting and
// scheduling counters, (GATE) per-warp rings of survivors, the solids of every group, per-thread interval end
// points and candidate-triangle queue, per-thread path lengths per material and run-end scratch of the voxel walk.
// Spectrum CDFs, guide tables and mu(E) tables are read through L1.
// ------------------------------------------------------------------------------------------------------------
constexpr size_t kRingBytes = (kBlock / 32) * 64 * sizeof(unsigned);  // per-warp rings of gate survivors
constexpr unsigned kTileMax = 8192;  // positions per work ticket (a power of two >= kBlock; smaller for short launches)

// resident blocks per SM the register budget is held to: the voxel walk and the primitives hide their loads with warps
// (3 x 80 registers; with 2 blocks c4 loses 14 %, c1 18 %), the mesh kernels spill at 80 and run 12 % faster with 2 x 128
constexpr int min_blocks(int feat) {
  return (feat == F_VOXELS || feat == (F_SOLIDS | F_PRIM)) ? 3 : (feat == (F_SOLIDS | F_MESH | F_PRIM) || feat == (F_SOLIDS | F_MESH)) ? 2
         : (feat == F_OPTICS || feat == F_LENS || feat == (F_VOXELS | F_SCATTER)) ? 2 : 1;
}

template <int FEAT, bool DUMP, bool GATE>
__global__ void __launch_bounds__(kBlock, min_blocks(FEAT)) trace_kernel(const DInstrument* __restrict__ g_inst, TraceArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned int* s_cnt = reinterpret_cast<unsigned int*>(smem_raw);  // [MCX_MAX_COMPONENTS + 4]
  unsigned int* s_sched = s_cnt + MCX_MAX_COMPONENTS + 4;  // [0..1] tile tickets, [2..3] slice counters (ping-pong)
  const int n_comps = A.n_comps, n_mats = A.n_mats;
  // Layout: counters (128 bytes), gate rings, then the per-thread scratch at offsets that do not depend on the instrument
  // (interval end points, triangle queue | voxel path lengths | tally cache), then the instrument itself, compact (SInst:
  // components, materials, tally pointers, solids).
  unsigned char* s_extra = smem_raw + 128 + (GATE ? kRingBytes : 0);
  Endpoints ep{nullptr, nullptr, 0};
  unsigned* tri_queue = nullptr;
  if (FEAT & F_SOLIDS) {  // per-thread interval end points (and, with meshes, the candidate-triangle queue)
    ep.cap = A.cap_endpoints;
    ep.t = reinterpret_cast<double*>(s_extra) + threadIdx.x;
    s_extra += (size_t)ep.cap * kBlock * sizeof(double);
    ep.tag = s_extra + threadIdx.x;
    s_extra += (size_t)ep.cap * kBlock;
    if (FEAT & F_MESH) {
      tri_queue = reinterpret_cast<unsigned*>(s_extra) + threadIdx.x;
      s_extra += (size_t)kTriQueue * kBlock * sizeof(unsigned);
    }
  }
  double* len_s = reinterpret_cast<double*>(s_extra) + threadIdx.x;  // per-thread path length per material (voxel walk)
  if (FEAT & F_VOXELS) s_extra += (size_t)(n_mats + VC_COUNT + ((FEAT & F_SCATTER) ? n_mats : 0)) * kBlock * sizeof(double);
  TallyCache tcache{nullptr, 0, A.tally_cache_dets};
  const int tally_mode = A.tally_mode;
  if (!DUMP && !(FEAT & (F_SOLIDS | F_VOXELS)) && A.tally_cache_log2 > 0) {  // block-private tally cache (chains without solids or voxels)
    tcache.key = reinterpret_cast<unsigned long long*>(s_extra);
    tcache.log2 = A.tally_cache_log2;
    s_extra += (size_t)32 << tcache.log2;
    for (int k = threadIdx.x; k < (4 << tcache.log2); k += kBlock) tcache.key[k] = 0ull;
    // (the barrier after the first ticket fetch below orders these stores before any update)
  }
  DComponent* s_comps = reinterpret_cast<DComponent*>(s_extra);
  DMaterial* s_mats = reinterpret_cast<DMaterial*>(s_comps + n_comps);
  TallyBin** s_tallies = reinterpret_cast<TallyBin**>(s_mats + n_mats);
  {
    static_assert(sizeof(DComponent) % 8 == 0 && sizeof(DMaterial) % 8 == 0, "copied as 8-byte words");
    const unsigned long long* src = reinterpret_cast<const unsigned long long*>(g_inst->comps);
    unsigned long long* dst = reinterpret_cast<unsigned long long*>(s_comps);
    for (int k = threadIdx.x; k < n_comps * (int)(sizeof(DComponent) / 8); k += kBlock) dst[k] = src[k];
    src = reinterpret_cast<const unsigned long long*>(g_inst->mats);
    dst = reinterpret_cast<unsigned long long*>(s_mats);
    for (int k = threadIdx.x; k < n_mats * (int)(sizeof(DMaterial) / 8); k += kBlock) dst[k] = src[k];
    if (threadIdx.x < MCX_MAX_DETECTORS) s_tallies[threadIdx.x] = g_inst->tallies[threadIdx.x];
    if (threadIdx.x < MCX_MAX_COMPONENTS + 4) s_cnt[threadIdx.x] = 0u;
  }
  const SInst I{n_comps, n_mats, s_comps, s_mats, s_tallies, g_inst->counters};
  __syncthreads();
  if (FEAT & F_SOLIDS) {  // stage the solids (poses, sizes, priorities) of every group and re-point the groups at the copy
    DSolid* s_solids = reinterpret_cast<DSolid*>(s_tallies + MCX_MAX_DETECTORS);
    int used = 0;
    for (int c = 1; c < n_comps; ++c) {
      if (s_comps[c].kind != MCX_SOLIDS) continue;
      const int ns = s_comps[c].u.solids.n_solids;
      const unsigned long long* src = reinterpret_cast<const unsigned long long*>(s_comps[c].u.solids.solids);
      unsigned long long* dst = reinterpret_cast<unsigned long long*>(s_solids + used);
      for (int k = threadIdx.x; k < ns * (int)(sizeof(DSolid) / 8); k += kBlock) dst[k] = src[k];
      __syncthreads();
      if (threadIdx.x == 0) s_comps[c].u.solids.solids = s_solids + used;
      used += ns;
    }
    __syncthreads();
  }
  const int lane = threadIdx.x & 31;
  // Staged trace (run_trace in mcx_host.cu): this launch is the part of the chain before (1) or after (2) a scattering
  // voxel volume, whose rays scatter_walk_kernel walks; stage 2 finds its rays, as many as stage 1 left, in the pool.
  constexpr bool STAGED = FEAT == (F_VOXELS | F_SCATTER);
  const int stage = STAGED ? A.stage : 0;
  const uint64_t first = A.first, n = (STAGED && stage == 2) ? (uint64_t)*A.pool_count : A.n, seed = A.seed;
  const uint32_t* __restrict__ order = A.order;
  mcx_ray_fate* __restrict__ dump = A.dump;
  // Lane scheduling (row a13): blocks pull tiles of A.tile consecutive positions from a global ticket counter (the
  // ticket of the next tile is fetched while the current one is traced), and the warps of a block pull 32-position
  // slices of the tile from a shared-memory counter, so neither a block nor a warp waits for a slower neighbour except
  // at the one barrier per tile.  With `order` set, position q holds the q-th ray of the chunk in detector-tile
  // order (kernels above); whole warps iterate together so the ballots are full-warp.
  const unsigned tile = A.tile;
  if (threadIdx.x == 0) {
    s_sched[0] = atomicAdd(A.ticket, 1u);
    s_sched[2] = 0u;
    // one read per block, before the barrier: every warp of the block must see the same value (it decides whether the
    // block takes the extra barrier after its first tile), whatever other blocks store meanwhile
    if (GATE) s_sched[5] = *reinterpret_cast<volatile unsigned int*>(A.gate_known);
  }
  __syncthreads();
  // Absorber gate (row a13, "warp-level compaction of absorbed rays").  Where the chain starts with slits, mirrors or
  // crystals (A.gate_max of them) and few rays survive those (c0 loses 84 % at its slit, c2 87 % at its two mirrors),
  // fresh rays are traced through components 1..gate only, and the offsets of the survivors go into a per-warp ring
  // in shared memory (ballot + prefix count); whenever the ring holds 32 the warp traces those through the WHOLE chain
  // from the source again, all lanes alive at the gate.  Legal because a ray is a pure function of its index
  // (slot-addressed draws), cheap because the replayed part is the source and a few apertures.  Rays absorbed up to
  // the gate are accounted in the first pass, everything a queued ray does in the second (it is counted there whatever
  // happens to it), so every ray is counted once.  The block picks the gate itself from what its first tile (traced
  // ungated) lost where: the first component after which at most 35 % of the rays are left, if there is one; the
  // choice (the first block's to finish a tile: one compare-and-swap decides for all) is left in the workspace, and
  // later launches on the instrument start with it.
  const unsigned known_gate = GATE ? s_sched[5] : 0u;
  int gate = known_gate ? (int)known_gate - 1 : 0;
  unsigned* ring = reinterpret_cast<unsigned*>(smem_raw + 128) + (threadIdx.x >> 5) * 64;
  unsigned ring_head = 0u, ring_n = 0u;  // warp-uniform
  // One warp-load of rays through components 1 .. (final_pass ? the end : the gate); see the loops below.
  auto trace_item = [&](const bool valid, uint64_t qi, bool final_pass) {
    int c_begin = 1, c_end = final_pass ? n_comps : gate + 1;
    Ray ray;
    int fate = MCX_FATE_MISSED;
    long long bin = -1;
    bool alive = valid;
    if (STAGED && stage == 2) {  // qi is a position in the pool: the ray as the walk stage left it
      c_begin = A.stage_comp + 1;
      if (valid) {
        const PoolRay& R = A.pool[qi];
        ray.r = {R.r[0], R.r[1], R.r[2]};
        ray.d = {R.d[0], R.d[1], R.d[2]};
        ray.E = R.E;
        ray.p = R.p;
        qi = R.offset;
      }
    } else {
      if (STAGED && stage == 1) {
        c_end = A.stage_comp;
        final_pass = false;
      }
      if (valid) sample_source(I.comps[0], seed, first + qi, ray);
    }
    for (int c = c_begin; c < c_end; ++c) {
      const DComponent& C = I.comps[c];
      const int kind = C.kind;  // warp-uniform
      bool pass = true, tally_now = false;
      const unsigned lanes_alive = (FEAT & F_SCATTER) ? __ballot_sync(0xffffffffu, alive) : 0u;  // (the legs of step 17 are walked by the warp)
      if ((FEAT & F_SOLIDS) && kind == MCX_SOLIDS) {  // whole warp: the mesh walk is warp-cooperative
        // (the walk without scattering is kept as its own function: the mesh kernel sits at the register limit)
        const int rc = (FEAT & F_SCATTER)
                           ? trace_solids_legs<(FEAT & F_MESH) != 0, (FEAT & F_PRIM) != 0, true>(I, C, c, ray, seed, first + qi, ep, tri_queue, alive,
                                                                                                 order != nullptr)
                           : trace_solids<(FEAT & F_MESH) != 0, (FEAT & F_PRIM) != 0>(I, C, ray, ep, tri_queue, alive, order != nullptr);
        if (alive && rc != 1) {
          pass = false;
          fate = MCX_FATE_DEGENERATE;
          if (rc < 0 && !DUMP) atomicAdd(&s_cnt[MCX_MAX_COMPONENTS + CNT_OVERFLOW], 1u);
        }
      } else if (alive) {
        if (kind == MCX_SLIT_RECT) {
          Vec3 h;
          pass = plane_hit(C.pose, ray, h) && fabs(h.x) <= C.u.slit.half_x && fabs(h.y) <= C.u.slit.half_y;
        } else if (kind == MCX_SLIT_CIRC) {
          Vec3 h;
          pass = plane_hit(C.pose, ray, h) && h.x * h.x + h.y * h.y <= C.u.slit.radius2;
        } else if ((FEAT & F_VOXELS) && kind == MCX_VOXELS) {
          trace_voxels<(FEAT & F_SCATTER) != 0>(I, C, c, ray, seed, first + qi, len_s, len_s + (size_t)I.n_mats * kBlock,
                                                len_s + (size_t)(I.n_mats + VC_COUNT) * kBlock, lanes_alive);
        } else if ((FEAT & F_OPTICS) && kind == MCX_MIRROR_ELLIPTIC) {
          pass = trace_mirror(C, ray);
        } else if ((FEAT & F_OPTICS) && kind == MCX_CRYSTAL_BRAGG) {
          pass = trace_crystal(C, ray);
        } else if ((FEAT & F_LENS) && kind == MCX_LENS_PARAB) {
          pass = trace_lens(I, C, ray);
        } else if (kind == MCX_DETECTOR) {
          const long long b = detector_bin(C, ray);
          if (b >= 0) {
            bin = b;
            fate = MCX_FATE_DETECTED;
            tally_now = true;
          } else {
            fate = MCX_FATE_MISSED;  // monitors do not absorb: the ray goes on
          }
        }
      }
      if (!DUMP && kind == MCX_DETECTOR) tally_add(I, tally_mode, tcache, (unsigned)C.u.detector.index, tally_now, bin, ray.p);  // whole warp
      if (alive) {
        if (kind != MCX_DETECTOR && pass) fate = MCX_FATE_MISSED;  // fate = what the last component said
        if (!pass) {
          alive = false;
          if (fate != MCX_FATE_DEGENERATE) fate = c;
        }
      }
      const unsigned alive_mask = __ballot_sync(0xffffffffu, alive);
      if (!DUMP) {
        // warp-aggregated ray accounting: one shared-memory add per warp and component
        const unsigned died = __ballot_sync(0xffffffffu, !pass && fate == c);
        if (lane == 0 && died) atomicAdd(&s_cnt[c], (unsigned)__popc(died));
      }
      if (alive_mask == 0u) break;
    }
    if (STAGED && stage == 1) {  // survivors go to the pool, packed
      const unsigned live = __ballot_sync(0xffffffffu, alive);
      unsigned at = 0u;
      if (lane == 0 && live) at = atomicAdd(A.pool_count, (unsigned)__popc(live));
      at = __shfl_sync(0xffffffffu, at, 0) + __popc(live & ((1u << lane) - 1u));
      if (alive) {
        PoolRay& R = A.pool[at];
        R.r[0] = ray.r.x; R.r[1] = ray.r.y; R.r[2] = ray.r.z;
        R.d[0] = ray.d.x; R.d[1] = ray.d.y; R.d[2] = ray.d.z;
        R.E = ray.E;
        R.p = ray.p;
        R.offset = qi;
        R.pad = 0ull;
      }
    }
    if (GATE && !final_pass) {  // survivors of the gate: queue their offsets for the full pass
      const unsigned live = __ballot_sync(0xffffffffu, alive);
      if (alive) ring[(ring_head + ring_n + __popc(live & ((1u << lane) - 1u))) & 63u] = (unsigned)qi;
      ring_n += __popc(live);
      __syncwarp();
    }
    if (DUMP) {
      if (valid && (final_pass || !alive)) {
        mcx_ray_fate f;
        f.fate = fate;
        f.reserved = 0;
        f.bin = fate == MCX_FATE_DETECTED ? bin : -1;
        f.p = ray.p;
        dump[qi] = f;
      }
    } else {
      const unsigned det = __ballot_sync(0xffffffffu, valid && final_pass && fate == MCX_FATE_DETECTED);
      const unsigned mis = __ballot_sync(0xffffffffu, valid && final_pass && fate == MCX_FATE_MISSED);
      const unsigned deg = __ballot_sync(0xffffffffu, valid && final_pass && fate == MCX_FATE_DEGENERATE);
      if (lane == 0) {
        if (det) atomicAdd(&s_cnt[MCX_MAX_COMPONENTS + CNT_DETECTED], (unsigned)__popc(det));
        if (mis) atomicAdd(&s_cnt[MCX_MAX_COMPONENTS + CNT_MISSED], (unsigned)__popc(mis));
        if (deg) atomicAdd(&s_cnt[MCX_MAX_COMPONENTS + CNT_DEGENERATE], (unsigned)__popc(deg));
      }
    }
  };
  if (!GATE) {
    for (unsigned it = 0;; ++it) {
      const unsigned par = it & 1u;
      const uint64_t tile_begin = (uint64_t)s_sched[par] * tile;
      if (tile_begin >= n) break;
      if (threadIdx.x == 0) {
        s_sched[par ^ 1u] = atomicAdd(A.ticket, 1u);
        s_sched[2 + (par ^ 1u)] = 0u;
      }
      for (;;) {
        unsigned slice = 0u;
        if (lane == 0) slice = atomicAdd(&s_sched[2 + par], 32u);
        slice = __shfl_sync(0xffffffffu, slice, 0);
        if (slice >= tile) break;
        const uint64_t q = tile_begin + slice + lane;
        if (q - lane >= n) break;  // the whole warp is beyond the end
        const bool valid = q < n;
        trace_item(valid, valid ? (order ? (uint64_t)order[q] : q) : 0, true);  // position in the chunk -> ray offset
      }
      __syncthreads();  // the tile is done and the next ticket is in place
    }
  } else {
    for (unsigned it = 0;; ++it) {
      const unsigned par = it & 1u;
      const uint64_t tile_begin = (uint64_t)s_sched[par] * tile;
      const bool last = tile_begin >= n;  // no tile left: drain the ring and leave
      if (!last && threadIdx.x == 0) {
        s_sched[par ^ 1u] = atomicAdd(A.ticket, 1u);
        s_sched[2 + (par ^ 1u)] = 0u;
      }
      for (;;) {
        bool valid, final_pass;
        uint64_t qi;
        if (GATE && (ring_n >= 32u || (last && ring_n > 0u))) {  // a warp-load of gate survivors
          const unsigned take = min(ring_n, 32u);
          valid = (unsigned)lane < take;
          qi = ring[(ring_head + lane) & 63u];
          ring_head = (ring_head + take) & 63u;
          ring_n -= take;
          final_pass = true;
        } else if (!last) {
          unsigned slice = 0u;
          if (lane == 0) slice = atomicAdd(&s_sched[2 + par], 32u);
          slice = __shfl_sync(0xffffffffu, slice, 0);
          if (slice >= tile) break;
          const uint64_t q = tile_begin + slice + lane;
          if (q - lane >= n) break;  // the whole warp is beyond the end
          valid = q < n;
          qi = valid ? (order ? (uint64_t)order[q] : q) : 0;  // position in the chunk -> ray offset
          final_pass = !GATE || gate == 0;
        } else {
          break;
        }
        trace_item(valid, qi, final_pass);
      }
      if (last) break;
      __syncthreads();  // the tile is done and the next ticket is in place
      if (GATE && it == 0u && known_gate == 0u) {
        if (threadIdx.x == 0) {
          const uint64_t left_in_range = n - tile_begin;
          const unsigned traced = left_in_range < tile ? (unsigned)left_in_range : tile;
          unsigned alive_after = traced, pick = 0u;
          for (int c = 1; c <= A.gate_max && pick == 0u; ++c) {
            alive_after -= s_cnt[c];
            if (100u * alive_after <= 35u * traced) pick = (unsigned)c;
          }
          const unsigned won = atomicCAS(A.gate_known, 0u, pick + 1u);  // 0: this block's choice stands
          s_sched[4] = won ? won - 1u : pick;
        }
        __syncthreads();
        gate = (int)s_sched[4];
      }
    }
  }
  // the last block to leave re-arms the ticket counter for the next launch
  if (threadIdx.x == 0) {
    __threadfence();
    if (atomicAdd(A.ticket + 1, 1u) == gridDim.x - 1) {
      A.ticket[0] = 0u;
      A.ticket[1] = 0u;
    }
  }
  if (!DUMP) {
    __syncthreads();
    tally_flush(I, tcache);
    if (threadIdx.x < MCX_MAX_COMPONENTS + 4) {
      const unsigned v = s_cnt[threadIdx.x];
      if (v) {
        const int slot = threadIdx.x < MCX_MAX_COMPONENTS ? threadIdx.x : n_comps + (threadIdx.x - MCX_MAX_COMPONENTS);
        if (threadIdx.x >= MCX_MAX_COMPONENTS || threadIdx.x < n_comps) atomicAdd(&I.counters[slot], (unsigned long long)v);
        if (threadIdx.x == MCX_MAX_COMPONENTS + CNT_OVERFLOW && A.host_flag) {
          // MCX_ERR_CAPACITY: tell the host (mapped pinned word) which reset epoch overflowed; include/mcx.h "Errors"
          *reinterpret_cast<volatile unsigned int*>(A.host_flag) = A.epoch + 1u;
          __threadfence_system();
        }
      }
    }
  }
}

// Step a14: tally finalise.  De-interleaves the 32-byte records into the three output arrays.
__global__ void __launch_bounds__(256) tally_read_kernel(const TallyBin* __restrict__ bins, uint64_t n_bins,
                                                         unsigned long long* __restrict__ N, double* __restrict__ P,
                                                         double* __restrict__ P2) {
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  for (uint64_t b = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; b < n_bins; b += stride) {
    const ulonglong4 rec = *reinterpret_cast<const ulonglong4*>(bins + b);
    N[b] = rec.x;
    P[b] = __longlong_as_double((long long)rec.y);
    P2[b] = __longlong_as_double((long long)rec.z);
  }
}

// Voxel volume from the interface layout [iz][iy][ix] into the traversal layout [i_a2 + 1][i_a1 + 1][i_fast + 1]
// (rows of `pitch` cells of 2 bytes: ID, run) with a guard border of kVoxelGuard around it.  Runs are filled in by
// voxel_runs_kernel.
__global__ void __launch_bounds__(256) voxel_relayout_kernel(const uint8_t* __restrict__ src, uint8_t* __restrict__ dst,
                                                             int nx, int ny, int nz, int fast, int a1, int a2, int pitch,
                                                             int n_mats) {
  const int n[3] = {nx, ny, nz};
  const long long total = (long long)(n[a2] + 2) * (n[a1] + 2) * pitch;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += stride) {
    const int jf = (int)(k % pitch) - 1;
    const long long rowi = k / pitch;
    const int j1 = (int)(rowi % (n[a1] + 2)) - 1, j2 = (int)(rowi / (n[a1] + 2)) - 1;
    unsigned v = kVoxelGuard;
    if (jf >= 0 && jf < n[fast] && j1 >= 0 && j1 < n[a1] && j2 >= 0 && j2 < n[a2]) {
      int idx[3];
      idx[fast] = jf; idx[a1] = j1; idx[a2] = j2;
      v = src[((long long)idx[2] * ny + idx[1]) * nx + idx[0]];
      if (v >= (unsigned)n_mats) v = 0u;  // not a material: vacuum (include/mcx.h)
    }
    reinterpret_cast<uint32_t*>(dst)[k] = v;  // run = radius = 0
  }
}

// run of a cell = number of cells following it along the row in direction run_dir that hold the same ID, capped at
// 255.  One thread per row, walking against run_dir.
__global__ void __launch_bounds__(256) voxel_runs_kernel(uint8_t* __restrict__ cells, long long n_rows, int pitch, int run_dir) {
  const long long row = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (row >= n_rows) return;
  uint8_t* r = cells + (long long)kVoxelCellBytes * row * pitch;
  int j = run_dir > 0 ? pitch - 1 : 0;
  unsigned prev_id = r[kVoxelCellBytes * j], run = 0u;
  for (int k = 1; k < pitch; ++k) {
    j -= run_dir;
    const unsigned id = r[kVoxelCellBytes * j];
    run = id == prev_id ? min(run + 1u, 255u) : 0u;
    r[kVoxelCellBytes * j + 1] = (uint8_t)run;
    prev_id = id;
  }
}

// Runs along one axis serve rays that follow it; a ray that crosses lateral faces every few slabs (the edge of a cone
// beam) or runs in any direction at all (after a scattering event, step 17) gets nothing from them.  Every cell therefore
// also carries the RADIUS of the largest cube of cells around it that holds its ID
// throughout (Chebyshev distance to the nearest cell of another ID, less one; capped at kVoxelRadiusMax): from a cell of
// radius R a ray may cross R - 1 slabs of its dominant axis, with whatever lateral faces come, without looking at
// anything (VoxWalk::step).  R = min(kVoxelRadiusMax, the chessboard distance to the nearest BOUNDARY cell) (a boundary cell
// has a neighbour, of its 26, of another ID; cells outside the arrays count as another ID).  Computed by doubling
// instead of kVoxelRadiusMax relaxation passes: with C_m(x) = "no boundary cell within chessboard distance m of x" (the
// cube of radius m around x is clear), C_0 is the boundary test, C_1 looks at the 26 neighbours' C_0, and
// C_2m(x) = AND of C_m at the eight cells x + (+-m, +-m, +-m), whose cubes cover the cube of radius 2m exactly.  Eight
// bits per cell (m = 0, 1, 2, 4, ..., 64) in one scratch byte, ping-ponged between two arrays.  Any other radius t = q + o,
// q the largest power of two <= t, is clear iff C_q holds at the eight cells x + (+-o, +-o, +-o) (o <= q - 1: the cubes
// overlap or touch), so R - 1 = the largest clear t <= 127 comes out of a seven-step binary search: about 120 byte
// look-ups per cell where the relaxation took up to 27 x 32.
constexpr int kVoxelRadiusMax = 128;  // a power of two <= 128 (eight C_m bits per scratch byte); 32 -> 64 -> 128: c7 +5 %, +2 %; c4, c9 +0 %
static_assert(kVoxelRadiusMax <= 128 && (kVoxelRadiusMax & (kVoxelRadiusMax - 1)) == 0, "C_m bits for m = 0, 1, 2, ..., kVoxelRadiusMax / 2 in one byte");

__device__ __forceinline__ long long vox_neighbour(long long k, int dx, int dy, int dz, int d0, int d1) {
  return k + dx + (long long)dy * d0 + (long long)dz * d0 * d1;
}

__global__ void __launch_bounds__(256) voxel_boundary_kernel(const uint8_t* __restrict__ cells, uint8_t* __restrict__ r0, int d0, int d1, int d2) {
  const long long total = (long long)d0 * d1 * d2, stride = (long long)gridDim.x * blockDim.x;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += stride) {
    const int x = (int)(k % d0), y = (int)((k / d0) % d1), z = (int)(k / ((long long)d0 * d1));
    const unsigned id = cells[kVoxelCellBytes * k];
    bool boundary = x == 0 || y == 0 || z == 0 || x == d0 - 1 || y == d1 - 1 || z == d2 - 1;
    if (!boundary)
      for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
          for (int dx = -1; dx <= 1; ++dx) boundary |= cells[kVoxelCellBytes * vox_neighbour(k, dx, dy, dz, d0, d1)] != id;
    r0[k] = boundary ? 0 : 1;  // bit 0 = C_0
  }
}

// bit `level` of rout = C_m from bit `level - 1` of rin (C_m/2, or C_0 for level 1); the lower bits are copied.
// level 1: the 26 neighbours; level >= 2: the eight cells at (+-off, +-off, +-off), off = m / 2.  (A cell whose own lower
// bit is clear cannot have the higher one; a cell with C_m set lies more than m cells inside the arrays, so the cells
// looked at exist.)
__global__ void __launch_bounds__(256) voxel_clear_pass_kernel(const uint8_t* __restrict__ rin, uint8_t* __restrict__ rout, int d0, int d1, int d2,
                                                               int level, int off) {
  const long long total = (long long)d0 * d1 * d2, stride = (long long)gridDim.x * blockDim.x;
  const unsigned below = 1u << (level - 1);
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += stride) {
    unsigned v = rin[k];
    if (v & below) {
      unsigned all = below;
      if (level == 1) {
        for (int dz = -1; dz <= 1; ++dz)
          for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) all &= rin[vox_neighbour(k, dx, dy, dz, d0, d1)];
      } else {
        for (int c = 0; c < 8; ++c)
          all &= rin[vox_neighbour(k, (c & 1) ? off : -off, (c & 2) ? off : -off, (c & 4) ? off : -off, d0, d1)];
      }
      if (all) v |= 1u << level;
    }
    rout[k] = (uint8_t)v;
  }
}

// bits: the six C_m bits of every cell (above).  Writes the radius into the third byte of every cell and, if asked, the
// compact cell (DVoxels::cmap).
__global__ void __launch_bounds__(256) voxel_radius_store_kernel(const uint8_t* __restrict__ bits, uint8_t* __restrict__ cells, uint8_t* __restrict__ cmap,
                                                                 int d0, int d1, int d2) {
  const long long total = (long long)d0 * d1 * d2, stride = (long long)gridDim.x * blockDim.x;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += stride) {
    unsigned R = 0u;
    if (bits[k] & 1u) {  // not a boundary cell: R - 1 = the largest clear radius t in 0 .. kVoxelRadiusMax - 1
      const int x = (int)(k % d0), y = (int)((k / d0) % d1), z = (int)(k / ((long long)d0 * d1));
      int t = 0;
      for (int step = kVoxelRadiusMax / 2; step >= 1; step >>= 1) {
        const int cand = t + step;  // <= kVoxelRadiusMax - 1
        const int lg = 31 - __clz(cand), q = 1 << lg, o = cand - q;
        // the cube of radius cand must lie inside the arrays' interior (their outermost cells are boundary cells)
        bool clear = x - cand >= 1 && x + cand <= d0 - 2 && y - cand >= 1 && y + cand <= d1 - 2 && z - cand >= 1 && z + cand <= d2 - 2;
        if (clear) {
          unsigned all = 1u << (lg + 1);  // the bit of C_q
          if (o == 0) all &= bits[k];
          else
            for (int c = 0; c < 8; ++c) all &= bits[vox_neighbour(k, (c & 1) ? o : -o, (c & 2) ? o : -o, (c & 4) ? o : -o, d0, d1)];
          clear = all != 0u;
        }
        if (clear) t = cand;
      }
      R = (unsigned)t + 1u;
    }
    cells[kVoxelCellBytes * k + 2] = (uint8_t)R;
    if (cmap) {  // the compact cell (DVoxels::cmap): the largest code whose radius is <= R
      const unsigned id = cells[kVoxelCellBytes * k];
      const unsigned code = R <= 6u ? R : R < 8u ? 6u : R < 10u ? 7u : R < 12u ? 8u : R < 16u ? 9u : R < 24u ? 10u : R < 32u ? 11u : R < 64u ? 12u : R < 128u ? 13u : 14u;
      cmap[k] = (uint8_t)(id == kVoxelGuard ? 0xF0u : (id | (code << 4)));
    }
  }
}

// FP64 pipe probe for the ALU roofline: 8 independent DFMA chains per thread.
__global__ void __launch_bounds__(256) probe_dfma_kernel(double* sink, long long n_iters) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1.0, a2 = a0 + 2.0, a3 = a0 + 3.0, a4 = a0 + 4.0, a5 = a0 + 5.0, a6 = a0 + 6.0,
         a7 = a0 + 7.0;
  const double m = 1.0000000001, c = 1e-12;
  for (long long k = 0; k < n_iters; ++k) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}


template <int FEAT, bool DUMP, bool GATE>
cudaError_t launch_one(const DInstrument* d_inst, int n_mats, const TraceArgs& A, cudaStream_t stream, int n_sm) {
  const size_t smem = 128 + (GATE ? kRingBytes : 0) + (size_t)A.n_comps * sizeof(DComponent) + (size_t)A.n_mats * sizeof(DMaterial) +
                      MCX_MAX_DETECTORS * sizeof(void*) +
                      ((FEAT & F_SOLIDS) ? (size_t)A.n_solids * sizeof(DSolid) + (size_t)A.cap_endpoints * kBlock * 9 : 0) +
                      ((FEAT & F_MESH) ? (size_t)kTriQueue * kBlock * sizeof(unsigned) : 0) +
                      ((FEAT & F_VOXELS) ? (size_t)(n_mats + VC_COUNT + ((FEAT & F_SCATTER) ? n_mats : 0)) * kBlock * sizeof(double) : 0) +
                      ((!DUMP && !(FEAT & (F_SOLIDS | F_VOXELS)) && A.tally_cache_log2 > 0) ? ((size_t)32 << A.tally_cache_log2) : 0);
  static std::atomic<unsigned long long> configured{0ull};  // bit d: the opt-in below was made on device d
  int blocks_per_sm = 1, dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev >= 64 || !((configured.load(std::memory_order_relaxed) >> dev) & 1ull)) {
    e = cudaFuncSetAttribute(trace_kernel<FEAT, DUMP, GATE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    if (dev < 64) configured.fetch_or(1ull << dev, std::memory_order_relaxed);
  }
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, trace_kernel<FEAT, DUMP, GATE>, kBlock, smem);
  if (e != cudaSuccess) return e;
  if (blocks_per_sm < 1) return cudaErrorInvalidConfiguration;
  const uint64_t full = (uint64_t)n_sm * blocks_per_sm;  // one resident wave: a multiple of the SM count
  TraceArgs B = A;
  B.tile = kTileMax;  // at least ~4 tiles per resident block, so that the tail of the launch is short
  while (B.tile > (unsigned)kBlock && A.n / B.tile < 2 * full) B.tile >>= 1;
  const uint64_t want = (A.n + B.tile - 1) / B.tile;
  const unsigned grid = (unsigned)(want < full ? (want ? want : 1) : full);
  trace_kernel<FEAT, DUMP, GATE><<<grid, kBlock, smem, stream>>>(d_inst, B);
  return cudaGetLastError();
}

std::atomic<int> g_sm_of_device[64];  // SM count per device, 0 = not asked yet

// SM count of the current device
cudaError_t sm_count(int* n_sm) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 64) {
    const int known = g_sm_of_device[dev].load(std::memory_order_relaxed);
    if (known) { *n_sm = known; return cudaSuccess; }
  }
  e = cudaDeviceGetAttribute(n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess && dev < 64) g_sm_of_device[dev].store(*n_sm, std::memory_order_relaxed);
  return e;
}

}  // namespace

cudaError_t launch_trace(const DInstrument* d_inst, int features, int n_mats, const TraceArgs& A, cudaStream_t stream) {
  int g_n_sm = 0;
  cudaError_t e = sm_count(&g_n_sm);
  if (e != cudaSuccess) return e;
  if (A.n == 0) return cudaSuccess;
  if (A.n > ((uint64_t)1 << 40)) return cudaErrorInvalidValue;  // tile tickets are 32-bit; the host chunks below this
  // the absorber gate is compiled into the tallying kernels of the chains that can start with absorbers and stay light
  // (no mesh, no voxels: those run at the register limit and their chains start at the sample)
#define MCX_DISPATCH(F)                                                              \
  return A.dump ? launch_one<F, true, false>(d_inst, n_mats, A, stream, g_n_sm)      \
                : launch_one<F, false, false>(d_inst, n_mats, A, stream, g_n_sm);
#define MCX_DISPATCH_GATED(F)                                                        \
  return A.dump         ? launch_one<F, true, false>(d_inst, n_mats, A, stream, g_n_sm)  \
         : A.gate_max > 0 ? launch_one<F, false, true>(d_inst, n_mats, A, stream, g_n_sm) \
                          : launch_one<F, false, false>(d_inst, n_mats, A, stream, g_n_sm);
  switch (features) {
    case 0: MCX_DISPATCH_GATED(0)
    case F_SOLIDS | F_PRIM: MCX_DISPATCH_GATED(F_SOLIDS | F_PRIM)
    case F_SOLIDS | F_MESH: MCX_DISPATCH(F_SOLIDS | F_MESH)
    case F_SOLIDS | F_MESH | F_PRIM: MCX_DISPATCH(F_SOLIDS | F_MESH | F_PRIM)
    case F_VOXELS: MCX_DISPATCH(F_VOXELS)
    case F_VOXELS | F_SCATTER: MCX_DISPATCH(F_VOXELS | F_SCATTER)
    case F_OPTICS: MCX_DISPATCH_GATED(F_OPTICS)
    case F_LENS: MCX_DISPATCH_GATED(F_LENS)
    default: MCX_DISPATCH_GATED(F_ALL)
  }
#undef MCX_DISPATCH
#undef MCX_DISPATCH_GATED
}

// The walk stage of a staged trace: at most n_max records are in the pool (the count itself is in device memory).
// (internal linkage: the local static of a template with external linkage is ONE object for every shared library of the
// process that holds the template, and the strict build's kernels would go without their own opt-in)
template <int CELL>
static cudaError_t launch_scatter_walk_as(const DInstrument* d_inst, const WalkArgs& A, uint64_t n_max, cudaStream_t stream, int n_sm) {
  int dev = 0, blocks_per_sm = 1;
  const size_t smem = (size_t)(2 * A.n_mats + VC_COUNT) * kBlock * sizeof(double) + sizeof(DComponent) + (size_t)A.n_mats * sizeof(DMaterial);
  static std::atomic<unsigned long long> configured{0ull};  // bit d: the opt-in below was made on device d
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev >= 64 || !((configured.load(std::memory_order_relaxed) >> dev) & 1ull)) {
    e = cudaFuncSetAttribute(scatter_walk_kernel<CELL>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    if (dev < 64) configured.fetch_or(1ull << dev, std::memory_order_relaxed);
  }
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, scatter_walk_kernel<CELL>, kBlock, smem);
  if (e != cudaSuccess) return e;
  if (blocks_per_sm < 1) return cudaErrorInvalidConfiguration;
  const uint64_t full = (uint64_t)n_sm * blocks_per_sm, per_block = (uint64_t)kWalkRange * (kBlock / 32), want = (n_max + per_block - 1) / per_block;
  scatter_walk_kernel<CELL><<<(unsigned)(want < full ? want : full), kBlock, smem, stream>>>(d_inst, A);
  return cudaGetLastError();
}

cudaError_t launch_scatter_walk(const DInstrument* d_inst, const WalkArgs& A, uint64_t n_max, cudaStream_t stream) {
  int g_n_sm = 0;
  const cudaError_t e = sm_count(&g_n_sm);
  if (e != cudaSuccess) return e;
  if (n_max == 0) return cudaSuccess;
  return A.compact ? launch_scatter_walk_as<1>(d_inst, A, n_max, stream, g_n_sm)
                   : launch_scatter_walk_as<kVoxelCellBytes>(d_inst, A, n_max, stream, g_n_sm);
}

// count -> scan -> scatter of one chunk (n <= 2^32 - 1 rays, 4^g buckets); cnt must be zero on entry
cudaError_t launch_sort(uint64_t first, uint32_t n, uint64_t seed, int g, unsigned int* cnt, unsigned int* bsum,
                        uint32_t* order, cudaStream_t stream) {
  int g_n_sm = 0;
  cudaError_t e = sm_count(&g_n_sm);
  if (e != cudaSuccess) return e;
  const uint32_t n_buckets = 1u << (2 * g);
  const int n_scan_blocks = (int)((n_buckets + kScanBlock - 1) / kScanBlock);
  if (g < 1 || g > MCX_SORT_MAX_G || n_scan_blocks > kMaxScanBlocks) return cudaErrorInvalidValue;
  const unsigned want = (n + 255u) / 256u;
  const unsigned grid = want < (unsigned)g_n_sm * 8u ? (want ? want : 1u) : (unsigned)g_n_sm * 8u;
  sort_count_kernel<<<grid, 256, 0, stream>>>(first, n, seed, g, cnt);
  sort_scan_kernel<<<n_scan_blocks, 256, 0, stream>>>(cnt, n_buckets, bsum);
  sort_scatter_kernel<<<grid, 256, 0, stream>>>(first, n, seed, g, cnt, bsum, n_scan_blocks, order);
  return cudaGetLastError();
}

cudaError_t launch_tally_read(const TallyBin* bins, uint64_t n_bins, unsigned long long* N, double* p, double* p2,
                              cudaStream_t stream) {
  int g_n_sm = 0;
  cudaError_t e = sm_count(&g_n_sm);
  if (e != cudaSuccess) return e;
  if (n_bins == 0) return cudaSuccess;
  const uint64_t want = (n_bins + 255) / 256;
  const unsigned grid = (unsigned)(want < (uint64_t)g_n_sm * 8 ? want : (uint64_t)g_n_sm * 8);
  tally_read_kernel<<<grid, 256, 0, stream>>>(bins, n_bins, N, p, p2);
  return cudaGetLastError();
}

cudaError_t launch_voxel_relayout(const uint8_t* src, uint8_t* dst, int nx, int ny, int nz, int fast, int a1, int a2,
                                  int pitch, int run_dir, int n_mats, cudaStream_t stream) {
  int g_n_sm = 0;
  cudaError_t e = sm_count(&g_n_sm);
  if (e != cudaSuccess) return e;
  voxel_relayout_kernel<<<g_n_sm * 8, 256, 0, stream>>>(src, dst, nx, ny, nz, fast, a1, a2, pitch, n_mats);
  const int n[3] = {nx, ny, nz};
  const long long n_rows = (long long)(n[a2] + 2) * (n[a1] + 2);
  voxel_runs_kernel<<<(unsigned)((n_rows + 255) / 256), 256, 0, stream>>>(dst, n_rows, pitch, run_dir);
  return cudaGetLastError();
}

// cells: the traversal layout of d0 x d1 x d2 cells {ID, .}; scratch: 2 * d0 * d1 * d2 bytes.  Leaves the radius in the
// second byte of every cell.
cudaError_t launch_voxel_radius(uint8_t* cells, uint8_t* scratch, uint8_t* cmap, int d0, int d1, int d2, cudaStream_t stream) {
  int g_n_sm = 0;
  cudaError_t e = sm_count(&g_n_sm);
  if (e != cudaSuccess) return e;
  const long long total = (long long)d0 * d1 * d2;
  uint8_t* a = scratch;
  uint8_t* b = scratch + total;
  voxel_boundary_kernel<<<g_n_sm * 16, 256, 0, stream>>>(cells, a, d0, d1, d2);
  for (int level = 1; (1 << (level - 1)) < kVoxelRadiusMax; ++level) {  // C_1, C_2, C_4, ..., C_(kVoxelRadiusMax / 2)
    voxel_clear_pass_kernel<<<g_n_sm * 16, 256, 0, stream>>>(a, b, d0, d1, d2, level, level == 1 ? 1 : (1 << (level - 2)));
    uint8_t* t = a; a = b; b = t;
  }
  voxel_radius_store_kernel<<<g_n_sm * 16, 256, 0, stream>>>(a, cells, cmap, d0, d1, d2);
  return cudaGetLastError();
}

// Tally probe for the atomics roofline: every thread does n_iters rounds of the three reductions of step 14 (u64 count,
// two fp64 sums) into one pseudo-random 32-byte record of a table of n_records (a power of two).
__global__ void __launch_bounds__(256) probe_tally_kernel(TallyBin* table, unsigned long long mask, long long n_iters) {
  unsigned long long x = ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) * 0x9E3779B97F4A7C15ull + 0x2545F4914F6CDD1Dull;
  for (long long k = 0; k < n_iters; ++k) {
    x ^= x >> 12; x ^= x << 25; x ^= x >> 27;  // xorshift64*
    TallyBin* rec = table + ((x * 0x2545F4914F6CDD1Dull) >> 20 & mask);
    atomicAdd(&rec->N, 1ull);
    atomicAdd(&rec->P, 0.5);
    atomicAdd(&rec->P2, 0.25);
  }
}

cudaError_t launch_probe_tally(void* table, unsigned long long n_records, int n_blocks, long long n_iters, cudaStream_t stream) {
  probe_tally_kernel<<<n_blocks, 256, 0, stream>>>(reinterpret_cast<TallyBin*>(table), n_records - 1, n_iters);
  return cudaGetLastError();
}

// L2 / L1 sector probe for the roofline of the mesh walk: independent loads of pseudo-random
// aligned 32-byte sectors (one BVH node) through the read-only path, four in flight per thread.
__global__ void __launch_bounds__(256) probe_l2_kernel(const uint4* __restrict__ table, unsigned long long sector_mask,
                                                       uint32_t* __restrict__ sink, long long n_iters) {
  unsigned long long x = ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) * 0x9E3779B97F4A7C15ull + 0x2545F4914F6CDD1Dull;
  unsigned acc = 0u;
  for (long long k = 0; k < n_iters; k += 4) {
    uint4 v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      x ^= x >> 12; x ^= x << 25; x ^= x >> 27;  // xorshift64*
      v[u] = __ldg(table + 2 * (((x * 0x2545F4914F6CDD1Dull) >> 24) & sector_mask));
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) acc += v[u].x ^ v[u].w;
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// Dependent-load latency probe: sector i of the table holds the index of the sector to read next (a full-period
// linear congruential permutation of the n sectors, written by probe_chain_init_kernel).
__global__ void __launch_bounds__(256) probe_chain_init_kernel(unsigned long long* __restrict__ table, unsigned long long n_sectors) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_sectors; i += stride)
    table[4 * i] = (i * 1664525ull + 1013904223ull) & (n_sectors - 1);  // Hull-Dobell: a = 1 mod 4, c odd
}
__global__ void __launch_bounds__(256) probe_latency_kernel(const unsigned long long* __restrict__ table, unsigned long long n_sectors,
                                                            uint32_t* __restrict__ sink, long long n_iters) {
  unsigned long long i = (((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) * 0x9E3779B97F4A7C15ull >> 20) & (n_sectors - 1);
  for (long long k = 0; k < n_iters; ++k) {
    unsigned long long nxt;
    asm volatile("ld.global.nc.u64 %0, [%1];" : "=l"(nxt) : "l"(table + 4 * i));
    i = nxt;
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = (uint32_t)i;
}

cudaError_t launch_probe_l2(const void* table, unsigned long long n_bytes, uint32_t* sink, int n_blocks, long long n_iters,
                            cudaStream_t stream) {
  probe_l2_kernel<<<n_blocks, 256, 0, stream>>>(reinterpret_cast<const uint4*>(table), n_bytes / 32 - 1, sink, n_iters);
  return cudaGetLastError();
}

cudaError_t launch_probe_latency(void* table, unsigned long long n_bytes, uint32_t* sink, int n_blocks, int n_threads,
                                 long long n_iters, cudaStream_t stream) {
  const unsigned long long n_sectors = n_bytes / 32;
  probe_chain_init_kernel<<<1024, 256, 0, stream>>>(reinterpret_cast<unsigned long long*>(table), n_sectors);
  probe_latency_kernel<<<n_blocks, n_threads, 0, stream>>>(reinterpret_cast<const unsigned long long*>(table), n_sectors, sink, n_iters);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// Contrast-to-noise ratio of PAPER.md:257 Eq. (1) (include/mcx.h, mcx_cnr).  One block per energy bin sums, over the pixels
// of the two regions, the bin's weight sums and its McXtrace error estimates (fixed-order tree: deterministic); one more
// block fits the least-squares line through the bins above e_fit_min.
// ------------------------------------------------------------------------------------------------------------
struct CnrRegions {
  int mat[4], ref[4];  // x0, x1, y0, y1
};

__device__ __forceinline__ double block_sum(double v, double* s_red) {
  __syncthreads();
  s_red[threadIdx.x] = v;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) s_red[threadIdx.x] += s_red[threadIdx.x + o];
    __syncthreads();
  }
  return s_red[0];
}

__global__ void __launch_bounds__(256) cnr_kernel(const unsigned long long* __restrict__ N, const double* __restrict__ P,
                                                  const double* __restrict__ P2, int nx, int ne, CnrRegions R,
                                                  double* __restrict__ cnr_out) {
  __shared__ double s_red[256];
  const int e = blockIdx.x;
  double mean[2], var[2];
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int* q = r == 0 ? R.mat : R.ref;
    const int w = q[1] - q[0], n_pix = w * (q[3] - q[2]);
    double sp = 0.0, sv = 0.0;
    for (int k = threadIdx.x; k < n_pix; k += 256) {
      const int ix = q[0] + k % w, iy = q[2] + k / w;
      const size_t b = ((size_t)iy * nx + ix) * ne + e;
      const double n = (double)N[b], p = P[b];
      sp += p;
      sv += n > 1.0 ? n / (n - 1.0) * fabs(P2[b] - (p / n) * (p / n)) : p * p;
    }
    mean[r] = block_sum(sp, s_red) / (double)n_pix;
    var[r] = block_sum(sv, s_red) / ((double)n_pix * (double)n_pix);
  }
  if (threadIdx.x == 0) {
    const double noise = sqrt(var[0] + var[1]);
    cnr_out[e] = noise > 0.0 ? fabs(mean[0] - mean[1]) / noise : 0.0;
  }
}

__global__ void __launch_bounds__(256) cnr_fit_kernel(const double* __restrict__ cnr, int ne, double emin, double emax, double e_fit_min,
                                                      double* __restrict__ fit_out) {
  __shared__ double s_red[256];
  const double de = (emax - emin) / (double)ne;
  double cnt = 0.0, sx = 0.0, sy = 0.0;
  for (int e = threadIdx.x; e < ne; e += 256) {
    const double x = emin + ((double)e + 0.5) * de;
    if (x >= e_fit_min) { cnt += 1.0; sx += x; sy += cnr[e]; }
  }
  const double n = block_sum(cnt, s_red);
  const double xm = block_sum(sx, s_red) / fmax(n, 1.0), ym = block_sum(sy, s_red) / fmax(n, 1.0);
  double sxy = 0.0, sxx = 0.0;
  for (int e = threadIdx.x; e < ne; e += 256) {
    const double x = emin + ((double)e + 0.5) * de;
    if (x >= e_fit_min) { sxy += (x - xm) * (cnr[e] - ym); sxx += (x - xm) * (x - xm); }
  }
  const double txy = block_sum(sxy, s_red), txx = block_sum(sxx, s_red);
  if (threadIdx.x == 0) {
    const double slope = (n >= 2.0 && txx > 0.0) ? txy / txx : 0.0;
    fit_out[0] = n >= 2.0 ? ym - slope * xm : 0.0;
    fit_out[1] = slope;
  }
}

cudaError_t launch_cnr(const unsigned long long* N, const double* p, const double* p2, int nx, int ny, int ne, const int* region_mat,
                       const int* region_ref, double emin, double emax, double e_fit_min, double* cnr_out, double* fit_out,
                       cudaStream_t stream) {
  (void)ny;
  CnrRegions R;
  for (int k = 0; k < 4; ++k) { R.mat[k] = region_mat[k]; R.ref[k] = region_ref[k]; }
  cnr_kernel<<<ne, 256, 0, stream>>>(N, p, p2, nx, ne, R, cnr_out);
  cnr_fit_kernel<<<1, 256, 0, stream>>>(cnr_out, ne, emin, emax, e_fit_min, fit_out);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// mcx_cnr_static (include/mcx.h): tally finalise + CNR for callers that cannot allocate device memory.  The
// intermediate arrays (N, p, p2 of the detector, the CNR per energy bin, the fit) live in this file-scope array: 6 MiB on
// every GPU that loads the library, until exit.  Shared by all calls, keeps the last call's contents: every byte a call
// reads it has written itself first (tally_read_kernel fills N, p, p2 [0, n_bins), cnr_kernel cnr [0, ne), the fit its 2),
// so nothing needs clearing; two calls in flight on the GPU at once would race on it (the header says so).
// In host code the array's name is a stand-in, not an address: the kernels get the device address from
// cudaGetSymbolAddress, asked once per device with that device current.
// ------------------------------------------------------------------------------------------------------------
constexpr size_t kCnrStaticOffCnr = (size_t)MCX_CNR_STATIC_MAX_BINS * 24;
constexpr size_t kCnrStaticBytes = kCnrStaticOffCnr + ((size_t)MCX_CNR_STATIC_MAX_NE + 2) * sizeof(double);
static __device__ __align__(256) unsigned char g_cnr_static_scratch[kCnrStaticBytes];
static std::atomic<unsigned char*> g_cnr_static_addr[64];  // per device, null = not asked yet

cudaError_t launch_cnr_static(const TallyBin* bins, uint64_t n_bins, int nx, int ny, int ne, const int* region_mat, const int* region_ref,
                              double emin, double emax, double e_fit_min, double* cnr_out, double* fit_out, cudaStream_t stream) {
  if (n_bins > (uint64_t)MCX_CNR_STATIC_MAX_BINS || ne > MCX_CNR_STATIC_MAX_NE || n_bins != (uint64_t)nx * ny * ne) return cudaErrorInvalidValue;
  int dev = 0, n_sm = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  unsigned char* scratch = dev < 64 ? g_cnr_static_addr[dev].load(std::memory_order_acquire) : nullptr;
  if (!scratch) {
    e = cudaGetSymbolAddress((void**)&scratch, g_cnr_static_scratch);  // this device's copy of the array
    if (e != cudaSuccess) return e;
    if (!scratch) return cudaErrorInvalidSymbol;
    if (dev < 64) g_cnr_static_addr[dev].store(scratch, std::memory_order_release);
  }
  e = sm_count(&n_sm);
  if (e != cudaSuccess) return e;
  unsigned long long* N = reinterpret_cast<unsigned long long*>(scratch);
  double* P = reinterpret_cast<double*>(scratch) + n_bins;
  double* P2 = P + n_bins;
  double* cnr = reinterpret_cast<double*>(scratch + kCnrStaticOffCnr);
  double* fit = cnr + MCX_CNR_STATIC_MAX_NE;
  const uint64_t want = (n_bins + 255) / 256;
  const unsigned grid = (unsigned)(want < (uint64_t)n_sm * 8 ? want : (uint64_t)n_sm * 8);
  tally_read_kernel<<<grid, 256, 0, stream>>>(bins, n_bins, N, P, P2);
  CnrRegions R;
  for (int k = 0; k < 4; ++k) { R.mat[k] = region_mat[k]; R.ref[k] = region_ref[k]; }
  cnr_kernel<<<ne, 256, 0, stream>>>(N, P, P2, nx, ne, R, cnr);
  cnr_fit_kernel<<<1, 256, 0, stream>>>(cnr, ne, emin, emax, e_fit_min, fit);
  e = cudaGetLastError();
  // outputs: host (pinned if the copy is to be asynchronous) or device memory, told apart by the unified address space
  if (e == cudaSuccess) e = cudaMemcpyAsync(cnr_out, cnr, (size_t)ne * sizeof(double), cudaMemcpyDefault, stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(fit_out, fit, 2 * sizeof(double), cudaMemcpyDefault, stream);
  return e;
}

cudaError_t launch_probe_dfma(double* sink, int n_blocks, long long n_iters, cudaStream_t stream) {
  probe_dfma_kernel<<<n_blocks, 256, 0, stream>>>(sink, n_iters);
  return cudaGetLastError();
}

}  // namespace mcx
