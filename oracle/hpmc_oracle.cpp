// =====================================================================================
// hpmc_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, sequential CPU restatement of the implicit-depletant hard-particle Monte
// Carlo trial move of arXiv 1508.07077 (Glaser, Karas, Glotzer), written from PAPER.md.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may load this library.  It shares no source, header, table or helper with the CUDA
// library under paper_1508_07077_b200/csrc/.
//
// What follows the paper (PAPER.md line numbers):
//   * move rule: propose M->M', draw N_p ~ Poisson(z_p V) depletants, reject if one of
//     them overlaps the new configuration only            -- Sec. III.B  L64-68, Fig. 2 L72
//   * insertion volume V_0 = circumsphere of diameter d_colloid + d_depletant around the
//     NEW pose; depletants overlapping the old pose or other colloids are ignored
//                                                         -- Sec. III.C  L117, L156
//   * configurational bias, Eq. (16)                      -- Sec. III.D  L170-174
//   * checkerboard: active cells separated by inactive ones, colouring permuted, grid
//     shifted, particles confined to their cell           -- Sec. III.E  L180
// Where the paper is silent (RNG, samplers, shape tests, Eq. 16's dropped prime ...) the
// readings R1..R23 of DESIGN.md ("Readings of the paper") are implemented; every function
// below names the reading it follows.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known answers; Poisson mean/variance
// and pmf; ball-sample moments; Steiner volumes of the dilated shapes; isolated-colloid
// acceptance exp(-n_R dV); Asakura-Oosawa two-sphere ratio test; CB forward/reverse ratio;
// explicit-depletant brute force; convex overlap test vs closed forms and an fp64 convex
// program.  PARITY UNPINNED BY THE PAPER (fixed by this file's definition only): the 0/0
// rule of Eq. 16 (R-G3), the particular samplers' bit patterns, and outcomes of the
// iterative convex test inside its 1e-5 contact band.
//
// Options (oracle_set_flags; default 0 = the path above, untouched by them): SURVEY 8(f) NEXT-1, the shell-restricted
// insertion volume of L158 (reading R-N1 of DESIGN.md), and NEXT-4, the exact Rosenbluth form of the configurational
// bias weight (refs 27, 28, 33; reading R-N4).  Their pins: radial cdf and isotropy of the shell sampler, cube-root
// accuracy, isolated-colloid and Asakura-Oosawa ratio tests with the shell on (and a literal-hard-core shell, built as a
// throw-away mutant of this file by the test, failing them), forward/reverse ratio of the Rosenbluth form to 3 sigma with no systematic allowance.
//
// Arithmetic: all pose arithmetic is IEEE fp32 with contraction OFF (-ffp-contract=off);
// an FMA is used only where fmaf() is written.  Integers u32/u64.  fp64 only for the
// Poisson threshold table.
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ----------------------------------------------------------------------------- Philox
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), R-S20.  Counter (c0..c3), key (k0,k1).
struct U4 { uint32_t v[4]; };

static inline U4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                               uint32_t k0, uint32_t k1) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)M0 * c0;
    const uint64_t p1 = (uint64_t)M1 * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  return U4{{c0, c1, c2, c3}};
}

// stream purposes, R-S20
enum { P_SWEEP = 0, P_SELECT = 1, P_MOVE = 2, P_NDEP = 3, P_DEPPOS = 4, P_CBPOS = 5, P_ACCEPT = 6, P_FREEVOL = 7 };

static inline uint32_t word3(uint32_t purpose, uint32_t colour, uint32_t attempt) {
  return purpose + (colour << 8) + (attempt << 16);
}

// R-S4: u32 -> symmetric unit variate s = 2u-1, u = ((x>>9)+0.5)/2^23; every step exact.
static inline float sym_unit(uint32_t x) {
  return ((float)(x >> 9) + 0.5f) * 2.384185791015625e-07f /* 2^-22 */ - 1.0f;
}
// R-S4: u in (0,1)
static inline float unit01(uint32_t x) {
  return ((float)(x >> 9) + 0.5f) * 1.1920928955078125e-07f /* 2^-23 */;
}
static inline uint32_t mulhi32(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) >> 32); }

// ----------------------------------------------------------------------------- vectors
struct V3 { float x, y, z; };
static inline V3 operator+(V3 a, V3 b) { return V3{a.x + b.x, a.y + b.y, a.z + b.z}; }
static inline V3 operator-(V3 a, V3 b) { return V3{a.x - b.x, a.y - b.y, a.z - b.z}; }
static inline V3 operator*(V3 a, float s) { return V3{a.x * s, a.y * s, a.z * s}; }
static inline V3 neg(V3 a) { return V3{-a.x, -a.y, -a.z}; }
// dot product: the one place an FMA chain is used (written identically on the device)
static inline float dot3(V3 a, V3 b) { return fmaf(a.z, b.z, fmaf(a.y, b.y, a.x * b.x)); }
static inline V3 cross3(V3 a, V3 b) {
  return V3{a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
struct Q4 { float w, x, y, z; };

// R-S19: body z axis in the space frame, third column of the rotation matrix of q.
static inline V3 quat_axis(Q4 q) {
  return V3{2.0f * (q.x * q.z + q.w * q.y), 2.0f * (q.y * q.z - q.w * q.x),
            1.0f - 2.0f * (q.x * q.x + q.y * q.y)};
}
// R-S6: q' = normalise((1,v) (x) q)   (Cayley rotation; left = space-frame multiplication)
static inline Q4 rotate_cayley(Q4 q, V3 v) {
  Q4 p;
  p.w = q.w - ((v.x * q.x + v.y * q.y) + v.z * q.z);
  p.x = (q.x + v.x * q.w) + (v.y * q.z - v.z * q.y);
  p.y = (q.y + v.y * q.w) + (v.z * q.x - v.x * q.z);
  p.z = (q.z + v.z * q.w) + (v.x * q.y - v.y * q.x);
  const float n2 = (p.w * p.w + p.x * p.x) + (p.y * p.y + p.z * p.z);
  const float n = sqrtf(n2);
  return Q4{p.w / n, p.x / n, p.y / n, p.z / n};
}

// ----------------------------------------------------------------------------- shapes
enum { SH_SPHERE = 0, SH_HALFBALL = 1, SH_SPHERODISK = 2, SH_ELLIPSOID = 3, SH_TETRAHEDRON = 4 };

struct Geo {                 // derived fp32 constants, R-0
  int shape;
  float dcirc, sigma_d, L, halfL, dmax_cap;
  float rd;                  // depletant radius
  float Rins, Rins2;         // insertion-sphere radius (dcirc+sigma_d)/2 and its square
  float dcirc2;              // circumsphere contact distance squared
  float rcut2;               // neighbour pre-filter
  float Rh;                  // half-ball radius
  float cen;                 // half-ball interior-point offset 3Rh/8
  float adisk, sdisk;        // spherodisk: disk radius, rounding radius; ellipsoid: equatorial and polar semi-axes A >= C
  float rs2;                 // (sdisk+rd)^2
  float rd2;                 // rd^2
};

static Geo make_geo(int shape, float sigma_c, float disk_a, float disk_s, float sigma_d, float L,
                    float dmax_cap) {
  Geo g;
  g.shape = shape; g.dcirc = sigma_c; g.sigma_d = sigma_d; g.L = L; g.halfL = 0.5f * L;
  g.dmax_cap = dmax_cap;
  g.rd = 0.5f * sigma_d;
  g.Rins = 0.5f * (sigma_c + sigma_d);
  g.Rins2 = g.Rins * g.Rins;
  g.dcirc2 = sigma_c * sigma_c;
  const float rcut = ((sigma_c + sigma_d) + dmax_cap * 1.7320508f) + 1e-3f;
  g.rcut2 = rcut * rcut;
  g.Rh = 0.5f * sigma_c;
  g.cen = 0.375f * g.Rh;
  g.adisk = disk_a; g.sdisk = disk_s;
  const float rs = disk_s + g.rd;
  g.rs2 = rs * rs;
  g.rd2 = g.rd * g.rd;
  return g;
}

// Orientation as the shape tests need it: the body z axis (x, y, z; w unused) for the bodies of revolution (R-S19), the
// whole unit quaternion (w, x, y, z stored as x = q.w, y = q.x, z = q.y, w = q.z) for the tetrahedron.
struct Ori { float x, y, z, w; };
static inline Ori ori_of(const Geo& g, Q4 q) {
  if (g.shape == SH_TETRAHEDRON) return Ori{q.w, q.x, q.y, q.z};
  const V3 a = quat_axis(q);
  return Ori{a.x, a.y, a.z, 0.0f};
}
static inline V3 axis_of(Ori o) { return V3{o.x, o.y, o.z}; }

// R-N2b (Fig. 1 L21 shows tetrahedra): regular tetrahedron with circumradius Rh = sigma_c / 2, body-frame
// vertices s u_i, s = Rh 0.57735026f, u_0 = (1,1,1), u_1 = (1,-1,-1), u_2 = (-1,1,-1), u_3 = (-1,-1,1); the face opposite
// vertex i lies in the plane u_i . x = -s.  Body axes = columns of the rotation matrix of q (the formula of R-S19 for all three).
struct Frame { V3 ex, ey, ez; };
static inline Frame frame_of(Ori o) {
  const float w = o.x, x = o.y, y = o.z, z = o.w;
  Frame f;
  f.ex = V3{1.0f - 2.0f * (y * y + z * z), 2.0f * (x * y + w * z), 2.0f * (x * z - w * y)};
  f.ey = V3{2.0f * (x * y - w * z), 1.0f - 2.0f * (x * x + z * z), 2.0f * (y * z + w * x)};
  f.ez = V3{2.0f * (x * z + w * y), 2.0f * (y * z - w * x), 1.0f - 2.0f * (x * x + y * y)};
  return f;
}
static const float TET_U[4][3] = {{1.0f, 1.0f, 1.0f}, {1.0f, -1.0f, -1.0f}, {-1.0f, 1.0f, -1.0f}, {-1.0f, -1.0f, 1.0f}};

// squared distance from p to the triangle (a, b, c): closest-point regions by barycentric signs (Ericson, Real-Time
// Collision Detection 5.1.5), only + x /
static inline float tri_dist2(V3 p, V3 a, V3 b, V3 c) {
  const V3 ab = b - a, ac = c - a, ap = p - a;
  const float d1 = dot3(ab, ap), d2 = dot3(ac, ap);
  if (d1 <= 0.0f && d2 <= 0.0f) return dot3(ap, ap);
  const V3 bp = p - b;
  const float d3 = dot3(ab, bp), d4 = dot3(ac, bp);
  if (d3 >= 0.0f && d4 <= d3) return dot3(bp, bp);
  const float vc = d1 * d4 - d3 * d2;
  if (vc <= 0.0f && d1 >= 0.0f && d3 <= 0.0f) { const float v = d1 / (d1 - d3); const V3 e = ap - ab * v; return dot3(e, e); }
  const V3 cp = p - c;
  const float d5 = dot3(ab, cp), d6 = dot3(ac, cp);
  if (d6 >= 0.0f && d5 <= d6) return dot3(cp, cp);
  const float vb = d5 * d2 - d1 * d6;
  if (vb <= 0.0f && d2 >= 0.0f && d6 <= 0.0f) { const float w = d2 / (d2 - d6); const V3 e = ap - ac * w; return dot3(e, e); }
  const float va = d3 * d6 - d5 * d4;
  if (va <= 0.0f && (d4 - d3) >= 0.0f && (d5 - d6) >= 0.0f) {
    const float w = (d4 - d3) / ((d4 - d3) + (d5 - d6));
    const V3 e = bp - (c - b) * w;
    return dot3(e, e);
  }
  const float den = 1.0f / (va + vb + vc);
  const float v = vb * den, w = vc * den;
  const V3 e = ap - (ab * v + ac * w);
  return dot3(e, e);
}
// depletant centre at body-frame point b vs the tetrahedron: inside, or closer than rd to a face it lies in front of
static inline bool near_tetrahedron(float s, float rd2, V3 b) {
  V3 v[4];
  for (int i = 0; i < 4; ++i) v[i] = V3{s * TET_U[i][0], s * TET_U[i][1], s * TET_U[i][2]};
  bool inside = true;
  float best = 3.0e38f;
  for (int i = 0; i < 4; ++i) {
    const float h = (TET_U[i][0] * b.x + TET_U[i][1] * b.y) + TET_U[i][2] * b.z;
    if (h < -s) {                                  // in front of the face opposite vertex i
      inside = false;
      const float d2 = tri_dist2(b, v[(i + 1) & 3], v[(i + 2) & 3], v[(i + 3) & 3]);
      if (d2 < best) best = d2;
    }
  }
  return inside || best < rd2;
}

// R-N2 (the paper's discoids are oblate ellipsoids a = b = 0.5, c = 0.25, L228): is the point at
// cylindrical coordinates (rho, z >= 0) of the body frame closer than rd to the solid spheroid x^2/A^2 + z^2/C^2 <= 1?
// Inside: yes.  Outside: the closest point of the ellipse is (A^2 rho/(t + A^2), C^2 z/(t + C^2)) for the root t of
// F(t) = (A rho/(t + A^2))^2 + (C z/(t + C^2))^2 - 1, which is convex and decreasing: SIX Newton steps from the lower bound
// t0 = max(A rho - A^2, C z - C^2) approach it monotonically (fp32-converged after five); only + x / on both sides.
static inline bool near_spheroid(float A, float Cc, float rd2, float rho, float z) {
  const float qa = rho / A, qc = z / Cc;
  if (fmaf(qa, qa, qc * qc) <= 1.0f) return true;
  const float A2 = A * A, C2 = Cc * Cc, ar = A * rho, cz = Cc * z;
  float t = ar - A2;
  const float t1 = cz - C2;
  if (t1 > t) t = t1;
  for (int it = 0; it < 6; ++it) {
    const float ia = 1.0f / (t + A2), ic = 1.0f / (t + C2);
    const float ua = ar * ia, uc = cz * ic;
    const float ua2 = ua * ua, uc2 = uc * uc;
    const float F = (ua2 + uc2) - 1.0f;
    const float dF = -2.0f * (ua2 * ia + uc2 * ic);
    t = t - F / dF;
  }
  const float ex = rho - (A2 * rho) / (t + A2), ez = z - (C2 * z) / (t + C2);
  return fmaf(ex, ex, ez * ez) < rd2;
}

// Depletant (sphere radius rd, centre at d relative to the colloid centre) vs colloid with
// body axis a.  R-S14 (strict <), R-S16 (half-ball), R-S17 (spherodisk), R-N2 (ellipsoid).
static inline bool dep_overlap(const Geo& g, V3 d, Ori o) {
  const float d2 = dot3(d, d);
  if (!(d2 < g.Rins2)) return false;          // circumsphere (+) depletant
  if (g.shape == SH_SPHERE) return true;
  if (g.shape == SH_TETRAHEDRON) {
    const Frame f = frame_of(o);
    return near_tetrahedron(g.Rh * 0.57735026f, g.rd2, V3{dot3(d, f.ex), dot3(d, f.ey), dot3(d, f.ez)});
  }
  const V3 a = axis_of(o);
  const float bz = dot3(d, a);
  if (g.shape == SH_ELLIPSOID) {
    const V3 p = V3{d.x - bz * a.x, d.y - bz * a.y, d.z - bz * a.z};
    return near_spheroid(g.adisk, g.sdisk, g.rd2, sqrtf(dot3(p, p)), fabsf(bz));
  }
  if (g.shape == SH_HALFBALL) {
    if (bz <= 0.0f) return true;              // below the flat face: inside ball radius Rh+rd
    const V3 p = V3{d.x - bz * a.x, d.y - bz * a.y, d.z - bz * a.z};
    const float rho = sqrtf(dot3(p, p));
    if (rho <= g.Rh) return bz < g.rd;
    const float e = rho - g.Rh;
    return fmaf(e, e, bz * bz) < g.rd2;
  }
  // spherodisk
  const V3 p = V3{d.x - bz * a.x, d.y - bz * a.y, d.z - bz * a.z};
  const float rho = sqrtf(dot3(p, p));
  if (rho <= g.adisk) return bz * bz < g.rs2;
  const float e = rho - g.adisk;
  return fmaf(e, e, bz * bz) < g.rs2;
}

// Support point of the shape with body axis a, centred at the origin, in direction n. R-S18.
static inline V3 support(const Geo& g, Ori o, V3 n) {
  if (g.shape == SH_TETRAHEDRON) {               // the vertex with the largest projection (first one on ties)
    const Frame f = frame_of(o);
    const V3 nb = V3{dot3(n, f.ex), dot3(n, f.ey), dot3(n, f.ez)};
    int best = 0;
    float hb = (TET_U[0][0] * nb.x + TET_U[0][1] * nb.y) + TET_U[0][2] * nb.z;
    for (int i = 1; i < 4; ++i) {
      const float h = (TET_U[i][0] * nb.x + TET_U[i][1] * nb.y) + TET_U[i][2] * nb.z;
      if (h > hb) { hb = h; best = i; }
    }
    const float s = g.Rh * 0.57735026f;
    return (f.ex * (s * TET_U[best][0]) + f.ey * (s * TET_U[best][1])) + f.ez * (s * TET_U[best][2]);
  }
  const V3 a = axis_of(o);
  const float nz = dot3(n, a);
  if (g.shape == SH_HALFBALL) {
    if (nz <= 0.0f) {
      const float len = sqrtf(dot3(n, n));
      if (!(len > 0.0f)) return V3{0.0f, 0.0f, 0.0f};
      return n * (g.Rh / len);
    }
    const V3 p = V3{n.x - nz * a.x, n.y - nz * a.y, n.z - nz * a.z};
    const float l = sqrtf(dot3(p, p));
    if (!(l > 0.0f)) return V3{0.0f, 0.0f, 0.0f};
    return p * (g.Rh / l);
  }
  if (g.shape == SH_ELLIPSOID) {               // (A^2 n_perp + C^2 n_par a) / sqrt(A^2 |n_perp|^2 + C^2 n_par^2)
    const V3 p = V3{n.x - nz * a.x, n.y - nz * a.y, n.z - nz * a.z};
    const float A2 = g.adisk * g.adisk, C2 = g.sdisk * g.sdisk;
    const float den = sqrtf(A2 * dot3(p, p) + C2 * (nz * nz));
    if (!(den > 0.0f)) return V3{0.0f, 0.0f, 0.0f};
    const float wa = A2 / den, wc = (C2 * nz) / den;
    return V3{wa * p.x + wc * a.x, wa * p.y + wc * a.y, wa * p.z + wc * a.z};
  }
  // spherodisk: disk rim point + rounding sphere
  const V3 p = V3{n.x - nz * a.x, n.y - nz * a.y, n.z - nz * a.z};
  const float l = sqrtf(dot3(p, p));
  const float len = sqrtf(dot3(n, n));
  V3 out = V3{0.0f, 0.0f, 0.0f};
  if (l > 0.0f) out = p * (g.adisk / l);
  if (len > 0.0f) out = out + n * (g.sdisk / len);
  return out;
}

static const int MPR_MAXIT = 48;
static const float MPR_TOL = 1e-5f;

// Support of the Minkowski difference B - A in direction n (A at origin, B at rho).
static inline V3 support_diff(const Geo& g, V3 rho, Ori aA, Ori aB, V3 n) {
  const V3 sb = support(g, aB, n);
  const V3 sa = support(g, aA, neg(n));
  return (sb + rho) - sa;
}

// Minkowski-portal-refinement (XenoCollide, G. Snethen 2008) boolean overlap test on the
// full convex shapes.  R-S18.  Returns true if overlapping.  Contact band (|gap| < MPR_TOL)
// counts as not overlapping; iteration cap counts as overlapping.
static bool mpr_overlap(const Geo& g, V3 rho, Ori aA, Ori aB) {
  V3 cA = V3{0.0f, 0.0f, 0.0f}, cB = rho;
  if (g.shape == SH_HALFBALL) {
    cA = neg(axis_of(aA) * g.cen);
    cB = rho - axis_of(aB) * g.cen;
  }
  V3 v0 = cB - cA;
  if (v0.x == 0.0f && v0.y == 0.0f && v0.z == 0.0f) v0 = V3{1e-5f, 0.0f, 0.0f};
  V3 n = neg(v0);
  V3 v1 = support_diff(g, rho, aA, aB, n);
  if (dot3(v1, n) <= 0.0f) return false;
  n = cross3(v1, v0);
  if (n.x == 0.0f && n.y == 0.0f && n.z == 0.0f) return true;
  V3 v2 = support_diff(g, rho, aA, aB, n);
  if (dot3(v2, n) <= 0.0f) return false;
  n = cross3(v1 - v0, v2 - v0);
  if (dot3(n, v0) > 0.0f) { V3 t = v1; v1 = v2; v2 = t; n = neg(n); }
  V3 v3;
  int it = 0;
  for (;;) {                                   // phase 1: find a portal the origin ray passes
    if (it++ >= MPR_MAXIT) return true;
    v3 = support_diff(g, rho, aA, aB, n);
    if (dot3(v3, n) <= 0.0f) return false;
    if (dot3(cross3(v1, v3), v0) < 0.0f) { v2 = v3; n = cross3(v1 - v0, v3 - v0); continue; }
    if (dot3(cross3(v3, v2), v0) < 0.0f) { v1 = v3; n = cross3(v3 - v0, v2 - v0); continue; }
    break;
  }
  for (it = 0;; ++it) {                        // phase 2: refine the portal
    if (it >= MPR_MAXIT) return true;
    n = cross3(v2 - v1, v3 - v1);
    const float len = sqrtf(dot3(n, n));
    if (!(len > 0.0f)) return true;
    n = V3{n.x / len, n.y / len, n.z / len};
    if (dot3(n, v1) >= 0.0f) return true;      // origin on the inner side of the portal
    const V3 v4 = support_diff(g, rho, aA, aB, n);
    if (dot3(v4, n) < 0.0f) return false;      // support plane separates the origin
    if (dot3(v4 - v3, n) <= MPR_TOL) return false;   // portal reached the surface: touching
    const V3 c = cross3(v4, v0);
    if (dot3(v1, c) > 0.0f) {
      if (dot3(v2, c) > 0.0f) v1 = v4; else v3 = v4;
    } else {
      if (dot3(v3, c) > 0.0f) v2 = v4; else v1 = v4;
    }
  }
}

// Hard overlap of colloid A (origin, axis aA) with colloid B (at rho, axis aB).  Eq. 5 L80.
static inline bool pair_overlap(const Geo& g, V3 rho, Ori aA, Ori aB) {
  const float r2 = dot3(rho, rho);
  if (!(r2 < g.dcirc2)) return false;          // circumsphere pre-test (exact test for spheres)
  if (g.shape == SH_SPHERE) return true;
  return mpr_overlap(g, rho, aA, aB);
}

// ----------------------------------------------------------------------------- Poisson
// R-S2: exact table inversion.  T[k-k_lo] = floor(CDF(k) 2^64) saturating; N = k_lo + #{T <= U}.
struct PoissonTable { double lambda = -1.0; int64_t k_lo = 0; std::vector<uint64_t> T; };

static void build_poisson(PoissonTable& pt, double lambda) {
  pt.lambda = lambda; pt.T.clear(); pt.k_lo = 0;
  if (!(lambda > 0.0)) return;
  const double sq = std::sqrt(lambda);
  int64_t lo = (int64_t)std::floor(lambda - 10.0 * sq - 10.0);
  if (lo < 0) lo = 0;
  const int64_t hi = (int64_t)std::ceil(lambda + 10.0 * sq + 20.0);
  const int64_t n = hi - lo + 1;
  int64_t m = (int64_t)std::floor(lambda);
  if (m < lo) m = lo;
  std::vector<double> p((size_t)n);
  p[(size_t)(m - lo)] = std::exp((double)m * std::log(lambda) - lambda - std::lgamma((double)m + 1.0));
  for (int64_t k = m; k < hi; ++k) p[(size_t)(k + 1 - lo)] = p[(size_t)(k - lo)] * lambda / (double)(k + 1);
  for (int64_t k = m; k > lo; --k) p[(size_t)(k - 1 - lo)] = p[(size_t)(k - lo)] * (double)k / lambda;
  double S = 0.0;
  for (int64_t j = 0; j < n; ++j) S += p[(size_t)j];
  pt.k_lo = lo; pt.T.resize((size_t)n);
  double c = 0.0;
  for (int64_t j = 0; j < n; ++j) {
    c += p[(size_t)j] / S;
    pt.T[(size_t)j] = (c >= 1.0) ? UINT64_MAX : (uint64_t)std::floor(c * 18446744073709551616.0);
  }
}
static inline int64_t poisson_draw(const PoissonTable& pt, uint64_t U) {
  if (pt.T.empty()) return 0;
  const size_t cnt = (size_t)(std::upper_bound(pt.T.begin(), pt.T.end(), U) - pt.T.begin());
  return pt.k_lo + (int64_t)cnt;
}

// ----------------------------------------------------------------------------- context
enum { C_TRIALS_TRANS, C_ACCEPT_TRANS, C_TRIALS_ROT, C_ACCEPT_ROT, C_REJ_BOUNDARY, C_REJ_HARD,
       C_REJ_DEPLETANT, C_REJ_CB, C_DEP_DRAWN, C_DEP_NEEDED, C_DEP_EVALUATED, C_CB_REINSERTIONS,
       C_PHILOX_BLOCKS, C_COUNT };

enum { OUT_NONE = 0, OUT_ACCEPT = 1, OUT_BOUNDARY = 2, OUT_HARD = 3, OUT_DEPLETANT = 4, OUT_CB = 5 };

struct Ctx {
  Geo g;
  int64_t N = 0;
  float* pos = nullptr;      // N x (x,y,z,unused), caller-owned host memory, updated in place
  float* quat = nullptr;     // N x (w,x,y,z) or null
  int nc = 0; float w = 0.0f;
  float shift[3] = {0, 0, 0};
  bool built = false; uint32_t b_seed = 0, b_step = 0;
  std::vector<uint32_t> cell_start, cell_pid;
  std::vector<uint8_t> outcome;
  std::vector<float> trial_pos, trial_quat;   // proposed pose of every particle tried this sweep
  uint64_t cnt[C_COUNT] = {0};
  PoissonTable pt;
  uint32_t flags = 0;          // F_* options (oracle_set_flags)
  float eval_dmax = -1.0f;     // d_max assumed by oracle_eval_move(s) for the shell (default: d_max_cap)
  std::string err;
};

struct Counters { uint64_t c[C_COUNT] = {0}; };

static inline Q4 load_q(const Ctx& c, int64_t i) {
  if (!c.quat) return Q4{1.0f, 0.0f, 0.0f, 0.0f};
  const float* q = c.quat + 4 * i;
  return Q4{q[0], q[1], q[2], q[3]};
}
static inline V3 load_r(const Ctx& c, int64_t i) {
  const float* p = c.pos + 4 * i;
  return V3{p[0], p[1], p[2]};
}

// R-1 (grid): cell index of a coordinate along one axis in the shifted grid.
static inline int cell_axis(const Ctx& c, float x, float gshift) {
  float t = x - gshift;
  if (t < 0.0f) t += c.g.L;
  int ci = (int)(t / c.w);
  if (ci >= c.nc) ci = c.nc - 1;
  return ci;
}
static inline int64_t cell_of(const Ctx& c, V3 r) {
  const int ix = cell_axis(c, r.x, c.shift[0]);
  const int iy = cell_axis(c, r.y, c.shift[1]);
  const int iz = cell_axis(c, r.z, c.shift[2]);
  return ((int64_t)iz * c.nc + iy) * c.nc + ix;
}
// R-S13: compare-and-shift minimum image of a - b
static inline float minimg1(const Geo& g, float d) {
  if (d > g.halfL) d -= g.L; else if (d < -g.halfL) d += g.L;
  return d;
}
static inline V3 minimg(const Geo& g, V3 a, V3 b) {
  return V3{minimg1(g, a.x - b.x), minimg1(g, a.y - b.y), minimg1(g, a.z - b.z)};
}
static inline float wrap1(const Geo& g, float x) {
  if (x < 0.0f) x += g.L;
  if (x >= g.L) x -= g.L;
  return x;
}

// R-S3: uniform point in the ball of given radius by cube rejection, one Philox block per attempt.
static inline V3 ball_sample(uint32_t seed, uint32_t step, uint32_t purpose, uint32_t colour,
                             uint32_t id, uint32_t k, uint32_t c2, uint32_t first_attempt,
                             float radius, float radius2, uint64_t& nblocks) {
  for (uint32_t a = 0; a < 64; ++a) {
    const U4 r = philox4x32_10(id, k, c2, word3(purpose, colour, first_attempt + a), seed, step);
    ++nblocks;
    const V3 d = V3{radius * sym_unit(r.v[0]), radius * sym_unit(r.v[1]), radius * sym_unit(r.v[2])};
    if (dot3(d, d) <= radius2) return d;
  }
  return V3{0.0f, 0.0f, 0.0f};
}

// ---- options of a sweep (oracle_set_flags)
enum { F_SHELL = 1u, F_ROSENBLUTH = 2u };

// R-N1 (L158 "restricting the sampling to the excluded volume shell of the moved colloid"): depletants are drawn
// uniformly in the shell R_in < |d| <= R about the NEW centre instead of the whole ball.  Eq. 12 (L136) needs
// V_0 >= V'_excl \ V_excl: the ball |d| <= R_in must lie inside the OLD pose's excluded volume for every move the
// sweep can propose.  The old excluded volume contains the ball of radius r_in about the old centre (r_in = R for a
// sphere, r_d for the half-ball whose centre lies on its flat face, s + r_d for the spherodisk), a translation moves
// the centre by at most sqrt(3) d_max and a rotation not at all, hence R_in = max(0, r_in - sqrt(3) d_max).
struct Shell { float Rin, Rin3, dR3; };
static inline Shell make_shell(const Geo& g, float d_max, uint32_t flags) {
  float rin = g.Rins;
  if (g.shape == SH_HALFBALL) rin = g.rd;
  else if (g.shape == SH_SPHERODISK || g.shape == SH_ELLIPSOID) rin = g.sdisk + g.rd;   // rounding radius / polar semi-axis
  else if (g.shape == SH_TETRAHEDRON) rin = g.Rh * 0.33333334f + g.rd;                   // inradius of the regular tetrahedron
  Shell sh;
  sh.Rin = rin - 1.7320508f * d_max;
  if (sh.Rin < 0.0f) sh.Rin = 0.0f;
  sh.Rin3 = (sh.Rin * sh.Rin) * sh.Rin;
  sh.dR3 = (g.Rins * g.Rins) * g.Rins - sh.Rin3;
  return sh;
}
// cube root by +, x, / only (libm's cbrtf is not reproducible on the device): exponent/3 seed, four Newton steps
static inline float cbrt_fixed(float t) {
  uint32_t b; std::memcpy(&b, &t, 4);
  b = b / 3u + 0x2a514067u;
  float y; std::memcpy(&y, &b, 4);
  for (int it = 0; it < 4; ++it) { const float q = t / (y * y); y = ((y + y) + q) * 0.33333334f; }
  return y;
}
// uniform point in the shell: direction by cube rejection (words 0-2 of the block, one block per attempt, as R-S3) and
// IEEE normalisation, radius (R_in^3 + u dR^3)^(1/3) from word 3 of the accepted block
static inline V3 shell_sample(uint32_t seed, uint32_t step, uint32_t purpose, uint32_t colour, uint32_t id,
                              uint32_t k, const Shell& sh, float radius, uint64_t& nblocks) {
  for (uint32_t a = 0; a < 64; ++a) {
    const U4 r = philox4x32_10(id, k, 0, word3(purpose, colour, a), seed, step);
    ++nblocks;
    const V3 v = V3{sym_unit(r.v[0]), sym_unit(r.v[1]), sym_unit(r.v[2])};
    const float n2 = dot3(v, v);
    if (n2 <= 1.0f && n2 >= 1e-6f) {
      const float t = sh.Rin3 + unit01(r.v[3]) * sh.dR3;
      const float sc = cbrt_fixed(t) / sqrtf(n2);
      return v * sc;
    }
  }
  return V3{radius, 0.0f, 0.0f};
}

struct Nbr { V3 rho; Ori axis; };

// Steps 3.4 - 3.8 of the move: neighbourhood, hard overlap, depletants.
// i = moved colloid, own = its cell, (r0,q0) old pose, (r1,q1) new pose (already wrapped).
static int evaluate_move(const Ctx& c, uint32_t seed, uint32_t step, uint32_t colour, int64_t i,
                         int64_t own, V3 r0, Q4 q0, V3 r1, Q4 q1, int n_trial, float d_max, Counters& cn) {
  const Geo& g = c.g;
  const int nc = c.nc;
  const int ix = (int)(own % nc), iy = (int)((own / nc) % nc), iz = (int)(own / ((int64_t)nc * nc));
  std::vector<Nbr> nb;
  for (int dz = -1; dz <= 1; ++dz)
    for (int dy = -1; dy <= 1; ++dy)
      for (int dx = -1; dx <= 1; ++dx) {
        const int jx = (ix + dx + nc) % nc, jy = (iy + dy + nc) % nc, jz = (iz + dz + nc) % nc;
        const int64_t cj = ((int64_t)jz * nc + jy) * nc + jx;
        for (uint32_t s = c.cell_start[(size_t)cj]; s < c.cell_start[(size_t)cj + 1]; ++s) {
          const int64_t j = c.cell_pid[s];
          if (j == i) continue;
          const V3 rho = minimg(g, load_r(c, j), r1);
          if (!(dot3(rho, rho) < g.rcut2)) continue;
          nb.push_back(Nbr{rho, ori_of(g, load_q(c, j))});
        }
      }
  const V3 rho_old = minimg(g, r0, r1);
  const Ori a_old = ori_of(g, q0), a_new = ori_of(g, q1);

  // 3.5 hard overlap of the new pose with any neighbour (Eq. 5's min(1, e^{-beta dH_cc}), L80)
  for (const Nbr& n : nb)
    if (pair_overlap(g, n.rho, a_new, n.axis)) return OUT_HARD;

  // 3.6 number of depletants N_d ~ Poisson(n_R V_ins)   (L67, L156)
  const U4 rn = philox4x32_10((uint32_t)i, 0, 0, word3(P_NDEP, colour, 0), seed, step);
  ++cn.c[C_PHILOX_BLOCKS];
  const uint64_t U = ((uint64_t)rn.v[0] << 32) | rn.v[1];
  const int64_t Nd = poisson_draw(c.pt, U);
  cn.c[C_DEP_DRAWN] += (uint64_t)Nd;

  const V3 zero = V3{0.0f, 0.0f, 0.0f};
  const Shell sh = make_shell(g, d_max, c.flags);
  // position of depletant k relative to the new centre: whole insertion ball (L156), or its shell (option R-N1)
  auto dep_position = [&](int64_t k) {
    if (c.flags & F_SHELL)
      return shell_sample(seed, step, P_DEPPOS, colour, (uint32_t)i, (uint32_t)k, sh, g.Rins, cn.c[C_PHILOX_BLOCKS]);
    return ball_sample(seed, step, P_DEPPOS, colour, (uint32_t)i, (uint32_t)k, 0, 0, g.Rins, g.Rins2,
                       cn.c[C_PHILOX_BLOCKS]);
  };
  auto free_of_nbrs = [&](V3 d) {
    for (const Nbr& n : nb)
      if (dep_overlap(g, d - n.rho, n.axis)) return false;
    return true;
  };
  // "rejecting" depletant (Fig. 2 L72): overlaps new pose, not the old pose, no other colloid
  auto new_only = [&](V3 d) { return dep_overlap(g, d - zero, a_new) && !dep_overlap(g, d - rho_old, a_old); };
  auto old_only = [&](V3 d) { return dep_overlap(g, d - rho_old, a_old) && !dep_overlap(g, d - zero, a_new); };

  if (n_trial <= 0) {                          // 3.7 plain rule, L68
    for (int64_t k = 0; k < Nd; ++k) {
      const V3 d = dep_position(k);
      ++cn.c[C_DEP_NEEDED]; ++cn.c[C_DEP_EVALUATED];
      if (new_only(d) && free_of_nbrs(d)) return OUT_DEPLETANT;
    }
    return OUT_ACCEPT;
  }

  // 3.8 configurational bias, Eq. 16 (L172) with the reading R-G1/G2/G3
  float P = 1.0f;
  bool any = false;
  // Option R-N4 (refs 27, 28, 33): the exact Rosenbluth weight N'_ins / (N_ins + 1) from n_trial forward and
  // n_trial - 1 FRESH reverse reinsertions (the original depletant is the n_trial-th reverse candidate, L174)
  const bool rosen = (c.flags & F_ROSENBLUTH) != 0;
  for (int64_t k = 0; k < Nd; ++k) {
    const V3 d = dep_position(k);
    ++cn.c[C_DEP_NEEDED]; ++cn.c[C_DEP_EVALUATED];
    if (!(new_only(d) && free_of_nbrs(d))) continue;
    any = true;
    uint32_t Ni = 0, Npins = 0, Npi = 0, Nins = 0;
    for (int t = 0; t < n_trial; ++t) {
      // forward: reinsertion about the OLD centre (Fig. 3)
      const V3 f = ball_sample(seed, step, P_CBPOS, colour, (uint32_t)i, (uint32_t)k, (uint32_t)t, 0,
                               g.Rins, g.Rins2, cn.c[C_PHILOX_BLOCKS]) + rho_old;
      if (old_only(f)) { ++Ni; if (free_of_nbrs(f)) ++Npins; }
      if (rosen && t == n_trial - 1) break;
      // reverse: reinsertion about the NEW centre
      const V3 b = ball_sample(seed, step, P_CBPOS, colour, (uint32_t)i, (uint32_t)k,
                               (uint32_t)t + (1u << 16), 0, g.Rins, g.Rins2, cn.c[C_PHILOX_BLOCKS]);
      if (new_only(b)) { ++Npi; if (free_of_nbrs(b)) ++Nins; }
    }
    cn.c[C_CB_REINSERTIONS] += 2u * (uint64_t)n_trial - (rosen ? 1u : 0u);
    if (Npins == 0) return OUT_CB;             // R-G3: zero forward weight
    if (rosen) { P = P * ((float)Npins / (float)(Nins + 1u)); continue; }
    const float wk = (float)(Npins * (Npi + 1u)) / (float)((Nins + 1u) * Ni);
    P = P * wk;
  }
  if (!any) return OUT_ACCEPT;
  const U4 ra = philox4x32_10((uint32_t)i, 0, 0, word3(P_ACCEPT, colour, 0), seed, step);
  ++cn.c[C_PHILOX_BLOCKS];
  return (unit01(ra.v[0]) < P) ? OUT_ACCEPT : OUT_CB;
}

// R-2 (L180 "the checkerboard coloring is permuted randomly"): the order in which a sweep visits the 8 colours, a
// Fisher-Yates shuffle of (0..7) driven by the 7 words of SWEEP blocks 1 and 2: position i (7 down to 1) is swapped
// with a position drawn uniformly from 0..i.  Pinned by tests/test_oracle_physics.py (uniform over positions and over
// neighbouring pairs; a constant order and an off-by-one range must fail).
static void colour_order(uint32_t seed, uint32_t step, uint32_t perm[8]) {
  for (uint32_t k = 0; k < 8; ++k) perm[k] = k;
  const U4 b1 = philox4x32_10(0, 0, 0, word3(P_SWEEP, 0, 1), seed, step);
  const U4 b2 = philox4x32_10(0, 0, 0, word3(P_SWEEP, 0, 2), seed, step);
  const uint32_t wds[7] = {b1.v[0], b1.v[1], b1.v[2], b1.v[3], b2.v[0], b2.v[1], b2.v[2]};
  for (int i = 7, j = 0; i >= 1; --i, ++j) {
    const uint32_t r = mulhi32(wds[j], (uint32_t)i + 1u);
    const uint32_t t = perm[i]; perm[i] = perm[r]; perm[r] = t;
  }
}

// Steps 3.1 - 3.3 + 3.9 for one active cell.
static void process_cell(Ctx& c, uint32_t seed, uint32_t step, uint32_t colour, int64_t cell,
                         float d_max, float a_max, int n_trial, Counters& cn) {
  const Geo& g = c.g;
  const uint32_t b = c.cell_start[(size_t)cell], e = c.cell_start[(size_t)cell + 1];
  const uint32_t nocc = e - b;
  if (nocc == 0) return;
  const U4 rs = philox4x32_10((uint32_t)cell, 0, 0, word3(P_SELECT, colour, 0), seed, step);
  const int64_t i = c.cell_pid[b + mulhi32(rs.v[0], nocc)];
  const V3 r0 = load_r(c, i);
  const Q4 q0 = load_q(c, i);
  const U4 rm = philox4x32_10((uint32_t)i, 0, 0, word3(P_MOVE, colour, 0), seed, step);
  cn.c[C_PHILOX_BLOCKS] += 2;
  const bool rot = (a_max > 0.0f) && (rm.v[3] & 1u);
  V3 r1 = r0; Q4 q1 = q0;
  if (!rot) {
    r1 = V3{wrap1(g, r0.x + d_max * sym_unit(rm.v[0])), wrap1(g, r0.y + d_max * sym_unit(rm.v[1])),
            wrap1(g, r0.z + d_max * sym_unit(rm.v[2]))};
    ++cn.c[C_TRIALS_TRANS];
  } else {
    const V3 v = ball_sample(seed, step, P_MOVE, colour, (uint32_t)i, 0, 0, 1, a_max, a_max * a_max,
                             cn.c[C_PHILOX_BLOCKS]);
    q1 = rotate_cayley(q0, v);
    ++cn.c[C_TRIALS_ROT];
  }
  float* tp = c.trial_pos.data() + 4 * i;
  tp[0] = r1.x; tp[1] = r1.y; tp[2] = r1.z; tp[3] = 0.0f;
  float* tq = c.trial_quat.data() + 4 * i;
  tq[0] = q1.w; tq[1] = q1.x; tq[2] = q1.y; tq[3] = q1.z;

  int out;
  if (cell_of(c, r1) != cell) out = OUT_BOUNDARY;      // confinement, L180
  else out = evaluate_move(c, seed, step, colour, i, cell, r0, q0, r1, q1, n_trial, d_max, cn);
  c.outcome[(size_t)i] = (uint8_t)out;
  switch (out) {
    case OUT_ACCEPT: {
      float* p = c.pos + 4 * i;
      p[0] = r1.x; p[1] = r1.y; p[2] = r1.z;
      if (c.quat) { float* q = c.quat + 4 * i; q[0] = q1.w; q[1] = q1.x; q[2] = q1.y; q[3] = q1.z; }
      ++cn.c[rot ? C_ACCEPT_ROT : C_ACCEPT_TRANS];
      break;
    }
    case OUT_BOUNDARY: ++cn.c[C_REJ_BOUNDARY]; break;
    case OUT_HARD: ++cn.c[C_REJ_HARD]; break;
    case OUT_DEPLETANT: ++cn.c[C_REJ_DEPLETANT]; break;
    case OUT_CB: ++cn.c[C_REJ_CB]; break;
  }
}

static double lambda_of(const Geo& g, double n_R) {
  const double Rd = (double)g.Rins;
  return n_R * ((4.0 * M_PI / 3.0) * (Rd * Rd * Rd));
}
// mean number of depletants of a move: fugacity x sampled volume (L67), the shell's volume with option R-N1
static double lambda_opt(const Geo& g, double n_R, float d_max, uint32_t flags) {
  if (!(flags & F_SHELL)) return lambda_of(g, n_R);
  const Shell sh = make_shell(g, d_max, flags);
  const double Rd = (double)g.Rins, Ri = (double)sh.Rin;
  return n_R * ((4.0 * M_PI / 3.0) * (Rd * Rd * Rd - Ri * Ri * Ri));
}

}  // namespace

// ===================================================================================== C ABI
extern "C" {

struct oracle_params {
  int32_t shape; float sigma_c; float disk_a; float disk_s; float sigma_d; float box_L; float d_max_cap;
};

void* oracle_create(const oracle_params* p, int64_t N, float* pos4, float* quat4) {
  if (!p || N <= 0 || !pos4 || !(p->box_L > 0.0f) || !(p->sigma_c > 0.0f) || p->sigma_d < 0.0f) return nullptr;
  if (p->shape != SH_SPHERE && !quat4) return nullptr;
  // near_spheroid's six Newton steps resolve the point-to-ellipse distance to fp32 rounding for aspect ratios up to 4
  // (pinned at 2 and at 4); flatter discoids would need more steps, so they are refused rather than answered loosely
  if (p->shape == SH_ELLIPSOID && !(p->disk_s > 0.0f && p->disk_a >= p->disk_s && p->disk_a <= 4.0f * p->disk_s)) return nullptr;
  Ctx* c = new Ctx();
  c->g = make_geo(p->shape, p->sigma_c, p->disk_a, p->disk_s, p->sigma_d, p->box_L, p->d_max_cap);
  c->N = N; c->pos = pos4; c->quat = quat4;
  // R-1: n_c = largest even integer <= L / (d_circ + sigma_d + 2 d_max_cap), n_c >= 4
  const double wmin = (double)p->sigma_c + (double)p->sigma_d + 2.0 * (double)p->d_max_cap;
  int64_t n = (int64_t)std::floor((double)p->box_L / wmin);
  n &= ~(int64_t)1;
  if (n < 4 || n > 1024) { delete c; return nullptr; }
  c->nc = (int)n;
  c->w = p->box_L / (float)c->nc;
  c->cell_start.assign((size_t)n * n * n + 1, 0);
  c->cell_pid.assign((size_t)N, 0);
  c->outcome.assign((size_t)N, 0);
  c->trial_pos.assign((size_t)N * 4, 0.0f);
  c->trial_quat.assign((size_t)N * 4, 0.0f);
  return c;
}
void oracle_destroy(void* h) { delete (Ctx*)h; }
// options of the following sweeps / evaluations: bit 0 shell-restricted insertion (R-N1), bit 1 Rosenbluth CB weight
// (R-N4); eval_dmax >= 0: the step size oracle_eval_move(s) assumes for the shell (their moves must obey it)
int oracle_set_flags(void* h, uint32_t flags, float eval_dmax) {
  Ctx* c = (Ctx*)h;
  c->flags = flags; c->eval_dmax = eval_dmax; c->pt.lambda = -1.0;
  return 0;
}
int oracle_grid(void* h, int32_t* nc, float* w) { Ctx* c = (Ctx*)h; *nc = c->nc; *w = c->w; return 0; }
void oracle_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}
int oracle_get_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// a2: grid shift from the SWEEP stream, then binning in ascending particle id (L180).
int oracle_build_cells(void* h, uint32_t seed, uint32_t step) {
  Ctx* c = (Ctx*)h;
  const U4 r = philox4x32_10(0, 0, 0, word3(P_SWEEP, 0, 0), seed, step);
  for (int a = 0; a < 3; ++a) c->shift[a] = unit01(r.v[a]) * c->w;
  const size_t ncell = (size_t)c->nc * c->nc * c->nc;
  std::vector<uint32_t> cnt(ncell + 1, 0);
  std::vector<int64_t> cid((size_t)c->N);
  for (int64_t i = 0; i < c->N; ++i) { cid[(size_t)i] = cell_of(*c, load_r(*c, i)); ++cnt[(size_t)cid[(size_t)i] + 1]; }
  for (size_t k = 0; k < ncell; ++k) cnt[k + 1] += cnt[k];
  c->cell_start = cnt;
  std::vector<uint32_t> fill(cnt.begin(), cnt.end() - 1);
  for (int64_t i = 0; i < c->N; ++i) c->cell_pid[fill[(size_t)cid[(size_t)i]]++] = (uint32_t)i;
  c->built = true; c->b_seed = seed; c->b_step = step;
  return 0;
}

// One sweep = 8 sub-lattice passes in a permuted order (L180).
int oracle_colour_order(uint32_t seed, uint32_t step, uint32_t* out8) { colour_order(seed, step, out8); return 0; }
int oracle_sweep(void* h, uint32_t seed, uint32_t step, double n_R, float d_max, float a_max, int32_t n_trial) {
  Ctx* c = (Ctx*)h;
  if (!c->built || c->b_seed != seed || c->b_step != step) return -3;
  if (!(d_max >= 0.0f) || d_max > c->g.dmax_cap || n_R < 0.0 || a_max < 0.0f || n_trial < 0 || n_trial > 65535) return -1;
  const double lambda = lambda_opt(c->g, n_R, d_max, c->flags);
  if (c->pt.lambda != lambda) build_poisson(c->pt, lambda);
  uint32_t perm[8];
  colour_order(seed, step, perm);
  std::fill(c->outcome.begin(), c->outcome.end(), (uint8_t)0);
  const int nc = c->nc, hc = nc / 2;
  const int64_t nact = (int64_t)hc * hc * hc;
  for (int pass = 0; pass < 8; ++pass) {
    const uint32_t col = perm[pass];
    const int px = col & 1, py = (col >> 1) & 1, pz = (col >> 2) & 1;
    // active cells in ascending linear index; independent of each other, so the
    // optional OpenMP loop gives the same bits as the sequential one
    Counters total;
#pragma omp parallel
    {
      Counters cn;
#pragma omp for schedule(dynamic, 256)
      for (int64_t a = 0; a < nact; ++a) {
        const int ax = (int)(a % hc), ay = (int)((a / hc) % hc), az = (int)(a / ((int64_t)hc * hc));
        const int64_t cell = ((int64_t)(2 * az + pz) * nc + (2 * ay + py)) * nc + (2 * ax + px);
        process_cell(*c, seed, step, col, cell, d_max, a_max, n_trial, cn);
      }
#pragma omp critical
      for (int k = 0; k < C_COUNT; ++k) total.c[k] += cn.c[k];
    }
    for (int k = 0; k < C_COUNT; ++k) c->cnt[k] += total.c[k];
  }
  c->built = false;   // the next sweep needs a new grid shift
  return 0;
}

int oracle_counters(void* h, uint64_t* out) { Ctx* c = (Ctx*)h; std::memcpy(out, c->cnt, sizeof(c->cnt)); return 0; }
int oracle_reset_counters(void* h) { Ctx* c = (Ctx*)h; std::memset(c->cnt, 0, sizeof(c->cnt)); return 0; }
int oracle_outcomes(void* h, uint8_t* out) { Ctx* c = (Ctx*)h; std::memcpy(out, c->outcome.data(), (size_t)c->N); return 0; }
int oracle_trial_poses(void* h, float* pos4, float* quat4) {
  Ctx* c = (Ctx*)h;
  std::memcpy(pos4, c->trial_pos.data(), sizeof(float) * 4 * (size_t)c->N);
  if (quat4) std::memcpy(quat4, c->trial_quat.data(), sizeof(float) * 4 * (size_t)c->N);
  return 0;
}
int oracle_cells(void* h, uint32_t* cell_start, uint32_t* cell_pid, float* shift3) {
  Ctx* c = (Ctx*)h;
  std::memcpy(cell_start, c->cell_start.data(), sizeof(uint32_t) * c->cell_start.size());
  std::memcpy(cell_pid, c->cell_pid.data(), sizeof(uint32_t) * (size_t)c->N);
  for (int a = 0; a < 3; ++a) shift3[a] = c->shift[a];
  return 0;
}

// n sweeps (build + sweep each, step = step0 + s).  traj (optional): n x N x 4 positions after
// each sweep; outc (optional): n x N outcome codes.
int oracle_run(void* h, uint32_t seed, uint32_t step0, int64_t n, double n_R, float d_max, float a_max,
               int32_t n_trial, float* traj, uint8_t* outc) {
  Ctx* c = (Ctx*)h;
  for (int64_t s = 0; s < n; ++s) {
    oracle_build_cells(h, seed, step0 + (uint32_t)s);
    const int rc = oracle_sweep(h, seed, step0 + (uint32_t)s, n_R, d_max, a_max, n_trial);
    if (rc) return rc;
    if (traj) std::memcpy(traj + (size_t)s * c->N * 4, c->pos, sizeof(float) * 4 * (size_t)c->N);
    if (outc) std::memcpy(outc + (size_t)s * c->N, c->outcome.data(), (size_t)c->N);
  }
  return 0;
}

// Evaluate (do not commit) a prescribed move of particle i to (pos3, quat4) against the current
// cell list: returns the outcome code (2 if the new centre leaves i's cell).  Used by the
// fixed-move ratio pins.  `draw` selects an independent random stream (it replaces `step` in the key).
int oracle_eval_move(void* h, uint32_t seed, uint32_t draw, int64_t i, const float* pos3, const float* quat4,
                     double n_R, int32_t n_trial) {
  Ctx* c = (Ctx*)h;
  if (!c->built) return -3;
  const float dm = c->eval_dmax >= 0.0f ? c->eval_dmax : c->g.dmax_cap;
  const double lambda = lambda_opt(c->g, n_R, dm, c->flags);
  if (c->pt.lambda != lambda) build_poisson(c->pt, lambda);
  const V3 r0 = load_r(*c, i); const Q4 q0 = load_q(*c, i);
  const V3 r1 = V3{pos3[0], pos3[1], pos3[2]};
  const Q4 q1 = quat4 ? Q4{quat4[0], quat4[1], quat4[2], quat4[3]} : q0;
  const int64_t own = cell_of(*c, r0);
  if (cell_of(*c, r1) != own) return OUT_BOUNDARY;
  Counters cn;
  return evaluate_move(*c, seed, draw, 0, i, own, r0, q0, r1, q1, n_trial, dm, cn);
}

// Batched form of oracle_eval_move for the statistical pins: out[j] = oracle_eval_move(h, seed, draw0 + j, ...) for
// j = 0..n-1.  A plain loop over the same evaluate_move (draws are independent random streams, so the optional
// OpenMP loop changes nothing); no arithmetic of its own.
int oracle_eval_moves(void* h, uint32_t seed, uint32_t draw0, int64_t n, int64_t i, const float* pos3,
                      const float* quat4, double n_R, int32_t n_trial, uint8_t* out) {
  Ctx* c = (Ctx*)h;
  if (!c->built) return -3;
  const float dm = c->eval_dmax >= 0.0f ? c->eval_dmax : c->g.dmax_cap;
  const double lambda = lambda_opt(c->g, n_R, dm, c->flags);
  if (c->pt.lambda != lambda) build_poisson(c->pt, lambda);
  const V3 r0 = load_r(*c, i); const Q4 q0 = load_q(*c, i);
  const V3 r1 = V3{pos3[0], pos3[1], pos3[2]};
  const Q4 q1 = quat4 ? Q4{quat4[0], quat4[1], quat4[2], quat4[3]} : q0;
  const int64_t own = cell_of(*c, r0);
  const bool outside = cell_of(*c, r1) != own;
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j) {
    Counters cn;
    out[j] = outside ? (uint8_t)OUT_BOUNDARY
                     : (uint8_t)evaluate_move(*c, seed, draw0 + (uint32_t)j, 0, i, own, r0, q0, r1, q1, n_trial, dm, cn);
  }
  return 0;
}

// Free-volume measurement (Sec. IV.A, Fig. 4: the depletant density in the
// system is n_R times the free-volume fraction): n test depletants at points uniform in the box, sample s from Philox
// block (s mod 2^32, s / 2^32, 0, FREEVOL) of key (seed, step), x_a = unit01(word a) L; counted if it overlaps no
// colloid (the insertion kernel's own predicate against the 27 cells around the point; cell width >= 2 R covers the
// range).  Needs the cell list of oracle_build_cells(seed, step).
int oracle_free_volume(void* h, uint32_t seed, uint32_t step, int64_t n, uint64_t* free_count) {
  Ctx* c = (Ctx*)h;
  if (!c->built || c->b_seed != seed || c->b_step != step) return -3;
  const Geo& g = c->g;
  const int nc = c->nc;
  uint64_t cnt = 0;
#pragma omp parallel for schedule(static) reduction(+ : cnt)
  for (int64_t s = 0; s < n; ++s) {
    const U4 r = philox4x32_10((uint32_t)((uint64_t)s & 0xffffffffu), (uint32_t)((uint64_t)s >> 32), 0,
                               word3(P_FREEVOL, 0, 0), seed, step);
    const V3 p = V3{unit01(r.v[0]) * g.L, unit01(r.v[1]) * g.L, unit01(r.v[2]) * g.L};
    const int ix = cell_axis(*c, p.x, c->shift[0]), iy = cell_axis(*c, p.y, c->shift[1]), iz = cell_axis(*c, p.z, c->shift[2]);
    bool is_free = true;
    for (int dz = -1; dz <= 1 && is_free; ++dz)
      for (int dy = -1; dy <= 1 && is_free; ++dy)
        for (int dx = -1; dx <= 1 && is_free; ++dx) {
          const int jx = (ix + dx + nc) % nc, jy = (iy + dy + nc) % nc, jz = (iz + dz + nc) % nc;
          const int64_t cj = ((int64_t)jz * nc + jy) * nc + jx;
          for (uint32_t t = c->cell_start[(size_t)cj]; t < c->cell_start[(size_t)cj + 1]; ++t) {
            const int64_t j = c->cell_pid[t];
            if (dep_overlap(g, minimg(g, p, load_r(*c, j)), ori_of(g, load_q(*c, j)))) { is_free = false; break; }
          }
        }
    cnt += is_free ? 1u : 0u;
  }
  *free_count = cnt;
  return 0;
}

// Number of overlapping pairs (i<j) under the fp32 hard-overlap predicate, evaluated with i as
// the "mover" and, if both_ways != 0, also requiring the predicate with j as the mover.  Check 1.
int64_t oracle_count_overlaps(void* h, int32_t both_ways) {
  Ctx* c = (Ctx*)h;
  const Geo& g = c->g;
  // own unshifted grid of width >= dcirc
  int n = (int)std::floor((double)g.L / (double)g.dcirc);
  if (n < 1) n = 1;
  if (n > 512) n = 512;
  const float wg = g.L / (float)n;
  auto ax = [&](float x) { int k = (int)(x / wg); if (k >= n) k = n - 1; if (k < 0) k = 0; return k; };
  std::vector<std::vector<uint32_t>> bins((size_t)n * n * n);
  for (int64_t i = 0; i < c->N; ++i) {
    const V3 r = load_r(*c, i);
    bins[((size_t)ax(r.z) * n + ax(r.y)) * n + ax(r.x)].push_back((uint32_t)i);
  }
  int64_t count = 0;
  for (int64_t i = 0; i < c->N; ++i) {
    const V3 ri = load_r(*c, i); const Ori ai = ori_of(g, load_q(*c, i));
    const int ix = ax(ri.x), iy = ax(ri.y), iz = ax(ri.z);
    std::vector<int64_t> seen;
    for (int dz = -1; dz <= 1; ++dz) for (int dy = -1; dy <= 1; ++dy) for (int dx = -1; dx <= 1; ++dx) {
      const int jx = (ix + dx + n) % n, jy = (iy + dy + n) % n, jz = (iz + dz + n) % n;
      for (uint32_t j : bins[((size_t)jz * n + jy) * n + jx]) {
        if ((int64_t)j <= i) continue;
        if (std::find(seen.begin(), seen.end(), (int64_t)j) != seen.end()) continue;   // n < 3 aliasing
        seen.push_back(j);
        const Ori aj = ori_of(g, load_q(*c, j));
        bool o = pair_overlap(g, minimg(g, load_r(*c, j), ri), ai, aj);
        if (o && both_ways) o = pair_overlap(g, minimg(g, ri, load_r(*c, j)), aj, ai);
        if (o) ++count;
      }
    }
  }
  return count;
}

// ------------------------------------------------------------------ unit-level exports (pins)
void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  const U4 r = philox4x32_10(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1]);
  for (int i = 0; i < 4; ++i) out[i] = r.v[i];
}
float oracle_unit01(uint32_t x) { return unit01(x); }
float oracle_sym_unit(uint32_t x) { return sym_unit(x); }
// thresholds of the Poisson table; returns number of entries (0 if cap too small), *k_lo set
int64_t oracle_poisson_table(double lambda, int64_t* k_lo, uint64_t* T, int64_t cap) {
  PoissonTable pt; build_poisson(pt, lambda);
  *k_lo = pt.k_lo;
  if ((int64_t)pt.T.size() > cap) return -(int64_t)pt.T.size();
  std::memcpy(T, pt.T.data(), sizeof(uint64_t) * pt.T.size());
  return (int64_t)pt.T.size();
}
void oracle_poisson_draws(double lambda, const uint64_t* U, int64_t n, int64_t* out) {
  PoissonTable pt; build_poisson(pt, lambda);
  for (int64_t i = 0; i < n; ++i) out[i] = poisson_draw(pt, U[i]);
}
double oracle_lambda(const oracle_params* p, double n_R) {
  return lambda_of(make_geo(p->shape, p->sigma_c, p->disk_a, p->disk_s, p->sigma_d, p->box_L, p->d_max_cap), n_R);
}
float oracle_cbrt_fixed(float t) { return cbrt_fixed(t); }
// lambda and inner radius of the shell option for step size d_max
double oracle_shell(const oracle_params* p, double n_R, float d_max, uint32_t flags, float* Rin) {
  const Geo g = make_geo(p->shape, p->sigma_c, p->disk_a, p->disk_s, p->sigma_d, p->box_L, p->d_max_cap);
  *Rin = make_shell(g, d_max, flags | F_SHELL).Rin;
  return lambda_opt(g, n_R, d_max, flags | F_SHELL);
}
// n shell samples k = 0..n-1 of the DEPPOS stream of colloid `id`
void oracle_shell_samples(const oracle_params* p, float d_max, uint32_t seed, uint32_t step, uint32_t colour, uint32_t id,
                          int64_t n, float* out3) {
  const Geo g = make_geo(p->shape, p->sigma_c, p->disk_a, p->disk_s, p->sigma_d, p->box_L, p->d_max_cap);
  const Shell sh = make_shell(g, d_max, F_SHELL);
  uint64_t nb = 0;
  for (int64_t k = 0; k < n; ++k) {
    const V3 d = shell_sample(seed, step, P_DEPPOS, colour, id, (uint32_t)k, sh, g.Rins, nb);
    out3[3 * k] = d.x; out3[3 * k + 1] = d.y; out3[3 * k + 2] = d.z;
  }
}
// n ball samples k = 0..n-1 of the DEPPOS stream of colloid `id`
void oracle_ball_samples(uint32_t seed, uint32_t step, uint32_t colour, uint32_t id, int64_t n, float radius,
                         float* out3) {
  uint64_t nb = 0;
  for (int64_t k = 0; k < n; ++k) {
    const V3 d = ball_sample(seed, step, P_DEPPOS, colour, id, (uint32_t)k, 0, 0, radius, radius * radius, nb);
    out3[3 * k] = d.x; out3[3 * k + 1] = d.y; out3[3 * k + 2] = d.z;
  }
}
// depletant-vs-colloid predicate for n displacement vectors d (depletant centre - colloid centre)
void oracle_dep_overlap(const oracle_params* p, const float* quat4, const float* d3, int64_t n, uint8_t* out) {
  const Geo g = make_geo(p->shape, p->sigma_c, p->disk_a, p->disk_s, p->sigma_d, p->box_L, p->d_max_cap);
  const Ori a = ori_of(g, Q4{quat4[0], quat4[1], quat4[2], quat4[3]});
  for (int64_t k = 0; k < n; ++k) out[k] = dep_overlap(g, V3{d3[3 * k], d3[3 * k + 1], d3[3 * k + 2]}, a) ? 1 : 0;
}
// colloid-colloid predicate for n pairs: A at origin with qA, B at rho with qB
void oracle_pair_overlap(const oracle_params* p, const float* rho3, const float* qA4, const float* qB4, int64_t n,
                         uint8_t* out) {
  const Geo g = make_geo(p->shape, p->sigma_c, p->disk_a, p->disk_s, p->sigma_d, p->box_L, p->d_max_cap);
  for (int64_t k = 0; k < n; ++k) {
    const Ori aA = ori_of(g, Q4{qA4[4 * k], qA4[4 * k + 1], qA4[4 * k + 2], qA4[4 * k + 3]});
    const Ori aB = ori_of(g, Q4{qB4[4 * k], qB4[4 * k + 1], qB4[4 * k + 2], qB4[4 * k + 3]});
    out[k] = pair_overlap(g, V3{rho3[3 * k], rho3[3 * k + 1], rho3[3 * k + 2]}, aA, aB) ? 1 : 0;
  }
}
void oracle_support(const oracle_params* p, const float* quat4, const float* n3, float* out3) {
  const Geo g = make_geo(p->shape, p->sigma_c, p->disk_a, p->disk_s, p->sigma_d, p->box_L, p->d_max_cap);
  const V3 s = support(g, ori_of(g, Q4{quat4[0], quat4[1], quat4[2], quat4[3]}), V3{n3[0], n3[1], n3[2]});
  out3[0] = s.x; out3[1] = s.y; out3[2] = s.z;
}
void oracle_quat_axis(const float* q, float* out3) {
  const V3 a = quat_axis(Q4{q[0], q[1], q[2], q[3]});
  out3[0] = a.x; out3[1] = a.y; out3[2] = a.z;
}
void oracle_rotate_cayley(const float* q, const float* v3, float* out4) {
  const Q4 r = rotate_cayley(Q4{q[0], q[1], q[2], q[3]}, V3{v3[0], v3[1], v3[2]});
  out4[0] = r.w; out4[1] = r.x; out4[2] = r.y; out4[3] = r.z;
}

}  // extern "C"
