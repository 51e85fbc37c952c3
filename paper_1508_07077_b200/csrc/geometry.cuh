// geometry.cuh -- fp32 shape arithmetic of the hot path.  Compiled with --fmad=false: no contraction; an FMA
// happens only where fmaf() is written (dot3).  Division and square root are IEEE (__fdiv_rn, __fsqrt_rn).
//   depletant-vs-colloid tests: sphere; point-to-half-ball (R-S16); point-to-disc (R-S17)
//   colloid-vs-colloid: sphere distance; support-function MPR test for the convex shapes (R-S18)
//   rotation: Cayley move (R-S6), body axis from the quaternion (R-S19)
// Paper: the overlap tests realise U_ij = infinity for overlapping pairs in Eq. 5 (L80) and the
// colloid-depletant overlap of Fig. 2 (L72); the paper gives no algorithm for them (ref. 35).
#pragma once
#include <cuda_runtime.h>

namespace hpmc {

enum : int { SH_SPHERE = 0, SH_HALFBALL = 1, SH_SPHERODISK = 2, SH_ELLIPSOID = 3, SH_TETRAHEDRON = 4 };

struct Geo {              // derived constants, computed once on the host in fp32
  float L, halfL, w;      // box edge, L/2, cell width
  int nc;                 // cells per axis
  float Rins, Rins2;      // insertion-sphere radius (sigma_c+sigma_d)/2 and square
  float dcirc2;           // sigma_c^2
  float rcut2;            // neighbour pre-filter radius squared
  float rd, rd2;          // depletant radius
  float Rh, cen;          // half-ball radius and interior-point offset 3 Rh / 8
  float adisk, sdisk, rs2;  // spherodisk: disk radius, rounding radius, (s + r_d)^2; ellipsoid: semi-axes A >= C in adisk, sdisk
};

struct V3 { float x, y, z; };

__device__ __forceinline__ V3 v3(float x, float y, float z) { return V3{x, y, z}; }
__device__ __forceinline__ V3 operator+(V3 a, V3 b) { return V3{a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ V3 operator-(V3 a, V3 b) { return V3{a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ V3 operator*(V3 a, float s) { return V3{a.x * s, a.y * s, a.z * s}; }
__device__ __forceinline__ V3 neg(V3 a) { return V3{-a.x, -a.y, -a.z}; }
__device__ __forceinline__ float dot3(V3 a, V3 b) { return fmaf(a.z, b.z, fmaf(a.y, b.y, a.x * b.x)); }
__device__ __forceinline__ V3 cross3(V3 a, V3 b) {
  return V3{a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
__device__ __forceinline__ bool is_zero(V3 a) { return a.x == 0.0f && a.y == 0.0f && a.z == 0.0f; }

// Quaternion (w,x,y,z); stored in memory as float4 with .x = w, .y = x, .z = y, .w = z.
struct Q4 { float w, x, y, z; };
__device__ __forceinline__ Q4 as_q(float4 f) { return Q4{f.x, f.y, f.z, f.w}; }
__device__ __forceinline__ float4 as_f4(Q4 q) { return make_float4(q.w, q.x, q.y, q.z); }

// body z axis in the space frame: third column of the rotation matrix of q (R-S19)
__device__ __forceinline__ V3 quat_axis(Q4 q) {
  return V3{2.0f * (q.x * q.z + q.w * q.y), 2.0f * (q.y * q.z - q.w * q.x), 1.0f - 2.0f * (q.x * q.x + q.y * q.y)};
}

// Orientation as the shape tests need it: the body z axis (x, y, z; w unused) for the bodies of revolution (R-S19), the
// whole unit quaternion (x = q.w, y = q.x, z = q.y, w = q.z) for the tetrahedron (R-N2b).  One float4 either way: the
// cell-ordered orientation array, the shared-memory records and the neighbour pool hold it as it is.
struct Ori { float x, y, z, w; };
template <int SHAPE>
__device__ __forceinline__ Ori ori_of(Q4 q) {
  if (SHAPE == SH_TETRAHEDRON) return Ori{q.w, q.x, q.y, q.z};
  const V3 a = quat_axis(q);
  return Ori{a.x, a.y, a.z, 0.0f};
}
__device__ __forceinline__ Ori as_ori(float4 f) { return Ori{f.x, f.y, f.z, f.w}; }
__device__ __forceinline__ float4 as_f4(Ori o) { return make_float4(o.x, o.y, o.z, o.w); }
__device__ __forceinline__ V3 axis_of(Ori o) { return V3{o.x, o.y, o.z}; }

// Cayley rotation move (R-S6): q' = normalise((1,v) (x) q), multiplication on the left (space frame)
__device__ __forceinline__ Q4 rotate_cayley(Q4 q, V3 v) {
  const float pw = q.w - ((v.x * q.x + v.y * q.y) + v.z * q.z);
  const float px = (q.x + v.x * q.w) + (v.y * q.z - v.z * q.y);
  const float py = (q.y + v.y * q.w) + (v.z * q.x - v.x * q.z);
  const float pz = (q.z + v.z * q.w) + (v.x * q.y - v.y * q.x);
  const float n2 = (pw * pw + px * px) + (py * py + pz * pz);
  const float n = __fsqrt_rn(n2);
  return Q4{__fdiv_rn(pw, n), __fdiv_rn(px, n), __fdiv_rn(py, n), __fdiv_rn(pz, n)};
}

// R-N2b: regular tetrahedron, circumradius Rh = sigma_c / 2, body-frame vertices s u_i with s = Rh 0.57735026f and
// u_0 = (1,1,1), u_1 = (1,-1,-1), u_2 = (-1,1,-1), u_3 = (-1,-1,1); the face opposite vertex i lies in the plane u_i . x = -s.
struct Frame { V3 ex, ey, ez; };               // body axes in the space frame: columns of the rotation matrix of q
__device__ __forceinline__ Frame frame_of(Ori o) {
  const float w = o.x, x = o.y, y = o.z, z = o.w;
  Frame f;
  f.ex = V3{1.0f - 2.0f * (y * y + z * z), 2.0f * (x * y + w * z), 2.0f * (x * z - w * y)};
  f.ey = V3{2.0f * (x * y - w * z), 1.0f - 2.0f * (x * x + z * z), 2.0f * (y * z + w * x)};
  f.ez = V3{2.0f * (x * z + w * y), 2.0f * (y * z - w * x), 1.0f - 2.0f * (x * x + y * y)};
  return f;
}
__device__ __forceinline__ V3 tet_u(int i) {
  return V3{(i & 2) ? -1.0f : 1.0f, (i == 1 || i == 3) ? -1.0f : 1.0f, (i == 1 || i == 2) ? -1.0f : 1.0f};
}
// squared distance from p to the triangle (a, b, c): closest-point regions by barycentric signs, only + x /
__device__ __forceinline__ float tri_dist2(V3 p, V3 a, V3 b, V3 c) {
  const V3 ab = b - a, ac = c - a, ap = p - a;
  const float d1 = dot3(ab, ap), d2 = dot3(ac, ap);
  if (d1 <= 0.0f && d2 <= 0.0f) return dot3(ap, ap);
  const V3 bp = p - b;
  const float d3 = dot3(ab, bp), d4 = dot3(ac, bp);
  if (d3 >= 0.0f && d4 <= d3) return dot3(bp, bp);
  const float vc = d1 * d4 - d3 * d2;
  if (vc <= 0.0f && d1 >= 0.0f && d3 <= 0.0f) { const float v = __fdiv_rn(d1, d1 - d3); const V3 e = ap - ab * v; return dot3(e, e); }
  const V3 cp = p - c;
  const float d5 = dot3(ab, cp), d6 = dot3(ac, cp);
  if (d6 >= 0.0f && d5 <= d6) return dot3(cp, cp);
  const float vb = d5 * d2 - d1 * d6;
  if (vb <= 0.0f && d2 >= 0.0f && d6 <= 0.0f) { const float w = __fdiv_rn(d2, d2 - d6); const V3 e = ap - ac * w; return dot3(e, e); }
  const float va = d3 * d6 - d5 * d4;
  if (va <= 0.0f && (d4 - d3) >= 0.0f && (d5 - d6) >= 0.0f) {
    const float w = __fdiv_rn(d4 - d3, (d4 - d3) + (d5 - d6));
    const V3 e = bp - (c - b) * w;
    return dot3(e, e);
  }
  const float den = __fdiv_rn(1.0f, va + vb + vc);
  const float v = vb * den, w = vc * den;
  const V3 e = ap - (ab * v + ac * w);
  return dot3(e, e);
}
// depletant centre at body-frame point b vs the tetrahedron: inside, or closer than r_d to a face it lies in front of
__device__ __forceinline__ bool near_tetrahedron(float s, float rd2, V3 b) {
  bool inside = true;
  float best = 3.0e38f;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const V3 u = tet_u(i);
    const float h = (u.x * b.x + u.y * b.y) + u.z * b.z;
    if (h < -s) {
      inside = false;
      const float d2 = tri_dist2(b, tet_u((i + 1) & 3) * s, tet_u((i + 2) & 3) * s, tet_u((i + 3) & 3) * s);
      if (d2 < best) best = d2;
    }
  }
  return inside || best < rd2;
}

// R-N2 (oblate spheroid x^2/A^2 + z^2/C^2 <= 1 in cylindrical body coordinates, the paper's discoids L228): is the point
// (rho, z >= 0) closer than r_d to the solid?  Inside: yes.  Outside: the closest point of the ellipse is
// (A^2 rho/(t + A^2), C^2 z/(t + C^2)) for the root t of F(t) = (A rho/(t + A^2))^2 + (C z/(t + C^2))^2 - 1 (convex,
// decreasing); six Newton steps from the lower bound max(A rho - A^2, C z - C^2), IEEE division throughout.
__device__ __forceinline__ bool near_spheroid(float A, float Cc, float rd2, float rho, float z) {
  const float qa = __fdiv_rn(rho, A), qc = __fdiv_rn(z, Cc);
  if (fmaf(qa, qa, qc * qc) <= 1.0f) return true;
  const float A2 = A * A, C2 = Cc * Cc, ar = A * rho, cz = Cc * z;
  float t = ar - A2;
  const float t1 = cz - C2;
  if (t1 > t) t = t1;
#pragma unroll 1
  for (int it = 0; it < 6; ++it) {
    const float ia = __fdiv_rn(1.0f, t + A2), ic = __fdiv_rn(1.0f, t + C2);
    const float ua = ar * ia, uc = cz * ic;
    const float ua2 = ua * ua, uc2 = uc * uc;
    const float F = (ua2 + uc2) - 1.0f;
    const float dF = -2.0f * (ua2 * ia + uc2 * ic);
    t = t - __fdiv_rn(F, dF);
  }
  const float ex = rho - __fdiv_rn(A2 * rho, t + A2), ez = z - __fdiv_rn(C2 * z, t + C2);
  return fmaf(ex, ex, ez * ez) < rd2;
}

// Does a depletant centred at d (relative to the colloid centre) overlap the colloid with body axis a?
template <int SHAPE>
__device__ __forceinline__ bool dep_overlap(const Geo& g, V3 d, Ori o) {
  const float d2 = dot3(d, d);
  if (!(d2 < g.Rins2)) return false;
  if (SHAPE == SH_SPHERE) return true;
  if (SHAPE == SH_TETRAHEDRON) {
    const Frame f = frame_of(o);
    return near_tetrahedron(g.Rh * 0.57735026f, g.rd2, V3{dot3(d, f.ex), dot3(d, f.ey), dot3(d, f.ez)});
  }
  const V3 a = axis_of(o);
  const float bz = dot3(d, a);
  if (SHAPE == SH_ELLIPSOID) {
    const V3 p = V3{d.x - bz * a.x, d.y - bz * a.y, d.z - bz * a.z};
    return near_spheroid(g.adisk, g.sdisk, g.rd2, __fsqrt_rn(dot3(p, p)), fabsf(bz));
  }
  if (SHAPE == SH_HALFBALL) {
    if (bz <= 0.0f) return true;
    const V3 p = V3{d.x - bz * a.x, d.y - bz * a.y, d.z - bz * a.z};
    const float rho = __fsqrt_rn(dot3(p, p));
    if (rho <= g.Rh) return bz < g.rd;
    const float e = rho - g.Rh;
    return fmaf(e, e, bz * bz) < g.rd2;
  }
  const V3 p = V3{d.x - bz * a.x, d.y - bz * a.y, d.z - bz * a.z};
  const float rho = __fsqrt_rn(dot3(p, p));
  if (rho <= g.adisk) return bz * bz < g.rs2;
  const float e = rho - g.adisk;
  return fmaf(e, e, bz * bz) < g.rs2;
}

template <int SHAPE>
__device__ __forceinline__ V3 support(const Geo& g, Ori o, V3 n) {
  if (SHAPE == SH_TETRAHEDRON) {               // the vertex with the largest projection (first one on ties)
    const Frame f = frame_of(o);
    const V3 nb = V3{dot3(n, f.ex), dot3(n, f.ey), dot3(n, f.ez)};
    int best = 0;
    float hb = (nb.x + nb.y) + nb.z;
#pragma unroll
    for (int i = 1; i < 4; ++i) {
      const V3 u = tet_u(i);
      const float h = (u.x * nb.x + u.y * nb.y) + u.z * nb.z;
      if (h > hb) { hb = h; best = i; }
    }
    const float s = g.Rh * 0.57735026f;
    const V3 u = tet_u(best);
    return (f.ex * (s * u.x) + f.ey * (s * u.y)) + f.ez * (s * u.z);
  }
  const V3 a = axis_of(o);
  const float nz = dot3(n, a);
  if (SHAPE == SH_HALFBALL) {
    if (nz <= 0.0f) {
      const float len = __fsqrt_rn(dot3(n, n));
      if (!(len > 0.0f)) return V3{0.0f, 0.0f, 0.0f};
      return n * __fdiv_rn(g.Rh, len);
    }
    const V3 p = V3{n.x - nz * a.x, n.y - nz * a.y, n.z - nz * a.z};
    const float l = __fsqrt_rn(dot3(p, p));
    if (!(l > 0.0f)) return V3{0.0f, 0.0f, 0.0f};
    return p * __fdiv_rn(g.Rh, l);
  }
  if (SHAPE == SH_ELLIPSOID) {               // (A^2 n_perp + C^2 n_par a) / sqrt(A^2 |n_perp|^2 + C^2 n_par^2)
    const V3 p = V3{n.x - nz * a.x, n.y - nz * a.y, n.z - nz * a.z};
    const float A2 = g.adisk * g.adisk, C2 = g.sdisk * g.sdisk;
    const float den = __fsqrt_rn(A2 * dot3(p, p) + C2 * (nz * nz));
    if (!(den > 0.0f)) return V3{0.0f, 0.0f, 0.0f};
    const float wa = __fdiv_rn(A2, den), wc = __fdiv_rn(C2 * nz, den);
    return V3{wa * p.x + wc * a.x, wa * p.y + wc * a.y, wa * p.z + wc * a.z};
  }
  const V3 p = V3{n.x - nz * a.x, n.y - nz * a.y, n.z - nz * a.z};
  const float l = __fsqrt_rn(dot3(p, p));
  const float len = __fsqrt_rn(dot3(n, n));
  V3 out = V3{0.0f, 0.0f, 0.0f};
  if (l > 0.0f) out = p * __fdiv_rn(g.adisk, l);
  if (len > 0.0f) out = out + n * __fdiv_rn(g.sdisk, len);
  return out;
}

template <int SHAPE>
__device__ __forceinline__ V3 support_diff(const Geo& g, V3 rho, Ori aA, Ori aB, V3 n) {
  const V3 sb = support<SHAPE>(g, aB, n);
  const V3 sa = support<SHAPE>(g, aA, neg(n));
  return (sb + rho) - sa;
}

#define HPMC_MPR_MAXIT 48
#define HPMC_MPR_TOL 1e-5f

// Minkowski portal refinement on the full convex shapes: A at the origin (axis aA), B at rho (axis aB).
template <int SHAPE>
__device__ __noinline__ bool mpr_overlap(const Geo& g, V3 rho, Ori aA, Ori aB) {
  V3 cA = V3{0.0f, 0.0f, 0.0f}, cB = rho;
  if (SHAPE == SH_HALFBALL) {
    cA = neg(axis_of(aA) * g.cen);
    cB = rho - axis_of(aB) * g.cen;
  }
  V3 v0 = cB - cA;
  if (is_zero(v0)) v0 = V3{1e-5f, 0.0f, 0.0f};
  V3 n = neg(v0);
  V3 v1 = support_diff<SHAPE>(g, rho, aA, aB, n);
  if (dot3(v1, n) <= 0.0f) return false;
  n = cross3(v1, v0);
  if (is_zero(n)) return true;
  V3 v2 = support_diff<SHAPE>(g, rho, aA, aB, n);
  if (dot3(v2, n) <= 0.0f) return false;
  n = cross3(v1 - v0, v2 - v0);
  if (dot3(n, v0) > 0.0f) { const V3 t = v1; v1 = v2; v2 = t; n = neg(n); }
  V3 v3;
  int it = 0;
  for (;;) {
    if (it++ >= HPMC_MPR_MAXIT) return true;
    v3 = support_diff<SHAPE>(g, rho, aA, aB, n);
    if (dot3(v3, n) <= 0.0f) return false;
    if (dot3(cross3(v1, v3), v0) < 0.0f) { v2 = v3; n = cross3(v1 - v0, v3 - v0); continue; }
    if (dot3(cross3(v3, v2), v0) < 0.0f) { v1 = v3; n = cross3(v3 - v0, v2 - v0); continue; }
    break;
  }
  for (it = 0;; ++it) {
    if (it >= HPMC_MPR_MAXIT) return true;
    n = cross3(v2 - v1, v3 - v1);
    const float len = __fsqrt_rn(dot3(n, n));
    if (!(len > 0.0f)) return true;
    n = V3{__fdiv_rn(n.x, len), __fdiv_rn(n.y, len), __fdiv_rn(n.z, len)};
    if (dot3(n, v1) >= 0.0f) return true;
    const V3 v4 = support_diff<SHAPE>(g, rho, aA, aB, n);
    if (dot3(v4, n) < 0.0f) return false;
    if (dot3(v4 - v3, n) <= HPMC_MPR_TOL) return false;
    const V3 c = cross3(v4, v0);
    if (dot3(v1, c) > 0.0f) {
      if (dot3(v2, c) > 0.0f) v1 = v4; else v3 = v4;
    } else {
      if (dot3(v3, c) > 0.0f) v2 = v4; else v1 = v4;
    }
  }
}

template <int SHAPE>
__device__ __forceinline__ bool pair_overlap(const Geo& g, V3 rho, Ori aA, Ori aB) {
  const float r2 = dot3(rho, rho);
  if (!(r2 < g.dcirc2)) return false;
  if (SHAPE == SH_SPHERE) return true;
  return mpr_overlap<SHAPE>(g, rho, aA, aB);
}

// periodic helpers (R-S13)
__device__ __forceinline__ float minimg1(const Geo& g, float d) {
  if (d > g.halfL) d -= g.L; else if (d < -g.halfL) d += g.L;
  return d;
}
__device__ __forceinline__ float wrap1(const Geo& g, float x) {
  if (x < 0.0f) x += g.L;
  if (x >= g.L) x -= g.L;
  return x;
}
__device__ __forceinline__ int cell_axis(const Geo& g, float x, float shift) {
  float t = x - shift;
  if (t < 0.0f) t += g.L;
  int c = (int)__fdiv_rn(t, g.w);
  if (c >= g.nc) c = g.nc - 1;
  return c;
}

}  // namespace hpmc
