"""Pins for the oracle's shape layer (CPU only): depletant-colloid predicates (S16, S17), support
functions and the convex-convex overlap test (S18), rotation algebra (S6, S19).

References used are independent of the oracle's code path: Steiner volumes (closed form), dense point
clouds of the solids (brute force), scipy's Rotation, closed-form contact distances, and an fp64 convex
program (scipy SLSQP) for random pair poses.
"""
import ctypes as C
import math
import os

import numpy as np
import pytest
from scipy.optimize import minimize
from scipy.spatial import cKDTree
from scipy.spatial.transform import Rotation

import oracle
from oracle.binding import make_params

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(key):
    with open(os.path.join(GOLD, "paper_values.txt")) as f:
        for line in f:
            if line.startswith(key + " "):
                return float(line.split()[1])
    raise KeyError(key)


HB = dict(shape="halfball", sigma_c=1.0, sigma_d=0.2, box_L=20.0, d_max_cap=0.1)
SD = dict(shape="spherodisk", sigma_c=1.0, sigma_d=0.15, box_L=20.0, d_max_cap=0.1, disk_a=0.4, disk_s=0.1)
SP = dict(shape="sphere", sigma_c=1.0, sigma_d=0.2, box_L=20.0, d_max_cap=0.1)
# the paper's discoids (L228): oblate ellipsoids a = b = 0.5, c = 0.25, depletant radius 0.25 (disk_a = A, disk_s = C)
# regular tetrahedron with circumradius 0.5 (Fig. 1 L21, reading R-N2b)
TE = dict(shape="tetrahedron", sigma_c=1.0, sigma_d=0.2, box_L=20.0, d_max_cap=0.1)
TET_V = (0.5 / math.sqrt(3.0)) * np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], np.float64)
EL = dict(shape="ellipsoid", sigma_c=1.0, sigma_d=0.5, box_L=20.0, d_max_cap=0.1, disk_a=0.5, disk_s=0.25)


def rand_quats(n, rng):
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    return q.astype(np.float32)


def q_to_R(q):
    """(w,x,y,z) -> scipy Rotation (scalar-last there)."""
    q = np.asarray(q, np.float64)
    return Rotation.from_quat(np.r_[q[1:], q[0]])


def dep_overlap(params, quat, d):
    p = make_params(**params)
    q = np.ascontiguousarray(quat, np.float32)
    d = np.ascontiguousarray(d, np.float32)
    out = np.zeros(len(d), np.uint8)
    oracle.lib().oracle_dep_overlap(C.byref(p), q.ctypes.data, d.ctypes.data, len(d), out.ctypes.data)
    return out.astype(bool)


def pair_overlap(params, rho, qA, qB):
    p = make_params(**params)
    rho = np.ascontiguousarray(np.atleast_2d(rho), np.float32)
    qA = np.ascontiguousarray(np.atleast_2d(qA), np.float32)
    qB = np.ascontiguousarray(np.atleast_2d(qB), np.float32)
    out = np.zeros(len(rho), np.uint8)
    oracle.lib().oracle_pair_overlap(C.byref(p), rho.ctypes.data, qA.ctypes.data, qB.ctypes.data, len(rho),
                                     out.ctypes.data)
    return out.astype(bool)


def shape_cloud(params, n, rng):
    """Dense fp64 point cloud of the solid in its body frame (volume + boundary points)."""
    if params["shape"] == "halfball":
        R = 0.5 * params["sigma_c"]
        v = rng.standard_normal((n, 3))
        v /= np.linalg.norm(v, axis=1, keepdims=True)
        vol = v * (R * rng.random((n, 1)) ** (1 / 3))
        vol[:, 2] = -np.abs(vol[:, 2])
        dome = v * R
        dome[:, 2] = -np.abs(dome[:, 2])
        ang, rad = rng.random(n) * 2 * np.pi, R * np.sqrt(rng.random(n))
        face = np.stack([rad * np.cos(ang), rad * np.sin(ang), np.zeros(n)], -1)
        rim = np.stack([R * np.cos(ang), R * np.sin(ang), np.zeros(n)], -1)
        return np.concatenate([vol, dome, face, rim])
    if params["shape"] == "tetrahedron":
        def bary(k, m):
            w = rng.dirichlet(np.ones(k), m)
            return w
        vol = bary(4, n) @ TET_V
        faces = np.concatenate([bary(3, n // 2) @ TET_V[[j for j in range(4) if j != i]] for i in range(4)])
        edges = np.concatenate([bary(2, n // 8) @ TET_V[[i, j]] for i in range(4) for j in range(i + 1, 4)])
        return np.concatenate([vol, faces, edges, TET_V])
    if params["shape"] == "ellipsoid":
        A, Cc = params["disk_a"], params["disk_s"]
        v = rng.standard_normal((n, 3))
        v /= np.linalg.norm(v, axis=1, keepdims=True)
        sc = np.array([A, A, Cc])
        # surface points (denser near the equator, where curvature is highest) and interior points
        th = rng.random(n) * np.pi
        ph = rng.random(n) * 2 * np.pi
        eq = np.stack([A * np.sin(th) * np.cos(ph), A * np.sin(th) * np.sin(ph), Cc * np.cos(th)], -1)
        return np.concatenate([v * sc, eq, v * sc * rng.random((n, 1)) ** (1 / 3)])
    a, s = params["disk_a"], params["disk_s"]
    ang, rad = rng.random(n) * 2 * np.pi, a * np.sqrt(rng.random(n))
    disk = np.stack([rad * np.cos(ang), rad * np.sin(ang), np.zeros(n)], -1)
    disk[: n // 4, :2] *= (a / np.maximum(1e-12, np.linalg.norm(disk[: n // 4, :2], axis=1)))[:, None]   # rim
    v = rng.standard_normal((n, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    return np.concatenate([disk + s * v, disk + s * v * rng.random((n, 1))])


# ----------------------------------------------------------------------------------- depletant tests
@pytest.mark.parametrize("params,key", [(HB, "halfball_steiner_fraction"), (SD, "spherodisk_steiner_fraction")])
def test_dilated_volume_steiner(olib, params, key):
    """Fraction of insertion-ball samples that overlap the shape = Steiner volume / ball volume."""
    n = 1000000
    R = 0.5 * (params["sigma_c"] + params["sigma_d"])
    d = np.zeros((n, 3), np.float32)
    olib.oracle_ball_samples(3, 1, 0, 77, n, R, d.ctypes.data)
    q = rand_quats(1, np.random.default_rng(5))[0]
    frac = dep_overlap(params, q, d).mean()
    want = _gold(key)
    assert abs(frac - want) < 4.5 * math.sqrt(want * (1 - want) / n) + 2e-5


def _spheroid_steiner_volume(A, Cc, r):
    """Volume of the oblate spheroid (A, A, Cc) dilated by a ball of radius r: V + S r + M r^2 + 4 pi r^3 / 3 (Steiner),
    with the surface area S and the integrated mean curvature M = 2 pi x (mean width) by quadrature of their closed-form
    integrands: surface of revolution (A sin t, Cc cos t); support function h(t) = sqrt(A^2 sin^2 t + Cc^2 cos^2 t)."""
    from scipy.integrate import quad
    V = 4.0 * math.pi * A * A * Cc / 3.0
    S = quad(lambda t: 2 * math.pi * A * math.sin(t) * math.sqrt((A * math.cos(t)) ** 2 + (Cc * math.sin(t)) ** 2), 0, math.pi)[0]
    M = 2 * math.pi * quad(lambda t: math.sqrt((A * math.sin(t)) ** 2 + (Cc * math.cos(t)) ** 2) * math.sin(t), 0, math.pi)[0]
    return V + S * r + M * r * r + 4.0 * math.pi * r ** 3 / 3.0


def test_steiner_formula_on_spheres_and_dilated_volume_ellipsoid(olib):
    """R-N2: fraction of insertion-ball samples that overlap the ellipsoid = Steiner volume / ball volume (4.5 sigma at 1e6).
    The quadrature itself is checked on the sphere (A = Cc), where the Steiner sum is 4 pi (A + r)^3 / 3."""
    assert abs(_spheroid_steiner_volume(0.5, 0.5, 0.25) / (4 * math.pi * 0.75 ** 3 / 3) - 1) < 1e-9
    n = 1000000
    R = 0.5 * (EL["sigma_c"] + EL["sigma_d"])
    d = np.zeros((n, 3), np.float32)
    olib.oracle_ball_samples(3, 1, 0, 79, n, R, d.ctypes.data)
    for seed in (5, 6):
        q = rand_quats(1, np.random.default_rng(seed))[0]
        frac = dep_overlap(EL, q, d).mean()
        want = _spheroid_steiner_volume(EL["disk_a"], EL["disk_s"], 0.5 * EL["sigma_d"]) / (4 * math.pi * R ** 3 / 3)
        assert abs(frac - want) < 4.5 * math.sqrt(want * (1 - want) / n) + 2e-5, (frac, want)


def test_dilated_volume_and_contacts_tetrahedron(olib):
    """R-N2b.  Steiner volume of the regular tetrahedron (edge a = R sqrt(8/3)) dilated by r: V + S r + M r^2 + 4 pi r^3/3
    with V = a^3/(6 sqrt 2), S = sqrt(3) a^2, M = (1/2) sum over edges of length x (pi - dihedral) = 3 a (pi - arccos(1/3));
    the fraction of insertion-ball samples that overlap must match (4.5 sigma at 1e6).  Contacts of two equally oriented
    tetrahedra (B = A + t): they overlap iff t lies inside A (+) (-A), i.e. |t| < h_A(n) + h_A(-n) along n:
    2 s along a body axis (edge midpoints: s = R/sqrt 3), R + R/3 along a vertex direction."""
    R, r = 0.5, 0.1
    a = R * math.sqrt(8.0 / 3.0)
    vdil = a ** 3 / (6 * math.sqrt(2)) + math.sqrt(3) * a * a * r + 3 * a * (math.pi - math.acos(1 / 3)) * r * r + 4 * math.pi * r ** 3 / 3
    n = 1000000
    d = np.zeros((n, 3), np.float32)
    olib.oracle_ball_samples(3, 1, 0, 80, n, 0.6, d.ctypes.data)
    want = vdil / (4 * math.pi * 0.6 ** 3 / 3)
    for seed in (5, 6):
        q = rand_quats(1, np.random.default_rng(seed))[0]
        frac = dep_overlap(TE, q, d).mean()
        assert abs(frac - want) < 4.5 * math.sqrt(want * (1 - want) / n) + 2e-5, (frac, want)
    ident = np.array([1, 0, 0, 0], np.float32)
    s = R / math.sqrt(3)
    for gap in (-0.05, -0.002, 0.002, 0.05):
        assert pair_overlap(TE, [2 * s + gap, 0, 0], ident, ident)[0] == (gap < 0)
        t = (R + R / 3 + gap) / math.sqrt(3)
        assert pair_overlap(TE, [t, t, t], ident, ident)[0] == (gap < 0)
        assert pair_overlap(TE, [-t, -t, -t], ident, ident)[0] == (gap < 0)


def test_ellipsoid_depletant_test_at_the_largest_aspect_ratio(olib):
    """R-N2: the closest point of the ellipse comes from a fixed six Newton steps, so accuracy depends on the aspect
    ratio; 4 is the largest the library and the oracle accept.  At A = 0.5, C = 0.125 the predicate must agree with the
    distance from a root finder (scipy brentq on F(t), fp64) for every point farther than 2e-6 from the decision surface,
    for a small, a matching and a large depletant; aspect 5 is refused."""
    from scipy.optimize import brentq
    A, Cc = 0.5, 0.125
    rng = np.random.default_rng(21)
    for sigma_d in (0.06, 0.25, 1.0):
        par = dict(EL, disk_s=Cc, sigma_d=sigma_d)
        rd, R = 0.5 * sigma_d, 0.5 + 0.5 * sigma_d
        pts = (rng.random((6000, 3)) * 2 - 1) * R
        rho, z = np.hypot(pts[:, 0], pts[:, 1]), np.abs(pts[:, 2])
        dist = np.zeros(len(pts))
        for k in range(len(pts)):
            if (rho[k] / A) ** 2 + (z[k] / Cc) ** 2 <= 1.0:
                continue
            F = lambda t: (A * rho[k] / (t + A * A)) ** 2 + (Cc * z[k] / (t + Cc * Cc)) ** 2 - 1.0
            lo = max(A * rho[k] - A * A, Cc * z[k] - Cc * Cc)
            t = brentq(F, lo, lo + 100.0, xtol=1e-15)
            dist[k] = math.hypot(rho[k] - A * A * rho[k] / (t + A * A), z[k] - Cc * Cc * z[k] / (t + Cc * Cc))
        want = (dist < rd) & (np.linalg.norm(pts, axis=1) < R)
        got = dep_overlap(par, np.array([1, 0, 0, 0], np.float32), pts)
        clear = (np.abs(dist - rd) > 2e-6) & (np.abs(np.linalg.norm(pts, axis=1) - R) > 2e-6)
        assert clear.sum() > 5900 and want[clear].sum() > 500 and (~want[clear]).sum() > 500
        assert np.array_equal(got[clear], want[clear]), (sigma_d, int((got[clear] != want[clear]).sum()))
    p4 = np.zeros((1, 4), np.float32); p4[0, :3] = 5.0
    q4 = np.array([[1, 0, 0, 0]], np.float32)
    ok = olib.oracle_create(C.byref(make_params(**dict(EL, disk_s=0.125))), 1, p4.ctypes.data, q4.ctypes.data)
    assert ok
    olib.oracle_destroy(ok)
    assert not olib.oracle_create(C.byref(make_params(**dict(EL, disk_s=0.1))), 1, p4.ctypes.data, q4.ctypes.data)


def test_pair_overlap_closed_forms_ellipsoid():
    """Coaxial spheroids overlap iff |dz| < 2 C; coplanar ones (same axis, separation in the equatorial plane) iff the
    distance is < 2 A; an edge-on spheroid above a flat one (axes perpendicular) iff the gap is < A + C."""
    A, Cc = EL["disk_a"], EL["disk_s"]
    z, x = quat_from_axis([0, 0, 1]), quat_from_axis([1, 0, 0])
    for gap in (-0.05, -0.002, 0.002, 0.05):
        assert pair_overlap(EL, [0, 0, 2 * Cc + gap], z, z)[0] == (gap < 0)
        assert pair_overlap(EL, [2 * A + gap, 0, 0], z, z)[0] == (gap < 0)
        assert pair_overlap(EL, [0, 0, A + Cc + gap], z, x)[0] == (gap < 0)


def test_dilated_volume_sphere(olib):
    n = 100000
    d = np.zeros((n, 3), np.float32)
    olib.oracle_ball_samples(3, 1, 0, 78, n, 0.6, d.ctypes.data)
    assert dep_overlap(SP, [1, 0, 0, 0], d).mean() > 0.9999
    assert not dep_overlap(SP, [1, 0, 0, 0], np.array([[0.6, 0.0, 0.0], [0.4, 0.4, 0.3]], np.float32)).any()


def test_spherodisk_volume_formula():
    import workloads
    assert abs(workloads.spherodisk_volume(0.4, 0.1) - _gold("spherodisk_volume")) < 1e-6


@pytest.mark.parametrize("params", [HB, SD, EL, TE])
def test_dep_overlap_vs_point_cloud(params):
    """Predicate == (distance from the depletant centre to the solid < r_d), by brute force."""
    rng = np.random.default_rng(11)
    cloud = shape_cloud(params, 150000, rng)
    tree = cKDTree(cloud)
    rd = 0.5 * params["sigma_d"]
    q = rand_quats(1, rng)[0]
    Rm = q_to_R(q)
    pts_body = (rng.random((4000, 3)) - 0.5) * 1.5
    dist, _ = tree.query(pts_body)
    pts_world = Rm.apply(pts_body)
    got = dep_overlap(params, q, pts_world)
    band = 0.012                                    # cloud resolution
    sure_in, sure_out = dist < rd - band, dist > rd + band
    assert sure_in.sum() > 200 and sure_out.sum() > 300
    assert got[sure_in].all()
    assert not got[sure_out].any()


# ----------------------------------------------------------------------------------- support function
@pytest.mark.parametrize("params", [HB, SD, EL, TE])
def test_support_is_argmax_over_cloud(olib, params):
    rng = np.random.default_rng(12)
    cloud = shape_cloud(params, 100000, rng)
    p = make_params(**params)
    for _ in range(40):
        q = rand_quats(1, rng)[0]
        n = (rng.standard_normal(3) * rng.choice([0.01, 1.0, 30.0])).astype(np.float32)
        out = np.zeros(3, np.float32)
        olib.oracle_support(C.byref(p), q.ctypes.data, n.ctypes.data, out.ctypes.data)
        world = q_to_R(q).apply(cloud)
        nn = n.astype(np.float64) / np.linalg.norm(n)
        h_cloud = (world @ nn).max()
        h = float(out.astype(np.float64) @ nn)
        assert h >= h_cloud - 1e-5                  # no point of the solid lies beyond the support plane
        assert h <= h_cloud + 0.01                  # and the support point is (nearly) attained by the cloud
    # special directions
    ident = np.array([1, 0, 0, 0], np.float32)
    for n, want in (([0, 0, 1], None), ([0, 0, -1], None), ([1, 0, 0], None)):
        out = np.zeros(3, np.float32)
        nv = np.array(n, np.float32)
        olib.oracle_support(C.byref(p), ident.ctypes.data, nv.ctypes.data, out.ctypes.data)
        if params["shape"] == "halfball":
            exp = {(0, 0, 1): 0.0, (0, 0, -1): 0.5, (1, 0, 0): 0.5}[tuple(n)]
        elif params["shape"] == "ellipsoid":
            exp = {(0, 0, 1): 0.25, (0, 0, -1): 0.25, (1, 0, 0): 0.5}[tuple(n)]
        elif params["shape"] == "tetrahedron":
            exp = 0.5 / math.sqrt(3.0)                 # an edge midpoint direction: two vertices tie
        else:
            exp = {(0, 0, 1): 0.1, (0, 0, -1): 0.1, (1, 0, 0): 0.5}[tuple(n)]
        assert abs(float(out @ nv) - exp) < 1e-6


# ----------------------------------------------------------------------------------- pair overlap
def quat_from_axis(z):
    """Any quaternion whose body z axis is the given unit vector."""
    z = np.asarray(z, np.float64) / np.linalg.norm(z)
    r, _ = Rotation.align_vectors([z], [[0, 0, 1]])
    x, y, zz, w = r.as_quat()
    return np.array([w, x, y, zz], np.float32)


def test_pair_overlap_closed_forms_spherodisk():
    """S18: coaxial spherodisks overlap iff |dz| < 2s; coplanar iff centre distance < 2(a+s)."""
    q = quat_from_axis([0, 0, 1])
    for dz in np.linspace(0.05, 0.4, 36):
        if abs(dz - 0.2) < 1e-3:
            continue
        assert pair_overlap(SD, [0, 0, dz], q, q)[0] == (dz < 0.2)
        assert pair_overlap(SD, [0.3, 0, dz], q, q)[0] == (dz < 0.2)       # still face to face
    for dx in np.linspace(0.8, 1.2, 41):
        if abs(dx - 1.0) < 1e-3:
            continue
        assert pair_overlap(SD, [dx, 0, 0], q, q)[0] == (dx < 1.0)
    # T configuration: B's axis along x, B's rim towards A's face: contact at dz = s + (a + s)
    qx = quat_from_axis([1, 0, 0])
    for dz in np.linspace(0.4, 0.8, 41):
        if abs(dz - 0.6) < 1e-3:
            continue
        assert pair_overlap(SD, [0, 0, dz], q, qx)[0] == (dz < 0.6)
    # tilted orientation-independent sanity: far apart never, coincident always
    rng = np.random.default_rng(3)
    qa, qb = rand_quats(200, rng), rand_quats(200, rng)
    assert pair_overlap(SD, np.tile([0.0, 0.0, 0.0], (200, 1)), qa, qb).all()
    assert not pair_overlap(SD, np.tile([1.0001, 0.0, 0.0], (200, 1)), qa, qb).any()
    # closer than the thickness 2s the two always overlap, whatever the orientations
    dirs = rng.standard_normal((200, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    assert pair_overlap(SD, 0.19 * dirs, qa, qb).all()


def test_pair_overlap_closed_forms_halfball():
    """S18/S15: solid {|x|<=R, x.a<=0}: dome towards -a, flat face through the centre with normal +a."""
    up, dn = quat_from_axis([0, 0, 1]), quat_from_axis([0, 0, -1])
    # domes facing each other along z: A's dome towards +z (a=-z), B above with dome towards -z (a=+z)
    for d in np.linspace(0.8, 1.2, 41):
        if abs(d - 1.0) < 1e-3:
            continue
        assert pair_overlap(HB, [0, 0, d], dn, up)[0] == (d < 1.0)
    # flat faces facing each other with a gap h > 0: never
    for h in (1e-3, 0.01, 0.1, 0.5):
        assert not pair_overlap(HB, [0, 0, h], up, dn)[0]
        assert not pair_overlap(HB, [0.3, 0.1, h], up, dn)[0]
    # ... and interpenetrating when the gap is negative
    for h in (-1e-3, -0.01, -0.1):
        assert pair_overlap(HB, [0, 0, h], up, dn)[0]
    # A's flat face (normal +z) against B's dome pointing down (a_B=+z): contact when d = R
    for d in np.linspace(0.3, 0.7, 41):
        if abs(d - 0.5) < 1e-3:
            continue
        assert pair_overlap(HB, [0, 0, d], up, up)[0] == (d < 0.5)
    # side by side, same axis: the great half-discs touch at d = 2R
    for d in np.linspace(0.8, 1.2, 41):
        if abs(d - 1.0) < 1e-3:
            continue
        assert pair_overlap(HB, [d, 0, 0], up, up)[0] == (d < 1.0)
    # back to back (flat faces outward): A dome +z? no: A a=+z has its dome towards -z; B below with a=-z
    # has its dome towards +z -> domes facing, contact at 2R; while B ABOVE A (d>0) with a_B=-z: faces facing
    for d in np.linspace(0.8, 1.2, 9):
        if abs(d - 1.0) < 1e-3:
            continue
        assert pair_overlap(HB, [0, 0, -d], up, dn)[0] == (d < 1.0)


def _gauge(params):
    """fp64 convex gauge g(x) <= 0 inside the solid (body frame at origin, axis = body z)."""
    if params["shape"] == "halfball":
        R = 0.5 * params["sigma_c"]
        return lambda b: max(np.linalg.norm(b) - R, b[2])
    if params["shape"] == "tetrahedron":
        s = 0.5 / math.sqrt(3.0)
        U = TET_V / s
        return lambda b: max(-(U @ b) - s) / math.sqrt(3.0)        # signed distance to the nearest face plane
    if params["shape"] == "ellipsoid":
        A, Cc = params["disk_a"], params["disk_s"]
        # convex, <= 0 inside, and at least as large as the signed distance scaled by 1/A near the surface
        return lambda b: Cc * (math.sqrt((b[0] * b[0] + b[1] * b[1]) / (A * A) + b[2] * b[2] / (Cc * Cc)) - 1.0)
    a, s = params["disk_a"], params["disk_s"]

    def g(b):
        rho = math.hypot(b[0], b[1])
        return math.hypot(max(rho - a, 0.0), b[2]) - s
    return g


def _deepest_common_point(params, rho, qA, qB):
    """min_x max(g_A(x), g_B(x)) by an epigraph convex program (SLSQP, several starts)."""
    g = _gauge(params)
    MA, MB = q_to_R(qA).as_matrix().T, q_to_R(qB).as_matrix().T     # space -> body
    rho = np.asarray(rho, np.float64)
    gA = lambda x: g(MA @ x)
    gB = lambda x: g(MB @ (x - rho))
    best = np.inf
    for x0 in (0.5 * rho, 0.3 * rho + 0.03):
        t0 = max(gA(x0), gB(x0))
        res = minimize(lambda z: z[3], np.r_[x0, t0], method="SLSQP",
                       constraints=[{"type": "ineq", "fun": lambda z: z[3] - gA(z[:3])},
                                    {"type": "ineq", "fun": lambda z: z[3] - gB(z[:3])}],
                       options={"ftol": 1e-12, "maxiter": 300})
        x = res.x[:3]
        best = min(best, max(gA(x), gB(x)))
    return best


@pytest.mark.parametrize("params", [HB, SD, EL, TE])
def test_pair_overlap_vs_convex_program(params):
    """Random poses inside the circumsphere range: MPR's verdict == sign of the fp64 convex program,
    outside a contact band."""
    rng = np.random.default_rng(21)
    n = 24
    dirs = rng.standard_normal((n, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    lo = 0.15 if params["shape"] == "spherodisk" else 0.05
    rho = (dirs * (lo + (1.0 - lo) * rng.random((n, 1)))).astype(np.float32)
    qA, qB = rand_quats(n, rng), rand_quats(n, rng)
    got = pair_overlap(params, rho, qA, qB)
    n_in = n_out = 0
    for k in range(n):
        f = _deepest_common_point(params, rho[k], qA[k], qB[k])
        if f < -2e-4:
            assert got[k], (k, f)
            n_in += 1
        elif f > 2e-4:
            assert not got[k], (k, f)
            n_out += 1
    assert n_in > 3 and n_out > 3


# ---- a second, vectorised fp64 reference: alternating projections between the two solids, with certificates
def _body_frames(q):
    """Rotation matrices (n,3,3), columns = body axes in the space frame, from (w,x,y,z) quaternions (fp64)."""
    q = np.asarray(q, np.float64)
    q = q / np.linalg.norm(q, axis=1, keepdims=True)
    return Rotation.from_quat(np.c_[q[:, 1:], q[:, 0]]).as_matrix()


def _closest_on_triangle(p, a, b, c):
    """Closest points (fp64, vectorised over p) of the triangle (a, b, c): projection onto the plane if it falls inside,
    else the best of the three clamped edge projections."""
    n = np.cross(b - a, c - a)
    n /= np.linalg.norm(n)
    q = p - ((p - a) @ n)[:, None] * n
    def inside(q):
        s0 = np.cross(b - a, q - a) @ n
        s1 = np.cross(c - b, q - b) @ n
        s2 = np.cross(a - c, q - c) @ n
        return (s0 >= 0) & (s1 >= 0) & (s2 >= 0)
    ins = inside(q)
    best, bd = q.copy(), np.where(ins, np.linalg.norm(q - p, axis=1), np.inf)
    for x, y in ((a, b), (b, c), (c, a)):
        t = np.clip(((p - x) @ (y - x)) / ((y - x) @ (y - x)), 0.0, 1.0)
        e = x + t[:, None] * (y - x)
        d = np.linalg.norm(e - p, axis=1)
        upd = d < bd
        best[upd] = e[upd]
        bd = np.where(upd, d, bd)
    return best


def _project_body(params, b, shrink):
    """Closest point (body frame, fp64) of the solid eroded by `shrink`, and the gauge (<= 0 inside) of b w.r.t. it.
    Half-ball eroded by e = ball(R-e) below the plane z = -e; spherodisk eroded by e = disk(a) (+) ball(s-e)."""
    if params["shape"] == "halfball":
        R = 0.5 * params["sigma_c"] - shrink
        z0 = -shrink
        nb = np.linalg.norm(b, axis=1)
        gauge = np.maximum(nb - R, b[:, 2] - z0)
        rc = math.sqrt(max(R * R - z0 * z0, 0.0))               # radius of the flat face of the eroded solid
        below = b[:, 2] <= z0
        # below the plane: radial projection onto the ball keeps z <= z0 unless it lands above the face level
        pb = b * np.minimum(1.0, R / np.maximum(nb, 1e-300))[:, None]
        ok_b = below & (pb[:, 2] <= z0)
        # otherwise the closest point lies on the face disc (z = z0, radius rc)
        r_xy = np.hypot(b[:, 0], b[:, 1])
        sc = np.minimum(1.0, rc / np.maximum(r_xy, 1e-300))
        pf = np.stack([b[:, 0] * sc, b[:, 1] * sc, np.full(len(b), z0)], -1)
        return np.where(ok_b[:, None], pb, pf), gauge
    if params["shape"] == "tetrahedron":
        # the tetrahedron eroded by e is the concentric one with inradius r_in - e; closest point = the point itself if
        # inside, else the nearest of the closest points on the four faces
        r_in = 0.5 * params["sigma_c"] / 3.0
        V = TET_V * ((r_in - shrink) / r_in)
        U = TET_V / np.linalg.norm(TET_V[0])                   # unit vertex directions; face i has outward normal -U[i]
        gauge = np.max(-(b @ U.T) - (r_in - shrink), axis=1)
        best = b.copy()
        bd = np.where(gauge <= 0, 0.0, np.inf)
        for i in range(4):
            tri = V[[j for j in range(4) if j != i]]
            q = _closest_on_triangle(b, tri[0], tri[1], tri[2])
            d = np.linalg.norm(q - b, axis=1)
            upd = d < bd
            best[upd] = q[upd]
            bd = np.where(upd, d, bd)
        return best, gauge
    a, s = params["disk_a"], params["disk_s"] - shrink
    r_xy = np.hypot(b[:, 0], b[:, 1])
    sc = np.minimum(1.0, a / np.maximum(r_xy, 1e-300))
    core = np.stack([b[:, 0] * sc, b[:, 1] * sc, np.zeros(len(b))], -1)
    v = b - core
    d = np.linalg.norm(v, axis=1)
    out = core + v * np.minimum(1.0, s / np.maximum(d, 1e-300))[:, None]
    return out, d - s


def _support_body(params, n):
    """Support function h(n) = max_{x in solid} n.x in the body frame (fp64)."""
    if params["shape"] == "halfball":
        R = 0.5 * params["sigma_c"]
        return np.where(n[:, 2] <= 0, R * np.linalg.norm(n, axis=1), R * np.hypot(n[:, 0], n[:, 1]))
    if params["shape"] == "tetrahedron":
        return np.max(n @ TET_V.T, axis=1)
    return params["disk_a"] * np.hypot(n[:, 0], n[:, 1]) + params["disk_s"] * np.linalg.norm(n, axis=1)


def _classify_pairs(params, rho, qA, qB, band, iters=4000):
    """+1 = certified overlapping by more than `band` (a common point of both solids eroded by `band`),
    -1 = certified separated by more than `band` (a separating plane with that much room), 0 = undecided."""
    rho = np.asarray(rho, np.float64)
    MA, MB = _body_frames(qA), _body_frames(qB)
    to_body = lambda M, x: np.einsum("nij,ni->nj", M, x)       # M^T x
    to_space = lambda M, b: np.einsum("nij,nj->ni", M, b)
    n = len(rho)
    res = np.zeros(n, int)
    # (1) overlap certificate on the eroded solids
    x = 0.5 * rho
    for _ in range(iters):
        pa, _ = _project_body(params, to_body(MA, x), band)
        x = to_space(MA, pa)
        pb, _ = _project_body(params, to_body(MB, x - rho), band)
        x = to_space(MB, pb) + rho
    _, ga = _project_body(params, to_body(MA, x), band)
    _, gb = _project_body(params, to_body(MB, x - rho), band)
    res[(ga <= 1e-12) & (gb <= 1e-12)] = 1
    # (2) separation certificate on the full solids: plane normal from the closest pair found
    x = 0.5 * rho
    for _ in range(iters):
        pa, _ = _project_body(params, to_body(MA, x), 0.0)
        xa = to_space(MA, pa)
        pb, _ = _project_body(params, to_body(MB, xa - rho), 0.0)
        x = to_space(MB, pb) + rho
    d = x - xa
    dn = np.linalg.norm(d, axis=1)
    nrm = d / np.maximum(dn, 1e-300)[:, None]
    gap = np.einsum("ni,ni->n", nrm, rho) - _support_body(params, to_body(MA, nrm)) - _support_body(params, to_body(MB, -nrm))
    sep = (dn > 0) & (gap > band)
    assert not (sep & (res == 1)).any()
    res[sep] = -1
    return res


def _structured_poses(params, n, rng):
    """Hard poses for an iterative test: nearly parallel flat faces a small gap apart, rims against rims / faces,
    coplanar side-by-side contacts, each with a small random tilt and offset."""
    rho, qA, qB = [], [], []
    R = 0.5 * params["sigma_c"]

    def tilt(axis_z, eps):
        v = np.array(axis_z, np.float64) + eps * rng.standard_normal(3)
        return quat_from_axis(v / np.linalg.norm(v))
    for k in range(n):
        kind = k % 4
        eps = 10 ** rng.uniform(-4, -1.3)
        gap = rng.choice([-1, 1]) * 10 ** rng.uniform(-3.3, -1.3)
        if params["shape"] == "halfball":
            if kind == 0:      # flat faces facing each other, nearly parallel, lateral offset
                off = rng.uniform(-0.4, 0.4, 2)
                rho.append([off[0], off[1], gap]); qA.append(tilt([0, 0, 1], eps)); qB.append(tilt([0, 0, -1], eps))
            elif kind == 1:    # rim of B on the flat face of A (B on edge)
                rho.append([rng.uniform(-0.2, 0.2), 0.0, R + gap]); qA.append(tilt([0, 0, 1], eps)); qB.append(tilt([1, 0, 0], eps))
            elif kind == 2:    # side by side, same axis: great half-discs near contact at 2R
                rho.append([2 * R + gap, 0.0, rng.uniform(-0.05, 0.05)]); qA.append(tilt([0, 0, 1], eps)); qB.append(tilt([0, 0, 1], eps))
            else:              # dome against dome
                rho.append([0.0, 0.0, -(2 * R + gap)]); qA.append(tilt([0, 0, 1], eps)); qB.append(tilt([0, 0, -1], eps))
        else:
            a, s = params["disk_a"], params["disk_s"]
            if kind == 0:      # coaxial, faces nearly parallel at 2 s
                off = rng.uniform(-0.3, 0.3, 2)
                rho.append([off[0], off[1], 2 * s + gap]); qA.append(tilt([0, 0, 1], eps)); qB.append(tilt([0, 0, 1], eps))
            elif kind == 1:    # coplanar rim against rim at 2 (a + s)
                rho.append([2 * (a + s) + gap, 0.0, rng.uniform(-0.02, 0.02)]); qA.append(tilt([0, 0, 1], eps)); qB.append(tilt([0, 0, 1], eps))
            elif kind == 2:    # rim of B (on edge) against the face of A
                rho.append([rng.uniform(-0.2, 0.2), 0.0, a + 2 * s + gap]); qA.append(tilt([0, 0, 1], eps)); qB.append(tilt([1, 0, 0], eps))
            else:              # crossed rims (T configuration in the plane)
                rho.append([a + s + s + gap, 0.0, 0.0]); qA.append(tilt([0, 0, 1], eps)); qB.append(tilt([0, 1, 0], eps))
    return np.array(rho, np.float32), np.array(qA, np.float32), np.array(qB, np.float32)


def test_pair_overlap_vs_certified_reference_tetrahedra():
    """R-N2b: 1,200 random poses of two tetrahedra inside the circumsphere range; wherever the fp64 reference certifies an
    overlap deeper than 2e-4 (common point of the eroded solids) or a separation wider than 2e-4 (separating plane), MPR
    with the vertex support must agree.  Face, edge and vertex contacts are covered by the closed forms above."""
    rng = np.random.default_rng(29)
    n = 1200
    dirs = rng.standard_normal((n, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    rho = (dirs * (0.1 + 0.9 * rng.random((n, 1)))).astype(np.float32)
    qA, qB = rand_quats(n, rng), rand_quats(n, rng)
    got = pair_overlap(TE, rho, qA, qB)
    cls = _classify_pairs(TE, rho, qA, qB, 2e-4, iters=2000)
    assert (cls != 0).mean() > 0.85, (cls != 0).mean()
    bad = np.nonzero(((cls == 1) & ~got) | ((cls == -1) & got))[0]
    assert len(bad) == 0, (len(bad), bad[:5], rho[bad[:5]], cls[bad[:5]])
    assert (cls == 1).sum() > 100 and (cls == -1).sum() > 100


@pytest.mark.parametrize("params", [HB, SD])
def test_pair_overlap_vs_certified_reference_many_poses(params):
    """>= 2,000 poses per shape (1,600 random inside the circumsphere range + 800 structured near-contact ones:
    nearly parallel faces, rim-rim, rim-face, dome-dome): wherever the fp64 reference certifies an overlap deeper
    than 2e-4 or a separation wider than 2e-4, MPR (two 48-iteration caps, 1e-5 tolerance) must agree."""
    rng = np.random.default_rng(23)
    n = 1600
    dirs = rng.standard_normal((n, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    lo = 0.15 if params["shape"] == "spherodisk" else 0.05
    rho = (dirs * (lo + (1.0 - lo) * rng.random((n, 1)))).astype(np.float32)
    qA, qB = rand_quats(n, rng), rand_quats(n, rng)
    srho, sqA, sqB = _structured_poses(params, 800, rng)
    rho, qA, qB = np.r_[rho, srho], np.r_[qA, sqA], np.r_[qB, sqB]
    got = pair_overlap(params, rho, qA, qB)
    cls = _classify_pairs(params, rho, qA, qB, 2e-4)
    assert (cls != 0).mean() > 0.9, (cls != 0).mean()            # the reference decides nearly every pose
    assert (cls[n:] != 0).mean() > 0.75
    bad = np.nonzero(((cls == 1) & ~got) | ((cls == -1) & got))[0]
    assert len(bad) == 0, (len(bad), bad[:5], rho[bad[:5]], cls[bad[:5]])
    for part in (slice(0, n), slice(n, None)):
        assert (cls[part] == 1).sum() > 100 and (cls[part] == -1).sum() > 100


def test_pair_overlap_symmetric_outside_band():
    """Swapping the roles of A and B (rho -> -rho) gives the same verdict for generic poses."""
    rng = np.random.default_rng(22)
    n = 20000
    dirs = rng.standard_normal((n, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    rho = (dirs * (0.2 + 0.8 * rng.random((n, 1)))).astype(np.float32)
    qA, qB = rand_quats(n, rng), rand_quats(n, rng)
    for params in (HB, SD):
        ab = pair_overlap(params, rho, qA, qB)
        ba = pair_overlap(params, -rho, qB, qA)
        assert (ab != ba).mean() < 2e-3            # only poses inside the 1e-5 contact band may differ
        assert 0.15 < ab.mean() < 0.9


def test_sphere_pair_overlap_exact():
    q = np.array([1, 0, 0, 0], np.float32)
    assert pair_overlap(SP, [0.999999, 0, 0], q, q)[0]
    assert not pair_overlap(SP, [1.0, 0, 0], q, q)[0]              # S14: touching is not overlapping
    assert not pair_overlap(SP, [0.6, 0.6, 0.6], q, q)[0]
    assert pair_overlap(SP, [0.57, 0.57, 0.57], q, q)[0]


# ----------------------------------------------------------------------------------- rotations
def test_quat_axis_and_cayley_vs_scipy(olib):
    rng = np.random.default_rng(31)
    for _ in range(200):
        q = rand_quats(1, rng)[0]
        ax = np.zeros(3, np.float32)
        olib.oracle_quat_axis(q.ctypes.data, ax.ctypes.data)
        assert np.allclose(ax, q_to_R(q).apply([0, 0, 1]), atol=2e-6)
        v = (rng.standard_normal(3) * 0.1).astype(np.float32)
        out = np.zeros(4, np.float32)
        olib.oracle_rotate_cayley(q.ctypes.data, v.ctypes.data, out.ctypes.data)
        assert abs(np.linalg.norm(out.astype(np.float64)) - 1.0) < 3e-7
        # (1,v)/sqrt(1+v^2) is the rotation by 2 atan|v| about v, applied on the left (space frame)
        ang = 2.0 * math.atan(np.linalg.norm(v.astype(np.float64)))
        dR = Rotation.from_rotvec(v.astype(np.float64) / np.linalg.norm(v) * ang)
        want = (dR * q_to_R(q)).as_matrix()
        got = q_to_R(out).as_matrix()
        assert np.allclose(got, want, atol=5e-6)
