"""Seeded synthetic inputs for the five BASELINE.json configurations (C1..C5).

This module serves BOTH the CUDA library and the CPU oracle and therefore contains none of the
method's arithmetic: no Philox, no cell list, no overlap predicate of the move, no sampler.  It
only places non-overlapping particles (fp64 distance checks with a safety margin, so that the
configuration is also overlap-free under any fp32 predicate) and draws orientations with numpy's
PCG64.  Recipes are stated in DESIGN.md ("Input recipe").

    cfg = workloads.config("C3")             # parameters (box, n_R, d_max ...)
    pos4, quat4 = workloads.generate(cfg)    # float32 (N,4) arrays; quat4 is None for spheres
    cfg_small = workloads.config("C3", N=4096)   # same densities, fewer particles (tests)
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SPHERE_VOL = math.pi / 6.0
HALFBALL_VOL = 2.0 * math.pi * 0.5 ** 3 / 3.0


def spherodisk_volume(a: float, s: float) -> float:
    """Volume of disk(radius a) (+) ball(radius s): Steiner formula 2 pi a^2 s + pi^2 a s^2 + 4 pi s^3/3."""
    return 2.0 * math.pi * a * a * s + math.pi ** 2 * a * s * s + 4.0 * math.pi * s ** 3 / 3.0


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    N: int
    shape: str            # "sphere" | "halfball" | "spherodisk" | "ellipsoid" | "tetrahedron"
    phi_c: float          # colloid packing fraction
    q: float              # sigma_d / sigma_c
    phi_d_r: tuple        # reservoir packing fraction(s) of the depletants
    d_max: float
    a_max: float
    n_trial: int
    sweeps: int
    init: str             # "rsa" | "fcc" | "sc" | "sca"
    sigma_c: float = 1.0  # circumsphere diameter
    disk_a: float = 0.0
    disk_s: float = 0.0
    seed: int = 1

    @property
    def particle_volume(self) -> float:
        if self.shape == "sphere":
            return SPHERE_VOL * self.sigma_c ** 3
        if self.shape == "halfball":
            return HALFBALL_VOL * self.sigma_c ** 3
        if self.shape == "tetrahedron":        # regular, circumradius sigma_c / 2: edge a = R sqrt(8/3), V = a^3 / (6 sqrt 2)
            return (0.5 * self.sigma_c * math.sqrt(8.0 / 3.0)) ** 3 / (6.0 * math.sqrt(2.0))
        if self.shape == "ellipsoid":          # oblate spheroid, semi-axes (disk_a, disk_a, disk_s)
            return 4.0 * math.pi * self.disk_a ** 2 * self.disk_s / 3.0
        return spherodisk_volume(self.disk_a, self.disk_s)

    @property
    def sigma_d(self) -> float:
        return self.q * self.sigma_c

    @property
    def box_L(self) -> float:
        return float(np.float32((self.N * self.particle_volume / self.phi_c) ** (1.0 / 3.0)))

    def n_R(self, phi_d_r=None) -> float:
        """Reservoir number density n_R = phi_d^r / (pi sigma_d^3 / 6)."""
        p = self.phi_d_r[0] if phi_d_r is None else phi_d_r
        return p / (math.pi * self.sigma_d ** 3 / 6.0)

    @property
    def lam(self) -> float:
        """Mean number of depletants drawn per move, n_R * 4 pi R^3 / 3 with R = (sigma_c+sigma_d)/2."""
        R = 0.5 * (self.sigma_c + self.sigma_d)
        return self.n_R() * 4.0 * math.pi * R ** 3 / 3.0


_CONFIGS = {
    "C1": Config("C1", 256, "sphere", 0.10, 0.20, (0.20,), 0.1, 0.0, 0, 100, "rsa"),
    "C2": Config("C2", 65536, "sphere", 0.30, 0.10, (0.1, 0.2, 0.3, 0.4), 0.05, 0.0, 0, 1000, "fcc"),
    "C3": Config("C3", 1048576, "sphere", 0.25, 0.05, (0.30,), 0.05, 0.0, 0, 200, "rsa"),
    "C4": Config("C4", 32768, "halfball", 0.20, 0.20, (0.25,), 0.1, 0.1, 0, 500, "sc"),
    "C5": Config("C5", 32768, "spherodisk", 0.15, 0.15, (0.35,), 0.1, 0.1, 4, 500, "sc", disk_a=0.4, disk_s=0.1),
    # SURVEY 8(f) NEXT-2, not a BASELINE.json config: the paper's own discoids (oblate ellipsoids
    # a = b = 0.5, c = 0.25, depletant radius 0.25, phi_p^r = 0.40, n_trial >~ 10), here 32^3 of them at phi_c = 0.10
    # (the paper's 500 at phi_c = 0.01 would leave every neighbourhood empty) with C4's step sizes
    "C6": Config("C6", 32768, "ellipsoid", 0.10, 0.50, (0.40,), 0.1, 0.1, 10, 200, "sc", disk_a=0.5, disk_s=0.25),
    # NEXT-2, second new shape: regular tetrahedra (Fig. 1 L21), circumradius 0.5, all with the same orientation
    # on a 32^3 lattice of spacing 0.685 (equally oriented tetrahedra are disjoint iff the lattice vector lies outside
    # their difference body, a cuboctahedron reaching 0.577 along the axes), C4's depletants and step sizes
    "C7": Config("C7", 32768, "tetrahedron", 0.20, 0.20, (0.25,), 0.1, 0.1, 0, 200, "sca"),
}


def config(name: str, N: int | None = None, **over) -> Config:
    cfg = _CONFIGS[name]
    if N is not None:
        over["N"] = int(N)
    return dataclasses.replace(cfg, **over) if over else cfg


# ------------------------------------------------------------------------------------------ placement
def _to_box_f32(x: np.ndarray, L: float) -> np.ndarray:
    """Round to float32 and keep inside [0, L)."""
    x32 = x.astype(np.float32)
    x32[x32 >= np.float32(L)] = 0.0
    x32[x32 < 0] = 0.0
    return x32


_RSA_LIB = None


def build() -> str:
    """Compile the placement helper rsa.c in-tree (gcc); returns the path of the shared object."""
    import os
    import subprocess
    here = os.path.dirname(os.path.abspath(__file__))
    src, so = os.path.join(here, "rsa.c"), os.path.join(here, "librsa.so")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        tmp = so + ".tmp%d" % os.getpid()
        subprocess.run(["gcc", "-O2", "-shared", "-fPIC", "-o", tmp, src, "-lm"], check=True)
        os.replace(tmp, so)
    return so


def _rsa_spheres(N: int, L: float, sigma: float, seed: int) -> np.ndarray:
    """Seeded random sequential placement (rsa.c): N centres with pair distance > sigma (1 + 5e-5)."""
    global _RSA_LIB
    import ctypes as C
    if _RSA_LIB is None:
        _RSA_LIB = C.CDLL(build())
        _RSA_LIB.rsa_place.restype = C.c_int64
        _RSA_LIB.rsa_place.argtypes = [C.c_int64, C.c_double, C.c_double, C.c_uint64, C.c_void_p, C.c_int64]
    pos4 = np.zeros((N, 4), np.float32)
    placed = _RSA_LIB.rsa_place(N, L, sigma, seed, pos4.ctypes.data_as(C.c_void_p), 400 * N + 100000)
    if placed != N:
        raise RuntimeError("random sequential placement stalled at %d of %d" % (placed, N))
    return pos4[:, :3].astype(np.float64)


def _fcc_sites(ncell: int, L: float) -> np.ndarray:
    a = L / ncell
    base = np.array([(0, 0, 0), (0.5, 0.5, 0), (0.5, 0, 0.5), (0, 0.5, 0.5)], np.float64)
    ii = np.arange(ncell)
    grid = np.stack(np.meshgrid(ii, ii, ii, indexing="ij"), -1).reshape(-1, 1, 3)
    return ((grid + base[None]) * a + 0.25 * a).reshape(-1, 3)


def _sc_sites(n: int, L: float) -> np.ndarray:
    a = L / n
    ii = np.arange(n)
    grid = np.stack(np.meshgrid(ii, ii, ii, indexing="ij"), -1).reshape(-1, 3)
    return (grid + 0.5) * a


def _random_quats(n: int, rng: np.random.Generator) -> np.ndarray:
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    q32 = q.astype(np.float32).astype(np.float64)
    q32 /= np.linalg.norm(q32, axis=1, keepdims=True)
    return q32          # (w,x,y,z)


def _body_z(q: np.ndarray) -> np.ndarray:
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    return np.stack([2 * (x * z + w * y), 2 * (y * z - w * x), 1 - 2 * (x * x + y * y)], -1)


def generate(cfg: Config):
    """Return (pos4, quat4) float32 arrays; quat4 is None for spheres."""
    rng = np.random.default_rng([cfg.seed, cfg.N, sum(map(ord, cfg.name))])
    L = cfg.box_L
    N = cfg.N
    quat = None
    if cfg.init == "rsa":
        pos = _rsa_spheres(N, L, cfg.sigma_c, 0x9E3779B9 * cfg.seed + N)
    elif cfg.init == "fcc":
        ncell = int(math.ceil((N / 4.0) ** (1.0 / 3.0) - 1e-9))
        sites = _fcc_sites(ncell, L)
        if (L / ncell) / math.sqrt(2.0) <= cfg.sigma_c * 1.0001:
            raise ValueError("fcc lattice too dense for this box")
        keep = np.sort(rng.permutation(len(sites))[:N])
        pos = sites[keep]
    elif cfg.init == "sca":
        n = int(round(N ** (1.0 / 3.0)))
        if n ** 3 != N:
            raise ValueError("simple-cubic initial state needs N = n^3")
        pos = _sc_sites(n, L)
        if cfg.shape != "tetrahedron" or L / n < 0.6 * cfg.sigma_c:
            raise ValueError("aligned lattice: tetrahedra at spacing >= 0.6 circumsphere diameters only")
        quat = np.tile(np.array([1.0, 0.0, 0.0, 0.0]), (N, 1))
    elif cfg.init == "sc":
        n = int(round(N ** (1.0 / 3.0)))
        if n ** 3 != N:
            raise ValueError("simple-cubic initial state needs N = n^3")
        pos = _sc_sites(n, L)
        spacing = L / n
        quat = _random_quats(N, rng)
        if cfg.shape in ("halfball", "ellipsoid", "tetrahedron"):
            if spacing < cfg.sigma_c * 1.0001:
                raise ValueError("circumspheres of the lattice overlap")
        elif cfg.shape == "spherodisk":
            # Lattice neighbours along axis e are disjoint if the two widths along e sum to less than
            # the spacing (separating plane); width of disk(a)+ball(s) along e is a sqrt(1-(n.e)^2)+s.
            # Second neighbours sit at spacing*sqrt(2) > circumsphere diameter.
            if spacing * math.sqrt(2.0) < cfg.sigma_c * 1.0001:
                raise ValueError("second lattice neighbours' circumspheres overlap")
            idx = np.arange(N).reshape(n, n, n)
            for _ in range(200):
                nz = _body_z(quat)
                bad = np.zeros(N, bool)
                for ax in range(3):
                    hw = cfg.disk_a * np.sqrt(np.maximum(0.0, 1.0 - nz[:, ax] ** 2)) + cfg.disk_s
                    nb = np.roll(idx, -1, axis=ax).reshape(-1)
                    clash = hw + hw[nb] >= spacing * (1.0 - 1e-4)
                    bad |= clash
                if not bad.any():
                    break
                quat[bad] = _random_quats(int(bad.sum()), rng)
            else:
                raise RuntimeError("could not orient the spherodisk lattice without overlaps")
    else:
        raise ValueError(cfg.init)
    pos4 = np.zeros((N, 4), np.float32)
    pos4[:, :3] = _to_box_f32(pos, L)
    quat4 = None if quat is None else np.ascontiguousarray(quat, np.float32)
    return pos4, quat4
