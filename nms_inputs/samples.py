"""Synthetic real-space samples and detector grids.

Only input construction lives here: lattices, magnetisation textures, particle
placement, detector abscissae and rotation matrices.  Everything is generated
in float64 with NumPy (seeded `np.random.Generator(np.random.Philox(seed))`
where random) and cast once to float32, which is what both the oracle and the
CUDA library receive.

Lattice conventions (Table I): "inside radius"
is inclusive (r^2 <= R^2); a node-centred lattice has integer coordinates
(4169 cells for R/a = 10), a cell-centred lattice half-integer ones (4224).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

KINDS = ["NUC", "MAG", "UNPOL", "PROJ", "NM", "SF", "CHI",
         "PM", "MP", "PP", "MM", "POL_PLUS", "POL_MINUS"]
KIND_INDEX = {k: i for i, k in enumerate(KINDS)}
ALL_KINDS = list(range(len(KINDS)))

GRID_POLAR, GRID_CARTESIAN, GRID_LIST = 0, 1, 2


# ----------------------------------------------------------------------------
# rotations (Eq. 37; convention fixed in SURVEY 8(c)-3)
# ----------------------------------------------------------------------------
def rot_y(a_deg: float) -> np.ndarray:
    a = np.deg2rad(a_deg)
    c, s = np.cos(a), np.sin(a)
    return np.array([[c, 0.0, s], [0.0, 1.0, 0.0], [-s, 0.0, c]], dtype=np.float64)


def rot_z(b_deg: float) -> np.ndarray:
    b = np.deg2rad(b_deg)
    c, s = np.cos(b), np.sin(b)
    return np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]], dtype=np.float64)


def rotation_alpha_beta(alpha_deg: float, beta_deg: float) -> np.ndarray:
    """R(alpha, beta) = R_z(beta) R_y(alpha), right-handed active matrices."""
    return rot_z(beta_deg) @ rot_y(alpha_deg)


# ----------------------------------------------------------------------------
# detector grids.  flat index = i0 * n1 + i1 (i1 fastest)
# ----------------------------------------------------------------------------
@dataclass
class Grid:
    type: int            # 0 polar (u0 = |q| [n0], u1 = theta [n1]); 1 cartesian (u0 = q_z [n0], u1 = q_y [n1]); 2 list (u0 = q_y [n], u1 = q_z [n], n1 = 1)
    n0: int
    n1: int
    u0: np.ndarray       # float32
    u1: np.ndarray       # float32

    @property
    def n_q(self) -> int:
        return self.n0 * self.n1

    def subset(self, idx: np.ndarray) -> "Grid":
        """Point-list grid holding the detector points with flat indices `idx`.

        The list carries (q_y, q_z) as float32, so it is only bit-identical to the
        parent for cartesian parents; polar parents are handled by the callers via
        `polar_points()` in float64 on the oracle side.
        """
        if self.type == GRID_CARTESIAN:
            i0, i1 = np.divmod(np.asarray(idx, dtype=np.int64), self.n1)
            return Grid(GRID_LIST, len(idx), 1, self.u1[i1].copy(), self.u0[i0].copy())
        if self.type == GRID_LIST:
            return Grid(GRID_LIST, len(idx), 1, self.u0[idx].copy(), self.u1[idx].copy())
        raise ValueError("subset() of a polar grid is not representable as an fp32 list")


def polar_grid(q: np.ndarray, n_theta: int) -> Grid:
    theta = (2.0 * np.pi * np.arange(n_theta, dtype=np.float64) / n_theta)
    return Grid(GRID_POLAR, len(q), n_theta, np.asarray(q, dtype=np.float32), theta.astype(np.float32))


def cartesian_grid(qz: np.ndarray, qy: np.ndarray) -> Grid:
    return Grid(GRID_CARTESIAN, len(qz), len(qy), np.asarray(qz, dtype=np.float32), np.asarray(qy, dtype=np.float32))


def list_grid(qy: np.ndarray, qz: np.ndarray) -> Grid:
    assert len(qy) == len(qz)
    return Grid(GRID_LIST, len(qy), 1, np.asarray(qy, dtype=np.float32), np.asarray(qz, dtype=np.float32))


def q_subset(n_q: int, count: int, seed: int) -> np.ndarray:
    """First, last and seeded random interior flat indices (sorted, unique)."""
    rng = np.random.Generator(np.random.Philox(seed))
    count = min(count, n_q)
    inner = rng.choice(np.arange(1, max(n_q - 1, 2)), size=max(count - 2, 0), replace=False) if n_q > 2 else np.array([], dtype=np.int64)
    idx = np.unique(np.concatenate([[0, n_q - 1], inner]).astype(np.int64))
    return idx


# ----------------------------------------------------------------------------
# workload container
# ----------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    pos: np.ndarray                   # float32 [W,3]
    N: Optional[np.ndarray]           # float32 [W] or None
    m: Optional[np.ndarray]           # float32 [W,3] or None
    grid: Grid
    kinds: List[int]
    R: np.ndarray = field(default_factory=lambda: np.eye(3))
    rotations: Optional[List[np.ndarray]] = None    # rocking scan (C4); R is rotations[0]
    offsets: Optional[np.ndarray] = None            # int64 [K+1]
    centres: Optional[np.ndarray] = None            # float32 [K,3]
    P: np.ndarray = field(default_factory=lambda: np.array([0.0, 0.0, 1.0]))
    n_bins: int = 0
    q_lo: float = 0.0
    q_hi: float = 0.0
    r: Optional[np.ndarray] = None                  # float32 [n_r]
    split: bool = False                             # form-factor / interference split requested

    @property
    def W(self) -> int:
        return int(self.pos.shape[0])

    @property
    def n_rot(self) -> int:
        return len(self.rotations) if self.rotations is not None else 1

    @property
    def pairs(self) -> int:
        return self.W * self.grid.n_q * self.n_rot


# ----------------------------------------------------------------------------
# lattices
# ----------------------------------------------------------------------------
def sphere_node_centred(radius: float, a: float) -> np.ndarray:
    """Integer-node lattice (i,j,k)*a with r^2 <= R^2; row order y outer, x middle, z inner (Table I)."""
    n = int(np.floor(radius / a + 1e-9))
    ax = np.arange(-n, n + 1, dtype=np.float64) * a
    y, x, z = np.meshgrid(ax, ax, ax, indexing="ij")          # y outer, x middle, z inner
    keep = (x * x + y * y + z * z) <= radius * radius * (1 + 1e-12)
    return np.stack([x[keep], y[keep], z[keep]], axis=1)


def sphere_cell_centred(radius: float, a: float) -> np.ndarray:
    """Half-integer lattice (i+1/2, j+1/2, k+1/2)*a with r^2 <= R^2 (same row order)."""
    n = int(np.ceil(radius / a))
    ax = (np.arange(-n, n, dtype=np.float64) + 0.5) * a
    y, x, z = np.meshgrid(ax, ax, ax, indexing="ij")
    keep = (x * x + y * y + z * z) <= radius * radius * (1 + 1e-12)
    return np.stack([x[keep], y[keep], z[keep]], axis=1)


def cuboid_lattice(nx: int, ny: int, nz: int, a: float) -> np.ndarray:
    """Uniform cuboid lattice centred on the origin, x fastest."""
    x = (np.arange(nx) - (nx - 1) / 2.0) * a
    y = (np.arange(ny) - (ny - 1) / 2.0) * a
    z = (np.arange(nz) - (nz - 1) / 2.0) * a
    zz, yy, xx = np.meshgrid(z, y, x, indexing="ij")
    return np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1)


def uniform_sphere_sample(radius: float = 20.0, a: float = 1.0, n=(0.0, 0.0, 1.0)):
    """PAPER.md Sec. IV A (Eq. 53-54): uniform N and uniform M = n inside a sphere."""
    pos = sphere_node_centred(radius, a)
    W = pos.shape[0]
    N = np.ones(W)
    m = np.tile(np.asarray(n, dtype=np.float64), (W, 1))
    return pos.astype(np.float32), N.astype(np.float32), m.astype(np.float32)


def linear_vortex_sphere_sample(radius: float = 20.0, a: float = 1.0, m1_over_m0: float = None):
    """PAPER.md Sec. IV B (Eq. 83): M = M0 e_z + M1 (x e_y - y e_x), in units of M0; M1 = 5 M0 / R by default."""
    pos = sphere_node_centred(radius, a)
    W = pos.shape[0]
    k = (5.0 / radius) if m1_over_m0 is None else m1_over_m0
    m = np.stack([-k * pos[:, 1], k * pos[:, 0], np.ones(W)], axis=1)
    return pos.astype(np.float32), np.ones(W, dtype=np.float32), m.astype(np.float32)


# ----------------------------------------------------------------------------
# C1 .. C5
# ----------------------------------------------------------------------------
def _kinds(names):
    return [KIND_INDEX[n] for n in names]


def config_c1() -> Workload:
    """Uniformly magnetised sphere, R = 10 nm, a = 1 nm, node-centred (W = 4169)."""
    pos = sphere_node_centred(10.0, 1.0)
    W = pos.shape[0]
    q = 0.01 + np.arange(64, dtype=np.float64) * (2.99 / 63.0)
    return Workload(
        name="C1", pos=pos.astype(np.float32), N=np.ones(W, dtype=np.float32),
        m=np.tile(np.array([0, 0, 1], dtype=np.float32), (W, 1)),
        grid=polar_grid(q, 64), kinds=_kinds(["NUC", "MAG", "UNPOL", "SF", "CHI"]),
        R=np.eye(3), n_bins=64)


def config_c2() -> Workload:
    """Vortex disc: radius 40 nm, height 20 nm, a = 2 nm cell-centred (W = 12640), rotated R_z(30) R_y(45)."""
    a = 2.0
    ax = (np.arange(-20, 20, dtype=np.float64) + 0.5) * a
    az = (np.arange(-5, 5, dtype=np.float64) + 0.5) * a
    z, y, x = np.meshgrid(az, ax, ax, indexing="ij")          # x fastest
    keep = (x * x + y * y) <= 40.0 ** 2
    x, y, z = x[keep], y[keep], z[keep]
    rho = np.sqrt(x * x + y * y)
    mz = np.exp(-(rho / 5.0) ** 2)
    s = np.sqrt(np.maximum(1.0 - mz * mz, 0.0))
    m = np.stack([-y * s / rho, x * s / rho, mz], axis=1)
    W = x.shape[0]
    qa = -1.5 + 3.0 * np.arange(128, dtype=np.float64) / 127.0
    r = 100.0 * np.arange(256, dtype=np.float64) / 255.0
    return Workload(
        name="C2", pos=np.stack([x, y, z], axis=1).astype(np.float32), N=np.ones(W, dtype=np.float32),
        m=m.astype(np.float32), grid=cartesian_grid(qa, qa), kinds=list(ALL_KINDS),
        R=rot_z(30.0) @ rot_y(45.0), n_bins=128, q_lo=0.0, q_hi=1.5, r=r.astype(np.float32))


def rsa_centres(K: int, half_box: float, min_dist: float, seed: int) -> np.ndarray:
    """Random sequential addition of K non-overlapping sphere centres in [-half_box, half_box]^3."""
    rng = np.random.Generator(np.random.Philox(seed))
    centres = np.empty((K, 3), dtype=np.float64)
    n = 0
    d2 = min_dist * min_dist
    while n < K:
        c = rng.uniform(-half_box, half_box, size=3)
        if n == 0 or np.min(np.sum((centres[:n] - c) ** 2, axis=1)) >= d2:
            centres[n] = c
            n += 1
    return centres


def config_c3(K: int = 1000, n_q: int = 256, n_theta: int = 256, separate_centres: bool = False) -> Workload:
    """Particle ensemble: K spheres of radius 5 nm on a 0.5 nm cell-centred lattice (4224 cells each)."""
    local = sphere_cell_centred(5.0, 0.5)
    Nk = local.shape[0]
    half = 245.0 if K > 8 else 40.0
    centres = rsa_centres(K, half, 10.0, 3001)
    rng = np.random.Generator(np.random.Philox(3002))
    d = rng.standard_normal((K, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    m = np.repeat(d, Nk, axis=0)
    if separate_centres:
        pos = np.tile(local, (K, 1))
        cen = centres.astype(np.float32)
    else:
        pos = (centres[:, None, :] + local[None, :, :]).reshape(-1, 3)
        cen = None
    W = K * Nk
    q = 0.005 * 400.0 ** (np.arange(n_q, dtype=np.float64) / max(n_q - 1, 1))
    return Workload(
        name="C3", pos=pos.astype(np.float32), N=np.ones(W, dtype=np.float32), m=m.astype(np.float32),
        grid=polar_grid(q, n_theta), kinds=_kinds(["NUC", "MAG", "UNPOL", "SF"]),
        offsets=(np.arange(K + 1, dtype=np.int64) * Nk), centres=cen, split=True)


def config_fig10(K: int, n_q: int = 256, n_theta: int = 256) -> Workload:
    """Context workload, not a BASELINE.json config: synthetic re-creation of the paper's runtime experiment
    (Sec. IV D, Eq. 109): K identical spheres D = 40 nm on a node-centred a = 2 nm lattice (4169 cells
    each), linear vortex m = (-5y/R, 5x/R, 1)/|.| in the particle's own frame, uniform N = 1; centres on a simple
    cubic lattice of 60 nm (the paper does not say where its copies sit); polar detector, |q| linear in 0.01-1.5."""
    local = sphere_node_centred(20.0, 2.0)
    x, y = local[:, 0] / 20.0, local[:, 1] / 20.0
    mv = np.stack([-5.0 * y, 5.0 * x, np.ones_like(x)], axis=1)
    mv /= np.linalg.norm(mv, axis=1, keepdims=True)
    n_side = int(np.ceil(K ** (1.0 / 3.0)))
    idx = np.arange(K)
    cen = np.stack([idx % n_side, (idx // n_side) % n_side, idx // (n_side * n_side)], axis=1).astype(np.float64)
    cen = (cen - 0.5 * (n_side - 1)) * 60.0
    pos = (cen[:, None, :] + local[None, :, :]).reshape(-1, 3).astype(np.float32)
    W = pos.shape[0]
    q = 0.01 + 1.49 * np.arange(n_q, dtype=np.float64) / max(n_q - 1, 1)
    return Workload(name="F10", pos=pos, N=np.ones(W, dtype=np.float32), m=np.tile(mv.astype(np.float32), (K, 1)),
                    grid=polar_grid(q, n_theta), kinds=list(ALL_KINDS), n_bins=n_q,
                    r=np.linspace(0.0, 60.0, 256).astype(np.float32))


def config_c4(nx: int = 512, ny: int = 512, nz: int = 8, n_rot: int = 36, n_grid: int = 256) -> Workload:
    """Neel-skyrmion-lattice film, hexagonal lattice period 50 nm; rocking scan about z in 10 degree steps."""
    x = np.arange(nx, dtype=np.float64) + 0.5 - nx / 2.0
    y = np.arange(ny, dtype=np.float64) + 0.5 - ny / 2.0
    z = np.arange(nz, dtype=np.float64) + 0.5 - nz / 2.0
    zz, yy, xx = np.meshgrid(z, y, x, indexing="ij")          # x fastest
    xx, yy, zz = xx.ravel(), yy.ravel(), zz.ravel()
    a1 = np.array([50.0, 0.0])
    a2 = np.array([25.0, 25.0 * np.sqrt(3.0)])
    A = np.stack([a1, a2], axis=1)                             # columns a1, a2
    frac = np.linalg.solve(A, np.stack([xx, yy], axis=0))      # fractional coordinates
    base = np.round(frac)
    best_d2 = np.full(xx.shape, np.inf)
    dx = np.zeros_like(xx)
    dy = np.zeros_like(yy)
    for di in (-1, 0, 1):
        for dj in (-1, 0, 1):
            site = A @ np.stack([base[0] + di, base[1] + dj], axis=0)
            ex, ey = xx - site[0], yy - site[1]
            d2 = ex * ex + ey * ey
            upd = d2 < best_d2
            best_d2 = np.where(upd, d2, best_d2)
            dx = np.where(upd, ex, dx)
            dy = np.where(upd, ey, dy)
    rho = np.sqrt(best_d2)
    phi = np.arctan2(dy, dx)
    Th = 2.0 * np.arctan(np.exp((8.0 - rho) / 3.0))
    m = np.stack([np.sin(Th) * np.cos(phi), np.sin(Th) * np.sin(phi), np.cos(Th)], axis=1)
    W = xx.shape[0]
    qa = -0.5 + 1.0 * np.arange(n_grid, dtype=np.float64) / (n_grid - 1)
    rots = [rot_z(10.0 * k) for k in range(n_rot)]
    return Workload(
        name="C4", pos=np.stack([xx, yy, zz], axis=1).astype(np.float32), N=np.ones(W, dtype=np.float32),
        m=m.astype(np.float32), grid=cartesian_grid(qa, qa), kinds=_kinds(["UNPOL", "SF"]),
        R=rots[0], rotations=rots)


def config_c5(n: int = 256, n_q: int = 512, n_theta: int = 512, n_r: int = 1024) -> Workload:
    """Micromagnetic block n^3 with a Gaussian-correlated unit vector field and 5 % spherical pores."""
    rng = np.random.Generator(np.random.Philox(5001))
    xi = 10.0
    sigma = xi / np.sqrt(2.0)
    k1 = 2.0 * np.pi * np.fft.fftfreq(n, d=1.0)
    kr = 2.0 * np.pi * np.fft.rfftfreq(n, d=1.0)
    filt = np.exp(-0.5 * sigma * sigma * (k1[:, None, None] ** 2 + k1[None, :, None] ** 2 + kr[None, None, :] ** 2))
    comps = []
    for _ in range(3):
        w = rng.standard_normal((n, n, n))
        f = np.fft.irfftn(np.fft.rfftn(w) * filt, s=(n, n, n), axes=(0, 1, 2))
        comps.append(f)
        del w
    norm = np.sqrt(comps[0] ** 2 + comps[1] ** 2 + comps[2] ** 2)
    m = np.stack([(c / norm).ravel() for c in comps], axis=1).astype(np.float32)   # arrays are [z][y][x]: x fastest
    del comps, norm, filt
    # pores: seeded uniform centres, radius 3, one at a time until >= 5 % of cells have N = 0
    rngp = np.random.Generator(np.random.Philox(5002))
    Nf = np.ones((n, n, n), dtype=np.float32)
    target = int(np.ceil(0.05 * n ** 3))
    zeroed = 0
    o = np.arange(-3, 5)
    while zeroed < target:
        c = rngp.uniform(0.0, float(n), size=3)                # (x, y, z) in index units; cell i has centre i + 0.5
        i0 = np.floor(c).astype(int)
        ix = i0[0] + o
        iy = i0[1] + o
        iz = i0[2] + o
        ix, iy, iz = (t[(t >= 0) & (t < n)] for t in (ix, iy, iz))
        gz, gy, gx = np.meshgrid(iz, iy, ix, indexing="ij")
        d2 = (gx + 0.5 - c[0]) ** 2 + (gy + 0.5 - c[1]) ** 2 + (gz + 0.5 - c[2]) ** 2
        inside = d2 <= 9.0
        sub = Nf[gz[inside], gy[inside], gx[inside]]
        zeroed += int(np.count_nonzero(sub))
        Nf[gz[inside], gy[inside], gx[inside]] = 0.0
    ax = np.arange(n, dtype=np.float32) + np.float32(0.5) - np.float32(n / 2.0)
    pos = np.empty((n ** 3, 3), dtype=np.float32)
    pos[:, 0] = np.tile(ax, n * n)
    pos[:, 1] = np.tile(np.repeat(ax, n), n)
    pos[:, 2] = np.repeat(ax, n * n)
    q = 0.01 + np.arange(n_q, dtype=np.float64) * (2.99 / max(n_q - 1, 1))
    r_max = float(np.ceil(n * np.sqrt(3.0)))                   # 444 nm for n = 256 (>= block diagonal, L270)
    r = r_max * np.arange(n_r, dtype=np.float64) / max(n_r - 1, 1)
    return Workload(
        name="C5", pos=pos, N=Nf.ravel(), m=m, grid=polar_grid(q, n_theta), kinds=list(ALL_KINDS),
        R=np.eye(3), n_bins=n_q, r=r.astype(np.float32))


def make_config(name: str, small: bool = False) -> Workload:
    """Full-size config by name, or a reduced version with the same structure (`small=True`)."""
    name = name.upper()
    if name == "C1":
        return config_c1()
    if name == "C2":
        return config_c2()
    if name == "C3":
        return config_c3(K=6, n_q=40, n_theta=48) if small else config_c3()
    if name == "C4":
        return config_c4(nx=64, ny=48, nz=4, n_rot=3, n_grid=40) if small else config_c4()
    if name == "C5":
        return config_c5(n=32, n_q=48, n_theta=64, n_r=96) if small else config_c5()
    raise ValueError(name)
