"""Seeded synthetic input generators (meshes, materials, initial fields) for the five
BASELINE.json configs.

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA library; it holds none
of the method's arithmetic (no shape functions, no matrices, no fields, no solver) --
only numpy random numbers, grid bookkeeping and the config tables.  It imports neither
the oracle nor the CUDA binding.

Recipe:
  * structured nx*ny*nz node grid over a box, node id = (iz*ny + iy)*nx + ix;
  * every hexahedron split into 6 Kuhn tetrahedra, one per permutation pi of the axes:
    {v, v+e_pi1, v+e_pi1+e_pi2, v+(1,1,1)};
  * interior nodes jittered uniformly by +-15 % of the grid spacing (face nodes are not,
    so box faces stay planar and "bottom face" is exactly z = 0);
  * node labels randomly permuted (seeded) so that the user ordering has no locality;
  * tets whose centroid lies inside a sphere / rotated ellipsoid are flagged
    non-magnetic with a second (x2 stiffer) elastic material.
These meshes stand in for the paper's COMSOL tetrahedral meshes, which
are not available; they have the same graph statistics (~14.8 nnz/row, ~23 tets/node).
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field, replace  # noqa: F401 (replace re-exported)
from typing import Optional, Tuple

import numpy as np

# physics term bits (same numeric values as include/cupymag_b200.h; plain constants)
TERM_ANIS = 1
TERM_ZEEMAN = 2
TERM_DEMAG = 4
TERM_FARFIELD = 8
TERM_MAGEL = 16

MU0 = 4.0e-7 * np.pi


@dataclass
class Material:
    Ms: float = 1.2e6            # A/m
    Aex: float = 1.3e-11         # J/m
    K1: float = 2.0e4            # J/m^3
    lambda100: float = 2.0e-4
    lambda111: float = -2.0e-5
    alpha: float = 0.5
    gamma: float = 2.211e5       # m/(A s)
    length_scale: float = 1.0e-9  # l_d, m
    Nd: Tuple[float, ...] = (1 / 3, 0, 0, 0, 1 / 3, 0, 0, 0, 1 / 3)   # sphere
    C_voigt: np.ndarray = field(default_factory=lambda: isotropic_voigt(200e9, 0.3)[None])   # crystal axes
    R: Optional[np.ndarray] = None   # App. D: crystal -> simulation frame (3x3, v_sim = R v_crystal); None = identity
    sigma_ext: Optional[np.ndarray] = None   # uniform external stress (6,) Pa, Voigt xx,yy,zz,yz,xz,xy (Eq. 1); None = 0


def isotropic_voigt(E: float, nu: float) -> np.ndarray:
    """6x6 isotropic stiffness (Pa), Voigt order xx,yy,zz,yz,xz,xy, engineering shears."""
    lam = E * nu / ((1 + nu) * (1 - 2 * nu))
    mu = E / (2 * (1 + nu))
    C = np.zeros((6, 6))
    C[:3, :3] = lam
    C[np.arange(3), np.arange(3)] = lam + 2 * mu
    C[np.arange(3, 6), np.arange(3, 6)] = mu
    return C


def cubic_voigt(C11: float, C12: float, C44: float) -> np.ndarray:
    """6x6 stiffness of a cubic crystal in its own axes (Voigt xx,yy,zz,yz,xz,xy; engineering shears), Pa."""
    C = np.zeros((6, 6))
    C[:3, :3] = C12
    C[np.arange(3), np.arange(3)] = C11
    C[np.arange(3, 6), np.arange(3, 6)] = C44
    return C


R_111 = np.array([[1 / np.sqrt(3), 1 / np.sqrt(3), 1 / np.sqrt(3)],
                  [-1 / np.sqrt(2), 1 / np.sqrt(2), 0.0],
                  [-1 / np.sqrt(6), -1 / np.sqrt(6), 2 / np.sqrt(6)]])   # Eq. D.1: axes <111>, <-110>, <-1-12>


@dataclass
class Mesh:
    xyz: np.ndarray          # (N,3) float64, metres, user node order
    tets: np.ndarray         # (Ne,4) int32, user node labels
    magnetic: np.ndarray     # (Ne,) uint8
    elastic_id: np.ndarray   # (Ne,) int32
    grid: Tuple[int, int, int]
    box: Tuple[float, float, float]
    node_perm: np.ndarray    # (N,) structured id -> user label

    @property
    def n_nodes(self) -> int:
        return self.xyz.shape[0]

    @property
    def n_tets(self) -> int:
        return self.tets.shape[0]

    def live_nodes(self) -> np.ndarray:
        """Nodes touched by at least one magnetic tet (mesh bookkeeping only)."""
        live = np.zeros(self.n_nodes, dtype=bool)
        live[self.tets[self.magnetic != 0].ravel()] = True
        return live


def kuhn_box(grid, box, jitter=0.15, seed_mesh=1, seed_perm=2, permute=True) -> Mesh:
    nx, ny, nz = grid
    Lx, Ly, Lz = box
    n = nx * ny * nz
    ix, iy, iz = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    # node id = (iz*ny + iy)*nx + ix  -> order arrays accordingly
    order = np.argsort(((iz * ny + iy) * nx + ix).ravel(), kind="stable")
    ix, iy, iz = ix.ravel()[order], iy.ravel()[order], iz.ravel()[order]
    h = np.array([Lx / (nx - 1), Ly / (ny - 1), Lz / (nz - 1)])
    xyz = np.stack([ix * h[0], iy * h[1], iz * h[2]], axis=1).astype(np.float64)
    interior = (ix > 0) & (ix < nx - 1) & (iy > 0) & (iy < ny - 1) & (iz > 0) & (iz < nz - 1)
    rng = np.random.default_rng(seed_mesh)
    d = rng.uniform(-jitter, jitter, size=(n, 3)) * h
    xyz[interior] += d[interior]

    # hexes
    hx, hy, hz = np.meshgrid(np.arange(nx - 1), np.arange(ny - 1), np.arange(nz - 1), indexing="ij")
    hx, hy, hz = hx.ravel(), hy.ravel(), hz.ravel()

    def nid(a, b, c):
        return (c * ny + b) * nx + a

    tets = []
    for pi in itertools.permutations(range(3)):
        off = np.zeros((4, 3), dtype=np.int64)
        off[1, pi[0]] = 1
        off[2, pi[0]] = 1
        off[2, pi[1]] = 1
        off[3, :] = 1
        cols = [nid(hx + off[k, 0], hy + off[k, 1], hz + off[k, 2]) for k in range(4)]
        tets.append(np.stack(cols, axis=1))
    # interleave so that the 6 tets of one hex are consecutive
    tets = np.stack(tets, axis=1).reshape(-1, 4)

    if permute:
        P = np.random.default_rng(seed_perm).permutation(n)     # structured id -> user label
    else:
        P = np.arange(n)
    xyz_u = np.empty_like(xyz)
    xyz_u[P] = xyz
    tets_u = P[tets].astype(np.int32)
    ne = tets_u.shape[0]
    return Mesh(xyz=xyz_u, tets=np.ascontiguousarray(tets_u),
                magnetic=np.ones(ne, dtype=np.uint8), elastic_id=np.zeros(ne, dtype=np.int32),
                grid=tuple(grid), box=tuple(box), node_perm=P)


@dataclass
class HexMesh:
    """Linear hexahedra; local node a = i + 2 j + 4 k of hexes[e] sits at corner (i, j, k) of the cell (R26)."""
    xyz: np.ndarray          # (N, 3) metres
    hexes: np.ndarray        # (Ne, 8) int32
    magnetic: np.ndarray
    elastic_id: np.ndarray
    grid: Tuple[int, int, int] = (0, 0, 0)
    box: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    node_perm: Optional[np.ndarray] = None

    @property
    def n_nodes(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def n_tets(self) -> int:          # number of elements (the name the binding and the oracle read)
        return int(self.hexes.shape[0])

    def live_nodes(self) -> np.ndarray:
        """Nodes touched by at least one magnetic cell (mesh bookkeeping only)."""
        live = np.zeros(self.n_nodes, dtype=bool)
        live[self.hexes[self.magnetic != 0].ravel()] = True
        return live


def hex_box(grid, box, jitter=0.15, seed_mesh=1, seed_perm=2, permute=True) -> HexMesh:
    """Structured nx x ny x nz node grid of linear hexahedra (the paper's Fig. 2-3 meshes): same node numbering,
    jitter and label permutation as kuhn_box, one hexahedron per cell."""
    t = kuhn_box(grid, box, jitter=jitter, seed_mesh=seed_mesh, seed_perm=seed_perm, permute=permute)
    nx, ny, nz = grid
    hx, hy, hz = np.meshgrid(np.arange(nx - 1), np.arange(ny - 1), np.arange(nz - 1), indexing="ij")
    hx, hy, hz = hx.ravel(), hy.ravel(), hz.ravel()
    cols = [((hz + k) * ny + (hy + j)) * nx + (hx + i) for k in (0, 1) for j in (0, 1) for i in (0, 1)]   # a = i + 2 j + 4 k
    hexes = t.node_perm[np.stack(cols, axis=1)].astype(np.int32)
    ne = hexes.shape[0]
    return HexMesh(xyz=t.xyz, hexes=np.ascontiguousarray(hexes), magnetic=np.ones(ne, np.uint8), elastic_id=np.zeros(ne, np.int32),
                   grid=tuple(grid), box=tuple(box), node_perm=t.node_perm)


def delaunay_box(grid, box, jitter=0.45, seed_mesh=1, seed_perm=2, permute=True) -> Mesh:
    """Unstructured tetrahedral mesh with the valence spread of a real mesh generator's output (the paper's COMSOL meshes,
    P:298-306: 8-30 neighbours per node, where the Kuhn split of kuhn_box has 14 almost everywhere): Delaunay
    tetrahedralisation (scipy / Qhull) of an nx x ny x nz lattice whose INTERIOR nodes are displaced uniformly by
    +-jitter of the spacing in every direction and whose face nodes slide within their face.  Flat cells that Qhull leaves
    between coplanar face nodes (volume below 1e-6 of the mean cell volume) are dropped.  Mesh bookkeeping only."""
    from scipy.spatial import Delaunay
    nx, ny, nz = grid
    n = nx * ny * nz
    ix, iy, iz = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    order = np.argsort(((iz * ny + iy) * nx + ix).ravel(), kind="stable")      # node id = (iz ny + iy) nx + ix
    idx = np.stack([ix.ravel()[order], iy.ravel()[order], iz.ravel()[order]], axis=1)
    h = np.array([box[d] / (grid[d] - 1) for d in range(3)])
    on_face = (idx == 0) | (idx == np.array(grid) - 1)           # per node, per direction: fixed in that direction
    rng = np.random.default_rng(seed_mesh)
    xyz = idx * h + np.where(on_face, 0.0, jitter * h * rng.uniform(-1.0, 1.0, size=(n, 3)))
    tets = Delaunay(xyz).simplices.astype(np.int64)
    a, b, c, d = (xyz[tets[:, k]] for k in range(4))
    vol = np.einsum("ij,ij->i", np.cross(b - a, c - a), d - a) / 6.0
    keep = np.abs(vol) > 1e-6 * np.abs(vol).mean()
    tets, vol = tets[keep], vol[keep]
    neg = vol < 0                                                # positive orientation, as kuhn_box gives
    tets[neg] = tets[neg][:, [0, 2, 1, 3]]
    n = xyz.shape[0]
    perm = np.random.default_rng(seed_perm).permutation(n) if permute else np.arange(n)
    xyz_p = np.empty_like(xyz); xyz_p[perm] = xyz                # old node i -> label perm[i]
    tets = perm[tets].astype(np.int32)
    ne = tets.shape[0]
    return Mesh(xyz=np.ascontiguousarray(xyz_p), tets=np.ascontiguousarray(tets), magnetic=np.ones(ne, np.uint8),
                elastic_id=np.zeros(ne, np.int32), grid=tuple(grid), box=tuple(box), node_perm=perm)


def flag_inclusion(mesh: Mesh, center, semi_axes, rotation: Optional[np.ndarray] = None) -> Mesh:
    """Flag elements (tets or hexahedra) whose centroid lies inside the (rotated) ellipsoid as non-magnetic,
    elastic material 1."""
    conn = mesh.hexes if hasattr(mesh, "hexes") else mesh.tets
    c = mesh.xyz[conn].mean(axis=1) - np.asarray(center)
    if rotation is not None:
        c = c @ rotation          # coordinates in the ellipsoid frame (columns = axes)
    inside = ((c / np.asarray(semi_axes)) ** 2).sum(axis=1) <= 1.0
    mag = mesh.magnetic.copy()
    eid = mesh.elastic_id.copy()
    mag[inside] = 0
    eid[inside] = 1
    return replace(mesh, magnetic=mag, elastic_id=eid)


def random_rotation(seed: int) -> np.ndarray:
    q = np.random.default_rng(seed).normal(size=4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def init_m_random(mesh: Mesh, seed: int) -> np.ndarray:
    m = np.random.default_rng(seed).normal(size=(mesh.n_nodes, 3))
    m /= np.linalg.norm(m, axis=1, keepdims=True)
    m[~mesh.live_nodes()] = 0.0
    return m


def init_m_noisy_x(mesh: Mesh, seed: int, amp: float = 0.1) -> np.ndarray:
    m = np.array([1.0, 0.0, 0.0]) + amp * np.random.default_rng(seed).normal(size=(mesh.n_nodes, 3))
    m /= np.linalg.norm(m, axis=1, keepdims=True)
    m[~mesh.live_nodes()] = 0.0
    return m


def clamp_bottom(mesh: Mesh) -> np.ndarray:
    """uint8 mask (N*3,) : all three displacement DOFs of nodes with z == 0 exactly."""
    c = np.zeros((mesh.n_nodes, 3), dtype=np.uint8)
    c[mesh.xyz[:, 2] == 0.0] = 1
    return c.ravel()


@dataclass
class Config:
    name: str
    mesh: Mesh
    material: Material
    m0: np.ndarray
    terms: int
    dt: float
    steps: int
    Hext: np.ndarray                     # (steps,3) A/m, field used at step k
    clamp_dof: Optional[np.ndarray] = None
    pin_node: int = 0
    dtypes: Tuple[str, ...] = ("f64",)


def _mT_to_Am(mT: float) -> float:
    return mT * 1e-3 / MU0


def make_config(idx: int, grid=None, box=None) -> Config:
    """BASELINE.json configs 0..3.  `grid` / `box` override the node grid / box lengths (same recipe,
    same seeds) so that parity tests and the timed CPU baseline can run a reduced instance of the big
    configs (e.g. a sub-box of config 3 at the same mesh spacing)."""
    nm = 1e-9
    if idx == 0:
        g = grid or (8, 8, 8)
        mesh = kuhn_box(g, (20 * nm,) * 3, seed_mesh=1, seed_perm=2)
        mat = Material()
        steps = 10
        return Config("config0_tiny_cube", mesh, mat, init_m_random(mesh, 3),
                      TERM_ANIS | TERM_DEMAG | TERM_FARFIELD, 1e-12, steps,
                      np.zeros((steps, 3)))
    if idx == 1:
        g = grid or (81, 81, 21)
        mesh = kuhn_box(g, (200 * nm, 200 * nm, 50 * nm), seed_mesh=11, seed_perm=12)
        mat = Material()
        steps = 100
        H = np.zeros((steps, 3))
        H[:, 0] = -_mT_to_Am(50.0)
        return Config("config1_cuboid", mesh, mat, init_m_noisy_x(mesh, 13),
                      TERM_ANIS | TERM_ZEEMAN, 5e-12, steps, H, dtypes=("f64", "f32"))
    if idx == 2:
        g = grid or (129, 129, 31)
        box = box or (400 * nm, 400 * nm, 100 * nm)
        mesh = kuhn_box(g, box, seed_mesh=21, seed_perm=22)
        mesh = flag_inclusion(mesh, np.array(box) / 2, (40 * nm,) * 3)
        C = isotropic_voigt(200e9, 0.3)
        mat = Material(C_voigt=np.stack([C, 2 * C]))
        steps = 50
        return Config("config2_magnetoelastic", mesh, mat, init_m_noisy_x(mesh, 23),
                      TERM_ANIS | TERM_ZEEMAN | TERM_DEMAG | TERM_FARFIELD | TERM_MAGEL,
                      10e-12, steps, np.zeros((steps, 3)), clamp_dof=clamp_bottom(mesh))
    if idx == 3:
        g = grid or (245, 245, 50)
        box = box or (1000 * nm, 1000 * nm, 200 * nm)
        mesh = kuhn_box(g, box, seed_mesh=31, seed_perm=32)
        mesh = flag_inclusion(mesh, np.array(box) / 2, (120 * nm, 60 * nm, 40 * nm),
                              rotation=random_rotation(34))
        C = isotropic_voigt(200e9, 0.3)
        mat = Material(C_voigt=np.stack([C, 2 * C]))
        steps = 20
        H = np.zeros((steps, 3))
        H[:, 0] = _mT_to_Am(-100.0 + 200.0 * np.arange(steps) / (steps - 1))
        return Config("config3_paper_scale", mesh, mat, init_m_noisy_x(mesh, 33),
                      TERM_ANIS | TERM_ZEEMAN | TERM_DEMAG | TERM_FARFIELD | TERM_MAGEL,
                      11e-12, steps, H, clamp_dof=clamp_bottom(mesh), dtypes=("f64", "f32"))
    raise ValueError(idx)


def make_config4_mesh(n_side: int, permute: bool = True) -> Mesh:
    """Config 4 (SpMV/CG microbenchmark): cube of n_side^3 nodes, 2.5 nm spacing."""
    L = 2.5e-9 * (n_side - 1)
    return kuhn_box((n_side,) * 3, (L, L, L), seed_mesh=41, seed_perm=42, permute=permute)


def make_config4_hex_mesh(n_side: int, permute: bool = True) -> HexMesh:
    """The same cube as make_config4_mesh meshed with linear hexahedra (the paper's Fig. 2 workload)."""
    L = (n_side - 1) * 2.5e-9
    return hex_box((n_side,) * 3, (L,) * 3, seed_mesh=41, seed_perm=42, permute=permute)


def clamp_face_x0(mesh: Mesh) -> np.ndarray:
    c = np.zeros((mesh.n_nodes, 3), dtype=np.uint8)
    c[mesh.xyz[:, 0] == 0.0] = 1
    return c.ravel()
