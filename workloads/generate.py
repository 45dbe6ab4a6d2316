"""Seeded synthetic workloads shaped like the paper's Chebyshev-filter benchmarks.

Stands in for the paper's benchmark systems (Mo supercells / Al nanoparticles with ONCV pseudopotentials,
PAPER.md:586-588, Sec. 5), whose structures and pseudopotential files are not available.  The five
configurations are BASELINE.json's `configs`, made concrete as in DESIGN.md ("Input recipe").

Conventions (the paper fixes none, PAPER.md:513-515 only fixes "vector index
fastest"):
  * cells      c = ci + n*(cj + n*ck), x fastest
  * cell nodes l = a + (p+1)*(b + (p+1)*c), x fastest, a,b,c in 0..p  (GLL node index per direction)
  * global dof g = gx + nd*(gy + nd*gz), periodic: nd = n*p, gx = (ci*p + a) mod nd
  * cell vertices v = vx + 2*vy + 4*vz, UNWRAPPED physical coordinates (a cell never straddles the seam)
  * quadrature points q = qa + nq1*(qb + nq1*qc), nq1 = p+2 Gauss-Legendre points per direction
  * vector block X[g, j], row-major, vector index j fastest

Nothing here evaluates shape functions, weights, matrices or the recurrence.  The Gauss-point *positions*
(needed to know where to sample V_eff and the projector functions) come from numpy's `leggauss`, a third
source independent of both the oracle's and the CUDA library's own tables.
"""
from __future__ import annotations

import json
import os
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

# --------------------------------------------------------------------------------------------------------
# configuration table (BASELINE.json configs 1..5; L for configs 3-5 chosen so that h = L/n = 2 bohr)
# --------------------------------------------------------------------------------------------------------


@dataclass(frozen=True)
class ConfigSpec:
    config: int
    n: int                 # cells per side
    p: int                 # FE degree
    L: float               # box side (bohr)
    atoms_per_side: int    # jittered lattice (0 => uniformly random centres, config 1)
    n_gaussians: int       # number of Gaussian wells if atoms_per_side == 0
    nonlocal_: bool
    smooth_field: float    # RMS (Ha) of the random smooth field, 0 => none
    N: int                 # total vectors
    B: int                 # chunk width
    m: int                 # Chebyshev degree
    precision: int         # 64 | 32
    seed_base: int         # seeds = seed_base + k
    bounds_key: str        # key into bounds.json


CONFIGS = {
    1: ConfigSpec(1, 4, 4, 8.0, 0, 4, False, 0.0, 32, 32, 10, 64, 1000, "1"),
    2: ConfigSpec(2, 8, 6, 16.0, 2, 0, True, 0.0, 256, 256, 20, 64, 2000, "2"),
    3: ConfigSpec(3, 16, 6, 32.0, 4, 0, True, 0.05, 1024, 256, 30, 64, 3000, "3"),
    # config 4 = config 3's mesh and potential (same seeds), FP32 storage
    4: ConfigSpec(4, 16, 6, 32.0, 4, 0, True, 0.05, 4096, 512, 30, 32, 3000, "3"),
    5: ConfigSpec(5, 20, 6, 40.0, 6, 0, True, 0.0, 4000, 400, 40, 64, 5000, "5"),
    # extra, NOT in BASELINE.json: config 2's box, atoms and block at FE degree 7 (the paper's other benchmark order,
    # PAPER.md:586, 601-603; M_cell = 512, 175,616 dofs) -- the p = 7 tiling of the persistent kernel
    6: ConfigSpec(6, 8, 7, 16.0, 2, 0, True, 0.0, 256, 256, 20, 64, 6000, "6"),
}

# seed offsets k: 0 V_eff centres/depths, 1 atom jitter, 2 D, 3 smooth field, 4 X,
# 5 Lanczos start, 6 Rayleigh-Ritz start
SEED_VEFF, SEED_JITTER, SEED_D, SEED_FIELD, SEED_X, SEED_LANCZOS, SEED_RR = range(7)

R_CUT = 3.0            # projector cut-off radius (bohr)
PROJ_WIDTHS = (0.6, 0.9)
GAUSS_SIGMA = 1.0      # width of the local Gaussian wells (bohr)
GAUSS_RANGE = 8.0      # wells are dropped beyond 8 sigma (exp(-32) ~ 1e-14)


@dataclass
class Workload:
    spec: Optional[ConfigSpec]
    p: int
    n_cells: int
    n_dofs: int
    cell_dofs: np.ndarray        # int32 [n_cells, (p+1)^3]
    cell_vertices: np.ndarray    # float64 [n_cells, 8, 3]
    veff_q: np.ndarray           # float64 [n_cells, (p+2)^3]
    # non-local part (n_proj == 0 => none)
    n_proj: int = 0
    D: np.ndarray = field(default_factory=lambda: np.zeros(0))
    proj_cell_ptr: np.ndarray = field(default_factory=lambda: np.zeros(1, dtype=np.int64))
    proj_cell_idx: np.ndarray = field(default_factory=lambda: np.zeros(0, dtype=np.int32))
    chi_q: np.ndarray = field(default_factory=lambda: np.zeros((0, 0)))
    L: float = 0.0
    n: int = 0
    periodic: bool = True
    atoms: np.ndarray = field(default_factory=lambda: np.zeros((0, 3)))
    # k-point variant: kvec [3] and the imaginary parts of the projector samples (chi_q then holds the real parts)
    kvec: Optional[np.ndarray] = None
    chi_q_im: Optional[np.ndarray] = None

    @property
    def m_cell(self) -> int:
        return (self.p + 1) ** 3

    @property
    def n_q(self) -> int:
        return (self.p + 2) ** 3


# --------------------------------------------------------------------------------------------------------
# mesh
# --------------------------------------------------------------------------------------------------------


def make_mesh(n: int, p: int, L: float, periodic: bool = True, jitter: float = 0.0, seed: int = 0):
    """Uniform n^3 hexahedral mesh of a cube of side L; returns (cell_dofs, cell_vertices, n_dofs).

    `jitter` (fraction of h) displaces the mesh vertices randomly (consistently across the periodic seam)
    so that cells become general trilinear hexahedra; only used by tests of the non-affine path.
    """
    if n < 1 or p < 1:
        raise ValueError("n >= 1 and p >= 1 required")
    if periodic and n < 2:
        raise ValueError("periodic meshes need n >= 2 (a dof may not repeat inside one cell)")
    h = L / n
    nd = n * p if periodic else n * p + 1
    nv = n if periodic else n + 1
    c = np.arange(n ** 3)
    ci, cj, ck = c % n, (c // n) % n, c // (n * n)
    l = np.arange((p + 1) ** 3)
    la, lb, lc = l % (p + 1), (l // (p + 1)) % (p + 1), l // ((p + 1) ** 2)
    gx = ci[:, None] * p + la[None, :]
    gy = cj[:, None] * p + lb[None, :]
    gz = ck[:, None] * p + lc[None, :]
    if periodic:
        gx, gy, gz = gx % nd, gy % nd, gz % nd
    cell_dofs = (gx + nd * (gy + nd * gz)).astype(np.int32)

    disp = np.zeros((nv, nv, nv, 3))
    if jitter != 0.0:
        rng = np.random.default_rng(seed)
        disp = rng.uniform(-jitter * h, jitter * h, size=(nv, nv, nv, 3))
        if not periodic:  # keep the outer boundary flat
            for d in range(3):
                sl = [slice(None)] * 3
                for edge in (0, nv - 1):
                    sl[d] = edge
                    disp[tuple(sl) + (d,)] = 0.0
    verts = np.empty((n ** 3, 8, 3))
    for v in range(8):
        vx, vy, vz = v & 1, (v >> 1) & 1, (v >> 2) & 1
        ix, iy, iz = ci + vx, cj + vy, ck + vz
        base = np.stack([ix * h, iy * h, iz * h], axis=1).astype(np.float64)
        verts[:, v, :] = base + disp[ix % nv, iy % nv, iz % nv]
    return cell_dofs, verts, nd ** 3


def gauss_points_physical(cell_vertices: np.ndarray, p: int) -> np.ndarray:
    """Physical coordinates [n_cells, (p+2)^3, 3] of the Gauss-Legendre points (x fastest) under the
    trilinear map of each cell.  Positions only (used to sample the synthetic fields)."""
    nq1 = p + 2
    xi, _ = np.polynomial.legendre.leggauss(nq1)
    q = np.arange(nq1 ** 3)
    ref = np.stack([xi[q % nq1], xi[(q // nq1) % nq1], xi[q // (nq1 * nq1)]], axis=1)  # [nq, 3]
    out = np.zeros((cell_vertices.shape[0], ref.shape[0], 3))
    for v in range(8):
        sx = (1 + (2 * (v & 1) - 1) * ref[:, 0]) / 2
        sy = (1 + (2 * ((v >> 1) & 1) - 1) * ref[:, 1]) / 2
        sz = (1 + (2 * ((v >> 2) & 1) - 1) * ref[:, 2]) / 2
        out += (sx * sy * sz)[None, :, None] * cell_vertices[:, v, None, :]
    return out


# --------------------------------------------------------------------------------------------------------
# synthetic fields
# --------------------------------------------------------------------------------------------------------


def _image_shifts(L: float, periodic: bool):
    if not periodic:
        return np.zeros((1, 3))
    s = np.array([-1.0, 0.0, 1.0]) * L
    return np.array([[a, b, c] for a in s for b in s for c in s])


def _cells_near(centres: np.ndarray, half_diag: float, pos: np.ndarray, radius: float) -> np.ndarray:
    d = np.linalg.norm(centres - pos[None, :], axis=1)
    return np.nonzero(d <= radius + half_diag)[0]


def _gaussian_wells(xq, centres, half_diag, atoms, depths, L, periodic):
    v = np.zeros(xq.shape[:2])
    for pos, dep in zip(atoms, depths):
        for sh in _image_shifts(L, periodic):
            cells = _cells_near(centres, half_diag, pos + sh, GAUSS_RANGE * GAUSS_SIGMA)
            if cells.size == 0:
                continue
            r2 = np.sum((xq[cells] - (pos + sh)[None, None, :]) ** 2, axis=2)
            v[cells] += dep * np.exp(-r2 / (2 * GAUSS_SIGMA ** 2))
    return v


def _smooth_field(xq, L, rms, seed):
    """Seeded low Fourier modes (|n|_inf <= 2, n != 0), scaled to the requested RMS."""
    rng = np.random.default_rng(seed)
    modes = [(i, j, k) for i in range(-2, 3) for j in range(-2, 3) for k in range(-2, 3) if (i, j, k) > (0, 0, 0)]
    amp = rng.standard_normal(len(modes))
    phase = rng.uniform(0, 2 * np.pi, len(modes))
    amp *= rms / np.sqrt(np.sum(amp ** 2) / 2)
    out = np.zeros(xq.shape[:2])
    w = 2 * np.pi / L
    # separable evaluation: cos(a+b+c+phi) via complex exponentials per direction
    ex = {k: np.exp(1j * w * k * xq[..., 0]) for k in range(-2, 3)}
    ey = {k: np.exp(1j * w * k * xq[..., 1]) for k in range(-2, 3)}
    ez = {k: np.exp(1j * w * k * xq[..., 2]) for k in range(-2, 3)}
    for (i, j, k), a, ph in zip(modes, amp, phase):
        out += a * np.real(ex[i] * ey[j] * ez[k] * np.exp(1j * ph))
    return out


def _radial_norms(s: float, rc: float):
    """1/sqrt(int chi^2) for the l=0 and l=1 projector shapes (fine composite Simpson rule)."""
    r = np.linspace(0.0, rc, 20001)
    f2 = (np.exp(-r ** 2 / (2 * s ** 2)) * (1 - (r / rc) ** 2) ** 2) ** 2
    w = np.ones_like(r)
    w[1:-1:2], w[2:-1:2] = 4.0, 2.0
    w *= (r[1] - r[0]) / 3
    n0 = 4 * np.pi * np.sum(w * f2 * r ** 2)
    n1 = 4 * np.pi / 3 * np.sum(w * f2 * r ** 4)
    return 1 / np.sqrt(n0), 1 / np.sqrt(n1)


def _projectors(xq, centres, half_diag, atoms, L, periodic, rc, kvec=None):
    """Per atom: support cells and chi values [8, n_support, nq] (l=0,1 x 2 radial widths).  With a k-point the values
    are the complex samples of sum_r e^{-i k.(x - L_r)} chi(x, R_a + L_r) (Eq. 33), L_r = image shift."""
    result = []
    norms = [_radial_norms(s, rc) for s in PROJ_WIDTHS]
    for pos in atoms:
        cells_all, chunks = [], {}
        for sh in _image_shifts(L, periodic):
            cells = _cells_near(centres, half_diag, pos + sh, rc)
            if cells.size == 0:
                continue
            d = xq[cells] - (pos + sh)[None, None, :]
            r = np.linalg.norm(d, axis=2)
            inside = r < rc
            keep = np.nonzero(inside.any(axis=1))[0]
            for kk in keep:
                c = int(cells[kk])
                vals = np.zeros((8, xq.shape[1]), dtype=np.float64 if kvec is None else np.complex128)
                phase = 1.0 if kvec is None else np.exp(-1j * ((xq[cells[kk]] - sh[None, :]) @ np.asarray(kvec)))
                for si, s in enumerate(PROJ_WIDTHS):
                    f = np.where(inside[kk], np.exp(-r[kk] ** 2 / (2 * s ** 2)) * (1 - (r[kk] / rc) ** 2) ** 2, 0.0)
                    vals[4 * si + 0] = norms[si][0] * f * phase
                    for ax in range(3):
                        vals[4 * si + 1 + ax] = norms[si][1] * f * d[kk, :, ax] * phase
                if c in chunks:
                    chunks[c] += vals
                else:
                    chunks[c] = vals
                    cells_all.append(c)
        cells_sorted = sorted(cells_all)
        chi = np.stack([chunks[c] for c in cells_sorted], axis=1) if cells_sorted else np.zeros((8, 0, xq.shape[1]))
        result.append((np.array(cells_sorted, dtype=np.int32), chi))
    return result


def _lattice_atoms(k: int, L: float, jitter: float, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    g = (np.arange(k) + 0.5) * (L / k)
    pts = np.array([[x, y, z] for z in g for y in g for x in g])
    return pts + rng.uniform(-jitter, jitter, size=pts.shape)


def make_workload(config: Optional[int] = None, *, n=None, p=None, L=None, periodic=True, mesh_jitter=0.0,
                  atoms_per_side=None, n_gaussians=None, nonlocal_=None, smooth_field=None, seed_base=None,
                  r_cut=R_CUT, kvec=None) -> Workload:
    """Build the operator inputs of a BASELINE.json config (or a custom small case for tests).  `kvec` (bohr^-1) selects
    the k-point variant: the projector samples then carry the Bloch phase of Eq. 33 (real and imaginary parts)."""
    spec = CONFIGS[config] if config is not None else None
    pick = lambda v, name: v if v is not None else getattr(spec, name)
    n, p, L = pick(n, "n"), pick(p, "p"), float(pick(L, "L"))
    aps, ng = pick(atoms_per_side, "atoms_per_side"), pick(n_gaussians, "n_gaussians")
    nl, sf, sb = pick(nonlocal_, "nonlocal_"), pick(smooth_field, "smooth_field"), pick(seed_base, "seed_base")

    cell_dofs, verts, n_dofs = make_mesh(n, p, L, periodic=periodic, jitter=mesh_jitter, seed=sb + 99)
    xq = gauss_points_physical(verts, p)
    centres = verts.mean(axis=1)
    half_diag = float(np.max(np.linalg.norm(verts - centres[:, None, :], axis=2)))

    rng = np.random.default_rng(sb + SEED_VEFF)
    if aps and aps > 0:
        atoms = _lattice_atoms(aps, L, 0.5, sb + SEED_JITTER)
    else:
        atoms = rng.uniform(0.0, L, size=(ng, 3))
    depths = rng.uniform(-2.0, -0.5, size=len(atoms))
    veff = _gaussian_wells(xq, centres, half_diag, atoms, depths, L, periodic)
    if sf and sf > 0:
        veff += _smooth_field(xq, L, sf, sb + SEED_FIELD)

    wl = Workload(spec=spec, p=p, n_cells=n ** 3, n_dofs=n_dofs, cell_dofs=cell_dofs, cell_vertices=verts,
                  veff_q=np.ascontiguousarray(veff), L=L, n=n, periodic=periodic, atoms=atoms)
    if nl:
        per_atom = _projectors(xq, centres, half_diag, atoms, L, periodic, r_cut, kvec)
        ptr, idx, chi = [0], [], []
        for cells, vals in per_atom:
            for j in range(8):
                idx.append(cells)
                chi.append(vals[j])
                ptr.append(ptr[-1] + len(cells))
        wl.n_proj = 8 * len(per_atom)
        wl.proj_cell_ptr = np.array(ptr, dtype=np.int64)
        wl.proj_cell_idx = np.concatenate(idx).astype(np.int32) if idx else np.zeros(0, dtype=np.int32)
        wl.chi_q = np.ascontiguousarray(np.concatenate(chi, axis=0)) if chi else np.zeros((0, xq.shape[1]))
        if kvec is not None:
            wl.chi_q_im = np.ascontiguousarray(wl.chi_q.imag)
            wl.chi_q = np.ascontiguousarray(wl.chi_q.real)
        wl.D = np.random.default_rng(sb + SEED_D).uniform(-1.0, 1.0, size=wl.n_proj)
    if kvec is not None:
        wl.kvec = np.asarray(kvec, dtype=np.float64)
    return wl


def random_block(n_dofs: int, cols, seed: int) -> np.ndarray:
    """Columns `cols` of the N(0,1) block X (each column has its own stream, so any subset of columns of a
    large block can be produced without generating the rest).  Returns float64 [n_dofs, len(cols)]."""
    cols = list(cols)
    out = np.empty((n_dofs, len(cols)))
    for k, j in enumerate(cols):
        out[:, k] = np.random.default_rng([seed, int(j)]).standard_normal(n_dofs)
    return out


def load_bounds(key: str, recipe: str = "B"):
    """(a0, a, b) stored by oracle/make_bounds.py (a committed script that calls only the oracle)."""
    path = os.path.join(os.path.dirname(__file__), "bounds.json")
    with open(path) as f:
        table = json.load(f)
    e = table[str(key)][recipe]
    return float(e["a0"]), float(e["a"]), float(e["b"])
