"""Seeded synthetic input generators (molecule, basis, grid, density) for the sn-K path.

This module is the ONE piece shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2303_14280_b200/snk.py``).  It holds none of the method's
arithmetic: it produces atoms, shells, quadrature points/weights and a density
matrix P, i.e. exactly the *inputs* of Alg. 1 ("Input: density
matrix D, basis set B") and of Eq. 38-40.

The five workloads are BASELINE.json's ``configs``; the recipe (RNG, draw order,
distributions) is stated in DESIGN.md "Input recipe" and follows SURVEY.md §8(d).
They *stand in* for the paper's Table I molecules / 6-31G(d) basis / Table II
grids, which are not available offline.

Units: the library API is in bohr; geometries are specified in Å and converted
with 1 bohr = 0.529177210903 Å.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

BOHR_PER_ANGSTROM = 1.0 / 0.529177210903
SEED_BASE = 230314280

__all__ = [
    "Basis", "Workload", "CONFIGS", "make_workload", "make_basis", "normalise_shell",
    "becke_grid", "ncart", "cart_components", "density_from_C", "custom_workload",
]


def ncart(l: int) -> int:
    return (l + 1) * (l + 2) // 2


def cart_components(l: int):
    """Cartesian component order inside a shell (include/snk.h): i from l down to 0,
    then j from l-i down to 0  ->  xx, xy, xz, yy, yz, zz for l = 2."""
    return [(i, j, l - i - j) for i in range(l, -1, -1) for j in range(l - i, -1, -1)]


@dataclasses.dataclass
class Basis:
    """Flattened contracted Cartesian Gaussian shells (Eq. 13).

    phi(r) = x_A^i y_A^j z_A^k * sum_k coef[k] * exp(-exp[k] r_A^2); ``coef`` is the FULL
    coefficient (normalisation already folded in)."""
    atom_xyz: np.ndarray      # [natoms,3] bohr
    shell_atom: np.ndarray    # [nshells] int32
    shell_l: np.ndarray       # [nshells] int32
    shell_nprim: np.ndarray   # [nshells] int32
    prim_exp: np.ndarray      # [sum nprim]
    prim_coef: np.ndarray     # [sum nprim]

    @property
    def nshells(self) -> int:
        return int(self.shell_l.shape[0])

    @property
    def nbf(self) -> int:
        return int(sum(ncart(int(l)) for l in self.shell_l))

    @property
    def shell_offset(self) -> np.ndarray:
        """first basis-function index of each shell, length nshells+1"""
        return np.concatenate([[0], np.cumsum([ncart(int(l)) for l in self.shell_l])]).astype(np.int64)

    @property
    def prim_offset(self) -> np.ndarray:
        return np.concatenate([[0], np.cumsum(self.shell_nprim)]).astype(np.int64)


@dataclasses.dataclass
class Workload:
    name: str
    cfg: int
    basis: Basis
    points: np.ndarray        # [npts,3] bohr, float64
    weights: np.ndarray       # [npts]   float64, >= 0
    P: np.ndarray             # [nbf,nbf] symmetric
    eps: float                # screening threshold (0 => none)
    batch_cell: float = 6.0   # h0, bohr
    batch_max: int = 2048     # N_max
    grid_shape: tuple = ()    # (n_r, n_theta, n_phi)
    atoms_z: tuple = ()


def _double_factorial(n: int) -> float:
    r = 1.0
    while n > 1:
        r *= n
        n -= 2
    return r


def normalise_shell(l: int, exps: np.ndarray, raw: np.ndarray) -> np.ndarray:
    """R5: primitive norm (2z/pi)^(3/4) (4z)^(l/2) / sqrt((2l-1)!!), then
    scale the contraction so that the (l,0,0) component has unit self-overlap
    sum_kl c_k c_l (2l-1)!!/(2p)^l (pi/p)^(3/2) = 1, p = z_k + z_l."""
    exps = np.asarray(exps, dtype=np.float64)
    df = _double_factorial(2 * l - 1)
    c = np.asarray(raw, dtype=np.float64) * (2.0 * exps / math.pi) ** 0.75 * (4.0 * exps) ** (l / 2.0) / math.sqrt(df)
    p = exps[:, None] + exps[None, :]
    S = (c[:, None] * c[None, :] * df / (2.0 * p) ** l * (math.pi / p) ** 1.5).sum()
    return c / math.sqrt(S)


# element -> list of (l, nprim); BASELINE.json configs
_SHELLS_WATER_SMALL = {8: [(0, 3), (0, 1), (1, 1)], 1: [(0, 2), (0, 1)]}
_SHELLS_WATER_D = {8: [(0, 6), (0, 3), (0, 1), (1, 3), (1, 1), (2, 1)], 1: [(0, 3), (0, 1), (1, 1)]}
_SHELLS_CARBON_F = {6: [(0, 6), (0, 3), (0, 1), (1, 3), (1, 1), (2, 2), (2, 1), (3, 1)]}

CONFIGS = {
    1: dict(name="water1", shells=_SHELLS_WATER_SMALL, exp_range=(0.1, 100.0), grid=(20, 8, 16), nocc=5, sigma=0.3, eps=0.0),
    2: dict(name="water8", shells=_SHELLS_WATER_D, exp_range=(0.1, 100.0), grid=(40, 14, 28), nocc=40, sigma=1.0, eps=1e-12, lattice=2),
    3: dict(name="water64", shells=_SHELLS_WATER_D, exp_range=(0.1, 100.0), grid=(50, 16, 32), nocc=320, sigma=None, eps=1e-11, lattice=4),
    4: dict(name="water343", shells=_SHELLS_WATER_D, exp_range=(0.1, 100.0), grid=(50, 16, 32), nocc=1715, sigma=None, eps=1e-10, lattice=7),
    5: dict(name="carbon32f", shells=_SHELLS_CARBON_F, exp_range=(0.05, 5000.0), grid=(60, 18, 36), nocc=96, sigma=1.0, eps=1e-12),
}

_WATER_ANG = np.array([[0.0, 0.0, 0.0], [0.757, 0.587, 0.0], [-0.757, 0.587, 0.0]])


def _water_cluster(rng: np.random.Generator, n: int, spacing=3.1, jitter=0.2):
    """n x n x n lattice of waters; per molecule: random rotation (unit quaternion from 4
    normals) about O, then O displaced by U(-jitter, jitter)^3 Å."""
    zs, xyz = [], []
    for ix in range(n):
        for iy in range(n):
            for iz in range(n):
                q = rng.standard_normal(4)
                q /= np.linalg.norm(q)
                w, x, y, z = q
                R = np.array([
                    [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                    [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                    [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
                ])
                o = np.array([ix, iy, iz], dtype=np.float64) * spacing + rng.uniform(-jitter, jitter, 3)
                mol = _WATER_ANG @ R.T + o
                xyz.append(mol)
                zs += [8, 1, 1]
    return np.array(zs), np.concatenate(xyz, axis=0)


def _random_atoms(rng: np.random.Generator, n: int, box=12.0, dmin=1.3, z=6):
    pts = []
    while len(pts) < n:
        c = rng.uniform(0.0, box, 3)
        if all(np.linalg.norm(c - p) >= dmin for p in pts):
            pts.append(c)
    return np.full(n, z), np.array(pts)


def make_basis(rng: np.random.Generator, zs: np.ndarray, xyz_bohr: np.ndarray, shells_by_z: dict, exp_range) -> Basis:
    """Per ELEMENT (all O alike, like a real basis set): for each shell draw nprim exponents
    10^U(log10 lo, log10 hi), sort descending; raw coefficients U(0.2, 1); normalise (R5)."""
    lo, hi = exp_range
    per_elem = {}
    for z in sorted(shells_by_z):           # fixed draw order: ascending Z
        sh = []
        for (l, nprim) in shells_by_z[z]:
            e = np.sort(10.0 ** rng.uniform(math.log10(lo), math.log10(hi), nprim))[::-1].copy()
            raw = rng.uniform(0.2, 1.0, nprim)
            sh.append((l, e, normalise_shell(l, e, raw)))
        per_elem[z] = sh
    s_atom, s_l, s_np, pe, pc = [], [], [], [], []
    for ia, z in enumerate(zs):
        for (l, e, c) in per_elem[int(z)]:
            s_atom.append(ia); s_l.append(l); s_np.append(len(e)); pe.append(e); pc.append(c)
    return Basis(
        atom_xyz=np.ascontiguousarray(xyz_bohr, dtype=np.float64),
        shell_atom=np.array(s_atom, dtype=np.int32), shell_l=np.array(s_l, dtype=np.int32),
        shell_nprim=np.array(s_np, dtype=np.int32),
        prim_exp=np.concatenate(pe).astype(np.float64), prim_coef=np.concatenate(pc).astype(np.float64),
    )


def becke_grid(xyz_bohr: np.ndarray, n_r: int, n_theta: int, n_phi: int, *, partner_cut_ang: float = 10.0,
               w_min: float = 1e-15, device: str = "cpu", chunk_bytes: int = 1 << 28, parents=None):
    """Product atomic grids + Becke partition (stands in for the
    paper's MK x Lebedev / SSF grid).

    radial: Gauss-Chebyshev 2nd kind x_i = cos(i pi/(n_r+1)), r = R(1+x)/(1-x), R = 1 bohr,
            w_r = pi/(n_r+1) sin^2(i pi/(n_r+1)) / sqrt(1-x^2) * 2R/(1-x)^2 * r^2
            (written as  pi/(n_r+1) * sin(.) * 2R/(1-x)^2 * r^2, since sqrt(1-x^2) = sin(.))
    angular: n_theta Gauss-Legendre nodes in cos(theta) x n_phi uniform phi, weight w_th * 2 pi / n_phi
    Becke: w <- w * p_A / sum_B p_B, p_A = prod_{B != A} s(mu_AB), s = (1 - f(f(f(mu))))/2,
           f = 1.5 mu - 0.5 mu^3; partners restricted to atoms within ``partner_cut_ang`` Å of the parent.
    Points with weight < w_min are dropped.  Order: atom, radial, theta, phi (phi fastest).
    ``parents``: generate only the atomic grids of these atoms (their points and weights are exactly those of the full
    molecular grid, the partition still sees every partner); tests use it to cut a piece out of a large config.
    Returns (points [n,3], weights [n]) as numpy float64.
    """
    import torch
    dev = torch.device(device)
    f64 = torch.float64
    xyz = torch.as_tensor(np.asarray(xyz_bohr), dtype=f64, device=dev)
    nat = xyz.shape[0]
    i = torch.arange(1, n_r + 1, dtype=f64, device=dev)
    ang = i * math.pi / (n_r + 1)
    x = torch.cos(ang)
    r = (1.0 + x) / (1.0 - x)
    w_r = math.pi / (n_r + 1) * torch.sin(ang) * 2.0 / (1.0 - x) ** 2 * r * r
    ct_np, wt_np = np.polynomial.legendre.leggauss(n_theta)
    ct = torch.as_tensor(ct_np, dtype=f64, device=dev)
    wt = torch.as_tensor(wt_np, dtype=f64, device=dev)
    st = torch.sqrt(1.0 - ct * ct)
    phi = torch.arange(n_phi, dtype=f64, device=dev) * (2.0 * math.pi / n_phi)
    # unit sphere points [n_theta, n_phi, 3]
    u = torch.stack([st[:, None] * torch.cos(phi)[None, :], st[:, None] * torch.sin(phi)[None, :],
                     ct[:, None].expand(n_theta, n_phi)], dim=-1)
    w_ang = (wt[:, None] * (2.0 * math.pi / n_phi)).expand(n_theta, n_phi)
    local = (r[:, None, None, None] * u[None]).reshape(-1, 3)           # [n_r*n_th*n_ph, 3]
    w_local = (w_r[:, None, None] * w_ang[None]).reshape(-1)
    npa = local.shape[0]

    dist_aa = torch.cdist(xyz, xyz)
    cut = partner_cut_ang * BOHR_PER_ANGSTROM
    pts_out, w_out = [], []
    for A in (range(nat) if parents is None else [int(a) for a in parents]):
        nb = torch.nonzero(dist_aa[A] <= cut).reshape(-1)              # includes A itself
        nn = int(nb.numel())
        pts = local + xyz[A]
        if nn == 1:
            pts_out.append(pts); w_out.append(w_local.clone())
            continue
        cxyz = xyz[nb]
        Rbc = dist_aa[nb][:, nb]
        Rbc = Rbc + torch.eye(nn, dtype=f64, device=dev)                # avoid 0/0 on the diagonal
        eye = torch.eye(nn, dtype=torch.bool, device=dev)
        ia = int(torch.nonzero(nb == A).reshape(-1)[0])
        chunk = max(1, int(chunk_bytes // (8 * nn * nn * 4)))
        wA = torch.empty(npa, dtype=f64, device=dev)
        for s in range(0, npa, chunk):
            p = pts[s:s + chunk]
            d = torch.cdist(p, cxyz)                                    # [c, nn]
            mu = (d[:, :, None] - d[:, None, :]) / Rbc[None]            # mu_BC = (r_B - r_C)/R_BC
            for _ in range(3):
                mu = 1.5 * mu - 0.5 * mu * mu * mu
            sfun = 0.5 * (1.0 - mu)
            sfun = torch.where(eye[None], torch.ones((), dtype=f64, device=dev), sfun)
            pB = torch.prod(sfun, dim=2)                                # [c, nn]
            wA[s:s + chunk] = pB[:, ia] / pB.sum(dim=1)
        pts_out.append(pts); w_out.append(w_local * wA)
    pts = torch.cat(pts_out, dim=0)
    w = torch.cat(w_out, dim=0)
    keep = w >= w_min
    return pts[keep].cpu().numpy().copy(), w[keep].cpu().numpy().copy()


def density_from_C(rng: np.random.Generator, nbf: int, nocc: int, sigma: float) -> np.ndarray:
    C = rng.standard_normal((nbf, nocc)) * sigma
    P = C @ C.T
    return 0.5 * (P + P.T)


def density_localised(rng: np.random.Generator, basis: Basis, nocc: int, decay_bohr: float, sigma: float = 1.0) -> np.ndarray:
    """Spatially decaying density: P = C C^T, every column of C a random orbital localised around
    one atom, C[mu, i] = N(0, sigma^2) * exp(-|R_mu - R_c(i)| / decay_bohr) with c(i) cycling through the atoms.  Symmetric,
    positive semi-definite, and |P[mu, nu]| falls off like exp(-|R_mu - R_nu| / decay_bohr) by the triangle inequality: the
    shape of the density of an insulator, for which Eq. 46 localises and sn-LinK deletes work."""
    fo = basis.shell_offset
    cen = np.repeat(basis.atom_xyz[basis.shell_atom], np.diff(fo), axis=0)             # centre of every basis function
    natoms = basis.atom_xyz.shape[0]
    home = basis.atom_xyz[np.arange(nocc) % natoms]                                    # centre of every column
    g = rng.standard_normal((basis.nbf, nocc)) * sigma
    d = np.linalg.norm(cen[:, None, :] - home[None, :, :], axis=2)
    C = g * np.exp(-d / decay_bohr)
    P = C @ C.T
    return 0.5 * (P + P.T)


def make_workload(cfg: int, *, grid=None, device: str = "cpu", lattice=None, natoms=None, grid_atoms=None,
                  density: str = "dense", decay_bohr: float = 1.5) -> Workload:
    """BASELINE.json config ``cfg`` (1..5).  ``grid=(n_r,n_theta,n_phi)`` overrides the grid level
    (reduced levels are what the CPU-sized parity tests use); ``lattice`` / ``natoms`` shrink
    the molecule (tests only); ``grid_atoms`` keeps the whole molecule, basis and P but only the atomic grids of the
    listed atoms (tests only); ``density="decay"`` swaps the dense random density for a spatially decaying one
    (density_localised).  Everything else (seed, draw order) is fixed."""
    c = CONFIGS[cfg]
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + cfg))
    # draw order: geometry -> basis -> C
    if cfg == 1:
        zs, xyz_ang = np.array([8, 1, 1]), _WATER_ANG.copy()
    elif cfg in (2, 3, 4):
        zs, xyz_ang = _water_cluster(rng, lattice or c["lattice"])
    else:
        zs, xyz_ang = _random_atoms(rng, natoms or 32)
    xyz = xyz_ang * BOHR_PER_ANGSTROM
    basis = make_basis(rng, zs, xyz, c["shells"], c["exp_range"])
    nbf = basis.nbf
    nocc = c["nocc"]
    if lattice or natoms:   # shrunk molecule: keep the occupied fraction
        full_atoms = {2: 24, 3: 192, 4: 1029, 5: 32}[cfg]
        nocc = max(1, int(round(nocc * len(zs) / full_atoms)))
    sigma = c["sigma"] if c["sigma"] is not None else 1.0 / math.sqrt(nocc)
    if density == "dense":            # BASELINE.json: P = C C^T, C i.i.d. Gaussian (no spatial decay)
        P = density_from_C(rng, nbf, nocc, sigma)
    elif density == "decay":          # section 8(f)-2: localised orbitals, exponentially decaying P
        P = density_localised(rng, basis, nocc, decay_bohr)
    else:
        raise ValueError("density must be 'dense' or 'decay'")
    g = grid or c["grid"]
    pts, w = becke_grid(xyz, *g, device=device, parents=grid_atoms)
    return Workload(name=c["name"], cfg=cfg, basis=basis, points=pts, weights=w, P=P, eps=c["eps"],
                    grid_shape=tuple(g), atoms_z=tuple(int(z) for z in zs))


def custom_workload(name: str, zs, xyz_ang, shells_by_z, *, seed: int, exp_range=(0.1, 100.0), grid=(12, 6, 12),
                    nocc=2, sigma=0.5, eps=0.0, device="cpu") -> Workload:
    """Small ad-hoc system with the same recipe (tests, pins)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    xyz = np.asarray(xyz_ang, dtype=np.float64) * BOHR_PER_ANGSTROM
    basis = make_basis(rng, np.asarray(zs), xyz, shells_by_z, exp_range)
    P = density_from_C(rng, basis.nbf, nocc, sigma)
    pts, w = becke_grid(xyz, *grid, device=device)
    return Workload(name=name, cfg=0, basis=basis, points=pts, weights=w, P=P, eps=eps, grid_shape=tuple(grid),
                    atoms_z=tuple(int(z) for z in zs))
