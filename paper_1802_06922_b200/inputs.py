"""Seeded synthetic inputs for the five BASELINE.json configs (and ad-hoc test shapes).

This module holds NONE of the method's arithmetic (no spline weights, no determinants): it
only draws random numbers and fills the coefficient table.  Both the oracle-side tests and
the CUDA-side tests/bench take their inputs from here, so the two see identical bits.

Recipe.  The paper measures on NiO-32 / NiO-128
B-spline orbital sets that are not available; these inputs stand in for
them with the same shapes: an fp32 table [nx][ny][nz][norb], smooth orbitals (a sum of 8
random plane waves each, |c| <= 1), electron positions uniform in the cell, isotropic
Gaussian displacements, uniforms in [0,1).

Generator: numpy.random.Generator(Philox(180206922 + config index)); draw order fixed:
plane-wave parameters (n, a, theta) or raw coefficients -> positions -> delta -> uniforms.
The table itself is filled with torch ops in fp64 on `device` and rounded once to fp32; a
table generated on the CPU and one generated on a GPU may differ in a few last bits, so a
test generates the table ONCE and hands the same bits to both sides.
"""
from dataclasses import dataclass, field
import math

import numpy as np
import torch

BASE_SEED = 180206922


@dataclass
class QmcConfig:
    name: str
    index: int
    grid: tuple            # (nx, ny, nz)
    norb: int              # = electrons per determinant
    lattice: tuple         # diagonal (Lx, Ly, Lz) in bohr, or a 3x3 nested tuple
    nw: int                # walkers
    nsweeps: int
    sigma: float           # std-dev of each displacement component (bohr)
    coef_kind: str         # "uniform" | "planewave"
    kmax: tuple = (0, 0, 0)  # plane-wave integer range per dimension
    nterms: int = 8

    def lattice_matrix(self):
        lat = np.asarray(self.lattice, dtype=np.float64)
        return np.diag(lat) if lat.ndim == 1 else lat.reshape(3, 3)

    def table_bytes(self):
        nx, ny, nz = self.grid
        return nx * ny * nz * self.norb * 4


# The five BASELINE.json configs.  sigma: R:A13 (tiny 0.05 L; others 0.8 x grid spacing 0.2).
CONFIGS = {
    "tiny": QmcConfig("tiny", 0, (16, 16, 16), 8, (1.0, 1.0, 1.0), 4, 1, 0.05, "uniform"),
    "small": QmcConfig("small", 1, (48, 48, 48), 128, (9.6, 10.8, 12.0), 256, 4, 0.16,
                       "planewave", (4, 4, 4)),
    "mid": QmcConfig("mid", 2, (96, 96, 96), 512, (19.2, 19.2, 19.2), 512, 2, 0.16,
                     "planewave", (6, 6, 6)),
    "large": QmcConfig("large", 3, (128, 128, 128), 1024, (25.6, 25.6, 25.6), 512, 1, 0.16,
                       "planewave", (8, 8, 8)),
    "xlarge": QmcConfig("xlarge", 4, (128, 128, 160), 2048, (25.6, 25.6, 32.0), 128, 1, 0.16,
                        "planewave", (8, 8, 10)),
}


@dataclass
class QmcInputs:
    cfg: QmcConfig
    lattice: np.ndarray          # [3][3] float64, rows = cell vectors
    coefs: torch.Tensor          # float32 [nx][ny][nz][norb] on `device`
    pos: np.ndarray              # float64 [nw][nel][3]
    delta: np.ndarray            # float64 [nsweeps][nel][nw][3]
    unif: np.ndarray             # float64 [nsweeps][nel][nw]
    pw: dict = field(default_factory=dict)   # plane-wave parameters (n, a, theta), if any

    def coefs_numpy(self):
        return self.coefs.detach().cpu().numpy()


def custom_config(name, grid, norb, lattice, nw, nsweeps=1, sigma=None, coef_kind="planewave",
                  kmax=None, index=100):
    """An ad-hoc shape for tests (ragged N, skewed cell, ...)."""
    lat = np.asarray(lattice, dtype=np.float64)
    if sigma is None:
        lens = lat if lat.ndim == 1 else np.linalg.norm(lat.reshape(3, 3), axis=1)
        sigma = 0.8 * float(np.min(lens / np.asarray(grid)))
    if kmax is None:
        # pool of (2k+1)^3 plane waves must exceed norb, or the Slater matrix is singular (R:A17)
        kmax = tuple(max(1, min(g // 3, 8)) for g in grid)
    lat_t = tuple(map(float, lat)) if lat.ndim == 1 else tuple(map(tuple, lat.reshape(3, 3).tolist()))
    return QmcConfig(name, index, tuple(grid), int(norb), lat_t, int(nw), int(nsweeps),
                     float(sigma), coef_kind, tuple(kmax))


def planewave_table(grid, n, a, theta, device="cpu", xchunk=None):
    """c[ix][iy][iz][j] = sum_m a[j][m] cos(2 pi (n_jm . (ix/nx, iy/ny, iz/nz)) + theta[j][m]),
    evaluated in fp64 (angle-addition form, exact integer phase reduction) -> fp32."""
    nx, ny, nz = grid
    norb, nterms = a.shape
    dev = torch.device(device)
    n_t = torch.as_tensor(n, dtype=torch.int64, device=dev)          # [norb][m][3]
    a_t = torch.as_tensor(a, dtype=torch.float64, device=dev)        # [norb][m]
    th_t = torch.as_tensor(theta, dtype=torch.float64, device=dev)   # [norb][m]
    two_pi = 2.0 * math.pi

    def frac(idx_count, nvec):                                       # [count][norb][m] in [0,1)
        i = torch.arange(idx_count, dtype=torch.int64, device=dev).view(-1, 1, 1)
        return torch.remainder(i * nvec.unsqueeze(0), idx_count).to(torch.float64) / idx_count

    fx, fy, fz = frac(nx, n_t[..., 0]), frac(ny, n_t[..., 1]), frac(nz, n_t[..., 2])
    bz = two_pi * fz + th_t.unsqueeze(0)                             # [nz][norb][m]
    # Q[j][2m][z]
    q = torch.cat([torch.cos(bz), -torch.sin(bz)], dim=2).permute(1, 2, 0).contiguous()
    out = torch.empty((nx, ny, nz, norb), dtype=torch.float32, device=dev)
    if xchunk is None:
        budget = 2 ** 27 if dev.type == "cpu" else 2 ** 28             # fp64 elements per chunk
        xchunk = max(1, min(nx, budget // max(1, ny * nz * norb)))
    for x0 in range(0, nx, xchunk):
        x1 = min(nx, x0 + xchunk)
        ang = two_pi * (fx[x0:x1].unsqueeze(1) + fy.unsqueeze(0))    # [xc][ny][norb][m]
        p = torch.cat([a_t * torch.cos(ang), a_t * torch.sin(ang)], dim=3)  # [xc][ny][norb][2m]
        p = p.permute(2, 0, 1, 3).reshape(norb, (x1 - x0) * ny, 2 * nterms)
        c = torch.bmm(p, q)                                          # [norb][xc*ny][nz]
        out[x0:x1] = c.permute(1, 2, 0).reshape(x1 - x0, ny, nz, norb).to(torch.float32)
        del ang, p, c
    return out


def make_inputs(cfg, device="cpu", nw=None, nsweeps=None, with_table=True):
    """Draw the inputs of `cfg` (a QmcConfig or one of the CONFIGS names).

    nw / nsweeps override the config's counts (the draw order keeps coefficients identical;
    positions, delta and uniforms are drawn for the overridden counts).
    """
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    nw = cfg.nw if nw is None else int(nw)
    nsweeps = cfg.nsweeps if nsweeps is None else int(nsweeps)
    rng = np.random.Generator(np.random.Philox(BASE_SEED + cfg.index))
    nx, ny, nz = cfg.grid
    nel = cfg.norb
    lat = cfg.lattice_matrix()
    pw = {}
    if cfg.coef_kind == "uniform":
        raw = rng.uniform(-1.0, 1.0, size=(nx, ny, nz, nel)).astype(np.float32)
        coefs = torch.from_numpy(raw).to(device) if with_table else None
    elif cfg.coef_kind == "planewave":
        kx, ky, kz = cfg.kmax
        n = np.stack([rng.integers(-kx, kx + 1, size=(nel, cfg.nterms)),
                      rng.integers(-ky, ky + 1, size=(nel, cfg.nterms)),
                      rng.integers(-kz, kz + 1, size=(nel, cfg.nterms))], axis=-1)
        a = rng.uniform(-1.0, 1.0, size=(nel, cfg.nterms)) / cfg.nterms
        theta = rng.uniform(0.0, 2.0 * math.pi, size=(nel, cfg.nterms))
        pw = dict(n=n, a=a, theta=theta)
        coefs = planewave_table(cfg.grid, n, a, theta, device=device) if with_table else None
    else:
        raise ValueError(cfg.coef_kind)
    u = rng.uniform(0.0, 1.0, size=(nw, nel, 3))
    pos = u @ lat
    delta = rng.normal(0.0, cfg.sigma, size=(nsweeps, nel, nw, 3))
    unif = rng.uniform(0.0, 1.0, size=(nsweeps, nel, nw))
    return QmcInputs(cfg, lat, coefs, np.ascontiguousarray(pos), np.ascontiguousarray(delta),
                     np.ascontiguousarray(unif), pw)


@dataclass
class JastrowInputs:
    funcs: list                  # [(r_c, control points p[0..M]), ...]: e-e same spin, e-e opposite spin, species 0, 1
    f_same: int
    f_opp: int
    ions: np.ndarray             # float64 [nion][3]
    ion_func: np.ndarray         # int32 [nion]: function of each ion's species
    other: np.ndarray            # float64 [nw][nother][3]: electrons of the other spin (fixed during a sweep)


def make_jastrow(cfg, lattice, nother=0, nion=None, nw=None, seed_offset=5000):
    """Seeded parameters of a one- and two-body B-spline Jastrow factor (eq. 30-33) shaped like the
    paper's solid-state workloads: cutoffs below the Wigner-Seitz radius of the cell (L375), 8-10 control
    points per function, two ionic species, nion = max(2, N / 6) ions uniform in the cell (NiO-128 has
    1536 valence electrons on 128 atoms; per spin determinant that is 6 electrons per atom).  Control
    points: a smooth decaying profile amp (1 - m / M)^2 with 20 % seeded noise and p_M = 0 (u continuous
    at the cutoff).  Draws only: none of the method's arithmetic lives here."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    rng = np.random.Generator(np.random.Philox(BASE_SEED + seed_offset + cfg.index))
    lat = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
    # inscribed-sphere radius of the Wigner-Seitz cell is at least half the smallest cell height
    vol = abs(np.linalg.det(lat))
    heights = [vol / np.linalg.norm(np.cross(lat[(d + 1) % 3], lat[(d + 2) % 3])) for d in range(3)]
    rws = 0.5 * min(heights)
    funcs = []
    for amp, frac, M in ((0.25, 0.95, 10), (0.5, 0.95, 10), (-0.6, 0.8, 8), (-0.9, 0.7, 8)):
        m = np.arange(M + 1, dtype=np.float64)
        p = amp * (1.0 - m / M) ** 2 * (1.0 + 0.2 * rng.uniform(-1.0, 1.0, M + 1))
        p[M] = 0.0
        funcs.append((float(frac * rws), p))
    nw = cfg.nw if nw is None else int(nw)
    nion = max(2, cfg.norb // 6) if nion is None else int(nion)
    ions = rng.uniform(0.0, 1.0, size=(nion, 3)) @ lat
    ion_func = (2 + (np.arange(nion) % 2)).astype(np.int32)
    other = rng.uniform(0.0, 1.0, size=(nw, nother, 3)) @ lat
    return JastrowInputs(funcs, 0, 1, np.ascontiguousarray(ions), ion_func, np.ascontiguousarray(other))
