"""Input generators for the five BASELINE.json configs.

Data only.  Every random array comes from ``numpy.random.default_rng([SEED, config, stream])``
in float64.  Array index order is ``U[field, patch, k, j, i]`` with ``i`` (x) fastest; the field
order is rho, m_x, m_y, m_z, E [, B_x, B_y, B_z, psi] (reading A20).  Units with mu_0 = 1.
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence

import numpy as np

SEED = 14120934
FIELDS_HYDRO = ("rho", "mx", "my", "mz", "E")
FIELDS_MHD = FIELDS_HYDRO + ("Bx", "By", "Bz", "psi")

BC_PERIODIC = 0
BC_OUTFLOW = 1

LIM_NONE, LIM_MINMOD, LIM_MC = 0, 1, 2
RS_HLL, RS_HLLC, RS_HLLD = 0, 1, 2


@dataclasses.dataclass
class Level:
    """One refinement level = one batch of equal-size cubic patches (interiors only)."""

    n: int                      # interior cells per side
    g: int                      # ghost layers carried by the API (3)
    level: int
    dx: float
    origin: np.ndarray          # int32 [npatch, 3] lower corner (x, y, z) in level-cell units
    domain_cells: tuple         # extent of this level's index space (x, y, z)
    bc: tuple                   # 6 entries: xlo, xhi, ylo, yhi, zlo, zhi
    self_periodic: bool
    U: np.ndarray               # float64 [nfields, npatch, n, n, n]

    @property
    def npatch(self) -> int:
        return int(self.U.shape[1])

    @property
    def nfields(self) -> int:
        return int(self.U.shape[0])

    @property
    def ncells(self) -> int:
        return self.npatch * self.n ** 3


@dataclasses.dataclass
class Workload:
    name: str
    levels: List[Level]
    gamma: float
    mhd: bool
    limiter: int
    riemann: int
    cfl: float
    nsteps: int
    alpha: float = 0.4
    note: str = ""


# --------------------------------------------------------------------------------------
# geometry helpers
# --------------------------------------------------------------------------------------

def _part1by2(v: np.ndarray) -> np.ndarray:
    """Spread the low 10 bits of v so that there are two zero bits between each."""
    v = v.astype(np.uint64) & np.uint64(0x3FF)
    v = (v | (v << np.uint64(16))) & np.uint64(0x30000FF)
    v = (v | (v << np.uint64(8))) & np.uint64(0x300F00F)
    v = (v | (v << np.uint64(4))) & np.uint64(0x30C30C3)
    v = (v | (v << np.uint64(2))) & np.uint64(0x9249249)
    return v


def morton_key(px, py, pz) -> np.ndarray:
    px, py, pz = (np.asarray(a) for a in (px, py, pz))
    return _part1by2(px) | (_part1by2(py) << np.uint64(1)) | (_part1by2(pz) << np.uint64(2))


def morton_patch_origins(npx: int, npy: int, npz: int, n: int) -> np.ndarray:
    """Origins (cell units) of an npx*npy*npz tiling by n^3 patches, ordered along a Morton
    (Z-order) curve -- the paper's own first step (space-filling-curve order)."""
    pz, py, px = np.meshgrid(np.arange(npz), np.arange(npy), np.arange(npx), indexing="ij")
    px, py, pz = px.ravel(), py.ravel(), pz.ravel()
    order = np.argsort(morton_key(px, py, pz), kind="stable")
    return (np.stack([px[order], py[order], pz[order]], axis=1) * n).astype(np.int32)


def split_into_patches(G: np.ndarray, n: int, origin: np.ndarray) -> np.ndarray:
    """G[nf, Nz, Ny, Nx] -> U[nf, npatch, n, n, n] for the given patch origins."""
    nf = G.shape[0]
    out = np.empty((nf, origin.shape[0], n, n, n), dtype=G.dtype)
    for p, (ox, oy, oz) in enumerate(origin):
        out[:, p] = G[:, oz:oz + n, oy:oy + n, ox:ox + n]
    return out


def join_patches(U: np.ndarray, origin: np.ndarray, shape: Sequence[int]) -> np.ndarray:
    """Inverse of split_into_patches; shape = (Nz, Ny, Nx)."""
    nf, _, n = U.shape[0], U.shape[1], U.shape[2]
    G = np.zeros((nf,) + tuple(shape), dtype=U.dtype)
    for p, (ox, oy, oz) in enumerate(origin):
        G[:, oz:oz + n, oy:oy + n, ox:ox + n] = U[:, p]
    return G


def add_ghost_frame(U: np.ndarray, g: int, fill: float = np.nan) -> np.ndarray:
    """[nf, np, n, n, n] -> [nf, np, n+2g, n+2g, n+2g]; ghost cells set to `fill`."""
    nf, npch, n = U.shape[0], U.shape[1], U.shape[2]
    m = n + 2 * g
    out = np.full((nf, npch, m, m, m), fill, dtype=U.dtype)
    out[:, :, g:g + n, g:g + n, g:g + n] = U
    return out


def strip_ghost_frame(Ug: np.ndarray, g: int) -> np.ndarray:
    m = Ug.shape[2]
    return np.ascontiguousarray(Ug[:, :, g:m - g, g:m - g, g:m - g])


def primitive_to_conserved(rho, v, p, gamma: float, B=None) -> np.ndarray:
    """Initial data are specified in primitive variables; this applies the ideal-gas energy
    definition E = p/(gamma-1) + rho|v|^2/2 [+ |B|^2/2] (SURVEY.md §8(c) Notation) to form the
    conserved input arrays.  psi = 0 initially (A8)."""
    rho = np.asarray(rho, dtype=np.float64)
    fields = [rho, rho * v[0], rho * v[1], rho * v[2]]
    E = np.asarray(p, dtype=np.float64) / (gamma - 1.0) + 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
    if B is not None:
        E = E + 0.5 * (B[0] ** 2 + B[1] ** 2 + B[2] ** 2)
    fields.append(E)
    if B is not None:
        fields += [np.asarray(B[0], dtype=np.float64) + 0.0 * rho,
                   np.asarray(B[1], dtype=np.float64) + 0.0 * rho,
                   np.asarray(B[2], dtype=np.float64) + 0.0 * rho,
                   np.zeros_like(rho)]
    return np.stack([np.broadcast_to(f, rho.shape) for f in fields]).astype(np.float64)


# --------------------------------------------------------------------------------------
# Gaussian random fields (reading A21)
# --------------------------------------------------------------------------------------

def _kgrid(N: int):
    kx = np.fft.rfftfreq(N) * N
    kf = np.fft.fftfreq(N) * N
    KZ, KY, KX = np.meshgrid(kf, kf, kx, indexing="ij")
    return KX, KY, KZ


def _amplitude(N: int, index: float):
    KX, KY, KZ = _kgrid(N)
    k = np.sqrt(KX ** 2 + KY ** 2 + KZ ** 2)
    amp = np.zeros_like(k)
    keep = (k > 0) & (k <= N / 2)
    amp[keep] = k[keep] ** (index / 2.0)
    return amp, (KX, KY, KZ), k


def _fft():
    import scipy.fft as sfft
    return sfft


def gaussian_random_field(N: int, index: float, rng: np.random.Generator) -> np.ndarray:
    """White noise -> rfftn -> * k^(index/2) (k=0 and k>N/2 zeroed) -> irfftn -> zero mean,
    unit variance.  `index` is the 3-D power-per-mode spectral index n in P(k) ~ k^n."""
    sfft = _fft()
    w = rng.standard_normal((N, N, N))
    amp, _, _ = _amplitude(N, index)
    wh = sfft.rfftn(w, workers=-1)
    del w
    wh *= amp
    f = sfft.irfftn(wh, s=(N, N, N), workers=-1)
    del wh
    f -= f.mean()
    f /= f.std()
    return f


def solenoidal_random_field(N: int, index: float, rng: np.random.Generator) -> np.ndarray:
    """Three filtered white-noise fields, projected B^ <- B^ - k (k.B^)/k^2, inverse
    transformed, mean removed, scaled so that <B.B> = 1.  Returns [3, N, N, N] (x, y, z)."""
    sfft = _fft()
    amp, (KX, KY, KZ), k = _amplitude(N, index)
    k2 = np.where(k > 0, k * k, 1.0)
    hats = []
    for _ in range(3):
        w = rng.standard_normal((N, N, N))
        h = sfft.rfftn(w, workers=-1)
        h *= amp
        hats.append(h)
        del w
    kdotb = (KX * hats[0] + KY * hats[1] + KZ * hats[2]) / k2
    hats[0] -= KX * kdotb
    hats[1] -= KY * kdotb
    hats[2] -= KZ * kdotb
    del kdotb
    out = np.empty((3, N, N, N))
    for c in range(3):
        out[c] = sfft.irfftn(hats[c], s=(N, N, N), workers=-1)
        out[c] -= out[c].mean()
    hats.clear()
    out /= np.sqrt(np.mean(out[0] ** 2 + out[1] ** 2 + out[2] ** 2))
    return out


def _rng(config: int, stream: int) -> np.random.Generator:
    return np.random.default_rng([SEED, config, stream])


# --------------------------------------------------------------------------------------
# the five configs
# --------------------------------------------------------------------------------------

def config1_sod(n: int = 32, axis: int = 0) -> Workload:
    """Config 1: Sod tube along `axis` on ONE n^3 patch, g=3, outflow, gamma=1.4, domain [0,1]^3.
    Left (cells 0..n/2-1): rho=1, p=1; right: rho=0.125, p=0.1; v=0.  The discontinuity sits on
    the cell face x=0.5."""
    gamma = 1.4
    idx = np.arange(n)
    shape = [1, 1, 1]
    shape[2 - axis] = n                      # array order is (k, j, i) = (z, y, x)
    left = (idx < n // 2).reshape(shape)
    rho = np.broadcast_to(np.where(left, 1.0, 0.125), (n, n, n)).copy()
    p = np.broadcast_to(np.where(left, 1.0, 0.1), (n, n, n)).copy()
    zero = np.zeros((n, n, n))
    U = primitive_to_conserved(rho, (zero, zero, zero), p, gamma)[:, None]
    lev = Level(n=n, g=3, level=0, dx=1.0 / n, origin=np.zeros((1, 3), np.int32),
                domain_cells=(n, n, n), bc=(BC_OUTFLOW,) * 6, self_periodic=False,
                U=np.ascontiguousarray(U))
    return Workload("config1_sod", [lev], gamma, False, LIM_MINMOD, RS_HLLC, 0.4, 20)


def config2_random_patches(npatch: int = 512, n: int = 16) -> Workload:
    """Config 2: `npatch` independent self-periodic hydro patches.  Per patch p (stream = p):
    rho = exp(0.5 g0) / patch mean; v_d = (c_s/sqrt3) g_d with c_s = sqrt(gamma); p = 1."""
    gamma = 5.0 / 3.0
    cs = np.sqrt(gamma * 1.0 / 1.0)
    U = np.empty((5, npatch, n, n, n))
    for p in range(npatch):
        rng = _rng(2, p)
        g = rng.standard_normal((4, n, n, n))
        rho = np.exp(0.5 * g[0])
        rho /= rho.mean()
        v = (cs / np.sqrt(3.0)) * g[1:4]
        U[:, p] = primitive_to_conserved(rho, v, np.ones_like(rho), gamma)
    origin = np.zeros((npatch, 3), np.int32)
    lev = Level(n=n, g=3, level=0, dx=1.0 / n, origin=origin, domain_cells=(n, n, n),
                bc=(BC_PERIODIC,) * 6, self_periodic=True, U=U)
    return Workload("config2_random_patches", [lev], gamma, False, LIM_MC, RS_HLLC, 0.4, 1)


def orszag_tang_state(N: int, eps: float = 0.2) -> np.ndarray:
    """Reading A16: 3-D (z-modulated) Orszag-Tang vortex at cell centres of an N^3 grid on
    [0,1]^3.  Returns conserved G[9, N, N, N]."""
    gamma = 5.0 / 3.0
    c = (np.arange(N) + 0.5) / N
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    rho = np.full((N, N, N), 25.0 / (36.0 * np.pi))
    p = np.full((N, N, N), 5.0 / (12.0 * np.pi))
    B0 = 1.0 / np.sqrt(4.0 * np.pi)
    mod = 1.0 + eps * np.sin(2 * np.pi * Z)
    vx = -mod * np.sin(2 * np.pi * Y)
    vy = mod * np.sin(2 * np.pi * X)
    vz = eps * np.sin(2 * np.pi * Z)
    Bx = -B0 * np.sin(2 * np.pi * Y)
    By = B0 * np.sin(4 * np.pi * X)
    Bz = np.zeros_like(Bx)
    return primitive_to_conserved(rho, (vx, vy, vz), p, gamma, B=(Bx, By, Bz))


def uniform_grid_workload(name: str, G: np.ndarray, n: int, gamma: float, mhd: bool, limiter: int,
                          riemann: int, cfl: float, nsteps: int, alpha: float = 0.4,
                          bc=(BC_PERIODIC,) * 6) -> Workload:
    """Tile a global grid G[nf, Nz, Ny, Nx] (domain [0,1] along x) into n^3 patches in Morton order."""
    Nz, Ny, Nx = G.shape[1:]
    origin = morton_patch_origins(Nx // n, Ny // n, Nz // n, n)
    U = split_into_patches(G, n, origin)
    lev = Level(n=n, g=3, level=0, dx=1.0 / Nx, origin=origin, domain_cells=(Nx, Ny, Nz),
                bc=tuple(bc), self_periodic=False, U=U)
    return Workload(name, [lev], gamma, mhd, limiter, riemann, cfl, nsteps, alpha)


def config3_orszag_tang(N: int = 256, n: int = 16, eps: float = 0.2) -> Workload:
    """Config 3: Orszag-Tang on N^3 periodic, (N/n)^3 patches of n^3 in Morton order; MC + HLLD +
    GLM alpha=0.4, cfl 0.3, 5 steps."""
    G = orszag_tang_state(N, eps)
    return uniform_grid_workload("config3_orszag_tang", G, n, 5.0 / 3.0, True, LIM_MC, RS_HLLD,
                                 0.3, 5)


def turbulence_state(N: int, config: int = 5, mach: float = 3.0, beta: float = 100.0,
                     index: float = -11.0 / 3.0) -> np.ndarray:
    """Config-5 state on an N^3 grid: rho=1, p=1, v = GRFs with P(k) ~ k^index scaled to
    sqrt<v.v> = mach*sqrt(gamma); B solenoidal, zero mean, <B.B> = 2p/beta."""
    gamma = 5.0 / 3.0
    cs = np.sqrt(gamma)
    v = np.stack([gaussian_random_field(N, index, _rng(config, s)) for s in range(3)])
    v *= mach * cs / np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    B = solenoidal_random_field(N, index, _rng(config, 3))
    B *= np.sqrt(2.0 * 1.0 / beta)
    one = np.ones((N, N, N))
    return primitive_to_conserved(one, v, one, gamma, B=B)


def config5_turbulence(N: int = 512, n: int = 32) -> Workload:
    """Config 5: N^3 periodic MHD turbulence, (N/n)^3 patches of n^3, Morton order; MC + HLLD +
    GLM, cfl 0.3, 10 steps."""
    G = turbulence_state(N)
    return uniform_grid_workload("config5_turbulence", G, n, 5.0 / 3.0, True, LIM_MC, RS_HLLD,
                                 0.3, 10)


# sigma(ln rho) tuned once (reading A15: start 1.2 flags 4007 blocks; 0.517 flags ~102) so that ~100 of the 4096 aligned 8^3 root blocks are
# flagged; the resulting count is recorded in Workload.note and DESIGN.md.
CONFIG4_SIGMA = 0.517


def config4_two_level(mhd: bool, nfine: int = 256, n: int = 16, sigma: float = CONFIG4_SIGMA,
                      threshold: float = 4.0) -> Workload:
    """Config 4: root (nfine/2)^3 periodic as n^3 patches + level-1 n^3 patches on aligned
    (n/2)^3 root blocks that contain a root cell with rho > threshold*mean (A15)."""
    gamma = 5.0 / 3.0
    N = nfine
    Gln = gaussian_random_field(N, -2.0, _rng(4, 0))
    rho = np.exp(sigma * Gln)
    rho /= rho.mean()
    v = np.stack([gaussian_random_field(N, -2.0, _rng(4, 1 + s)) for s in range(3)])
    v *= 2.0 * np.sqrt(gamma * 1.0 / 1.0) / np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    p = np.ones_like(rho)
    if mhd:
        dB = solenoidal_random_field(N, -2.0, _rng(4, 4)) * 1.0e-4
        B = (dB[0], dB[1], dB[2] + 1.0e-3)
        Gf = primitive_to_conserved(rho, v, p, gamma, B=B)
    else:
        Gf = primitive_to_conserved(rho, v, p, gamma)
    nf = Gf.shape[0]
    Nc = N // 2
    # root = 2x2x2 mean of the conserved variables
    Gc = Gf.reshape(nf, Nc, 2, Nc, 2, Nc, 2).mean(axis=(2, 4, 6))
    # flag aligned (n/2)^3 root blocks
    nb = n // 2
    nblk = Nc // nb
    blkmax = Gc[0].reshape(nblk, nb, nblk, nb, nblk, nb).max(axis=(1, 3, 5))
    bz, by, bx = np.nonzero(blkmax > threshold * Gc[0].mean())
    order = np.argsort(morton_key(bx, by, bz), kind="stable")
    bx, by, bz = bx[order], by[order], bz[order]
    origin1 = (np.stack([bx, by, bz], axis=1) * n).astype(np.int32)      # level-1 cell units
    origin0 = morton_patch_origins(Nc // n, Nc // n, Nc // n, n)
    lev0 = Level(n=n, g=3, level=0, dx=1.0 / Nc, origin=origin0, domain_cells=(Nc, Nc, Nc),
                 bc=(BC_PERIODIC,) * 6, self_periodic=False, U=split_into_patches(Gc, n, origin0))
    lev1 = Level(n=n, g=3, level=1, dx=1.0 / N, origin=origin1, domain_cells=(N, N, N),
                 bc=(BC_PERIODIC,) * 6, self_periodic=False, U=split_into_patches(Gf, n, origin1))
    w = Workload("config4_two_level_" + ("mhd" if mhd else "hydro"), [lev0, lev1], gamma, mhd,
                 LIM_MC, RS_HLLD if mhd else RS_HLLC, 0.3, 1)
    w.note = "sigma=%g refined_blocks=%d extra_cell_fraction=%.4f" % (
        sigma, origin1.shape[0], origin1.shape[0] * n ** 3 / float(Nc ** 3))
    return w


def two_level_outflow(mhd: bool = False, n: int = 16) -> Workload:
    """Two-level test set-up with OUTFLOW faces in x (periodic in y, z) and fine patches ON the x faces:
    a 32^3 root ([0,1]^3, 2x2x2 patches) at rest; left state (rho, p) = (1, 1) for x < 3/8, right state
    (0.5, 0.4) beyond, the jump modulated in y, z only for 1/4 < x < 3/4, so both x faces see a uniform state
    at rest for a whole step.  Fine patches: (0,16,16) on the lower x face, its x-sibling (16,16,16) (holds
    the jump), (48,32,32) on the upper x face.  Used by the pins of the boundary readings of O8 / O9."""
    gamma = 1.4
    N = 64
    c = (np.arange(N) + 0.5) / N
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    left = X < 0.375
    mod = np.where((X > 0.25) & (X < 0.75), 1.0 + 0.2 * np.sin(2 * np.pi * Y) * np.cos(2 * np.pi * Z), 1.0)
    rho = np.where(left, 1.0, 0.5) * mod
    p = np.where(left, 1.0, 0.4) * np.where((X > 0.25) & (X < 0.75), 1.0 + 0.1 * np.cos(2 * np.pi * Y), 1.0)
    v = np.zeros((3, N, N, N))
    if mhd:
        B = (np.full_like(rho, 0.05), np.full_like(rho, 0.1), np.full_like(rho, -0.07))
        Gf = primitive_to_conserved(rho, v, p, gamma, B=B)
    else:
        Gf = primitive_to_conserved(rho, v, p, gamma)
    nf = Gf.shape[0]
    Nc = N // 2
    Gc = Gf.reshape(nf, Nc, 2, Nc, 2, Nc, 2).mean(axis=(2, 4, 6))
    bc = (BC_OUTFLOW, BC_OUTFLOW, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC)
    origin0 = morton_patch_origins(Nc // n, Nc // n, Nc // n, n)
    origin1 = np.array([[0, 16, 16], [16, 16, 16], [48, 32, 32]], np.int32)
    lev0 = Level(n=n, g=3, level=0, dx=1.0 / Nc, origin=origin0, domain_cells=(Nc, Nc, Nc), bc=bc,
                 self_periodic=False, U=split_into_patches(Gc, n, origin0))
    lev1 = Level(n=n, g=3, level=1, dx=1.0 / N, origin=origin1, domain_cells=(N, N, N), bc=bc,
                 self_periodic=False, U=split_into_patches(Gf, n, origin1))
    w = Workload("two_level_outflow_" + ("mhd" if mhd else "hydro"), [lev0, lev1], gamma, mhd,
                 LIM_MC, RS_HLLD if mhd else RS_HLLC, 0.3, 1)
    w.note = "p_left=1 p_right=0.4"
    return w


def _dilate_periodic(m: np.ndarray) -> np.ndarray:
    out = np.zeros_like(m)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                out |= np.roll(m, (dz, dy, dx), axis=(0, 1, 2))
    return out


def _erode_periodic(m: np.ndarray) -> np.ndarray:
    return ~_dilate_periodic(~m)


def select_blocks(flag: np.ndarray, cover_prev: Optional[np.ndarray], grow: bool) -> np.ndarray:
    """Geometry policy of a (re)grid: which flagged (n/2)^3 blocks of level l-1 [bool, (z, y, x) block grid]
    become level-l patches.  cover_prev = the block grid of level l-1's own patches one level down (None: level
    l-1 covers the domain).  A block is allowed only where all 27 blocks around it lie inside level l-1
    (proper nesting); `grow` adds one block around the flagged ones (for a level that will carry a finer one)."""
    if cover_prev is None:
        allowed = np.ones_like(flag)
    else:                                               # a level l-1 patch = 2x2x2 blocks of this grid
        up = np.repeat(np.repeat(np.repeat(cover_prev, 2, axis=0), 2, axis=1), 2, axis=2)
        allowed = _erode_periodic(up)
    flag = flag & allowed
    if grow:
        flag = _dilate_periodic(flag) & allowed
    return flag


def blocks_to_origins(flag: np.ndarray, n: int) -> np.ndarray:
    """Patch origins (level-l cell units, Morton order) of the selected blocks of level l-1."""
    bz, by, bx = np.nonzero(flag)
    order = np.argsort(morton_key(bx, by, bz), kind="stable")
    return (np.stack([bx[order], by[order], bz[order]], axis=1) * n).astype(np.int32)


def origins_to_blocks(origin: np.ndarray, n: int, nblk: int) -> np.ndarray:
    """Inverse of blocks_to_origins: bool block grid [nblk]^3 (z, y, x) of a level's patches."""
    g = np.zeros((nblk, nblk, nblk), bool)
    o = np.asarray(origin) // n
    g[o[:, 2], o[:, 1], o[:, 0]] = True
    return g


def patch_flags_to_block_grid(level: Level, flags: np.ndarray) -> np.ndarray:
    """Per-patch block flags [np, 2, 2, 2] (z, y, x halves) of `level` -> its block grid [2 N / n]^3."""
    nb = level.n // 2
    nblk = level.domain_cells[0] // nb
    g = np.zeros((nblk, nblk, nblk), bool)
    o = np.asarray(level.origin) // nb
    for dz in range(2):
        for dy in range(2):
            for dx in range(2):
                g[o[:, 2] + dz, o[:, 1] + dy, o[:, 0] + dx] = flags[:, dz, dy, dx]
    return g


def nested_hierarchy_from_fine(name: str, Gfine: np.ndarray, nlevels: int, n: int, thresholds: Sequence[float],
                               gamma: float, mhd: bool, limiter: int, riemann: int) -> Workload:
    """an L-level properly nested hierarchy cut from one fine periodic state Gfine
    [nf, N, N, N] (N = the finest level's index space).  Level l's data are the 2x2x2 means of level l+1's
    (so every level is the restriction of the next).  Level 0 covers the domain.  For l >= 1 a patch sits on
    an aligned (n/2)^3 block of level l-1 cells; blocks are flagged where the level l-1 density exceeds
    thresholds[l-1] x mean, grown by one block (for every level that has a finer one above it) and kept
    only where all 27 blocks around them lie inside level l-1's patches (proper nesting: a level-l halo and
    its prolongation stencil never leave level l-1).  Patches in Morton order."""
    nf, N = Gfine.shape[0], Gfine.shape[1]
    fields = [None] * nlevels
    fields[nlevels - 1] = Gfine
    for l in range(nlevels - 2, -1, -1):
        M = fields[l + 1].shape[1] // 2
        fields[l] = fields[l + 1].reshape(nf, M, 2, M, 2, M, 2).mean(axis=(2, 4, 6))
    nb = n // 2
    N0 = fields[0].shape[1]
    origin0 = morton_patch_origins(N0 // n, N0 // n, N0 // n, n)
    levels = [Level(n=n, g=3, level=0, dx=1.0 / N0, origin=origin0, domain_cells=(N0,) * 3, bc=(BC_PERIODIC,) * 6,
                    self_periodic=False, U=split_into_patches(fields[0], n, origin0))]
    cover_prev = None                                   # bool on level l-1's block grid (None: everything)
    for l in range(1, nlevels):
        Np = fields[l - 1].shape[1]                     # cells per side of level l-1
        nblk = Np // nb
        rho = fields[l - 1][0]
        flag = rho.reshape(nblk, nb, nblk, nb, nblk, nb).max(axis=(1, 3, 5)) > thresholds[l - 1] * rho.mean()
        flag = select_blocks(flag, cover_prev, grow=l < nlevels - 1)
        origin = blocks_to_origins(flag, n)
        Nl = fields[l].shape[1]
        levels.append(Level(n=n, g=3, level=l, dx=1.0 / Nl, origin=origin, domain_cells=(Nl,) * 3,
                            bc=(BC_PERIODIC,) * 6, self_periodic=False, U=split_into_patches(fields[l], n, origin)))
        cover_prev = flag
    w = Workload(name, levels, gamma, mhd, limiter, riemann, 0.3, 1)
    w.note = "patches per level: " + ", ".join(str(lv.npatch) for lv in levels)
    return w


def config_hierarchy(mhd: bool, nlevels: int = 3, nfine: int = 128, n: int = 16, sigma: float = CONFIG4_SIGMA,
                     thresholds: Sequence[float] = (2.8, 4.0, 5.0, 6.0), mach: float = 0.5) -> Workload:
    """Config 4's lognormal state (A15) refined over `nlevels` levels (f3); nfine = finest index space.
    The velocity field is scaled to rms `mach` x the sound speed of the mean state (config 4 itself uses 2):
    the finest level takes 2^(L-1) steps per root step, and at Mach 2 the grid-scale velocity differences of
    the k^-2 field at 256^3 drive single cells to negative pressure within four steps (the method has no
    pressure floor), which is not what these cases are for."""
    gamma = 5.0 / 3.0
    N = nfine
    rho = np.exp(sigma * gaussian_random_field(N, -2.0, _rng(4, 0)))
    rho /= rho.mean()
    v = np.stack([gaussian_random_field(N, -2.0, _rng(4, 1 + s)) for s in range(3)])
    v *= mach * np.sqrt(gamma) / np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    p = np.ones_like(rho)
    if mhd:
        dB = solenoidal_random_field(N, -2.0, _rng(4, 4))
        dB *= 0.05 / np.sqrt(np.mean(dB[0] ** 2 + dB[1] ** 2 + dB[2] ** 2))
        Gf = primitive_to_conserved(rho, v, p, gamma, B=(dB[0], dB[1], dB[2] + 0.3))   # beta ~ 20 (config 4: 2e6)
    else:
        Gf = primitive_to_conserved(rho, v, p, gamma)
    return nested_hierarchy_from_fine("hierarchy%d_%s" % (nlevels, "mhd" if mhd else "hydro"), Gf, nlevels, n,
                                      thresholds, gamma, mhd, LIM_MC, RS_HLLD if mhd else RS_HLLC)


# --------------------------------------------------------------------------------------
# smooth test states (pins P10, P12): single self-periodic patch of n^3 on [0,1]^3
# --------------------------------------------------------------------------------------

def smooth_wave_patchset(kind: str, N: int, axis: int = 0, t: float = 0.0, n: int = 8) -> Workload:
    """Plane wave along `axis` on a periodic domain of N cells along the axis and n cells across,
    tiled by n^3 patches; dx = 1/N.
    `density`: rho = 1 + 0.2 sin(2 pi (s - t)), u_axis = 1, p = 1 (exact: translation).
    `alfven`: circularly polarised Alfven wave along `axis` (rho=1, p=0.1, B_par=1,
    B_perp = 0.1 (cos, sin)(2 pi (s - t)), v_perp = -B_perp: travels in +axis at speed 1).
    Evaluated at cell centres at time t, so t>0 gives the exact solution to compare with."""
    gamma = 5.0 / 3.0
    dims = [n, n, n]                          # (Nx, Ny, Nz)
    dims[axis] = N
    c = (np.arange(N) + 0.5) / N
    shape = [1, 1, 1]
    shape[2 - axis] = N
    full = (dims[2], dims[1], dims[0])
    s = np.broadcast_to(c.reshape(shape), full)
    ph = 2.0 * np.pi * (s - t)
    zero = np.zeros(full)
    a, b1, b2 = axis, (axis + 1) % 3, (axis + 2) % 3
    if kind == "density":
        v = [zero, zero, zero]
        v[a] = zero + 1.0
        G = primitive_to_conserved(1.0 + 0.2 * np.sin(ph), v, zero + 1.0, gamma)
        mhd = False
    elif kind == "alfven":
        B = [None, None, None]
        v = [None, None, None]
        B[a] = zero + 1.0
        B[b1] = 0.1 * np.cos(ph)
        B[b2] = 0.1 * np.sin(ph)
        v[a] = zero
        v[b1] = -B[b1]
        v[b2] = -B[b2]
        G = primitive_to_conserved(zero + 1.0, v, zero + 0.1, gamma, B=B)
        mhd = True
    else:
        raise ValueError(kind)
    w = uniform_grid_workload("smooth_" + kind, G, n, gamma, mhd, LIM_MC, RS_HLLD if mhd else RS_HLLC,
                              0.3, 0)
    w.levels[0].dx = 1.0 / N
    return w


# --------------------------------------------------------------------------------------
# device-side generator for the full-size config 5 (512^3): same recipe (A21) evaluated with
# torch.fft on the GPU from a seeded torch.Generator, because 512^3 float64 FFTs on the host
# would dominate the benchmark's run time (SURVEY.md §8(d) allows exactly this).  Data only.
# --------------------------------------------------------------------------------------

def morton_permutation(npx: int, npy: int, npz: int) -> np.ndarray:
    """perm[m] = raster index (pz*npy + py)*npx + px of the m-th patch along the Morton curve."""
    pz, py, px = np.meshgrid(np.arange(npz), np.arange(npy), np.arange(npx), indexing="ij")
    px, py, pz = px.ravel(), py.ravel(), pz.ravel()
    return np.argsort(morton_key(px, py, pz), kind="stable")


def turbulence_patches_torch(N: int, n: int, device, mach: float = 3.0, beta: float = 100.0,
                             index: float = -11.0 / 3.0, config: int = 5):
    """Config-5 state on an N^3 grid, built on `device` in float32: rho=1, p=1, v = Gaussian random
    fields with P(k) ~ k^index scaled to sqrt<v.v> = mach*sqrt(gamma); B = solenoidally projected
    field of the same spectrum, zero mean, <B.B> = 2p/beta; psi = 0.  Returns (U, origin) with U a
    torch float32 tensor [9, npatch, n, n, n] in Morton patch order and origin int32 [npatch, 3]."""
    import torch
    gamma = 5.0 / 3.0
    gen = torch.Generator(device=device)
    gen.manual_seed(SEED * 10 + config)
    kf = torch.fft.fftfreq(N, device=device) * N
    kx = torch.fft.rfftfreq(N, device=device) * N
    KZ, KY, KX = torch.meshgrid(kf, kf, kx, indexing="ij")
    k2 = KX * KX + KY * KY + KZ * KZ
    k = torch.sqrt(k2)
    amp = torch.where((k > 0) & (k <= N / 2), torch.clamp(k, min=1.0) ** (index / 2.0), torch.zeros_like(k))
    del k

    def filtered_hat():
        w = torch.randn((N, N, N), generator=gen, device=device, dtype=torch.float32)
        return torch.fft.rfftn(w) * amp

    v = []
    for _ in range(3):
        f = torch.fft.irfftn(filtered_hat(), s=(N, N, N))
        f -= f.mean()
        f /= f.std()
        v.append(f)
    norm = torch.sqrt((v[0] ** 2 + v[1] ** 2 + v[2] ** 2).mean())
    v = [c * (mach * np.sqrt(gamma) / norm) for c in v]
    hats = [filtered_hat() for _ in range(3)]
    kdotb = (KX * hats[0] + KY * hats[1] + KZ * hats[2]) / torch.clamp(k2, min=1.0)
    hats = [hats[0] - KX * kdotb, hats[1] - KY * kdotb, hats[2] - KZ * kdotb]
    del kdotb
    B = []
    for h in hats:
        f = torch.fft.irfftn(h, s=(N, N, N))
        f -= f.mean()
        B.append(f)
    del hats
    bn = torch.sqrt((B[0] ** 2 + B[1] ** 2 + B[2] ** 2).mean())
    B = [c * (np.sqrt(2.0 / beta) / bn) for c in B]
    rho = torch.ones((N, N, N), device=device, dtype=torch.float32)
    E = 1.0 / (gamma - 1.0) + 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2) + 0.5 * (B[0] ** 2 + B[1] ** 2 + B[2] ** 2)
    fields = [rho, rho * v[0], rho * v[1], rho * v[2], E, B[0], B[1], B[2], torch.zeros_like(rho)]
    npd = N // n
    perm = torch.as_tensor(morton_permutation(npd, npd, npd), device=device)
    out = torch.empty((9, npd ** 3, n, n, n), device=device, dtype=torch.float32)
    for q, f in enumerate(fields):
        t = f.reshape(npd, n, npd, n, npd, n).permute(0, 2, 4, 1, 3, 5).reshape(npd ** 3, n, n, n)
        out[q] = t.index_select(0, perm)
    origin = morton_patch_origins(npd, npd, npd, n)
    return out, origin


def refined_level_cells(bits: int = 8, frac: float = 0.25, nfields: int = 9, dtype=np.float32, stream: int = 0):
    """Input of the patch builder: the leaf cells of one refined level as a
    fully threaded tree would hand them over -- scattered in memory, in no spatial order.  Level index space
    (2^bits)^3.  Octs (2^3 cells, what an AMR tree refines) are flagged where a lognormal density with
    P(k) ~ k^-4 (the recipe of A21 with a steeper index: smooth blobs, as collapsed structures are) exceeds its
    (1 - frac) quantile, so about `frac` of the volume is refined in blobs: compact cubes of every size in
    the interiors, single octs along the rims.
    Returns (xyz int32 [3, ncell] in a seeded scrambled order, fields [nfields, ncell] = seeded normals).
    DATA ONLY: no curve ordering, no grouping happens here."""
    rng = _rng(6, stream)
    N = 1 << bits
    Nc = N // 2
    G = gaussian_random_field(Nc, -4.0, rng)
    thr = np.quantile(G, 1.0 - frac)
    oz, oy, ox = np.nonzero(G > thr)          # arrays are indexed [z, y, x]
    d = np.arange(2)
    cx = (2 * ox[:, None, None, None] + d[None, None, None, :]).repeat(2, axis=1).repeat(2, axis=2)
    cy = (2 * oy[:, None, None, None] + d[None, None, :, None]).repeat(2, axis=1).repeat(2, axis=3)
    cz = (2 * oz[:, None, None, None] + d[None, :, None, None]).repeat(2, axis=2).repeat(2, axis=3)
    xyz = np.stack([cx.ravel(), cy.ravel(), cz.ravel()]).astype(np.int32)
    order = rng.permutation(xyz.shape[1])
    xyz = np.ascontiguousarray(xyz[:, order])
    fields = rng.standard_normal((nfields, xyz.shape[1])).astype(dtype)
    return xyz, fields
