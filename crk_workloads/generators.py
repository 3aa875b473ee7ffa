"""Seeded input generators (see package docstring; recipes in DESIGN.md).

Nothing here evaluates an SPH kernel or any CRKSPH quantity.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

N_H = 2.4          # particles per support radius: (4/3) pi n_h^3 = 57.9 (PAPER.md:336 with n_h=4 -> 268)
GAMMA = 5.0 / 3.0
BOX = 1.0

CONFIG_NAMES = ("tiny_uniform", "blast_wave", "clustered", "cosmo", "cosmo_large", "clustered_large")


@dataclass
class ParticleSet:
    name: str
    seed: int
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    vx: np.ndarray
    vy: np.ndarray
    vz: np.ndarray
    m: np.ndarray
    h: np.ndarray
    u: np.ndarray
    box: float = BOX
    gamma: float = GAMMA
    n_h: float = N_H
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    def subset(self, idx: np.ndarray) -> "ParticleSet":
        f = lambda a: np.ascontiguousarray(a[idx])
        return ParticleSet(self.name + "[sub]", self.seed, f(self.x), f(self.y), f(self.z),
                           f(self.vx), f(self.vy), f(self.vz), f(self.m), f(self.h), f(self.u),
                           self.box, self.gamma, self.n_h, dict(self.meta))


def _rng(seed: int, stream: int) -> np.random.Generator:
    # counter-based, machine independent; one independent stream per quantity
    return np.random.Generator(np.random.Philox(key=[np.uint64(seed), np.uint64(stream)]))


def _wrap32(p64: np.ndarray) -> np.ndarray:
    """wrap into [0,1) in float64, cast to float32, and fix the cast rounding up to 1.0"""
    p = p64 - np.floor(p64)
    p32 = p.astype(np.float32)
    p32[p32 >= np.float32(1.0)] = np.float32(0.0)
    return p32


def _lattice(n_side: int) -> np.ndarray:
    """cell-centred cubic lattice, shape (n_side^3, 3), float64, x fastest-varying last"""
    g = (np.arange(n_side, dtype=np.float64) + 0.5) / n_side
    q = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    return q


def _pack(name, seed, pos64, vel, u, h, meta=None) -> ParticleSet:
    n = pos64.shape[0]
    m = np.full(n, 1.0 / n, dtype=np.float32)
    c = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return ParticleSet(name, seed, _wrap32(pos64[:, 0]), _wrap32(pos64[:, 1]), _wrap32(pos64[:, 2]),
                       c(vel[:, 0]), c(vel[:, 1]), c(vel[:, 2]), m, c(h), c(u), meta=meta or {})


# --------------------------------------------------------------------------- config 1
def tiny_uniform(n_side: int = 16, seed: int = 1001, jitter: float = 0.1) -> ParticleSet:
    """BASELINE config 1: jittered lattice, Gaussian velocities sigma=0.1, u~U[1,2], equal h=2.4*spacing."""
    n = n_side ** 3
    d = 1.0 / n_side
    q = _lattice(n_side)
    pos = q + _rng(seed, 0).uniform(-jitter * d, jitter * d, size=(n, 3))
    vel = _rng(seed, 1).normal(0.0, 0.1, size=(n, 3))
    u = _rng(seed, 2).uniform(1.0, 2.0, size=n)
    h = np.full(n, N_H * d)
    return _pack("tiny_uniform", seed, pos, vel, u, h, {"n_side": n_side})


# --------------------------------------------------------------------------- config 2
def blast_wave(n_side: int = 64, seed: int = 1002, jitter: float = 0.05) -> ParticleSet:
    """BASELINE config 2: jittered lattice at rest, u=1e-5 except the 8 particles nearest the centre,
    which share total thermal energy sum(m u) = 1  (shape of the paper's Sedov-Taylor set-up)."""
    n = n_side ** 3
    d = 1.0 / n_side
    q = _lattice(n_side)
    pos = q + _rng(seed, 0).uniform(-jitter * d, jitter * d, size=(n, 3))
    vel = np.zeros((n, 3))
    u = np.full(n, 1.0e-5)
    r2 = ((pos - 0.5) ** 2).sum(axis=1)
    hot = np.argsort(r2, kind="stable")[:8]
    u[hot] = 1.0 / (8.0 * (1.0 / n))
    h = np.full(n, N_H * d)
    return _pack("blast_wave", seed, pos, vel, u, h, {"n_side": n_side, "hot": hot.tolist()})


# --------------------------------------------------------------------------- config 3
def _knn_support(pos32: np.ndarray, k: int) -> np.ndarray:
    """support radius = midpoint of the k-th and (k+1)-th neighbour distances (periodic),
    so every particle has exactly k neighbours strictly inside its support."""
    from scipy.spatial import cKDTree
    p = pos32.astype(np.float64)
    tree = cKDTree(p, boxsize=BOX, balanced_tree=False, compact_nodes=False)
    h = np.empty(p.shape[0])
    step = 1 << 20
    for s in range(0, p.shape[0], step):
        dist, _ = tree.query(p[s:s + step], k=k + 2, workers=-1)   # column 0 is the particle itself
        h[s:s + step] = 0.5 * (dist[:, k] + dist[:, k + 1])
    return h


def clustered_plummer(n_side: int = 128, seed: int = 1003, frac_clustered: float = 0.7,
                      n_spheres: int | None = None, k_nbr: int = 58, name: str = "clustered") -> ParticleSet:
    """BASELINE config 3: 70% of particles in Plummer spheres (centres uniform, scale radii log-uniform in
    [0.002, 0.02]), 30% uniform background; v ~ N(0, 0.05^2); u log-uniform in [0.1, 10]; adaptive h with
    exactly k_nbr neighbours inside the support (k-th-neighbour rule; >10x range in h)."""
    n = n_side ** 3
    if n_spheres is None:
        n_spheres = max(1, (512 * n) // (128 ** 3))
    n_cl = int(round(frac_clustered * n))
    r = _rng(seed, 0)
    centres = r.uniform(0.0, 1.0, size=(n_spheres, 3))
    a = np.exp(r.uniform(np.log(0.002), np.log(0.02), size=n_spheres))
    owner = _rng(seed, 1).integers(0, n_spheres, size=n_cl)
    # Plummer cumulative mass M(<r)/M = r^3 / (r^2 + a^2)^{3/2}  ->  r = a / sqrt(U^{-2/3} - 1)
    U = _rng(seed, 2).uniform(1e-9, 1.0 - 1e-9, size=n_cl)
    rad = a[owner] / np.sqrt(U ** (-2.0 / 3.0) - 1.0)
    rad = np.minimum(rad, 0.45)                      # keep the far tail inside one periodic image
    mu = _rng(seed, 3).uniform(-1.0, 1.0, size=n_cl)
    ph = _rng(seed, 4).uniform(0.0, 2.0 * np.pi, size=n_cl)
    s = np.sqrt(1.0 - mu * mu)
    pos_cl = centres[owner] + rad[:, None] * np.stack([s * np.cos(ph), s * np.sin(ph), mu], axis=1)
    pos_bg = _rng(seed, 5).uniform(0.0, 1.0, size=(n - n_cl, 3))
    pos = np.concatenate([pos_cl, pos_bg], axis=0)
    order = _rng(seed, 6).permutation(n)             # no generator-side spatial order leaks to the solver
    pos = pos[order]
    vel = _rng(seed, 7).normal(0.0, 0.05, size=(n, 3))
    u = np.exp(_rng(seed, 8).uniform(np.log(0.1), np.log(10.0), size=n))
    ps = _pack(name, seed, pos, vel, u, np.ones(n), {"n_side": n_side, "n_spheres": n_spheres})
    del pos, vel, u
    p32 = np.stack([ps.x, ps.y, ps.z], axis=1)
    h = _knn_support(p32, k_nbr)
    ps.h = np.minimum(h, 0.49 * BOX).astype(np.float32)
    return ps


# --------------------------------------------------------------------------- configs 4, 5
def zeldovich(n_side: int = 256, seed: int = 1004, rms_disp: float = 0.3, k_cut: float | None = None,
              name: str = "cosmo") -> ParticleSet:
    """BASELINE configs 4/5: lattice displaced by a Zel'dovich field from a Gaussian random field with
    P(k) ~ k^-2 exp(-(k/k_c)^2), k_c = 64*2pi; 3-D rms displacement = rms_disp lattice spacings; v = psi (f=1);
    u = 1 + 0.01 N(0,1); h = 2.4 * spacing * J^{1/3} with J = |det(I + d psi / d q)| the Zel'dovich volume
    factor (generator-side density, no neighbour sums)."""
    n = n_side ** 3
    d = 1.0 / n_side
    if k_cut is None:
        k_cut = 64.0 * 2.0 * np.pi
    white = _rng(seed, 0).standard_normal(size=(n_side, n_side, n_side)).astype(np.float64)
    wk = np.fft.rfftn(white)
    del white
    k1 = 2.0 * np.pi * np.fft.fftfreq(n_side, d=d)
    kz1 = 2.0 * np.pi * np.fft.rfftfreq(n_side, d=d)
    kx, ky, kz = np.meshgrid(k1, k1, kz1, indexing="ij", sparse=True)
    k2 = kx * kx + ky * ky + kz * kz
    k2[0, 0, 0] = 1.0
    amp = np.sqrt(np.exp(-k2 / (k_cut * k_cut)) / k2)      # sqrt(P(k))
    amp[0, 0, 0] = 0.0
    # zero the Nyquist planes so that i*k*delta_k is Hermitian and psi is real
    nyq = n_side // 2
    dk = wk * amp / k2                                       # delta_k / k^2
    del wk, amp
    dk[nyq, :, :] = 0.0
    dk[:, nyq, :] = 0.0
    dk[:, :, -1] = 0.0
    kvec = (kx, ky, kz)
    shape = (n_side, n_side, n_side)
    psi = [np.fft.irfftn(1j * kvec[a] * dk, s=shape, axes=(0, 1, 2)) for a in range(3)]
    rms = np.sqrt(sum(float((p * p).mean()) for p in psi))
    scale = rms_disp * d / rms
    # deformation tensor d psi_a / d q_b = -k_a k_b delta_k / k^2   (symmetric)
    T = {}
    for a in range(3):
        for b in range(a, 3):
            T[(a, b)] = scale * np.fft.irfftn(-(kvec[a] * kvec[b]) * dk, s=shape, axes=(0, 1, 2))
    del dk
    a00 = 1.0 + T[(0, 0)]; a11 = 1.0 + T[(1, 1)]; a22 = 1.0 + T[(2, 2)]
    a01 = T[(0, 1)]; a02 = T[(0, 2)]; a12 = T[(1, 2)]
    J = (a00 * (a11 * a22 - a12 * a12) - a01 * (a01 * a22 - a12 * a02) + a02 * (a01 * a12 - a11 * a02))
    del T, a00, a11, a22, a01, a02, a12
    J = np.clip(np.abs(J), 1.0 / 64.0, 64.0).reshape(-1)
    psi = np.stack([p.reshape(-1) for p in psi], axis=1) * scale
    q = _lattice(n_side)
    pos = q + psi
    vel = psi.copy()
    u = 1.0 + 0.01 * _rng(seed, 1).standard_normal(size=n)
    h = N_H * d * np.cbrt(J)
    ps = _pack(name, seed, pos, vel, u, np.minimum(h, 0.49 * BOX),
               {"n_side": n_side, "rms_disp": rms_disp, "k_cut": float(k_cut)})
    return ps


# --------------------------------------------------------------------------- dispatch
def make_config(name: str, n_side: int | None = None, seed: int | None = None) -> ParticleSet:
    """name in CONFIG_NAMES; n_side overrides the BASELINE size (used for scaled-down parity cases)."""
    if name == "tiny_uniform":
        return tiny_uniform(n_side or 16, seed or 1001)
    if name == "blast_wave":
        return blast_wave(n_side or 64, seed or 1002)
    if name == "clustered":
        return clustered_plummer(n_side or 128, seed or 1003)
    if name == "cosmo":
        return zeldovich(n_side or 256, seed or 1004, rms_disp=0.3, name="cosmo")
    if name == "cosmo_large":
        return zeldovich(n_side or 512, seed or 1005, rms_disp=1.5, name="cosmo_large")
    if name == "clustered_large":
        # BASELINE configs[4] read literally ("generated as in config 3"): the Plummer generator of config 3 at 512^3
        # (the same sphere number density: 512 * 64 spheres), k-th-neighbour h
        return clustered_plummer(n_side or 512, seed or 1006, name="clustered_large")
    raise ValueError(f"unknown config {name!r}; choose from {CONFIG_NAMES}")


def select_window(ps: ParticleSet, centre, half: float, pad: float):
    """Indices of particles whose min-image offset from `centre` is within half+pad on every axis, and a
    boolean mask (over those indices) of the ones within `half` (the un-padded core).  Plain geometry."""
    c = np.asarray(centre, dtype=np.float64)
    L = ps.box

    def off(a, c0):
        dd = a.astype(np.float64) - c0
        dd -= L * np.round(dd / L)
        return np.abs(dd)

    ox, oy, oz = off(ps.x, c[0]), off(ps.y, c[1]), off(ps.z, c[2])
    lim = half + pad
    sel = (ox <= lim) & (oy <= lim) & (oz <= lim)
    idx = np.nonzero(sel)[0]
    core = (ox[idx] <= half) & (oy[idx] <= half) & (oz[idx] <= half)
    return idx, core
