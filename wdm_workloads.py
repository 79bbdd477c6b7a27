"""Seeded synthetic input generators shared by the tests, bench.py and smoke().

This module is the ONLY code both the CUDA path and the CPU oracle are fed from.
It holds none of the method's arithmetic (no kick, drift, Poisson, CIC): it only
builds initial wave functions and particle sets shaped like the paper's
workloads (soliton + granular halo, soliton merger, exponential stellar disc;
PAPER.md:39, 609; Eq. 30) from numpy's PCG64 stream.  numpy's FFT
is used here only to synthesise a random-phase halo from a list of modes, which
is input synthesis, not the split-step method.

Recipe (stated in DESIGN.md "Input recipe"): seed = 26062500 + config number;
L = 1, hbar/m = 1, G = 1/(4 pi); arrays are generated in float64 (float32 for
N >= 512 to bound host memory), cast to the config dtype, and the *cast* arrays
are what both sides receive.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 26062500
FOUR_PI = 4.0 * math.pi


@dataclass
class Workload:
    name: str
    N: int
    dtype: str                      # "c64" | "c128"
    nsteps: int
    L: float = 1.0
    hbar_over_m: float = 1.0
    G: float = 1.0 / FOUR_PI
    dt: float | None = None         # None -> CFL from the initial potential
    psi: np.ndarray | None = None   # (N,N,N) complex64/complex128
    pos: np.ndarray | None = None   # (Np,3) float32/float64 in [-L/2, L/2)
    vel: np.ndarray | None = None
    mass: float = 0.0               # equal particle mass
    meta: dict = field(default_factory=dict)

    @property
    def dx(self) -> float:
        return self.L / self.N

    @property
    def cdtype(self):
        return np.complex64 if self.dtype == "c64" else np.complex128

    @property
    def rdtype(self):
        return np.float32 if self.dtype == "c64" else np.float64


def _rng(cfg: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + cfg))


def _axis(N: int, L: float, dtype=np.float64) -> np.ndarray:
    """Grid coordinates x_i = -L/2 + i dx, dx = L/N (Eq. 20; reading G1)."""
    return (-0.5 * L + (L / N) * np.arange(N)).astype(dtype)


def _min_image(d: np.ndarray, L: float) -> np.ndarray:
    return d - L * np.round(d / L)


def _work_dtypes(N: int):
    return (np.float32, np.complex64) if N >= 512 else (np.float64, np.complex128)


def soliton_density(r, rho_c: float, r_c: float):
    """rho_c / (1 + 0.091 (r/r_c)^2)^8 (BASELINE.json config 2)."""
    return rho_c / (1.0 + 0.091 * (r / r_c) ** 2) ** 8


def _add_soliton(psi: np.ndarray, N: int, L: float, centre, rho_c: float, r_c: float,
                 kvec=None) -> None:
    """psi += sqrt(rho_sol(|x - centre|_minimum-image)) * exp(i k.x), slab by slab."""
    rdt = psi.real.dtype
    x = _axis(N, L, rdt)
    dx2 = _min_image(x - centre[0], L) ** 2
    dy2 = _min_image(x - centre[1], L) ** 2
    dz2 = _min_image(x - centre[2], L) ** 2
    yz = dy2[:, None] + dz2[None, :]
    if kvec is not None:
        py = np.exp(1j * (kvec[1] * x)).astype(psi.dtype)
        pz = np.exp(1j * (kvec[2] * x)).astype(psi.dtype)
        pyz = py[:, None] * pz[None, :]
    for i in range(N):
        r2 = dx2[i] + yz
        amp = np.sqrt(rho_c) / (1.0 + (0.091 / r_c ** 2) * r2) ** 4
        if kvec is None:
            psi[i] += amp
        else:
            psi[i] += amp * (pyz * np.exp(1j * kvec[0] * x[i]).astype(psi.dtype))


def _halo(N: int, L: float, nmodes: int, sigma_n: float, rng: np.random.Generator,
          mean_density: float, cdt) -> np.ndarray:
    """Random-phase halo: sum_j a e^{i(k_j.x + phi_j)}, lattice modes n_j = round(N(0, sigma_n^2))
    per component (a Maxwellian in |v|), equal |a_j| after sampling, phases U[0, 2pi),
    scaled to the requested mean density.  Built by scattering the modes into k-space and
    one inverse FFT (input synthesis only)."""
    import scipy.fft as sfft
    n = np.rint(rng.normal(0.0, sigma_n, size=(nmodes, 3))).astype(np.int64)
    phi = rng.uniform(0.0, 2.0 * math.pi, size=nmodes)
    spec = np.zeros((N, N, N), dtype=cdt)
    np.add.at(spec, (n[:, 0] % N, n[:, 1] % N, n[:, 2] % N), np.exp(1j * phi).astype(cdt))
    # sum_k c_k e^{ik.x}: unnormalised inverse transform
    halo = sfft.ifftn(spec, norm="forward", workers=-1, overwrite_x=True)
    del spec
    msq = 0.0
    for i in range(N):                                # slab-wise mean |halo|^2 (bounded temporaries)
        msq += float(np.sum(np.abs(halo[i]).astype(np.float64) ** 2))
    msq /= float(N) ** 3
    halo *= cdt(math.sqrt(mean_density / msq))
    return halo


def _soliton_halo(cfg_seed: int, N: int, nmodes: int, L: float = 1.0) -> np.ndarray:
    rng = _rng(cfg_seed)
    _, cdt = _work_dtypes(N)
    sigma_v = 20.0
    sigma_n = sigma_v * L / (2.0 * math.pi)          # hbar/m = 1
    psi = _halo(N, L, nmodes, sigma_n, rng, mean_density=1.0, cdt=cdt)
    _add_soliton(psi, N, L, centre=(0.0, 0.0, 0.0), rho_c=1000.0, r_c=0.05 * L)
    return psi


def config1() -> Workload:
    """32^3 complex128: normalised sum of 3 Gaussian packets (sigma = 0.08 L), lattice momenta
    |n| <= 4, one random phase per packet; 10 steps, dt = 0.2 dx^2 (BASELINE.json configs[0])."""
    N, L = 32, 1.0
    rng = _rng(1)
    x = _axis(N, L)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    psi = np.zeros((N, N, N), dtype=np.complex128)
    sigma = 0.08 * L
    for _ in range(3):
        c = rng.uniform(-0.5 * L, 0.5 * L, size=3)
        while True:
            n = rng.integers(-4, 5, size=3)
            if n @ n <= 16:
                break
        k = 2.0 * math.pi * n / L
        ph = rng.uniform(0.0, 2.0 * math.pi)
        r2 = _min_image(X - c[0], L) ** 2 + _min_image(Y - c[1], L) ** 2 + _min_image(Z - c[2], L) ** 2
        psi += np.exp(-r2 / (4.0 * sigma ** 2) + 1j * (k[0] * X + k[1] * Y + k[2] * Z + ph))
    dx = L / N
    psi /= math.sqrt(float(np.sum(np.abs(psi) ** 2)) * dx ** 3)
    return Workload("cfg1_32_c128_packets", N, "c128", 10, dt=0.2 * dx * dx, psi=psi)


def config2(N: int = 128, nsteps: int = 100, nmodes: int = 4096, dtype: str = "c64",
            name: str | None = None, seed: int = 2) -> Workload:
    """soliton (rho_c = 1000, r_c = 0.05 L) + Maxwellian random-phase halo (BASELINE.json configs[1])."""
    psi = _soliton_halo(seed, N, nmodes)
    w = Workload(name or f"cfg2_{N}_{dtype}_soliton_halo", N, dtype, nsteps)
    w.psi = np.ascontiguousarray(psi.astype(w.cdtype, copy=False))
    return w


def config3(N: int = 256, nsteps: int = 200) -> Workload:
    """Merger of 8 solitons with bulk velocities (BASELINE.json configs[2])."""
    L = 1.0
    rng = _rng(3)
    _, cdt = _work_dtypes(N)
    psi = np.zeros((N, N, N), dtype=cdt)
    for _ in range(8):
        r_c = rng.uniform(0.02, 0.06) * L
        rho_c = 1000.0 * (0.05 * L / r_c) ** 4
        c = rng.uniform(-0.25 * L, 0.25 * L, size=3)
        v = rng.normal(0.0, 10.0, size=3)
        n = np.rint(v * L / (2.0 * math.pi))
        _add_soliton(psi, N, L, c, rho_c, r_c, kvec=2.0 * math.pi * n / L)
    w = Workload(f"cfg3_{N}_c64_merger", N, "c64", nsteps)
    w.psi = np.ascontiguousarray(psi.astype(np.complex64))
    return w


def config4(N: int = 1024, nsteps: int = 20) -> Workload:
    """1024^3 soliton + 65536-mode halo, fixed dt = dx^2/6 (BASELINE.json configs[3])."""
    w = config2(N=N, nsteps=nsteps, nmodes=65536, name=f"cfg4_{N}_c64_soliton_halo", seed=4)
    w.dt = (w.L / N) ** 2 / 6.0
    return w


def t512(nsteps: int = 50) -> Workload:
    """512^3 complex64 soliton + 65536-mode halo: the north_star target measurement."""
    w = config2(N=512, nsteps=nsteps, nmodes=65536, name="t512_c64_soliton_halo", seed=4)
    w.dt = (w.L / 512) ** 2 / 6.0
    return w


def disk_particles(rng: np.random.Generator, n: int, L: float, G: float, m_dm_soliton: float,
                   rho_halo: float, m_disk: float, R_d: float, z_d: float, r_c: float, rho_c: float,
                   rdtype=np.float32):
    """Exponential disc rho ~ exp(-|z|/z_d - R/R_d) (Eq. 30): R ~ Gamma(2, R_d) (R < L/2),
    phi ~ U, z ~ Laplace(z_d); v = v_c(R) e_phi + N(0, (0.1 v_c)^2) per component with
    v_c^2 = G M(<R)/R from the soliton + mean halo + disc enclosed mass (spherical approximation)."""
    R = np.empty(0)
    while R.size < n:
        cand = rng.gamma(2.0, R_d, size=n)
        R = np.concatenate([R, cand[cand < 0.5 * L]])
    R = R[:n]
    phi = rng.uniform(0.0, 2.0 * math.pi, size=n)
    z = rng.laplace(0.0, z_d, size=n)
    z = _min_image(z, L)
    pos = np.stack([R * np.cos(phi), R * np.sin(phi), z], axis=1)
    # enclosed masses on a radial table
    rt = np.linspace(0.0, 0.5 * L, 4097)[1:]
    shell = 4.0 * math.pi * rt ** 2 * soliton_density(rt, rho_c, r_c)
    m_sol = np.cumsum(shell) * (rt[1] - rt[0])
    m_halo = rho_halo * 4.0 / 3.0 * math.pi * rt ** 3
    m_d = m_disk * (1.0 - np.exp(-rt / R_d) * (1.0 + rt / R_d))
    vc_t = np.sqrt(G * (m_sol + m_halo + m_d) / rt)
    vc = np.interp(R, rt, vc_t)
    vel = np.stack([-vc * np.sin(phi), vc * np.cos(phi), np.zeros(n)], axis=1)
    vel += rng.normal(0.0, 1.0, size=(n, 3)) * (0.1 * vc)[:, None]
    pos = pos.astype(rdtype)
    # wrap into [-L/2, L/2) after the cast
    half = rdtype(0.5 * L)
    pos = np.where(pos >= half, pos - rdtype(L), pos)
    pos = np.where(pos < -half, pos + rdtype(L), pos).astype(rdtype)
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel.astype(rdtype))


def config5(N: int = 256, nsteps: int = 100, n_particles: int = 1 << 20, nmodes: int = 4096) -> Workload:
    """Coupled run: soliton + halo at N^3 plus 2^20 equal-mass disc particles carrying 5 % of the
    dark-matter mass (BASELINE.json configs[4])."""
    w = config2(N=N, nsteps=nsteps, nmodes=nmodes, name=f"cfg5_{N}_c64_coupled_disk", seed=5)
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 55))
    dx = w.L / N
    m_dm = float(np.sum(np.abs(w.psi.astype(np.complex128)) ** 2)) * dx ** 3
    m_disk = 0.05 * m_dm
    w.pos, w.vel = disk_particles(rng, n_particles, w.L, w.G, 0.0, 1.0, m_disk,
                                  R_d=0.05 * w.L, z_d=0.005 * w.L, r_c=0.05 * w.L, rho_c=1000.0,
                                  rdtype=w.rdtype)
    w.mass = m_disk / n_particles
    w.meta["m_dm"] = m_dm
    return w


def small_coupled(N: int = 16, n_particles: int = 257, dtype: str = "c128", seed: int = 77,
                  nsteps: int = 5) -> Workload:
    """Small coupled case for element-by-element parity: smooth two-mode wave field + a clump of
    particles carrying ~20 % of the mass (includes particles within one cell of the box faces)."""
    L = 1.0
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + seed))
    x = _axis(N, L)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    k = 2.0 * math.pi / L
    psi = (3.0 + np.exp(1j * k * X) + 0.5 * np.exp(1j * (k * Y - 2 * k * Z)) +
           0.3 * np.exp(-((X - 0.1) ** 2 + Y ** 2 + (Z + 0.2) ** 2) / (2 * 0.15 ** 2)))
    w = Workload(f"small_coupled_{N}_{dtype}", N, dtype, nsteps)
    w.psi = np.ascontiguousarray(psi.astype(w.cdtype))
    pos = rng.normal(0.0, 0.12 * L, size=(n_particles, 3))
    pos[:8] = rng.uniform(0.5 * L - 1.5 * L / N, 0.5 * L, size=(8, 3)) * rng.choice([-1.0, 1.0], size=(8, 3))
    pos = _min_image(pos, L)
    vel = rng.normal(0.0, 1.0, size=(n_particles, 3))
    rdt = w.rdtype
    pos = pos.astype(rdt)
    half = rdt(0.5 * L)
    pos = np.where(pos >= half, pos - rdt(L), pos)
    pos = np.where(pos < -half, pos + rdt(L), pos).astype(rdt)
    w.pos = np.ascontiguousarray(pos)
    w.vel = np.ascontiguousarray(vel.astype(rdt))
    m_dm = float(np.sum(np.abs(psi) ** 2)) * (L / N) ** 3
    w.mass = 0.2 * m_dm / n_particles
    w.dt = 0.2 * (L / N) ** 2
    w.G = 40.0 / FOUR_PI      # strong gravity so that the coupling terms are not lost in roundoff
    return w


def random_field(N: int, dtype: str, seed: int) -> np.ndarray:
    """White complex noise (test-only input: exercises every Fourier mode)."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 1000 + seed))
    cdt = np.complex64 if dtype == "c64" else np.complex128
    return np.ascontiguousarray((rng.normal(size=(N, N, N)) + 1j * rng.normal(size=(N, N, N))).astype(cdt))


def cfl_dt(w: Workload, max_abs_phi: float) -> float:
    """dt = min(dx^2/6, 1/max|Phi0|) with m/hbar = 1 (BASELINE.json configs 2, 3, 5; reading G17)."""
    dx = w.L / w.N
    kin = dx * dx / (6.0 * w.hbar_over_m)
    if max_abs_phi <= 0.0:
        return kin
    return min(kin, w.hbar_over_m / max_abs_phi)
