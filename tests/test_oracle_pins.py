"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself by retyping its formula: each expected value is a
closed form, an invariant, a brute-force sum, or a library routine used as a check OF the oracle.
"""
import math

import numpy as np
import pytest

import oracle
import wdm_workloads as wl

FOUR_PI = 4.0 * math.pi


def grid(N, L=1.0):
    x = -0.5 * L + (L / N) * np.arange(N)
    return np.meshgrid(x, x, x, indexing="ij")


def relerr(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


def run(N, psi, nsteps, dt, L=1.0, mu=1.0, G=1.0 / FOUR_PI, particles=None):
    o = oracle.Oracle(N, L, mu, G)
    o.set_psi(psi)
    if particles is not None:
        o.set_particles(*particles)
    o.step(nsteps, dt)
    return o


# ---------------------------------------------------------------- P5 / P10: the FFT itself

@pytest.mark.parametrize("n", [2, 4, 8, 16, 64, 256, 1024])
def test_p5_fft1d_vs_direct_dft(n):
    rng = np.random.default_rng(n)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    f = oracle.fft1d(x, -1)
    d = oracle.dft1d_direct(x, -1)
    assert relerr(f, d) < 1e-13
    # the direct sum is itself the definition sum_j x_j e^{-2 pi i jk/n}: spot-check one bin by hand
    k = n // 3
    assert abs(d[k] - sum(x[j] * np.exp(-2j * np.pi * j * k / n) for j in range(n))) < 1e-10
    # inverse carries 1/n and round-trips
    assert relerr(oracle.fft1d(f, +1), x) < 1e-13


def test_p5_fft3_vs_bruteforce_triple_sum_8cubed():
    a = wl.random_field(8, "c128", 5)
    assert relerr(oracle.fft3(a, -1), oracle.dft3_direct(a, -1)) < 1e-13
    assert relerr(oracle.fft3(a, +1), oracle.dft3_direct(a, +1)) < 1e-13
    # a delta at (1,2,3) transforms to the plane wave e^{-2 pi i (kx+2ky+3kz)/8}: fixes sign + axis order
    d = np.zeros((8, 8, 8), complex); d[1, 2, 3] = 1.0
    k = np.arange(8)
    KX, KY, KZ = np.meshgrid(k, k, k, indexing="ij")
    assert relerr(oracle.fft3(d, -1), np.exp(-2j * np.pi * (KX + 2 * KY + 3 * KZ) / 8)) < 1e-14


@pytest.mark.parametrize("N", [16, 32, 64])
def test_p10_fft3_vs_numpy(N):
    a = wl.random_field(N, "c128", N)
    assert relerr(oracle.fft3(a, -1), np.fft.fftn(a)) < 1e-13
    assert relerr(oracle.fft3(a, +1), np.fft.ifftn(a)) < 1e-13


# ---------------------------------------------------------------- P1: unitarity

def test_p1_norm_conserved_config1():
    w = wl.config1()
    n0 = np.sum(np.abs(w.psi) ** 2) * w.dx ** 3
    assert abs(n0 - 1.0) < 1e-12                      # G19: normalised input
    o = run(w.N, w.psi, 10, w.dt)
    n1 = np.sum(np.abs(o.psi()) ** 2) * w.dx ** 3
    assert abs(n1 - n0) < 1e-13


def test_p1_norm_conserved_strong_gravity():
    N = 16
    psi = wl.random_field(N, "c128", 1) + 3.0
    o = run(N, psi, 20, 1e-3, G=50.0)
    assert abs(np.sum(np.abs(o.psi()) ** 2) / np.sum(np.abs(psi) ** 2) - 1.0) < 1e-13


# ---------------------------------------------------------------- P2: free Gaussian packet

def gaussian_packet(X, Y, Z, sigma, k0, t, mu):
    """psi(x,t) for psi(x,0) = (2 pi s^2)^(-3/4) exp(-|x|^2/4s^2 + i k0.x), free Schroedinger
    i psi_t = -(mu/2) lap psi  (textbook spreading Gaussian)."""
    tau = mu * t / (2.0 * sigma ** 2)
    xc = [X - mu * k0[0] * t, Y - mu * k0[1] * t, Z - mu * k0[2] * t]
    r2 = xc[0] ** 2 + xc[1] ** 2 + xc[2] ** 2
    kk = float(np.dot(k0, k0))
    phase = k0[0] * xc[0] + k0[1] * xc[1] + k0[2] * xc[2] + 0.5 * mu * kk * t
    return (2 * np.pi * sigma ** 2) ** -0.75 * (1 + 1j * tau) ** -1.5 * np.exp(-r2 / (4 * sigma ** 2 * (1 + 1j * tau)) + 1j * phase)


@pytest.mark.parametrize("nsteps", [1, 7])
def test_p2_free_gaussian_closed_form(nsteps):
    N, L, mu = 64, 1.0, 0.7
    sigma = 0.04 * L
    k0 = 2 * np.pi / L * np.array([3.0, -2.0, 1.0])
    X, Y, Z = grid(N, L)
    psi0 = gaussian_packet(X, Y, Z, sigma, k0, 0.0, mu)
    T = 2.0 * sigma ** 2 / mu * 0.6            # tau = 0.6: width grows by sqrt(1.36)
    o = run(N, psi0, nsteps, T / nsteps, L=L, mu=mu, G=0.0)
    exact = gaussian_packet(X, Y, Z, sigma, k0, T, mu)
    # spectral drift is exact for any dt: residual = periodic images + sampling only
    assert relerr(o.psi(), exact) < 1e-9
    # and the packet really moved and spread (guards a no-op)
    assert relerr(psi0, exact) > 0.5


def test_p2_sign_of_drift_phase():
    """A wrong sign of the kinetic phase conjugates the evolution: check against the conjugate too."""
    N, L, mu = 32, 1.0, 1.0
    X, Y, Z = grid(N, L)
    sigma = 0.08
    k0 = 2 * np.pi * np.array([1.0, 0.0, 0.0])
    T = 0.004
    o = run(N, gaussian_packet(X, Y, Z, sigma, k0, 0.0, mu), 2, T / 2, G=0.0)
    good = gaussian_packet(X, Y, Z, sigma, k0, T, mu)
    bad = gaussian_packet(X, Y, Z, sigma, k0, -T, mu)
    assert relerr(o.psi(), good) < 1e-3 < 0.1 < relerr(o.psi(), bad)   # 1e-3: periodic images of a sigma=0.08L packet


# ---------------------------------------------------------------- P3: plane wave with gravity on

def test_p3_plane_wave_exact():
    N, L, mu = 16, 2.0, 1.3
    X, Y, Z = grid(N, L)
    n = np.array([2, -1, 3])
    k = 2 * np.pi * n / L
    A = 0.8 - 0.3j
    psi0 = A * np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z))
    dt, ns = 0.01, 9
    o = run(N, psi0, ns, dt, L=L, mu=mu, G=3.0)
    exact = psi0 * np.exp(-0.5j * mu * float(k @ k) * dt * ns)
    assert relerr(o.psi(), exact) < 1e-13
    assert np.max(np.abs(o.potential())) < 1e-12        # uniform density -> Phi = 0 (k=0 zeroed)
    assert np.allclose(o.density(), abs(A) ** 2, rtol=1e-13)


# ---------------------------------------------------------------- P4: single-mode Poisson

def test_p4_single_mode_poisson_closed_form():
    N, L, G = 32, 1.5, 0.37
    X, Y, Z = grid(N, L)
    n = np.array([1, 2, -3])
    k = 2 * np.pi * n / L
    rho0, rho1 = 5.0, 0.25
    arg = k[0] * X + k[1] * Y + k[2] * Z
    rho = rho0 + rho1 * np.cos(arg)
    phi = oracle.poisson(rho, L, G)
    exact = -4 * np.pi * G * rho1 * np.cos(arg) / float(k @ k)
    assert relerr(phi, exact) < 1e-13
    assert abs(phi.mean()) < 1e-15
    # through the context as well: psi = sqrt(rho) gives the same potential
    o = oracle.Oracle(N, L, 1.0, G); o.set_psi(np.sqrt(rho).astype(complex))
    assert relerr(o.potential(), exact) < 1e-12


def test_p4_poisson_discrete_laplacian_of_smooth_field():
    """lap Phi = 4 pi G (rho - <rho>) checked spectrally-independent: 2nd-order FD Laplacian converges."""
    L, G = 1.0, 1.0 / FOUR_PI
    errs = []
    for N in (16, 32):
        X, Y, Z = grid(N, L)
        rho = np.exp(np.cos(2 * np.pi * X) + np.sin(2 * np.pi * Y) * np.cos(2 * np.pi * Z))
        phi = oracle.poisson(rho, L, G)
        dx = L / N
        lap = sum(np.roll(phi, 1, a) + np.roll(phi, -1, a) - 2 * phi for a in range(3)) / dx ** 2
        errs.append(relerr(lap, FOUR_PI * G * (rho - rho.mean())))
    assert errs[1] < errs[0] / 3.5 and errs[1] < 0.02


# ---------------------------------------------------------------- P6: second-order energy error

def total_energy(psi, phi, L, mu):
    """E = T + W: T = (mu^2/2) sum_k k^2 |psi_k|^2 dV/N^3 (Parseval), W = (1/2) sum rho Phi dV."""
    N = psi.shape[0]
    dV = (L / N) ** 3
    k = 2 * np.pi * np.fft.fftfreq(N, d=L / N)
    K2 = k[:, None, None] ** 2 + k[None, :, None] ** 2 + k[None, None, :] ** 2
    pk = np.fft.fftn(psi)
    T = 0.5 * mu ** 2 * float(np.sum(K2 * np.abs(pk) ** 2)) * dV / N ** 3
    W = 0.5 * float(np.sum(np.abs(psi) ** 2 * phi)) * dV
    return T + W


def test_p6_energy_error_is_second_order():
    N, L, mu, G = 16, 1.0, 1.0, 200.0 / FOUR_PI
    X, Y, Z = grid(N, L)
    psi0 = (2.0 + np.exp(2j * np.pi * X) + 0.7 * np.exp(2j * np.pi * (Y - Z)) + 0.4 * np.cos(2 * np.pi * Z)).astype(complex)
    Tend = 0.02
    drifts = []
    for ns in (8, 16, 32, 64):
        o = oracle.Oracle(N, L, mu, G); o.set_psi(psi0)
        e0 = total_energy(o.psi(), o.potential(), L, mu)
        worst = 0.0
        for _ in range(ns):
            o.step(1, Tend / ns)
            worst = max(worst, abs(total_energy(o.psi(), o.potential(), L, mu) - e0))
        drifts.append(worst / abs(e0))
    ratios = [drifts[i] / drifts[i + 1] for i in range(3)]
    assert drifts[0] > 1e-9                      # gravity is actually doing something
    assert all(3.6 < r < 4.4 for r in ratios), (drifts, ratios)


def test_p6_solution_self_convergence_second_order():
    N, L, G = 16, 1.0, 100.0 / FOUR_PI
    psi0 = wl.small_coupled(N).psi
    Tend = 0.004
    sols = [run(N, psi0, ns, Tend / ns, G=G).psi() for ns in (4, 8, 16, 32)]
    d = [np.linalg.norm(sols[i] - sols[i + 1]) for i in range(3)]
    assert 3.6 < d[0] / d[1] < 4.4 and 3.6 < d[1] / d[2] < 4.4, d


# ---------------------------------------------------------------- P7: time reversal (whole coupled step)

def test_p7_time_reversal_with_particles():
    w = wl.small_coupled(16)
    o = oracle.Oracle(w.N, w.L, w.hbar_over_m, w.G)
    o.set_psi(w.psi); o.set_particles(w.pos, w.vel, w.mass)
    o.step(12, w.dt)
    moved = relerr(o.psi(), w.psi)
    o.step(12, -w.dt)
    pos, vel = o.particles()
    assert moved > 1e-3
    assert relerr(o.psi(), w.psi) < 1e-12
    d = pos - w.pos; d -= w.L * np.round(d / w.L)
    assert np.max(np.abs(d)) < 1e-13 and np.max(np.abs(vel - w.vel)) < 1e-11


# ---------------------------------------------------------------- P8: CIC deposit / gather pair

def test_p8_cic_mass_node_and_weights():
    N, L = 8, 2.0
    dx = L / N
    # a particle exactly on node (3,0,7) deposits m/dx^3 there and nothing elsewhere
    pos = np.array([[-L / 2 + 3 * dx, -L / 2, -L / 2 + 7 * dx]])
    rho = oracle.cic_deposit(N, L, pos, 2.5)
    assert rho[3, 0, 7] == pytest.approx(2.5 / dx ** 3, rel=1e-14)
    assert np.count_nonzero(rho) == 1
    # a quarter of the way from node (7,7,7) towards (0,0,0) across the periodic face, per axis
    pos = np.array([[L / 2 - 0.75 * dx] * 3])
    rho = oracle.cic_deposit(N, L, pos, 1.0) * dx ** 3
    assert rho[7, 7, 7] == pytest.approx(0.75 ** 3) and rho[0, 0, 0] == pytest.approx(0.25 ** 3)
    assert rho[0, 7, 7] == pytest.approx(0.25 * 0.75 ** 2) and rho[7, 0, 0] == pytest.approx(0.75 * 0.25 ** 2)
    assert rho.sum() == pytest.approx(1.0, rel=1e-14)
    # total mass of a random cloud with individual masses
    rng = np.random.default_rng(3)
    p = rng.uniform(-L / 2, L / 2, size=(500, 3)); m = rng.uniform(0.1, 2.0, size=500)
    assert oracle.cic_deposit(N, L, p, m).sum() * dx ** 3 == pytest.approx(m.sum(), rel=1e-13)


def test_p8_zero_self_force_and_momentum_conservation():
    N, L, G = 16, 1.0, 1.0
    rng = np.random.default_rng(8)
    o = oracle.Oracle(N, L, 1.0, G)
    o.set_psi(np.zeros((N, N, N), complex))
    # single particle: no self force
    o.set_particles(rng.uniform(-0.5, 0.5, size=(1, 3)), np.zeros((1, 3)), 1.0)
    assert np.max(np.abs(o.accel())) < 1e-12
    # many particles: total momentum change vanishes
    p = rng.uniform(-0.5, 0.5, size=(200, 3)); m = rng.uniform(0.5, 1.5, size=200)
    o.set_particles(p, np.zeros((200, 3)), m)
    a = o.accel()
    assert np.max(np.abs(a)) > 1.0
    assert np.max(np.abs((m[:, None] * a).sum(0))) < 1e-11 * np.abs(m[:, None] * a).sum()
    # two particles attract each other (sign of gravity)
    o.set_particles(np.array([[-0.1, 0.02, 0.0], [0.1, 0.0, 0.03]]), np.zeros((2, 3)), 1.0)
    a = o.accel()
    assert a[0, 0] > 0 > a[1, 0]


# ---------------------------------------------------------------- P9: gather in a known field

def test_p9_gather_closed_form():
    N, L = 16, 1.0
    dx = L / N
    X, Y, Z = grid(N, L)
    kk = 2 * np.pi * 2 / L
    A = 0.3
    phi = A * np.cos(kk * Y)                       # varies along axis 1 only
    rng = np.random.default_rng(9)
    pos = rng.uniform(-0.5, 0.5, size=(64, 3))
    acc = oracle.cic_gather(phi, L, pos)
    # node gradient of A cos(k y): -(phi[j+1]-phi[j-1])/(2dx) = A sin(k y_j) sin(k dx)/dx ; CIC = linear interp in y
    u = (pos[:, 1] + L / 2) / dx
    j0 = np.floor(u).astype(int); f = u - j0
    y = -L / 2 + dx * np.arange(N + 1)
    g = A * np.sin(kk * y) * np.sin(kk * dx) / dx
    expect = (1 - f) * g[j0] + f * g[j0 + 1]
    assert np.max(np.abs(acc[:, 1] - expect)) < 1e-13
    assert np.max(np.abs(acc[:, 0])) < 1e-13 and np.max(np.abs(acc[:, 2])) < 1e-13


def test_particle_leapfrog_free_streaming_and_wrap():
    """G = 0: particles stream freely, x(t) = x0 + v t wrapped into [-L/2, L/2)."""
    N, L = 8, 1.0
    o = oracle.Oracle(N, L, 1.0, 0.0)
    o.set_psi(np.ones((N, N, N), complex))
    pos = np.array([[0.49, -0.49, 0.0]]); vel = np.array([[1.0, -2.0, 0.5]])
    o.set_particles(pos, vel, 1.0)
    o.step(10, 0.01)
    p, v = o.particles()
    assert np.allclose(p, [[0.59 - 1.0, -0.69 + 1.0, 0.05]], atol=1e-14)
    assert np.allclose(v, vel)


def test_kick_sign_and_half_step():
    """Drift-free limit: for a k=0 wave function in a *given* potential the KDK step is a pure phase
    exp(-i Phi dt/mu).  Use particles to impose Phi without touching |psi| (uniform)."""
    N, L, mu, G = 8, 1.0, 2.0, 1.0
    o = oracle.Oracle(N, L, mu, G)
    o.set_psi(np.full((N, N, N), 1e-9, complex))        # negligible self-gravity, uniform
    pos = np.array([[0.0, 0.0, 0.0]])
    o.set_particles(pos, np.zeros((1, 3)), 3.0)          # static source (zero self force keeps it put)
    phi = o.potential()
    dt = 1e-4                                            # drift of a non-uniform phase is O(dt^2) here
    o.step(1, dt)
    ratio = o.psi() / 1e-9
    assert relerr(ratio, np.exp(-1j * phi * dt / mu)) < 1e-5
    assert np.max(np.abs(phi)) * dt / mu > 1e-3          # the phase is resolvable
    assert phi[4, 4, 4] == phi.min() < 0                 # attractive well at the particle


# ---------------------------------------------------------------- P11-P13: the extra kick terms

def test_p11_self_interaction_plane_wave_closed_form():
    """V = kappa |psi|^2 (Eq. 14): for psi = A e^{ik.x} the density is uniform, so Phi = 0 and
    psi(t) = A exp(i(k.x - mu k^2 t/2 - kappa A^2 t/mu)) exactly, for any dt (the split step is exact here)."""
    N, L, mu, kappa, A = 16, 1.3, 0.7, 2.5, 0.8
    X, Y, Z = grid(N, L)
    n = np.array([2, -1, 3]); k = 2 * np.pi * n / L
    psi0 = A * np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z))
    for nsteps, dt in ((1, 0.05), (7, 0.011)):
        o = oracle.Oracle(N, L, mu, 1.0 / FOUR_PI)
        o.set_kick_terms(kappa=kappa)
        o.set_psi(psi0)
        o.step(nsteps, dt)
        t = nsteps * dt
        exact = psi0 * np.exp(-1j * (0.5 * mu * (k @ k) * t + kappa * A * A * t / mu))
        assert relerr(o.psi(), exact) < 1e-12
    # sign: an attractive interaction (kappa < 0) advances the phase the other way
    o = oracle.Oracle(N, L, mu, 0.0); o.set_kick_terms(kappa=-kappa); o.set_psi(psi0); o.step(1, 0.05)
    exact = psi0 * np.exp(-1j * (0.5 * mu * (k @ k) * 0.05 - kappa * A * A * 0.05 / mu))
    assert relerr(o.psi(), exact) < 1e-12


def test_p12_external_potential_harmonic_ground_state_second_order():
    """Phi_ext = omega^2 r^2 / 2 (Eq. 13 with a static V): the Gaussian of width a^2 = mu/omega is stationary,
    psi(t) = psi0 exp(-3 i omega t / 2).  The split step reaches it with an error that falls 4x per halving
    of dt, which pins the sign and the 1/mu of the external term and its place in the potential."""
    N, L, mu, a = 32, 1.0, 1.0, 0.06
    omega = mu / a ** 2
    X, Y, Z = grid(N, L)
    r2 = X ** 2 + Y ** 2 + Z ** 2
    psi0 = np.exp(-r2 / (2 * a * a)).astype(complex)
    T = 1.0 / omega
    errs = []
    for nsteps in (8, 16, 32):
        o = oracle.Oracle(N, L, mu, 0.0)
        o.set_kick_terms(phi_ext=0.5 * omega ** 2 * r2)
        o.set_psi(psi0)
        o.step(nsteps, T / nsteps)
        errs.append(relerr(o.psi(), psi0 * np.exp(-1.5j * omega * T)))
        assert relerr(o.potential(), 0.5 * omega ** 2 * r2) < 1e-15      # G = 0: Phi_total is the external term
    assert errs[2] < 2e-4
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5


def test_p12_particles_feel_the_external_potential():
    """Phi_total = Phi_DM + Phi_ext (Alg. 1 l.15) is what the particles gather: massless particle on a node of
    A cos(k x) gets a = A sin(k x_i) sin(k dx)/dx (central difference of the cosine)."""
    N, L, A = 16, 1.0, 0.3
    dx = L / N
    X, Y, Z = grid(N, L)
    kk = 2 * np.pi * 3 / L
    o = oracle.Oracle(N, L, 1.0, 0.0)
    o.set_kick_terms(phi_ext=A * np.cos(kk * X))
    o.set_psi(np.ones((N, N, N), complex))
    xi = -0.5 * L + 5 * dx
    o.set_particles(np.array([[xi, 0.0, 0.0]]), np.zeros((1, 3)), 0.0)
    o.step(0, 0.0)
    acc = o.accel()
    assert abs(acc[0, 0] - A * np.sin(kk * xi) * np.sin(kk * dx) / dx) < 1e-12
    assert abs(acc[0, 1]) < 1e-13 and abs(acc[0, 2]) < 1e-13


def test_p13_absorbing_layer_special_points():
    """Eq. 22 after every step.  From a uniform field (the drift leaves it uniform, G = 0) one step gives
    psi = B(x).  What the formula fixes without retyping it: B = 1 deep inside; on a face (x = -L/2, the
    other two coordinates inside) b = 2 - tanh(0) + tanh(-nb) = 1, so B = e^{-alpha dt}; on an edge
    e^{-2 alpha dt}; at the corner e^{-3 alpha dt}; B is even in every coordinate; the norm only decreases."""
    N, L, alpha, nb, dt = 32, 2.0, 10.0, 50, 0.013
    o = oracle.Oracle(N, L, 1.0, 0.0)
    o.set_kick_terms(absorb_alpha=alpha, absorb_nb=nb)
    o.set_psi(np.ones((N, N, N), complex))
    o.step(1, dt)
    B = o.psi()
    assert np.max(np.abs(B.imag)) < 1e-15
    B = B.real
    m = N // 2
    assert abs(B[m, m, m] - 1.0) < 1e-14 and abs(B[m - 5, m + 6, m + 3] - 1.0) < 1e-12
    e = math.exp(-alpha * dt)
    assert abs(B[0, m, m] - e) < 1e-12 and abs(B[m, 0, m] - e) < 1e-12 and abs(B[m, m, 0] - e) < 1e-12
    assert abs(B[0, 0, m] - e ** 2) < 1e-12 and abs(B[0, 0, 0] - e ** 3) < 1e-12
    for i in range(1, N // 2):                    # x_i = -x_{N-i}: even profile
        assert abs(B[i, m, m] - B[N - i, m, m]) < 1e-13
    assert np.all(np.diff(B[: m + 1, m, m]) >= -1e-15)       # rises monotonically from the face to the centre
    # several steps: the layer only removes norm (the drift in between is unitary)
    n0 = float(np.sum(np.abs(o.psi()) ** 2))
    o.step(3, dt)
    assert float(np.sum(np.abs(o.psi()) ** 2)) < n0


# ---------------------------------------------------------------- P14: diagnostics

def test_p14_diagnostics_plane_wave_closed_forms():
    """psi = A e^{ik.x}: rho = A^2, rho v = mu A^2 sin(k dx)/dx per axis (central difference of the phase), so
    K = A^2 mu^2 sum_a (sin(k_a dx)/dx)^2 L^3 / 2, Q = 0, M = A^2 L^3, Phi = 0 => V = 0, max rho = A^2."""
    N, L, mu, A = 16, 1.3, 0.7, 0.8
    dx = L / N
    X, Y, Z = grid(N, L)
    k = 2 * np.pi * np.array([2, -1, 3]) / L
    o = oracle.Oracle(N, L, mu, 1.0 / FOUR_PI)
    o.set_psi(A * np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z)))
    d = o.diagnostics()
    assert abs(d["M"] - A * A * L ** 3) < 1e-12
    assert abs(d["max_rho"] - A * A) < 1e-14 and d["max_phi"] < 1e-12 and abs(d["V"]) < 1e-12
    assert abs(d["K"] - 0.5 * A * A * mu * mu * np.sum((np.sin(k * dx) / dx) ** 2) * L ** 3) < 1e-10
    assert abs(d["Q"]) < 1e-12
    # Eq. 26: Phi = 0, kappa = 0 -> the kinetic bound alone, 0.5 * 4/(3 pi) dx^2 (m/hbar)
    assert abs(d["dt_max"] - 0.5 * 4 / (3 * np.pi) * dx * dx / mu) < 1e-15


def test_p14_diagnostics_real_gaussian_and_cosine_density():
    """Real psi: K = 0.  Gaussian psi = exp(-r^2/2a^2): Q -> (mu^2/2) (3/2a^2) pi^{3/2} a^3 with second-order
    convergence in dx.  rho = r0 + r1 cos(kx): Phi = -4 pi G r1 cos(kx)/k^2, V = int rho Phi = -4 pi G r1^2 L^3/(2 k^2);
    max|Phi| = 4 pi G r1/k^2 then bounds dt through the second term of Eq. 26."""
    L, mu, a = 1.0, 0.9, 0.09
    exact = 0.5 * mu * mu * 1.5 / a ** 2 * np.pi ** 1.5 * a ** 3
    errs = []
    for N in (16, 32, 64):
        X, Y, Z = grid(N, L)
        o = oracle.Oracle(N, L, mu, 0.0)
        o.set_psi(np.exp(-(X ** 2 + Y ** 2 + Z ** 2) / (2 * a * a)).astype(complex))
        d = o.diagnostics()
        assert abs(d["K"]) < 1e-20
        errs.append(abs(d["Q"] - exact) / exact)
    assert errs[2] < 0.05 and 3.0 < errs[1] / errs[2] < 5.0
    N, G, r0, r1 = 32, 7.0, 2.0, 0.5
    X, Y, Z = grid(N, L)
    kk = 2 * np.pi * 3 / L
    o = oracle.Oracle(N, L, mu, G)
    o.set_psi(np.sqrt(r0 + r1 * np.cos(kk * X)).astype(complex))
    d = o.diagnostics()
    assert abs(d["V"] + 4 * np.pi * G * r1 * r1 * L ** 3 / (2 * kk * kk)) < 1e-10
    assert abs(d["max_phi"] - 4 * np.pi * G * r1 / kk ** 2) < 1e-10 and abs(d["max_rho"] - (r0 + r1)) < 1e-12
    o.set_kick_terms(kappa=-1e4)
    d = o.diagnostics()
    assert abs(d["dt_max"] - 0.5 * 2 * np.pi * mu / (1e4 * (r0 + r1))) < 1e-15     # third term of Eq. 26 is the smallest


# ---------------------------------------------------------------- P15: particle variants

def test_p15_substeps_harmonic_leapfrog_closed_form():
    """G = 0, Phi_ext = omega^2 x^2/2: the central difference of x^2 and the CIC interpolation of a linear
    function are exact, so the particle feels a = -omega^2 x exactly and the KDK leapfrog of sub-step h = dt/nsub
    has the closed form x_n = x0 cos(n theta), cos(theta) = 1 - (omega h)^2/2 (v0 = 0).  nsub = 1 is the default
    scheme; more sub-steps follow the same closed form with the smaller h."""
    N, L, omega = 32, 1.0, 3.0
    X, Y, Z = grid(N, L)
    x0 = 0.2137
    for nsub in (1, 4):
        dt, nsteps = 0.05, 6
        o = oracle.Oracle(N, L, 1.0, 0.0)
        o.set_kick_terms(phi_ext=0.5 * omega ** 2 * X ** 2)
        o.set_psi(np.ones((N, N, N), complex))
        o.set_particles(np.array([[x0, 0.01, -0.02]]), np.zeros((1, 3)), 0.0)
        o.set_particle_mode(substeps=nsub)
        o.step(nsteps, dt)
        h = dt / nsub
        theta = math.acos(1 - 0.5 * (omega * h) ** 2)
        p, v = o.particles()
        assert abs(p[0, 0] - x0 * math.cos(nsteps * nsub * theta)) < 1e-12
        assert abs(p[0, 1] - 0.01) < 1e-15 and abs(p[0, 2] + 0.02) < 1e-15
    # default mode == one sub-step, bit for bit
    res = []
    for mode in (None, 1):
        o = oracle.Oracle(16, 1.0, 1.0, 1.0 / FOUR_PI)
        w = wl.small_coupled(16, dtype="c128")
        o.set_psi(w.psi); o.set_particles(w.pos, w.vel, w.mass)
        if mode:
            o.set_particle_mode(substeps=mode)
        o.step(3, w.dt)
        res.append(o.particles())
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])


def test_p15_static_particles_only_source_the_potential():
    """:particles_static: positions and velocities never change, but the particles' mass is in the
    Poisson source: the potential at step 0 equals the dynamic mode's, and psi evolves differently from a run
    without particles."""
    w = wl.small_coupled(16, dtype="c128")
    o = oracle.Oracle(w.N, w.L, w.hbar_over_m, w.G)
    o.set_psi(w.psi); o.set_particles(w.pos, w.vel, w.mass); o.set_particle_mode(static=True)
    o.step(0, 0.0)
    phi_static = o.potential()
    od = oracle.Oracle(w.N, w.L, w.hbar_over_m, w.G)
    od.set_psi(w.psi); od.set_particles(w.pos, w.vel, w.mass); od.step(0, 0.0)
    assert np.array_equal(phi_static, od.potential())
    o.step(4, w.dt)
    p, v = o.particles()
    pw = w.pos - w.L * np.floor((w.pos + w.L / 2) / w.L)
    assert np.array_equal(p, pw) and np.array_equal(v, w.vel)
    o0 = oracle.Oracle(w.N, w.L, w.hbar_over_m, w.G)
    o0.set_psi(w.psi); o0.step(4, w.dt)
    assert relerr(o.psi(), o0.psi()) > 1e-6
    # total mass in the source: sum rho dx^3 = M_psi + sum m_p
    dx3 = (w.L / w.N) ** 3
    assert abs(o.density().sum() * dx3 - (np.sum(np.abs(o.psi()) ** 2) * dx3 + np.sum(np.broadcast_to(w.mass, (len(w.pos),))))) < 1e-10


# ---------------------------------------------------------------- P16: triangular-shaped cloud (reading G30)

def test_p16_tsc_hand_computed_weights():
    N, L = 8, 2.0
    dx = L / N
    # on a node: (1/8, 3/4, 1/8) per axis, across the periodic face for node 0
    rho = oracle.tsc_deposit(N, L, np.array([[-L / 2 + 3 * dx, -L / 2, -L / 2 + 7 * dx]]), 1.0) * dx ** 3
    assert rho[3, 0, 7] == pytest.approx(0.75 ** 3) and rho[2, 7, 6] == pytest.approx(0.125 ** 3)
    assert rho[4, 1, 0] == pytest.approx(0.125 ** 3) and rho[3, 7, 0] == pytest.approx(0.75 * 0.125 ** 2)
    assert np.count_nonzero(rho) == 27 and rho.sum() == pytest.approx(1.0, rel=1e-14)
    # a quarter cell past node 5 along x (d = 1/4): 1/32, 11/16, 9/32; on nodes along y and z
    rho = oracle.tsc_deposit(N, L, np.array([[-L / 2 + 5.25 * dx, -L / 2 + 2 * dx, -L / 2 + 2 * dx]]), 1.0) * dx ** 3
    line = rho[:, 2, 2] / 0.75 ** 2
    assert line[4] == pytest.approx(1 / 32) and line[5] == pytest.approx(11 / 16) and line[6] == pytest.approx(9 / 32)
    assert np.count_nonzero(line) == 3
    # exactly half way between nodes 5 and 6: the far node's weight vanishes, 1/2 each (the cloud is continuous there)
    for eps in (0.0, -1e-9, 1e-9):
        rho = oracle.tsc_deposit(N, L, np.array([[-L / 2 + (5.5 + eps) * dx, -L / 2 + 2 * dx, -L / 2 + 2 * dx]]), 1.0) * dx ** 3
        line = rho[:, 2, 2] / 0.75 ** 2
        assert abs(line[5] - 0.5) < 2e-9 and abs(line[6] - 0.5) < 2e-9 and abs(line[4]) < 1e-16 + 1e-17 and abs(line[7]) < 1e-16


def test_p16_tsc_moments_mass_centre_and_constant_variance():
    """Per axis: sum w = 1, sum w (i - u) = 0, sum w (i - u)^2 = 1/4 for every position (what defines the scheme
    among three-point assignments)."""
    N, L = 16, 1.0
    dx = L / N
    rng = np.random.default_rng(16)
    idx = np.arange(N)
    for x in rng.uniform(-L / 2, L / 2, size=(40, 3)):
        rho = oracle.tsc_deposit(N, L, x[None, :], 3.0) * dx ** 3 / 3.0
        assert rho.min() >= 0 and rho.sum() == pytest.approx(1.0, rel=1e-13)
        for a in range(3):
            marg = rho.sum(axis=tuple(b for b in range(3) if b != a))
            u = (x[a] + L / 2) / dx
            off = (idx - u + N / 2) % N - N / 2                    # minimum-image offset in cells
            assert abs((marg * off).sum()) < 1e-12
            assert (marg * off ** 2).sum() == pytest.approx(0.25, abs=1e-12)
    p = rng.uniform(-L / 2, L / 2, size=(500, 3)); m = rng.uniform(0.1, 2.0, size=500)
    assert oracle.tsc_deposit(N, L, p, m).sum() * dx ** 3 == pytest.approx(m.sum(), rel=1e-13)


def test_p16_tsc_gather_closed_form():
    """phi = A cos(k y): node gradient g_j = A sin(k y_j) sin(k dx)/dx; three-point interpolation with
    w- + w+ = 1/4 + d^2 and w+ - w- = d gives sin(k y_j)[3/4 - d^2 + (1/4 + d^2) cos(k dx)] + d cos(k y_j) sin(k dx)."""
    N, L = 16, 1.0
    dx = L / N
    X, Y, Z = grid(N, L)
    kk = 2 * np.pi * 2 / L
    A = 0.3
    phi = A * np.cos(kk * Y)
    rng = np.random.default_rng(17)
    pos = rng.uniform(-0.5, 0.5, size=(64, 3))
    acc = oracle.tsc_gather(phi, L, pos)
    u = (pos[:, 1] + L / 2) / dx
    j = np.floor(u + 0.5); d = u - j
    yj = -L / 2 + dx * j
    expect = A * np.sin(kk * dx) / dx * (np.sin(kk * yj) * (0.75 - d ** 2 + (0.25 + d ** 2) * np.cos(kk * dx))
                                         + d * np.cos(kk * yj) * np.sin(kk * dx))
    assert np.max(np.abs(acc[:, 1] - expect)) < 1e-13
    assert np.max(np.abs(acc[:, 0])) < 1e-13 and np.max(np.abs(acc[:, 2])) < 1e-13
    assert np.max(np.abs(acc - oracle.cic_gather(phi, L, pos))) > 1e-3          # and it is not the CIC value


def test_p16_tsc_zero_self_force_momentum_and_context_switch():
    N, L, G = 16, 1.0, 1.0
    rng = np.random.default_rng(18)
    o = oracle.Oracle(N, L, 1.0, G)
    o.set_psi(np.zeros((N, N, N), complex))
    o.set_assignment(3)
    o.set_particles(rng.uniform(-0.5, 0.5, size=(1, 3)), np.zeros((1, 3)), 1.0)
    assert np.max(np.abs(o.accel())) < 1e-12
    p = rng.uniform(-0.5, 0.5, size=(200, 3)); m = rng.uniform(0.5, 1.5, size=200)
    o.set_particles(p, np.zeros((200, 3)), m)
    a3 = o.accel()
    assert np.max(np.abs((m[:, None] * a3).sum(0))) < 1e-11 * np.abs(m[:, None] * a3).sum()
    dx3 = (L / N) ** 3
    assert np.allclose(o.density(), oracle.tsc_deposit(N, L, p, m), rtol=0, atol=1e-12 / dx3)
    o.set_assignment(2)                                                        # back to CIC: the potential is refreshed
    a2 = o.accel()
    assert np.allclose(o.density(), oracle.cic_deposit(N, L, p, m), rtol=0, atol=1e-12 / dx3)
    assert np.max(np.abs(a2 - a3)) > 1e-3 * np.max(np.abs(a2))
    with pytest.raises(Exception):
        o.set_assignment(4)


# ---------------------------------------------------------------- P17: spectral kinetic energy, W, E, per-step diagnostics

def test_p17_spectral_kinetic_energy_plane_waves_closed_form():
    """psi = sum_j A_j e^{i k_j . x}, distinct lattice k_j: T_a = (mu^2/2) sum_j k_ja^2 |A_j|^2 L^3 exactly (orthogonality),
    including a Nyquist component (index N/2 <-> s = -N/2, reading G4: k^2 is sign-blind)."""
    N, L, mu = 16, 1.3, 0.7
    X, Y, Z = grid(N, L)
    ns = np.array([[2, -1, 3], [0, 5, -4], [-7, 0, 8], [1, 1, 0]])
    A = np.array([0.8, 0.5 - 0.2j, 0.3j, 1.1])
    k = 2 * np.pi * ns / L
    psi = sum(a * np.exp(1j * (kk[0] * X + kk[1] * Y + kk[2] * Z)) for a, kk in zip(A, k))
    o = oracle.Oracle(N, L, mu, 0.0)
    o.set_psi(psi)
    d = o.diagnostics()
    Ta = 0.5 * mu * mu * (np.abs(A)[:, None] ** 2 * k ** 2).sum(axis=0) * L ** 3
    assert abs(d["T"] - Ta.sum()) < 1e-10 * Ta.sum()
    assert d["W"] == 0.5 * d["V"] and abs(d["E"] - (d["T"] + d["W"])) < 1e-15 * abs(d["E"])
    # per axis, and unchanged by a drift (G = 0: the step is Eq. 18(b) alone, unit-modulus factors in k-space)
    o.set_step_diagnostics(True)
    o.step(1, 0.37 * (L / N) ** 2)
    s = o.step_diagnostics()
    for a, key in enumerate(("Tx", "Ty", "Tz")):
        assert abs(s[key] - Ta[a]) < 1e-10 * Ta.sum()
    assert abs(s["T"] - Ta.sum()) < 1e-10 * Ta.sum() and abs(o.diagnostics()["T"] - Ta.sum()) < 1e-10 * Ta.sum()
    assert abs(s["M"] - (np.abs(A) ** 2).sum() * L ** 3) < 1e-10


def test_p17_T_equals_K_plus_Q_in_the_continuum_limit():
    """T (spectral) and K + Q (central differences, Eq. 21) are the same integral (Eq. 11-12 PAPER.md:118-128 with the
    hbar^2/2m prefactors): for a smooth moving Gaussian the difference falls by 4 per halving of dx, and
    T -> (mu^2/2) (|k0|^2 + 3/(4 s^2)) M for psi = exp(-r^2/(4 s^2) + i k0 . x)."""
    L, mu, s = 1.0, 0.9, 0.07
    k0 = 2 * np.pi * np.array([2, -1, 1]) / L
    diffs = []
    for N in (16, 32, 64):
        X, Y, Z = grid(N, L)
        psi = np.exp(-(X ** 2 + Y ** 2 + Z ** 2) / (4 * s * s) + 1j * (k0[0] * X + k0[1] * Y + k0[2] * Z))
        o = oracle.Oracle(N, L, mu, 0.0)
        o.set_psi(psi)
        d = o.diagnostics()
        diffs.append(abs(d["T"] - (d["K"] + d["Q"])) / d["T"])
    assert diffs[2] < 0.02 and 3.3 < diffs[1] / diffs[2] < 4.7, diffs
    M = (2 * np.pi * s * s) ** 1.5
    assert abs(d["T"] - 0.5 * mu * mu * (k0 @ k0 + 3 / (4 * s * s)) * M) < 1e-6 * d["T"]     # spectral: exact up to the periodic images


def test_p17_energy_from_diagnostics_matches_numpy_and_is_second_order():
    """E = T + W of wdmo_diagnostics against the numpy.fft evaluation of P6 (a library routine used as a check OF
    the oracle), and its drift over a fixed time falls by 4 per halving of dt."""
    N, L, mu, G = 16, 1.0, 1.0, 200.0 / FOUR_PI
    X, Y, Z = grid(N, L)
    psi0 = (2.0 + np.exp(2j * np.pi * X) + 0.7 * np.exp(2j * np.pi * (Y - Z)) + 0.4 * np.cos(2 * np.pi * Z)).astype(complex)
    Tend, drifts = 0.02, []
    for ns in (8, 16, 32):
        o = oracle.Oracle(N, L, mu, G); o.set_psi(psi0)
        e0 = o.diagnostics()["E"]
        assert abs(e0 - total_energy(o.psi(), o.potential(), L, mu)) < 1e-12 * abs(e0)
        o.step(ns, Tend / ns)
        drifts.append(abs(o.diagnostics()["E"] - e0) / abs(e0))
    assert 3.5 < drifts[0] / drifts[1] < 4.5 and 3.5 < drifts[1] / drifts[2] < 4.5, drifts


def test_p17_step_diagnostics_are_those_of_psi2():
    """The per-step record belongs to psi_2 = the field between Eq. 18(c) and (d).  Undo the closing half kick of the
    last step by hand (psi_2 = psi exp(+i Phi dt / 2 mu), |psi| unchanged, so rho and Phi are those of the end state)
    and hand psi_2 to a fresh oracle: its diagnostics must be the record."""
    N, L, mu, G = 16, 1.3, 0.8, 60.0 / FOUR_PI
    X, Y, Z = grid(N, L)
    psi0 = (1.5 + np.exp(2j * np.pi * X / L) + 0.6 * np.exp(2j * np.pi * (2 * Y - Z) / L)).astype(complex)
    dt = 0.3 * (L / N) ** 2
    o = oracle.Oracle(N, L, mu, G); o.set_psi(psi0)
    with pytest.raises(RuntimeError):
        o.step_diagnostics()                              # nothing recorded yet
    o.set_step_diagnostics(True)
    o.step(3, dt)
    s = o.step_diagnostics()
    psi2 = o.psi() * np.exp(1j * o.potential() * dt / (2 * mu))
    o2 = oracle.Oracle(N, L, mu, G); o2.set_psi(psi2)
    d = o2.diagnostics()
    for key in ("M", "max_rho", "max_phi", "T", "W"):
        assert abs(s[key] - d[key]) <= 1e-11 * abs(d[key]), (key, s[key], d[key])
    assert abs(s["Tx"] + s["Ty"] + s["Tz"] - s["T"]) < 1e-12 * s["T"]
    # with particles W counts the whole source: 1/2 sum (|psi|^2 + rho_p) Phi
    w = wl.small_coupled(16)
    o = oracle.Oracle(w.N, w.L, w.hbar_over_m, w.G); o.set_psi(w.psi); o.set_particles(w.pos, w.vel, w.mass)
    o.set_step_diagnostics(True)
    o.step(2, w.dt)
    s = o.step_diagnostics()
    W = 0.5 * float(np.sum(o.density() * o.potential())) * (w.L / w.N) ** 3
    assert abs(s["W"] - W) < 1e-12 * abs(W)


def test_density_getter_is_that_of_the_returned_psi_with_a_layer():
    """Reading G22: wdmo_get_density = |psi|^2 of the psi the getter returns (+ particles).  With the absorbing layer of
    Alg. 1 l.17-18 that is the attenuated field; Phi stays the potential solved at l.13 from the un-attenuated one."""
    w = wl.small_coupled(16)
    o = oracle.Oracle(w.N, w.L, w.hbar_over_m, w.G)
    o.set_psi(w.psi); o.set_particles(w.pos, w.vel, w.mass)
    o.set_kick_terms(absorb_alpha=0.2 / w.dt, absorb_nb=8)
    o.step(2, w.dt)
    pos, _ = o.particles()
    want = np.abs(o.psi()) ** 2 + oracle.cic_deposit(w.N, w.L, pos, w.mass)
    assert relerr(o.density(), want) < 1e-14
    # the potential is NOT that of the attenuated field
    assert relerr(o.potential(), oracle.poisson(want, w.L, w.G)) > 1e-4
