"""Small cases that draw every synchronisation path of the kernels, sized so that they also run under
compute-sanitizer (memcheck, racecheck, synccheck; see profiles/r2_sanitizer.md for the commands):

  * two-level and three-level tiles, complex64 and complex128, with fewer tiles than CTAs (static assignment only);
  * 128^3: more tiles than the first static round, so the ticket path hands out tiles dynamically;
  * coupled particles (shared-memory atomics of the deposit, the sort, both assignment schemes);
  * the extra kick terms and the external potential (separate instantiations of the z and complex-to-real sweeps).

Each case is also a parity test against the CPU oracle, so a plain `pytest -m gpu` run checks the same code.
"""
import math

import numpy as np
import pytest

import oracle
import wdm_workloads as wl

pytestmark = pytest.mark.gpu


def rel(a, b):
    a = np.asarray(a, dtype=np.complex128 if np.iscomplexobj(a) else np.float64)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


@pytest.fixture(scope="module")
def wdm():
    import torch
    assert torch.cuda.is_available()
    import paper_2606_25026_b200 as w
    w.lib()
    return w


def run_pair(wdm, w, nsteps, kick=None, order=2, substeps=1):
    npart = 0 if w.pos is None else len(w.pos)
    sim = wdm.Sim(w.N, w.L, w.hbar_over_m, w.G, w.dtype, max_particles=npart)
    o = oracle.Oracle(w.N, w.L, w.hbar_over_m, w.G)
    sim.set_psi(w.psi); o.set_psi(w.psi)
    if npart:
        sim.set_particles(w.pos, w.vel, w.mass); o.set_particles(w.pos, w.vel, w.mass)
        for x in (sim, o):
            x.set_assignment(order)
            x.set_particle_mode(substeps=substeps)
    if kick:
        sim.set_kick_terms(**kick); o.set_kick_terms(**kick)
    sim.step(nsteps, w.dt); o.step(nsteps, w.dt)
    t = (1e-12 if w.dtype == "c128" else 2e-5)
    assert rel(sim.psi().cpu().numpy(), o.psi()) <= t
    if w.G > 0 or kick:
        assert rel(sim.potential().cpu().numpy(), o.potential()) <= t
    if npart:
        p, _ = sim.particles()
        po, _ = o.particles()
        d = p.cpu().numpy().astype(np.float64) - po
        d -= w.L * np.round(d / w.L)
        assert np.abs(d).max() <= (1e-5 if w.dtype == "c64" else 1e-12) * w.L
    sim.close()


def noise(N, dtype, G=30.0):
    psi0 = (0.3 * wl.random_field(N, dtype, 500 + N) + 1.0).astype(np.complex64 if dtype == "c64" else np.complex128)
    w = wl.Workload(f"san{N}", N, dtype, 2, L=1.3, hbar_over_m=0.8, G=G, psi=psi0)
    w.dt = 0.2 * (w.L / N) ** 2
    return w


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_san_32_static_tiles(wdm, dtype):
    run_pair(wdm, noise(32, dtype), 2)


def test_san_config1(wdm):
    run_pair(wdm, wl.config1(), 2)


def test_san_128_ticket_path(wdm):
    run_pair(wdm, noise(128, "c64"), 2)


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("order", [2, 3])
def test_san_16_coupled(wdm, dtype, order):
    run_pair(wdm, wl.small_coupled(16, dtype=dtype), 3, order=order, substeps=2 if order == 3 else 1)


def test_san_kick_terms(wdm):
    N = 32
    w = noise(N, "c64")
    x = -0.5 * w.L + (w.L / N) * np.arange(N)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    ext = (5.0 * np.cos(2 * math.pi * X / w.L) + 3.0 * (Y * Y + Z * Z)).astype(np.float32)
    run_pair(wdm, w, 2, kick=dict(kappa=-3.0, phi_ext=ext, absorb_alpha=0.1 / w.dt, absorb_nb=10))


# ---------------------------------------------------------------- stand-ins for racecheck / memcheck
# compute-sanitizer is closed on the GPU pool this repository is measured on (profiles/r2_sanitizer.md).  Two properties
# that a race or an out-of-bounds store would break are checked directly instead.

@pytest.mark.parametrize("dtype,N", [("c64", 128), ("c128", 64), ("c64", 256), ("c128", 128)])
def test_runs_are_bitwise_reproducible(wdm, dtype, N):
    """Pure SPE steps use no atomics: whichever CTA draws a tile (dynamic tickets), the tile's arithmetic is the same, so
    repeated runs from the same input must agree BIT FOR BIT.  A buffer refilled before its last reader left, or read
    before its copy landed, shows up as a run-to-run difference."""
    import torch
    w = noise(N, dtype)
    outs = []
    for rep in range(3):
        sim = wdm.Sim(w.N, w.L, w.hbar_over_m, w.G, w.dtype)
        sim.set_psi(w.psi)
        sim.step(6, w.dt)
        outs.append((sim.psi().clone(), sim.potential().clone()))
        sim.close()
    for psi, phi in outs[1:]:
        assert torch.equal(psi, outs[0][0]) and torch.equal(phi, outs[0][1])


@pytest.mark.parametrize("dtype,N,npart", [("c64", 32, 0), ("c128", 32, 0), ("c64", 16, 257), ("c64", 128, 0)])
def test_no_store_outside_the_workspace(wdm, dtype, N, npart):
    """The context lives in a caller workspace; guard bands on both sides must come back untouched, and a workspace of
    exactly wdm_workspace_bytes must suffice (no hidden allocation for the grid)."""
    import torch
    w = wl.small_coupled(N, dtype=dtype, n_particles=npart) if npart else noise(N, dtype)
    code = wdm.WDM_C64 if dtype == "c64" else wdm.WDM_C128
    need = wdm.wdm_workspace_bytes(N, code, npart)
    guard = 1 << 20
    buf = torch.full((need + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda")
    ws = buf[guard:guard + need]
    h = wdm.wdm_create_ws(N, w.L, w.hbar_over_m, w.G, code, npart, ws)
    cdt = torch.complex64 if dtype == "c64" else torch.complex128
    rdt = torch.float32 if dtype == "c64" else torch.float64
    wdm.wdm_set_psi(h, torch.as_tensor(w.psi).to("cuda", cdt).contiguous())
    if npart:
        wdm.wdm_set_particles(h, npart, torch.as_tensor(w.pos).to("cuda", rdt).contiguous(),
                              torch.as_tensor(w.vel).to("cuda", rdt).contiguous(), None, float(w.mass))
    wdm.wdm_step(h, 4, w.dt)
    out = torch.empty((N,) * 3, dtype=cdt, device="cuda")
    wdm.wdm_get_psi(h, out)
    torch.cuda.synchronize()
    wdm.wdm_destroy(h)
    assert bool((buf[:guard] == 0xA5).all()) and bool((buf[guard + need:] == 0xA5).all())
    assert bool(torch.isfinite(torch.view_as_real(out)).all())
