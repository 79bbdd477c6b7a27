"""Slab-decomposed step (include/wdm_dist.h) against the CPU oracle, on ONE GPU: `world` contexts in one process run the
phase program in lock step and the all-to-all exchanges are device-to-device block copies (paper_2606_25026_b200.dist.
run_emulated).  No phase waits on another rank's kernel, so these are exactly the kernels and index maps of a real
multi-GPU run; only the NCCL call itself is not exercised (no multi-GPU node in this build: unmeasured on hardware)."""
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
def wd():
    import torch
    assert torch.cuda.is_available()
    import paper_2606_25026_b200.dist as wd
    wd._lib()
    return wd


def gather_psi(wd, sims):
    wd.run_emulated(sims, [s.prog_get_psi() for s in sims])
    return np.concatenate([s._get_psi().cpu().numpy() for s in sims], axis=0)


def gather_phi(sims):
    # Phi^T[y_l][x][z] per rank -> Phi[x][y][z]
    return np.concatenate([s.potential_t().cpu().numpy().transpose(1, 0, 2) for s in sims], axis=1)


@pytest.mark.parametrize("dtype,N,world,G", [("c128", 32, 1, 30.0), ("c128", 32, 2, 30.0), ("c128", 32, 4, 30.0), ("c64", 64, 4, 30.0),
                                             ("c64", 128, 8, 30.0), ("c64", 128, 4, 30.0), ("c128", 64, 8, 30.0), ("c64", 32, 2, 0.0),
                                             ("c64", 256, 8, 30.0), ("c64", 16, 16, 30.0)])
def test_slab_decomposed_step_matches_oracle(wd, dtype, N, world, G):
    L, mu = 1.3, 0.8
    psi0 = (0.3 * wl.random_field(N, dtype, 60 + N) + 1.0).astype(np.complex64 if dtype == "c64" else np.complex128)
    dt = 0.2 * (L / N) ** 2
    xl = N // world
    sims = [wd.DistSim(N, L, mu, G, dtype, r, world) for r in range(world)]
    o = oracle.Oracle(N, L, mu, G)
    o.set_psi(psi0)
    wd.run_emulated(sims, [s.prog_set_psi(psi0[r * xl:(r + 1) * xl]) for r, s in enumerate(sims)])
    t10 = 1e-12 if dtype == "c128" else 2e-5
    if G > 0:
        assert rel(gather_phi(sims), o.potential()) <= t10               # refresh: Phi of the initial state
    assert np.array_equal(gather_psi(wd, sims), psi0)                     # two transposes bring psi back bit for bit
    for nsteps in (3, 1):                                                 # a second call: closing kick applied, then reopened
        wd.run_emulated(sims, [s.prog_step(nsteps, dt) for s in sims])
        o.step(nsteps, dt)
        assert rel(gather_psi(wd, sims), o.psi()) <= t10
        if G > 0:
            assert rel(gather_phi(sims), o.potential()) <= t10
    for s in sims:
        s.close()


def test_slab_decomposed_equals_single_gpu_path(wd):
    """Same kernels on slabs: the decomposed run agrees with the single-GPU library to a few roundings."""
    import torch
    import paper_2606_25026_b200 as wdm
    N, world = 128, 4
    psi0 = (0.3 * wl.random_field(N, "c64", 9) + 1.0).astype(np.complex64)
    dt = (1.0 / N) ** 2 / 6
    sims = [wd.DistSim(N, 1.0, 1.0, 1.0 / (4 * math.pi), "c64", r, world) for r in range(world)]
    xl = N // world
    wd.run_emulated(sims, [s.prog_set_psi(psi0[r * xl:(r + 1) * xl]) for r, s in enumerate(sims)])
    wd.run_emulated(sims, [s.prog_step(4, dt) for s in sims])
    one = wdm.Sim(N, dtype="c64")
    one.set_psi(psi0)
    one.step(4, dt)
    a, b = gather_psi(wd, sims), one.psi().cpu().numpy()
    assert np.abs(a - b).max() <= 2e-6 * np.abs(b).max()
    assert np.abs(gather_phi(sims) - one.potential().cpu().numpy()).max() <= 2e-5 * float(one.potential().abs().max())
    for s in sims:
        s.close()
    one.close()


def test_dist_errors(wd):
    import paper_2606_25026_b200 as wdm
    with pytest.raises(wdm.WdmError) as e:
        wd.DistSim(64, world=3)
    assert e.value.code == wdm.WDM_EUNSUPPORTED
    s = wd.DistSim(32, world=2, rank=1)
    with pytest.raises(wdm.WdmError) as e:
        s.phase(wd.S1, 1e-4, 5e-5)                                        # no psi, no potential yet
    assert e.value.code == wdm.WDM_ESTATE
    s.close()
