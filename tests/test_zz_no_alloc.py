"""wdm_deposit_static (include/wdm_static.h): the entry point that allocates nothing -- the deterministic particle
deposit with its fixed-point accumulator mesh in a static device array (N <= 64).

Collected last on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`, and a failure
in this side entry point must not hide the parity tests of the hot path.  The GPU test compares the new entry point with
the EXISTING path -- a wdm_ctx in deterministic deposit mode, read back with wdm_get_density over psi = 0 -- on several
calls in a row that share the static scratch, and with the CPU oracle's deposit."""
import os
import re

import numpy as np
import pytest

import oracle
import wdm_workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


# ---------------------------------------------------------------- host side (no GPU)

@pytest.fixture(scope="module")
def st():
    from paper_2606_25026_b200 import build
    build.build()
    from paper_2606_25026_b200 import static
    static._lib()
    return static


def test_static_header_symbols_are_exported(st):
    import paper_2606_25026_b200 as w
    header = open(os.path.join(ROOT, "include", "wdm_static.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(wdm_[a-z_0-9]+)\s*\(", header))
    assert declared == set(st.EXPORTS)
    for name in declared:
        assert hasattr(w.lib(), name)
        assert callable(getattr(st, name))
    assert st.wdm_static_scratch_bytes() == 64 ** 3 * 8
    assert f"#define WDM_STATIC_MAX_N {st.WDM_STATIC_MAX_N}" in header


def test_static_rejects_sizes_beyond_the_scratch_without_a_gpu(st):
    """Argument validation precedes every CUDA call, so it runs here."""
    import paper_2606_25026_b200 as w
    for N in (128, 256, 1024):
        with pytest.raises(w.WdmError) as e:
            st.wdm_deposit_static(None, None, 1.0, 10, N, 1.0, w.WDM_C64, 2, 10.0, None, stream=0)
        assert e.value.code == w.WDM_EUNSUPPORTED
        assert "exceed the static scratch" in str(e.value) and "N <= 64" in str(e.value)
    bad = [dict(N=48), dict(N=4)]
    for kw in bad:
        with pytest.raises(w.WdmError) as e:
            st.wdm_deposit_static(None, None, 1.0, 10, kw["N"], 1.0, w.WDM_C64, 2, 10.0, None, stream=0)
        assert e.value.code == w.WDM_EUNSUPPORTED
    for args in ((1.0, 10, 32, 1.0, 7, 2, 10.0), (1.0, 10, 32, 1.0, 0, 4, 10.0), (1.0, -1, 32, 1.0, 0, 2, 10.0),
                 (1.0, 10, 32, 0.0, 0, 2, 10.0), (1.0, 10, 32, 1.0, 0, 2, 0.0), (1.0, 10, 32, 1.0, 0, 2, float("nan")),
                 (float("inf"), 10, 32, 1.0, 0, 2, 1.0)):
        with pytest.raises(w.WdmError) as e:
            st.wdm_deposit_static(None, None, *args, None, stream=0)
        assert e.value.code == w.WDM_EINVAL
    with pytest.raises(w.WdmError) as e:                      # null output
        st.wdm_deposit_static(None, None, 1.0, 0, 32, 1.0, 0, 2, 1.0, None, stream=0)
    assert e.value.code == w.WDM_EINVAL and "null" in str(e.value)


def test_static_entry_point_has_no_allocating_call():
    """The source of the entry point: no cudaMalloc / cudaFree / allocating container between its braces."""
    text = open(os.path.join(ROOT, "paper_2606_25026_b200", "csrc", "wdm_particles.cu")).read()
    tail = text[text.index("static __device__ __align__(256) unsigned long long g_static_acc"):]
    for word in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "std::vector", "new ", "malloc("):
        assert word not in tail, word
    assert "cudaGetSymbolAddress((void **)&p, g_static_acc)" in tail


# ---------------------------------------------------------------- GPU: against the existing path, calls in a row

TOL = {"c64": 2e-5, "c128": 1e-12}          # rel-L2 tolerances of tests/test_sanitizer_cases.py


def existing_path(wdm, w, order, deterministic, masses=None):
    """The deposit as a wdm_ctx does it: psi = 0, so wdm_get_density returns 0 + rho_p exactly."""
    sim = wdm.Sim(w.N, w.L, w.hbar_over_m, w.G, w.dtype, max_particles=len(w.pos))
    sim.set_psi(np.zeros_like(w.psi))
    sim.set_particles(w.pos, w.vel, w.mass if masses is None else masses)
    sim.set_assignment(order)
    sim.set_deposit_mode(deterministic)
    rho = sim.density().clone()
    sim.close()
    return rho


def oracle_deposit(w, order, masses=None):
    o = oracle.Oracle(w.N, w.L, w.hbar_over_m, w.G)
    o.set_psi(np.zeros(w.psi.shape, dtype=np.complex128))
    o.set_particles(w.pos, w.vel, w.mass if masses is None else masses)
    o.set_assignment(order)
    return o.density()


def static_path(st, wdm, w, order, out, masses=None):
    import torch
    rdt = torch.float32 if w.dtype == "c64" else torch.float64
    code = wdm.WDM_C64 if w.dtype == "c64" else wdm.WDM_C128
    pos = torch.as_tensor(w.pos).to("cuda", rdt).contiguous()
    n = pos.shape[0]
    if masses is None:
        m, ms, total = None, float(w.mass), abs(float(w.mass)) * n
    else:
        m, ms = torch.as_tensor(masses).to("cuda", rdt).contiguous(), 0.0
        total = float(np.abs(np.asarray(masses, dtype=np.float64)).sum()) * 1.001
    st.wdm_deposit_static(pos, m, ms, n, w.N, w.L, code, order, total, out)
    torch.cuda.synchronize()
    return out


@pytest.mark.gpu
def test_static_deposit_matches_the_existing_path_on_calls_in_a_row(st):
    """Four calls in a row through the shared scratch -- different meshes, precisions, schemes and particle sets, the
    largest mesh first so that anything a call left behind would reach the next one -- each compared with the existing
    deterministic deposit (bit for bit: same kernels, same scale), the floating-point deposit and the oracle."""
    import torch
    assert torch.cuda.is_available()
    import paper_2606_25026_b200 as wdm
    wdm.lib()
    cases = [(wl.small_coupled(64, dtype="c64", n_particles=1 << 14, seed=81), 2),
             (wl.small_coupled(32, dtype="c64", n_particles=3000, seed=82), 2),
             (wl.small_coupled(16, dtype="c128", n_particles=257, seed=83), 3),
             (wl.small_coupled(32, dtype="c64", n_particles=500, seed=84), 3)]
    for w, order in cases:
        rdt = torch.float32 if w.dtype == "c64" else torch.float64
        out = torch.full((w.N,) * 3, float("nan"), dtype=rdt, device="cuda")     # every cell must be written
        got = static_path(st, wdm, w, order, out)
        assert bool(torch.isfinite(got).all())
        det = existing_path(wdm, w, order, True)
        assert torch.equal(got, det), (w.name, order, float((got - det).abs().max()))
        flt = existing_path(wdm, w, order, False)
        assert rel(got.cpu().numpy(), flt.cpu().numpy()) <= TOL[w.dtype]
        assert rel(got.cpu().numpy(), oracle_deposit(w, order)) <= TOL[w.dtype]
        # mass conservation: sum rho dx^3 = n m
        total = float(got.double().sum()) * (w.L / w.N) ** 3
        assert abs(total - len(w.pos) * w.mass) <= 1e-5 * len(w.pos) * w.mass


@pytest.mark.gpu
def test_static_deposit_repeats_bitwise_and_takes_particle_masses(st):
    """The same call twice in a row gives the same bits (the scratch is cleared, not accumulated into); per-particle
    masses; an empty particle set writes an all-zero mesh over whatever the output held."""
    import torch
    import paper_2606_25026_b200 as wdm
    wdm.lib()
    w = wl.small_coupled(32, dtype="c64", n_particles=2000, seed=85)
    rng = np.random.Generator(np.random.PCG64(4242))
    masses = (w.mass * rng.uniform(0.2, 3.0, size=len(w.pos))).astype(np.float32)
    outs = []
    for rep in range(2):
        out = torch.full((w.N,) * 3, float("nan"), dtype=torch.float32, device="cuda")
        outs.append(static_path(st, wdm, w, 2, out, masses=masses).clone())
    assert torch.equal(outs[0], outs[1])
    flt = existing_path(wdm, w, 2, False, masses=masses)
    assert rel(outs[0].cpu().numpy(), flt.cpu().numpy()) <= TOL["c64"]
    assert rel(outs[0].cpu().numpy(), oracle_deposit(w, 2, masses=masses)) <= TOL["c64"]
    out = torch.full((w.N,) * 3, float("nan"), dtype=torch.float32, device="cuda")
    st.wdm_deposit_static(None, None, 1.0, 0, w.N, w.L, wdm.WDM_C64, 2, 1.0, out)
    torch.cuda.synchronize()
    assert bool((out == 0).all())


@pytest.mark.gpu
def test_static_deposit_calls_no_allocator(st):
    """torch's view of the device: free memory is the same before and after a batch of calls (the driver would show a
    cudaMalloc of the call as a drop), and a call works on a side stream."""
    import torch
    import paper_2606_25026_b200 as wdm
    wdm.lib()
    w = wl.small_coupled(64, dtype="c64", n_particles=4096, seed=86)
    pos = torch.as_tensor(w.pos).to("cuda", torch.float32).contiguous()
    out = torch.empty((w.N,) * 3, dtype=torch.float32, device="cuda")
    ref = torch.empty_like(out)
    st.wdm_deposit_static(pos, None, w.mass, len(w.pos), w.N, w.L, wdm.WDM_C64, 2, w.mass * len(w.pos), ref)   # set-up call
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):                       # first use of the stream (driver-side set-up) before the reading
        torch.zeros(16, device="cuda").sum().item()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(20):
        st.wdm_deposit_static(pos, None, w.mass, len(w.pos), w.N, w.L, wdm.WDM_C64, 2, w.mass * len(w.pos), out)
    torch.cuda.synchronize()
    side.wait_stream(torch.cuda.current_stream())
    st.wdm_deposit_static(pos, None, w.mass, len(w.pos), w.N, w.L, wdm.WDM_C64, 2, w.mass * len(w.pos), out, stream=side)
    side.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    assert torch.equal(out, ref)
