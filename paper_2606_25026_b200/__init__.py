"""paper_2606_25026_b200 -- B200 (sm_100a) split-step Schroedinger-Poisson + CIC particle step.

Thin ctypes binding of libwdm.so (include/wdm.h): the functions below have the C ABI's names and only
marshal arguments (torch tensors -> device pointers).  Every step of the path runs in the CUDA kernels
of csrc/; there is no CPU or PyTorch fallback -- a missing or unloadable library raises.
PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libwdm.so")

WDM_C64, WDM_C128 = 0, 1
WDM_OK, WDM_EINVAL, WDM_EUNSUPPORTED, WDM_ENOMEM, WDM_ECUDA, WDM_ESTATE = range(6)
_CODE = {1: "WDM_EINVAL", 2: "WDM_EUNSUPPORTED", 3: "WDM_ENOMEM", 4: "WDM_ECUDA", 5: "WDM_ESTATE"}

_lib = None


class WdmError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"{_CODE.get(code, code)}: {text}")
        self.code = code


def lib():
    """Load libwdm.so (built by paper_2606_25026_b200.build / __graft_entry__.build()).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_25026_b200.build` (needs nvcc); "
                              "there is no fallback path")
        L = C.CDLL(LIB_PATH)
        vp, i, d, ll, sz = C.c_void_p, C.c_int, C.c_double, C.c_longlong, C.c_size_t
        sig = {
            "wdm_workspace_bytes": [i, i, ll, C.POINTER(sz)],
            "wdm_create": [C.POINTER(vp), i, d, d, d, i],
            "wdm_create_ws": [C.POINTER(vp), i, d, d, d, i, ll, vp, sz],
            "wdm_destroy": [vp], "wdm_set_stream": [vp, vp],
            "wdm_set_psi": [vp, vp], "wdm_set_psi_host": [vp, vp],
            "wdm_set_particles": [vp, ll, vp, vp, vp, d], "wdm_set_particles_host": [vp, ll, vp, vp, vp, d],
            "wdm_step": [vp, i, d], "wdm_run_host": [vp, vp, i, d, vp],
            "wdm_get_psi": [vp, vp], "wdm_get_density": [vp, vp], "wdm_get_potential": [vp, vp],
            "wdm_get_particles": [vp, vp, vp],
            "wdm_get_psi_host": [vp, vp], "wdm_get_density_host": [vp, vp], "wdm_get_potential_host": [vp, vp],
            "wdm_get_particles_host": [vp, vp, vp],
            "wdm_launch_count": [vp, C.POINTER(ll)], "wdm_set_profiling": [vp, i],
            "wdm_set_kick_terms": [vp, d, vp, d, i], "wdm_get_diagnostics": [vp, C.POINTER(d)], "wdm_set_step_diagnostics": [vp, i], "wdm_get_step_diagnostics": [vp, C.POINTER(d)], "wdm_set_particle_mode": [vp, i, i], "wdm_set_assignment": [vp, i], "wdm_set_deposit_mode": [vp, i], "wdm_get_assignment": [vp, C.POINTER(i)],
            "wdm_kernel_stats": [vp, C.POINTER(i), C.POINTER(C.c_char_p), C.POINTER(ll), C.POINTER(d)],
        }
        for name, args in sig.items():
            fn = getattr(L, name)
            fn.argtypes = args
            fn.restype = i
        L.wdm_last_error.argtypes = [vp]
        L.wdm_last_error.restype = C.c_char_p
        _lib = L
    return _lib


EXPORTS = ["wdm_workspace_bytes", "wdm_create", "wdm_create_ws", "wdm_destroy", "wdm_set_stream", "wdm_set_psi",
           "wdm_set_psi_host", "wdm_set_particles", "wdm_set_particles_host", "wdm_step", "wdm_run_host",
           "wdm_get_psi", "wdm_get_density", "wdm_get_potential", "wdm_get_particles", "wdm_get_psi_host",
           "wdm_get_density_host", "wdm_get_potential_host", "wdm_get_particles_host", "wdm_launch_count",
           "wdm_set_profiling", "wdm_kernel_stats", "wdm_last_error", "wdm_set_kick_terms", "wdm_get_diagnostics", "wdm_set_particle_mode", "wdm_set_assignment", "wdm_get_assignment", "wdm_set_deposit_mode", "wdm_set_step_diagnostics", "wdm_get_step_diagnostics"]


def _chk(rc, h=None):
    if rc != WDM_OK:
        raise WdmError(rc, (lib().wdm_last_error(h) or b"").decode())


def _ptr(t):
    """device (or host) pointer of a contiguous torch tensor / numpy array; None -> NULL"""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        assert t.is_contiguous()
        return C.c_void_p(t.data_ptr())
    assert t.flags["C_CONTIGUOUS"]
    return C.c_void_p(t.ctypes.data)


# ---- the C ABI, same names, tensors instead of raw pointers -------------------------------------------

def wdm_workspace_bytes(N, dtype, max_particles=0):
    out = C.c_size_t()
    _chk(lib().wdm_workspace_bytes(N, dtype, max_particles, C.byref(out)))
    return out.value


def wdm_create(N, L, hbar_over_m, G, dtype):
    h = C.c_void_p()
    _chk(lib().wdm_create(C.byref(h), N, L, hbar_over_m, G, dtype))
    return h


def wdm_create_ws(N, L, hbar_over_m, G, dtype, max_particles, workspace):
    h = C.c_void_p()
    _chk(lib().wdm_create_ws(C.byref(h), N, L, hbar_over_m, G, dtype, max_particles, _ptr(workspace),
                             workspace.numel() * workspace.element_size()))
    return h


def wdm_destroy(h):
    _chk(lib().wdm_destroy(h))


def wdm_set_stream(h, cuda_stream):
    _chk(lib().wdm_set_stream(h, C.c_void_p(cuda_stream)), h)


def wdm_set_psi(h, psi):
    _chk(lib().wdm_set_psi(h, _ptr(psi)), h)


def wdm_set_psi_host(h, psi):
    _chk(lib().wdm_set_psi_host(h, _ptr(psi)), h)


def wdm_set_particles(h, n, pos, vel, mass=None, mass_scalar=0.0):
    _chk(lib().wdm_set_particles(h, n, _ptr(pos), _ptr(vel), _ptr(mass), mass_scalar), h)


def wdm_set_particles_host(h, n, pos, vel, mass=None, mass_scalar=0.0):
    _chk(lib().wdm_set_particles_host(h, n, _ptr(pos), _ptr(vel), _ptr(mass), mass_scalar), h)


def wdm_step(h, nsteps, dt):
    _chk(lib().wdm_step(h, nsteps, dt), h)


def wdm_run_host(h, psi_in, nsteps, dt, psi_out):
    _chk(lib().wdm_run_host(h, _ptr(psi_in), nsteps, dt, _ptr(psi_out)), h)


def wdm_get_psi(h, out):
    _chk(lib().wdm_get_psi(h, _ptr(out)), h)


def wdm_get_density(h, out):
    _chk(lib().wdm_get_density(h, _ptr(out)), h)


def wdm_get_potential(h, out):
    _chk(lib().wdm_get_potential(h, _ptr(out)), h)


def wdm_get_particles(h, pos, vel):
    _chk(lib().wdm_get_particles(h, _ptr(pos), _ptr(vel)), h)


def wdm_get_psi_host(h, out):
    _chk(lib().wdm_get_psi_host(h, _ptr(out)), h)


def wdm_get_density_host(h, out):
    _chk(lib().wdm_get_density_host(h, _ptr(out)), h)


def wdm_get_potential_host(h, out):
    _chk(lib().wdm_get_potential_host(h, _ptr(out)), h)


def wdm_get_particles_host(h, pos, vel):
    _chk(lib().wdm_get_particles_host(h, _ptr(pos), _ptr(vel)), h)


def wdm_launch_count(h):
    out = C.c_longlong()
    _chk(lib().wdm_launch_count(h, C.byref(out)), h)
    return out.value


def wdm_set_kick_terms(h, kappa=0.0, phi_ext=None, absorb_alpha=0.0, absorb_nb=50):
    """phi_ext: device tensor of N^3 reals or None; the library keeps the pointer (caller keeps the tensor alive)."""
    _chk(lib().wdm_set_kick_terms(h, float(kappa), _ptr(phi_ext), float(absorb_alpha), int(absorb_nb)), h)


def wdm_set_particle_mode(h, substeps=1, static=False):
    _chk(lib().wdm_set_particle_mode(h, int(substeps), 1 if static else 0), h)


def wdm_set_assignment(h, order=2):
    """2: cloud-in-cell, 3: triangular-shaped cloud (deposit and gather alike)."""
    _chk(lib().wdm_set_assignment(h, int(order)), h)


def wdm_set_deposit_mode(h, deterministic=False):
    """True: fixed-point deposit, bit-identical from run to run (debugging mode)."""
    _chk(lib().wdm_set_deposit_mode(h, 1 if deterministic else 0), h)


def wdm_get_assignment(h):
    out = C.c_int(0)
    _chk(lib().wdm_get_assignment(h, C.byref(out)), h)
    return out.value


def wdm_get_diagnostics(h):
    """dict(M, max_rho, max_phi, V, K, Q, dt_max, T, W, E) of the current state (synchronises)."""
    out = (C.c_double * 12)()
    _chk(lib().wdm_get_diagnostics(h, out), h)
    return dict(zip(("M", "max_rho", "max_phi", "V", "K", "Q", "dt_max", "T", "W", "E"), list(out)[:10]))


def wdm_set_step_diagnostics(h, on=True):
    _chk(lib().wdm_set_step_diagnostics(h, 1 if on else 0), h)


def wdm_get_step_diagnostics(h):
    """dict(M, max_rho, max_phi, T, W, Tx, Ty, Tz) of the field between the drift and the closing kick of the last step."""
    out = (C.c_double * 8)()
    _chk(lib().wdm_get_step_diagnostics(h, out), h)
    return dict(zip(("M", "max_rho", "max_phi", "T", "W", "Tx", "Ty", "Tz"), list(out)))


def wdm_set_profiling(h, on):
    _chk(lib().wdm_set_profiling(h, 1 if on else 0), h)


def wdm_kernel_stats(h):
    """{kernel name: (timed launches, summed ms)} since the last call (CUDA events on the context stream)."""
    n = C.c_int(32)
    names = (C.c_char_p * 32)()
    cnt = (C.c_longlong * 32)()
    ms = (C.c_double * 32)()
    _chk(lib().wdm_kernel_stats(h, C.byref(n), names, cnt, ms), h)
    return {names[i].decode(): (cnt[i], ms[i]) for i in range(n.value)}


def wdm_last_error(h=None):
    return (lib().wdm_last_error(h) or b"").decode()


# ---- convenience wrapper: owns the context and takes its device memory from PyTorch ------------------

class Sim:
    """One periodic box on the current CUDA device.  All device memory comes from one torch allocation
    handed to wdm_create_ws; work is enqueued on torch's current stream at construction."""

    def __init__(self, N, L=1.0, hbar_over_m=1.0, G=1.0 / (4.0 * 3.141592653589793), dtype="c64", max_particles=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_25026_b200 needs a CUDA device (sm_100a); there is no CPU path")
        self.torch = torch
        self.N, self.L = N, L
        self.dtype = WDM_C64 if dtype in ("c64", WDM_C64) else WDM_C128
        self.cdtype = torch.complex64 if self.dtype == WDM_C64 else torch.complex128
        self.rdtype = torch.float32 if self.dtype == WDM_C64 else torch.float64
        nbytes = wdm_workspace_bytes(N, self.dtype, max_particles)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        self.h = wdm_create_ws(N, L, hbar_over_m, G, self.dtype, max_particles, self.workspace)
        wdm_set_stream(self.h, torch.cuda.current_stream().cuda_stream)
        self.n_particles = 0

    def close(self):
        if getattr(self, "h", None):
            wdm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev(self, a, dt):
        t = self.torch.as_tensor(a)
        return t.to(device="cuda", dtype=dt).contiguous()

    def set_psi(self, psi):
        t = self._dev(psi, self.cdtype)
        assert tuple(t.shape) == (self.N,) * 3
        wdm_set_psi(self.h, t)
        self.torch.cuda.current_stream().synchronize()      # t may be a temporary

    def set_particles(self, pos, vel, mass):
        p, v = self._dev(pos, self.rdtype), self._dev(vel, self.rdtype)
        n = p.shape[0]
        if self.torch.is_tensor(mass) or hasattr(mass, "shape") and getattr(mass, "shape", ()) != ():
            m = self._dev(mass, self.rdtype)
            wdm_set_particles(self.h, n, p, v, m, 0.0)
        else:
            wdm_set_particles(self.h, n, p, v, None, float(mass))
        self.n_particles = n
        self.torch.cuda.current_stream().synchronize()

    def set_kick_terms(self, kappa=0.0, phi_ext=None, absorb_alpha=0.0, absorb_nb=50):
        self._phi_ext = None if phi_ext is None else self._dev(phi_ext, self.rdtype)     # kept alive here
        wdm_set_kick_terms(self.h, kappa, self._phi_ext, absorb_alpha, absorb_nb)

    def set_particle_mode(self, substeps=1, static=False):
        wdm_set_particle_mode(self.h, substeps, static)

    def set_assignment(self, order=2):
        wdm_set_assignment(self.h, order)

    def set_deposit_mode(self, deterministic=False):
        wdm_set_deposit_mode(self.h, deterministic)

    def assignment(self):
        return wdm_get_assignment(self.h)

    def diagnostics(self):
        return wdm_get_diagnostics(self.h)

    def set_step_diagnostics(self, on=True):
        wdm_set_step_diagnostics(self.h, on)

    def step_diagnostics(self):
        return wdm_get_step_diagnostics(self.h)

    def step(self, nsteps, dt):
        wdm_step(self.h, nsteps, dt)

    def psi(self):
        out = self.torch.empty((self.N,) * 3, dtype=self.cdtype, device="cuda")
        wdm_get_psi(self.h, out)
        return out

    def density(self):
        out = self.torch.empty((self.N,) * 3, dtype=self.rdtype, device="cuda")
        wdm_get_density(self.h, out)
        return out

    def potential(self):
        out = self.torch.empty((self.N,) * 3, dtype=self.rdtype, device="cuda")
        wdm_get_potential(self.h, out)
        return out

    def particles(self):
        pos = self.torch.empty((self.n_particles, 3), dtype=self.rdtype, device="cuda")
        vel = self.torch.empty((self.n_particles, 3), dtype=self.rdtype, device="cuda")
        wdm_get_particles(self.h, pos, vel)
        return pos, vel
