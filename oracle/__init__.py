"""CPU oracle (test infrastructure, NOT the product): ctypes binding of oracle/wdmo.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2606_25026_b200 and shares no code with it.
Everything is float64 on the host; complex arrays are numpy complex128.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wdmo.c")
_LIB = os.path.join(_HERE, "libwdmo.so")
_lib = None

OK, EINVAL, EUNSUPPORTED, ENOMEM, ESTATE = 0, 1, 2, 3, 5


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp oracle/wdmo.c -> oracle/libwdmo.so (rebuilt when the source is newer)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu99", "-fPIC", "-shared", "-fopenmp", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp, ll, i, d, vp = C.POINTER(C.c_double), C.c_longlong, C.c_int, C.c_double, C.c_void_p
        sig = {
            "wdmo_fft1d": [i, dp, dp, i], "wdmo_dft1d_direct": [i, dp, dp, i],
            "wdmo_fft3": [i, dp, dp, i], "wdmo_dft3_direct": [i, dp, dp, i],
            "wdmo_poisson": [i, d, d, dp, dp],
            "wdmo_cic_deposit": [i, d, ll, dp, dp, dp], "wdmo_cic_gather": [i, d, dp, ll, dp, dp],
            "wdmo_tsc_deposit": [i, d, ll, dp, dp, dp], "wdmo_tsc_gather": [i, d, dp, ll, dp, dp], "wdmo_set_assignment": [vp, i],
            "wdmo_create": [C.POINTER(vp), i, d, d, d], "wdmo_destroy": [vp],
            "wdmo_set_psi": [vp, dp], "wdmo_set_particles": [vp, ll, dp, dp, dp, d],
            "wdmo_step": [vp, i, d], "wdmo_get_psi": [vp, dp], "wdmo_get_density": [vp, dp],
            "wdmo_get_potential": [vp, dp], "wdmo_get_particles": [vp, dp, dp],
            "wdmo_get_accel": [vp, dp], "wdmo_threads": [],
            "wdmo_set_kick_terms": [vp, d, dp, d, i], "wdmo_diagnostics": [vp, dp], "wdmo_set_particle_mode": [vp, i, i],
            "wdmo_set_step_diagnostics": [vp, i], "wdmo_step_diagnostics": [vp, dp],
        }
        for name, args in sig.items():
            fn = getattr(_lib, name)
            fn.argtypes = args
            fn.restype = C.c_int
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _check(rc, what):
    if rc != OK:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def threads() -> int:
    return lib().wdmo_threads()


def fft1d(x, sign=-1):
    x = _c128(x); out = np.empty_like(x)
    _check(lib().wdmo_fft1d(x.size, _dp(x), _dp(out), sign), "fft1d")
    return out


def dft1d_direct(x, sign=-1):
    x = _c128(x); out = np.empty_like(x)
    _check(lib().wdmo_dft1d_direct(x.size, _dp(x), _dp(out), sign), "dft1d_direct")
    return out


def fft3(a, sign=-1):
    a = _c128(a); out = np.empty_like(a)
    _check(lib().wdmo_fft3(a.shape[0], _dp(a), _dp(out), sign), "fft3")
    return out


def dft3_direct(a, sign=-1):
    a = _c128(a); out = np.empty_like(a)
    _check(lib().wdmo_dft3_direct(a.shape[0], _dp(a), _dp(out), sign), "dft3_direct")
    return out


def poisson(rho, L, G):
    rho = _f64(rho); phi = np.empty_like(rho)
    _check(lib().wdmo_poisson(rho.shape[0], L, G, _dp(rho), _dp(phi)), "poisson")
    return phi


def cic_deposit(N, L, pos, mass):
    pos = _f64(pos); mass = _f64(np.broadcast_to(mass, (pos.shape[0],)))
    rho = np.zeros((N, N, N))
    _check(lib().wdmo_cic_deposit(N, L, pos.shape[0], _dp(pos), _dp(mass), _dp(rho)), "cic_deposit")
    return rho


def cic_gather(phi, L, pos):
    phi = _f64(phi); pos = _f64(pos); acc = np.empty_like(pos)
    _check(lib().wdmo_cic_gather(phi.shape[0], L, _dp(phi), pos.shape[0], _dp(pos), _dp(acc)), "cic_gather")
    return acc


def tsc_deposit(N, L, pos, mass):
    """Triangular-shaped-cloud deposit (27 nodes; reading G30)."""
    pos = _f64(pos); mass = _f64(np.broadcast_to(mass, (pos.shape[0],)))
    rho = np.zeros((N, N, N))
    _check(lib().wdmo_tsc_deposit(N, L, pos.shape[0], _dp(pos), _dp(mass), _dp(rho)), "tsc_deposit")
    return rho


def tsc_gather(phi, L, pos):
    phi = _f64(phi); pos = _f64(pos); acc = np.empty_like(pos)
    _check(lib().wdmo_tsc_gather(phi.shape[0], L, _dp(phi), pos.shape[0], _dp(pos), _dp(acc)), "tsc_gather")
    return acc


class Oracle:
    """Same call sequence as the product's Sim (wdm_create / set / step / get), float64 on the host."""

    def __init__(self, N, L=1.0, hbar_over_m=1.0, G=1.0 / (4.0 * np.pi)):
        self._h = C.c_void_p()
        self.N = N
        self.np_ = 0
        rc = lib().wdmo_create(C.byref(self._h), N, L, hbar_over_m, G)
        if rc != OK:
            self._h = None
            raise RuntimeError(f"wdmo_create failed with code {rc}")

    def close(self):
        if getattr(self, "_h", None):
            lib().wdmo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_psi(self, psi):
        psi = _c128(psi)
        assert psi.shape == (self.N,) * 3
        _check(lib().wdmo_set_psi(self._h, _dp(psi)), "set_psi")

    def set_particles(self, pos, vel, mass):
        pos = _f64(pos); vel = _f64(vel)
        self.np_ = pos.shape[0]
        if np.ndim(mass) == 0:
            _check(lib().wdmo_set_particles(self._h, self.np_, _dp(pos), _dp(vel), None, float(mass)), "set_particles")
        else:
            m = _f64(mass)
            _check(lib().wdmo_set_particles(self._h, self.np_, _dp(pos), _dp(vel), _dp(m), 0.0), "set_particles")

    def set_kick_terms(self, kappa=0.0, phi_ext=None, absorb_alpha=0.0, absorb_nb=50):
        """V = Phi + phi_ext + kappa |psi|^2 in the kicks (Eq. 13-14); absorbing layer of Eq. 22 after every step."""
        pe = None if phi_ext is None else _f64(phi_ext)
        _check(lib().wdmo_set_kick_terms(self._h, float(kappa), _dp(pe), float(absorb_alpha), int(absorb_nb)), "set_kick_terms")

    def step(self, nsteps, dt):
        _check(lib().wdmo_step(self._h, nsteps, dt), "step")

    def psi(self):
        out = np.empty((self.N,) * 3, dtype=np.complex128)
        _check(lib().wdmo_get_psi(self._h, _dp(out)), "get_psi")
        return out

    def density(self):
        out = np.empty((self.N,) * 3)
        _check(lib().wdmo_get_density(self._h, _dp(out)), "get_density")
        return out

    def potential(self):
        out = np.empty((self.N,) * 3)
        _check(lib().wdmo_get_potential(self._h, _dp(out)), "get_potential")
        return out

    def set_particle_mode(self, substeps=1, static=False):
        """Leapfrog sub-steps per SPE step; static: particles only source the potential."""
        _check(lib().wdmo_set_particle_mode(self._h, int(substeps), 1 if static else 0), "set_particle_mode")

    def set_assignment(self, order=2):
        """2 = cloud-in-cell (G12-G13), 3 = triangular-shaped cloud (G30), for deposit and gather alike."""
        _check(lib().wdmo_set_assignment(self._h, int(order)), "set_assignment")

    def diagnostics(self):
        """dict(M, max_rho, max_phi, V, K, Q, dt_max, T, W, E) of the current state (Sect. 3.5-3.6): K, Q by central
        differences, T spectral, W = V/2, E = T + W."""
        out = np.zeros(12)
        _check(lib().wdmo_diagnostics(self._h, _dp(out)), "diagnostics")
        return dict(zip(("M", "max_rho", "max_phi", "V", "K", "Q", "dt_max", "T", "W", "E"), out[:10]))

    def set_step_diagnostics(self, on=True):
        _check(lib().wdmo_set_step_diagnostics(self._h, 1 if on else 0), "set_step_diagnostics")

    def step_diagnostics(self):
        """dict(M, max_rho, max_phi, T, W, Tx, Ty, Tz) of the field between the drift and the closing half kick of the
        last step (recorded while set_step_diagnostics is on)."""
        out = np.zeros(8)
        _check(lib().wdmo_step_diagnostics(self._h, _dp(out)), "step_diagnostics")
        return dict(zip(("M", "max_rho", "max_phi", "T", "W", "Tx", "Ty", "Tz"), out))

    def particles(self):
        pos = np.empty((self.np_, 3)); vel = np.empty((self.np_, 3))
        _check(lib().wdmo_get_particles(self._h, _dp(pos), _dp(vel)), "get_particles")
        return pos, vel

    def accel(self):
        acc = np.empty((self.np_, 3))
        _check(lib().wdmo_get_accel(self._h, _dp(acc)), "get_accel")
        return acc
