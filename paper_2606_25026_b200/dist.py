"""Slab-decomposed (multi-GPU) form of the step: ctypes binding of include/wdm_dist.h plus the driver that runs
the phase program and performs the exchanges between phases.

The library does every kernel of the path; this module only sequences phases and moves the exchange blocks:
with torch.distributed (NCCL all_to_all_single, one process per GPU) in `DistSim.run`, or -- for tests on one
GPU -- between several contexts of one process by device-to-device copies in `run_emulated`.  The phases of the
different ranks never wait on one another's kernels, so the emulation executes exactly the kernels of a real run.
"""
from __future__ import annotations

import ctypes as C

from . import WDM_C64, WDM_C128, WdmError, lib

R1, R2, R3, R4, S1, S2, S3, S4, S5, KICK, G1, G2 = range(12)
EXPORTS = ["wdm_dist_create", "wdm_dist_destroy", "wdm_dist_set_stream", "wdm_dist_exchange_bytes", "wdm_dist_set_buffers",
           "wdm_dist_set_psi", "wdm_dist_local_sum", "wdm_dist_set_mean", "wdm_dist_phase", "wdm_dist_get_psi",
           "wdm_dist_get_potential_t", "wdm_dist_copy_plan", "wdm_dist_last_error"]
_ready = False


def _lib():
    global _ready
    L = lib()
    if not _ready:
        vp, i, d, sz = C.c_void_p, C.c_int, C.c_double, C.c_size_t
        sig = {
            "wdm_dist_create": [C.POINTER(vp), i, d, d, d, i, i, i], "wdm_dist_destroy": [vp], "wdm_dist_set_stream": [vp, vp],
            "wdm_dist_exchange_bytes": [vp, C.POINTER(sz)], "wdm_dist_set_buffers": [vp, vp, vp], "wdm_dist_set_psi": [vp, vp],
            "wdm_dist_local_sum": [vp, C.POINTER(d)], "wdm_dist_set_mean": [vp, d],
            "wdm_dist_phase": [vp, i, d, d, C.POINTER(sz)], "wdm_dist_get_psi": [vp, vp], "wdm_dist_get_potential_t": [vp, vp],
            "wdm_dist_copy_plan": [i, i, i, C.POINTER(C.c_longlong)],
        }
        for name, args in sig.items():
            fn = getattr(L, name)
            fn.argtypes = args
            fn.restype = i
        L.wdm_dist_last_error.argtypes = [vp]
        L.wdm_dist_last_error.restype = C.c_char_p
        _ready = True
    return L


def _chk(rc, h=None):
    if rc != 0:
        raise WdmError(rc, (_lib().wdm_dist_last_error(h) or b"").decode())


def wdm_dist_copy_plan(N, world, op):
    """(n0, n1, n2, s0, s1, s2, d0, d1, d2, kmul, ksel, klim) of pack / unpack copy `op` (host logic only)."""
    out = (C.c_longlong * 12)()
    _chk(_lib().wdm_dist_copy_plan(N, world, op, out))
    return tuple(out)


class DistSim:
    """This rank's slab of one periodic box.  psi slabs are (N / world, N, N) tensors: the rank's x-planes."""

    def __init__(self, N, L=1.0, hbar_over_m=1.0, G=1.0 / (4.0 * 3.141592653589793), dtype="c64", rank=0, world=1):
        import torch
        self.torch = torch
        self.N, self.rank, self.world, self.xl = N, rank, world, N // world
        self.dtype = WDM_C64 if dtype in ("c64", WDM_C64) else WDM_C128
        self.cdtype = torch.complex64 if self.dtype == WDM_C64 else torch.complex128
        self.rdtype = torch.float32 if self.dtype == WDM_C64 else torch.float64
        self.h = C.c_void_p()
        _chk(_lib().wdm_dist_create(C.byref(self.h), N, L, hbar_over_m, G, self.dtype, rank, world))
        _chk(_lib().wdm_dist_set_stream(self.h, C.c_void_p(torch.cuda.current_stream().cuda_stream)), self.h)
        nb = C.c_size_t()
        _chk(_lib().wdm_dist_exchange_bytes(self.h, C.byref(nb)), self.h)
        self.send = torch.empty(nb.value, dtype=torch.uint8, device="cuda")
        self.recv = torch.empty(nb.value, dtype=torch.uint8, device="cuda")
        _chk(_lib().wdm_dist_set_buffers(self.h, C.c_void_p(self.send.data_ptr()), C.c_void_p(self.recv.data_ptr())), self.h)
        self.launched_phases = 0

    def close(self):
        if getattr(self, "h", None):
            _lib().wdm_dist_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- single calls of the ABI
    def phase(self, ph, dt=0.0, kick_dt=0.0):
        nb = C.c_size_t()
        _chk(_lib().wdm_dist_phase(self.h, ph, float(dt), float(kick_dt), C.byref(nb)), self.h)
        self.launched_phases += 1
        return nb.value

    def local_sum(self):
        s = C.c_double()
        _chk(_lib().wdm_dist_local_sum(self.h, C.byref(s)), self.h)
        return s.value

    def set_mean(self, mean):
        _chk(_lib().wdm_dist_set_mean(self.h, float(mean)), self.h)

    def _set_psi(self, slab):
        t = self.torch.as_tensor(slab).to(device="cuda", dtype=self.cdtype).contiguous()
        assert tuple(t.shape) == (self.xl, self.N, self.N)
        _chk(_lib().wdm_dist_set_psi(self.h, C.c_void_p(t.data_ptr())), self.h)
        self.torch.cuda.current_stream().synchronize()

    def _get_psi(self):
        out = self.torch.empty((self.xl, self.N, self.N), dtype=self.cdtype, device="cuda")
        _chk(_lib().wdm_dist_get_psi(self.h, C.c_void_p(out.data_ptr())), self.h)
        return out

    def potential_t(self):
        """Phi^T[y_l][x][z]: this rank's y-rows of the potential, x complete."""
        out = self.torch.empty((self.xl, self.N, self.N), dtype=self.rdtype, device="cuda")
        _chk(_lib().wdm_dist_get_potential_t(self.h, C.c_void_p(out.data_ptr())), self.h)
        return out

    # ---- programs: generators that yield what the ranks must do together
    #      ("a2a", bytes_per_peer) | ("sum", value) -> the global sum is sent back into the generator
    def prog_set_psi(self, slab):
        self._set_psi(slab)
        total = yield ("sum", self.local_sum())
        self.set_mean(total / float(self.N) ** 3)
        for ph in (R1, R2, R3, R4):
            nb = self.phase(ph)
            if nb:
                yield ("a2a", nb)

    def prog_step(self, nsteps, dt):
        for s in range(nsteps):
            for ph in (S1, S2, S3, S4, S5):
                nb = self.phase(ph, dt, 0.5 * dt if s == 0 else dt)
                if nb:
                    yield ("a2a", nb)
        if nsteps > 0:
            self.phase(KICK, dt, 0.5 * dt)

    def prog_get_psi(self):
        for ph in (G1, G2):
            nb = self.phase(ph)
            if nb:
                yield ("a2a", nb)

    # ---- real run: one process per GPU, torch.distributed (NCCL)
    def run(self, prog, group=None):
        import torch.distributed as dist
        reply = None
        while True:
            try:
                op, val = prog.send(reply)
            except StopIteration:
                return
            reply = None
            if op == "a2a":
                n = val * self.world
                dist.all_to_all_single(self.recv[:n], self.send[:n], group=group)
            else:
                t = self.torch.tensor([val], dtype=self.torch.float64, device="cuda")
                dist.all_reduce(t, group=group)
                reply = float(t.item())

    def set_psi(self, slab, group=None):
        self.run(self.prog_set_psi(slab), group)

    def step(self, nsteps, dt, group=None):
        self.run(self.prog_step(nsteps, dt), group)

    def psi(self, group=None):
        self.run(self.prog_get_psi(), group)
        return self._get_psi()


def run_emulated(sims, progs):
    """Drive the same program on several contexts of ONE process (one GPU) in lock step; the all-to-all is a set of
    device-to-device block copies, the all-reduce a host sum."""
    replies = [None] * len(sims)
    while True:
        ops = []
        for k, g in enumerate(progs):
            try:
                ops.append(g.send(replies[k]))
            except StopIteration:
                ops.append(None)
        if all(o is None for o in ops):
            return
        assert all(o is not None and o[0] == ops[0][0] for o in ops), "ranks diverged"
        replies = [None] * len(sims)
        if ops[0][0] == "a2a":
            nb = ops[0][1]
            assert all(o[1] == nb for o in ops)
            for d, dst in enumerate(sims):
                for s, src in enumerate(sims):
                    dst.recv[s * nb:(s + 1) * nb].copy_(src.send[d * nb:(d + 1) * nb])
        else:
            total = sum(o[1] for o in ops)
            replies = [total] * len(sims)
