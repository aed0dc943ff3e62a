"""Thin ctypes binding of libdns_b200.so (include/dns.h): argument marshalling only -- every step of the path
runs in the library's CUDA kernels.  There is NO CPU fallback: if the shared library is missing the import of
any entry point raises, and without a CUDA device dns_plan_create returns DNS_ECUDA (raised as DnsError).

Module-level functions carry the C names (dns_plan_create, dns_plan_bind, dns_set_state, dns_step,
dns_get_state, dns_diagnostics, ...); `Plan` is a small convenience wrapper that allocates the device
workspace with torch (PyTorch is used for device memory and streams only).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

DNS_COUETTE, DNS_POISEUILLE_CMF = 0, 1
DNS_OK, DNS_EINVAL, DNS_ENOMEM, DNS_ECUDA, DNS_ENONFINITE, DNS_ESTATE, DNS_ELIMIT = 0, -1, -2, -3, -4, -5, -6
DNS_NOALLOC_MAX_DOUBLES = 65536
DNS_FORM_CONVECTIVE, DNS_FORM_ROTATIONAL = 0, 1
DNS_COUPLING_NONE, DNS_COUPLING_STREAMWISE_MEAN = 0, 1
DNS_NCLASS = 4
CLASS_NAMES = ("fft_z_inv", "line_fft_x_products", "fft_z_fwd", "ypair_dmma")

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libdns_b200.so")
_lib = None

# every symbol include/dns.h declares, then the test / measurement hooks of include/dns_debug.h
EXPORTS = ("dns_plan_create", "dns_plan_set_form", "dns_plan_set_coupling", "dns_plan_set_exchange", "dns_add_increment",
           "dns_plan_workspace_bytes", "dns_plan_bind", "dns_set_state", "dns_step",
           "dns_step_profile", "dns_get_state", "dns_diagnostics", "dns_stats_reset", "dns_stats_accumulate", "dns_stats_get",
           "dns_launches_per_step", "dns_plan_destroy", "dns_strerror",
           "dns_lin_plan_create", "dns_lin_set_base", "dns_lin_set_state", "dns_lin_get_state", "dns_lin_step",
           "dns_lin_energy", "dns_lin_orthonormalise", "dns_lin_optimals", "dns_lin_launches_per_step",
           "dns_energy_noalloc",
           "dns_debug_fetch", "dns_debug_stage", "dns_debug_set_option", "dns_debug_fp64_peak")
EXCHANGE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)


class DnsError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: {dns_strerror(status)} ({status})")


def lib():
    """Loads libdns_b200.so; fails loudly when it has not been built (python -m paper_2306_12739_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} is missing: build it with `python -m paper_2306_12739_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(_LIB_PATH)
        vp, dp, i, d = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.dns_plan_create.argtypes = [ctypes.POINTER(vp), i, i, i, i, d, d, d, d, i]
        L.dns_plan_create.restype = i
        L.dns_plan_workspace_bytes.argtypes = [vp]
        L.dns_plan_workspace_bytes.restype = ctypes.c_size_t
        L.dns_plan_bind.argtypes = [vp, vp, ctypes.c_size_t, vp]
        L.dns_plan_bind.restype = i
        L.dns_set_state.argtypes = [vp, dp, dp, dp, dp]
        L.dns_set_state.restype = i
        L.dns_step.argtypes = [vp, i]
        L.dns_step.restype = i
        L.dns_step_profile.argtypes = [vp, i, dp]
        L.dns_step_profile.restype = i
        L.dns_get_state.argtypes = [vp, dp, dp, dp, dp]
        L.dns_get_state.restype = i
        L.dns_diagnostics.argtypes = [vp, dp]
        L.dns_diagnostics.restype = i
        L.dns_debug_fetch.argtypes = [vp, i, vp, ctypes.c_size_t]
        L.dns_debug_fetch.restype = i
        L.dns_stats_reset.argtypes = [vp]
        L.dns_stats_reset.restype = i
        L.dns_stats_accumulate.argtypes = [vp]
        L.dns_stats_accumulate.restype = i
        L.dns_stats_get.argtypes = [vp, dp, ctypes.POINTER(ctypes.c_longlong)]
        L.dns_stats_get.restype = i
        L.dns_debug_stage.argtypes = [vp, i]
        L.dns_debug_stage.restype = i
        L.dns_launches_per_step.argtypes = [vp]
        L.dns_launches_per_step.restype = i
        L.dns_plan_destroy.argtypes = [vp]
        L.dns_plan_destroy.restype = i
        L.dns_strerror.argtypes = [i]
        L.dns_strerror.restype = ctypes.c_char_p
        L.dns_plan_set_form.argtypes = [vp, i]
        L.dns_plan_set_form.restype = i
        L.dns_plan_set_coupling.argtypes = [vp, i, ctypes.c_longlong]
        L.dns_plan_set_coupling.restype = i
        L.dns_plan_set_exchange.argtypes = [vp, EXCHANGE_FN, vp]
        L.dns_plan_set_exchange.restype = i
        L.dns_add_increment.argtypes = [vp, dp, dp]
        L.dns_add_increment.restype = i
        L.dns_lin_plan_create.argtypes = [ctypes.POINTER(vp), i, i, i, i, ctypes.POINTER(i), i, d, d, d, d]
        L.dns_lin_plan_create.restype = i
        L.dns_lin_set_base.argtypes = [vp, vp, i]
        L.dns_lin_set_base.restype = i
        L.dns_lin_set_state.argtypes = [vp, dp, dp]
        L.dns_lin_set_state.restype = i
        L.dns_lin_get_state.argtypes = [vp, dp, dp]
        L.dns_lin_get_state.restype = i
        L.dns_lin_step.argtypes = [vp, i, i]
        L.dns_lin_step.restype = i
        L.dns_lin_energy.argtypes = [vp, dp]
        L.dns_lin_energy.restype = i
        L.dns_lin_orthonormalise.argtypes = [vp]
        L.dns_lin_orthonormalise.restype = i
        L.dns_lin_optimals.argtypes = [vp, i, i, dp]
        L.dns_lin_optimals.restype = i
        L.dns_lin_launches_per_step.argtypes = [vp]
        L.dns_lin_launches_per_step.restype = i
        L.dns_energy_noalloc.argtypes = [vp, dp]
        L.dns_energy_noalloc.restype = i
        L.dns_debug_set_option.argtypes = [ctypes.c_char_p, i]
        L.dns_debug_set_option.restype = i
        L.dns_debug_fp64_peak.argtypes = [i, d, ctypes.POINTER(d)]
        L.dns_debug_fp64_peak.restype = i
        _lib = L
    return _lib


def _ptr(a):
    """Address of a numpy array (host) or torch tensor (host or device); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return ctypes.c_void_p(a.ctypes.data)
    return ctypes.c_void_p(a.data_ptr())          # torch tensor


def dns_strerror(status: int) -> str:
    return lib().dns_strerror(int(status)).decode()


def dns_plan_create(Nx, Ny, Nz, E, Re, Lx, Lz, dt, flow):
    h = ctypes.c_void_p()
    st = lib().dns_plan_create(ctypes.byref(h), int(Nx), int(Ny), int(Nz), int(E), float(Re), float(Lx), float(Lz),
                               float(dt), int(flow))
    return st, h


def dns_plan_set_form(h, form: int) -> int:
    return lib().dns_plan_set_form(h, int(form))


def dns_plan_set_coupling(h, mode: int, E_total: int) -> int:
    return lib().dns_plan_set_coupling(h, int(mode), int(E_total))


def dns_plan_set_exchange(h, fn) -> int:
    """fn: an EXCHANGE_FN instance (the caller keeps it alive) or None."""
    return lib().dns_plan_set_exchange(h, fn if fn is not None else EXCHANGE_FN(0), None)


def dns_add_increment(h, dvhat, detahat) -> int:
    return lib().dns_add_increment(h, _ptr(dvhat), _ptr(detahat))


def dns_debug_set_option(name: str, value: int) -> int:
    return lib().dns_debug_set_option(name.encode(), int(value))


def dns_debug_fp64_peak(kind: int, seconds: float):
    t = ctypes.c_double(0.0)
    st = lib().dns_debug_fp64_peak(int(kind), float(seconds), ctypes.byref(t))
    return st, float(t.value)


def dns_lin_plan_create(Nx, Ny, Nz, n_list, Eg, Re, Lx, Lz, dt_lin):
    h = ctypes.c_void_p()
    arr = (ctypes.c_int * len(n_list))(*[int(n) for n in n_list])
    st = lib().dns_lin_plan_create(ctypes.byref(h), int(Nx), int(Ny), int(Nz), len(n_list), arr, int(Eg), float(Re),
                                   float(Lx), float(Lz), float(dt_lin))
    return st, h


def dns_lin_set_base(h, dns_h, member: int) -> int:
    return lib().dns_lin_set_base(h, dns_h, int(member))


def dns_lin_set_state(h, vhat, etahat) -> int:
    return lib().dns_lin_set_state(h, _ptr(vhat), _ptr(etahat))


def dns_lin_get_state(h, vhat, etahat) -> int:
    return lib().dns_lin_get_state(h, _ptr(vhat), _ptr(etahat))


def dns_lin_step(h, nsteps: int, adjoint: int) -> int:
    return lib().dns_lin_step(h, int(nsteps), int(adjoint))


def dns_lin_energy(h, out) -> int:
    return lib().dns_lin_energy(h, _ptr(out))


def dns_lin_orthonormalise(h) -> int:
    return lib().dns_lin_orthonormalise(h)


def dns_lin_optimals(h, nsteps: int, niter: int, gains) -> int:
    return lib().dns_lin_optimals(h, int(nsteps), int(niter), _ptr(gains))


def dns_energy_noalloc(h, energy_dev) -> int:
    """energy_dev: a float64 CUDA tensor of E elements that the caller made beforehand; the call itself allocates nothing
    and does not synchronise (include/dns.h).  Works on DNS and linearised plans with Ny * E <= DNS_NOALLOC_MAX_DOUBLES."""
    return lib().dns_energy_noalloc(h, _ptr(energy_dev))


def dns_lin_launches_per_step(h) -> int:
    return lib().dns_lin_launches_per_step(h)


def dns_plan_workspace_bytes(h) -> int:
    return int(lib().dns_plan_workspace_bytes(h))


def dns_plan_bind(h, dev_ptr: int, nbytes: int, stream: int = 0) -> int:
    return lib().dns_plan_bind(h, ctypes.c_void_p(dev_ptr), ctypes.c_size_t(nbytes), ctypes.c_void_p(stream))


def dns_set_state(h, vhat, etahat, U00, W00) -> int:
    return lib().dns_set_state(h, _ptr(vhat), _ptr(etahat), _ptr(U00), _ptr(W00))


def dns_step(h, nsteps: int) -> int:
    return lib().dns_step(h, int(nsteps))


def dns_step_profile(h, nsteps: int, ms: np.ndarray) -> int:
    return lib().dns_step_profile(h, int(nsteps), _ptr(ms))


def dns_get_state(h, vhat, etahat, U00, W00) -> int:
    return lib().dns_get_state(h, _ptr(vhat), _ptr(etahat), _ptr(U00), _ptr(W00))


def dns_diagnostics(h, out) -> int:
    return lib().dns_diagnostics(h, _ptr(out))


def dns_debug_fetch(h, which: int, out: np.ndarray) -> int:
    return lib().dns_debug_fetch(h, int(which), _ptr(out), ctypes.c_size_t(out.nbytes))


def dns_stats_reset(h) -> int:
    return lib().dns_stats_reset(h)


def dns_stats_accumulate(h) -> int:
    return lib().dns_stats_accumulate(h)


def dns_stats_get(h, out: np.ndarray):
    n = ctypes.c_longlong(0)
    st = lib().dns_stats_get(h, _ptr(out), ctypes.byref(n))
    return st, int(n.value)


def dns_debug_stage(h, stage: int) -> int:
    return lib().dns_debug_stage(h, int(stage))


def dns_launches_per_step(h) -> int:
    return lib().dns_launches_per_step(h)


def dns_plan_destroy(h) -> int:
    return lib().dns_plan_destroy(h)


class Plan:
    """dns_plan_create + a torch-allocated workspace bound on torch's current stream."""

    def __init__(self, Nx, Ny, Nz, E, Re, Lx, Lz, dt, flow, device="cuda:0", form=DNS_FORM_CONVECTIVE,
                 coupling=DNS_COUPLING_NONE, E_total=None, allreduce=None):
        """form / coupling: dns_plan_set_form / dns_plan_set_coupling.  allreduce (coupled ensembles sharded over ranks):
        a callable taking a float64 torch tensor that views the exchange buffer and summing it over all ranks in place
        (e.g. shard.allreduce_sum_); E_total = members over all ranks."""
        import torch

        self.shape = (int(E), int(Nx) // 2, int(Nz) - 1, int(Ny))
        self.E, self.Ny = int(E), int(Ny)
        self.device = torch.device(device)
        self.h = None
        if not torch.cuda.is_available():
            raise DnsError(DNS_ECUDA, "Plan (no CUDA device; this library has no CPU path)")
        torch.cuda.set_device(self.device)
        st, h = dns_plan_create(Nx, Ny, Nz, E, Re, Lx, Lz, dt, flow)
        if st != DNS_OK:
            raise DnsError(st, "dns_plan_create")
        self.h = h
        nbytes = dns_plan_workspace_bytes(h)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) & ~255
        self.stream = torch.cuda.current_stream(self.device)
        st = dns_plan_bind(h, base, nbytes, self.stream.cuda_stream)
        if st != DNS_OK:
            raise DnsError(st, "dns_plan_bind")
        self.workspace_bytes = nbytes
        self._exchange_cb = None
        if form != DNS_FORM_CONVECTIVE:
            self._chk(dns_plan_set_form(h, form), "dns_plan_set_form")
        if coupling != DNS_COUPLING_NONE:
            self._chk(dns_plan_set_coupling(h, coupling, int(E) if E_total is None else int(E_total)), "dns_plan_set_coupling")
            if allreduce is not None:
                ws, base_ptr = self.workspace, self.workspace.data_ptr()

                def _cb(ctx, dev_buf, count, stream):                 # marshalling only: a tensor view of the buffer
                    try:
                        off = int(dev_buf) - base_ptr
                        # the library promises the exchange is ordered on ITS stream (include/dns.h), whatever torch's
                        # current stream is in the thread that calls dns_step: make that stream current for the call
                        s = torch.cuda.ExternalStream(int(stream), device=ws.device) if stream else torch.cuda.default_stream(ws.device)
                        with torch.cuda.stream(s):
                            allreduce(ws[off:off + 8 * int(count)].view(torch.float64))
                        return 0
                    except Exception:                                  # nothing may propagate through the C frames
                        return 1
                self._exchange_cb = EXCHANGE_FN(_cb)
                self._chk(dns_plan_set_exchange(h, self._exchange_cb), "dns_plan_set_exchange")

    def _chk(self, st, where):
        if st != DNS_OK:
            raise DnsError(st, where)

    def set_state(self, vhat, etahat, U00, W00):
        if isinstance(vhat, np.ndarray):
            vhat = np.ascontiguousarray(vhat, dtype=np.complex128)
            etahat = np.ascontiguousarray(etahat, dtype=np.complex128)
            U00 = np.ascontiguousarray(U00, dtype=np.float64)
            W00 = np.ascontiguousarray(W00, dtype=np.float64)
            assert vhat.shape == self.shape and etahat.shape == self.shape
            assert U00.shape == (self.E, self.Ny) and W00.shape == (self.E, self.Ny)
        self._chk(dns_set_state(self.h, vhat, etahat, U00, W00), "dns_set_state")

    def add_increment(self, dvhat, detahat):
        if isinstance(dvhat, np.ndarray):
            dvhat = np.ascontiguousarray(dvhat, dtype=np.complex128)
            detahat = np.ascontiguousarray(detahat, dtype=np.complex128)
            assert dvhat.shape == self.shape and detahat.shape == self.shape
        self._chk(dns_add_increment(self.h, dvhat, detahat), "dns_add_increment")

    def step(self, nsteps=1):
        self._chk(dns_step(self.h, nsteps), "dns_step")

    def step_profile(self, nsteps=1):
        ms = np.zeros(DNS_NCLASS)
        self._chk(dns_step_profile(self.h, nsteps, ms), "dns_step_profile")
        return dict(zip(CLASS_NAMES, ms.tolist()))

    def get_state(self, out=None):
        if out is None:
            out = (np.empty(self.shape, np.complex128), np.empty(self.shape, np.complex128),
                   np.empty((self.E, self.Ny)), np.empty((self.E, self.Ny)))
        self._chk(dns_get_state(self.h, *out), "dns_get_state")
        return out

    def diagnostics(self):
        out = np.empty((self.E, 6))
        st = dns_diagnostics(self.h, out)
        if st not in (DNS_OK, DNS_ENONFINITE):
            raise DnsError(st, "dns_diagnostics")
        return out

    def debug_fetch(self, which):
        """Internal arrays (test hook): spectral ones come back in ABI order [E][nkx][nkz][Ny]."""
        E, nkx, nkz, Ny = self.shape
        if which == 10:
            out = np.empty((1, Ny, nkx, nkz, E), np.complex128)
            self._chk(dns_debug_fetch(self.h, which, out), "dns_debug_fetch")
            return np.ascontiguousarray(out.transpose(0, 4, 2, 3, 1))[0]
        if which in (8, 9):
            out = np.empty((Ny, E))
            self._chk(dns_debug_fetch(self.h, which, out), "dns_debug_fetch")
            return np.ascontiguousarray(out.T)
        nf = 3 if which == 4 else 1
        out = np.empty((nf, Ny, nkx, nkz, E), np.complex128)
        self._chk(dns_debug_fetch(self.h, which, out), "dns_debug_fetch")
        out = np.ascontiguousarray(out.transpose(0, 4, 2, 3, 1))
        return out if nf > 1 else out[0]

    def stats_reset(self):
        self._chk(dns_stats_reset(self.h), "dns_stats_reset")

    def stats_accumulate(self):
        self._chk(dns_stats_accumulate(self.h), "dns_stats_accumulate")

    def stats(self):
        """(mean one-point statistics [E][Ny][5] = U, <u'u'>, <v'v'>, <w'w'>, <u'v'>; number of samples)"""
        out = np.empty((self.E, self.Ny, 5))
        st, n = dns_stats_get(self.h, out)
        self._chk(st, "dns_stats_get")
        return out, n

    def energy_noalloc(self, out):
        """dns_energy_noalloc: fills `out` (float64 CUDA tensor, E elements, made by the caller beforehand) with the members'
        kinetic energies in stream order; allocates nothing and does not synchronise."""
        self._chk(dns_energy_noalloc(self.h, out), "dns_energy_noalloc")

    def debug_stage(self, stage):
        self._chk(dns_debug_stage(self.h, stage), "dns_debug_stage")

    def launches_per_step(self):
        return dns_launches_per_step(self.h)

    def close(self):
        if self.h is not None:
            dns_plan_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class LinPlan:
    """dns_lin_plan_create + a torch-allocated workspace bound on torch's current stream (linearised forward / adjoint
    ensemble).  E = len(n_list) * Eg members, [E][nkz][Ny] complex128."""

    def __init__(self, Nx, Ny, Nz, n_list, Eg, Re, Lx, Lz, dt_lin, device="cuda:0"):
        import torch

        self.E = len(n_list) * int(Eg)
        self.shape = (self.E, int(Nz) - 1, int(Ny))
        self.device = torch.device(device)
        self.h = None
        if not torch.cuda.is_available():
            raise DnsError(DNS_ECUDA, "LinPlan (no CUDA device; this library has no CPU path)")
        torch.cuda.set_device(self.device)
        st, h = dns_lin_plan_create(Nx, Ny, Nz, n_list, Eg, Re, Lx, Lz, dt_lin)
        if st != DNS_OK:
            raise DnsError(st, "dns_lin_plan_create")
        self.h = h
        nbytes = dns_plan_workspace_bytes(h)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) & ~255
        self.stream = torch.cuda.current_stream(self.device)
        st = dns_plan_bind(h, base, nbytes, self.stream.cuda_stream)
        if st != DNS_OK:
            raise DnsError(st, "dns_plan_bind")
        self.workspace_bytes = nbytes

    def _chk(self, st, where):
        if st != DNS_OK:
            raise DnsError(st, where)

    def set_base(self, dns_plan, member=0):
        self._chk(dns_lin_set_base(self.h, dns_plan.h, member), "dns_lin_set_base")

    def set_state(self, vhat, etahat):
        if isinstance(vhat, np.ndarray):
            vhat = np.ascontiguousarray(vhat, dtype=np.complex128)
            etahat = np.ascontiguousarray(etahat, dtype=np.complex128)
            assert vhat.shape == self.shape and etahat.shape == self.shape
        self._chk(dns_lin_set_state(self.h, vhat, etahat), "dns_lin_set_state")

    def get_state(self):
        out = (np.empty(self.shape, np.complex128), np.empty(self.shape, np.complex128))
        self._chk(dns_lin_get_state(self.h, *out), "dns_lin_get_state")
        return out

    def step(self, nsteps=1, adjoint=False):
        self._chk(dns_lin_step(self.h, nsteps, 1 if adjoint else 0), "dns_lin_step")

    def energy(self):
        out = np.empty(self.E)
        self._chk(dns_lin_energy(self.h, out), "dns_lin_energy")
        return out

    def energy_noalloc(self, out):
        """dns_energy_noalloc: fills `out` (float64 CUDA tensor, E elements, made by the caller beforehand) with the members'
        kinetic energies in stream order; allocates nothing and does not synchronise."""
        self._chk(dns_energy_noalloc(self.h, out), "dns_energy_noalloc")

    def orthonormalise(self):
        self._chk(dns_lin_orthonormalise(self.h), "dns_lin_orthonormalise")

    def optimals(self, nsteps, niter):
        out = np.empty(self.E)
        self._chk(dns_lin_optimals(self.h, nsteps, niter, out), "dns_lin_optimals")
        return out

    def close(self):
        if self.h is not None:
            dns_plan_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
