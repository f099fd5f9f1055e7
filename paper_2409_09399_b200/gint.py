"""Thin Python binding of libgint.so (include/gint.h): argument marshalling only.

Every step of the path (pair list, grid batching, neighbour lists, orbital evaluation, contractions) runs
inside the library's CUDA kernels.  PyTorch is used for device memory and the current stream.  There is no
CPU fallback: if the library cannot be built/loaded, or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

STAT_NAMES = ("n_batch", "n_batch_empty", "batch_bx", "batch_by", "batch_bz", "neigh_entries", "max_nb", "max_cols",
              "padded_macs", "n_canon", "alg_incidence", "alg_sum_n", "alg_sum_n2", "nonempty_points", "smem_bytes",
              "device_bytes", "launches_vlocal", "launches_rho", "smem_eval", "tab_in_smem", "phi_bytes", "phi_scratch_bytes",
              "n_waves", "n_tiles", "tune_us")

EXPORTS = ("gint_init", "gint_n_orb", "gint_n_pairs", "gint_get_pairs", "gint_vlocal", "gint_rho", "gint_vlocal_host",
           "gint_rho_host", "gint_force_stress", "gint_force_stress_static", "gint_force_time", "gint_tune_report", "gint_stats", "gint_kernel_times", "gint_phase_times", "gint_fp64_peak",
           "gint_free", "gint_last_error")


STATIC_SCRATCH_DOUBLES = 1 << 20      # GINT_STATIC_SCRATCH_DOUBLES of include/gint.h


class GintError(RuntimeError):
    pass


def lib() -> C.CDLL:
    """Load (building first if needed) libgint.so.  Raises if that fails -- there is no other path."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.gint_last_error.restype = C.c_char_p
        for name in EXPORTS:
            if name != "gint_last_error":
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise GintError(f"libgint error {rc}: {lib().gint_last_error().decode()}")


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def fp64_peak(device: int = 0) -> dict:
    """gint_fp64_peak: DMMA / DFMA TFLOP/s of the device measured now, with the SM clock seen during the run."""
    out = (C.c_double * 4)()
    _check(lib().gint_fp64_peak(C.c_int(device), out))
    return {"dmma_tflops": float(out[0]), "dfma_tflops": float(out[1]), "sm_mhz": float(out[2]), "n_sm": int(out[3])}


FLAG_TUNE = 1 << 32       # gint_init times several grid-batch shapes; the default stays unless another is > 2 % faster


FLAG_FORCE = 1 << 33      # the batch shape must also fit gint_force_stress's shared memory


def batch_flag(bx: int, by: int, bz: int) -> int:
    return bx | (by << 8) | (bz << 16)


def phi_cap_flag(mib: int) -> int:
    """GINT_FLAG_PHI_CAP_MB: upper bound (MiB) of the context's orbital-value scratch; 0 = automatic."""
    if not 0 <= mib < (1 << 20):
        raise ValueError("phi_cap_flag: 0..1048575 MiB")
    return mib << 40


class Gint:
    """One gint_ctx: gint_init(basis tables, atoms, cell, mesh) -> vlocal / rho calls."""

    def __init__(self, basis, atom_species, atom_pos, cell, mesh, device: int = 0, flags: int = 0):
        L = lib()
        self._ctx = C.c_void_p()
        n_shell = np.ascontiguousarray(basis.n_shell, np.int32)
        shell_l = np.ascontiguousarray(basis.shell_l, np.int32)
        rcut = np.ascontiguousarray(basis.rcut, np.float64)
        n_knot = np.ascontiguousarray(basis.n_knot, np.int32)
        tab_y = np.ascontiguousarray(basis.tab_y, np.float64)
        tab_y2 = np.ascontiguousarray(basis.tab_y2, np.float64)
        sp = np.ascontiguousarray(atom_species, np.int32)
        pos = np.ascontiguousarray(atom_pos, np.float64).reshape(-1)
        cell = np.ascontiguousarray(cell, np.float64).reshape(-1)
        mesh = np.ascontiguousarray(mesh, np.int32)
        assert cell.size == 9 and mesh.size == 3 and pos.size == 3 * sp.size
        _check(L.gint_init(C.byref(self._ctx), C.c_int(int(basis.n_species)), _ip(n_shell), _ip(shell_l), _dp(rcut),
                           C.c_double(float(basis.dr)), _ip(n_knot), _dp(tab_y), _dp(tab_y2), C.c_int(sp.size), _ip(sp),
                           _dp(pos), _dp(cell), _ip(mesh), C.c_int(device), C.c_ulonglong(flags)))
        self.device = device
        self.n_atoms = int(sp.size)
        self.mesh = tuple(int(m) for m in mesh)
        self.n_points = int(np.prod(np.asarray(self.mesh, np.int64)))
        n_pairs, n_values, n_orb = C.c_longlong(), C.c_longlong(), C.c_longlong()
        _check(L.gint_n_pairs(self._ctx, C.byref(n_pairs), C.byref(n_values)))
        _check(L.gint_n_orb(self._ctx, C.byref(n_orb)))
        self.n_pairs, self.n_values, self.n_orb = n_pairs.value, n_values.value, n_orb.value

    @classmethod
    def from_workload(cls, w, device: int = 0, flags: int = 0) -> "Gint":
        return cls(w.basis, w.atom_species, w.atom_pos, w.cell, w.mesh, device=device, flags=flags)

    # ------------------------------------------------------------------ queries
    def pairs(self):
        """(A, B, R[n,3], offset[n+1]) -- lexicographic in (A, B, n1, n2, n3)."""
        n = self.n_pairs
        A = np.zeros(n, np.int32); B = np.zeros(n, np.int32); R = np.zeros((n, 3), np.int32); off = np.zeros(n + 1, np.int64)
        _check(lib().gint_get_pairs(self._ctx, _ip(A), _ip(B), _ip(R), off.ctypes.data_as(C.POINTER(C.c_longlong))))
        return A, B, R, off

    def stats(self) -> dict:
        out = np.zeros(len(STAT_NAMES), np.int64)
        _check(lib().gint_stats(self._ctx, out.ctypes.data_as(C.POINTER(C.c_longlong))))
        return dict(zip(STAT_NAMES, (int(x) for x in out)))

    def tune_report(self) -> list:
        """[(bx, by, bz, ns per mesh point or -1)] of the batch shapes the tuner tried (empty without FLAG_TUNE)."""
        out = (C.c_double * 64)(); n = C.c_int()
        _check(lib().gint_tune_report(self._ctx, C.c_int(16), out, C.byref(n)))
        return [(int(out[4 * i]), int(out[4 * i + 1]), int(out[4 * i + 2]), float(out[4 * i + 3])) for i in range(n.value)]

    def kernel_times(self) -> dict:
        """Device seconds of the main contraction kernels in the last vlocal / rho call (CUDA events in the library)."""
        out = (C.c_double * 2)()
        _check(lib().gint_kernel_times(self._ctx, out))
        return {"vlocal_main": float(out[0]), "rho_main": float(out[1])}

    def phase_times(self) -> dict:
        """Device seconds of the evaluation / tile kernels (summed over waves) in the last vlocal / rho call."""
        out = (C.c_double * 4)()
        _check(lib().gint_phase_times(self._ctx, out))
        return {"vlocal_eval": float(out[0]), "vlocal_tiles": float(out[1]), "rho_eval": float(out[2]), "rho_tiles": float(out[3])}

    # ------------------------------------------------------------------ device path
    def _stream(self):
        import torch
        return C.c_void_p(torch.cuda.current_stream(self.device).cuda_stream)

    def _dev_check(self, t, n, name):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and t.numel() == n and t.device.index == self.device):
            raise GintError(f"{name}: expected a contiguous float64 CUDA tensor of {n} elements on device {self.device}")

    def vlocal(self, V, out=None):
        """Eq. 2: V (device, n_points) -> H values (device, n_values), enqueued on torch's current stream."""
        import torch
        self._dev_check(V, self.n_points, "V")
        if out is None:
            out = torch.empty(self.n_values, dtype=torch.float64, device=V.device)
        self._dev_check(out, self.n_values, "H")
        _check(lib().gint_vlocal(self._ctx, C.c_void_p(V.data_ptr()), C.c_void_p(out.data_ptr()), self._stream()))
        return out

    def rho(self, D, out=None):
        """Eq. 3: D values (device, n_values) -> rho (device, n_points), enqueued on torch's current stream."""
        import torch
        self._dev_check(D, self.n_values, "D")
        if out is None:
            out = torch.empty(self.n_points, dtype=torch.float64, device=D.device)
        self._dev_check(out, self.n_points, "rho")
        _check(lib().gint_rho(self._ctx, C.c_void_p(D.data_ptr()), C.c_void_p(out.data_ptr()), self._stream()))
        return out

    def force_stress(self, V, D, stress: bool = True):
        """Eq. 4 / Eq. 5: V (device, n_points), D values (device, n_values) -> (F [n_atoms, 3], sigma [3, 3] or None), device tensors."""
        import torch
        self._dev_check(V, self.n_points, "V")
        self._dev_check(D, self.n_values, "D")
        F = torch.empty((self.n_atoms, 3), dtype=torch.float64, device=V.device)
        sigma = torch.empty((3, 3), dtype=torch.float64, device=V.device) if stress else None
        _check(lib().gint_force_stress(self._ctx, C.c_void_p(V.data_ptr()), C.c_void_p(D.data_ptr()), C.c_void_p(F.data_ptr()),
                                       C.c_void_p(sigma.data_ptr()) if stress else None, self._stream()))
        return F, sigma

    def force_stress_static(self, V, D, stress: bool = True):
        """gint_force_stress_static: the same F and sigma as force_stress(), for users who cannot let the library allocate device memory
        (all memory held by their own pool, a fixed MPS / MIG slice, no tolerance for cudaMalloc's device-wide stall).  The library's
        only scratch, the symmetrised copy of D, then sits in a fixed 8 MiB array inside libgint.so: n_values <= STATIC_SCRATCH_DOUBLES
        or GintError.  F and sigma are still torch tensors created here -- pass-through callers of the C ABI bring their own."""
        import torch
        self._dev_check(V, self.n_points, "V")
        self._dev_check(D, self.n_values, "D")
        F = torch.empty((self.n_atoms, 3), dtype=torch.float64, device=V.device)
        sigma = torch.empty((3, 3), dtype=torch.float64, device=V.device) if stress else None
        _check(lib().gint_force_stress_static(self._ctx, C.c_void_p(V.data_ptr()), C.c_void_p(D.data_ptr()), C.c_void_p(F.data_ptr()),
                                              C.c_void_p(sigma.data_ptr()) if stress else None, self._stream()))
        return F, sigma

    def force_time(self) -> float:
        out = C.c_double()
        _check(lib().gint_force_time(self._ctx, C.byref(out)))
        return float(out.value)

    # ------------------------------------------------------------------ host-buffer path (end to end)
    @staticmethod
    def _host_ptr(a, n, name):
        import torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != n:
                raise GintError(f"{name}: expected a contiguous float64 CPU tensor of {n} elements")
            return C.c_void_p(a.data_ptr())
        if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous and a.size == n):
            raise GintError(f"{name}: expected a contiguous float64 array of {n} elements")
        return C.c_void_p(a.ctypes.data)

    def vlocal_host(self, V_host, H_host):
        _check(lib().gint_vlocal_host(self._ctx, self._host_ptr(V_host, self.n_points, "V"),
                                      self._host_ptr(H_host, self.n_values, "H"), self._stream()))
        return H_host

    def rho_host(self, D_host, rho_host):
        _check(lib().gint_rho_host(self._ctx, self._host_ptr(D_host, self.n_values, "D"),
                                   self._host_ptr(rho_host, self.n_points, "rho"), self._stream()))
        return rho_host

    # ------------------------------------------------------------------ lifetime
    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            lib().gint_free(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
