"""Thin Python binding of libmsm_b200 (include/msm.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; PyTorch supplies device memory
and streams. There is no CPU fallback: loading fails loudly if the extension is missing, and
creating a plan fails with MSM_ERR_CUDA without a usable device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libmsm_b200.so")
_lib = None

MSM_FP64, MSM_FP32 = 0, 1
MSM_MAX_LEVELS = 32

STATUS = {0: "MSM_OK", 1: "MSM_ERR_INVALID_ARG", 2: "MSM_ERR_UNSUPPORTED", 3: "MSM_ERR_CUTOFF_TOO_LARGE",
          4: "MSM_ERR_TOO_MANY_PARTICLES", 5: "MSM_ERR_OUT_OF_BOX", 6: "MSM_ERR_NOMEM", 7: "MSM_ERR_CUDA",
          8: "MSM_ERR_SCRATCH_LIMIT"}

EXPORTS = ["msm_plan_create", "msm_plan_info", "msm_evaluate", "msm_evaluate_async", "msm_get_results",
           "msm_evaluate_host", "msm_set_profiling",
           "msm_get_stage_times", "msm_get_launch_count", "msm_debug_copy_grid", "msm_plan_destroy",
           "msm_status_string", "msm_measure_fma_peak", "msm_batch_create", "msm_evaluate_batch",
           "msm_batch_destroy", "msm_plan_create_dynamic", "msm_plan_set_box", "msm_restrict_noalloc"]


class MsmError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        super().__init__(f"{where}: {STATUS.get(int(status), status)}")


class Params(C.Structure):
    _fields_ = [("box", C.c_double * 3), ("periodic", C.c_int * 3), ("h", C.c_double), ("a", C.c_double),
                ("p", C.c_int), ("levels", C.c_int), ("precision", C.c_int), ("mu", C.c_int),
                ("max_particles", C.c_int), ("device", C.c_int)]


class PlanInfo(C.Structure):
    _fields_ = [("L_full", C.c_int), ("n_tiled", C.c_int), ("mu", C.c_int), ("omega_halfwidth", C.c_int),
                ("grid_dims", (C.c_int * 3) * MSM_MAX_LEVELS), ("grid_lo", (C.c_int * 3) * MSM_MAX_LEVELS),
                ("grid_h", (C.c_double * 3) * MSM_MAX_LEVELS), ("stencil_taps", C.c_int * MSM_MAX_LEVELS),
                ("pair_cells", C.c_int * 3), ("top_points", C.c_int), ("device_bytes", C.c_size_t)]


def lib():
    """Load libmsm_b200.so (built in-tree by paper_2510_05961_b200/build.py). Raises if missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} is missing: run `python -m paper_2510_05961_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_SO)
        vp, i, dp = C.c_void_p, C.c_int, C.POINTER(C.c_double)
        L.msm_plan_create.restype = i; L.msm_plan_create.argtypes = [C.POINTER(Params), C.POINTER(vp)]
        L.msm_plan_create_dynamic.restype = i
        L.msm_plan_create_dynamic.argtypes = [C.POINTER(Params), C.c_double, C.POINTER(vp)]
        L.msm_plan_set_box.restype = i; L.msm_plan_set_box.argtypes = [vp, dp]
        L.msm_plan_info.restype = i; L.msm_plan_info.argtypes = [vp, C.POINTER(PlanInfo)]
        L.msm_evaluate.restype = i; L.msm_evaluate.argtypes = [vp, i, vp, vp, vp, vp, dp, dp, vp]
        L.msm_evaluate_async.restype = i; L.msm_evaluate_async.argtypes = [vp, i, vp, vp, vp, vp, i, vp]
        L.msm_get_results.restype = i; L.msm_get_results.argtypes = [vp, dp, dp]
        L.msm_evaluate_host.restype = i; L.msm_evaluate_host.argtypes = [vp, i, vp, vp, vp, vp, dp, dp, vp]
        L.msm_set_profiling.restype = i; L.msm_set_profiling.argtypes = [vp, i]
        L.msm_get_stage_times.restype = i
        L.msm_get_stage_times.argtypes = [vp, C.POINTER(i), C.POINTER(C.POINTER(C.c_char_p)),
                                          C.POINTER(C.POINTER(C.c_float))]
        L.msm_get_launch_count.restype = i; L.msm_get_launch_count.argtypes = [vp, C.POINTER(i)]
        L.msm_debug_copy_grid.restype = i; L.msm_debug_copy_grid.argtypes = [vp, i, i, dp, C.c_size_t]
        L.msm_batch_create.restype = i; L.msm_batch_create.argtypes = [C.POINTER(Params), i, C.POINTER(vp)]
        L.msm_evaluate_batch.restype = i
        L.msm_evaluate_batch.argtypes = [vp, C.POINTER(i), vp, vp, vp, vp, dp, dp, vp]
        L.msm_batch_destroy.restype = None; L.msm_batch_destroy.argtypes = [vp]
        L.msm_plan_destroy.restype = None; L.msm_plan_destroy.argtypes = [vp]
        L.msm_status_string.restype = C.c_char_p; L.msm_status_string.argtypes = [i]
        L.msm_measure_fma_peak.restype = i; L.msm_measure_fma_peak.argtypes = [i, i, dp]
        ip = C.POINTER(i)
        L.msm_restrict_noalloc.restype = i
        L.msm_restrict_noalloc.argtypes = [i, i, i, ip, ip, ip, ip, ip, vp, vp, vp]
        _lib = L
    return _lib


def measure_fma_peak(kind: str = "fp32", device: int = 0) -> float:
    """TFLOP/s of back-to-back FFMA ("fp32"), DFMA ("fp64") or packed FFMA2 ("fp32x2") on the CUDA cores."""
    out = C.c_double(0.0)
    st = lib().msm_measure_fma_peak(device, {"fp32": 0, "fp64": 1, "fp32x2": 2}[kind], C.byref(out))
    if st:
        raise MsmError(st, "msm_measure_fma_peak")
    return out.value


NOALLOC_SCRATCH_BYTES = 16 << 20


def restrict_noalloc(fine, coarse, p, fine_lo, coarse_lo, periodic, stream=None):
    """msm_restrict_noalloc: coarse <- restriction of fine. Both are torch CUDA tensors indexed
    [z][y][x] (float32 or float64, contiguous, caller-owned); nothing is allocated on the device."""
    import torch
    assert fine.is_cuda and coarse.is_cuda and fine.is_contiguous() and coarse.is_contiguous()
    assert fine.dtype == coarse.dtype and fine.dim() == 3 and coarse.dim() == 3
    i3 = C.c_int * 3
    fd, cd = i3(*reversed(fine.shape)), i3(*reversed(coarse.shape))
    s = stream if stream is not None else torch.cuda.current_stream(fine.device)
    st = lib().msm_restrict_noalloc(fine.device.index, MSM_FP32 if fine.dtype == torch.float32 else MSM_FP64, int(p),
                                    fd, i3(*[int(v) for v in fine_lo]), cd, i3(*[int(v) for v in coarse_lo]),
                                    i3(*[int(bool(v)) for v in periodic]), fine.data_ptr(), coarse.data_ptr(),
                                    s.cuda_stream)
    if st:
        raise MsmError(st, "msm_restrict_noalloc")


class Plan:
    """msm_plan_create / msm_evaluate / msm_plan_destroy with torch tensors as buffers."""

    def __init__(self, box, periodic, h, a, p, levels, precision="fp64", mu=-1, max_particles=1 << 20, device=0,
                 reserve=0.0):
        """reserve > 0: room for set_box() to shrink periodic box edges by that fraction."""
        prm = Params()
        prm.box[:] = [float(b) for b in box]
        prm.periodic[:] = [int(b) for b in periodic]
        prm.h, prm.a, prm.p, prm.levels = float(h), float(a), int(p), int(levels)
        prm.precision = MSM_FP32 if precision == "fp32" else MSM_FP64
        prm.mu, prm.max_particles, prm.device = int(mu), int(max_particles), int(device)
        self._h = C.c_void_p()
        st = lib().msm_plan_create_dynamic(C.byref(prm), float(reserve), C.byref(self._h))
        if st:
            self._h = None
            raise MsmError(st, "msm_plan_create")
        self.precision = precision
        self.device = int(device)
        self.info = PlanInfo()
        lib().msm_plan_info(self._h, C.byref(self.info))

    @classmethod
    def for_workload(cls, w, precision=None, mu=-1, device=0, max_particles=None):
        return cls(w.box, w.periodic, w.h, w.a, w.p, w.levels, precision or w.precision, mu,
                   max_particles or w.n, device)

    def set_box(self, box):
        """Move the plan to new box edges (same grid counts): stencils rebuilt on the device."""
        b = (C.c_double * 3)(*[float(v) for v in box])
        st = lib().msm_plan_set_box(self._h, b)
        if st:
            raise MsmError(st, "msm_plan_set_box")
        lib().msm_plan_info(self._h, C.byref(self.info))

    def close(self):
        if getattr(self, "_h", None) and lib is not None:     # (module globals are gone at interpreter exit)
            lib().msm_plan_destroy(self._h)
            self._h = None

    __del__ = close

    @property
    def torch_dtype(self):
        import torch
        return torch.float32 if self.precision == "fp32" else torch.float64

    def grid_dims(self, level):
        return tuple(int(v) for v in self.info.grid_dims[level - 1])

    def evaluate(self, positions, charges, forces=None, potentials=None, want_energy=True, want_virial=True,
                 stream=None):
        """positions (n,3), charges (n,) CUDA tensors of the plan's dtype; forces/potentials are
        written in place if given. Returns (energy or None, virial ndarray(6) or None)."""
        import torch
        n = int(charges.shape[0])
        for t in (positions, charges, forces, potentials):
            if t is not None:
                assert t.is_cuda and t.dtype == self.torch_dtype and t.is_contiguous()
        e = C.c_double(0.0)
        w = (C.c_double * 6)()
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = lib().msm_evaluate(self._h, n, positions.data_ptr(), charges.data_ptr(),
                                forces.data_ptr() if forces is not None else None,
                                potentials.data_ptr() if potentials is not None else None,
                                C.byref(e) if want_energy else None, w if want_virial else None,
                                C.c_void_p(s.cuda_stream))
        if st:
            raise MsmError(st, "msm_evaluate")
        return (e.value if want_energy else None), (np.array(w[:]) if want_virial else None)

    def evaluate_async(self, positions, charges, forces=None, potentials=None, want_virial=False, stream=None):
        """Enqueue one evaluation on `stream` (default: torch's current stream) and return at once;
        forces / potentials are valid for work enqueued on that stream afterwards. results() waits."""
        import torch
        n = int(charges.shape[0])
        for t in (positions, charges, forces, potentials):
            if t is not None:
                assert t.is_cuda and t.dtype == self.torch_dtype and t.is_contiguous()
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = lib().msm_evaluate_async(self._h, n, positions.data_ptr(), charges.data_ptr(),
                                      forces.data_ptr() if forces is not None else None,
                                      potentials.data_ptr() if potentials is not None else None,
                                      1 if want_virial else 0, C.c_void_p(s.cuda_stream))
        if st:
            raise MsmError(st, "msm_evaluate_async")

    def results(self):
        """Wait for the last evaluation -> (energy, virial ndarray(6))."""
        e = C.c_double(0.0)
        w = (C.c_double * 6)()
        st = lib().msm_get_results(self._h, C.byref(e), w)
        if st:
            raise MsmError(st, "msm_get_results")
        return e.value, np.array(w[:])

    def evaluate_host(self, positions, charges, forces=None, potentials=None, want_virial=True, stream=None):
        """The same call on HOST buffers (numpy arrays or pinned CPU tensors of the plan's dtype)."""
        import torch
        n = int(charges.shape[0])

        def ptr(t):
            if t is None:
                return None
            return t.data_ptr() if hasattr(t, "data_ptr") else t.ctypes.data
        e = C.c_double(0.0)
        w = (C.c_double * 6)()
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = lib().msm_evaluate_host(self._h, n, ptr(positions), ptr(charges), ptr(forces), ptr(potentials),
                                     C.byref(e), w if want_virial else None, C.c_void_p(s.cuda_stream))
        if st:
            raise MsmError(st, "msm_evaluate_host")
        return e.value, (np.array(w[:]) if want_virial else None)

    def set_profiling(self, on: bool):
        lib().msm_set_profiling(self._h, 1 if on else 0)

    def stage_times(self):
        n = C.c_int(0)
        names = C.POINTER(C.c_char_p)()
        ms = C.POINTER(C.c_float)()
        lib().msm_get_stage_times(self._h, C.byref(n), C.byref(names), C.byref(ms))
        return {names[i].decode(): float(ms[i]) for i in range(n.value)}

    def launch_count(self):
        n = C.c_int(0)
        lib().msm_get_launch_count(self._h, C.byref(n))
        return n.value

    def debug_grid(self, level, kind):
        """kind 'Q' or 'E' -> float64 array [z, y, x] of the last evaluate."""
        M = self.grid_dims(level)
        out = np.zeros((M[2], M[1], M[0]))
        st = lib().msm_debug_copy_grid(self._h, level, 0 if kind == "Q" else 1,
                                       out.ctypes.data_as(C.POINTER(C.c_double)), out.size)
        if st:
            raise MsmError(st, "msm_debug_copy_grid")
        return out


class Batch:
    """msm_batch_create / msm_evaluate_batch: B systems of one geometry, tensors [B, max_particles, ...]."""

    def __init__(self, batch, box, periodic, h, a, p, levels, precision="fp64", mu=-1, max_particles=1024, device=0):
        prm = Params()
        prm.box[:] = [float(b) for b in box]
        prm.periodic[:] = [int(b) for b in periodic]
        prm.h, prm.a, prm.p, prm.levels = float(h), float(a), int(p), int(levels)
        prm.precision = MSM_FP32 if precision == "fp32" else MSM_FP64
        prm.mu, prm.max_particles, prm.device = int(mu), int(max_particles), int(device)
        self._h = C.c_void_p()
        st = lib().msm_batch_create(C.byref(prm), int(batch), C.byref(self._h))
        if st:
            self._h = None
            raise MsmError(st, "msm_batch_create")
        self.batch, self.cap, self.precision, self.device = int(batch), int(max_particles), precision, int(device)

    def close(self):
        if getattr(self, "_h", None) and lib is not None:
            lib().msm_batch_destroy(self._h)
            self._h = None

    __del__ = close

    def evaluate(self, n, positions, charges, forces=None, potentials=None, want_energy=True, want_virial=True,
                 stream=None):
        """n: B particle counts; positions [B, cap, 3], charges [B, cap] CUDA tensors of the batch's
        dtype. Returns (energies ndarray(B) or None, virials ndarray(B, 6) or None)."""
        import torch
        nn = (C.c_int * self.batch)(*[int(v) for v in n])
        e = (C.c_double * self.batch)()
        w = (C.c_double * (6 * self.batch))()
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = lib().msm_evaluate_batch(self._h, nn, positions.data_ptr(), charges.data_ptr(),
                                      forces.data_ptr() if forces is not None else None,
                                      potentials.data_ptr() if potentials is not None else None,
                                      e if want_energy else None, w if want_virial else None,
                                      C.c_void_p(s.cuda_stream))
        if st:
            raise MsmError(st, "msm_evaluate_batch")
        return (np.array(e[:]) if want_energy else None), (np.array(w[:]).reshape(self.batch, 6) if want_virial else None)


def evaluate_workload(w, precision=None, mu=-1, want_virial=True, device=0):
    """Convenience: run one workload end to end on the GPU, returning numpy results."""
    import torch
    prec = precision or w.precision
    plan = Plan.for_workload(w, prec, mu, device)
    dt = plan.torch_dtype
    dev = torch.device("cuda", device)
    pos = torch.tensor(w.positions, dtype=dt, device=dev).contiguous()
    q = torch.tensor(w.charges, dtype=dt, device=dev).contiguous()
    F = torch.zeros((w.n, 3), dtype=dt, device=dev)
    V = torch.zeros(w.n, dtype=dt, device=dev)
    U, W = plan.evaluate(pos, q, F, V, True, want_virial)
    res = {"energy": U, "forces": F.cpu().numpy().astype(np.float64),
           "potentials": V.cpu().numpy().astype(np.float64), "virial": W, "plan": plan}
    return res
