"""paper_1204_1121_b200 — thin Python binding of the blipgpu C ABI (include/blipgpu.h, plus the
test / benchmark instrumentation of include/blipgpu_dev.h).

Argument marshalling only: every step of the hot path (cell map, B-spline weights, 64-row
gather + FMA, grouping, output; Eq. 6-8) runs in the sm_100a kernels of
csrc/.  torch is used for device memory and streams.  There is no CPU fallback: if
libblipgpu.so cannot be built/loaded, or no sm_100 device is present, calls raise.
"""
import ctypes
import os

import numpy as np

from . import _build

VALUE, VGL, VGH = 0, 1, 2
OK, EINVAL, ENOMEM, ECUDA, EARCH, ELIMIT = 0, -1, -2, -3, -4, -5
STATIC_MAX_POSITIONS, STATIC_MAX_BRICKS = 65536, 32768     # blipgpu_eval_static: BLIPGPU_STATIC_MAX_* of blipgpu.h

_lib = None
_c_dp = ctypes.POINTER(ctypes.c_double)
_c_ip = ctypes.POINTER(ctypes.c_int)
_c_fp = ctypes.POINTER(ctypes.c_float)
_c_llp = ctypes.POINTER(ctypes.c_longlong)

# name -> (restype, argtypes): every symbol include/blipgpu.h declares
SIGNATURES = {
    "blipgpu_create": (ctypes.c_int, [_c_dp, _c_ip, ctypes.c_int, ctypes.c_void_p, ctypes.c_int,
                                      ctypes.c_void_p, ctypes.POINTER(ctypes.c_void_p)]),
    "blipgpu_eval": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int,
                                    ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                    ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]),
    "blipgpu_eval_host": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int,
                                         ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                         ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]),
    "blipgpu_eval_contract": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int,
                                             ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p,
                                             ctypes.c_void_p, ctypes.c_void_p]),
    "blipgpu_eval_f64": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int,
                                        ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                        ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]),
    "blipgpu_set_kpoints": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "blipgpu_eval_complex": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int,
                                            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                            ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]),
    "blipgpu_eval_static": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int,
                                           ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                           ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]),
    "blipgpu_reserve": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong]),
    "blipgpu_destroy": (ctypes.c_int, [ctypes.c_void_p]),
    "blipgpu_info": (ctypes.c_int, [ctypes.c_void_p, _c_ip, _c_ip, _c_llp, _c_llp]),
    "blipgpu_set_tuning": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int]),
    "blipgpu_probe_fp32": (ctypes.c_int, [ctypes.c_void_p, _c_dp, ctypes.c_void_p]),
    "blipgpu_last_path": (ctypes.c_int, [ctypes.c_void_p]),
    "blipgpu_launch_count": (ctypes.c_longlong, [ctypes.c_void_p]),
    "blipgpu_set_profiling": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]),
    "blipgpu_last_kernel_ms": (ctypes.c_int, [ctypes.c_void_p, _c_fp, _c_fp]),
    "blipgpu_strerror": (ctypes.c_char_p, [ctypes.c_int]),
    "blipgpu_last_cuda_error": (ctypes.c_int, [ctypes.c_void_p]),
}


class BlipGpuError(RuntimeError):
    def __init__(self, code, where, cuda=0):
        self.code, self.cuda = code, cuda
        msg = lib().blipgpu_strerror(code).decode()
        super().__init__(f"{where}: {msg} (code {code}" + (f", cudaError {cuda})" if cuda else ")"))


def lib():
    """Load (building if stale) the C-ABI library.  Fails loudly — there is no other path."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(rc, where, handle=None):
    if rc != OK:
        raise BlipGpuError(rc, where, lib().blipgpu_last_cuda_error(handle))


def _stream_ptr(stream):
    import torch
    if stream is None:
        if not torch.cuda.is_available():
            return ctypes.c_void_p(0)          # the C call then reports the missing device
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(int(stream.cuda_stream))


def _ptr(x):
    """device/host pointer of a torch tensor or numpy array, or NULL."""
    if x is None:
        return ctypes.c_void_p(0)
    if isinstance(x, np.ndarray):
        return ctypes.c_void_p(x.ctypes.data)
    return ctypes.c_void_p(x.data_ptr())


# ---- the C calls, same names ---------------------------------------------------------------
def blipgpu_create(lattice, grid, norb, coeffs, stream=None):
    """coeffs: torch CUDA tensor or numpy array, fp32, [n1][n2][n3][norb] contiguous."""
    A = np.ascontiguousarray(np.asarray(lattice, dtype=np.float64).reshape(9))
    n = np.ascontiguousarray(np.asarray(grid, dtype=np.int32).reshape(3))
    on_device = 0
    if isinstance(coeffs, np.ndarray):
        assert coeffs.dtype == np.float32 and coeffs.flags.c_contiguous
    else:
        import torch
        assert coeffs.dtype == torch.float32 and coeffs.is_contiguous()
        on_device = 1 if coeffs.is_cuda else 0
    assert coeffs.size == int(n[0]) * int(n[1]) * int(n[2]) * int(norb) if isinstance(coeffs, np.ndarray) \
        else coeffs.numel() == int(n[0]) * int(n[1]) * int(n[2]) * int(norb)
    out = ctypes.c_void_p(0)
    rc = lib().blipgpu_create(A.ctypes.data_as(_c_dp), n.ctypes.data_as(_c_ip), int(norb), _ptr(coeffs),
                              on_device, _stream_ptr(stream), ctypes.byref(out))
    _check(rc, "blipgpu_create")
    return out


def blipgpu_eval(handle, positions, M, mode, val, grad, lap, ld, cell=None, stream=None):
    rc = lib().blipgpu_eval(handle, _ptr(positions), int(M), int(mode), _ptr(val), _ptr(grad), _ptr(lap),
                            int(ld), _ptr(cell), _stream_ptr(stream))
    _check(rc, "blipgpu_eval", handle)


def blipgpu_eval_host(handle, positions, M, mode, val, grad, lap, ld, cell=None, stream=None):
    rc = lib().blipgpu_eval_host(handle, _ptr(positions), int(M), int(mode), _ptr(val), _ptr(grad),
                                 _ptr(lap), int(ld), _ptr(cell), _stream_ptr(stream))
    _check(rc, "blipgpu_eval_host", handle)


def blipgpu_eval_contract(handle, positions, M, mode, d, ldd, out, cell=None, stream=None):
    rc = lib().blipgpu_eval_contract(handle, _ptr(positions), int(M), int(mode), _ptr(d), int(ldd), _ptr(out),
                                     _ptr(cell), _stream_ptr(stream))
    _check(rc, "blipgpu_eval_contract", handle)


def blipgpu_eval_f64(handle, positions, M, mode, val, grad, lap, ld, cell=None, stream=None):
    rc = lib().blipgpu_eval_f64(handle, _ptr(positions), int(M), int(mode), _ptr(val), _ptr(grad), _ptr(lap),
                                int(ld), _ptr(cell), _stream_ptr(stream))
    _check(rc, "blipgpu_eval_f64", handle)


def blipgpu_set_kpoints(handle, kpoints):
    """kpoints: [L/2][3] Cartesian k-points (rad / bohr) of the complex orbitals, or None to drop them."""
    if kpoints is None:
        _check(lib().blipgpu_set_kpoints(handle, ctypes.c_void_p(0)), "blipgpu_set_kpoints", handle)
        return
    k = np.ascontiguousarray(np.asarray(kpoints, dtype=np.float64).reshape(-1, 3))
    info = blipgpu_info(handle)
    assert k.shape[0] * 2 == info["norb"], "one k-point per complex orbital (pair of real channels)"
    _check(lib().blipgpu_set_kpoints(handle, _ptr(k)), "blipgpu_set_kpoints", handle)


def blipgpu_eval_complex(handle, positions, M, mode, val, grad, lap, ld, cell=None, stream=None):
    rc = lib().blipgpu_eval_complex(handle, _ptr(positions), int(M), int(mode), _ptr(val), _ptr(grad), _ptr(lap),
                                    int(ld), _ptr(cell), _stream_ptr(stream))
    _check(rc, "blipgpu_eval_complex", handle)


def blipgpu_eval_static(handle, positions, M, mode, val, grad, lap, ld, cell=None, stream=None):
    """blipgpu_eval for callers that may not allocate device memory while sampling (their own arena owns
    the GPU's memory, or cudaMalloc's device-wide stall would hit walkers on other streams): the grouping
    workspace is a fixed 768 KiB array inside the library instead of a cudaMalloc'ed one.  At most
    STATIC_MAX_POSITIONS positions and STATIC_MAX_BRICKS 4x4x4-cell bricks (else ELIMIT); calls on one GPU
    share that array, so they must not overlap; make the first call on a device before any stream capture."""
    rc = lib().blipgpu_eval_static(handle, _ptr(positions), int(M), int(mode), _ptr(val), _ptr(grad), _ptr(lap),
                                   int(ld), _ptr(cell), _stream_ptr(stream))
    _check(rc, "blipgpu_eval_static", handle)


def blipgpu_reserve(handle, M_max):
    _check(lib().blipgpu_reserve(handle, int(M_max)), "blipgpu_reserve", handle)


def blipgpu_destroy(handle):
    _check(lib().blipgpu_destroy(handle), "blipgpu_destroy")


def blipgpu_set_tuning(handle, path=0, nq=0):
    """path: 0 auto, 1 direct-gather kernel, 2 staged kernel (FP32 pipe), 5 staged kernel on the tensor cores;
    nq: direct kernel quads per lane (0 = default)."""
    _check(lib().blipgpu_set_tuning(handle, int(path), int(nq)), "blipgpu_set_tuning", handle)


def blipgpu_probe_fp32(handle, stream=None):
    """Measured packed-FP32 FMA rate of the device, TFLOP/s."""
    v = ctypes.c_double()
    _check(lib().blipgpu_probe_fp32(handle, ctypes.byref(v), _stream_ptr(stream)), "blipgpu_probe_fp32", handle)
    return v.value


def blipgpu_last_path(handle):
    """1 direct, 2 staged, 3 split: the gather+FMA kernel of the handle's last evaluation."""
    return int(lib().blipgpu_last_path(handle))


def blipgpu_launch_count(handle):
    return int(lib().blipgpu_launch_count(handle))


def blipgpu_set_profiling(handle, on):
    _check(lib().blipgpu_set_profiling(handle, int(bool(on))), "blipgpu_set_profiling", handle)


def blipgpu_last_kernel_ms(handle):
    """(grouping ms, gather+FMA kernel ms) of the last profiled blipgpu_eval."""
    a, b = ctypes.c_float(), ctypes.c_float()
    _check(lib().blipgpu_last_kernel_ms(handle, ctypes.byref(a), ctypes.byref(b)),
           "blipgpu_last_kernel_ms", handle)
    return a.value, b.value


def blipgpu_info(handle):
    g = (ctypes.c_int * 3)()
    L = ctypes.c_int()
    pitch, nbytes = ctypes.c_longlong(), ctypes.c_longlong()
    _check(lib().blipgpu_info(handle, g, ctypes.byref(L), ctypes.byref(pitch), ctypes.byref(nbytes)),
           "blipgpu_info", handle)
    return {"grid": tuple(g), "norb": L.value, "pitch": pitch.value, "table_bytes": nbytes.value}


# ---- convenience wrapper (allocation of outputs with torch; no arithmetic) ------------------
class BlipTable:
    def __init__(self, lattice, grid, norb, coeffs, stream=None):
        self.handle = blipgpu_create(lattice, grid, norb, coeffs, stream)
        self.norb = int(norb)
        self.ld = (self.norb + 3) // 4 * 4

    def eval(self, positions, mode=VGL, want_cell=False, stream=None):
        """positions: CUDA fp64 [M][3].  Returns (val [M][L], grad [M][3][L] | None, lap | None, cell | None)."""
        import torch
        assert positions.is_cuda and positions.dtype == torch.float64 and positions.is_contiguous()
        M = positions.shape[0]
        dev = positions.device
        val = torch.empty((M, self.ld), dtype=torch.float32, device=dev)
        grad = torch.empty((M, 3, self.ld), dtype=torch.float32, device=dev) if mode != VALUE else None
        lap = None
        if mode == VGL:
            lap = torch.empty((M, self.ld), dtype=torch.float32, device=dev)
        elif mode == VGH:
            lap = torch.empty((M, 6, self.ld), dtype=torch.float32, device=dev)      # Hessian xx yy zz xy xz yz
        cell = torch.empty((M, 3), dtype=torch.int32, device=dev) if want_cell else None
        blipgpu_eval(self.handle, positions, M, mode, val, grad, lap, self.ld, cell, stream)
        L = self.norb
        return (val[:, :L], grad[:, :, :L] if grad is not None else None,
                lap[..., :L] if lap is not None else None, cell)

    def launch_count(self):
        return blipgpu_launch_count(self.handle)

    def close(self):
        if self.handle is not None:
            blipgpu_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
