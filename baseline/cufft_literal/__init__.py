"""cuFFT-backed LITERAL variant of the paper's GPU implementation — a timed reference point, not the product
(complex psi_l^m, one 3-D FFT per field, eq.(10) in k-space, inverse FFT, pointwise
potential + eq.(11)).  ctypes binding over libcufft_literal.so plus the real <-> complex basis change of DESIGN.md R6
(torch ops on the device) so that its state can be compared with the [C][z][y][x] real-basis fields of the C ABI.
3-D only.  Nothing under paper_1801_06364_b200/ or oracle/ is imported here.
"""
import ctypes as C
import math
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcufft_literal.so")
_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: python baseline/cufft_literal/build.py")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.cl_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_int, C.c_float, C.c_float, C.c_float, vp, vp,
                                vp, vp]
        L.cl_destroy.argtypes = [vp]
        L.cl_destroy.restype = None
        L.cl_set_state.argtypes = [vp, vp]
        L.cl_get_state.argtypes = [vp, vp]
        L.cl_step.argtypes = [vp, C.c_int]
        L.cl_device_bytes.argtypes = [vp]
        L.cl_device_bytes.restype = C.c_ulonglong
        L.cl_own_kernel_launches.argtypes = [vp]
        L.cl_own_kernel_launches.restype = C.c_longlong
        _lib = L
    return _lib


def real_to_complex(psi_real):
    """[C,nz,ny,nx] real-basis fields (c = l*l+l+m; m>=0 cos-type a_l^m, m<0 sin-type b_l^|m|) -> complex psi_l^m
    (same index, m in [-l,l]):  psi_l^m = (-1)^m (a - i b)/sqrt2,  psi_l^-m = (a + i b)/sqrt2 (m>0),  psi_l^0 = a_l^0."""
    Cn = psi_real.shape[0]
    N = int(round(math.sqrt(Cn))) - 1
    out = torch.zeros(psi_real.shape, dtype=torch.complex64, device=psi_real.device)
    r = 1.0 / math.sqrt(2.0)
    for l in range(N + 1):
        out[l * l + l] = psi_real[l * l + l]
        for m in range(1, l + 1):
            a, b = psi_real[l * l + l + m], psi_real[l * l + l - m]
            out[l * l + l + m] = ((-1) ** m) * r * torch.complex(a, -b)
            out[l * l + l - m] = r * torch.complex(a, b)
    return out


def complex_to_real(psi_c):
    """Inverse of real_to_complex for a real radiance: a = sqrt2 Re psi_l^-m, b = sqrt2 Im psi_l^-m."""
    Cn = psi_c.shape[0]
    N = int(round(math.sqrt(Cn))) - 1
    out = torch.zeros(psi_c.shape, dtype=torch.float32, device=psi_c.device)
    s = math.sqrt(2.0)
    for l in range(N + 1):
        out[l * l + l] = psi_c[l * l + l].real
        for m in range(1, l + 1):
            out[l * l + l + m] = s * psi_c[l * l + l - m].real
            out[l * l + l - m] = s * psi_c[l * l + l - m].imag
    return out


class Solver:
    """sa/ss/gm: fp32 CUDA maps [nz,ny,nx] with the PML folded in (sa = mu_a in Omega | mu_b in the layer, ss = mu_s | 0)."""

    def __init__(self, nx, ny, nz, N, dx, dt, c, sa, ss, gm):
        self._keep = [t.contiguous() for t in (sa, ss, gm)]
        for t in self._keep:
            assert t.is_cuda and t.dtype == torch.float32 and t.numel() == nx * ny * nz
        self.h = C.c_void_p()
        self.shape = ((N + 1) ** 2, nz, ny, nx)
        rc = lib().cl_create(C.byref(self.h), nx, ny, nz, N, dx, dt, c, *[C.c_void_p(t.data_ptr()) for t in self._keep],
                             C.c_void_p(torch.cuda.current_stream().cuda_stream))
        if rc != 0:
            raise RuntimeError(f"cl_create failed ({rc}): out of device memory or bad arguments")

    def set_state(self, psi_complex):
        assert psi_complex.dtype == torch.complex64 and psi_complex.is_cuda and tuple(psi_complex.shape) == self.shape
        lib().cl_set_state(self.h, C.c_void_p(psi_complex.contiguous().data_ptr()))
        torch.cuda.current_stream().synchronize()

    def get_state(self):
        out = torch.empty(self.shape, dtype=torch.complex64, device="cuda")
        lib().cl_get_state(self.h, C.c_void_p(out.data_ptr()))
        torch.cuda.current_stream().synchronize()
        return out

    def step(self, n):
        if lib().cl_step(self.h, int(n)) != 0:
            raise RuntimeError("cl_step failed")

    def device_bytes(self):
        return int(lib().cl_device_bytes(self.h))

    def own_kernel_launches(self):
        return int(lib().cl_own_kernel_launches(self.h))

    def close(self):
        if self.h:
            lib().cl_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
