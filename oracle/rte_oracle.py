"""ctypes wrapper around the fp64 CPU oracle (oracle/rte_oracle.cpp).

TEST INFRASTRUCTURE ONLY: import this from tests/, from __graft_entry__.smoke() and from bench.py's
cpu_baseline / --impl reference legs, never from the product package.  It holds no arithmetic of its own:
every number comes from the C++ translation unit, which follows PAPER.md eq.(6)-(12) (see its header).
"""
import ctypes as C
import os

import numpy as np

from . import build_oracle

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = build_oracle.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        L.orc_num_coeffs.restype = C.c_int
        L.orc_num_coeffs.argtypes = [C.c_int, C.c_int]
        L.orc_degrees.argtypes = [C.c_int, C.c_int, ip]
        L.orc_coupling_real.restype = C.c_double
        L.orc_coupling_real.argtypes = [C.c_int, C.c_int, C.c_int, dp]
        L.orc_coupling_complex.argtypes = [C.c_int, C.c_int, C.c_int, dp, dp]
        L.orc_wavenumbers.argtypes = [C.c_int, C.c_double, dp]
        L.orc_dft.argtypes = [C.c_int, C.c_int, dp, dp, dp, dp]
        L.orc_deriv.argtypes = [dp, dp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double]
        L.orc_pml_map.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, dp,
                                  C.POINTER(C.c_ubyte)]
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                 dp, C.c_int, dp, C.c_int, dp, C.c_int, C.c_int, C.c_double, C.c_double]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_state.argtypes = [C.c_void_p, dp]
        L.orc_get_state.argtypes = [C.c_void_p, dp]
        L.orc_fluence.argtypes = [C.c_void_p, dp]
        L.orc_set_source.restype = C.c_int
        L.orc_set_source.argtypes = [C.c_void_p, dp, dp, ip, ip, C.c_int, C.c_double, C.c_double]
        L.orc_step.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_step_ssprk3.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_time_ps.restype = C.c_double
        L.orc_time_ps.argtypes = [C.c_void_p]
        L.orc_streaming.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_step_cell.argtypes = [C.c_void_p, dp, C.c_int, C.c_int, C.c_int, dp]
        L.orc_apply_operator.argtypes = [C.c_void_p, C.c_int, dp, dp]
        L.orc_source_field.argtypes = [C.c_void_p, dp]
        L.orc_solve_steady.restype = C.c_long
        L.orc_solve_steady.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_int, dp]
        L.orc_step_exp.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_step_cell_f32.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int, C.c_int, C.c_int, dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


LITERAL = 0   # the paper's recipe: complex fields, d-dim DFT, eq.(10) in k-space
PER_AXIS = 1  # T = sum_a A_a D_a psi in the real basis


def num_threads():
    return int(lib().orc_num_threads())


def set_num_threads(n):
    lib().orc_set_num_threads(int(n))


def num_coeffs(dim, N):
    return int(lib().orc_num_coeffs(dim, N))


def degrees(dim, N):
    out = np.zeros(num_coeffs(dim, N), dtype=np.int32)
    lib().orc_degrees(dim, N, _ip(out))
    return out


def coupling_real(dim, N, axis):
    """A[c, c'] with T_c = sum_c' A[c, c'] d_axis psi_c' (real basis); also returns max |imag| residue."""
    n = num_coeffs(dim, N)
    A = np.zeros((n, n))
    im = lib().orc_coupling_real(dim, N, axis, _dp(A))
    return A, float(im)


def coupling_complex(dim, N, axis):
    n = num_coeffs(dim, N)
    re = np.zeros((n, n))
    im = np.zeros((n, n))
    lib().orc_coupling_complex(dim, N, axis, _dp(re), _dp(im))
    return re + 1j * im


def wavenumbers(n, dx):
    k = np.zeros(n)
    lib().orc_wavenumbers(n, float(dx), _dp(k))
    return k


def dft(x, sign=-1):
    x = np.asarray(x, dtype=np.complex128)
    n = x.shape[0]
    re, im = _f64(x.real), _f64(x.imag)
    ore, oim = np.zeros(n), np.zeros(n)
    lib().orc_dft(n, sign, _dp(re), _dp(im), _dp(ore), _dp(oim))
    return ore + 1j * oim


def deriv(f, axis, dx):
    """Spectral derivative of a field f[z, y, x] (or f[y, x]) along axis 0=x, 1=y, 2=z."""
    f = _f64(f)
    shp = f.shape
    f3 = f.reshape((1,) + shp) if f.ndim == 2 else f
    nz, ny, nx = f3.shape
    out = np.zeros_like(f3)
    lib().orc_deriv(_dp(f3), _dp(out), nx, ny, nz, axis, float(dx))
    return out.reshape(shp)


def pml_map(dim, nx, ny, nz, W, mu_lo, mu_hi):
    mu_b = np.zeros((nz, ny, nx))
    inside = np.zeros((nz, ny, nx), dtype=np.uint8)
    lib().orc_pml_map(dim, nx, ny, nz, W, float(mu_lo), float(mu_hi), _dp(mu_b),
                      inside.ctypes.data_as(C.POINTER(C.c_ubyte)))
    return mu_b, inside


class Oracle:
    """One fp64 solver instance.  Arrays are [C, nz, ny, nx] (nz = 1 in 2-D)."""

    def __init__(self, dim, nx, ny, nz, N, dx, dt, c, mu_a, mu_s, g, pml_width=0, mu_lo=0.0, mu_hi=0.0):
        self.dim, self.nx, self.ny, self.nz, self.N = dim, nx, ny, nz, N
        self.C = num_coeffs(dim, N)
        self.G = nx * ny * nz
        args = []
        self._keep = []
        for m in (mu_a, mu_s, g):
            a = _f64(np.asarray(m, dtype=np.float64).reshape(-1))
            if a.size not in (1, self.G):
                raise ValueError("media must be a scalar or a full map")
            self._keep.append(a)
            args += [_dp(a), int(a.size == self.G)]
        self.h = lib().orc_create(dim, nx, ny, nz, N, float(dx), float(dt), float(c), *args, int(pml_width),
                                  float(mu_lo), float(mu_hi))
        if not self.h:
            raise ValueError("orc_create rejected the arguments")

    def close(self):
        if self.h:
            lib().orc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, psi):
        psi = _f64(psi).reshape(self.C, self.nz, self.ny, self.nx)
        lib().orc_set_state(self.h, _dp(psi))

    def get_state(self):
        out = np.zeros((self.C, self.nz, self.ny, self.nx))
        lib().orc_get_state(self.h, _dp(out))
        return out

    def fluence(self):
        out = np.zeros((self.nz, self.ny, self.nx))
        lib().orc_fluence(self.h, _dp(out))
        return out

    def set_source(self, w, S, origin, extent, kind, t0=0.0, sigma_t=1.0):
        w = _f64(w)
        S = _f64(S)
        org = np.asarray(origin, dtype=np.int32)
        ext = np.asarray(extent, dtype=np.int32)
        rc = lib().orc_set_source(self.h, _dp(w), _dp(S), _ip(org), _ip(ext), int(kind), float(t0), float(sigma_t))
        if rc != 0:
            raise ValueError("orc_set_source rejected the arguments")

    def step(self, nsteps=1, formulation=PER_AXIS):
        lib().orc_step(self.h, int(nsteps), int(formulation))

    def step_ssprk3(self, nsteps=1, formulation=PER_AXIS):
        """NOT the paper's integrator: three-stage SSP Runge-Kutta built from the Euler update."""
        lib().orc_step_ssprk3(self.h, int(nsteps), int(formulation))

    def step_exp(self, nsteps=1, formulation=PER_AXIS):
        """Exponential (integrating-factor) Euler step, SURVEY §8(f2) / PAPER.md:109 — not eq.(11)."""
        lib().orc_step_exp(self.h, int(nsteps), int(formulation))

    def apply_operator(self, x, formulation=PER_AXIS):
        """L x = T[x] + sigma_l x, the steady-state operator of eq.(9)."""
        x = _f64(x).reshape(self.C, self.nz, self.ny, self.nx)
        out = np.zeros_like(x)
        lib().orc_apply_operator(self.h, int(formulation), _dp(x), _dp(out))
        return out

    def source_field(self):
        """q_c(r) = w_c S(r) 1_Omega(r) (temporal factor 1)."""
        out = np.zeros((self.C, self.nz, self.ny, self.nx))
        lib().orc_source_field(self.h, _dp(out))
        return out

    def solve_steady(self, restart=30, tol=1e-10, max_restarts=200, formulation=PER_AXIS):
        """Steady state L psi = q by restarted GMRES from the current state (which becomes the solution).
        Returns (operator applications, true relative residual)."""
        rr = C.c_double(0)
        n = lib().orc_solve_steady(self.h, int(formulation), int(restart), float(tol), int(max_restarts), C.byref(rr))
        return int(n), float(rr.value)

    def time_ps(self):
        return float(lib().orc_time_ps(self.h))

    def streaming(self, formulation=PER_AXIS):
        out = np.zeros((self.C, self.nz, self.ny, self.nx))
        lib().orc_streaming(self.h, int(formulation), _dp(out))
        return out

    def step_cell(self, psi, x, y, z):
        """psi_new[:, z, y, x] after one step from state `psi` (fp64 [C,nz,ny,nx]), computed for that cell alone."""
        out = np.zeros(self.C)
        if psi.dtype == np.float32 and psi.flags["C_CONTIGUOUS"]:
            lib().orc_step_cell_f32(self.h, psi.ctypes.data_as(C.POINTER(C.c_float)), int(x), int(y), int(z), _dp(out))
        else:
            psi = _f64(psi)
            lib().orc_step_cell(self.h, _dp(psi), int(x), int(y), int(z), _dp(out))
        return out
