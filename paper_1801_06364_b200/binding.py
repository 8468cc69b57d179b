"""Thin ctypes binding over the C ABI of include/rte.h — argument marshalling only.

Every function has the name and meaning of its C counterpart; torch tensors are passed as device pointers
(`data_ptr()`), PyTorch supplies device memory and the stream, nothing else.  There is NO fallback: if the CUDA
library has not been built (python paper_1801_06364_b200/build.py) importing this module raises.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librte_b200.so")

RTE_OK, RTE_EINVAL, RTE_ENOMEM, RTE_ECUDA, RTE_ESTATE, RTE_EUNSUPPORTED = 0, 1, 2, 3, 4, 5
_CODES = {0: "RTE_OK", 1: "RTE_EINVAL", 2: "RTE_ENOMEM", 3: "RTE_ECUDA", 4: "RTE_ESTATE", 5: "RTE_EUNSUPPORTED"}


class rte_grid(C.Structure):
    _fields_ = [("dim", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int)]


class rte_pml(C.Structure):
    _fields_ = [("width", C.c_int), ("mu_lo", C.c_float), ("mu_hi", C.c_float)]


class rte_media(C.Structure):
    _fields_ = [("mu_a", C.c_void_p), ("mu_s", C.c_void_p), ("g", C.c_void_p),
                ("mu_a_is_map", C.c_int), ("mu_s_is_map", C.c_int), ("g_is_map", C.c_int)]


class RteError(RuntimeError):
    def __init__(self, code, text=""):
        super().__init__(f"{_CODES.get(code, code)}: {text}")
        self.code = code


if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python paper_1801_06364_b200/build.py` "
                      "(there is no CPU or PyTorch fallback)")

_lib = C.CDLL(LIB_PATH)
_vp, _i, _f = C.c_void_p, C.c_int, C.c_float
_i3 = C.POINTER(C.c_int)
_lib.rte_num_coeffs.argtypes = [_i, _i]
_lib.rte_coupling_table.argtypes = [_i, _i, _i, C.POINTER(C.c_double)]
_lib.rte_storage_layout.argtypes = [_i, _i, C.POINTER(_i), C.POINTER(_i), C.POINTER(_i)]
_lib.rte_workspace_bytes.argtypes = [C.POINTER(rte_grid), _i, C.POINTER(C.c_size_t)]
_lib.rte_create.argtypes = [C.POINTER(_vp), C.POINTER(rte_grid), _i, _f, _f, _f, C.POINTER(rte_media),
                            C.POINTER(rte_pml), _vp, C.c_size_t, _vp]
_lib.rte_destroy.argtypes = [_vp]
_lib.rte_destroy.restype = None
for _n in ("rte_set_state", "rte_get_state", "rte_set_state_host", "rte_get_state_host", "rte_fluence",
           "rte_fluence_host"):
    getattr(_lib, _n).argtypes = [_vp, _vp]
_lib.rte_reset_time.argtypes = [_vp]
_lib.rte_set_source.argtypes = [_vp, C.POINTER(C.c_float), _vp, _i3, _i3, _i, _f, _f]
_lib.rte_set_source_host.argtypes = [_vp, C.POINTER(C.c_float), _vp, _i3, _i3, _i, _f, _f]
_lib.rte_step.argtypes = [_vp, _i]
_lib.rte_step_ssprk3.argtypes = [_vp, _i]
_lib.rte_step_exp.argtypes = [_vp, _i]
_lib.rte_extra_workspace_bytes.argtypes = [C.POINTER(rte_grid), _i, _i, C.POINTER(C.c_size_t)]
_lib.rte_set_extra_workspace.argtypes = [_vp, _vp, C.c_size_t]
_lib.rte_stable_dt.argtypes = [_i, _i, _i, _f, _f, _f, _f, _f, C.POINTER(C.c_double), C.POINTER(C.c_double)]
_lib.rte_apply_operator.argtypes = [_vp, _vp, _vp]
_lib.rte_solve_steady.argtypes = [_vp, _i, C.c_double, _i, _i, _f, C.POINTER(_i), C.POINTER(C.c_double)]
_lib.rte_step_profile.argtypes = [_vp, _i, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
_lib.rte_fluence_change.argtypes = [_vp, C.POINTER(C.c_double)]
_lib.rte_time_ps.argtypes = [_vp, C.POINTER(C.c_double)]
_lib.rte_energy.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
_lib.rte_sync.argtypes = [_vp]
_lib.rte_last_error.argtypes = [_vp]
_lib.rte_last_error.restype = C.c_char_p
_lib.rte_launch_count.argtypes = [_vp, C.POINTER(C.c_longlong)]
_lib.rte_media_ellipsoids.argtypes = [C.POINTER(rte_grid), _f, C.POINTER(C.c_float), _i, C.POINTER(C.c_float), _vp,
                                      _vp, _vp, _vp]
_lib.rte_media_lognormal.argtypes = [C.POINTER(rte_grid), _f, C.c_uint64, _f, _f, _f, _vp, _vp, _vp]
_lib.rte_media_lognormal_noalloc.argtypes = [C.POINTER(rte_grid), _f, C.c_uint64, _f, _f, _f, _vp, _vp]
_lib.rte_pml_profile.argtypes = [C.POINTER(rte_grid), C.POINTER(rte_pml), _vp, _vp, _vp]

EXPORTED = ["rte_num_coeffs", "rte_coupling_table", "rte_storage_layout", "rte_workspace_bytes", "rte_create", "rte_destroy",
            "rte_set_state", "rte_get_state", "rte_set_state_host", "rte_get_state_host", "rte_reset_time",
            "rte_set_source", "rte_set_source_host", "rte_step", "rte_step_ssprk3", "rte_step_exp", "rte_step_profile",
            "rte_extra_workspace_bytes", "rte_set_extra_workspace", "rte_stable_dt", "rte_apply_operator",
            "rte_solve_steady", "rte_fluence", "rte_fluence_host",
            "rte_fluence_change", "rte_energy", "rte_time_ps", "rte_sync", "rte_last_error", "rte_launch_count",
            "rte_media_ellipsoids", "rte_media_lognormal", "rte_media_lognormal_noalloc", "rte_pml_profile"]


def _check(rc, ctx=None):
    if rc != RTE_OK:
        msg = _lib.rte_last_error(ctx)
        raise RteError(rc, msg.decode() if msg else "")


def _stream_ptr(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _dev(t, dtype=torch.float32):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"expected a contiguous CUDA tensor of {dtype}")
    return C.c_void_p(t.data_ptr())


def _grid(grid):
    if isinstance(grid, rte_grid):
        return grid
    dim, nx, ny, nz = grid
    return rte_grid(int(dim), int(nx), int(ny), int(nz))


# ---- host-only helpers -------------------------------------------------------------------------------------------
def rte_num_coeffs(dim, N):
    return int(_lib.rte_num_coeffs(dim, N))


def rte_coupling_table(dim, N, axis):
    import numpy as np
    n = rte_num_coeffs(dim, N)
    if n < 0:
        raise RteError(RTE_EINVAL, "bad dim/N")
    A = np.zeros((n, n))
    _check(_lib.rte_coupling_table(dim, N, axis, A.ctypes.data_as(C.POINTER(C.c_double))))
    return A


def rte_storage_layout(dim, N):
    """(ext_of_slot[Cp] int array, (cost_natural, cost_chosen, cost_ideal)) — host only, see include/rte.h."""
    import numpy as np
    cp = _i(0)
    _check(_lib.rte_storage_layout(dim, N, C.byref(cp), None, None))
    ext = np.zeros(cp.value, dtype=np.int32)
    cost = (_i * 3)()
    _check(_lib.rte_storage_layout(dim, N, C.byref(cp), ext.ctypes.data_as(C.POINTER(_i)), cost))
    return ext, tuple(cost)


def rte_workspace_bytes(grid, N):
    out = C.c_size_t(0)
    g = _grid(grid)
    _check(_lib.rte_workspace_bytes(C.byref(g), N, C.byref(out)))
    return int(out.value)


# ---- life cycle ----------------------------------------------------------------------------------------------------
class Context:
    """Owns the opaque rte_ctx*, the workspace tensor and the media tensors' lifetimes (nothing else)."""

    def __init__(self, handle, keep):
        self.handle = handle
        self._keep = keep

    def __del__(self):
        try:
            rte_destroy(self)
        except Exception:
            pass


def rte_create(grid, N, dx_mm, dt_ps, c_mm_per_ps, mu_a, mu_s, g, pml=(0, 0.0, 0.0), stream=None, device=None):
    """mu_a/mu_s/g: python floats or fp32 CUDA tensors with G elements ([z][y][x])."""
    if not torch.cuda.is_available():
        raise RteError(RTE_ECUDA, "no CUDA device (this library has no CPU fallback)")
    dev = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
    g_ = _grid(grid)
    G = g_.nx * g_.ny * g_.nz
    keep, ptrs, flags = [], [], []
    for m in (mu_a, mu_s, g):
        if isinstance(m, torch.Tensor):
            t = m.to(device=dev, dtype=torch.float32).contiguous().reshape(-1)
            if t.numel() not in (1, G):
                raise RteError(RTE_EINVAL, "media map must have nx*ny*nz elements")
        else:
            t = torch.tensor([float(m)], dtype=torch.float32, device=dev)
        keep.append(t)
        ptrs.append(t.data_ptr())
        flags.append(int(t.numel() == G and G > 1))
    media = rte_media(ptrs[0], ptrs[1], ptrs[2], flags[0], flags[1], flags[2])
    pm = rte_pml(int(pml[0]), float(pml[1]), float(pml[2]))
    nbytes = rte_workspace_bytes(g_, N)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    keep.append(ws)
    h = C.c_void_p()
    with torch.cuda.device(dev):
        rc = _lib.rte_create(C.byref(h), C.byref(g_), int(N), float(dx_mm), float(dt_ps), float(c_mm_per_ps),
                             C.byref(media), C.byref(pm), C.c_void_p(ws.data_ptr()), nbytes, _stream_ptr(stream))
    _check(rc, None)
    ctx = Context(h, keep)
    ctx.grid, ctx.N, ctx.C, ctx.G, ctx.device = g_, int(N), rte_num_coeffs(g_.dim, N), G, dev
    return ctx


def rte_destroy(ctx):
    if ctx.handle:
        _lib.rte_destroy(ctx.handle)
        ctx.handle = None


# ---- state / source / hot path ---------------------------------------------------------------------------------------
def rte_set_state(ctx, psi_dev):
    _check(_lib.rte_set_state(ctx.handle, _dev(psi_dev)), ctx.handle)


def rte_get_state(ctx, psi_dev):
    _check(_lib.rte_get_state(ctx.handle, _dev(psi_dev)), ctx.handle)


def _host(t):
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("expected a contiguous fp32 host tensor")
    return C.c_void_p(t.data_ptr())


def rte_set_state_host(ctx, psi_host):
    _check(_lib.rte_set_state_host(ctx.handle, _host(psi_host)), ctx.handle)


def rte_get_state_host(ctx, psi_host):
    _check(_lib.rte_get_state_host(ctx.handle, _host(psi_host)), ctx.handle)


def rte_reset_time(ctx):
    _check(_lib.rte_reset_time(ctx.handle), ctx.handle)


def _source_args(w, origin, extent):
    wa = (C.c_float * len(w))(*[float(v) for v in w])
    org = (C.c_int * 3)(*[int(v) for v in origin])
    ext = (C.c_int * 3)(*[int(v) for v in extent])
    return wa, org, ext


def rte_set_source(ctx, w, S_dev, box_origin, box_extent, temporal_kind, t0_ps=0.0, sigma_t_ps=1.0):
    if temporal_kind == 0:
        _check(_lib.rte_set_source(ctx.handle, None, None, None, None, 0, 0.0, 1.0), ctx.handle)
        return
    wa, org, ext = _source_args(w, box_origin, box_extent)
    _check(_lib.rte_set_source(ctx.handle, wa, _dev(S_dev), org, ext, int(temporal_kind), float(t0_ps),
                               float(sigma_t_ps)), ctx.handle)


def rte_set_source_host(ctx, w, S_host, box_origin, box_extent, temporal_kind, t0_ps=0.0, sigma_t_ps=1.0):
    wa, org, ext = _source_args(w, box_origin, box_extent)
    _check(_lib.rte_set_source_host(ctx.handle, wa, _host(S_host), org, ext, int(temporal_kind), float(t0_ps),
                                    float(sigma_t_ps)), ctx.handle)


def rte_step(ctx, nsteps=1):
    _check(_lib.rte_step(ctx.handle, int(nsteps)), ctx.handle)


def rte_extra_workspace_bytes(grid, N, n_fields):
    out = C.c_size_t(0)
    g = _grid(grid)
    _check(_lib.rte_extra_workspace_bytes(C.byref(g), N, int(n_fields), C.byref(out)))
    return int(out.value)


def rte_set_extra_workspace(ctx, n_fields):
    """Allocate n_fields state-sized device buffers with torch (the caller-owned extra workspace of include/rte.h),
    hand them to the library and keep them alive with the context.  n_fields = 0 takes the workspace back."""
    if n_fields <= 0:
        _check(_lib.rte_set_extra_workspace(ctx.handle, None, 0), ctx.handle)
        ctx._extra, ctx._extra_fields = None, 0
        return
    if getattr(ctx, "_extra_fields", 0) >= n_fields:
        return
    nbytes = rte_extra_workspace_bytes(ctx.grid, ctx.N, n_fields)
    _check(_lib.rte_set_extra_workspace(ctx.handle, None, 0), ctx.handle)     # drop (and free) the old one first
    ctx._extra = None
    buf = torch.empty(nbytes, dtype=torch.uint8, device=ctx.device)
    _check(_lib.rte_set_extra_workspace(ctx.handle, C.c_void_p(buf.data_ptr()), nbytes), ctx.handle)
    ctx._extra, ctx._extra_fields = buf, n_fields


def rte_stable_dt(dim, N, n_min, dx_mm, c_mm_per_ps, mu_a_min, mu_s_min, g_max):
    """(bound, recommended dt = bound / 2) of the forward-Euler step in ps (host only; include/rte.h)."""
    b, d = C.c_double(0), C.c_double(0)
    _check(_lib.rte_stable_dt(int(dim), int(N), int(n_min), float(dx_mm), float(c_mm_per_ps), float(mu_a_min),
                              float(mu_s_min), float(g_max), C.byref(b), C.byref(d)))
    return float(b.value), float(d.value)


def rte_step_ssprk3(ctx, nsteps=1):
    """NOT the paper's integrator: SSP-RK3 built from the Euler update (include/rte.h)."""
    rte_set_extra_workspace(ctx, max(1, getattr(ctx, "_extra_fields", 0)))
    _check(_lib.rte_step_ssprk3(ctx.handle, int(nsteps)), ctx.handle)


def rte_step_exp(ctx, nsteps=1):
    """Exponential (integrating-factor) Euler step (include/rte.h) — not eq.(11)."""
    _check(_lib.rte_step_exp(ctx.handle, int(nsteps)), ctx.handle)


def rte_apply_operator(ctx, x_dev, y_dev):
    """y = L x = T[x] + sigma_l x (include/rte.h); [C,nz,ny,nx] fp32 CUDA tensors."""
    rte_set_extra_workspace(ctx, max(2, getattr(ctx, "_extra_fields", 0)))
    _check(_lib.rte_apply_operator(ctx.handle, _dev(x_dev), _dev(y_dev)), ctx.handle)


def rte_solve_steady(ctx, restart=30, tol=1e-5, max_restarts=100, precond_steps=0, precond_dt_ps=0.0):
    """Device-resident GMRES(restart) for L psi = q from the current state, optionally preconditioned by precond_steps
    SSP-RK3 steps of size precond_dt_ps (include/rte.h); returns (operator sweeps, true relative residual).  Allocates
    the extra workspace the solve needs if the context has less."""
    need = restart + 3 + (3 if precond_steps > 0 else 0)
    rte_set_extra_workspace(ctx, max(need, getattr(ctx, "_extra_fields", 0)))
    n, rr = _i(0), C.c_double(0)
    _check(_lib.rte_solve_steady(ctx.handle, int(restart), float(tol), int(max_restarts), int(precond_steps),
                                 float(precond_dt_ps), C.byref(n), C.byref(rr)), ctx.handle)
    return int(n.value), float(rr.value)


def rte_step_profile(ctx, nsteps=1):
    """Returns (ms per axis [3], launches per axis [3]) accumulated over nsteps; synchronises."""
    ms = (C.c_double * 3)()
    nl = (C.c_longlong * 3)()
    _check(_lib.rte_step_profile(ctx.handle, int(nsteps), ms, nl), ctx.handle)
    return [float(v) for v in ms], [int(v) for v in nl]


def rte_fluence(ctx, phi_dev):
    _check(_lib.rte_fluence(ctx.handle, _dev(phi_dev)), ctx.handle)


def rte_fluence_host(ctx, phi_host):
    _check(_lib.rte_fluence_host(ctx.handle, _host(phi_host)), ctx.handle)


def rte_fluence_change(ctx):
    out = C.c_double(0)
    _check(_lib.rte_fluence_change(ctx.handle, C.byref(out)), ctx.handle)
    return float(out.value)


def rte_energy(ctx):
    """(weighted energy sum_c w_l ||psi_c||^2, number of non-finite state values) — the instability guard of include/rte.h."""
    e, n = C.c_double(0), C.c_longlong(0)
    _check(_lib.rte_energy(ctx.handle, C.byref(e), C.byref(n)), ctx.handle)
    return float(e.value), int(n.value)


def rte_time_ps(ctx):
    out = C.c_double(0)
    _check(_lib.rte_time_ps(ctx.handle, C.byref(out)), ctx.handle)
    return float(out.value)


def rte_sync(ctx):
    _check(_lib.rte_sync(ctx.handle), ctx.handle)


def rte_last_error(ctx=None):
    msg = _lib.rte_last_error(ctx.handle if ctx is not None else None)
    return msg.decode() if msg else ""


def rte_launch_count(ctx):
    out = C.c_longlong(0)
    _check(_lib.rte_launch_count(ctx.handle, C.byref(out)), ctx.handle)
    return int(out.value)


# ---- geometry layer ------------------------------------------------------------------------------------------------
def rte_media_ellipsoids(grid, dx_mm, background, ellipsoids, mu_a_dev=None, mu_s_dev=None, g_dev=None, stream=None):
    """ellipsoids: sequence of rows {cx,cy,cz,ax,ay,az,mu_a,mu_s,g} (host)."""
    g_ = _grid(grid)
    flat = [float(v) for row in ellipsoids for v in row]
    n = len(flat) // 9
    arr = (C.c_float * max(1, len(flat)))(*flat)
    bg = (C.c_float * 3)(*[float(v) for v in background])
    ptr = lambda t: _dev(t) if t is not None else None
    _check(_lib.rte_media_ellipsoids(C.byref(g_), float(dx_mm), bg, n, arr, ptr(mu_a_dev), ptr(mu_s_dev), ptr(g_dev),
                                     _stream_ptr(stream)))


def rte_media_lognormal(grid, dx_mm, seed, mean, sigma_log, corr_len_mm, out_dev, scratch_dev, stream=None):
    g_ = _grid(grid)
    _check(_lib.rte_media_lognormal(C.byref(g_), float(dx_mm), C.c_uint64(int(seed)), float(mean), float(sigma_log),
                                    float(corr_len_mm), _dev(out_dev), _dev(scratch_dev), _stream_ptr(stream)))


def rte_media_lognormal_noalloc(grid, dx_mm, seed, mean, sigma_log, corr_len_mm, out_dev, stream=None):
    """Allocation-free variant (static in-library scratch, at most 2 097 152 cells; include/rte.h)."""
    g_ = _grid(grid)
    _check(_lib.rte_media_lognormal_noalloc(C.byref(g_), float(dx_mm), C.c_uint64(int(seed)), float(mean), float(sigma_log),
                                            float(corr_len_mm), _dev(out_dev), _stream_ptr(stream)))


def rte_pml_profile(grid, pml, mu_b_dev=None, inside_dev=None, stream=None):
    g_ = _grid(grid)
    pm = rte_pml(int(pml[0]), float(pml[1]), float(pml[2]))
    _check(_lib.rte_pml_profile(C.byref(g_), C.byref(pm), _dev(mu_b_dev) if mu_b_dev is not None else None,
                                _dev(inside_dev, torch.uint8) if inside_dev is not None else None,
                                _stream_ptr(stream)))
