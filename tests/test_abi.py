"""Host-side tests of the C-ABI boundary (no GPU): the in-tree library loads, exports every symbol include/rte.h
declares, validates arguments, and its host-only coefficient tables agree with quadrature and with the oracle."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1801_06364_b200 as rte
from oracle import rte_oracle as orc
from test_oracle_pins import quad_coupling

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "rte.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rte_[a-z_0-9]+)\s*\(", text)))


def test_library_is_in_tree_and_exports_every_declared_symbol():
    assert os.path.dirname(rte.LIB_PATH) == os.path.join(ROOT, "paper_1801_06364_b200")
    lib = ctypes.CDLL(rte.LIB_PATH)
    syms = declared_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in include/rte.h but not exported"
    assert sorted(rte.EXPORTED) == syms


def test_binding_has_same_names():
    for s in declared_symbols():
        assert hasattr(rte, s), f"binding lacks {s}"


def test_num_coeffs():
    assert rte.rte_num_coeffs(3, 3) == 16 and rte.rte_num_coeffs(3, 7) == 64 and rte.rte_num_coeffs(3, 5) == 36
    assert rte.rte_num_coeffs(2, 3) == 7 and rte.rte_num_coeffs(2, 7) == 15
    assert rte.rte_num_coeffs(4, 3) < 0 and rte.rte_num_coeffs(3, 0) < 0


@pytest.mark.parametrize("dim,N", [(3, 1), (3, 2), (3, 3), (3, 5), (3, 7), (2, 1), (2, 3), (2, 7)])
def test_product_coupling_tables_vs_quadrature_and_oracle(dim, N):
    """The library's own R7/R8 tables (written in the real basis) vs sphere quadrature and vs the oracle's
    (complex eq.(10) + change of basis): three independent derivations."""
    Aq = quad_coupling(dim, N)
    for axis in range(3):
        A = rte.rte_coupling_table(dim, N, axis)
        assert np.abs(A - Aq[axis]).max() < 1e-13
        Ao, _ = orc.coupling_real(dim, N, axis)
        assert np.abs(A - Ao).max() < 1e-14


@pytest.mark.parametrize("dim,N", [(2, 3), (2, 7), (3, 1), (3, 2), (3, 3), (3, 5), (3, 7), (3, 9)])
def test_storage_layout_is_a_valid_slot_assignment(dim, N):
    """Host logic of the bank-conflict-minimising pair layout: every external coefficient appears in exactly one slot,
    pads fill the rest, slot 0 is the fluence, pairs stay together, and the chosen layout is never worse than the
    natural order in the library's own wavefront model (cfg4's order: within 10 % of conflict-free; cfg3's: at least
    20 % fewer wavefronts than the natural order)."""
    ext, (c0, c1, ideal) = rte.rte_storage_layout(dim, N)
    Cn = rte.rte_num_coeffs(dim, N)
    assert len(ext) % 2 == 0 and len(ext) >= Cn
    assert ext[0] == 0
    assert sorted(e for e in ext if e >= 0) == list(range(Cn))
    assert sum(1 for e in ext if e < 0) == len(ext) - Cn
    assert ideal <= c1 <= c0
    if (dim, N) == (3, 7):
        assert c1 <= 1.1 * ideal
    if (dim, N) == (3, 5):
        assert c1 <= 0.8 * c0
    if dim == 3:
        # m >= 1: a_l^m (index l*l+l+m) and b_l^m (l*l+l-m) share a pair; m = 0 fields pair with m = 0 fields
        for s in range(0, len(ext), 2):
            a, b = int(ext[s]), int(ext[s + 1])
            la = int(np.floor(np.sqrt(a)))
            ma = a - la * la - la
            if ma > 0:
                assert b == la * la + la - ma
            elif b >= 0:
                lb = int(np.floor(np.sqrt(b)))
                assert b - lb * lb - lb == 0 and ma == 0
    # deterministic: a second call gives the same layout
    ext2, _ = rte.rte_storage_layout(dim, N)
    assert (ext == ext2).all()


def test_workspace_bytes_and_validation():
    b = rte.rte_workspace_bytes((3, 128, 128, 128), 3)
    G = 128 ** 3
    assert b >= 2 * G * 16 * 4 + 3 * G * 4 and b < 2 * G * 16 * 4 + 3 * G * 4 + 5 * 256
    # 2-D P_3 pads 7 -> 8 fields, P_7 15 -> 16
    assert rte.rte_workspace_bytes((2, 64, 64, 1), 3) >= 2 * 64 * 64 * 8 * 4
    with pytest.raises(rte.RteError):
        rte.rte_workspace_bytes((3, 100, 128, 128), 3)      # unsupported extent
    with pytest.raises(rte.RteError):
        rte.rte_workspace_bytes((2, 64, 64, 2), 3)          # nz must be 1 in 2-D
    with pytest.raises(rte.RteError):
        rte.rte_workspace_bytes((3, 64, 64, 64), 0)


def test_create_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(rte.RteError) as e:
        rte.rte_create((3, 16, 16, 16), 3, 0.1, 0.001, 0.3, 0.01, 10.0, 0.9)
    assert e.value.code == rte.RTE_ECUDA
    # and the raw C entry point reports RTE_ECUDA or RTE_EINVAL, never a silent success
    lib = ctypes.CDLL(rte.LIB_PATH)
    out = ctypes.c_void_p()
    assert lib.rte_create(ctypes.byref(out), None, 3, ctypes.c_float(0.1), ctypes.c_float(0.1), ctypes.c_float(0.3),
                          None, None, None, 0, None) == rte.RTE_EINVAL
    assert lib.rte_step(None, 1) == rte.RTE_ESTATE


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1801_06364_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("rte_tables.h, the oracle", "").lower() or f in ("rte_tables.h", "rte_lib.cu"), f
    for f in ("rte_lib.cu", "rte_pass.cuh", "rte_fft.cuh", "rte_tables.h"):
        text = open(os.path.join(pkg, "csrc", f)).read()
        assert "#include \"../../oracle" not in text and "rte_oracle" not in text


# ---- round 2: stability helper, general extents, extra workspace (host only) ---------------------------------------------
def numpy_stable_dt_bound(dim, N, n, dx, c, mu_a, mu_s, g):
    """R10 written with numpy.linalg on the quadrature-built coupling matrix (independent of the library's own
    eigenvalue routine and tables)."""
    A = quad_coupling(dim, N)[2 if dim == 3 else 0]
    L = np.array([int(np.floor(np.sqrt(i))) for i in range(A.shape[0])]) if dim == 3 else \
        np.array([0] + [m for m in range(1, N + 1) for _ in range(2)])
    sigma = mu_a + mu_s * (1 - g ** L)
    kmax = np.sqrt(dim) * np.pi / dx * (1 - 2.0 / n)
    best = np.inf
    for k in np.linspace(kmax / 200, kmax, 200):
        lam = np.linalg.eigvals(-c * (1j * k * A + np.diag(sigma)))
        best = min(best, np.min(-2 * lam.real / np.abs(lam) ** 2))
    return best


@pytest.mark.parametrize("dim,N,n,dx,med", [(2, 3, 64, 0.1, (0.01, 10.0, 0.9)), (3, 3, 128, 0.8, (0.01, 10.0, 0.9)),
                                            (3, 5, 256, 0.04, (0.01, 5.0, 0.95)), (3, 7, 384, 0.25, (0.01, 3.0, 0.9)),
                                            (2, 7, 512, 0.05, (0.005, 5.0, 0.9)), (3, 2, 32, 0.3, (0.2, 1.0, 0.0))])
def test_stable_dt_matches_numpy_eigenvalues(dim, N, n, dx, med):
    bound, dt = rte.rte_stable_dt(dim, N, n, dx, 0.3, *med)
    ref = numpy_stable_dt_bound(dim, N, n, dx, 0.3, *med)
    assert abs(bound - ref) <= 1e-6 * ref          # media arrive as fp32
    assert dt == 0.5 * bound


def test_stable_dt_reproduces_the_survey_table_and_rejects_bad_input():
    """SURVEY R10 [verified] bounds: cfg0 4.68 fs, cfg2 268 fs, the paper's exp.1 background 66 fs."""
    assert abs(rte.rte_stable_dt(2, 3, 64, 0.1, 0.3, 0.01, 10.0, 0.9)[0] - 4.68e-3) < 2e-5
    assert abs(rte.rte_stable_dt(3, 3, 128, 0.8, 0.3, 0.01, 10.0, 0.9)[0] - 0.268) < 1e-3
    assert abs(rte.rte_stable_dt(3, 21, 64, 50.0 / 64, 0.3, 0.01, 1.0, 0.9)[0] - 0.066) < 1e-3
    import rte_workloads as wl
    for name, weak in [("cfg0", (0.01, 10.0, 0.9)), ("cfg1", (0.005, 5.0, 0.9)), ("cfg2", (0.01, 10.0, 0.9)),
                       ("cfg3", (0.01, 5.0, 0.95)), ("cfg4", (0.01, 3.0, 0.9))]:
        cfg = wl.CONFIGS[name]
        assert cfg.dt <= 0.55 * rte.rte_stable_dt(cfg.dim, cfg.N, cfg.nx, cfg.dx, cfg.c, *weak)[0]
    for bad in [(4, 3, 64, 0.1, 0.3, 0.01, 10.0, 0.9), (3, 0, 64, 0.1, 0.3, 0.01, 10.0, 0.9), (3, 32, 64, 0.1, 0.3, 0.01, 10.0, 0.9),
                (3, 3, 64, 0.0, 0.3, 0.01, 10.0, 0.9), (3, 3, 64, 0.1, 0.3, 0.01, 10.0, 1.5), (3, 3, 2, 0.1, 0.3, 0.01, 10.0, 0.9)]:
        with pytest.raises(rte.RteError):
            rte.rte_stable_dt(*bad)


def test_supported_extents_are_the_even_2a3b_numbers():
    ok = sorted(n for n in range(16, 1025) if n % 2 == 0 and all(p in (2, 3) for p in _prime_factors(n)))
    assert len(ok) == 29 and ok[:6] == [16, 18, 24, 32, 36, 48] and ok[-3:] == [864, 972, 1024]
    for n in range(2, 1100):
        try:
            rte.rte_workspace_bytes((2, n, 16, 1), 1)
            accepted = True
        except rte.RteError:
            accepted = False
        assert accepted == (n in ok), n


def _prime_factors(n):
    out, p = [], 2
    while n > 1:
        while n % p == 0:
            out.append(p)
            n //= p
        p += 1
    return out


def test_extra_workspace_bytes_and_order_cap():
    one = rte.rte_extra_workspace_bytes((3, 32, 32, 32), 3, 1)
    assert one >= 32 ** 3 * 16 * 4 and one % 256 == 0
    assert rte.rte_extra_workspace_bytes((3, 32, 32, 32), 3, 33) == 33 * one
    assert rte.rte_extra_workspace_bytes((3, 32, 32, 32), 3, 0) == 0
    assert rte.rte_num_coeffs(3, 31) == 1024 and rte.rte_num_coeffs(3, 32) < 0 and rte.rte_num_coeffs(3, 50000) < 0
    with pytest.raises(rte.RteError):
        rte.rte_coupling_table(3, 50000, 0)
    with pytest.raises(rte.RteError):
        rte.rte_storage_layout(3, 40)
