"""Pins P1..P16: the fp64 oracle checked against what the paper and the
mathematics fix, never against itself.  CPU only.

Every expected value below comes from (a) direct quadrature on the sphere / circle written here with numpy + scipy's
Legendre functions, (b) closed forms, (c) numpy.linalg on small matrices built from (a), (d) brute-force O(n^2)
definitions written here, or (e) the small text fixtures under tests/golden/ (mathematical constants, cited there).
"""
import math
import os

import numpy as np
import pytest
from scipy.special import lpmv

from oracle import rte_oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------------------------------------------------------
# independent spherical / circular harmonics (eq.(3); reading R6, R12: orthonormal, Condon-Shortley)
# ------------------------------------------------------------------------------------------------------------------
def sph_Y(l, m, ct, ph):
    """Orthonormal complex Y_l^m with Condon-Shortley phase (scipy's lpmv includes it)."""
    am = abs(m)
    norm = math.sqrt((2 * l + 1) / (4 * math.pi) * math.factorial(l - am) / math.factorial(l + am))
    y = norm * lpmv(am, l, ct) * np.exp(1j * am * ph)
    if m < 0:
        y = (-1) ** am * np.conj(y)
    return y


def sphere_quadrature(nt=40, nph=80):
    x, w = np.polynomial.legendre.leggauss(nt)
    ph = 2 * np.pi * np.arange(nph) / nph
    CT, PH = np.meshgrid(x, ph, indexing="ij")
    W = np.outer(w, np.full(nph, 2 * np.pi / nph))
    return CT, PH, W


def real_Y(l, m, ct, ph):
    """Reading R6: Y^R_{l,m>0} = sqrt2 (-1)^m Re Y_l^m ; Y^R_{l,m<0} = sqrt2 (-1)^|m| Im Y_l^|m| ; Y^R_{l0} = Y_l^0."""
    if m == 0:
        return sph_Y(l, 0, ct, ph).real
    y = sph_Y(l, abs(m), ct, ph)
    s = math.sqrt(2.0) * (-1) ** abs(m)
    return s * (y.real if m > 0 else y.imag)


def quad_coupling_real3(N):
    """A_a[c,c'] = (n_l'/n_l) int Y^R_c s_a Y^R_c' ds,  n_l = sqrt((2l+1)/4pi)  (projection of s.grad phi, eq.(3),(6))."""
    CT, PH, W = sphere_quadrature()
    st = np.sqrt(1 - CT ** 2)
    s = [st * np.cos(PH), st * np.sin(PH), CT]
    lm = [(l, m) for l in range(N + 1) for m in range(-l, l + 1)]
    Y = [real_Y(l, m, CT, PH) for (l, m) in lm]
    C = len(lm)
    A = np.zeros((3, C, C))
    for a in range(3):
        for i, (l, m) in enumerate(lm):
            for j, (lp, mp) in enumerate(lm):
                A[a, i, j] = math.sqrt((2 * lp + 1) / (2 * l + 1)) * np.sum(W * Y[i] * s[a] * Y[j])
    return A


def quad_coupling_complex3(N):
    CT, PH, W = sphere_quadrature()
    st = np.sqrt(1 - CT ** 2)
    s = [st * np.cos(PH), st * np.sin(PH), CT]
    lm = [(l, m) for l in range(N + 1) for m in range(-l, l + 1)]
    Y = [sph_Y(l, m, CT, PH) for (l, m) in lm]
    C = len(lm)
    A = np.zeros((3, C, C), dtype=complex)
    for a in range(3):
        for i, (l, m) in enumerate(lm):
            for j, (lp, mp) in enumerate(lm):
                A[a, i, j] = math.sqrt((2 * lp + 1) / (2 * l + 1)) * np.sum(W * np.conj(Y[i]) * s[a] * Y[j])
    return A


def quad_coupling_real2(N):
    """Reading R8: phi = (1/2pi)[a_0 + 2 sum (a_m cos m th + b_m sin m th)], a_m = int phi cos m th, b_m = int phi sin m th."""
    nth = 256
    th = 2 * np.pi * np.arange(nth) / nth
    w = 2 * np.pi / nth
    C = 2 * N + 1
    expand, project = [None] * C, [None] * C
    expand[0] = np.full(nth, 1 / (2 * np.pi))
    project[0] = np.ones(nth)
    for m in range(1, N + 1):
        expand[2 * m - 1] = np.cos(m * th) / np.pi
        expand[2 * m] = np.sin(m * th) / np.pi
        project[2 * m - 1] = np.cos(m * th)
        project[2 * m] = np.sin(m * th)
    s = [np.cos(th), np.sin(th)]
    A = np.zeros((3, C, C))
    for a in range(2):
        for i in range(C):
            for j in range(C):
                A[a, i, j] = w * np.sum(project[i] * s[a] * expand[j])
    return A


def quad_coupling(dim, N):
    return quad_coupling_real3(N) if dim == 3 else quad_coupling_real2(N)


# ------------------------------------------------------------------------------------------------------------------
# P1 — coupling coefficients vs direct quadrature  (alpha, beta, 1/(2l+1), signs; R1, R6, R7, R8, R12)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [1, 3, 5, 7])
def test_P1_real_coupling_vs_quadrature_3d(N):
    Aq = quad_coupling_real3(N)
    for a in range(3):
        A, im = orc.coupling_real(3, N, a)
        assert im < 1e-14
        assert np.abs(A - Aq[a]).max() < 1e-13


@pytest.mark.parametrize("N", [2, 5])
def test_P1_complex_coupling_eq10_vs_quadrature(N):
    """eq.(10) itself, in the paper's complex basis, with the 1/(2l+1) on all brackets (R1)."""
    Aq = quad_coupling_complex3(N)
    for a in range(3):
        A = orc.coupling_complex(3, N, a)
        assert np.abs(A - Aq[a]).max() < 1e-13


def test_P1_literal_eq6_reading_is_rejected():
    """If the 1/(2l+1) enclosed only the d/dz bracket (eq.(6) as printed) the x coupling would be off by O(1)."""
    Aq = quad_coupling_complex3(2)
    A = orc.coupling_complex(3, 2, 0)
    l_of = np.array([l for l in range(3) for m in range(-l, l + 1)])
    A_literal = A * (2 * l_of[:, None] + 1)
    assert np.abs(A_literal - Aq[0]).max() > 0.1


@pytest.mark.parametrize("N", [1, 3, 7])
def test_P1_coupling_vs_quadrature_2d(N):
    Aq = quad_coupling_real2(N)
    for a in range(2):
        A, im = orc.coupling_real(2, N, a)
        assert im < 1e-14
        assert np.abs(A - Aq[a]).max() < 1e-13
    A, _ = orc.coupling_real(2, N, 2)
    assert np.abs(A).max() == 0.0


def test_P1_fan_in():
    """Sparsity the CUDA tables rely on: <=2 z-neighbours, <=4 x, <=4 y per output coefficient."""
    for N in (3, 5, 7):
        for a, cap in ((0, 4), (1, 4), (2, 2)):
            A, _ = orc.coupling_real(3, N, a)
            assert (np.count_nonzero(A, axis=1) <= cap).all()


# ------------------------------------------------------------------------------------------------------------------
# own DFT vs the O(n^2) definition (eq.(8): exp(-ik.r) forward)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 12, 24, 64, 96, 35])
def test_dft_vs_definition(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    j = np.arange(n)
    for sign in (-1, +1):
        Wm = np.exp(sign * 2j * np.pi * np.outer(j, j) / n)
        assert np.abs(orc.dft(x, sign) - Wm @ x).max() < 1e-12 * max(1, n)


# ------------------------------------------------------------------------------------------------------------------
# P2 — spectral derivative of band-limited trigonometric fields vs analytic derivative (R2, R5)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [16, 24, 64])
def test_P2_spectral_derivative_analytic(n):
    dx = 0.37
    Lx = n * dx
    x = np.arange(n) * dx
    for axis in range(3):
        for j in (1, 3, n // 2 - 1):
            kx = 2 * np.pi * j / Lx
            shape = [1, 1, 1]
            shape[2 - axis] = n
            full = [n if (2 - axis) == d else 3 for d in range(3)]
            f = np.broadcast_to(np.sin(kx * x + 0.3).reshape(shape), full).copy()
            df = orc.deriv(f, axis, dx)
            ex = np.broadcast_to((kx * np.cos(kx * x + 0.3)).reshape(shape), f.shape)
            assert np.abs(df - ex).max() < 1e-12 * kx * n
    # constants and the Nyquist mode differentiate to zero (R5)
    f = np.ones((3, 3, n))
    assert np.abs(orc.deriv(f, 0, dx)).max() < 1e-13
    f = np.broadcast_to(np.cos(np.pi * np.arange(n)), (3, 3, n)).copy()
    assert np.abs(orc.deriv(f, 0, dx)).max() < 1e-12


def test_P2_wavenumbers():
    k = orc.wavenumbers(8, 0.5)
    ex = 2 * np.pi * np.array([0, 1, 2, 3, 0, -3, -2, -1]) / (8 * 0.5)
    assert np.abs(k - ex).max() < 1e-15
    k = orc.wavenumbers(6, 1.0)
    ex = 2 * np.pi * np.array([0, 1, 2, 0, -2, -1]) / 6
    assert np.abs(k - ex).max() < 1e-15


# ------------------------------------------------------------------------------------------------------------------
# degrees(): which power of g each external coefficient takes in sigma = mu_a + mu_s (1 - g^l)  (eq.(5), PAPER.md:66-69;
# 2-D: l == |m|, reading R8).  The expected side of P3 / P4 below uses THIS hand-written table, not orc.degrees.
# ------------------------------------------------------------------------------------------------------------------
def hand_degrees(dim, N):
    """Written out from the coefficient order alone: 3-D c = l*l + l + m, m = -l..l  =>  2l+1 consecutive entries of l;
    2-D c = 0 -> a_0, c = 2m-1 -> a_m, c = 2m -> b_m  =>  0, 1, 1, 2, 2, ..."""
    if dim == 3:
        return np.array([l for l in range(N + 1) for _ in range(2 * l + 1)])
    return np.array([0] + [m for m in range(1, N + 1) for _ in (0, 1)])


def test_degrees_tables_written_out():
    assert list(orc.degrees(2, 3)) == [0, 1, 1, 2, 2, 3, 3]
    assert list(orc.degrees(2, 1)) == [0, 1, 1]
    assert list(orc.degrees(2, 7)) == [0, 1, 1, 2, 2, 3, 3, 4, 4, 5, 5, 6, 6, 7, 7]
    assert list(orc.degrees(3, 2)) == [0, 1, 1, 1, 2, 2, 2, 2, 2]
    assert list(orc.degrees(3, 3)) == [0] + [1] * 3 + [2] * 5 + [3] * 7


def test_henyey_greenstein_eigenvalues_are_g_to_the_order():
    """Why the diagonal is mu_s g^l (3-D, eq.(2),(5)) and mu_s g^|m| (2-D, R8): the Legendre /
    Fourier coefficients of the phase function, by quadrature."""
    g = 0.87
    x, w = np.polynomial.legendre.leggauss(200)
    p3 = (1 - g * g) / (4 * np.pi * (1 + g * g - 2 * g * x) ** 1.5)           # eq.(2)
    for l in range(8):
        Pl = np.polynomial.legendre.Legendre.basis(l)(x)
        assert abs(2 * np.pi * np.sum(w * p3 * Pl) - g ** l) < 1e-12
    th = 2 * np.pi * np.arange(4096) / 4096
    p2 = (1 - g * g) / (2 * np.pi * (1 + g * g - 2 * g * np.cos(th)))         # 2-D Henyey-Greenstein kernel (R8)
    for m in range(8):
        assert abs(np.sum(p2 * np.cos(m * th)) * (2 * np.pi / 4096) - g ** m) < 1e-12


# ------------------------------------------------------------------------------------------------------------------
# P3 — uniform field decays as (1 - c dt sigma_l)^n -> exp(-c sigma_l t)  (sigma_l = mu_a + mu_s (1-g^l); R3, R4)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim,N,form", [(3, 3, orc.PER_AXIS), (3, 2, orc.LITERAL), (2, 3, orc.PER_AXIS), (2, 3, orc.LITERAL)])
def test_P3_uniform_decay(dim, N, form):
    n = 8
    nz = n if dim == 3 else 1
    mu_a, mu_s, g, c, dt = 0.013, 9.0, 0.87, 0.3, 0.004
    o = orc.Oracle(dim, n, n, nz, N, 0.1, dt, c, mu_a, mu_s, g)
    C = o.C
    amp = 1.0 + np.arange(C)
    o.set_state(np.broadcast_to(amp[:, None, None, None], (C, nz, n, n)))
    steps = 25
    o.step(steps, form)
    psi = o.get_state()
    L = hand_degrees(dim, N)                    # not orc.degrees: the expected side is independent of the oracle
    sigma = mu_a + mu_s * (1 - g ** L)
    ex = amp * (1 - c * dt * sigma) ** steps
    assert np.abs(psi - ex[:, None, None, None]).max() < 1e-13 * amp.max()
    # l = 0 decays with mu_a only: exp(-c mu_a t) to first order in dt
    t = steps * dt
    assert abs(psi[0, 0, 0, 0] / amp[0] - math.exp(-c * mu_a * t)) < (c * mu_a) ** 2 * dt * t
    # first-order convergence of the l>=1 decay to exp(-c sigma_l t)
    errs = []
    for fac in (1, 2):
        o2 = orc.Oracle(dim, n, n, nz, N, 0.1, dt / fac, c, mu_a, mu_s, g)
        o2.set_state(np.broadcast_to(amp[:, None, None, None], (C, nz, n, n)))
        o2.step(steps * fac, form)
        errs.append(abs(o2.get_state()[1, 0, 0, 0] / amp[1] - math.exp(-c * sigma[1] * t)))
    assert 1.7 < errs[0] / errs[1] < 2.3


def test_P3_uniform_decay_inside_pml():
    """eq.(12): in the layer every l decays with mu_b alone (mu_s = 0 there, mu_a not added; R11)."""
    n, W = 8, 4                       # W = n/2: every cell belongs to the layer
    mu_b, c, dt = 0.7, 0.3, 0.01
    o = orc.Oracle(3, n, n, n, 2, 0.1, dt, c, 0.01, 10.0, 0.9, pml_width=W, mu_lo=mu_b, mu_hi=mu_b)
    C = o.C
    amp = 1.0 + np.arange(C)
    o.set_state(np.broadcast_to(amp[:, None, None, None], (C, n, n, n)))
    o.step(10)
    ex = amp * (1 - c * dt * mu_b) ** 10
    assert np.abs(o.get_state() - ex[:, None, None, None]).max() < 1e-13 * amp.max()


def test_P3_heterogeneous_maps_pointwise():
    """Uniform psi => T = 0, so one step is psi (1 - c dt sigma_l(r)) cell by cell: pins map indexing and g^l (R16)."""
    rng = np.random.default_rng(7)
    nx, ny, nz, N = 6, 4, 8, 3
    mu_a = rng.uniform(0.01, 1, (nz, ny, nx))
    mu_s = rng.uniform(5, 20, (nz, ny, nx))
    g = rng.uniform(0.8, 0.95, (nz, ny, nx))
    c, dt = 0.3, 1e-3
    o = orc.Oracle(3, nx, ny, nz, N, 0.1, dt, c, mu_a, mu_s, g)
    o.set_state(np.ones((o.C, nz, ny, nx)))
    o.step(1)
    L = hand_degrees(3, N)
    ex = 1 - c * dt * (mu_a[None] + mu_s[None] * (1 - g[None] ** L[:, None, None, None]))
    assert np.abs(o.get_state() - ex).max() < 1e-14


# ------------------------------------------------------------------------------------------------------------------
# P4 — one Fourier mode against the matrix power / exponential of the per-k system built from quadrature
# ------------------------------------------------------------------------------------------------------------------
def mode_matrix(dim, N, kvec, mu_a, mu_s, g, c):
    A = quad_coupling(dim, N)
    L = hand_degrees(dim, N)                    # not orc.degrees: M(k) is built without the oracle
    sigma = mu_a + mu_s * (1 - g ** L)
    M = -c * (1j * sum(kvec[a] * A[a] for a in range(dim)) + np.diag(sigma))
    return M


@pytest.mark.parametrize("dim,N,n,form", [(3, 3, 8, orc.PER_AXIS), (3, 2, 8, orc.LITERAL), (2, 3, 16, orc.PER_AXIS),
                                          (2, 4, 12, orc.LITERAL), (3, 3, 12, orc.PER_AXIS)])
def test_P4_single_mode_matrix_power(dim, N, n, form):
    rng = np.random.default_rng(100 * dim + N)
    dx, c, dt = 0.2, 0.3, 0.002
    mu_a, mu_s, g = 0.02, 4.0, 0.8
    nz = n if dim == 3 else 1
    j = np.array([2, -1, 3][:dim] + [0] * (3 - dim))
    kvec = 2 * np.pi * j / (n * dx)
    C = orc.num_coeffs(dim, N)
    v = rng.standard_normal(C) + 1j * rng.standard_normal(C)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(n), np.arange(n), indexing="ij")
    phase = np.exp(1j * dx * (kvec[0] * x + kvec[1] * y + kvec[2] * z))
    o = orc.Oracle(dim, n, n, nz, N, dx, dt, c, mu_a, mu_s, g)
    o.set_state((v[:, None, None, None] * phase[None]).real)
    steps = 20
    o.step(steps, form)
    M = mode_matrix(dim, N, kvec, mu_a, mu_s, g, c)
    vn = np.linalg.matrix_power(np.eye(C) + dt * M, steps) @ v
    ex = (vn[:, None, None, None] * phase[None]).real
    assert np.abs(o.get_state() - ex).max() < 1e-12 * np.abs(v).max()


def test_P4_single_mode_converges_to_matrix_exponential():
    from scipy.linalg import expm
    dim, N, n = 3, 3, 8
    dx, c = 0.2, 0.3
    mu_a, mu_s, g = 0.02, 4.0, 0.8
    kvec = 2 * np.pi * np.array([1, 2, -1]) / (n * dx)
    C = orc.num_coeffs(dim, N)
    rng = np.random.default_rng(5)
    v = rng.standard_normal(C) + 1j * rng.standard_normal(C)
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    phase = np.exp(1j * dx * (kvec[0] * x + kvec[1] * y + kvec[2] * z))
    M = mode_matrix(dim, N, kvec, mu_a, mu_s, g, c)
    t = 0.04
    ex = ((expm(M * t) @ v)[:, None, None, None] * phase[None]).real
    errs = []
    for steps in (20, 40):
        o = orc.Oracle(dim, n, n, n, N, dx, t / steps, c, mu_a, mu_s, g)
        o.set_state((v[:, None, None, None] * phase[None]).real)
        o.step(steps)
        errs.append(np.abs(o.get_state() - ex).max())
    assert 1.7 < errs[0] / errs[1] < 2.3


# ------------------------------------------------------------------------------------------------------------------
# P5 — conservation of the total l=0 moment when mu_a = 0, periodic, no PML, no source
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim,form", [(3, orc.PER_AXIS), (2, orc.PER_AXIS), (3, orc.LITERAL)])
def test_P5_conservation(dim, form):
    rng = np.random.default_rng(11)
    n = 8 if dim == 3 else 16
    nz = n if dim == 3 else 1
    o = orc.Oracle(dim, n, n, nz, 3, 0.1, 0.002, 0.3, 0.0, 6.0, 0.9)
    psi0 = rng.standard_normal((o.C, nz, n, n))
    o.set_state(psi0)
    tot0 = psi0[0].sum()
    for _ in range(5):
        o.step(3, form)
        assert abs(o.fluence().sum() - tot0) < 1e-13 * np.abs(psi0[0]).sum()


# ------------------------------------------------------------------------------------------------------------------
# P6 — D_a real antisymmetric; streaming skew-adjoint; eigen-speeds = Gauss-Legendre nodes (golden constants)
# ------------------------------------------------------------------------------------------------------------------
def test_P6_derivative_antisymmetric():
    rng = np.random.default_rng(3)
    u = rng.standard_normal((6, 8, 12))
    v = rng.standard_normal((6, 8, 12))
    for axis in range(3):
        a = np.sum(u * orc.deriv(v, axis, 0.3))
        b = np.sum(orc.deriv(u, axis, 0.3) * v)
        assert abs(a + b) < 1e-11 * (abs(a) + 1)


def test_P6_symmetrisable_and_eigen_speeds_golden():
    rows = [ln.split() for ln in open(os.path.join(GOLD, "eigen_speeds.txt")) if ln.strip() and not ln.startswith("#")]
    for dim, N, val in rows:
        dim, N, val = int(dim), int(N), float(val)
        L = orc.degrees(dim, N)
        for a in range(dim):
            A, _ = orc.coupling_real(dim, N, a)
            if dim == 3:
                d = np.sqrt(2 * L + 1.0)
            else:
                d = np.where(L == 0, 1.0, math.sqrt(2.0))       # 2-D weights: a_0 once, m>=1 twice
            S = A * d[:, None] / d[None, :]
            assert np.abs(S - S.T).max() < 1e-14
            ev = np.linalg.eigvalsh(0.5 * (S + S.T))
            assert abs(np.abs(ev).max() - val) < 2e-10


# ------------------------------------------------------------------------------------------------------------------
# P7 — source scaling and sign: fixed point of the Euler map is psi_c = q_c / sigma_l
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim", [2, 3])
def test_P7_source_fixed_point(dim):
    n = 4
    nz = n if dim == 3 else 1
    mu_a, mu_s, g, c, dt = 0.5, 3.0, 0.5, 0.3, 0.05
    o = orc.Oracle(dim, n, n, nz, 2, 0.1, dt, c, mu_a, mu_s, g)
    w = np.arange(1, o.C + 1) * 0.25
    S = np.full((nz, n, n), 2.0)
    o.set_source(w, S, (0, 0, 0), (n, n, nz), 1)
    L = hand_degrees(dim, 2)
    sigma = mu_a + mu_s * (1 - g ** L)
    fixed = 2.0 * w / sigma
    o.set_state(np.broadcast_to(fixed[:, None, None, None], (o.C, nz, n, n)))
    o.step(7)
    assert np.abs(o.get_state() - fixed[:, None, None, None]).max() < 1e-13 * fixed.max()
    # and it is reached geometrically from zero: after n steps psi_0 = (q/mu_a)(1 - (1 - c dt mu_a)^n)
    o2 = orc.Oracle(dim, n, n, nz, 2, 0.1, dt, c, mu_a, mu_s, g)
    o2.set_source(w, S, (0, 0, 0), (n, n, nz), 1)
    o2.step(9)
    ex = fixed[0] * (1 - (1 - c * dt * sigma[0]) ** 9)
    assert abs(o2.fluence()[0, 0, 0] - ex) < 1e-13


def test_P7_gaussian_temporal_profile_sampled_at_tn():
    """R14: q(t_n); uniform isotropic source, mu=0: psi_0(n) = c dt sum_{j<n} f(j dt)."""
    n, c, dt, t0, sg = 4, 0.3, 0.1, 0.5, 0.2
    o = orc.Oracle(2, n, n, 1, 1, 0.1, dt, c, 0.0, 0.0, 0.0)
    o.set_source([1, 0, 0], np.ones((1, n, n)), (0, 0, 0), (n, n, 1), 2, t0, sg)
    o.step(10)
    ex = c * dt * sum(math.exp(-0.5 * ((j * dt - t0) / sg) ** 2) for j in range(10))
    assert abs(o.fluence()[0, 0, 0] - ex) < 1e-14
    assert abs(o.time_ps() - 1.0) < 1e-14


def test_P7_source_masked_in_pml_and_boxed():
    n, W = 16, 3
    o = orc.Oracle(2, n, n, 1, 1, 0.1, 0.01, 0.3, 0.0, 0.0, 0.0, pml_width=W, mu_lo=0.0, mu_hi=0.0)
    S = np.arange(1, 1 + 5 * 4, dtype=float).reshape(1, 4, 5)
    o.set_source([1, 0, 0], S, (1, 2, 0), (5, 4, 1), 1)
    o.step(1)
    phi = o.fluence()[0]
    ex = np.zeros((n, n))
    ex[2:6, 1:6] = 0.3 * 0.01 * S[0]
    ex[:W, :] = 0
    ex[:, :W] = 0
    assert np.abs(phi - ex).max() < 1e-16


# ------------------------------------------------------------------------------------------------------------------
# P8 — direction sign with anisotropic data: the centroid of psi_0 moves toward +x at c sum(Jx)/sum(Phi)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim", [2, 3])
def test_P8_centroid_moves_along_plus_x(dim):
    n, dx, c, dt = 32, 0.1, 0.3, 0.002
    nz = 8 if dim == 3 else 1
    o = orc.Oracle(dim, n, n, nz, 3, dx, dt, c, 0.0, 0.0, 0.0)
    xs = (np.arange(n) - n // 2) * dx
    Gs = np.exp(-(xs[None, None, :] ** 2 + xs[None, :, None] ** 2) / (2 * 0.3 ** 2)) * np.ones((nz, 1, 1))
    psi = np.zeros((o.C, nz, n, n))
    psi[0] = Gs
    jx = 3 if dim == 3 else 1                        # a_1^1 (3-D, c = l*l+l+m = 3) / a_1 (2-D)
    psi[jx] = 0.5 * Gs
    o.set_state(psi)
    steps = 250
    o.step(steps)
    phi = o.fluence()
    cx = (phi * xs[None, None, :]).sum() / phi.sum()
    cy = (phi * xs[None, :, None]).sum() / phi.sum()
    expected = c * 0.5 * steps * dt
    assert cx > 0
    assert abs(cx - expected) < 0.03 * expected
    assert abs(cy) < 1e-5            # only the unpaired tail cell at -n/2 (e^-14) breaks the y symmetry of the sum


# ------------------------------------------------------------------------------------------------------------------
# P9 — cubic / square symmetry of an isotropic centred pulse
# ------------------------------------------------------------------------------------------------------------------
def test_P9_symmetry_3d():
    n, dx = 12, 0.2
    o = orc.Oracle(3, n, n, n, 3, dx, 0.004, 0.3, 0.01, 2.0, 0.8)
    xs = (np.arange(n) - n // 2) * dx
    r2 = xs[None, None, :] ** 2 + xs[None, :, None] ** 2 + xs[:, None, None] ** 2
    psi = np.zeros((o.C, n, n, n))
    psi[0] = np.exp(-r2 / (2 * 0.3 ** 2))
    o.set_state(psi)
    o.step(12)
    p = o.get_state()
    f = p[0]
    scale = np.abs(f).max()
    assert np.abs(f - f.transpose(1, 0, 2)).max() < 1e-13 * scale
    assert np.abs(f - f.transpose(2, 1, 0)).max() < 1e-13 * scale
    # reflection about the centre cell n/2: index i -> (n - i) mod n
    refl = lambda a: np.roll(a[::-1, ::-1, ::-1], 1, axis=(0, 1, 2))
    L = orc.degrees(3, 3)
    for cc in range(o.C):
        assert np.abs(refl(p[cc]) - (-1) ** L[cc] * p[cc]).max() < 1e-13 * scale
    # flux components map into each other under axis swaps: a_1^1 (c=3) <-> b_1^1 (c=1) <-> a_1^0 (c=2)
    assert np.abs(p[3] - p[1].transpose(0, 2, 1)).max() < 1e-13 * scale
    assert np.abs(p[3] - p[2].transpose(2, 1, 0)).max() < 1e-13 * scale
    assert np.abs(p[3]).max() > 1e-3 * scale


# ------------------------------------------------------------------------------------------------------------------
# P10 — PML map (R11)
# ------------------------------------------------------------------------------------------------------------------
def test_P10_pml_map():
    n, W, lo, hi = 20, 4, 0.01, 1.0
    mu_b, inside = orc.pml_map(3, n, n, n, W, lo, hi)
    assert inside.sum() == (n - 2 * W) ** 3
    assert inside[W:n - W, W:n - W, W:n - W].all()
    assert (mu_b[inside == 1] == 0).all()
    # outer faces carry mu_hi, first layer cell carries the half-cosine value at delta = 1/W
    assert np.allclose(mu_b[0], hi) and np.allclose(mu_b[:, :, n - 1], hi) and np.allclose(mu_b[:, 0, :], hi)
    first = lo + (hi - lo) * 0.5 * (1 - math.cos(math.pi / W))
    assert abs(mu_b[n // 2, n // 2, W - 1] - first) < 1e-15
    assert abs(mu_b[n // 2, n // 2, n - W] - first) < 1e-15
    assert abs(mu_b[n // 2, W - 2, n // 2] - (lo + (hi - lo) * 0.5 * (1 - math.cos(2 * math.pi / W)))) < 1e-15
    # symmetric under i -> n-1-i, corner = max rule
    assert np.array_equal(mu_b, mu_b[::-1, ::-1, ::-1])
    assert abs(mu_b[W - 1, W - 3, n // 2] - (lo + (hi - lo) * 0.5 * (1 - math.cos(3 * math.pi / W)))) < 1e-15
    # 2-D: z is not an axis
    mu2, in2 = orc.pml_map(2, n, n, 1, W, lo, hi)
    assert in2.sum() == (n - 2 * W) ** 2
    # no PML
    mu0, in0 = orc.pml_map(3, 6, 6, 6, 0, lo, hi)
    assert in0.all() and (mu0 == 0).all()


def test_P10_scattering_switched_off_in_layer():
    """In the layer sigma_l = mu_b for every l (mu_s = 0, mu_a not added): uniform psi, one step, cell by cell."""
    n, W, N = 12, 3, 2
    c, dt = 0.3, 0.01
    o = orc.Oracle(3, n, n, n, N, 0.1, dt, c, 0.05, 8.0, 0.9, pml_width=W, mu_lo=0.05, mu_hi=2.0)
    o.set_state(np.ones((o.C, n, n, n)))
    o.step(1)
    mu_b, inside = orc.pml_map(3, n, n, n, W, 0.05, 2.0)
    L = hand_degrees(3, N)
    sig_in = 0.05 + 8.0 * (1 - 0.9 ** L)
    ex = np.where(inside[None] == 1, 1 - c * dt * sig_in[:, None, None, None], 1 - c * dt * mu_b[None])
    assert np.abs(o.get_state() - ex).max() < 1e-15


# ------------------------------------------------------------------------------------------------------------------
# P11 — P_1 reduction (textbook telegraph system; golden fixture)
# ------------------------------------------------------------------------------------------------------------------
def test_P11_p1_reduction_golden():
    rows = [ln.split() for ln in open(os.path.join(GOLD, "p1_reduction.txt")) if ln.strip() and not ln.startswith("#")]
    for dim in (2, 3):
        C = orc.num_coeffs(dim, 1)
        ex = np.zeros((3, C, C))
        for d, a, r, cc, v in rows:
            if int(d) == dim:
                ex[int(a), int(r), int(cc)] = float(v)
        for a in range(3):
            A, _ = orc.coupling_real(dim, 1, a)
            assert np.abs(A - ex[a]).max() < 1e-15


# ------------------------------------------------------------------------------------------------------------------
# P12 — the paper's literal complex / full-DFT / k-space formulation == per-axis real-basis formulation (R6, R18)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim,N,shape", [(3, 3, (8, 6, 12)), (3, 4, (6, 6, 6)), (2, 3, (1, 12, 16)), (2, 7, (1, 8, 8))])
def test_P12_literal_equals_per_axis(dim, N, shape):
    rng = np.random.default_rng(12)
    nz, ny, nx = shape
    mu_a = rng.uniform(0.01, 0.1, shape)
    mu_s = rng.uniform(5, 20, shape)
    g = rng.uniform(0.8, 0.95, shape)
    psi0 = rng.standard_normal((orc.num_coeffs(dim, N),) + shape)
    res = []
    for form in (orc.LITERAL, orc.PER_AXIS):
        o = orc.Oracle(dim, nx, ny, nz, N, 0.1, 0.001, 0.3, mu_a, mu_s, g, pml_width=2, mu_lo=0.01, mu_hi=3.0)
        o.set_state(psi0)
        o.step(5, form)
        res.append(o.get_state())
    assert np.abs(res[0] - res[1]).max() < 1e-12 * np.abs(psi0).max()


def test_streaming_is_sum_of_coupled_derivatives():
    """T = sum_a A_a D_a psi with A from quadrature (not the oracle's tables) and D from the analytic k multiply of
    numpy's FFT: an end-to-end check of the streaming term that shares nothing with the oracle."""
    rng = np.random.default_rng(21)
    N, n, dx = 3, 8, 0.25
    o = orc.Oracle(3, n, n, n, N, dx, 0.001, 0.3, 0.0, 0.0, 0.0)
    psi = rng.standard_normal((o.C, n, n, n))
    o.set_state(psi)
    T = o.streaming(orc.LITERAL)
    A = quad_coupling_real3(N)
    f = np.fft.fftfreq(n, d=dx) * 2 * np.pi
    f[n // 2] = 0.0
    ex = np.zeros_like(psi)
    for a in range(3):
        shape = [1, 1, 1, 1]
        shape[3 - a] = n
        D = np.fft.ifft(1j * f.reshape(shape) * np.fft.fft(psi, axis=3 - a), axis=3 - a).real
        ex += np.einsum("ij,jzyx->izyx", A[a], D)
    assert np.abs(T - ex).max() < 1e-12 * np.abs(ex).max()


def test_step_cell_matches_full_step():
    """The one-cell evaluator used for sampled parity at full size == the full step (and uses a different
    derivative evaluation: the direct circulant sum)."""
    rng = np.random.default_rng(33)
    nz, ny, nx, N = 6, 8, 12, 3
    shape = (nz, ny, nx)
    mu_a = rng.uniform(0.01, 0.1, shape)
    mu_s = rng.uniform(5, 20, shape)
    g = rng.uniform(0.8, 0.95, shape)
    S = rng.standard_normal((2, 3, 4))
    C = orc.num_coeffs(3, N)
    psi0 = rng.standard_normal((C,) + shape)

    def make():
        o = orc.Oracle(3, nx, ny, nz, N, 0.1, 0.001, 0.3, mu_a, mu_s, g, pml_width=2, mu_lo=0.01, mu_hi=3.0)
        o.set_source(np.arange(C) + 1.0, S, (3, 2, 2), (4, 3, 2), 1)
        return o

    o = make()
    o.set_state(psi0)
    o.step(1, orc.LITERAL)
    full = o.get_state()
    o2 = make()
    for (x, y, z) in [(0, 0, 0), (4, 3, 2), (11, 7, 5), (5, 4, 3), (1, 6, 0), (6, 4, 3)]:
        v = o2.step_cell(psi0, x, y, z)
        assert np.abs(v - full[:, z, y, x]).max() < 1e-12 * np.abs(psi0).max()


# ------------------------------------------------------------------------------------------------------------------
# P13 — SSP-RK3 (NOT the paper's integrator): stability polynomial, order, stage times, large steps
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim,N,n,form", [(3, 3, 8, orc.PER_AXIS), (2, 4, 12, orc.LITERAL)])
def test_P13_ssprk3_single_mode_stability_polynomial(dim, N, n, form):
    """For u' = M u the Shu-Osher scheme is u_{n+1} = (I + z + z^2/2 + z^3/6) u_n, z = dt M(k), with M(k) built
    independently from quadrature (as in P4)."""
    rng = np.random.default_rng(13 * dim + N)
    dx, c, dt = 0.2, 0.3, 0.05
    mu_a, mu_s, g = 0.02, 4.0, 0.8
    nz = n if dim == 3 else 1
    j = np.array([2, -1, 3][:dim] + [0] * (3 - dim))
    kvec = 2 * np.pi * j / (n * dx)
    C = orc.num_coeffs(dim, N)
    v = rng.standard_normal(C) + 1j * rng.standard_normal(C)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(n), np.arange(n), indexing="ij")
    phase = np.exp(1j * dx * (kvec[0] * x + kvec[1] * y + kvec[2] * z))
    o = orc.Oracle(dim, n, n, nz, N, dx, dt, c, mu_a, mu_s, g)
    o.set_state((v[:, None, None, None] * phase[None]).real)
    steps = 7
    o.step_ssprk3(steps, form)
    Z = dt * mode_matrix(dim, N, kvec, mu_a, mu_s, g, c)
    Pz = np.eye(C) + Z + Z @ Z / 2 + Z @ Z @ Z / 6
    vn = np.linalg.matrix_power(Pz, steps) @ v
    ex = (vn[:, None, None, None] * phase[None]).real
    assert np.abs(o.get_state() - ex).max() < 1e-12 * np.abs(v).max()
    assert abs(o.time_ps() - steps * dt) < 1e-12


def test_P13_ssprk3_third_order_and_stable_where_euler_is_not():
    """(i) error against the matrix exponential falls by ~8 when dt halves; (ii) with mu_s = 0 (no damping) and
    dt = 0.5 dx/c forward Euler amplifies a high mode every step while SSP-RK3 does not (|P(i y)| <= 1 for |y| <= sqrt 3)."""
    from scipy.linalg import expm
    dim, N, n = 3, 3, 8
    dx, c = 0.2, 0.3
    kvec = 2 * np.pi * np.array([1, 2, -1]) / (n * dx)
    C = orc.num_coeffs(dim, N)
    rng = np.random.default_rng(5)
    v = rng.standard_normal(C) + 1j * rng.standard_normal(C)
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    phase = np.exp(1j * dx * (kvec[0] * x + kvec[1] * y + kvec[2] * z))
    M = mode_matrix(dim, N, kvec, 0.02, 4.0, 0.8, c)
    t = 0.4
    ex = ((expm(M * t) @ v)[:, None, None, None] * phase[None]).real
    errs = []
    for steps in (8, 16):
        o = orc.Oracle(dim, n, n, n, N, dx, t / steps, c, 0.02, 4.0, 0.8)
        o.set_state((v[:, None, None, None] * phase[None]).real)
        o.step_ssprk3(steps)
        errs.append(np.abs(o.get_state() - ex).max())
    assert 6.0 < errs[0] / errs[1] < 10.0
    dt = 0.5 * dx / c
    norms = {}
    wgt = np.sqrt(2 * orc.degrees(dim, N) + 1.0)[:, None, None, None]     # streaming is skew-adjoint in this norm (P6)
    for name in ("euler", "ssprk3"):
        o = orc.Oracle(dim, n, n, n, N, dx, dt, c, 0.0, 0.0, 0.0)
        o.set_state((v[:, None, None, None] * phase[None]).real)
        n0 = np.linalg.norm(wgt * o.get_state())
        (o.step if name == "euler" else o.step_ssprk3)(40)
        norms[name] = np.linalg.norm(wgt * o.get_state()) / n0
    assert norms["euler"] > 5.0 and norms["ssprk3"] <= 1.0 + 1e-9


def test_P13_ssprk3_source_stage_times():
    """Uniform medium, uniform isotropic source with Gaussian time profile, psi = 0 initially, no streaming (uniform
    field): the scheme reduces to the scalar SSP-RK3 of y' = -a y + b f(t) with stages at t_n, t_n + dt, t_n + dt/2."""
    n, N, dx, dt, c = 4, 1, 0.3, 0.5, 0.3
    mu_a, mu_s, g = 0.4, 0.0, 0.0
    t0, sig = 1.2, 0.9
    o = orc.Oracle(3, n, n, n, N, dx, dt, c, mu_a, mu_s, g)
    w = np.zeros(o.C); w[0] = 1.0
    o.set_source(w, np.full((n, n, n), 2.5), (0, 0, 0), (n, n, n), 2, t0, sig)
    o.set_state(np.zeros((o.C, n, n, n)))
    f = lambda t: np.exp(-0.5 * ((t - t0) / sig) ** 2)
    E = lambda yv, t: yv + dt * (-c * mu_a * yv + c * 2.5 * f(t))
    yv = 0.0
    for s in range(5):
        tn = s * dt
        u1 = E(yv, tn)
        u2 = 0.75 * yv + 0.25 * E(u1, tn + dt)
        yv = yv / 3 + 2 / 3 * E(u2, tn + dt / 2)
    o.step_ssprk3(5)
    got = o.get_state()
    assert np.abs(got[0] - yv).max() < 1e-13 and np.abs(got[1:]).max() < 1e-15


# ------------------------------------------------------------------------------------------------------------------
# P14 — the steady-state operator L = T + sigma_l of eq.(9)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim,N,n,form", [(3, 3, 8, orc.PER_AXIS), (3, 2, 8, orc.LITERAL), (2, 4, 12, orc.PER_AXIS)])
def test_P14_operator_on_a_single_mode_is_minus_M_over_c(dim, N, n, form):
    """L Re(v e^{ik.r}) = Re(-(M(k)/c) v e^{ik.r}) with M(k) = -c(i k.A + diag sigma) built from quadrature (P4's)."""
    rng = np.random.default_rng(14 + dim)
    dx, c = 0.2, 0.3
    mu_a, mu_s, g = 0.02, 4.0, 0.8
    nz = n if dim == 3 else 1
    j = np.array([1, -2, 3][:dim] + [0] * (3 - dim))
    kvec = 2 * np.pi * j / (n * dx)
    C = orc.num_coeffs(dim, N)
    v = rng.standard_normal(C) + 1j * rng.standard_normal(C)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(n), np.arange(n), indexing="ij")
    phase = np.exp(1j * dx * (kvec[0] * x + kvec[1] * y + kvec[2] * z))
    o = orc.Oracle(dim, n, n, nz, N, dx, 1.0, c, mu_a, mu_s, g)
    got = o.apply_operator((v[:, None, None, None] * phase[None]).real, form)
    M = mode_matrix(dim, N, kvec, mu_a, mu_s, g, c)
    ex = (((-M / c) @ v)[:, None, None, None] * phase[None]).real
    assert np.abs(got - ex).max() < 1e-12 * np.abs(ex).max()


def test_P14_operator_diagonal_in_layer_and_omega():
    """A uniform field has T = 0: L x = sigma_l(r) x cell by cell — mu_b in the layer for every l, mu_a+mu_s(1-g^l) in
    Omega (hand-written degrees, explicit PML cells: P10's formula)."""
    n, W, N = 12, 3, 2
    mu_a, mu_s, g, lo, hi = 0.05, 7.0, 0.8, 0.05, 2.0
    o = orc.Oracle(3, n, n, n, N, 0.1, 1.0, 0.3, mu_a, mu_s, g, pml_width=W, mu_lo=lo, mu_hi=hi)
    y = o.apply_operator(np.ones((o.C, n, n, n)))
    L = hand_degrees(3, N)
    assert np.allclose(y[:, 6, 6, 6], mu_a + mu_s * (1 - g ** L), rtol=0, atol=1e-14)
    assert np.allclose(y[:, 6, 6, 0], hi, rtol=0, atol=1e-14)                       # outer face: delta = 1
    first = lo + (hi - lo) * 0.5 * (1 - math.cos(math.pi / W))                     # first layer cell: delta = 1/W
    assert np.allclose(y[:, 6, W - 1, 6], first, rtol=0, atol=1e-14)
    # and the Euler step is psi - c dt (L psi - q): tie the operator to eq.(11) on random data
    rng = np.random.default_rng(3)
    psi = rng.standard_normal((o.C, n, n, n))
    o2 = orc.Oracle(3, n, n, n, N, 0.1, 0.01, 0.3, mu_a, mu_s, g, pml_width=W, mu_lo=lo, mu_hi=hi)
    o2.set_state(psi)
    o2.step(1)
    assert np.abs(o2.get_state() - (psi - 0.3 * 0.01 * o2.apply_operator(psi))).max() < 1e-13


# ------------------------------------------------------------------------------------------------------------------
# P15 — the Krylov steady-state solve: dense solve on a tiny grid, closed form, true residual
# ------------------------------------------------------------------------------------------------------------------
def test_P15_gmres_equals_dense_solve_on_a_tiny_grid():
    n, N = 6, 1
    rng = np.random.default_rng(15)
    mu_a = rng.uniform(0.05, 0.5, (n, n, n)); mu_s = rng.uniform(1, 4, (n, n, n)); g = rng.uniform(0.5, 0.9, (n, n, n))
    o = orc.Oracle(3, n, n, n, N, 0.3, 1.0, 0.3, mu_a, mu_s, g, pml_width=1, mu_lo=0.05, mu_hi=1.5)
    w = np.array([1.0, 0.2, -0.3, 0.5])
    S = rng.uniform(0, 1, (2, 2, 2))
    o.set_source(w, S, (2, 2, 1), (2, 2, 2), 1)
    q = o.source_field()
    assert np.count_nonzero(q[0]) == 8 and q[:, 0, :, :].max() == 0          # boxed, nothing in the layer
    nunk = o.C * n ** 3
    Lmat = np.zeros((nunk, nunk))
    e = np.zeros(nunk)
    for i in range(nunk):                                                     # dense matrix, column by column
        e[:] = 0; e[i] = 1
        Lmat[:, i] = o.apply_operator(e.reshape(o.C, n, n, n)).ravel()
    ex = np.linalg.solve(Lmat, q.ravel()).reshape(q.shape)
    napp, rr = o.solve_steady(restart=20, tol=1e-12, max_restarts=100)
    got = o.get_state()
    assert rr <= 1e-12 and napp > 5
    assert np.abs(got - ex).max() < 1e-9 * np.abs(ex).max()
    assert np.linalg.norm(o.apply_operator(got) - q) <= 2e-12 * np.linalg.norm(q)   # its own true residual


@pytest.mark.parametrize("dim", [2, 3])
def test_P15_gmres_uniform_source_closed_form(dim):
    """Uniform constant source in a uniform periodic medium: psi_c = q_c / sigma_l (P7's closed form)."""
    n = 6
    nz = n if dim == 3 else 1
    mu_a, mu_s, g = 0.5, 3.0, 0.5
    o = orc.Oracle(dim, n, n, nz, 2, 0.1, 1.0, 0.3, mu_a, mu_s, g)
    w = np.arange(1, o.C + 1) * 0.25
    o.set_source(w, np.full((nz, n, n), 2.0), (0, 0, 0), (n, n, nz), 1)
    o.solve_steady(restart=10, tol=1e-13, max_restarts=20)
    L = hand_degrees(dim, 2)
    fixed = 2.0 * w / (mu_a + mu_s * (1 - g ** L))
    assert np.abs(o.get_state() - fixed[:, None, None, None]).max() < 1e-11 * fixed.max()


def test_P15_steady_state_is_the_fixed_point_of_the_paper_step():
    """The GMRES solution does not move under the paper's Euler step eq.(11) with the same constant source."""
    n, N = 8, 2
    rng = np.random.default_rng(16)
    mu_s = rng.uniform(2, 6, (n, n, n))
    o = orc.Oracle(3, n, n, n, N, 0.25, 0.01, 0.3, 0.1, mu_s, 0.7, pml_width=2, mu_lo=0.1, mu_hi=2.0)
    w = np.zeros(o.C); w[0] = 1.0; w[2] = 0.5
    o.set_source(w, np.ones((1, 2, 2)), (3, 3, 3), (2, 2, 1), 1)
    o.solve_steady(restart=30, tol=1e-12, max_restarts=200)
    ss = o.get_state()
    o.step(5)
    assert np.abs(o.get_state() - ss).max() < 1e-11 * np.abs(ss).max()


# ------------------------------------------------------------------------------------------------------------------
# P16 — exponential (integrating-factor) Euler step: exact diagonal, exact source response
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim,form", [(3, orc.PER_AXIS), (2, orc.LITERAL)])
def test_P16_exp_step_uniform_decay_is_exact(dim, form):
    n, N = 6, 3
    nz = n if dim == 3 else 1
    mu_a, mu_s, g, c, dt = 0.013, 9.0, 0.87, 0.3, 0.35            # c dt sigma_l up to ~0.4: Euler would be far off
    o = orc.Oracle(dim, n, n, nz, N, 0.1, dt, c, mu_a, mu_s, g)
    amp = 1.0 + np.arange(o.C)
    o.set_state(np.broadcast_to(amp[:, None, None, None], (o.C, nz, n, n)))
    o.step_exp(11, form)
    L = hand_degrees(dim, N)
    ex = amp * np.exp(-c * (mu_a + mu_s * (1 - g ** L)) * 11 * dt)
    # (round-off of the spectral derivative of a constant, ~1e-14 k_max, enters times c dt = 0.1 per step)
    assert np.abs(o.get_state() - ex[:, None, None, None]).max() < 1e-11 * amp.max()
    assert abs(o.time_ps() - 11 * dt) < 1e-15


def test_P16_exp_step_exact_in_layer_and_source_response():
    """Whole-domain layer: every l decays as exp(-c mu_b t) exactly.  Uniform constant source from zero:
    psi_c(t_n) = (q_c/sigma_l)(1 - exp(-c sigma_l t_n)) exactly (phi_1 weighting), fixed point q_c/sigma_l."""
    n, c, dt = 8, 0.3, 0.5
    o = orc.Oracle(3, n, n, n, 2, 0.1, dt, c, 0.01, 10.0, 0.9, pml_width=4, mu_lo=0.7, mu_hi=0.7)
    amp = 1.0 + np.arange(o.C)
    o.set_state(np.broadcast_to(amp[:, None, None, None], (o.C, n, n, n)))
    o.step_exp(6)
    assert np.abs(o.get_state() - (amp * math.exp(-c * 0.7 * 6 * dt))[:, None, None, None]).max() < 1e-11 * amp.max()
    mu_a, mu_s, g = 0.5, 3.0, 0.5
    o2 = orc.Oracle(3, 4, 4, 4, 2, 0.1, dt, c, mu_a, mu_s, g)
    w = np.arange(1, o2.C + 1) * 0.25
    o2.set_source(w, np.full((4, 4, 4), 2.0), (0, 0, 0), (4, 4, 4), 1)
    o2.step_exp(9)
    sigma = mu_a + mu_s * (1 - g ** hand_degrees(3, 2))
    ex = 2.0 * w / sigma * (1 - np.exp(-c * sigma * 9 * dt))
    assert np.abs(o2.get_state() - ex[:, None, None, None]).max() < 1e-11 * ex.max()


def test_P16_exp_step_single_mode_matrix_and_convergence():
    """One Fourier mode: psi_{n+1} = diag(E) (I - c dt i k.A) psi_n with E = exp(-c dt sigma_l), A from quadrature;
    first-order convergence to expm(M t); and the diagonal no longer limits dt: with streaming switched off by k = 0
    the step is exact at c dt sigma = 6 where eq.(11) blows up."""
    from scipy.linalg import expm
    dim, N, n = 3, 3, 8
    dx, c, dt = 0.2, 0.3, 0.002
    mu_a, mu_s, g = 0.02, 4.0, 0.8
    kvec = 2 * np.pi * np.array([2, -1, 3]) / (n * dx)
    C = orc.num_coeffs(dim, N)
    rng = np.random.default_rng(160)
    v = rng.standard_normal(C) + 1j * rng.standard_normal(C)
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    phase = np.exp(1j * dx * (kvec[0] * x + kvec[1] * y + kvec[2] * z))
    A = quad_coupling(dim, N)
    sigma = mu_a + mu_s * (1 - g ** hand_degrees(dim, N))
    kA = sum(kvec[a] * A[a] for a in range(dim))
    step = np.diag(np.exp(-c * dt * sigma)) @ (np.eye(C) - c * dt * 1j * kA)
    o = orc.Oracle(dim, n, n, n, N, dx, dt, c, mu_a, mu_s, g)
    o.set_state((v[:, None, None, None] * phase[None]).real)
    o.step_exp(20)
    ex = ((np.linalg.matrix_power(step, 20) @ v)[:, None, None, None] * phase[None]).real
    assert np.abs(o.get_state() - ex).max() < 1e-12 * np.abs(v).max()
    M = mode_matrix(dim, N, kvec, mu_a, mu_s, g, c)
    t, errs = 0.04, []
    for steps in (20, 40):
        o = orc.Oracle(dim, n, n, n, N, dx, t / steps, c, mu_a, mu_s, g)
        o.set_state((v[:, None, None, None] * phase[None]).real)
        o.step_exp(steps)
        errs.append(np.abs(o.get_state() - ((expm(M * t) @ v)[:, None, None, None] * phase[None]).real).max())
    assert 1.7 < errs[0] / errs[1] < 2.3
    # stiff diagonal: c dt sigma_1 = 0.3 * 20 * 1.0 = 6
    big = orc.Oracle(dim, n, n, n, 1, dx, 20.0, c, 0.5, 1.0, 0.5)
    big.set_state(np.ones((4, n, n, n)))
    big.step_exp(3)
    assert np.allclose(big.get_state()[1], math.exp(-c * 1.0 * 60.0), rtol=1e-12, atol=0)
    eul = orc.Oracle(dim, n, n, n, 1, dx, 20.0, c, 0.5, 1.0, 0.5)
    eul.set_state(np.ones((4, n, n, n)))
    eul.step(3)
    assert abs(eul.get_state()[1, 0, 0, 0]) > 100          # (1 - 6)^3 = -125
