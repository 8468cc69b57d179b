"""GPU parity for the round-2 rows (SURVEY 8(b) general extents, 8(f1) operator + Krylov steady state, 8(f2) exponential
step, CUDA-graph stepping): the CUDA path through the C ABI against the fp64 oracle on the same seeded fp32 inputs.
Same acceptance as test_gpu_parity.py.  Run with -m gpu."""
import numpy as np
import pytest
import torch

import paper_1801_06364_b200 as rte
import rte_workloads as wl
from oracle import rte_oracle as orc
from test_gpu_parity import DEV, assert_parity, dev, field_errors, gpu_create, gpu_state, make_oracle, run_both

pytestmark = pytest.mark.gpu


def random_case(dim, nx, ny, nz, N, dx=0.2, dt=0.002, W=3, seed=0):
    rng = np.random.default_rng(seed + nx * 7 + ny * 3 + nz + N)
    cfg = wl.Config("rand", dim, nx, ny, nz, N, dx, dt, 0.3, 3, (W, 0.01, 2.0), "random", "box", 0)
    mu_a = rng.uniform(0.01, 0.5, cfg.shape).astype(np.float32)
    mu_s = rng.uniform(2.0, 20.0, cfg.shape).astype(np.float32)
    g = rng.uniform(0.7, 0.95, cfg.shape).astype(np.float32)
    ext = (5, 4, 3 if dim == 3 else 1)
    src = dict(w=rng.standard_normal(cfg.C).astype(np.float32), S=rng.standard_normal(ext[::-1]).astype(np.float32),
               origin=(1, 2, 4 if dim == 3 else 0), extent=ext, kind=1, t0=0.0, sigma_t=1.0)
    return cfg, mu_a, mu_s, g, src


# ---- every pencil length the generic kernels add this round (even 2^a 3^b), on every axis position ------------------------
NEW_SHAPES_3D = [(18, 24, 36, 3), (36, 18, 24, 2), (24, 36, 18, 1), (54, 16, 72, 3), (72, 54, 16, 2), (16, 72, 54, 3),
                 (108, 16, 16, 3), (16, 144, 16, 2), (16, 16, 162, 3), (216, 16, 16, 1), (16, 288, 16, 3), (16, 16, 324, 2),
                 (432, 16, 16, 3), (16, 486, 16, 1), (16, 16, 576, 3), (648, 16, 16, 2), (16, 768, 16, 3), (16, 16, 864, 1),
                 (972, 16, 16, 3), (16, 1024, 16, 2), (16, 16, 1024, 3)]


@pytest.mark.parametrize("nx,ny,nz,N", NEW_SHAPES_3D)
def test_general_extents_3d(nx, ny, nz, N):
    cfg, mu_a, mu_s, g, src = random_case(3, nx, ny, nz, N)
    got, ref, _ = run_both(cfg, mu_a, mu_s, g, wl.random_state(cfg, seed=N), src, cfg.steps)
    assert_parity(got, ref, f"{nx}x{ny}x{nz} P{N}")


@pytest.mark.parametrize("nx,ny,N", [(18, 54, 3), (144, 24, 2), (1024, 16, 3), (36, 972, 1), (768, 108, 4)])
def test_general_extents_2d(nx, ny, N):
    cfg, mu_a, mu_s, g, src = random_case(2, nx, ny, 1, N, dx=0.1, dt=0.001, W=4)
    got, ref, _ = run_both(cfg, mu_a, mu_s, g, wl.random_state(cfg, seed=N), src, 4)
    assert_parity(got, ref, f"{nx}x{ny} P{N}")


def test_unsupported_extents_are_rejected():
    for n in (20, 27, 81, 100, 2048):
        with pytest.raises(rte.RteError) as e:
            rte.rte_create((3, n, 16, 16), 1, 0.1, 0.001, 0.3, 0.01, 10.0, 0.9)
        assert e.value.code == rte.RTE_EINVAL
    with pytest.raises(rte.RteError) as e:      # one pencil of all coefficients must fit a shared-memory tile
        rte.rte_create((3, 1024, 16, 16), 9, 0.1, 0.001, 0.3, 0.01, 10.0, 0.9)
    assert e.value.code == rte.RTE_EUNSUPPORTED


# ---- the steady-state operator and the device-resident GMRES -------------------------------------------------
@pytest.mark.parametrize("shape,N,maps", [((32, 48, 16), 3, True), ((64, 64, 1), 4, True), ((128, 128, 128), 3, False),
                                          ((18, 24, 36), 2, True)])
def test_apply_operator_vs_oracle(shape, N, maps):
    """y = L x = T[x] + sigma_l x on random x: generic kernels (maps, PML), 2-D, and the specialised cfg2 kernels with
    scalar media (the uniform-g instance) at 128^3."""
    nx, ny, nz = shape
    dim = 3 if nz > 1 else 2
    cfg, mu_a, mu_s, g, _ = random_case(dim, nx, ny, nz, N, W=4)
    if not maps:
        mu_a, mu_s, g = 0.02, 8.0, 0.85
    ctx = gpu_create(cfg, mu_a, mu_s, g)
    x = wl.random_state(cfg, seed=11)
    xd = dev(x)
    yd = torch.empty_like(xd)
    rte.rte_set_state(ctx, dev(wl.random_state(cfg, seed=12)))
    before = gpu_state(ctx, cfg)
    rte.rte_apply_operator(ctx, xd, yd)
    rte.rte_sync(ctx)
    got = yd.cpu().numpy().astype(np.float64)
    ref = make_oracle(cfg, mu_a, mu_s, g).apply_operator(x)
    assert_parity(got, ref, f"operator {shape} P{N}")
    assert np.array_equal(before, gpu_state(ctx, cfg)) and rte.rte_time_ps(ctx) == 0.0     # state and clock untouched


def steady_case(n, N, W, n_incl, dx):
    cfg = wl.reduced(wl.CONFIGS["cfg3"], n, pml_width=W, dx=dx)
    cfg = wl.replace(cfg, n_inclusions=n_incl, N=N)
    return cfg, wl.media_maps(cfg), wl.source_term(cfg)


@pytest.mark.parametrize("n,N,W,dx,otol,prec", [(32, 3, 5, 0.16, 1e-10, False), (32, 3, 5, 0.16, 1e-10, True),
                                                 (48, 5, 6, 0.2, 1e-8, True)])
def test_solve_steady_vs_oracle(n, N, W, dx, otol, prec):
    """Converged steady state of the cfg3 structure (ellipsoid inclusions with varying mu_a, mu_s, g; PML; constant
    collimated source): device GMRES(30) in fp32 against the oracle's fp64 GMRES solved to 1e-10 (32^3 P_3) / 1e-8
    (48^3 P_5: the size the plain oracle finishes in minutes)."""
    cfg, (mu_a, mu_s, g), src = steady_case(n, N, W, 8, dx)
    ctx = gpu_create(cfg, mu_a, mu_s, g)
    rte.rte_set_source(ctx, src["w"], dev(src["S"]), src["origin"], src["extent"], 1)
    if prec:      # GMRES on (I - Phi^s) psi = Phi^s(0; q), Phi = one SSP-RK3 step at 0.3 dx/c
        napp, rr = rte.rte_solve_steady(ctx, restart=20, tol=2e-6, max_restarts=60, precond_steps=8,
                                        precond_dt_ps=0.3 * cfg.dx / cfg.c)
    else:
        napp, rr = rte.rte_solve_steady(ctx, restart=30, tol=2e-6, max_restarts=60)
    got = gpu_state(ctx, cfg)
    o = make_oracle(cfg, mu_a, mu_s, g)
    o.set_source(src["w"], src["S"], src["origin"], src["extent"], 1)
    onapp, orr = o.solve_steady(restart=30 if n <= 32 else 60, tol=otol, max_restarts=200)
    ref = o.get_state()
    assert orr <= otol and rr <= 2e-6, (rr, orr)
    assert 10 < napp < (40 if prec else 4) * onapp
    assert_parity(got, ref, f"steady {n}^3 P{N} ({napp} applications, oracle {onapp})")
    # the oracle's own true residual of the GPU field (fp64 operator on the fp32 solution)
    q = o.source_field()
    assert np.linalg.norm(o.apply_operator(got) - q) <= 1e-4 * np.linalg.norm(q)


def test_solve_steady_uniform_source_breakdown_and_restart_from_solution():
    """Uniform source, uniform periodic medium: the Krylov space is exhausted after a few steps (happy breakdown) and
    psi_c = q_c / sigma_l exactly (P7's closed form); solving again from the solution does (almost) no work."""
    cfg = wl.Config("uni", 3, 16, 16, 16, 2, 0.1, 0.01, 0.3, 1, (0, 0.0, 0.0), "homogeneous", "box", 0)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, 0.5, 3.0, 0.5)
    w = (np.arange(1, cfg.C + 1) * 0.25).astype(np.float32)
    rte.rte_set_source(ctx, w, dev(np.full(cfg.shape, 2.0, np.float32)), (0, 0, 0), (16, 16, 16), 1)
    napp, rr = rte.rte_solve_steady(ctx, restart=12, tol=1e-6, max_restarts=5)
    L = np.array([0, 1, 1, 1, 2, 2, 2, 2, 2])
    fixed = 2.0 * w / (0.5 + 3.0 * (1 - 0.5 ** L))
    got = gpu_state(ctx, cfg)
    assert rr <= 1e-6 and napp <= 12
    assert np.abs(got - fixed[:, None, None, None]).max() <= 2e-6 * fixed.max()
    napp2, rr2 = rte.rte_solve_steady(ctx, restart=12, tol=1e-6, max_restarts=5)
    assert napp2 == 1 and rr2 <= 1e-6
    with pytest.raises(rte.RteError):
        rte.rte_solve_steady(ctx, restart=65)
    rte.rte_set_source(ctx, None, None, None, None, 0)
    with pytest.raises(rte.RteError):
        rte.rte_solve_steady(ctx, restart=8)


# ---- exponential (integrating-factor) Euler step -------------------------------------------------------------
@pytest.mark.parametrize("shape,N,dt", [((32, 48, 16), 3, 0.004), ((64, 96, 1), 4, 0.002), ((128, 16, 16), 2, 0.05)])
def test_exp_step_vs_oracle(shape, N, dt):
    nx, ny, nz = shape
    dim = 3 if nz > 1 else 2
    cfg, mu_a, mu_s, g, src = random_case(dim, nx, ny, nz, N, dt=dt, W=4)
    if dt >= 0.05:                       # stiff diagonal (c dt sigma up to ~3: eq.(11) would diverge), weak streaming
        cfg = wl.replace(cfg, dx=2.0)
    src = dict(src, kind=2, t0=3 * dt, sigma_t=2 * dt)
    psi0 = wl.random_state(cfg, seed=N)
    ctx = gpu_create(cfg, mu_a, mu_s, g)
    rte.rte_set_state(ctx, dev(psi0))
    rte.rte_set_source(ctx, src["w"], dev(src["S"]), src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
    o = make_oracle(cfg, mu_a, mu_s, g)
    o.set_state(psi0)
    o.set_source(src["w"], src["S"], src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
    rte.rte_step_exp(ctx, 6)
    o.step_exp(6)
    assert_parity(gpu_state(ctx, cfg), o.get_state(), f"exp step {shape} P{N}")
    assert abs(rte.rte_time_ps(ctx) - 6 * dt) < 1e-6


@pytest.mark.parametrize("name", ["cfg2", "cfg0"])
def test_exp_step_on_specialised_grids_vs_oracle(name):
    """The grids of the BASELINE configurations take the two-kernel route of rte_step_exp (specialised passes for -c dt T,
    then the pointwise exp / phi_1 / source kernel): cfg2 at full size with scalar media (uniform-g instance), PML and its
    temporal-Gaussian source; cfg0's grid with a PML, maps and a constant source."""
    if name == "cfg2":
        cfg = wl.CONFIGS["cfg2"]
        mu_a, mu_s, g = (float(v) for v in cfg.background)
        src = wl.source_term(cfg)
        src = dict(src, t0=2 * cfg.dt, sigma_t=1.5 * cfg.dt)
        steps = 4
    else:
        cfg = wl.Config("cfg0pml", 2, 64, 64, 1, 3, 0.1, 0.002, 0.3, 12, (8, 0.01, 5.0), "random", "box", 0)
        rng = np.random.default_rng(40)
        mu_a = rng.uniform(0.01, 0.5, cfg.shape).astype(np.float32)
        mu_s = rng.uniform(2.0, 20.0, cfg.shape).astype(np.float32)
        g = rng.uniform(0.7, 0.95, cfg.shape).astype(np.float32)
        src = dict(w=rng.standard_normal(cfg.C).astype(np.float32), S=rng.standard_normal((1, 7, 9)).astype(np.float32),
                   origin=(5, 20, 0), extent=(9, 7, 1), kind=1, t0=0.0, sigma_t=1.0)      # the box reaches into the PML
        steps = 12
    psi0 = wl.random_state(cfg, seed=8)
    ctx = gpu_create(cfg, mu_a, mu_s, g)
    rte.rte_set_state(ctx, dev(psi0))
    rte.rte_set_source(ctx, src["w"], dev(src["S"]), src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
    o = make_oracle(cfg, mu_a, mu_s, g)
    o.set_state(psi0)
    o.set_source(src["w"], src["S"], src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
    l0 = rte.rte_launch_count(ctx)
    rte.rte_step_exp(ctx, steps)
    assert rte.rte_launch_count(ctx) - l0 == steps * (cfg.dim + 1)          # passes + the finish kernel: the two-kernel route
    o.step_exp(steps)
    assert_parity(gpu_state(ctx, cfg), o.get_state(), f"exp step on {name}'s grid")


def test_exp_step_uniform_decay_exact_on_device():
    """P16 on the device: a uniform field decays as exp(-c sigma_l t) with no O(dt) error at c dt sigma_l ~ 1."""
    cfg = wl.Config("uni", 3, 16, 16, 16, 3, 0.1, 0.35, 0.3, 1, (0, 0.0, 0.0), "homogeneous", "none", 0)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, 0.013, 9.0, 0.87)
    amp = (1.0 + np.arange(cfg.C)).astype(np.float32)
    rte.rte_set_state(ctx, dev(np.broadcast_to(amp[:, None, None, None], (cfg.C,) + cfg.shape).copy()))
    rte.rte_step_exp(ctx, 11)
    L = np.array([int(np.floor(np.sqrt(c))) for c in range(cfg.C)])
    ex = amp * np.exp(-0.3 * (0.013 + 9.0 * (1 - 0.87 ** L)) * 11 * 0.35)
    got = gpu_state(ctx, cfg)
    assert np.abs(got / ex[:, None, None, None] - 1).max() < 2e-5


# ---- CUDA-graph replay on L2-resident grids --------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim", [2, 3])
def test_graph_stepping_is_bit_identical_to_eager(dim):
    """rte_step(n) with n > 32 on a small grid replays captured launches; the time-dependent source amplitude comes from
    a device table.  Same bits as n single eager steps, and both match the oracle."""
    nz = 32 if dim == 3 else 1
    cfg, mu_a, mu_s, g, src = random_case(dim, 64, 48, nz, 3, dx=0.1, dt=0.001, W=4)
    src = dict(src, kind=2, t0=0.04, sigma_t=0.02)
    psi0 = wl.random_state(cfg, seed=5)
    states = []
    for mode in ("graph", "eager"):
        ctx = gpu_create(cfg, mu_a, mu_s, g)
        rte.rte_set_state(ctx, dev(psi0))
        rte.rte_set_source(ctx, src["w"], dev(src["S"]), src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
        if mode == "graph":
            rte.rte_step(ctx, 70)       # 1 eager + 2 x 32 replayed + 5 eager
            rte.rte_step(ctx, 37)       # 1 x 32 replayed + 5 eager
        else:
            for _ in range(107):
                rte.rte_step(ctx, 1)
        assert abs(rte.rte_time_ps(ctx) - 107 * cfg.dt) < 1e-6          # dt is an fp32 argument
        states.append(gpu_state(ctx, cfg))
    assert np.array_equal(states[0], states[1])
    o = make_oracle(cfg, mu_a, mu_s, g)
    o.set_state(psi0)
    o.set_source(src["w"], src["S"], src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
    o.step(107)
    assert_parity(states[0], o.get_state(), "graph stepping")


# ---- the cuFFT-backed literal variant (reference point, not the product) vs the oracle's LITERAL formulation ----
@pytest.mark.parametrize("shape,N", [((32, 48, 16), 3), ((16, 18, 20), 2)])
def test_cufft_literal_reference_point_vs_oracle_literal(shape, N):
    from baseline import cufft_literal as cl
    nx, ny, nz = shape
    cfg, mu_a, mu_s, g, _ = random_case(3, nx, ny, nz, N, W=3)
    o = make_oracle(cfg, mu_a, mu_s, g)
    mu_b, inside = orc.pml_map(3, nx, ny, nz, *cfg.pml)
    ins = inside.reshape(cfg.shape).astype(bool)
    sa = np.where(ins, mu_a, mu_b.reshape(cfg.shape)).astype(np.float32)
    ss = np.where(ins, mu_s, 0.0).astype(np.float32)
    psi0 = wl.random_state(cfg, seed=21)
    sol = cl.Solver(nx, ny, nz, N, cfg.dx, cfg.dt, cfg.c, dev(sa), dev(ss), dev(g))
    pc = cl.real_to_complex(dev(psi0))
    assert torch.allclose(cl.complex_to_real(pc), dev(psi0), atol=1e-6)          # R6 round trip
    sol.set_state(pc)
    sol.step(5)
    out_c = sol.get_state()
    got = cl.complex_to_real(out_c).cpu().numpy().astype(np.float64)
    # a real radiance keeps psi_l^-m = (-1)^m conj(psi_l^m): the imaginary remainder of the reconstruction is round-off
    l, m = 2, 1
    sym = out_c[l * l + l - m] - ((-1) ** m) * torch.conj(out_c[l * l + l + m])
    assert float(sym.abs().max()) <= 1e-5 * float(out_c[l * l + l + m].abs().max())
    o.set_state(psi0)
    o.step(5, orc.LITERAL)
    assert_parity(got, o.get_state(), f"cufft literal {shape} P{N}")


def test_graph_survives_source_changes_and_other_integrators():
    """The captured launches hold the source box by value and the state buffers by address: rte_set_source drops the graph,
    and a step of another integrator (which leaves the state in a different buffer) must not let a replay read stale data."""
    cfg, mu_a, mu_s, g, src = random_case(2, 64, 48, 1, 3, dx=0.1, dt=0.001, W=4)
    rng = np.random.default_rng(77)
    src2 = dict(w=rng.standard_normal(cfg.C).astype(np.float32), S=rng.standard_normal((1, 9, 11)).astype(np.float32),
                origin=(20, 10, 0), extent=(11, 9, 1), kind=1, t0=0.0, sigma_t=1.0)
    psi0 = wl.random_state(cfg, seed=6)
    ctx = gpu_create(cfg, mu_a, mu_s, g)
    o = make_oracle(cfg, mu_a, mu_s, g)
    rte.rte_set_state(ctx, dev(psi0))
    o.set_state(psi0)
    for s_ in (src, src2):
        rte.rte_set_source(ctx, s_["w"], dev(s_["S"]), s_["origin"], s_["extent"], s_["kind"], s_["t0"], s_["sigma_t"])
        o.set_source(s_["w"], s_["S"], s_["origin"], s_["extent"], s_["kind"], s_["t0"], s_["sigma_t"])
        rte.rte_step(ctx, 70)                 # graph replays
        o.step(70)
        rte.rte_step_ssprk3(ctx, 1)           # leaves the state in the other buffer
        o.step_ssprk3(1)
        rte.rte_step(ctx, 41)                 # replays again: must pick up the right buffer
        o.step(41)
    assert_parity(gpu_state(ctx, cfg), o.get_state(), "graph + source change + ssprk3")
    assert abs(rte.rte_time_ps(ctx) - o.time_ps()) < 1e-6


def test_solve_steady_2d_vs_oracle():
    """2-D steady state (circular harmonics P_4, disks, PML, constant source), preconditioned GMRES vs the oracle's GMRES."""
    cfg = wl.reduced(wl.CONFIGS["cfg1"], 64, pml_width=6, dx=0.25)
    cfg = wl.replace(cfg, N=4, n_inclusions=5)
    mu_a, mu_s, g = wl.media_maps(cfg)
    w = np.zeros(cfg.C, np.float32); w[0] = 1.0; w[1] = 0.5
    S = np.ones((1, 3, 3), np.float32)
    ctx = gpu_create(cfg, mu_a, mu_s, g)
    rte.rte_set_source(ctx, w, dev(S), (30, 31, 0), (3, 3, 1), 1)
    napp, rr = rte.rte_solve_steady(ctx, restart=20, tol=2e-6, max_restarts=60, precond_steps=6,
                                    precond_dt_ps=0.3 * cfg.dx / cfg.c)
    o = make_oracle(cfg, mu_a, mu_s, g)
    o.set_source(w, S, (30, 31, 0), (3, 3, 1), 1)
    _, orr = o.solve_steady(restart=40, tol=1e-10, max_restarts=200)
    assert orr <= 1e-10 and rr <= 2e-6, (rr, orr)
    assert_parity(gpu_state(ctx, cfg), o.get_state(), f"2-D steady ({napp} sweeps)")


# ---- instability / NaN guard --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim", [3, 2])
def test_energy_guard(dim):
    """rte_energy = sum_c w_l ||psi_c||^2 (w = 2l+1 in 3-D; 1, 2, 2, ... in 2-D) against numpy; it never grows in a source-free
    run at the dt recommended by rte_stable_dt and blows up at 4x the bound (reading R10); NaNs are counted, not summed."""
    n, N, dx, c = 32, 3, 0.2, 0.3
    med = (0.02, 4.0, 0.8)
    nz = n if dim == 3 else 1
    bound, dt_ok = rte.rte_stable_dt(dim, N, n, dx, c, *med)
    cfg = wl.Config("e", dim, n, n, nz, N, dx, dt_ok, c, 0, (0, 0.0, 0.0), "homogeneous", "none", 0)
    psi0 = wl.random_state(cfg, seed=9, decay=1.0)          # white in space and degree: every mode up to the corner Nyquist
    L = np.array([int(np.floor(np.sqrt(i))) for i in range(cfg.C)]) if dim == 3 else np.array([0] + [m for m in range(1, N + 1) for _ in range(2)])
    w = (2 * L + 1) if dim == 3 else np.where(L == 0, 1.0, 2.0)
    ctx = rte.rte_create(cfg.grid, N, dx, dt_ok, c, *med)
    rte.rte_set_state(ctx, dev(psi0))
    e0, bad = rte.rte_energy(ctx)
    ref = float((w[:, None, None, None] * psi0.astype(np.float64) ** 2).sum())
    assert bad == 0 and abs(e0 / ref - 1) < 1e-6
    prev = e0
    for _ in range(8):
        rte.rte_step(ctx, 25)
        e, bad = rte.rte_energy(ctx)
        assert bad == 0 and e <= prev * (1 + 1e-6)
        prev = e
    # 4x the bound: the corner modes are amplified every step
    ctx2 = rte.rte_create(cfg.grid, N, dx, 4.0 * bound, c, *med)
    rte.rte_set_state(ctx2, dev(psi0))
    rte.rte_step(ctx2, 200)
    e2, _ = rte.rte_energy(ctx2)
    assert e2 > 10 * e0
    # NaNs / Infs are counted and kept out of the sum
    bad_state = psi0.copy()
    bad_state[1, 0, 3, 4] = np.nan
    bad_state[2, 0, 5, 6] = np.inf
    rte.rte_set_state(ctx, dev(bad_state))
    e3, bad3 = rte.rte_energy(ctx)
    assert bad3 == 2 and np.isfinite(e3) and e3 < e0


def test_exchange_microbenchmark_runs_and_both_variants_transpose():
    """DESIGN.md 6 "Why no warp-shuffle butterflies": the micro-benchmark that measured the 16 x 16 inter-factor exchange through
    shared memory against a warp-shuffle butterfly transpose (B200: 0.45 vs 0.63 ps per element, profiles/r2_exchange_microbench.md).
    Here: it runs and both variants produce the transpose; the timing is printed, not asserted."""
    import json
    import os
    import subprocess
    exe = os.path.join(os.path.dirname(os.path.abspath(__file__)), "microbench", "exchange_bench")
    if not os.path.exists(exe):
        pytest.skip("tests/microbench/exchange_bench not built (python __graft_entry__.py)")
    out = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert out.returncode == 0, out.stdout + out.stderr
    res = json.loads(out.stdout.strip().splitlines()[-1])
    print(res)
    assert res["smem_ok"] and res["shfl_ok"] and res["smem_ms"] > 0 and res["shfl_ms"] > 0
