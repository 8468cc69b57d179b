"""GPU parity: the CUDA path (through the C ABI of include/rte.h) against the fp64 oracle on the same seeded fp32
inputs.  Acceptance (BASELINE.json north_star): relative L2 error <= 1e-4 on every coefficient field (fields whose
oracle norm is below 1e-6 ||psi_0|| are judged against that floor) and max pointwise fluence error <= 1e-3 of the
fluence maximum.  All tests need a B200: run with -m gpu.
"""
import math

import numpy as np
import pytest
import torch

import paper_1801_06364_b200 as rte
import rte_workloads as wl
from oracle import rte_oracle as orc

pytestmark = pytest.mark.gpu

TOL_FIELD = 1e-4
TOL_FLUENCE = 1e-3
DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def gpu_create(cfg, mu_a, mu_s, g):
    """Media as numpy maps (-> device maps) or python floats (-> 1-value device arrays: is_map = 0, which is what
    bench.py passes for homogeneous workloads and what selects the uniform-g kernel instances)."""
    m = [v if isinstance(v, float) else dev(v) for v in (mu_a, mu_s, g)]
    return rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, m[0], m[1], m[2], cfg.pml)


def media_of(cfg, kind):
    """'maps': full fp32 maps from the CPU generators; 'scalars': the background as three python floats (homogeneous
    configs only) — bench.py's launch configuration for cfg0 / cfg2 (bench.py device_media)."""
    if kind == "maps":
        return wl.media_maps(cfg)
    assert cfg.media == "homogeneous"
    return tuple(float(v) for v in cfg.background)


def gpu_state(ctx, cfg):
    out = torch.empty((cfg.C,) + cfg.shape, dtype=torch.float32, device=DEV)
    rte.rte_get_state(ctx, out)
    rte.rte_sync(ctx)
    return out.cpu().numpy().astype(np.float64)


def make_oracle(cfg, mu_a, mu_s, g):
    return orc.Oracle(cfg.dim, cfg.nx, cfg.ny, cfg.nz, cfg.N, cfg.dx, cfg.dt, cfg.c, mu_a, mu_s, g, *cfg.pml)


def field_errors(got, ref):
    n0 = np.linalg.norm(ref[0])
    return np.array([np.linalg.norm(got[c] - ref[c]) / max(np.linalg.norm(ref[c]), 1e-6 * n0) for c in range(ref.shape[0])])


def assert_parity(got, ref, what=""):
    assert np.isfinite(got).all(), f"{what}: non-finite GPU output"
    err = field_errors(got, ref)
    assert err.max() <= TOL_FIELD, f"{what}: per-field rel L2 error {err.max():.3e} (field {err.argmax()})"
    fl = np.abs(got[0] - ref[0]).max() / np.abs(ref[0]).max()
    assert fl <= TOL_FLUENCE, f"{what}: fluence error {fl:.3e} of max"
    return err.max(), fl


def run_both(cfg, mu_a, mu_s, g, psi0, src, steps):
    ctx = gpu_create(cfg, mu_a, mu_s, g)
    rte.rte_set_state(ctx, dev(psi0))
    o = make_oracle(cfg, mu_a, mu_s, g)
    o.set_state(psi0)
    if src is not None:
        rte.rte_set_source(ctx, src["w"], dev(src["S"]), src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
        o.set_source(src["w"], src["S"], src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
    rte.rte_step(ctx, steps)
    got = gpu_state(ctx, cfg)
    o.step(steps)
    ref = o.get_state()
    assert abs(rte.rte_time_ps(ctx) - o.time_ps()) < 1e-9 * max(1.0, o.time_ps()) + 1e-6 * steps * cfg.dt
    return got, ref, ctx


# ---------------------------------------------------------------------------------------------------------------------
# every supported pencil length, on every axis position, several orders (N even -> padded pair), random heterogeneous
# media, PML, box source: a few steps from a random state
# ---------------------------------------------------------------------------------------------------------------------
SHAPES_3D = [
    (16, 32, 48, 3), (48, 16, 32, 2), (32, 48, 16, 1),
    (64, 16, 96, 3), (96, 64, 16, 4), (16, 96, 64, 5),
    (128, 16, 16, 3), (16, 128, 32, 3), (16, 16, 128, 7),
    (192, 16, 16, 3), (16, 192, 16, 2), (16, 16, 192, 3),
    (256, 16, 16, 5), (16, 256, 16, 3), (16, 16, 256, 3),
    (384, 16, 16, 3), (16, 384, 16, 3), (16, 16, 384, 7),
    (512, 16, 16, 3), (16, 512, 16, 1), (16, 16, 512, 3),
]


@pytest.mark.parametrize("nx,ny,nz,N", SHAPES_3D)
def test_few_steps_random_state_3d(nx, ny, nz, N):
    rng = np.random.default_rng(nx * 7 + ny * 3 + nz + N)
    cfg = wl.Config("rand3d", 3, nx, ny, nz, N, 0.2, 0.002, 0.3, 3, (3, 0.01, 2.0), "random", "box", 0)
    mu_a = rng.uniform(0.01, 0.5, cfg.shape).astype(np.float32)
    mu_s = rng.uniform(2.0, 20.0, cfg.shape).astype(np.float32)
    g = rng.uniform(0.7, 0.95, cfg.shape).astype(np.float32)
    psi0 = wl.random_state(cfg, seed=N)
    ext = (5, 4, 3)
    src = dict(w=rng.standard_normal(cfg.C).astype(np.float32), S=rng.standard_normal(ext[::-1]).astype(np.float32),
               origin=(1, 2, 4), extent=ext, kind=1, t0=0.0, sigma_t=1.0)
    got, ref, _ = run_both(cfg, mu_a, mu_s, g, psi0, src, cfg.steps)
    assert_parity(got, ref, f"{nx}x{ny}x{nz} P{N}")


SHAPES_2D = [(16, 32, 3), (48, 96, 2), (64, 64, 3), (128, 192, 7), (256, 16, 4), (384, 32, 3), (512, 64, 7), (32, 512, 1)]


@pytest.mark.parametrize("nx,ny,N", SHAPES_2D)
def test_few_steps_random_state_2d(nx, ny, N):
    rng = np.random.default_rng(nx + ny + N)
    cfg = wl.Config("rand2d", 2, nx, ny, 1, N, 0.1, 0.001, 0.3, 4, (4, 0.01, 5.0), "random", "box", 0)
    mu_a = rng.uniform(0.01, 0.5, cfg.shape).astype(np.float32)
    mu_s = rng.uniform(2.0, 20.0, cfg.shape).astype(np.float32)
    g = rng.uniform(0.7, 0.95, cfg.shape).astype(np.float32)
    psi0 = wl.random_state(cfg, seed=N)
    ext = (6, 5, 1)
    src = dict(w=rng.standard_normal(cfg.C).astype(np.float32), S=rng.standard_normal(ext[::-1]).astype(np.float32),
               origin=(2, 3, 0), extent=ext, kind=2, t0=0.002, sigma_t=0.001)
    got, ref, _ = run_both(cfg, mu_a, mu_s, g, psi0, src, cfg.steps)
    assert_parity(got, ref, f"{nx}x{ny} P{N}")


def test_scalar_media_no_pml_no_source():
    cfg = wl.Config("scalar", 3, 32, 32, 32, 3, 0.1, 0.002, 0.3, 5, (0, 0.0, 0.0), "homogeneous", "none", 0)
    psi0 = wl.random_state(cfg, seed=3)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, 0.02, 8.0, 0.85, cfg.pml)
    rte.rte_set_state(ctx, dev(psi0))
    rte.rte_step(ctx, 5)
    got = gpu_state(ctx, cfg)
    o = make_oracle(cfg, 0.02, 8.0, 0.85)
    o.set_state(psi0)
    o.step(5)
    assert_parity(got, o.get_state(), "scalar media")


# ---------------------------------------------------------------------------------------------------------------------
# the five configs
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("media", ["maps", "scalars"])
def test_cfg0_full(media):
    """configs[0]: 2-D 64x64 P_3, homogeneous, periodic, Gaussian pulse, 200 steps — full size, full step count.
    'scalars' is bench.py's launch configuration (uniform-g instance of the specialised x-pass kernel)."""
    cfg = wl.CONFIGS["cfg0"]
    mu = media_of(cfg, media)
    got, ref, ctx = run_both(cfg, *mu, wl.initial_state(cfg), wl.source_term(cfg), cfg.steps)
    e, f = assert_parity(got, ref, "cfg0")
    # conservation-type sanity on the GPU result itself: total fluence decays as (1 - c dt mu_a)^n (P5/P3 combined)
    tot = got[0].sum() / wl.initial_state(cfg)[0].astype(np.float64).sum()
    assert abs(tot - (1 - cfg.c * cfg.dt * 0.01) ** cfg.steps) < 1e-5
    phi = torch.empty(cfg.shape, dtype=torch.float32, device=DEV)
    rte.rte_fluence(ctx, phi)
    rte.rte_sync(ctx)
    assert np.array_equal(phi.cpu().numpy(), got[0].astype(np.float32))


def test_cfg1_reduced_full_steps():
    """configs[1] structure (P_7, disks, PML, point pulse) on 128^2 with the full 1000 steps.  dx is enlarged so that
    the pulse (20 ps, ~6 mm ballistic) reaches inclusions (SURVEY.md §8(d) extra case (i))."""
    cfg = wl.reduced(wl.CONFIGS["cfg1"], 128, dx=0.4, dt=0.02)      # Euler bound for the weakest disk: 0.058 ps
    mu = wl.media_maps(cfg)
    got, ref, _ = run_both(cfg, *mu, wl.initial_state(cfg), None, 1000)
    assert_parity(got, ref, "cfg1@128")


def test_cfg1_full_size_40_steps():
    cfg = wl.CONFIGS["cfg1"]
    mu = wl.media_maps(cfg)
    got, ref, _ = run_both(cfg, *mu, wl.initial_state(cfg), None, 40)
    assert_parity(got, ref, "cfg1 full size")


@pytest.mark.parametrize("media", ["maps", "scalars"])
def test_cfg2_reduced_full_steps(media):
    """configs[2] structure (P_3, homogeneous, PML, temporal-Gaussian face source) on 32^3, all 2000 steps."""
    cfg = wl.reduced(wl.CONFIGS["cfg2"], 32, pml_width=6)
    mu = media_of(cfg, media)
    got, ref, _ = run_both(cfg, *mu, wl.initial_state(cfg), wl.source_term(cfg), 2000)
    assert_parity(got, ref, "cfg2@32")
    assert np.abs(ref[0]).max() > 0


@pytest.mark.parametrize("media", ["scalars", "maps"])
def test_cfg2_full_size_few_steps(media):
    """configs[2] at 128^3, 16-cell PML, temporal-Gaussian source: 4 whole oracle steps around the source peak from a
    random state.  'scalars' passes mu_a, mu_s, g as single values exactly as bench.py does for this homogeneous
    workload (bench.py device_media), i.e. the uniform-g instance pass_kernel<..., UG = true> of the x pass with its
    2-number diagonal table — bench.py's launch configuration; 'maps' runs the g-map instance."""
    cfg = wl.CONFIGS["cfg2"]
    cfg = wl.replace(cfg, extra=dict(cfg.extra, t0_ps=0.2))
    mu = media_of(cfg, media)
    got, ref, _ = run_both(cfg, *mu, wl.random_state(cfg, seed=2), wl.source_term(cfg), 4)
    assert_parity(got, ref, f"cfg2 full size ({media})")


@pytest.mark.parametrize("name,n,N,W,steps", [("cfg0", 64, 3, 8, 50), ("cfg1", 512, 7, 16, 12)])
def test_2d_uniform_g_instance_with_pml_and_source(name, n, N, W, steps):
    """The uniform-g instances of the 2-D specialised x-pass kernels (64^2 P_3 and 512^2 P_7 tiles) with a PML and a
    Gaussian-in-time box source, scalar media, from a random state (UG + PML + source had no oracle check)."""
    base = wl.CONFIGS[name]
    cfg = wl.replace(base, name=f"{name}-ug", media="homogeneous", pml=(W, 0.01, 4.0), steps=steps, n_inclusions=0)
    rng = np.random.default_rng(n + N)
    ext = (7, 5, 1)
    src = dict(w=rng.standard_normal(cfg.C).astype(np.float32), S=rng.standard_normal(ext[::-1]).astype(np.float32),
               origin=(W + 3, n - W - 9, 0), extent=ext, kind=2, t0=3.5 * cfg.dt, sigma_t=2.0 * cfg.dt)
    got, ref, _ = run_both(cfg, *media_of(cfg, "scalars"), wl.random_state(cfg, seed=N), src, steps)
    assert_parity(got, ref, f"{name} 2-D UG + PML + source")


def test_cfg3_reduced():
    """configs[3] structure (P_5, ellipsoids with heterogeneous g, PML, constant collimated source) on 64^3, 200 steps;
    dx/dt enlarged (forward Euler's limit scales like dx^2)."""
    cfg = wl.reduced(wl.CONFIGS["cfg3"], 64, pml_width=8, dx=0.16, dt=0.0015)     # Euler bound 0.0038 ps
    mu = wl.media_maps(cfg)
    # a weak random background on top of the source-driven field makes every inclusion and PML cell matter
    got, ref, _ = run_both(cfg, *mu, 1e-3 * wl.random_state(cfg, seed=3), wl.source_term(cfg), 200)
    assert_parity(got, ref, "cfg3@64")


def test_cfg4_reduced():
    """configs[4] structure (P_7, log-normal mu_s, PML, point pulse) on 96^3 (3*2^5: exercises the radix-3 path)."""
    cfg = wl.reduced(wl.CONFIGS["cfg4"], 96, pml_width=8)
    mu = wl.media_maps(cfg)
    got, ref, _ = run_both(cfg, *mu, wl.initial_state(cfg), None, 12)
    assert_parity(got, ref, "cfg4@96")


def structural_cells(cfg, mu, src, rng, n_surface=40):
    """Cells a heterogeneous-media / PML / source bug would show up in first: the 8 corners, the 6 face centres, cells of
    the outermost-but-one PML layer boundary (last PML cell next to Omega and first Omega cell) on every side at random
    transverse positions, source-box cells, and cells on inclusion surfaces (where a medium map changes along x, y or z)."""
    n = (cfg.nx, cfg.ny, cfg.nz)
    W = cfg.pml[0]
    cells = [(x, y, z) for x in (0, n[0] - 1) for y in (0, n[1] - 1) for z in (0, n[2] - 1)]
    for a in range(3):
        for v in (0, n[a] - 1):
            c = [n[0] // 2, n[1] // 2, n[2] // 2]
            c[a] = v
            cells.append(tuple(c))
    if W > 0:
        for a in range(3):
            for v in (W - 1, W, n[a] - 1 - W, n[a] - W):        # last PML cell | first Omega cell | last Omega | first PML
                for _ in range(3):
                    c = [int(rng.integers(W, n[k] - W)) for k in range(3)]
                    c[a] = v
                    cells.append(tuple(c))
    if src is not None:
        o, e = src["origin"], src["extent"]
        for _ in range(8):
            cells.append(tuple(int(o[k] + rng.integers(e[k])) for k in range(3)))
        cells.append((o[0] + e[0] // 2, o[1] + e[1] // 2, o[2]))
    for m in mu:                                               # inclusion / field surfaces
        if isinstance(m, np.ndarray) and m.ndim == 3:
            for axis in range(3):
                d = np.diff(m, axis=axis) != 0
                idx = np.argwhere(d)
                if len(idx) == 0 or len(idx) > 0.5 * m.size:  # homogeneous, or a smooth field (every cell differs)
                    continue
                pick = idx[rng.choice(len(idx), size=min(n_surface // 3, len(idx)), replace=False)]
                cells += [(int(x), int(y), int(z)) for z, y, x in pick]
    return cells


def sampled_full_size_check(cfg, mu, psi0, src, ncells, seed):
    """One step at full size in bench.py's launch configuration, checked on sampled cells the oracle computes one by
    one (orc_step_cell: direct circulant sum along the three pencils through the cell): ncells random cells plus the
    structural ones (corners, faces, PML/Omega interface, source box, inclusion surfaces)."""
    mu_a, mu_s, g = mu
    ctx = gpu_create(cfg, mu_a, mu_s, g)
    rte.rte_set_state(ctx, dev(psi0))
    o = make_oracle(cfg, mu_a, mu_s, g)
    if src is not None:
        rte.rte_set_source(ctx, src["w"], dev(src["S"]), src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
        o.set_source(src["w"], src["S"], src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
    rte.rte_step(ctx, 1)
    out = torch.empty((cfg.C,) + cfg.shape, dtype=torch.float32, device=DEV)
    rte.rte_get_state(ctx, out)
    rte.rte_sync(ctx)
    rng = np.random.default_rng(seed)
    cells = [(int(rng.integers(cfg.nx)), int(rng.integers(cfg.ny)), int(rng.integers(cfg.nz))) for _ in range(ncells)]
    cells += structural_cells(cfg, mu, src, rng)
    ix = torch.tensor(cells, dtype=torch.long, device=DEV)
    got_all = out[:, ix[:, 2], ix[:, 1], ix[:, 0]].cpu().numpy().astype(np.float64)        # [C, ncells]
    scale = np.sqrt(np.mean(psi0.astype(np.float64) ** 2, axis=(1, 2, 3)))
    worst = 0.0
    for j, (x, y, z) in enumerate(cells):
        ref = o.step_cell(psi0, x, y, z)
        worst = max(worst, np.max(np.abs(got_all[:, j] - ref) / np.maximum(np.abs(ref), scale)))
    assert len(cells) >= 200
    assert worst < 2e-5, f"{cfg.name}: sampled one-step error {worst:.3e} over {len(cells)} cells"


def test_cfg3_full_size_sampled():
    cfg = wl.CONFIGS["cfg3"]
    mu = wl.media_maps(cfg)
    sampled_full_size_check(cfg, mu, wl.random_state(cfg, seed=3), wl.source_term(cfg), 200, 3)


def test_cfg2_full_size_sampled_scalar_media():
    """cfg2 exactly as bench.py launches it (scalar media => UG instance, 16-cell PML, temporal source at its peak)."""
    cfg = wl.CONFIGS["cfg2"]
    cfg = wl.replace(cfg, extra=dict(cfg.extra, t0_ps=0.0))
    sampled_full_size_check(cfg, media_of(cfg, "scalars"), wl.random_state(cfg, seed=2), wl.source_term(cfg), 200, 2)


def host_ram_gb():
    try:
        for ln in open("/proc/meminfo"):
            if ln.startswith("MemAvailable"):
                return int(ln.split()[1]) / 1e6
    except OSError:
        pass
    return 0.0


def test_cfg4_full_size_sampled():
    cfg = wl.CONFIGS["cfg4"]
    if host_ram_gb() < 80:
        pytest.skip("needs ~60 GB of host RAM for the fp32 state and its download")
    mu_a = np.full(cfg.shape, 0.01, dtype=np.float32)
    g = np.full(cfg.shape, 0.9, dtype=np.float32)
    # media from the DEVICE generator, downloaded and fed to the oracle (decouples stepper parity from generator parity)
    mu_s_d = torch.empty(cfg.shape, dtype=torch.float32, device=DEV)
    scratch = torch.empty_like(mu_s_d)
    rte.rte_media_lognormal(cfg.grid, cfg.dx, cfg.seed, 10.0, cfg.extra["sigma_log"], cfg.extra["corr_len_mm"], mu_s_d, scratch)
    mu_s = mu_s_d.cpu().numpy()
    del scratch
    sampled_full_size_check(cfg, (mu_a, mu_s, g), wl.random_state(cfg, seed=4), None, 200, 4)


# ---------------------------------------------------------------------------------------------------------------------
# properties that hold at any size (full-size launch configuration, no oracle run needed beyond small matrices)
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4"])
def test_full_size_single_mode_matrix_power(name):
    """Homogeneous periodic medium at the config's full grid and order: psi(r,0) = Re(v e^{ik.r}) must evolve to
    Re((I + dt M(k))^n v e^{ik.r}) with M(k) = -c (i k.A + diag sigma_l) from the ORACLE's coupling tables (pin P4)."""
    base = wl.CONFIGS[name]
    cfg = wl.replace(base, pml=(0, 0.0, 0.0))
    if cfg.C * cfg.G * 4 * 5 > 0.8 * torch.cuda.get_device_properties(0).total_memory:
        pytest.skip("not enough device memory")
    mu_a, mu_s, g = cfg.background
    rng = np.random.default_rng(cfg.seed)
    j = np.array([3, -5, 2])
    n = np.array([cfg.nx, cfg.ny, cfg.nz])
    kvec = 2 * np.pi * j / (n * cfg.dx)
    L = orc.degrees(cfg.dim, cfg.N)
    A = [orc.coupling_real(cfg.dim, cfg.N, a)[0] for a in range(3)]
    M = -cfg.c * (1j * sum(kvec[a] * A[a] for a in range(3)) + np.diag(mu_a + mu_s * (1 - g ** L)))
    v = (rng.standard_normal(cfg.C) + 1j * rng.standard_normal(cfg.C)) * 0.5 ** L
    steps = 3
    vn = np.linalg.matrix_power(np.eye(cfg.C) + cfg.dt * M, steps) @ v
    # phase factor evaluated with torch in fp64 on the device (test plumbing, not the CUDA path under test)
    ax = [torch.arange(m, dtype=torch.float64, device=DEV) for m in (cfg.nz, cfg.ny, cfg.nx)]
    ph = (kvec[2] * cfg.dx * ax[0])[:, None, None] + (kvec[1] * cfg.dx * ax[1])[None, :, None] + (kvec[0] * cfg.dx * ax[2])[None, None, :]
    cs, sn = torch.cos(ph), torch.sin(ph)
    del ph
    psi0 = torch.empty((cfg.C,) + cfg.shape, dtype=torch.float32, device=DEV)
    for c in range(cfg.C):
        psi0[c] = (v[c].real * cs - v[c].imag * sn).to(torch.float32)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, mu_a, mu_s, g, cfg.pml)
    rte.rte_set_state(ctx, psi0)
    rte.rte_step(ctx, steps)
    rte.rte_get_state(ctx, psi0)
    rte.rte_sync(ctx)
    worst = 0.0
    for c in range(cfg.C):
        ex = vn[c].real * cs - vn[c].imag * sn
        err = (psi0[c].to(torch.float64) - ex).norm() / ex.norm()
        worst = max(worst, float(err))
    assert worst < 2e-5, f"{name}: single-mode error {worst:.3e}"


def test_uniform_decay_and_conservation_on_device():
    """P3 + P5 on the device at a multi-tile size: uniform field decays as (1 - c dt sigma_l)^n; sum of psi_0 conserved
    when mu_a = 0."""
    cfg = wl.Config("decay", 3, 64, 48, 32, 3, 0.1, 0.002, 0.3, 10, (0, 0, 0), "homogeneous", "none", 0)
    amp = 1.0 + np.arange(cfg.C)
    psi0 = np.broadcast_to(amp[:, None, None, None], (cfg.C,) + cfg.shape).astype(np.float32)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, 0.013, 9.0, 0.87)
    rte.rte_set_state(ctx, dev(psi0))
    rte.rte_step(ctx, 10)
    got = gpu_state(ctx, cfg)
    L = orc.degrees(3, 3)
    ex = amp * (1 - 0.3 * 0.002 * (0.013 + 9.0 * (1 - 0.87 ** L))) ** 10
    assert np.abs(got / ex[:, None, None, None] - 1).max() < 5e-6
    ctx2 = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, 0.0, 6.0, 0.9)
    r = wl.random_state(cfg, seed=9)
    rte.rte_set_state(ctx2, dev(r))
    rte.rte_step(ctx2, 10)
    got = gpu_state(ctx2, cfg)
    assert abs(got[0].sum() - r[0].astype(np.float64).sum()) < 2e-6 * np.abs(r[0]).sum()


# ---------------------------------------------------------------------------------------------------------------------
# boundary behaviour on the device
# ---------------------------------------------------------------------------------------------------------------------
def test_host_buffer_entry_points_and_state_roundtrip():
    cfg = wl.Config("host", 3, 32, 16, 48, 4, 0.1, 0.002, 0.3, 2, (2, 0.01, 1.0), "homogeneous", "none", 0)
    psi0 = wl.random_state(cfg, seed=5)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, 0.02, 8.0, 0.85, cfg.pml)
    h = torch.from_numpy(psi0).pin_memory()
    rte.rte_set_state_host(ctx, h)
    back = torch.empty_like(h)
    rte.rte_get_state_host(ctx, back)
    assert torch.equal(back, h)                       # layout transposes are exact
    S = torch.ones((1, 2, 3), dtype=torch.float32).pin_memory()
    rte.rte_set_source_host(ctx, [1.0] + [0.0] * (cfg.C - 1), S, (5, 6, 7), (3, 2, 1), 1)
    rte.rte_step(ctx, 2)
    phi_h = torch.empty(cfg.shape, dtype=torch.float32).pin_memory()
    rte.rte_fluence_host(ctx, phi_h)
    o = make_oracle(cfg, 0.02, 8.0, 0.85)
    o.set_state(psi0)
    o.set_source([1.0] + [0.0] * (cfg.C - 1), np.ones((1, 2, 3)), (5, 6, 7), (3, 2, 1), 1)
    o.step(2)
    ref = o.fluence()
    assert np.abs(phi_h.numpy() - ref).max() <= 1e-5 * np.abs(ref).max()
    assert rte.rte_launch_count(ctx) >= 2 * 3
    ms, nl = rte.rte_step_profile(ctx, 2)
    assert nl == [2, 2, 2] and all(m > 0 for m in ms)
    assert abs(rte.rte_time_ps(ctx) - 4 * cfg.dt) < 1e-9


@pytest.mark.parametrize("grid,N", [((128, 16, 16), 3), ((32, 32, 32), 4)])
def test_double_buffer_odd_steps_and_determinism(grid, N):
    """The state is double buffered (each pass reads psi^n and reduces into the buffer that becomes psi^{n+1}; the
    accumulating passes use fire-and-forget red.global.add — one reduction per address per pass).  (i) Reading the state
    and the fluence after an ODD number of steps, through device and host entry points, then stepping on, matches the
    oracle stepped straight through; (ii) two identical runs are bit-identical (no scheduling dependence)."""
    cfg = wl.Config("dbuf", 3, grid[0], grid[1], grid[2], N, 0.2, 0.002, 0.3, 5, (2, 0.01, 2.0), "homogeneous", "none", 0)
    rng = np.random.default_rng(11)
    mu_a = rng.uniform(0.01, 0.5, cfg.shape).astype(np.float32)
    mu_s = rng.uniform(2.0, 20.0, cfg.shape).astype(np.float32)
    g = rng.uniform(0.7, 0.95, cfg.shape).astype(np.float32)
    psi0 = wl.random_state(cfg, seed=7)
    outs = []
    for rep in range(2):
        ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, dev(mu_a), dev(mu_s), dev(g), cfg.pml)
        rte.rte_set_state(ctx, dev(psi0))
        rte.rte_step(ctx, 3)
        mid = gpu_state(ctx, cfg)
        h = torch.empty((cfg.C,) + cfg.shape, dtype=torch.float32).pin_memory()
        rte.rte_get_state_host(ctx, h)
        assert np.array_equal(h.numpy().astype(np.float64), mid)
        phi_h = torch.empty(cfg.shape, dtype=torch.float32).pin_memory()
        rte.rte_fluence_host(ctx, phi_h)
        assert np.array_equal(phi_h.numpy().astype(np.float64), mid[0])
        rte.rte_step(ctx, 2)
        outs.append((mid, gpu_state(ctx, cfg)))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    o = make_oracle(cfg, mu_a, mu_s, g)
    o.set_state(psi0)
    o.step(3)
    assert_parity(outs[0][0], o.get_state(), "double buffer, 3 steps")
    o.step(2)
    assert_parity(outs[0][1], o.get_state(), "double buffer, 5 steps")


def test_paper_experiment_2_first_steps():
    """the paper's second run (64^3, P_7, PML, constant offset Gaussian source,
    dt = 0.04 ps) at full size for its first 25 of 25 000 steps, against the oracle."""
    cfg = wl.replace(wl.PAPER_EXPERIMENTS["paper_exp2"], steps=25)
    got, ref, _ = run_both(cfg, *wl.media_maps(cfg), wl.initial_state(cfg), wl.source_term(cfg), cfg.steps)
    assert np.abs(ref[0]).max() > 0
    assert_parity(got, ref, "paper exp. 2")


def test_paper_experiment_1_full_size_two_steps():
    """the paper's first run at its REAL size (64^3, P_21 = 484 coefficients, P = 242
    pairs: the large-C generic kernels), 2 whole oracle steps from a random state on top of the Gaussian initial
    radiance."""
    cfg = wl.replace(wl.PAPER_EXPERIMENTS["paper_exp1"], steps=2)
    if host_ram_gb() < 24:
        pytest.skip("needs ~12 GB of host RAM for the fp64 oracle state and its streaming term")
    mu = wl.media_maps(cfg)
    psi0 = wl.initial_state(cfg) + 1e-3 * wl.random_state(cfg, seed=21, decay=0.8)
    got, ref, _ = run_both(cfg, *mu, psi0.astype(np.float32), None, cfg.steps)
    assert_parity(got, ref, "paper exp. 1 (64^3, P_21)")


def test_paper_experiment_1_structure_reduced():
    """the paper's first run (P_21 = 484 coefficients, sharp mu_s slab, Gaussian
    initial radiance, dt = 0.1 ps) on a 32^3 grid with the same dx for 6 steps (the oracle needs ~1 s per step here)."""
    base = wl.PAPER_EXPERIMENTS["paper_exp1"]
    cfg = wl.reduced(base, 32, steps=6)
    mu = wl.media_maps(cfg)
    assert mu[1].max() == 5.0 and mu[1].min() == 1.0
    got, ref, _ = run_both(cfg, *mu, wl.initial_state(cfg), None, cfg.steps)
    assert_parity(got, ref, "paper exp. 1 (32^3)")


@pytest.mark.parametrize("dim,n,N", [(3, 32, 3), (2, 64, 4), (3, 128, 3)])
def test_ssprk3_against_oracle(dim, n, N):
    """SURVEY 8(f2) (NOT the paper's integrator): rte_step_ssprk3 vs the oracle's SSP-RK3 on heterogeneous media with a
    PML and a Gaussian-in-time source (pins the stage times), at a time step 12x above the forward-Euler bound of this
    medium (dt = 0.5 dx/c; Euler would blow up) — generic kernels, 2-D, and the specialised 128-point x pass."""
    nz = (n if dim == 3 else 1) if n != 128 else 16
    ny = n if n != 128 else 16
    dx, c = 0.2, 0.3
    dt = 0.5 * dx / c
    cfg = wl.Config("rk3", dim, n, ny, nz, N, dx, dt, c, 12, (3, 0.01, 2.0), "random", "box", 0)
    rng = np.random.default_rng(n + N)
    mu_a = rng.uniform(0.01, 0.5, cfg.shape).astype(np.float32)
    mu_s = rng.uniform(0.5, 5.0, cfg.shape).astype(np.float32)
    g = rng.uniform(0.7, 0.95, cfg.shape).astype(np.float32)
    psi0 = wl.random_state(cfg, seed=N)
    ext = (5, 4, 3 if dim == 3 else 1)
    w = rng.standard_normal(cfg.C).astype(np.float32)
    S = rng.standard_normal(ext[::-1]).astype(np.float32)
    org = (4, 5, 6 if dim == 3 else 0)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, dev(mu_a), dev(mu_s), dev(g), cfg.pml)
    rte.rte_set_state(ctx, dev(psi0))
    rte.rte_set_source(ctx, w, dev(S), org, ext, 2, 3.5 * dt, 2.0 * dt)
    rte.rte_step_ssprk3(ctx, cfg.steps)
    got = gpu_state(ctx, cfg)
    assert abs(rte.rte_time_ps(ctx) - cfg.steps * dt) < 1e-6 * cfg.steps * dt     # dt is fp32 inside the library
    o = make_oracle(cfg, mu_a, mu_s, g)
    o.set_state(psi0)
    o.set_source(w, S, org, ext, 2, 3.5 * dt, 2.0 * dt)
    o.step_ssprk3(cfg.steps)
    assert_parity(got, o.get_state(), f"ssprk3 {dim}-D n={n}")
    # mixing integrators on one context keeps the buffers straight: two Euler steps after the RK steps
    rte.rte_step(ctx, 2)
    # (Euler at this dt is unstable, but two steps stay finite and must match the oracle exactly as well)
    o.step(2)
    assert_parity(gpu_state(ctx, cfg), o.get_state(), "euler after ssprk3")


def test_steady_state_by_ssprk3_is_a_fixed_point_of_the_paper_step():
    """configs[3]'s steady state, reached with the non-paper SSP-RK3 step at dt = 0.3 dx/c and the R17 stopping rule, must
    be a fixed point of the PAPER's forward-Euler map: one oracle Euler step (small stable dt) of the converged GPU state
    changes it by no more than the residual the stopping rule allows."""
    n, N, dx, c = 32, 3, 0.2, 0.3
    dt_rk = 0.3 * dx / c
    cfg = wl.Config("ss3d", 3, n, n, n, N, dx, dt_rk, c, 0, (4, 0.05, 3.0), "homogeneous", "none", 0)
    mu_a, mu_s, g = 0.05, 4.0, 0.8
    w = wl.collimated_weights(cfg)
    S = np.zeros((1, 5, 5), dtype=np.float32)
    S[0, 2, 2] = 1.0 / dx ** 3
    S[0, 1:4, 1:4] += 0.2 / dx ** 3
    org, ext = (14, 14, 5), (5, 5, 1)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, mu_a, mu_s, g, cfg.pml)
    rte.rte_set_source(ctx, w, dev(S), org, ext, 1)
    rte.rte_fluence_change(ctx)
    steps, change = 0, float("inf")
    while steps < 6000 and not change < 1e-6:
        rte.rte_step_ssprk3(ctx, 100)
        steps += 100
        change = rte.rte_fluence_change(ctx)
    assert change < 1e-6, f"no steady state after {steps} steps (change {change:.2e})"
    star = gpu_state(ctx, cfg)
    assert np.isfinite(star).all() and np.abs(star[0]).max() > 0
    dt_e = 0.002                                            # stable forward-Euler step of this medium
    o = orc.Oracle(3, n, n, n, N, dx, dt_e, c, np.full(cfg.shape, mu_a), np.full(cfg.shape, mu_s), np.full(cfg.shape, g),
                   *cfg.pml)
    o.set_source(w, S, org, ext, 1)
    o.set_state(star)
    o.step(1)
    after = o.get_state()
    # d psi/dt at the converged state, relative to the state, per unit time: the RK run's own rate was
    # change / (100 dt_rk) ~ 5e-8 / ps for the fluence; allow a generous multiple (fp32 state, all coefficients)
    rate = np.linalg.norm(after[0] - star[0]) / np.linalg.norm(star[0]) / dt_e
    assert rate < 1e-5, f"converged state is not a fixed point of the Euler map: relative rate {rate:.2e} per ps"


def test_fluence_change_steady_state_rule():
    """configs[3]'s stopping rule (R17): relative L2 change of the fluence over Omega between calls, against the same
    quantity computed from the oracle's fluence (dt = 0.02 ps is below the Euler bound of this medium, ~0.044 ps)."""
    cfg = wl.Config("ss", 2, 64, 64, 1, 3, 0.2, 0.02, 0.3, 0, (8, 0.01, 2.0), "homogeneous", "none", 0)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, 0.5, 5.0, 0.5, cfg.pml)
    S = torch.ones((1, 3, 3), dtype=torch.float32, device=DEV)
    w = [1.0] + [0.0] * (cfg.C - 1)
    rte.rte_set_source(ctx, w, S, (30, 30, 0), (3, 3, 1), 1)
    o = make_oracle(cfg, 0.5, 5.0, 0.5)
    o.set_source(w, np.ones((1, 3, 3)), (30, 30, 0), (3, 3, 1), 1)
    _, inside = orc.pml_map(2, 64, 64, 1, 8, 0.01, 2.0)
    m = inside == 1
    assert math.isinf(rte.rte_fluence_change(ctx))
    prev, oprev = None, o.fluence()
    for _ in range(16):
        rte.rte_step(ctx, 200)
        ch = rte.rte_fluence_change(ctx)
        o.step(200)
        of = o.fluence()
        och = np.linalg.norm((of - oprev)[m]) / np.linalg.norm(of[m])
        oprev = of
        assert np.isfinite(ch)
        assert abs(ch - och) <= 0.02 * och + 1e-6, (ch, och)
        if prev is not None:
            assert ch < prev
        prev = ch
    assert prev < 1e-4      # approaching a steady state


def test_argument_validation_on_device():
    with pytest.raises(rte.RteError) as e:
        rte.rte_create((3, 32, 32, 32), 3, 0.1, 0.001, 0.3, 0.01, 10.0, 0.9, (16, 0.01, 1.0))   # PML wider than half
    assert e.value.code == rte.RTE_EINVAL
    with pytest.raises(rte.RteError):
        rte.rte_create((3, 32, 32, 32), 3, -0.1, 0.001, 0.3, 0.01, 10.0, 0.9)
    ctx = rte.rte_create((3, 32, 32, 32), 3, 0.1, 0.001, 0.3, 0.01, 10.0, 0.9)
    with pytest.raises(rte.RteError):
        rte.rte_set_source(ctx, [1.0] * 16, torch.ones(8, device=DEV), (30, 0, 0), (4, 2, 1), 1)   # box leaves the grid
    with pytest.raises(rte.RteError):
        rte.rte_step(ctx, -1)
    rte.rte_step(ctx, 0)
    rte.rte_sync(ctx)


# ---------------------------------------------------------------------------------------------------------------------
# geometry layer vs the CPU generators
# ---------------------------------------------------------------------------------------------------------------------
def test_device_geometry_generators():
    cfg = wl.reduced(wl.CONFIGS["cfg3"], 64, dx=0.16)
    rows = wl.inclusion_list(cfg)
    a, s, g = (torch.empty(cfg.shape, dtype=torch.float32, device=DEV) for _ in range(3))
    rte.rte_media_ellipsoids(cfg.grid, cfg.dx, cfg.background, rows, a, s, g)
    ra, rs, rg = wl.rasterize_inclusions(cfg, rows)
    torch.cuda.synchronize()
    for got, ref in ((a, ra), (s, rs), (g, rg)):
        mism = (got.cpu().numpy() != ref).mean()
        assert mism < 1e-4          # only cells exactly on an ellipsoid surface may differ by rounding
    c2 = wl.reduced(wl.CONFIGS["cfg1"], 128, dx=0.2)
    rows2 = wl.inclusion_list(c2)
    a2 = torch.empty(c2.shape, dtype=torch.float32, device=DEV)
    rte.rte_media_ellipsoids(c2.grid, c2.dx, c2.background, rows2, a2, None, None)
    assert (a2.cpu().numpy() != wl.rasterize_inclusions(c2, rows2)[0]).mean() < 1e-3
    # PML profile vs the oracle's map (fp32 vs fp64)
    mb = torch.empty(cfg.shape, dtype=torch.float32, device=DEV)
    ins = torch.empty(cfg.shape, dtype=torch.uint8, device=DEV)
    rte.rte_pml_profile(cfg.grid, (8, 0.01, 8.0), mb, ins)
    ob, oi = orc.pml_map(3, 64, 64, 64, 8, 0.01, 8.0)
    assert np.array_equal(ins.cpu().numpy(), oi)
    assert np.abs(mb.cpu().numpy() - ob).max() < 1e-5 * 8.0
    # log-normal field vs the CPU generator (transcendental functions differ in the last ulp)
    c4 = wl.reduced(wl.CONFIGS["cfg4"], 48)
    out = torch.empty(c4.shape, dtype=torch.float32, device=DEV)
    scr = torch.empty_like(out)
    rte.rte_media_lognormal(c4.grid, c4.dx, c4.seed, 10.0, 0.3, 2.0, out, scr)
    ref = wl.lognormal_field(c4)
    assert np.abs(out.cpu().numpy() / ref - 1).max() < 1e-4
