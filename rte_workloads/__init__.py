"""rte_workloads — the five BASELINE.json configs and the seeded synthetic-input generators (numpy, CPU).

This module serves BOTH the oracle-side tests and the CUDA-side harness, so it holds none of the method's arithmetic
(no derivative, coupling, scattering diagonal, PML profile or time step): only workload parameters, geometry
rasterisation of inclusion lists, initial radiance / source footprints, and the counter-based random numbers of the
log-normal field recipe.  Recipes follow SURVEY.md §8(d) / DESIGN.md "Synthetic inputs"; the workloads are shaped like
the paper's diffuse-regime runs (mu_s ~ 10 mm^-1, mu_a ~ 0.01 mm^-1, g ~ 0.9) and stand in
for them — the paper publishes no dataset.
"""
from dataclasses import dataclass, field, replace  # noqa: F401 (replace is re-exported)
import math

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    dim: int
    nx: int
    ny: int
    nz: int
    N: int
    dx: float            # mm
    dt: float            # ps   (R10)
    c: float             # mm/ps
    steps: int
    pml: tuple           # (width, mu_lo, mu_hi)
    media: str           # 'homogeneous' | 'disks' | 'ellipsoids' | 'lognormal'
    source: str          # 'gaussian_pulse_ic' | 'point_pulse_ic' | 'gaussian_face_temporal' | 'collimated_constant'
    seed: int
    background: tuple = (0.01, 10.0, 0.9)   # mu_a, mu_s, g
    n_inclusions: int = 0
    extra: dict = field(default_factory=dict)

    @property
    def grid(self):
        return (self.dim, self.nx, self.ny, self.nz)

    @property
    def C(self):
        return (self.N + 1) ** 2 if self.dim == 3 else 2 * self.N + 1

    @property
    def G(self):
        return self.nx * self.ny * self.nz

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)


CONFIGS = {
    "cfg0": Config("cfg0", 2, 64, 64, 1, 3, 0.1, 0.002, 0.3, 200, (0, 0.0, 0.0), "homogeneous", "gaussian_pulse_ic",
                   1801, extra={"sigma_mm": 0.3}),
    "cfg1": Config("cfg1", 2, 512, 512, 1, 7, 0.05, 0.0004, 0.3, 1000, (16, 0.01, 10.0), "disks", "point_pulse_ic",
                   6364, n_inclusions=20),
    "cfg2": Config("cfg2", 3, 128, 128, 128, 3, 0.8, 0.1, 0.3, 2000, (16, 0.01, 1.0), "homogeneous",
                   "gaussian_face_temporal", 2018, extra={"sigma_mm": 1.0, "fwhm_ps": 10.0, "t0_ps": 15.0}),
    "cfg3": Config("cfg3", 3, 256, 256, 256, 5, 0.04, 0.0001, 0.3, 200, (24, 0.01, 8.0), "ellipsoids",
                   "collimated_constant", 3, n_inclusions=50, extra={"sigma_mm": 0.5}),
    "cfg4": Config("cfg4", 3, 384, 384, 384, 7, 0.25, 0.005, 0.3, 500, (32, 0.01, 1.0), "lognormal", "point_pulse_ic",
                   5, extra={"sigma_log": 0.3, "corr_len_mm": 2.0}),
}


# The paper's own two runs, as workloads: like-for-like wall-clock beside
# the Tesla-K40 timings the paper prints (70 s / 223 s).  No expected output exists (Figures 1-4 carry no numbers).
#   exp1: 50 mm cube, 64^3, P_21, mu_a 0.01, mu_s 1.0 (5.0 for x <= 15 mm), g 0.9, dt 0.1 ps, 400 steps, no PML,
#         isotropic Gaussian initial radiance of 1/e diameter 1.5 mm (sigma = D / (2 sqrt 2)) at the centre.
#   exp2: 35.5 mm real cube inside the 50 mm / 64^3 domain (PML of 9 cells, half-cosine 0.01 -> 1.0 mm^-1), P_7,
#         mu_a 0.01, mu_s 10, g 0.95, dt 0.04 ps, 25 000 steps, constant isotropic Gaussian source (same width) offset
#         8 mm in x from the centre.
PAPER_EXPERIMENTS = {
    "paper_exp1": Config("paper_exp1", 3, 64, 64, 64, 21, 50.0 / 64, 0.1, 0.3, 400, (0, 0.0, 0.0), "slab",
                         "gaussian_pulse_ic", 0, background=(0.01, 1.0, 0.9),
                         extra={"sigma_mm": 1.5 / (2.0 * math.sqrt(2.0)), "slab_mu_s": 5.0, "slab_x_mm": 15.0}),
    "paper_exp2": Config("paper_exp2", 3, 64, 64, 64, 7, 50.0 / 64, 0.04, 0.3, 25000, (9, 0.01, 1.0), "homogeneous",
                         "gaussian_constant_offset", 0, background=(0.01, 10.0, 0.95),
                         extra={"sigma_mm": 1.5 / (2.0 * math.sqrt(2.0)), "offset_x_mm": 8.0}),
}


def reduced(cfg: Config, n: int, steps=None, pml_width=None, dt=None, dx=None) -> Config:
    """Same structure on an n^d grid (for parity runs the fp64 oracle can finish)."""
    W = cfg.pml[0] if pml_width is None else pml_width
    W = min(W, max(0, n // 2 - 2)) if cfg.pml[0] > 0 else 0
    return replace(cfg, name=f"{cfg.name}@{n}", nx=n, ny=n, nz=(n if cfg.dim == 3 else 1),
                   steps=cfg.steps if steps is None else steps, pml=(W, cfg.pml[1], cfg.pml[2]),
                   dt=cfg.dt if dt is None else dt, dx=cfg.dx if dx is None else dx)


# ---------------------------------------------------------------------------------------------------------------------
# geometry
# ---------------------------------------------------------------------------------------------------------------------
def cell_coords(cfg: Config):
    """Cell i along an axis sits at (i - n/2) dx."""
    x = (np.arange(cfg.nx) - cfg.nx // 2) * cfg.dx
    y = (np.arange(cfg.ny) - cfg.ny // 2) * cfg.dx
    z = (np.arange(cfg.nz) - cfg.nz // 2) * cfg.dx
    return x, y, z


def inclusion_list(cfg: Config):
    """Rows {cx,cy,cz,ax,ay,az,mu_a,mu_s,g}; centres ~U(Omega), later rows overwrite earlier ones."""
    rng = np.random.default_rng(cfg.seed)
    W = cfg.pml[0]
    rows = []
    ext = [cfg.nx, cfg.ny, cfg.nz]
    for _ in range(cfg.n_inclusions):
        ctr = []
        for a in range(3):
            if a >= cfg.dim:
                ctr.append(0.0)
                rng.uniform()   # keep the stream independent of dim
                continue
            lo = (W - ext[a] // 2) * cfg.dx
            hi = (ext[a] - 1 - W - ext[a] // 2) * cfg.dx
            ctr.append(rng.uniform(lo, hi))
        if cfg.media == "disks":
            r = rng.uniform(0.5, 3.0) * cfg.extra.get("radius_scale", 1.0)
            ax = [r, r, 1.0]
            mu_a, mu_s, g = rng.uniform(0.005, 0.1), rng.uniform(5.0, 20.0), cfg.background[2]
        else:
            sc = cfg.extra.get("radius_scale", 1.0)
            ax = [rng.uniform(0.2, 1.5) * sc for _ in range(3)]
            mu_a, mu_s, g = rng.uniform(0.01, 1.0), rng.uniform(5.0, 20.0), rng.uniform(0.8, 0.95)
        rows.append([*ctr, *ax, mu_a, mu_s, g])
    return np.asarray(rows, dtype=np.float32).reshape(-1, 9)


def rasterize_inclusions(cfg: Config, rows):
    """CPU counterpart of rte_media_ellipsoids (fp32 arithmetic in the same order)."""
    x, y, z = [v.astype(np.float32) for v in cell_coords(cfg)]
    mu_a = np.full(cfg.shape, cfg.background[0], dtype=np.float32)
    mu_s = np.full(cfg.shape, cfg.background[1], dtype=np.float32)
    g = np.full(cfg.shape, cfg.background[2], dtype=np.float32)
    X = x[None, None, :]
    Y = y[None, :, None]
    Z = z[:, None, None]
    for r in np.asarray(rows, dtype=np.float32):
        ux = (X - r[0]) / r[3]
        uy = (Y - r[1]) / r[4]
        d = ux * ux + uy * uy
        if cfg.dim == 3:
            uz = (Z - r[2]) / r[5]
            d = d + uz * uz
        m = np.broadcast_to(d <= np.float32(1.0), cfg.shape)
        mu_a[m], mu_s[m], g[m] = r[6], r[7], r[8]
    return mu_a, mu_s, g


_M64 = (1 << 64) - 1


def splitmix64(x):
    """splitmix64 finaliser on uint64 arrays (the counter-based generator of the log-normal recipe)."""
    x = (x + np.uint64(0x9E3779B97F4A7C15)) & np.uint64(_M64)
    x = ((x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & np.uint64(_M64)
    x = ((x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & np.uint64(_M64)
    return x ^ (x >> np.uint64(31))


def white_noise(G, seed):
    """Normal deviates: h = splitmix64(seed*0x100000001B3 + i); u1 = (top 24 bits + 1)/2^24, u2 = next 24 bits/2^24;
    z = sqrt(-2 ln u1) cos(2 pi u2)."""
    with np.errstate(over="ignore"):
        i = np.arange(G, dtype=np.uint64)
        h = splitmix64(np.uint64((seed * 0x100000001B3) & _M64) + i)
    a = (h >> np.uint64(40)).astype(np.float64)
    b = ((h >> np.uint64(16)) & np.uint64(0xFFFFFF)).astype(np.float64)
    u1 = (a + 1.0) / 16777216.0
    u2 = b / 16777216.0
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def lognormal_field(cfg: Config, mean=None):
    """CPU counterpart of rte_media_lognormal: white noise -> separable circular Gaussian blur (std corr_len/sqrt2 per
    axis, truncated at R = ceil(4 std) cells, weights normalised) -> zero mean, unit sample variance ->
    exp(ln mean - s^2/2 + s f)."""
    mean = cfg.background[1] if mean is None else mean
    s_log, lc = cfg.extra["sigma_log"], cfg.extra["corr_len_mm"]
    f = white_noise(cfg.G, cfg.seed).reshape(cfg.shape)
    s_cells = np.float32(lc) / np.float32(1.41421356237) / np.float32(cfg.dx)
    R = int(math.ceil(4.0 * float(s_cells)))
    j = np.arange(-R, R + 1)
    w = np.exp(-(j * j) / (2.0 * float(s_cells) ** 2))
    w /= w.sum()
    for axis_np in ([2, 1, 0] if cfg.dim == 3 else [2, 1]):      # x, y, (z)
        acc = np.zeros_like(f)
        for jj, ww in zip(j, w):
            acc += ww * np.roll(f, -jj, axis=axis_np)
        f = acc
    f = (f - f.mean()) / f.std()
    return np.exp(math.log(mean) - 0.5 * s_log ** 2 + s_log * f).astype(np.float32)


def media_maps(cfg: Config):
    """(mu_a, mu_s, g) as fp32 maps [nz,ny,nx] (CPU generators)."""
    if cfg.media == "homogeneous":
        return tuple(np.full(cfg.shape, v, dtype=np.float32) for v in cfg.background)
    if cfg.media in ("disks", "ellipsoids"):
        return rasterize_inclusions(cfg, inclusion_list(cfg))
    if cfg.media == "slab":       # the paper's sharp mu_s step: cells whose x, measured from the domain edge, is <= slab_x
        mu_a, mu_s, g = (np.full(cfg.shape, v, dtype=np.float32) for v in cfg.background)
        x_from_edge = np.arange(cfg.nx) * cfg.dx
        mu_s[:, :, x_from_edge <= cfg.extra["slab_x_mm"]] = cfg.extra["slab_mu_s"]
        return mu_a, mu_s, g
    if cfg.media == "lognormal":
        mu_a = np.full(cfg.shape, cfg.background[0], dtype=np.float32)
        g = np.full(cfg.shape, cfg.background[2], dtype=np.float32)
        return mu_a, lognormal_field(cfg), g
    raise ValueError(cfg.media)


# ---------------------------------------------------------------------------------------------------------------------
# initial radiance and sources (R13)
# ---------------------------------------------------------------------------------------------------------------------
def gaussian_footprint(cfg: Config, centre_cell, sigma_mm, ndim=None, radius_sigmas=5.0):
    """Unit-integral Gaussian S(r) = exp(-|r-r0|^2/(2 sigma^2)), normalised so that sum S dx^d = 1, on a box of
    +-radius_sigmas sigma cells clipped to the grid.  Returns (S[bz,by,bx] fp32, origin, extent)."""
    ndim = cfg.dim if ndim is None else ndim
    R = int(math.ceil(radius_sigmas * sigma_mm / cfg.dx))
    ext_n = [cfg.nx, cfg.ny, cfg.nz]
    lo, hi = [], []
    for a in range(3):
        if a < ndim:
            lo.append(max(0, centre_cell[a] - R))
            hi.append(min(ext_n[a] - 1, centre_cell[a] + R))
        else:
            lo.append(centre_cell[a])
            hi.append(centre_cell[a])
    ax = [np.arange(lo[a], hi[a] + 1) - centre_cell[a] for a in range(3)]
    r2 = (ax[0][None, None, :] ** 2 + ax[1][None, :, None] ** 2 + ax[2][:, None, None] ** 2) * cfg.dx ** 2
    S = np.exp(-r2 / (2.0 * sigma_mm ** 2))
    S /= S.sum() * cfg.dx ** ndim
    return S.astype(np.float32), tuple(lo), tuple(hi[a] - lo[a] + 1 for a in range(3))


def collimated_weights(cfg: Config, direction=(0.0, 0.0, 1.0)):
    """Angular weights of a delta(s - s0) source in the expansion of PAPER.md eq.(4): w_c = sqrt(4 pi/(2l+1)) Y^R_c(s0).
    Only s0 = +z (3-D: w_{l0} = 1, others 0) and s0 at angle theta0 in 2-D (a_m = cos m theta0, b_m = sin m theta0) are
    needed by the configs."""
    w = np.zeros(cfg.C, dtype=np.float32)
    if cfg.dim == 3:
        if tuple(direction) != (0.0, 0.0, 1.0):
            raise NotImplementedError("only +z collimation is used by the configs")
        for l in range(cfg.N + 1):
            w[l * l + l] = 1.0
    else:
        th = math.atan2(direction[1], direction[0])
        w[0] = 1.0
        for m in range(1, cfg.N + 1):
            w[2 * m - 1] = math.cos(m * th)
            w[2 * m] = math.sin(m * th)
    return w


def isotropic_weights(cfg: Config):
    w = np.zeros(cfg.C, dtype=np.float32)
    w[0] = 1.0
    return w


def initial_state(cfg: Config):
    """psi(0) [C,nz,ny,nx] fp32: the delta(t) pulses of cfg0/1/4 enter as an initial radiance."""
    psi = np.zeros((cfg.C,) + cfg.shape, dtype=np.float32)
    cz = cfg.nz // 2 if cfg.dim == 3 else 0
    centre = (cfg.nx // 2, cfg.ny // 2, cz)
    if cfg.source == "gaussian_pulse_ic":
        S, org, ext = gaussian_footprint(cfg, centre, cfg.extra["sigma_mm"])
        psi[0, org[2]:org[2] + ext[2], org[1]:org[1] + ext[1], org[0]:org[0] + ext[0]] = S
    elif cfg.source == "point_pulse_ic":
        psi[0, centre[2], centre[1], centre[0]] = 1.0 / cfg.dx ** cfg.dim
    return psi


def source_term(cfg: Config):
    """None, or dict(w, S, origin, extent, kind, t0, sigma_t) for rte_set_source / Oracle.set_source."""
    W = cfg.pml[0]
    if cfg.source == "gaussian_face_temporal":
        # isotropic, spatial Gaussian centred one cell inside Omega on the -z face, temporal Gaussian (FWHM given)
        centre = (cfg.nx // 2, cfg.ny // 2, W + 1)
        S, org, ext = gaussian_footprint(cfg, centre, cfg.extra["sigma_mm"])
        sig_t = cfg.extra["fwhm_ps"] / (2.0 * math.sqrt(2.0 * math.log(2.0)))
        return dict(w=isotropic_weights(cfg), S=S, origin=org, extent=ext, kind=2, t0=cfg.extra["t0_ps"], sigma_t=sig_t)
    if cfg.source == "gaussian_constant_offset":
        # constant isotropic Gaussian source, offset along +x from the centre
        centre = (cfg.nx // 2 + int(round(cfg.extra["offset_x_mm"] / cfg.dx)), cfg.ny // 2, cfg.nz // 2)
        S, org, ext = gaussian_footprint(cfg, centre, cfg.extra["sigma_mm"])
        return dict(w=isotropic_weights(cfg), S=S, origin=org, extent=ext, kind=1, t0=0.0, sigma_t=1.0)
    if cfg.source == "collimated_constant":
        # +z collimated Gaussian disc on the first Omega layer at the -z face
        centre = (cfg.nx // 2, cfg.ny // 2, W)
        S, org, ext = gaussian_footprint(cfg, centre, cfg.extra["sigma_mm"], ndim=2)
        S = S / cfg.dx      # a disc of one cell thickness: sum S dx^3 = 1
        return dict(w=collimated_weights(cfg), S=S.astype(np.float32), origin=org, extent=ext, kind=1, t0=0.0, sigma_t=1.0)
    return None


def random_state(cfg: Config, seed=0, decay=0.5):
    """Seeded random fp32 state with amplitudes decaying in the degree (stress input for one-step parity)."""
    rng = np.random.default_rng(seed)
    psi = rng.standard_normal((cfg.C,) + cfg.shape).astype(np.float32)
    if cfg.dim == 3:
        L = np.array([l for l in range(cfg.N + 1) for _ in range(2 * l + 1)])
    else:
        L = np.array([0] + [m for m in range(1, cfg.N + 1) for _ in range(2)])
    return psi * (decay ** L)[:, None, None, None].astype(np.float32)
