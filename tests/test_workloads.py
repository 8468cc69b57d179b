"""Host tests of the seeded input generators and of the time-step choices (R10, R13)."""
import math

import numpy as np
import pytest

import rte_workloads as wl
from oracle import rte_oracle as orc


def test_config_table_matches_baseline():
    c = wl.CONFIGS
    assert (c["cfg0"].C, c["cfg1"].C, c["cfg2"].C, c["cfg3"].C, c["cfg4"].C) == (7, 15, 16, 36, 64)
    assert c["cfg4"].C * c["cfg4"].G * 4 == 384 ** 3 * 64 * 4          # "~14.5 GB per fp32 state"
    assert c["cfg2"].pml[0] == 16 and c["cfg3"].pml[0] == 24 and c["cfg4"].pml[0] == 32


def stable_dt_bound(cfg, mu_a, mu_s, g):
    """Forward-Euler bound dt <= -2 Re(lambda)/|lambda|^2 over the eigenvalues of M(k) = -c (i k A_axis + diag sigma),
    k along one axis up to the corner Nyquist magnitude sqrt(d) pi/dx (R10).  Uses only the oracle's tables."""
    A, _ = orc.coupling_real(cfg.dim, cfg.N, 2 if cfg.dim == 3 else 0)
    L = orc.degrees(cfg.dim, cfg.N)
    sigma = mu_a + mu_s * (1 - g ** L)
    n = cfg.nx
    kmax = math.sqrt(cfg.dim) * math.pi / cfg.dx * (1 - 2.0 / n)
    best = np.inf
    for k in np.linspace(kmax / 200, kmax, 200):
        lam = np.linalg.eigvals(-cfg.c * (1j * k * A + np.diag(sigma)))
        best = min(best, np.min(-2 * lam.real / np.abs(lam) ** 2))
    return best


@pytest.mark.parametrize("name,weak", [("cfg0", (0.01, 10.0, 0.9)), ("cfg1", (0.005, 5.0, 0.9)), ("cfg2", (0.01, 10.0, 0.9)),
                                       ("cfg3", (0.01, 5.0, 0.95)), ("cfg4", (0.01, 3.0, 0.9))])
def test_config_time_steps_are_stable(name, weak):
    """dt of every config is below half the bound for the weakest-damping medium present (R10)."""
    cfg = wl.CONFIGS[name]
    bound = stable_dt_bound(cfg, *weak)
    assert cfg.dt <= 0.55 * bound, (cfg.dt, bound)


def test_inclusions_are_seeded_and_inside_omega():
    cfg = wl.CONFIGS["cfg1"]
    rows = wl.inclusion_list(cfg)
    assert rows.shape == (20, 9) and np.array_equal(rows, wl.inclusion_list(cfg))
    half = (cfg.nx // 2 - cfg.pml[0]) * cfg.dx
    assert (np.abs(rows[:, 0]) <= half).all() and (np.abs(rows[:, 1]) <= half).all()
    assert (rows[:, 3] >= 0.5).all() and (rows[:, 3] <= 3.0).all() and (rows[:, 8] == np.float32(0.9)).all()
    small = wl.reduced(cfg, 64)
    mu_a, mu_s, g = wl.media_maps(small)
    assert mu_a.shape == (1, 64, 64) and mu_a.dtype == np.float32
    assert len(np.unique(mu_s)) > 1


def test_gaussian_footprint_normalisation_and_point_source():
    cfg = wl.CONFIGS["cfg0"]
    psi = wl.initial_state(cfg)
    assert abs(psi[0].sum() * cfg.dx ** 2 - 1.0) < 1e-5 and np.abs(psi[1:]).max() == 0
    assert psi[0, 0, 32, 32] == psi[0].max()
    c4 = wl.reduced(wl.CONFIGS["cfg4"], 16)
    p4 = wl.initial_state(c4)
    assert p4[0, 8, 8, 8] == np.float32(1 / c4.dx ** 3) and np.count_nonzero(p4) == 1
    s2 = wl.source_term(wl.CONFIGS["cfg2"])
    assert s2["kind"] == 2 and abs(s2["sigma_t"] - 4.2466) < 1e-3 and abs(s2["S"].sum() * 0.8 ** 3 - 1) < 1e-4
    s3 = wl.source_term(wl.reduced(wl.CONFIGS["cfg3"], 64))
    assert s3["kind"] == 1 and s3["extent"][2] == 1 and s3["w"][0] == 1 and s3["w"][2] == 1 and s3["w"][1] == 0


def test_white_noise_moments_and_lognormal_field():
    z = wl.white_noise(1 << 16, 5)
    assert abs(z.mean()) < 0.02 and abs(z.std() - 1) < 0.02
    assert np.array_equal(z, wl.white_noise(1 << 16, 5)) and not np.array_equal(z, wl.white_noise(1 << 16, 6))
    cfg = wl.reduced(wl.CONFIGS["cfg4"], 64)
    f = wl.lognormal_field(cfg)
    lf = np.log(f.astype(np.float64))
    assert abs(lf.std() - 0.3) < 1e-3
    assert abs(lf.mean() - (math.log(10.0) - 0.045)) < 1e-3
    # correlation at lag of one correlation length ~ exp(-1/2) (periodic domain, truncated kernel): loose check
    lag = int(round(cfg.extra["corr_len_mm"] / cfg.dx))
    g0 = (lf - lf.mean())
    rho = (g0 * np.roll(g0, lag, axis=2)).mean() / g0.var()
    assert 0.45 < rho < 0.75        # exp(-1/2) = 0.607 up to sampling noise on a 64^3 periodic box
