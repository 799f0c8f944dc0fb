"""Equilibrium of the Brownian-dynamics step above a wall (initial heights are "sampled from the equilibrium
Gibbs-Boltzmann distribution P(z) ~ exp(-m g z / k_B T)"; eq. (14) PAPER.md:224-228 with the thermal-drift term;
PAPER.md:87: the drift is what makes eq. (9) consistent with that distribution).

Particles above a no-slip wall under gravity and the soft wall repulsion of eq. (13) have the stationary height
distribution P(h) ~ exp(-(m g h + U_wall(h)) / k_B T) WHATEVER the mobility -- provided the noise is M^{1/2} W
(fluctuation-dissipation) and the drift k_B T d/dX . M is there.  The test starts a dilute layer in that distribution and
checks that lm_bd_step_rfd (steric + gravity, M.F, Lanczos noise, RFD drift, Adams-Bashforth) KEEPS it over two relaxation
times, while the same run without the drift term (lm_bd_step) leaves it: the height-dependent mobility then piles
particles up near the wall.  No oracle run is involved: the expected distribution is a closed form."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

A, ETA, KT, MG, U0, B = 1.0, 1.0, 1.0, 1.0, 4.0, 0.1


def wall_potential(h):
    return np.where(h < A, U0 * (1.0 + (A - h) / B), U0 * np.exp((A - h) / B))          # eq. (13), d = a


def equilibrium_cdf():
    h = np.linspace(0.0, 25.0, 250001)
    w = np.exp(-(MG * h + wall_potential(h)) / KT)
    c = np.concatenate([[0.0], np.cumsum(0.5 * (w[1:] + w[:-1]) * np.diff(h))])
    return h, c / c[-1]


def ks_distance(sample, h, cdf):
    s = np.sort(sample)
    f = np.interp(s, h, cdf)
    n = s.size
    return max(np.abs(f - np.arange(1, n + 1) / n).max(), np.abs(f - np.arange(0, n) / n).max())


def run(lm, torch, with_drift, steps, every, seed):
    N, L, dt = 2048, 700.0, 0.02
    rng = np.random.default_rng(seed)
    h, cdf = equilibrium_cdf()
    z0 = np.interp(rng.random(N), cdf, h)
    pos = np.column_stack([rng.random(N) * L, rng.random(N) * L, z0]).astype(np.float32)
    s = lm.Solver("f32", N, ETA, A, False)
    s.set_wall(True, 0.0)
    s.set_max_iter(200)
    X = torch.from_numpy(pos.reshape(-1)).cuda()
    F = torch.zeros(N, 3, dtype=torch.float32, device="cuda")
    F[:, 2] = -MG
    F = F.reshape(-1)
    g = torch.Generator(device="cuda")
    g.manual_seed(seed)
    heights = []
    for n in range(steps):
        W = torch.randn(3 * N, dtype=torch.float32, device="cuda", generator=g)
        if with_drift:
            Wt = torch.randn(3 * N, dtype=torch.float32, device="cuda", generator=g)
            s.bd_step_rfd(X, F, None, W, Wt, 0.05, dt, KT, U0, B, 1e-3, allow_noconv=True)
        else:
            s.bd_step(X, F, None, W, dt, KT, U0, B, 1e-3, allow_noconv=True)
        if (n + 1) % every == 0 and n + 1 >= steps // 2:
            heights.append(X.reshape(N, 3)[:, 2].cpu().numpy().astype(np.float64))
    s.close()
    return np.concatenate(heights), h, cdf


def test_gibbs_boltzmann_heights_are_kept_only_with_the_drift_term():
    import torch
    import paper_2510_02135_b200 as lm
    assert torch.cuda.is_available()
    # relaxation time ~ (k_B T / m g)^2 / (k_B T mu_0) = 6 pi ~ 19 time units = 940 steps of dt = 0.02
    steps, every = 3000, 250
    with_drift, h, cdf = run(lm, torch, True, steps, every, 1)
    without, _, _ = run(lm, torch, False, steps, every, 1)
    mean_exact = np.trapezoid(h * np.gradient(cdf, h), h)
    d_with, d_without = ks_distance(with_drift, h, cdf), ks_distance(without, h, cdf)
    m_with, m_without = with_drift.mean(), without.mean()
    assert np.isfinite(with_drift).all() and (with_drift > 0).all()
    # measured (2000 steps, two seeds): with the drift KS distance 0.008 / 0.010 and mean height 2.184 / 2.175 against the
    # exact 2.181; without it 0.094 / 0.085 and 2.04 / 2.05 (particles pile up near the wall)
    assert d_with <= 0.03 and abs(m_with / mean_exact - 1.0) <= 0.02, (d_with, m_with, mean_exact)
    assert d_without >= 0.05 and d_without >= 3 * d_with and m_without < 0.96 * mean_exact, (d_without, d_with, m_without, mean_exact)
