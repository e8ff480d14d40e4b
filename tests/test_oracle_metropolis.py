"""Pins of the oracle's Metropolis update ("standard Metropolis algorithm"; DESIGN R21), -m "not gpu".

The paper states the algorithm but not its proposal; DESIGN R21 takes one hit per link with a symmetric
uniform proposal of half-width delta.  What fixes the implementation independently of itself:
the proposal map and the Philox keying recomputed here word by word (beta = 0: every proposal is accepted);
the von Mises law exp(beta k cos(theta - alpha)) being stationary under the update (KS test against the
scipy CDF on links that all see the same staple; a wrong sign or a missing beta fails it); the strong-coupling
closed form <cos theta_P> = I1(beta)/I0(beta); agreement with the heatbath chain (already pinned) at beta = 1.
"""
import numpy as np
from scipy import special, stats

from tests import inputs


def _series_mean_err(v, nbin=10):
    v = np.asarray(v, dtype=np.float64)
    b = v[: len(v) // nbin * nbin].reshape(nbin, -1).mean(axis=1)
    return v.mean(), b.std(ddof=1) / np.sqrt(nbin)


def test_beta_zero_accepts_everything_and_follows_the_keying(ulo):
    seed, delta = (0x77 << 32) | 0x1234567, 0.9
    o = ulo.Oracle(4, 4, 0.0, seed)
    o.set_update_algorithm(1, delta)
    o.set_counter(5)
    before = o.get_links().reshape(4, -1).astype(np.float64)
    o.substep(2, 1, 2, 0)                                           # Metropolis, parity 1, mu = 2
    after = o.get_links().reshape(4, -1)
    coords = np.indices((4, 4, 4, 4)).reshape(4, -1)               # t, x3, x2, x1 of every site
    par = coords.sum(axis=0) & 1
    assert np.array_equal(after[[0, 1, 3]], before[[0, 1, 3]].astype(np.float32))
    assert np.array_equal(after[2][par == 0], before[2][par == 0].astype(np.float32))
    for site in (1, 4, 16, 77, 254):                                # odd sites
        assert par[site] == 1
        w = ulo.philox4x32_10([site, 5, 0, (3 << 3) | (1 << 2) | 2], [seed & 0xffffffff, seed >> 32])
        u1 = (2 * (int(w[0]) >> 9) + 1) * 2.0 ** -24
        want = before[2, site] + delta * (2 * u1 - 1)
        want -= 2 * np.pi * np.round(want / (2 * np.pi))
        assert after[2, site] == np.float32(want)
    assert o.get_counter() == 5                                     # a sub-step does not advance the counter
    o.sweep(1, 0)
    assert o.get_counter() == 6                                     # a Metropolis sweep does


def test_rejections_keep_links_bit_for_bit_and_acceptance_falls_with_delta(ulo):
    acc = []
    for delta in (0.2, 1.0, np.pi):
        o = ulo.Oracle(6, 4, 2.0, 3)
        o.set_update_algorithm(1, delta)
        for _ in range(6):
            o.sweep(1, 0)
        before = o.get_links()
        o.sweep(1, 0)
        after = o.get_links()
        moved = before != after
        acc.append(moved.mean())
        d = np.abs(after.astype(np.float64) - before)[moved]
        d = np.minimum(d, 2 * np.pi - d)
        assert d.max() <= delta + 1e-6                               # never further than the proposal width
    assert acc[0] > acc[1] > acc[2] > 0.05 and acc[0] > 0.8


def test_von_mises_is_stationary_under_the_update(ulo):
    # All links 0 except theta_0 on even sites: those links all see the staple S = 6 (k = 6, alpha = 0) and do
    # not appear in each other's staples, so each sub-step is an independent Metropolis hit per link at a = 6 beta.
    Ns, Nt, beta = 8, 8, 0.5
    a = 6 * beta
    rng = np.random.default_rng(4)
    coords = np.indices((Nt, Ns, Ns, Ns))
    even = (coords.sum(axis=0) & 1) == 0
    for start in ("vonmises", "uniform"):
        o = ulo.Oracle(Ns, Nt, beta, 21)
        o.set_update_algorithm(1, 2.0)
        links = np.zeros((4, Nt, Ns, Ns, Ns), dtype=np.float32)
        n = int(even.sum())
        links[0][even] = (rng.vonmises(0.0, a, n) if start == "vonmises" else rng.uniform(-np.pi, np.pi, n)).astype(np.float32)
        o.set_links(links)
        for it in range(1 if start == "vonmises" else 40):
            o.set_counter(it)
            o.substep(2, 0, 0, 0)
        th = o.get_links()[0][even].astype(np.float64)
        assert not o.get_links()[1:].any()
        _, p = stats.kstest(th, stats.vonmises(kappa=a).cdf)
        assert p > 1e-3, (start, p)
        _, p_wrong = stats.kstest(th, stats.vonmises(kappa=1.5 * a).cdf)
        assert p_wrong < 1e-4                                        # the test has the power to see a wrong beta
        assert abs(np.cos(th).mean() - special.iv(1, a) / special.iv(0, a)) < 4 * np.sqrt(0.5 / n)


def test_strong_coupling_plaquette_with_metropolis(ulo):
    o = ulo.Oracle(6, 6, 0.1, 31)
    o.set_update_algorithm(1, np.pi)
    o.sweep(10, 0)
    vals = []
    for _ in range(150):
        o.sweep(1, 1)
        vals.append(o.plaquette()[0])
    m, e = _series_mean_err(vals)
    want = special.iv(1, 0.1) / special.iv(0, 0.1)
    assert e < 2e-3 and abs(m - want) < 4 * e, (m, e, want)


def test_metropolis_and_heatbath_chains_agree_at_beta_one(ulo):
    res = []
    for alg in (0, 1):
        o = ulo.Oracle(4, 4, 1.0, 41 + alg)
        o.set_update_algorithm(alg, 1.2)
        o.sweep(60, 60)
        vals = []
        for _ in range(300):
            o.sweep(1, 3)                                           # the paper's recipe: 1 stochastic + 3 overrelaxation
            vals.append(o.plaquette()[0])
        res.append(_series_mean_err(vals))
    (m0, e0), (m1, e1) = res
    assert abs(m0 - m1) < 4 * np.hypot(e0, e1), res
    assert max(e0, e1) < 0.02                                       # the comparison has teeth (errors scatter 0.004-0.014 with the seed at beta = 1)


def test_error_codes(ulo):
    o = ulo.Oracle(4, 4, 1.0, 1)
    for bad in ((2, 1.0), (1, 0.0), (1, 4.0), (-1, 1.0)):
        try:
            o.set_update_algorithm(*bad)
        except Exception:
            continue
        raise AssertionError(bad)
    o.set_update_algorithm(0)
