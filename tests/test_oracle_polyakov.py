"""Pins of the oracle's Polyakov-loop average with analytic multihit (Eqs. 15-16), -m "not gpu".

Closed forms (cold start: r(6 beta)^Nt; constant temporal angle; beta = 0), gauge invariance on random
configurations (a wrong sign of alpha breaks it), a numpy restatement from the pinned staple with scipy's Bessel
functions, and the statistical statement that the multihit estimator has the same mean and a smaller variance.
"""
import numpy as np
from scipy import special

from tests import inputs


def _ratio(a):
    return special.ive(1, a) / special.ive(0, a)


def test_closed_forms(ulo):
    Ns, Nt, beta = 4, 6, 0.8
    o = ulo.Oracle(Ns, Nt, beta, 1)
    o.init(0)
    assert abs(o.polyakov(0) - 1) < 1e-15
    assert abs(o.polyakov(1) - _ratio(6 * beta) ** Nt) < 1e-14           # every staple sum is 6
    links = np.zeros((4, Nt, Ns, Ns, Ns), dtype=np.float32)
    links[0] = 0.25                                                      # constant temporal angle: P = e^{i Nt phi}
    o.set_links(links)
    assert abs(o.polyakov(0) - np.exp(1j * Nt * float(np.float32(0.25)))) < 1e-14
    assert abs(o.polyakov(1) - _ratio(6 * beta) ** Nt * np.exp(1j * Nt * float(np.float32(0.25)))) < 1e-13   # plaquettes are all trivial
    z = ulo.Oracle(Ns, Nt, 0.0, 1)
    assert z.polyakov(1) == 0                                            # beta = 0: the link average vanishes
    assert abs(z.polyakov(0) - z.polyakov_naive(0)[1]) < 1e-15


def test_gauge_invariance(ulo):
    Ns, Nt = 4, 4
    links = inputs.hot_links(Ns, Nt, 8) * 0.5
    lam = inputs.gauge_function(Ns, Nt, 9)
    o = ulo.Oracle(Ns, Nt, 1.1, 1)
    vals = []
    for cfg in (links, inputs.gauge_transform(links, lam)):
        o.set_links(cfg)
        vals.append((o.polyakov(0), o.polyakov(1)))
    assert abs(vals[0][0] - vals[1][0]) < 2e-6 and abs(vals[0][1] - vals[1][1]) < 2e-6   # fp32 storage of the transformed links
    assert abs(vals[0][1]) > 1e-4


def test_numpy_restatement_from_the_staple(ulo):
    Ns, Nt, beta = 4, 4, 0.9
    o = ulo.Oracle(Ns, Nt, beta, 5)
    o.sweep(3, 1)
    Vs = Ns ** 3
    P = np.ones(Vs, dtype=complex)
    for t in range(Nt):
        for xs in range(Vs):
            k, alpha = o.staple(0, xs + Vs * t)
            P[xs] *= _ratio(beta * k) * np.exp(1j * alpha)
    assert abs(o.polyakov(1) - P.mean()) < 1e-13


def test_multihit_has_the_same_mean_and_less_noise(ulo):
    # Re <P conj(P_ref)> is not available without a reference phase, so compare <|mean_x P|^2>-free quantities:
    # the lattice means over an ensemble, real and imaginary parts, and their spreads.
    Ns, Nt, beta = 4, 2, 1.3                                             # deconfined, short time extent: |<P>| is sizeable
    o = ulo.Oracle(Ns, Nt, beta, 17)
    o.init(0)
    o.sweep(30, 30)
    plain, mh = [], []
    for _ in range(200):
        o.sweep(1, 2)
        plain.append(o.polyakov(0))
        mh.append(o.polyakov(1))
    plain, mh = np.array(plain), np.array(mh)
    d = mh - plain                                                       # same configurations: the difference has mean zero
    nb = 10
    db = d.reshape(nb, -1).mean(axis=1)
    err = np.hypot(db.real.std(ddof=1), db.imag.std(ddof=1)) / np.sqrt(nb)
    assert abs(d.mean()) < 4 * err + 1e-3, (d.mean(), err)
    assert abs(plain.mean()) > 0.05                                      # there is a signal to speak of
    assert np.abs(d).mean() < 0.5 * np.abs(plain).mean()                 # and the two estimators track each other
