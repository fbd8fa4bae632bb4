"""Pins of the oracle's extended likelihood (reading D4): the identity with the fraction
form, -log L_ext = NLL(f = ns/(ns+nb)) + (ns+nb) - N log(ns+nb); the closed-form minimum over the total yield at
fixed fraction, nu_hat = N; and the mpmath definition on a few events."""
import mpmath as mp
import numpy as np

import ipa_inputs as inp
from test_oracle_ipatia import MPModel

LO, HI = inp.LO, inp.HI


def test_extended_equals_fraction_form_plus_yield_terms(orc):
    x = orc.generate_mixture(3, 5000, inp.GEN, LO, HI)
    for P, ns, nb in ((inp.GEN, 1500.0, 3400.0), (inp.P2, 10.0, 7000.0), (inp.GEN, 0.0, 5000.0), (inp.P2, 4000.0, 0.0)):
        nu = ns + nb
        frac = orc.nll(x, dict(P, f=ns / nu), LO, HI)[0]
        ext = orc.nll_extended(x, P, ns, nb, LO, HI)
        assert abs(ext - (frac + nu - x.size * np.log(nu))) <= 1e-12 * abs(ext)


def test_total_yield_minimum_is_the_number_of_events(orc):
    x = orc.generate_mixture(4, 2000, inp.GEN, LO, HI)
    f = 0.3
    v = [orc.nll_extended(x, inp.GEN, f * nu, (1 - f) * nu, LO, HI) for nu in (1990.0, 2000.0, 2010.0)]
    assert v[1] < v[0] and v[1] < v[2]
    # parabola through the three points: vertex at nu = N up to O((dnu/N)^2)
    a = (v[0] + v[2] - 2 * v[1]) / 2 / 100.0
    b = (v[2] - v[0]) / 20.0
    assert abs(-b / (2 * a)) < 0.1


def test_extended_definition_mpmath(orc):
    mp.mp.dps = 30
    xs = [5004.0, 5251.5, 5280.25, 5309.0, 5577.0]
    ns, nb = 2.5, 3.75
    m = MPModel(inp.P2)
    ref = (mp.mpf(ns) + mp.mpf(nb)) - sum(mp.log(ns * m.I(mp.mpf(x) - m.mu) / m.NS + nb * mp.exp(m.k * (mp.mpf(x) - m.lo)) / m.NB)
                                           for x in xs)
    got = orc.nll_extended(np.array(xs), inp.P2, ns, nb, LO, HI)
    assert abs(got - float(ref)) <= 1e-12 * abs(float(ref))
