"""The seeded input generators: shapes and structure BASELINE.json's configs state; determinism."""
import numpy as np
import pytest

from paper_1607_03884_b200 import synth


@pytest.mark.parametrize("kind,ns,nr,ntb,ntroe", [("h2co", 13, 27, 4, 2), ("gri", 53, 325, 30, 29)])
def test_mechanism_shape(kind, ns, nr, ntb, ntroe):
    m = synth.make_mechanism(kind, synth.MECH_SEED)
    assert m["n_species"] == ns and m["n_reactions"] == nr
    assert (m["rxn_type"] == synth.RXN_THREE_BODY).sum() == ntb
    assert (m["rxn_type"] == synth.RXN_FALLOFF_TROE).sum() == ntroe
    assert m["species_names"][-1] == "N2"
    synth.check_mechanism(m)                       # element balance, every reactive species used
    assert np.all((m["arr_A"] >= 1e6) & (m["arr_A"] <= 1e14))
    assert np.all((m["arr_b"] >= -2) & (m["arr_b"] <= 2))
    assert np.all((m["arr_Ea"] >= 0) & (m["arr_Ea"] <= 50000))
    assert np.all((m["eff_val"] >= 0.5) & (m["eff_val"] <= 12.0))
    # N2 takes part in no reaction
    assert (ns - 1) not in set(m["reac_sp"]) | set(m["prod_sp"])
    m2 = synth.make_mechanism(kind, synth.MECH_SEED)
    for k, v in m.items():
        if isinstance(v, np.ndarray):
            assert np.array_equal(v, m2[k]), k
    m3 = synth.make_mechanism(kind, synth.MECH_SEED + 1)
    assert not np.array_equal(m["arr_A"], m3["arr_A"])


@pytest.mark.parametrize("kind", ["h2co", "gri"])
@pytest.mark.parametrize("dist", ["uniform", "ignition"])
def test_states_shape(kind, dist):
    m = synth.make_mechanism(kind, synth.MECH_SEED)
    y = synth.make_states(m, 2000, dist, 3)
    assert y.shape == (2000, m["n_species"]) and y.dtype == np.float64
    assert y[:, 0].min() >= 800.0 and y[:, 0].max() <= (2400.0 if kind == "h2co" else 2600.0)
    Ylast = 1.0 - y[:, 1:].sum(axis=1)
    assert np.all(y[:, 1:] > 0) and np.all(Ylast > -1e-12)
    if dist == "ignition":
        band = (1000.0, 1400.0) if kind == "h2co" else (1100.0, 1600.0)
        frac = ((y[:, 0] >= band[0]) & (y[:, 0] <= band[1])).mean()
        assert frac > 0.6
    assert np.array_equal(y, synth.make_states(m, 2000, dist, 3))
    assert np.array_equal(y[:100], synth.make_states(m, 2000, dist, 3)[:100])
