"""The oracle against stored values of itself (tests/golden/oracle_regression.json, written by
tests/golden/make_golden.py, which calls only oracle/): guards its arithmetic against accidental
changes.  The physics of those numbers is pinned elsewhere (test_oracle_physics.py); config 1's
energy is also checked here against the closed form it must approach (hbar (wx + wy) / 2 = 1)."""
import importlib.util
import json
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
MG = importlib.util.module_from_spec(spec)
spec.loader.exec_module(MG)

with open(os.path.join(HERE, "golden", "oracle_regression.json")) as f:
    GOLD = json.load(f)


@pytest.mark.parametrize("name", sorted(GOLD))
def test_oracle_reproduces_stored_values(name):
    got = MG.run(*MG.cases()[name])
    want = GOLD[name]
    for k, v in want.items():
        a, b = np.asarray(got[k], dtype=np.float64), np.asarray(v, dtype=np.float64)
        # OpenMP reduction order moves the last digits of the sums that feed back into psi
        assert np.allclose(a, b, rtol=1e-9, atol=1e-12), (name, k)


def test_config1_energy_near_closed_form():
    e = GOLD["config1_g0"]
    assert e["e_kin"] + e["e_pot"] == pytest.approx(1.0, abs=2e-4)       # E - 1 ~ 1e-4 at tau = 2
    assert e["norm"] == pytest.approx(1.0, abs=1e-12)
    assert GOLD["config1_g10"]["e_kin"] + GOLD["config1_g10"]["e_pot"] + GOLD["config1_g10"]["e_int"] > 1.5
