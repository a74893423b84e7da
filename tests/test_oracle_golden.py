"""The oracle reproduces its own stored config-1 anchor (tests/golden/, written from oracle/ only)."""
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def test_config1_anchor():
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_c1_golden", os.path.join(HERE, "golden", "make_c1_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    prof, rmin, rmax = mod.compute()
    with open(os.path.join(HERE, "golden", "c1_oracle_u_profile_step200.txt")) as fh:
        rows = [ln for ln in fh if not ln.startswith("#")]
    g_rmin, g_rmax = (float(v) for v in rows[0].split())
    g_prof = np.array([float(r) for r in rows[1:]])
    assert abs(rmin - g_rmin) < 1e-12 and abs(rmax - g_rmax) < 1e-12
    np.testing.assert_allclose(prof, g_prof, atol=1e-12)
    # physically sane: wake deficit below roof height (z < 16) relative to the inlet log law, recovery above
    assert prof[4] < prof[24]
