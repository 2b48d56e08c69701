"""Golden fixtures (tests/golden/): hand-derived closed-form windows with their citations, and an
oracle-written regression fixture (written by tests/golden/make_golden.py, which calls only oracle/)."""
import os

import numpy as np
import pytest

from oracle import rfi_oracle as orc

HERE = os.path.dirname(os.path.abspath(__file__))
GOLDEN = os.path.join(HERE, "golden")


def _cases():
    out = []
    with open(os.path.join(GOLDEN, "closed_forms.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            name, W, d, samples, tau, r_re, r_im = [x.strip() for x in line.split("|")]
            win = np.array([[complex(v.strip()) for v in s.split(",")] for s in samples.split(";")], np.complex128)
            assert win.shape == (int(W), 4), name
            out.append(pytest.param(win, float(d), float(tau), float(r_re), float(r_im), id=name))
    return out


@pytest.mark.parametrize("win,d,tau,r_re,r_im", _cases())
def test_closed_form_windows(win, d, tau, r_re, r_im):
    got = orc.window_stats(win, d)
    assert got[0] == pytest.approx(tau, rel=1e-14, abs=1e-15)
    assert got[1] == pytest.approx(r_re, rel=1e-14, abs=1e-15)
    assert got[2] == pytest.approx(r_im, rel=1e-14, abs=1e-15)


def test_oracle_regression_fixture():
    """The stored outputs of the oracle on a tiny seeded chunk (make_golden.py) still come out: guards the
    oracle's arithmetic against silent drift.  A deliberate change must regenerate the file and cite the passage."""
    from tests.golden import make_golden as mg
    stored = mg.read(os.path.join(GOLDEN, "tiny_oracle.txt"))
    fresh = mg.compute()
    assert stored.keys() == fresh.keys()
    for key in stored:
        np.testing.assert_allclose(fresh[key], stored[key], rtol=1e-12, atol=1e-14, err_msg=key)
