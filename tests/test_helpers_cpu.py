"""The sub-box trick used by the large-grid GPU parity tests, checked on the CPU against a full
oracle step, and the input generators' stated properties."""
import math

import numpy as np

from oracle import mhd_c, mhd_numpy as mn
from paper_2012_08758_b200 import inputs
import helpers


def test_subbox_equals_full_oracle_step():
    state = inputs.smooth_strong_state((40, 36, 32), 3)
    lengths = (2 * math.pi, 2 * math.pi, 2 * math.pi)
    forcing = helpers.oracle_forcing(5, 2, 3, 1.0, 2e-3, 0.02, 1.0)
    full = mhd_c.step(state, 2e-3, lengths, 1e-3, 2e-3, 1.0, forcing)
    for centre in ((0, 0, 0), (39, 35, 31), (7, 20, 30), (20, 1, 16)):
        got = helpers.subbox_oracle_step(state, centre, 2e-3, lengths, 1e-3, 2e-3, 1.0, forcing)
        want = full[:, centre[0], centre[1], centre[2]]
        assert np.abs(got - want).max() < 1e-14 * np.abs(full).max()


def test_input_generators():
    s = inputs.gaussian_state(16, 1001)
    assert s.shape == (7, 16, 16, 16) and np.all(s[0] == 0)
    assert 0.8e-3 < s[1:4].std() < 1.2e-3 and 0.8e-5 < s[4:7].std() < 1.2e-5
    assert np.array_equal(s, inputs.gaussian_state(16, 1001))
    v = inputs.solenoidal_state((16, 20, 24), 1003)
    u2 = (v[1:4] ** 2).sum(axis=0).mean()
    assert abs(math.sqrt(u2) - 0.1) < 1e-12
    # solenoidal to truncation error of the 6th-order stencil at |k| <= 4 (not to round-off)
    h = mn.grid_spacing(v.shape[1:], helpers.TWO_PI3)
    div = mn.der1(v[1], 0, h) + mn.der1(v[2], 1, h) + mn.der1(v[3], 2, h)
    grad = abs(mn.der1(v[1], 0, h)).max()
    assert np.abs(div).max() < 0.05 * grad
    ks, amps = inputs.solenoidal_modes(1003)
    assert len(ks) == 128 and all(abs(np.dot(k, a)) < 1e-12 for k, a in zip(ks, amps))
    w = inputs.uniform_state(8, 3)
    assert w.min() >= 0.0 and w.max() < 1.0
