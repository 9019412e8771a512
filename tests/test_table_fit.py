"""Host-side spline fit of the library (gm_fit_pair_table, Eq. (12)) against the oracle's own fit:
two independent implementations (Thomas algorithm in C++ / elimination in numpy) of the same natural cubic spline."""
import numpy as np

from oracle import oracle as orc
from paper_1310_2041_b200 import gm


def test_library_spline_fit_matches_the_oracle_fit():
    interval = 6.25 / 2000
    z = interval * np.arange(2001)
    zz = np.maximum(z, 0.49)
    v = 4.0 * (zz ** -6 - zz ** -3)                       # Lennard-Jones in terms of z = r^2 (Eq. (1))
    c_lib = gm.gm_fit_pair_table(v, interval)
    c_orc = orc.spline_table(v, interval)
    assert c_lib.shape == (2000, 4) and c_lib.dtype == np.float32
    scale = np.abs(c_orc).max(axis=0)
    assert (np.abs(c_lib - c_orc).max(axis=0) <= 1e-6 * scale + 1e-30).all()
    # continuity of value, first and second derivative across the grid points (what Eq. (12) promises)
    h = interval
    c = c_orc
    assert np.allclose(c[:-1, 0] + h * (c[:-1, 1] + h * (c[:-1, 2] + h * c[:-1, 3])), c[1:, 0], rtol=0, atol=1e-9 * scale[0])
    assert np.allclose(c[:-1, 1] + h * (2 * c[:-1, 2] + 3 * h * c[:-1, 3]), c[1:, 1], rtol=0, atol=1e-9 * scale[1])
    assert np.allclose(2 * c[:-1, 2] + 6 * h * c[:-1, 3], 2 * c[1:, 2], rtol=0, atol=1e-8 * scale[2])
    assert gm.lib().gm_fit_pair_table(0, 1.0, None, None) == gm.GM_ERR_INVALID_ARG
