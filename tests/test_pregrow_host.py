"""Host helpers of pregrow.py (numpy only, no GPU): extent of the occupied set and the radial profile."""
import numpy as np

from paper_2303_08123_b200 import pregrow
from tests._helpers import blank_state, K_G1, K_DEAD


def test_extent_and_radial_profile_of_a_layered_ball():
    n = 40
    st = blank_state(n, n, n)
    z, y, x = np.indices(st.shape)
    r = np.sqrt((x - 20) ** 2 + (y - 20) ** 2 + (z - 20) ** 2)
    st[(r <= 12) & (r > 8)] = K_G1 | (0 << 3)            # proliferating aerobic rim
    st[(r <= 8) & (r > 5)] = K_G1 | (3 << 3)             # quiescent anaerobic shell
    st[(r <= 5) & (r > 2)] = K_DEAD                      # necrotic core, lysed in the middle
    assert pregrow.extent(st) == 25
    assert pregrow.extent(blank_state(8, 8, 8)) == 0
    prof = pregrow.radial_profile(dict(state=st))
    assert prof["proliferating"][1] > prof["quiescent"][1] > prof["dead"][1]
    assert prof["anaerobic"][0] == prof["quiescent"][0]
    assert abs(prof["r_max"] - 12.0) < 0.2
    assert prof["empty_inside_half_radius"] == int((r <= 2).sum())
    one = blank_state(9, 9, 9); one[4, 4, 4] = K_G1
    assert pregrow.extent(one) == 1
