"""The mode-group recipe of workloads.py (Table 2): 120 modes in 15 groups of 1, 2, ..., 15."""
import numpy as np

from paper_1901_01895_b200 import workloads


def test_fifteen_groups_for_120_modes():
    p = workloads.problem(3, N=64)
    kap, group_of = p.kappa_grouped()
    assert p.M == 120 and kap.shape == (120, 120) and int(group_of.max()) + 1 == 15
    assert [int((group_of == g).sum()) for g in range(15)] == list(range(1, 16))        # 1 + 2 + ... + 15 = 120
    assert np.array_equal(kap, kap.T) and len({tuple(r) for r in kap}) == 15
    assert np.all(kap[group_of[:, None] == group_of[None, :]] == 1.0)                   # within a group: 1
    k2, _ = p.kappa_grouped()
    assert np.array_equal(kap, k2)                                                       # seeded
