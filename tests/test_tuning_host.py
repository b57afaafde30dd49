"""Host logic of the tuning study (paper_2110_13115_b200/tuning.py) pinned directly, without the oracle: Eq. 16 on
counts worked out by hand.  The oracle has its own implementation and its own pins
(tests/test_oracle_pins.py); the two are only ever compared through their results (tests/test_gpu_tuning.py)."""
import numpy as np

from paper_2110_13115_b200 import tuning


def test_rho_target_on_hand_counted_lists():
    """flat = {4.0 x100, 5.0 x100, 6.0 x100, 7.0 x10}; the hierarchical search lost 30 of the 4.0s, 2 of the 5.0s and
    none above.  Counted by hand at rho_II = 4, 5, 5.5, 6, 7, 8: n_flat = 310, 210, 110, 110, 10, 0 and
    n_final = 278, 208, 110, 110, 10, 0, i.e. recovered fractions 0.897, 0.9905, 1, 1, 1, -."""
    grid = [4.0, 5.0, 5.5, 6.0, 7.0, 8.0]
    n_flat = [310, 210, 110, 110, 10, 0]
    n_final = [278, 208, 110, 110, 10, 0]
    assert tuning.rho_target(n_final, n_flat, grid, 0.99) == 5.0       # 208 / 210 = 0.9905
    assert tuning.rho_target(n_final, n_flat, grid, 0.995) == 5.5
    assert tuning.rho_target(n_final, n_flat, grid, 0.85) == 4.0
    assert tuning.rho_target(n_flat, n_flat, grid, 0.99) == 4.0        # the flat search recovers itself everywhere
    # nothing recovered, or no flat triggers at all: no target
    assert tuning.rho_target([0] * 6, n_flat, grid, 0.99) is None
    assert tuning.rho_target([0] * 6, [0] * 6, grid, 0.99) is None
    # the threshold must hold for every larger grid value: 4.0 passes (100 / 100) but 5.0 fails (70 / 80)
    assert tuning.rho_target([100, 70, 50], [100, 80, 50], [4.0, 5.0, 6.0], 0.99) == 6.0
    # a failure at the last populated threshold leaves only the empty tail
    assert tuning.rho_target([100, 80, 40, 0], [100, 80, 50, 0], [4.0, 5.0, 6.0, 7.0], 0.99) is None
    # numpy inputs of integer dtype, as tune() passes them
    assert tuning.rho_target(np.array(n_final), np.array(n_flat), np.array(grid), 0.99) == 5.0


def test_cost_ratio_reproduces_the_papers_first_stage_figures():
    """Eq. 14 / Eq. 13 at the paper's block N = 2^18: about 1/6 for w = 8 and about 1/10 for w = 16 (PAPER.md:316:
    'speed up factor of 6 ... w = 8', '~10 times ... w = 16'), and Eq. 15 adds p / T plus the second-stage term."""
    N, T, p = 1 << 18, 6250, 254
    total8, first8 = tuning.cost_ratio(N, T, 8, p, 0.0)
    total16, first16 = tuning.cost_ratio(N, T, 16, p, 0.0)
    assert abs(1.0 / first8 - 6.0) < 0.35 and abs(1.0 / first16 - 10.0) < 1.5
    assert abs((total8 - first8) - p / T) < 1e-12 and abs((total16 - first16) - p / T) < 1e-12
    more, _ = tuning.cost_ratio(N, T, 8, p, 1000.0)
    z_basic = N * T * (5.0 * 18 + 6.0)
    assert abs((more - total8) - 4.0 * p * 8 * 1000.0 * T / z_basic) < 1e-12
