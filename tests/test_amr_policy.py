"""Algorithm 1 of the paper (reading B13 in DESIGN.md): the capacity N_max of a refinement layer."""
from paper_2504_13750_b200.amr import update_n_max


def test_doubles_until_the_valid_blocks_fit():
    assert update_n_max(0, 1) == 1
    assert update_n_max(1, 1) == 2                    # N_valid + 1 > N_max -> 2 N_max
    assert update_n_max(8, 1) == 16                   # one regrid may add many blocks: applied until stable
    assert update_n_max(100, 16) == 128


def test_halves_only_below_the_hysteresis_band():
    assert update_n_max(8, 16) == 16                  # 9 * 2.5 = 22.5 >= 16: stays
    assert update_n_max(6, 16) == 16                  # 7 * 2.5 = 17.5 >= 16: stays
    assert update_n_max(5, 16) == 8                   # 6 * 2.5 = 15 < 16 -> N_max / 2
    assert update_n_max(0, 64) == 2


def test_is_stable_and_always_holds_the_valid_blocks():
    for n_max in (1, 2, 8, 64, 1024):
        for n_valid in range(0, 300, 7):
            m = update_n_max(n_valid, n_max)
            assert m >= n_valid + 1 or (n_valid == 0 and m == 1)
            assert update_n_max(n_valid, m) == m      # a second application changes nothing
            assert m == 1 or (n_valid + 1) * 2.5 >= m
