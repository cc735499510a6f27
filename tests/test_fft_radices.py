"""Host logic of the mixed-radix transforms (csrc/pz_fft_generic.cu): the
factorisation the kernels run with, through the C ABI (pz_fft_radices; no GPU needed).  Checked
against what the arithmetic fixes: the radices multiply to n, each is one the kernels implement,
7-smooth lengths are exactly the ones accepted, no factorisation with fewer passes exists (brute
force), an odd radix goes first whenever n has an odd factor within the fewest passes (its
first-pass writes are free of bank conflicts), and the points-per-thread constraint is respected."""
import itertools
import math

import pytest

from paper_2502_06296_b200 import binding as pz

RADICES = (2, 3, 4, 5, 6, 7, 8, 9, 10, 12, 14, 15, 16)
# points a thread keeps per pass (kE = 16): ceil(16 / R) butterflies up to radix 9, one above
POINTS = {R: min(16, (-(-16 // R) if R <= 9 else 1) * R) for R in RADICES}


def smooth7(n):
    for f in (2, 3, 5, 7):
        while n % f == 0:
            n //= f
    return n == 1


def fewest_passes(n, allowed):
    best = {1: 0}
    for m in range(2, n + 1):
        if n % m:
            continue
        c = [best[m // r] + 1 for r in allowed if m % r == 0 and (m // r) in best]
        if c:
            best[m] = min(c)
    return best.get(n)


LENGTHS = [4, 6, 12, 30, 48, 60, 192, 384, 448, 1536, 1600, 1728, 3072, 3200, 3456, 3584, 4096, 5000, 6144, 7168, 8192]


@pytest.mark.parametrize("n", LENGTHS)
def test_radices_multiply_to_n_and_are_fewest(n):
    r = pz.pz_fft_radices(n)
    assert r and all(x in RADICES for x in r)
    assert math.prod(r) == n
    # the cost model charges 10 per pass and at most 2 * 7 for conflicts: never more than one pass above the minimum
    assert len(r) <= fewest_passes(n, RADICES) + 1


@pytest.mark.parametrize("n", range(2, 400))
def test_exactly_the_7_smooth_lengths_are_accepted(n):
    r = pz.pz_fft_radices(n)
    assert bool(r) == smooth7(n)
    if r:
        assert math.prod(r) == n


def test_paper_grid_lengths():
    """7168 / 2, 3200 / 2, 3456 / 2 along x (half-length complex transforms)."""
    assert sorted(pz.pz_fft_radices(1728)) == [9, 12, 16] and pz.pz_fft_radices(1728)[0] == 9
    assert sorted(pz.pz_fft_radices(3584)) == [14, 16, 16] and pz.pz_fft_radices(3584)[0] == 14
    assert sorted(pz.pz_fft_radices(1600)) == [10, 10, 16] and pz.pz_fft_radices(1600)[0] == 10
    assert math.prod(pz.pz_fft_radices(3072, 12, 2)) == 3072 and len(pz.pz_fft_radices(3072, 12, 2)) == 3


@pytest.mark.parametrize("n", [27, 45, 105, 225, 1728, 3375, 2 * 3 * 5 * 7 * 8])
def test_odd_radix_first_when_it_costs_no_pass(n):
    r = pz.pz_fft_radices(n)
    odd_sets = [c for k in range(1, len(r) + 1) for c in itertools.combinations_with_replacement(RADICES, k)
                if math.prod(c) == n and any(x % 2 for x in c)] if n < 4000 else [r]
    if any(len(c) == len(r) for c in odd_sets):
        assert r[0] % 2 == 1


@pytest.mark.parametrize("n,min_points", [(8192, 16), (7680, 15), (6144, 12), (5120, 10), (7776, 16)])
def test_points_per_thread_constraint(n, min_points):
    r = pz.pz_fft_radices(n, min_points)
    if r:
        assert math.prod(r) == n and all(POINTS[x] >= min_points for x in r)
    else:
        # only acceptable where no allowed set of radices exists
        allowed = [x for x in RADICES if POINTS[x] >= min_points]
        assert fewest_passes(n, allowed) is None


def test_refusals():
    assert pz.pz_fft_radices(1) == [] and pz.pz_fft_radices(0) == [] and pz.pz_fft_radices(11) == []
    assert pz.pz_fft_radices(2 * 11) == [] and pz.pz_fft_radices(64, 17) == []
