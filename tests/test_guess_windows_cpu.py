"""The index claim behind k_guess_rhs (csrc/guess.cuh): for one source (xs) the table indices a
tile of 64 mesh columns plus its ring uses -- the difference index |x - xs| and the folded sum index f(x + xs + 1),
f(t) = t if t <= n else 2n - t -- each form a CONTIGUOUS run of at most 66 values whose smallest member is what
guess_origin computes; rounded down to a multiple of four entries (the TMA box origin must be 16-byte aligned) every
index still falls inside the 72-wide box.  Brute force over mesh sizes, tiles and sources; integers only."""
import itertools

TX, BW = 64, 72


def fold(t, n):
    return t if t <= n else 2 * n - t


def origin(lo, hi, s, n):
    """guess_origin of csrc/guess.cuh, restated: smallest |x - s| and smallest f(x + s + 1) over x in [lo, hi]."""
    a_d = max(lo - s, s - hi, 0)
    tlo, thi = lo + s + 1, hi + s + 1
    a_s = tlo if thi <= n else (2 * n - thi if tlo > n else min(tlo, 2 * n - thi))
    return a_d, a_s


def check(n, tile_w, box_w, align):
    for t0 in range(0, n, tile_w):
        lo, hi = max(t0 - 1, 0), min(t0 + tile_w, n - 1)      # the tile and its ring, clamped to the mesh
        for s in range(n):
            d = {abs(x - s) for x in range(lo, hi + 1)}
            f = {fold(x + s + 1, n) for x in range(lo, hi + 1)}
            for vals, a in zip((d, f), origin(lo, hi, s, n)):
                assert min(vals) == a
                assert vals == set(range(min(vals), max(vals) + 1)), "a gap in the window"
                assert max(vals) - min(vals) + 1 <= tile_w + 2
                a4 = a - a % align
                assert a4 >= 0 and max(vals) - a4 < box_w
                assert max(vals) <= n                           # inside the (n + 1)-wide table


def test_column_windows_are_contiguous_and_fit_the_box():
    for n in (192, 193, 255, 256, 301, 512):
        check(n, TX, BW, 4)


def test_row_windows_fit_the_box_height():
    for n, ty in itertools.product((192, 257, 300), (16, 24, 32)):
        check(n, ty, ty + 2, 1)   # rows need no alignment: the box is TY + 2 high
