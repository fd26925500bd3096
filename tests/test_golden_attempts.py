"""The paper's printed multi-start arithmetic, the only numbers in the text that a program here
can reproduce: 35.7 / 6.3 / 4.3 % success -> 11 / 71 / 105 attempts for a < 1 % miss probability."""
import os

from oracle.multistart import attempts_needed, miss_probability

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "attempts.txt")


def _rows():
    with open(GOLDEN) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                name, rate, n = line.split()
                yield name, float(rate) / 100.0, int(n)


def test_attempts_match_the_paper():
    rows = list(_rows())
    assert len(rows) == 3
    for name, rate, n in rows:
        assert attempts_needed(rate) == n, name
        assert miss_probability(rate, n) < 0.01 <= miss_probability(rate, n - 1), name
