"""Multi-start bookkeeping of the fit comparison (TEST INFRASTRUCTURE, see oracle/__init__.py).

PAPER.md:133: with a per-fit success rate alpha, the number of random starts N needed so that the chance of
never reaching the global optimum is below `miss` satisfies (1 - alpha)^N < miss.  The paper prints N = 11, 71
and 105 for alpha = 35.7 %, 6.3 % and 4.3 % at miss = 1 % (tests/golden/attempts.txt)."""
import math


def attempts_needed(success_rate: float, miss: float = 0.01) -> int:
    if not (0.0 < success_rate < 1.0 and 0.0 < miss < 1.0):
        raise ValueError("rates must lie in (0, 1)")
    return math.ceil(math.log(miss) / math.log(1.0 - success_rate))


def miss_probability(success_rate: float, n_starts: int) -> float:
    return (1.0 - success_rate) ** n_starts
