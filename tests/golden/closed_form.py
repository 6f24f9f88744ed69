"""Textbook closed forms used as statistical pins (no oracle, no CUDA)."""
from math import comb


def expected_bins_hit(E: int, k: int, bins: int) -> float:
    """E[#distinct bins hit] when a uniform k-subset of E items is drawn and the items are
    spread evenly over `bins` bins: bins * (1 - C(E - E/bins, k) / C(E, k))."""
    per = E // bins
    return bins * (1.0 - comb(E - per, k) / comb(E, k))
