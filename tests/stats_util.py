"""Small statistics helpers for the Monte Carlo pins (tests only)."""
import numpy as np


def blocked_mean_se(series, n_blocks=20):
    """Mean and standard error from a blocking (binning) analysis of a correlated series.

    SURVEY section 8c: raw per-sweep standard errors underestimate the error near T_c, so every
    statistical pin uses block means."""
    x = np.asarray(series, dtype=np.float64)
    n = (len(x) // n_blocks) * n_blocks
    b = x[len(x) - n:].reshape(n_blocks, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / np.sqrt(n_blocks)


def within(value, target, se, n_sigma=3.0, floor=0.0):
    return abs(value - target) <= n_sigma * se + floor
