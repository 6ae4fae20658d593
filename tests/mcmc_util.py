"""Minimal Monte Carlo standard errors (batch means) for the posterior-agreement tests."""
import numpy as np


def mcse_batch_means(x, n_batches=30):
    """MCSE of the mean of each column of the chain x (T, d) by non-overlapping batch means."""
    x = np.asarray(x, dtype=np.float64)
    if x.ndim == 1:
        x = x[:, None]
    T = (x.shape[0] // n_batches) * n_batches
    b = x[:T].reshape(n_batches, T // n_batches, -1).mean(1)
    return b.std(0, ddof=1) / np.sqrt(n_batches)


def mean_and_var_with_mcse(x, n_batches=30):
    """(mean, mcse of mean, variance, mcse of variance) per column."""
    x = np.asarray(x, dtype=np.float64)
    if x.ndim == 1:
        x = x[:, None]
    m = x.mean(0)
    sq = (x - m) ** 2
    return m, mcse_batch_means(x, n_batches), x.var(0, ddof=1), mcse_batch_means(sq, n_batches)
