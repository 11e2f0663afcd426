import numpy as np


def binned_mean_se(x, nbins=32, drop=0.0):
    """Mean and binned standard error of a time series (first `drop` fraction discarded)."""
    x = np.asarray(x, dtype=np.float64)
    x = x[int(len(x) * drop):]
    m = (len(x) // nbins) * nbins
    b = x[:m].reshape(nbins, -1).mean(axis=1)
    return float(b.mean()), float(b.std(ddof=1) / np.sqrt(nbins))
