"""O9 / O10 analysis (TEST INFRASTRUCTURE): volume-perturbation pressure from snapshots.

"We compute pressure in NVT simulations by building a histogram of scale factors s that cause two
neighboring particles to overlap and extrapolate the probability of overlap at s=0".
Compressing every separation by (1 - s) changes the volume by dV/V = -dim*s; the probability that the
compressed configuration has an overlap is, to first order, the mean number of pairs whose touch scale
1 - lambda* lies below s.  Hence

    beta P / rho = 1 + h(0) / (dim * N),     h(0) = d<pairs with touch scale < s>/ds at s -> 0+.

For disks h(0) = N rho pi sigma^2 g(sigma+), i.e. the textbook 1 + (pi/2) rho sigma^2 g(sigma+).

The histogram itself comes from oracle/hpmc_oracle.c:orc_scale_histogram, applied identically to snapshots
taken from the CUDA path and from the oracle; nothing here is on the product path.
"""
import numpy as np

S_MAX = 0.02
NBINS = 40


def contact_density(hist_sum, n_snapshots, s_max=S_MAX):
    """Weighted quadratic fit of the pair-count density h(s) = counts / (snapshots * ds); returns h(0).

    Bin b holds Poisson-like counts c_b, so the weight of its density is ~ 1/var = 1/c_b (in count units)."""
    c = np.asarray(hist_sum, dtype=np.float64)
    nb = c.size
    ds = s_max / nb
    x = (np.arange(nb) + 0.5) * ds
    y = c / (n_snapshots * ds)
    sig = np.sqrt(np.maximum(c, 1.0)) / (n_snapshots * ds)
    A = np.stack([np.ones(nb), x, x * x], axis=1) / sig[:, None]
    coef, *_ = np.linalg.lstsq(A, y / sig, rcond=None)
    return float(coef[0])


def compressibility(hist_sum, n_snapshots, N, dim, s_max=S_MAX):
    """beta P / rho from the summed scale-factor histogram of n_snapshots snapshots of N particles."""
    return 1.0 + contact_density(hist_sum, n_snapshots, s_max) / (dim * N)


def mean_and_se(per_seed_values):
    v = np.asarray(per_seed_values, dtype=np.float64)
    return float(v.mean()), float(v.std(ddof=1) / np.sqrt(v.size))
