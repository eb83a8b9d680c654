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


def contact_density(hist_sum, n_snapshots, s_max=S_MAX, skip_bins=0):
    """Weighted quadratic fit of the pair-count density h(s) = counts / (snapshots * ds); returns h(0).

    Bin b holds Poisson-like counts c_b, so the weight of its density is ~ 1/var = 1/c_b (in count units).

    skip_bins: leave the first bins out of the fit.  The sweep accepts a move only if every margin is >= eps_g = 2e-6
    (R15), so no pair ever has a touch scale below s_g ~ eps_g / |r| ~ 2e-6: the first bin really covers
    [s_g, ds), i.e. it is short of s_g / ds of its counts (1 % for ds = 2e-4), and as the end point of a quadratic fit over n
    bins (leverage ~ 9 / n) it pulls h(0) down by ~0.2 % at n = 40.  Invisible at the 0.5 % level of the short runs, 3-4
    standard errors in runs that resolve 0.08 %; those fit bins 1.. and extrapolate across the first bin."""
    c = np.asarray(hist_sum, dtype=np.float64)
    nb = c.size
    ds = s_max / nb
    x = (np.arange(nb) + 0.5) * ds
    y = c / (n_snapshots * ds)
    sig = np.sqrt(np.maximum(c, 1.0)) / (n_snapshots * ds)
    x, y, sig = x[skip_bins:], y[skip_bins:], sig[skip_bins:]
    A = np.stack([np.ones(x.size), x, x * x], axis=1) / sig[:, None]
    coef, *_ = np.linalg.lstsq(A, y / sig, rcond=None)
    return float(coef[0])


def compressibility(hist_sum, n_snapshots, N, dim, s_max=S_MAX, skip_bins=0):
    """beta P / rho from the summed scale-factor histogram of n_snapshots snapshots of N particles."""
    return 1.0 + contact_density(hist_sum, n_snapshots, s_max, skip_bins) / (dim * N)


def mean_and_se(per_seed_values):
    v = np.asarray(per_seed_values, dtype=np.float64)
    return float(v.mean()), float(v.std(ddof=1) / np.sqrt(v.size))
