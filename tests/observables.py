"""Long-run observables and their statistical error bars (test helper; plain numpy, none of the method's arithmetic).

BASELINE.json north_star: "Long-run averages (T, potential energy, RDF, diffusion constant) must agree within stated
statistical error bars" and "the hybrid process still samples mu (temperature, RDF and energy distributions on small
systems)" (the velocity-jump process leaves mu invariant; P:L527-531, L575-589 are the paper's own
evidence of this kind: temperatures, radial distribution functions, diffusion constants).
"""
import numpy as np


def block_mean_se(x, n_blocks=8):
    """Mean of a correlated time series and its standard error from n_blocks block averages."""
    x = np.asarray(x, dtype=np.float64)
    m = (len(x) // n_blocks) * n_blocks
    b = x[:m].reshape(n_blocks, -1).mean(axis=1)
    return float(x[:m].mean()), float(b.std(ddof=1) / np.sqrt(n_blocks))


def agree(a, b, n_sigma=4.0, slack=0.0):
    """(mean, se) pairs agree within n_sigma combined standard errors plus an absolute slack (time-step bias)."""
    return abs(a[0] - b[0]) <= n_sigma * np.hypot(a[1], b[1]) + slack


def rdf(snapshots, box, r_max, n_bins):
    """g(r) of one species from a list of (n, 3) position snapshots in a cubic periodic box (minimum image)."""
    edges = np.linspace(0.0, r_max, n_bins + 1)
    hist = np.zeros(n_bins)
    n = snapshots[0].shape[0]
    iu = np.triu_indices(n, 1)
    for x in snapshots:
        d = x[:, None, :] - x[None, :, :]
        d -= box * np.round(d / box)
        r = np.sqrt((d ** 2).sum(-1))[iu]
        hist += np.histogram(r, bins=edges)[0]
    shell = 4.0 / 3.0 * np.pi * (edges[1:] ** 3 - edges[:-1] ** 3)
    ideal = 0.5 * n * (n - 1) / box ** 3 * shell * len(snapshots)
    return 0.5 * (edges[1:] + edges[:-1]), hist / ideal


def rdf_blocks(snapshots, box, r_max, n_bins, n_blocks=4):
    """g(r) and its per-bin standard error from n_blocks blocks of snapshots."""
    per = len(snapshots) // n_blocks
    gs = np.array([rdf(snapshots[k * per:(k + 1) * per], box, r_max, n_bins)[1] for k in range(n_blocks)])
    r = rdf(snapshots[:1], box, r_max, n_bins)[0]
    return r, gs.mean(0), gs.std(0, ddof=1) / np.sqrt(n_blocks)


def unwrap(snapshots, box):
    """Continuous trajectories from wrapped snapshots taken often enough that no atom moves box/2 in between."""
    out = [snapshots[0].astype(np.float64)]
    for x in snapshots[1:]:
        d = x - (out[-1] - box * np.floor(out[-1] / box))
        d -= box * np.round(d / box)
        out.append(out[-1] + d)
    return np.array(out)


def diffusion_atoms(snapshots, box, dt_ps, lag_lo, lag_hi):
    """Apparent self-diffusion constant (A^2/ps) from the MSD slope between two lags (in snapshots), averaged over
    all time origins; the error bar is the standard error over the atoms' individual estimates."""
    traj = unwrap(snapshots, box)
    per_atom = []
    for lag in (lag_lo, lag_hi):
        d = traj[lag:] - traj[:-lag]
        per_atom.append((d ** 2).sum(-1).mean(0))
    est = (per_atom[1] - per_atom[0]) / (6.0 * (lag_hi - lag_lo) * dt_ps)
    return float(est.mean()), float(est.std(ddof=1) / np.sqrt(len(est)))
