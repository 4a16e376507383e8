"""Adaptive importance-sampling grid of the integration step (oracle; test infrastructure).

The paper integrates with BASES: "a grid-optimisation step followed by an integration
step", a VEGAS-type grid in every integration variable (refs [10], [11] of the paper; the algorithm itself is not
printed in PAPER.md -- reading A22 in DESIGN.md restates the published VEGAS algorithm of Lepage):

  * every integration variable d (here: every uniform draw of an event, a1 of SURVEY.md 8a) has its own grid of
    NB bins with edges 0 = g[d][0] < g[d][1] < ... < g[d][NB] = 1;
  * a uniform y in (0,1) picks bin i = floor(y NB) and the point x = g[i] + (y NB - i) (g[i+1] - g[i]) inside it, so
    every bin is drawn equally often; the Jacobian is dx/dy = NB (g[i+1] - g[i]); the event weight is multiplied by
    the product of the Jacobians of all variables;
  * the grid-optimisation step accumulates, per variable and bin, the sum of the squared event weights
    (h[d][i] = sum w^2 over the events whose variable d fell in bin i);
  * refinement: h is smoothed over neighbouring bins ((h[i-1] + h[i] + h[i+1]) / 3, two-point at the ends),
    normalised, compressed with r = ((1 - h) / ln(1 / h)) ** alpha, and the new edges are placed so that every new
    bin holds the same amount sum(r) / NB, assuming r is spread evenly inside an old bin.

The fixed point equalises the contribution of every bin to the variance: bin widths ~ 1 / |f| for a one-dimensional
integrand (pinned in tests/test_oracle_vegas.py against the analytic optimal grid).
"""
import math

import numpy as np

X_MAX = 1.0 - 2.0 ** -53      # mapped points stay strictly inside (0, 1): RAMBO takes log x


def uniform_grid(ndim, nb):
    return np.tile(np.linspace(0.0, 1.0, nb + 1), (ndim, 1))


def apply_grid(grid, y):
    """y [N, ndim] uniforms -> x [N, ndim] mapped points, jac [N] product of the Jacobians, bins [N, ndim]."""
    ndim, nb1 = grid.shape
    nb = nb1 - 1
    x = np.empty_like(y)
    jac = np.ones(y.shape[0])
    bins = np.empty(y.shape, dtype=np.int64)
    for d in range(ndim):
        t = y[:, d] * nb
        i = np.minimum(t.astype(np.int64), nb - 1)
        lo = grid[d][i]
        w = grid[d][i + 1] - lo
        x[:, d] = np.minimum(lo + (t - i) * w, X_MAX)
        jac *= nb * w
        bins[:, d] = i
    return x, jac, bins


def accumulate(bins, w, nb):
    """h[d][i] = sum of w^2 over the events with bins[:, d] == i."""
    n, ndim = bins.shape
    h = np.zeros((ndim, nb))
    w2 = w * w
    for d in range(ndim):
        h[d] = np.bincount(bins[:, d], weights=w2, minlength=nb)
    return h


def refine(grid, h, alpha=1.5):
    """One refinement of every variable's grid from the accumulated h (module docstring)."""
    ndim, nb1 = grid.shape
    nb = nb1 - 1
    new = grid.copy()
    for d in range(ndim):
        hd = h[d]
        if not np.all(np.isfinite(hd)) or hd.sum() <= 0.0:
            continue
        s = np.empty(nb)
        s[0] = (hd[0] + hd[1]) / 2.0
        s[-1] = (hd[-2] + hd[-1]) / 2.0
        s[1:-1] = (hd[:-2] + hd[1:-1] + hd[2:]) / 3.0
        s = s / s.sum()
        r = np.zeros(nb)
        for i in range(nb):
            if s[i] > 0.0:
                # ((1 - s) / ln(1 / s)) ** alpha; s = 1 (everything in one bin) has the limit 1
                r[i] = 1.0 if s[i] >= 1.0 else ((1.0 - s[i]) / math.log(1.0 / s[i])) ** alpha
        per = r.sum() / nb
        if per <= 0.0:
            continue
        edges = np.empty(nb + 1)
        edges[0], edges[nb] = 0.0, 1.0
        k = 0           # old bin being consumed
        acc = 0.0       # amount of r taken from bins before k
        for j in range(1, nb):
            target = j * per
            while k < nb - 1 and acc + r[k] < target:
                acc += r[k]
                k += 1
            frac = (target - acc) / r[k] if r[k] > 0.0 else 0.0
            frac = min(max(frac, 0.0), 1.0)
            edges[j] = grid[d][k] + frac * (grid[d][k + 1] - grid[d][k])
        # edges must increase strictly (a bin of zero width would give a zero Jacobian)
        for j in range(1, nb + 1):
            if edges[j] <= edges[j - 1]:
                edges[j] = np.nextafter(edges[j - 1], 2.0)
        edges[nb] = 1.0
        new[d] = edges
    return new
