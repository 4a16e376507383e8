"""Pins of the adaptive grid (oracle/vegas.py, reading A22): mapping, Jacobian, accumulation and the refinement's
fixed point on a one-dimensional analytic integrand."""
import math

import numpy as np

from oracle import phase_space as ops
from oracle import philox
from oracle import sm
from oracle import vegas


def test_map_is_a_change_of_variables():
    """For any grid, E_y[f(x(y)) J(y)] = int_0^1 f(x) dx: checked with f = x^3 (exact value 1/4) on a grid with very
    unequal bins, by a midpoint rule in y fine enough to resolve every bin."""
    edges = np.concatenate([[0.0], np.sort(np.random.default_rng(1).uniform(0, 1, 9)), [1.0]])
    grid = np.array([edges])
    n = 200000
    y = ((np.arange(n) + 0.5) / n)[:, None]
    x, jac, bins = vegas.apply_grid(grid, y)
    assert abs(np.mean(x[:, 0] ** 3 * jac) - 0.25) < 1e-9
    assert abs(np.mean(jac) - 1.0) < 1e-12                       # f = 1
    assert np.array_equal(np.bincount(bins[:, 0], minlength=10), np.full(10, n // 10))   # every bin equally often
    assert x.min() > 0 and x.max() < 1
    # the point lies in the bin it reports
    assert np.all(x[:, 0] >= edges[bins[:, 0]]) and np.all(x[:, 0] <= edges[bins[:, 0] + 1])


def test_refinement_converges_to_the_analytic_optimum():
    """f(x) = 1 / (x + a) on (0, 1): the variance-optimal grid has equal int_bin |f| dx in every bin, i.e. edges
    x_i = a ((1 + 1/a)^(i/NB) - 1).  Iterating accumulate -> refine (alpha = 1: no damping towards... the compression
    exponent only sets the speed) from a uniform grid must approach these edges, and the Monte-Carlo variance must
    drop by the factor the optimum predicts."""
    a, nb, n = 0.01, 32, 200000
    f = lambda x: 1.0 / (x + a)
    exact = math.log(1.0 + 1.0 / a)
    grid = vegas.uniform_grid(1, nb)
    var = []
    for it in range(12):
        y = philox.uniforms(3, it * n, n, 1, 99)
        x, jac, bins = vegas.apply_grid(grid, y)
        w = f(x[:, 0]) * jac
        var.append(w.var())
        est, err = w.mean(), w.std() / math.sqrt(n)
        assert abs(est - exact) < 5 * err
        grid = vegas.refine(grid, vegas.accumulate(bins, w, nb), alpha=1.0)
    optimum = a * ((1.0 + 1.0 / a) ** (np.arange(nb + 1) / nb) - 1.0)
    assert np.abs(grid[0] - optimum).max() < 0.02                     # edges (in x)
    assert np.abs(np.log((grid[0][1:] + a) / (optimum[1:] + a))).max() < 0.15    # ... and on the scale that matters
    # flat sampling: var = int f^2 - I^2; on the optimal grid f J is constant up to the variation inside a bin
    var_flat = (1.0 / a - 1.0 / (1.0 + a)) - exact ** 2
    assert abs(var[0] / var_flat - 1) < 0.05
    assert var[-1] < var_flat / 500


def test_accumulate_and_degenerate_input():
    bins = np.array([[0, 1], [0, 0], [2, 1]])
    w = np.array([1.0, 2.0, 3.0])
    h = vegas.accumulate(bins, w, 3)
    assert np.array_equal(h, [[5.0, 0.0, 9.0], [4.0, 10.0, 0.0]])
    g = vegas.uniform_grid(2, 3)
    assert np.array_equal(vegas.refine(g, np.zeros((2, 3))), g)         # nothing accumulated: grid unchanged
    g2 = vegas.refine(g, h)
    assert np.all(np.diff(g2, axis=1) > 0) and np.all(g2[:, 0] == 0) and np.all(g2[:, -1] == 1)


def test_generate_with_grid_is_generate_on_mapped_uniforms():
    par = sm.default_params()
    cfg, n, rs = 5, 200, 2000.0
    rng = np.random.default_rng(5)
    grid = np.sort(np.concatenate([np.zeros((20, 1)), rng.uniform(0, 1, (20, 7)), np.ones((20, 1))], 1), 1)
    p, w, bins = ops.generate(cfg, 11, 0, n, rs, par, grid=grid, with_bins=True)
    u = philox.uniforms(11, 0, n, 20, cfg)
    x, jac, b2 = vegas.apply_grid(grid, u)
    p2, w2 = ops.from_uniforms(cfg, x, rs, par)
    assert np.array_equal(p, p2) and np.array_equal(w, w2 * jac) and np.array_equal(bins, b2)
    # the flat grid changes nothing
    p3, w3 = ops.generate(cfg, 11, 0, n, rs, par, grid=vegas.uniform_grid(20, 8))
    p0, w0 = ops.generate(cfg, 11, 0, n, rs, par)
    assert np.allclose(p3, p0, rtol=0, atol=1e-9) and np.allclose(w3, w0, rtol=1e-13)
