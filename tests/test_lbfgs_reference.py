"""Pins for oracle/lbfgs.py, the fp64 reference of the L-BFGS back-end of the optimizer driver (f4(i); PAPER.md:L605,
reading R19 of DESIGN.md).  The paper names the solver (L-BFGS, Liu & Nocedal 1989) and how the box is handled (sigmoid
reparameterisation) and gives no trajectory, so what is pinned is what the mathematics fixes: the minimiser of a strictly
convex quadratic inside the box is its closed form; the iterates never leave the box and the objective never
increases; a minimum beyond the box is approached at the bound; on a textbook non-convex function and on the spectral
likelihood itself the minimum is the one scipy's independent implementations find."""
import numpy as np

import gen
import oracle
from oracle.lbfgs import lbfgs


def _quadratic(n, seed, lo_t, hi_t):
    g = gen.rng_for("misc", seed)
    Q = g.normal(size=(n, n))
    C = Q @ Q.T / n + np.diag(0.5 + g.random(n))           # symmetric positive definite, not diagonal
    t = g.uniform(lo_t, hi_t, n)

    def fun(x, want_grad):
        r = x - t
        return 0.5 * float(r @ C @ r), (C @ r if want_grad else None)
    return fun, C, t


def test_quadratic_inside_the_box_reaches_the_closed_form():
    fun, C, t = _quadratic(12, 90, 0.25, 0.75)
    tr = []
    x, L = lbfgs(fun, np.full(12, 0.5), np.zeros(12), np.ones(12), iters=80, trace=tr)
    assert np.max(np.abs(x - t)) < 1e-7 and L < 1e-13, (np.max(np.abs(x - t)), L)
    assert all(b <= a for a, b in zip(tr, tr[1:]))          # Armijo: never increases
    # a start on a bound is moved inside, not stuck (sigma' = 0 at the bound itself)
    x0 = np.full(12, 0.5)
    x0[0], x0[1] = 0.0, 1.0
    x2, _ = lbfgs(fun, x0, np.zeros(12), np.ones(12), iters=120)
    assert np.max(np.abs(x2 - t)) < 1e-6


def test_minimum_beyond_the_box_is_approached_at_the_bound():
    fun, C, t = _quadratic(8, 91, 0.3, 0.7)
    C[:] = np.diag(np.diag(C))                               # separable: the constrained minimiser is clip(t)
    t[0], t[1] = 1.6, -0.5
    x, L = lbfgs(fun, np.full(8, 0.5), np.zeros(8), np.ones(8), iters=200)
    assert np.all(x >= 0.0) and np.all(x <= 1.0)             # the sigmoid keeps the iterate in the box (it saturates to
                                                             # the bound itself in floating point)
    assert x[0] > 1.0 - 2e-3 and x[1] < 2e-3
    assert np.max(np.abs(x[2:] - t[2:])) < 1e-4


def test_history_one_and_history_many_find_the_same_minimum():
    fun, C, t = _quadratic(10, 92, 0.3, 0.7)
    for h in (1, 3, 20):
        x, L = lbfgs(fun, np.full(10, 0.5), np.zeros(10), np.ones(10), iters=300, history=h)
        assert np.max(np.abs(x - t)) < 1e-6, h


def test_rosenbrock_agrees_with_scipy_bfgs():
    from scipy.optimize import minimize, rosen, rosen_der

    def fun(x, want_grad):
        return float(rosen(x)), (rosen_der(x) if want_grad else None)
    lo, hi = np.full(4, -3.0), np.full(4, 3.0)
    x, L = lbfgs(fun, np.array([-1.2, 1.0, -1.2, 1.0]), lo, hi, iters=400)
    ref = minimize(rosen, np.array([-1.2, 1.0, -1.2, 1.0]), jac=rosen_der, method="BFGS", options={"gtol": 1e-10})
    assert np.max(np.abs(x - ref.x)) < 1e-5 and np.max(np.abs(x - 1.0)) < 1e-5 and L < 1e-10, (x, ref.x, L)


def test_spectral_likelihood_minimum_is_the_one_scipy_finds():
    # noisy nside-8 sky, the standard bounds (no bound active at the minimum): the same minimum as scipy's L-BFGS-B
    from scipy.optimize import minimize
    w = gen.make_config(0, nside=8, K=(6, 2, 3), cluster_truth=True)
    model, K = oracle.Model(w.freqs), w.K_of_cfg(0)
    d, idx = w.data()[0], w.maps[w.cfg_maps[0]]

    def fun(x, want_grad):
        r = oracle.nll_grad(model, d, w.ninv, idx, K, x, want_grad=want_grad)
        return r["nll"][0], r["grad"]
    lo = np.concatenate([np.full(K[0], 0.5), np.full(K[1], 8.0), np.full(K[2], -5.0)])
    hi = np.concatenate([np.full(K[0], 3.0), np.full(K[1], 40.0), np.full(K[2], -1.0)])
    tr = []
    x, L = lbfgs(fun, w.params_const(), lo, hi, iters=150, trace=tr)
    assert all(b <= a for a, b in zip(tr, tr[1:]))
    res = minimize(lambda z: fun(z, True), w.params_const(), jac=True, method="L-BFGS-B", bounds=list(zip(lo, hi)),
                   options={"maxiter": 2000, "ftol": 1e-15, "gtol": 1e-10, "maxcor": 20})
    assert not ((res.x <= lo) | (res.x >= hi)).any()
    dd = d.astype(np.float64)
    half_dNd = 0.5 * float(np.einsum("f,fsp,fsp->", w.ninv.astype(np.float64), dd, dd))
    m, m_ref = L + half_dNd, res.fun + half_dNd
    assert abs(m - m_ref) <= 1e-9 * m_ref, (m, m_ref)
    assert np.max(np.abs(x - res.x) / (hi - lo)) < 1e-5, np.max(np.abs(x - res.x) / (hi - lo))
