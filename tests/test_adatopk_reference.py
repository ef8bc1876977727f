"""Pins for oracle/adatopk.py, the fp64 reference of the fixed-budget AdaTopK driver (a5; App. A, Alg. 1,
readings R13/R14 of DESIGN.md).  The paper publishes neither hyper-parameters nor a worked trajectory, so what is
pinned is what it states about the algorithm: iterates stay inside the bounds, every accepted step decreases the
objective (L263), a bound that the gradient pushes away from is released (L519-L525), a bound that the minimum lies
beyond stays active, and on a sky whose optimum is known by construction (L287) the truth is recovered."""
import numpy as np

import gen
import oracle
from oracle.adatopk import adatopk


def test_quadratic_with_active_bounds():
    # f(x) = 1/2 sum c_i (x_i - t_i)^2 on [0,1]^n with some targets outside the box: the minimiser is clip(t, 0, 1)
    g = gen.rng_for("misc", 77)
    n = 12
    c = 1.0 + 9.0 * g.random(n)
    t = g.uniform(-0.5, 1.5, n)
    t[0], t[1] = 1.7, -0.4                       # beyond the upper / lower bound

    def fun(x, want_grad):
        return 0.5 * float(np.sum(c * (x - t) ** 2)), (c * (x - t) if want_grad else None)
    hist = []
    x0 = np.full(n, 0.5)
    x0[2] = 0.0                                  # starts ON the lower bound although its target is inside: must be released
    t[2] = 0.6
    x, L = adatopk(fun, x0, np.zeros(n), np.ones(n), iters=600, lr=0.05, history=hist)
    assert np.all(x >= 0.0) and np.all(x <= 1.0)
    assert all(b <= a for a, b in zip(hist, hist[1:]))
    assert x[0] == 1.0 and x[1] == 0.0           # pinned exactly at the bound
    assert np.max(np.abs(x - np.clip(t, 0.0, 1.0))) < 2e-3
    assert L <= fun(np.clip(t, 0, 1), False)[0] + 1e-4


def test_rescale_keeps_the_trajectory_scale_invariant():
    # A4 (L541-L546): objectives scaled out of [1e-15, 1e15] are rescaled; the iterates must not depend on the scale
    def make(scale):
        def fun(x, want_grad):
            return scale * float(np.sum((x - 0.3) ** 2)), (scale * 2 * (x - 0.3) if want_grad else None)
        return fun
    xs = [adatopk(make(s), np.full(4, 0.9), np.zeros(4), np.ones(4), iters=50)[0] for s in (1.0, 1e20, 1e-20)]
    assert np.allclose(xs[0], xs[1], rtol=0, atol=1e-9) and np.allclose(xs[0], xs[2], rtol=0, atol=1e-9)


def test_recovers_known_optimum_on_noiseless_cluster_constant_sky():
    w = gen.make_config(0, nside=8, K=(6, 2, 3), noiseless=True, cluster_truth=True)
    model, K = oracle.Model(w.freqs), w.K_of_cfg(0)
    d, idx = w.data()[0], w.maps[w.cfg_maps[0]]

    def fun(x, want_grad):
        r = oracle.nll_grad(model, d, w.ninv, idx, K, x, want_grad=want_grad)
        return r["nll"][0], r["grad"]
    lo = np.concatenate([np.full(K[0], 0.5), np.full(K[1], 8.0), np.full(K[2], -5.0)])
    hi = np.concatenate([np.full(K[0], 3.0), np.full(K[1], 40.0), np.full(K[2], -1.0)])
    hist = []
    x, L = adatopk(fun, w.params_const(), lo, hi, iters=300, history=hist)
    truth = np.concatenate(w.truth["per_cluster"])
    assert np.all(x >= lo) and np.all(x <= hi)
    assert all(b <= a for a, b in zip(hist, hist[1:]))
    err = np.abs(x - truth)
    assert err[:K[0]].max() < 5e-3 and err[K[0]:K[0] + K[1]].max() < 0.2 and err[K[0] + K[1]:].max() < 5e-3, err
    dd = d.astype(np.float64)
    dNd = float(np.einsum("f,fsp,fsp->", w.ninv.astype(np.float64), dd, dd))
    assert L + 0.5 * dNd < 1e-3 * abs(hist[0] + 0.5 * dNd)      # misfit reduced by > 1000x towards the noiseless optimum 0


def test_reaches_the_bounded_minimum_an_independent_solver_finds():
    # The result of a5 is the bound-constrained minimiser of the spectral likelihood: scipy's L-BFGS-B (an independent
    # implementation of bounded minimisation, run to convergence on the same oracle objective) must find the same
    # minimum, on a noisy sky with tight bounds so that several parameters end pinned ("reaches the same
    # minimum as scipy L-BFGS-B").
    from scipy.optimize import minimize
    w = gen.make_config(0, nside=8, K=(6, 2, 3), cluster_truth=True)
    model, K = oracle.Model(w.freqs), w.K_of_cfg(0)
    d, idx = w.data()[0], w.maps[w.cfg_maps[0]]

    def fun(x, want_grad):
        r = oracle.nll_grad(model, d, w.ninv, idx, K, x, want_grad=want_grad)
        return r["nll"][0], r["grad"]
    lo = np.concatenate([np.full(K[0], 1.50), np.full(K[1], 8.0), np.full(K[2], -5.0)])
    hi = np.concatenate([np.full(K[0], 1.56), np.full(K[1], 40.0), np.full(K[2], -2.95)])   # tight: some minima lie beyond
    x, L = adatopk(fun, np.clip(w.params_const(), lo, hi), lo, hi, iters=600)
    res = minimize(lambda z: fun(z, True), np.clip(w.params_const(), lo, hi), jac=True, method="L-BFGS-B",
                   bounds=list(zip(lo, hi)), options={"maxiter": 2000, "ftol": 1e-15, "gtol": 1e-10, "maxcor": 20})
    dd = d.astype(np.float64)
    half_dNd = 0.5 * float(np.einsum("f,fsp,fsp->", w.ninv.astype(np.float64), dd, dd))
    m_ada, m_ref = L + half_dNd, res.fun + half_dNd          # misfits 1/2 chi^2: the part that depends on the parameters
    assert abs(m_ada - m_ref) <= 1e-9 * m_ref, (m_ada, m_ref)            # measured 1.6e-12
    at_bound_ref = (res.x <= lo) | (res.x >= hi)
    assert at_bound_ref.any()                                 # the test is about active bounds
    assert np.array_equal((x <= lo) | (x >= hi), at_bound_ref)
    free = ~at_bound_ref
    assert np.max(np.abs(x - res.x)[free] / (hi - lo)[free]) < 1e-5   # measured 2e-8


def _box_problem(n=40, seed=78):
    """Separable quadratic on [0,1]^n whose targets are all inside the box, started with every parameter ON a bound."""
    g = gen.rng_for("misc", seed)
    c = 1.0 + 9.0 * g.random(n)
    t = g.uniform(0.2, 0.8, n)

    def fun(x, want_grad):
        return 0.5 * float(np.sum(c * (x - t) ** 2)), (c * (x - t) if want_grad else None)
    x0 = np.where(np.arange(n) % 2 == 0, 0.0, 1.0)
    return fun, x0, t


def test_topk_zero_releases_exactly_one_bound_per_iteration():
    # A3 (L535): "K=0 (single-parameter release per iteration, matching the classical TNC strategy)"
    fun, x0, t = _box_problem()
    rel = []
    adatopk(fun, x0, np.zeros_like(x0), np.ones_like(x0), iters=25, released=rel)
    assert rel == [1] * 25


def test_topk_one_releases_every_bound_pushed_inwards_at_once():
    # A3 (L531): "K=1.0 (all constraints released simultaneously)"; every start value sits on the wrong side of its target
    fun, x0, t = _box_problem()
    rel = []
    x, L = adatopk(fun, x0, np.zeros_like(x0), np.ones_like(x0), iters=400, lr=0.05, topk=1.0, released=rel)
    assert rel[0] == len(x0) and sum(rel[1:]) == 0
    assert np.max(np.abs(x - t)) < 5e-3


def test_topk_fraction_releases_floor_of_the_fraction_of_the_bound_set():
    # n = max(1, floor(topk * n_bound)); the bound set shrinks as parameters are released
    fun, x0, t = _box_problem(n=40)
    rel = []
    adatopk(fun, x0, np.zeros_like(x0), np.ones_like(x0), iters=6, topk=0.25, released=rel)
    nb, want = 40, []
    for _ in range(6):
        n = max(1, int(np.floor(0.25 * nb)))
        want.append(n)
        nb -= n
    assert rel == want                                   # 10, 7, 5, 4, 3, 2
    # and the released ones are those with the largest scores: after one iteration the 10 largest c_i |x0_i - t_i| are free
    hist = []
    x1, _ = adatopk(fun, x0, np.zeros_like(x0), np.ones_like(x0), iters=1, topk=0.25, history=hist)
    moved = np.flatnonzero(x1 != x0)
    c_t = np.abs(fun(x0, True)[1])
    assert set(moved.tolist()) == set(np.argsort(c_t)[::-1][:10].tolist())


def test_topk_keeps_bounds_and_monotonicity():
    fun, x0, t = _box_problem(n=30, seed=79)
    t[:5] = [1.4, -0.3, 1.2, -0.1, 1.6]                  # minima beyond the box: those parameters must stay / end pinned
    for topk in (0.0, 0.3, 1.0):
        hist = []
        x, L = adatopk(fun, x0, np.zeros_like(x0), np.ones_like(x0), iters=500, lr=0.05, topk=topk, history=hist)
        assert np.all(x >= 0.0) and np.all(x <= 1.0)
        assert all(b <= a for a, b in zip(hist, hist[1:]))
        assert np.max(np.abs(x - np.clip(t, 0, 1))) < 5e-3, topk
