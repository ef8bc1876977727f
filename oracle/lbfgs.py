"""CPU fp64 reference of the fixed-budget L-BFGS back-end of the optimizer driver (f4(i); "Unified
minimize() interface supporting multiple solvers (L-BFGS, AdaTopK, SciPy back-ends), box constraints via sigmoid
reparameterisation").  TEST INFRASTRUCTURE ONLY (same rules as cs_oracle.c and adatopk.py): it follows the textbook
algorithm step by step -- two-loop recursion (Liu & Nocedal 1989, cited L247; Nocedal & Wright, Numerical Optimization,
Alg. 7.4) inside the limited-memory loop (Alg. 7.5) -- and calls the oracle likelihood for every objective / gradient
evaluation.  The paper names the solver and the reparameterisation and nothing else; reading R19 of DESIGN.md:

  box constraints   x = l + (u - l) sigma(z), sigma(z) = 1 / (1 + exp(-z)) = (1 + tanh(z/2)) / 2; the iteration runs in the unconstrained z;
                    a start on (or beyond) a bound is moved to y = clip((x - l)/(u - l), ymin, 1 - ymin), ymin = 1e-6
  gradient          dL/dz = dL/dx (u - l) y (1 - y),  y = sigma(z)
  direction         d = -H g by the two-loop recursion over the last `history` pairs (s, yv) = (z+ - z, g+ - g) with
                    H0 = gamma I, gamma = s.yv / yv.yv of the newest pair; no pair yet: d = -g / |g| (a unit step in z)
  pair update       skipped when s.yv <= curv_eps |s| |yv| (keeps H positive definite); a direction with g.d >= 0
                    (possible only through rounding) is replaced by -g / |g| and the history dropped
  line search       backtracking from alpha = 1, halving, at most ls_max trials, Armijo test
                    L(z + alpha d) <= L + c1 alpha g.d + ls_noise |L|; no trial accepted: no move, history dropped
  budget            a fixed number of iterations, no convergence test (as the AdaTopK driver)
"""
import numpy as np


def _sigmoid(z):
    return 0.5 * (1.0 + np.tanh(0.5 * z))                          # = 1 / (1 + exp(-z)), without overflow for large |z|


def lbfgs(fun, x0, lower, upper, iters=100, history=10, ls_c1=1e-4, ls_max=8, ls_noise=0.0, curv_eps=1e-10, ymin=1e-6,
          trace=None):
    """fun(x, want_grad) -> (L, g or None).  Returns (x, L(x)).  trace, if given, receives L after every iteration."""
    lo, hi = np.asarray(lower, float), np.asarray(upper, float)
    span = hi - lo
    y = np.clip((np.asarray(x0, float) - lo) / span, ymin, 1.0 - ymin)
    z = np.log(y) - np.log1p(-y)                                  # logit
    S, Y = [], []                                                  # newest last
    L, gx = fun(lo + span * _sigmoid(z), True)
    yy = _sigmoid(z)
    g = gx * span * yy * (1.0 - yy)
    for _ in range(iters):
        # two-loop recursion (Nocedal & Wright Alg. 7.4)
        q = g.copy()
        al = []
        for s, yv in zip(reversed(S), reversed(Y)):
            a = float(np.dot(s, q)) / float(np.dot(s, yv))
            al.append(a)
            q -= a * yv
        if S:
            q *= float(np.dot(S[-1], Y[-1])) / float(np.dot(Y[-1], Y[-1]))
        for (s, yv), a in zip(zip(S, Y), reversed(al)):
            b = float(np.dot(yv, q)) / float(np.dot(s, yv))
            q += s * (a - b)
        d = -q
        gd = float(np.dot(g, d))
        nrm = float(np.linalg.norm(g))
        if not S or not gd < 0.0:
            S, Y = [], []
            d = -g / nrm if nrm > 0 else np.zeros_like(g)
            gd = -nrm
        # backtracking line search
        alpha, acc = 1.0, 0.0
        for _ls in range(ls_max):
            Lt, _g = fun(lo + span * _sigmoid(z + alpha * d), False)
            if Lt <= L + ls_c1 * alpha * gd + ls_noise * abs(L):
                acc = alpha
                break
            alpha *= 0.5
        if acc > 0.0:
            z_new = z + acc * d
            L_new, gx = fun(lo + span * _sigmoid(z_new), True)
            yy = _sigmoid(z_new)
            g_new = gx * span * yy * (1.0 - yy)
            s, yv = z_new - z, g_new - g
            sy = float(np.dot(s, yv))
            if sy > curv_eps * float(np.linalg.norm(s)) * float(np.linalg.norm(yv)):
                S.append(s); Y.append(yv)
                if len(S) > history:
                    S.pop(0); Y.pop(0)
            z, g, L = z_new, g_new, L_new
        else:
            S, Y = [], []
        if trace is not None:
            trace.append(L)
    x = lo + span * _sigmoid(z)
    return x, fun(x, False)[0]
