"""CPU fp64 reference of the fixed-budget AdaTopK driver (App. A, Alg. 1) with the readings R13/R14
of DESIGN.md.  TEST INFRASTRUCTURE ONLY (same rules as cs_oracle.c): it follows Alg. 1 step by step in the paper's
order and calls the oracle likelihood for every objective / gradient evaluation.  Parity with the paper's own
AdaTopK is unpinned (its hyper-parameters are not published); what is pinned in tests is that this reading never
leaves the bounds, never increases the objective and recovers a known optimum.

Top-K release (A2-A3, L519-L537): `topk` is the paper's "Top-K fraction K" in [0, 1].  Per iteration the
n = max(1, floor(topk * n_bound)) bound parameters with the highest positive release scores are released together
(n_bound = parameters currently pinned at a bound); topk = 0 releases one per iteration (the paper's production
setting, L535), topk = 1 every bound parameter whose score is positive (L531).  Scores equal to the n-th highest are
released with it.  (Reading R18 of DESIGN.md: the paper gives the range of K and its two end points, not the rounding.)

Armijo test (L263 "every accepted step decreases the objective"): the sufficient-decrease term uses min(g.d, 0), so
that a momentum direction with g.d >= 0 can never license an increase.
"""
import numpy as np


def adatopk(fun, x0, lower, upper, iters=200, lr=0.02, beta1=0.9, beta2=0.999, eps=1e-16, ls_c1=1e-4, ls_max=8,
            safe_lo=1e-15, safe_hi=1e15, ls_noise=0.0, history=None, topk=0.0, released=None):
    """fun(x, want_grad) -> (L, g or None).  Returns (x, L(x))."""
    lo, hi = np.asarray(lower, float), np.asarray(upper, float)
    span = hi - lo
    y = np.clip((np.asarray(x0, float) - lo) / span, 0.0, 1.0)          # A1 (L509-L513): y = (x - l)/(u - l)
    piv = np.where(y <= 0.0, -1, np.where(y >= 1.0, 1, 0))               # p in {-1, 0, +1} (L519)
    m = np.zeros_like(y)
    v = np.zeros_like(y)
    cs = 1.0                                                             # cumulative objective scale (A4)
    for it in range(iters):
        L, g = fun(lo + y * span, True)
        L *= cs
        gint = cs * g * span                                             # g_int = g * s (L513, Alg. 1 line 3)
        # A2 (L519-L525): release the n bound parameters pushed hardest into the feasible region; K = 0 -> n = 1 (L249, L535)
        score = np.where(piv < 0, -gint, np.where(piv > 0, gint, 0.0))
        nrel = 0
        if (score > 0).any():
            n = max(1, int(np.floor(topk * np.count_nonzero(piv))))
            pos = np.sort(score[score > 0])[::-1]
            thr = pos[min(n, len(pos)) - 1]
            rel = score >= thr
            if n == 1:                                                   # ties at the top: the lowest index only
                rel = np.zeros_like(rel)
                rel[int(np.argmax(score))] = True
            nrel = int(np.count_nonzero(rel))
            piv[rel] = 0
        if released is not None:
            released.append(nrel)
        free = piv == 0
        gp = np.where(free, gint, 0.0)                                   # projected gradient (line 8)
        nrm = float(np.linalg.norm(gp))
        f = 1.0 / nrm if nrm > 0 and (nrm < safe_lo or nrm > safe_hi) else 1.0   # A4 (L541-L546)
        cs *= f; L *= f; gp = gp * f; m *= f; v *= f * f
        # AdaBelief direction (Zhuang et al. 2020), masked by the active set (lines 14-16)
        m = beta1 * m + (1 - beta1) * gp
        v = beta2 * v + (1 - beta2) * (gp - m) ** 2 + eps
        t = it + 1
        d = np.where(free, -lr * (m / (1 - beta1 ** t)) / (np.sqrt(v / (1 - beta2 ** t)) + eps), 0.0)
        gd = float(np.dot(gp, d))
        with np.errstate(divide="ignore", invalid="ignore"):
            a = np.where(d > 0, (1 - y) / d, np.where(d < 0, y / (-d), np.inf))   # distance to the nearest bound (line 17)
        il = int(np.argmin(a))
        amax = float(a[il])
        alpha, acc = min(1.0, amax), 0.0
        for _ in range(ls_max):                                          # backtracking (line 18, L263)
            Lt, _ = fun(lo + np.clip(y + alpha * d, 0, 1) * span, False)
            if Lt * cs <= L + ls_c1 * alpha * min(gd, 0.0) + ls_noise * abs(L):
                acc = alpha
                break
            alpha *= 0.5
        if acc > 0:                                                      # lines 19-25
            y = np.clip(y + acc * d, 0, 1)
            if acc == amax:
                y[il] = 1.0 if d[il] > 0 else 0.0
                piv[il] = 1 if d[il] > 0 else -1
            hit = free & ((y <= 0) | (y >= 1))
            piv[hit & (y <= 0)] = -1
            piv[hit & (y >= 1)] = 1
        if history is not None:
            history.append(L / cs)
    x = lo + y * span
    return x, fun(x, False)[0]
