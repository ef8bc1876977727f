"""Pins for the CPU fp64 oracle against what the paper and the mathematics fix.

Nothing here compares the oracle with itself through the same formula: every check is a closed form, an
invariant, a special case that reduces to a textbook identity, a finite difference, a statistical law or a
brute-force search.  Data come from gen/ (an independent numpy forward model), never from the CUDA path.
"""
import numpy as np
import pytest

import gen
import oracle

H_OVER_K = 6.62607015e-34 / 1.380649e-23 * 1e9      # K / GHz, exact SI (R3)


@pytest.fixture(scope="module")
def model():
    return oracle.Model(gen.BANDS_GHZ)


@pytest.fixture(scope="module")
def model_lit():
    return oracle.Model(gen.BANDS_GHZ, units=oracle.UNITS_LITERAL)


@pytest.fixture(scope="module")
def c1():
    return gen.make_config(0)


def _entry(w, e=0):
    c = int(w.cfg_of[e])
    return w.data()[int(w.data_of[e])], w.maps[w.cfg_maps[c]], w.K_of_cfg(c)


# ----------------------------------------------------------------------------- SED (Eq. 2, R1-R3)

def test_sed_unity_at_reference_frequency(model, model_lit):
    # "both normalized to unity at the reference frequency nu0"
    for m in (model, model_lit):
        for bd, Td, bs in ((1.54, 20.0, -3.0), (0.5, 8.0, -5.0), (3.0, 40.0, -1.0)):
            assert oracle.sed_dust(m, 353.0, bd, Td) == 1.0
            assert oracle.sed_sync(m, 23.0, bs) == 1.0


def test_sed_dust_is_modified_blackbody_in_RJ_units(model_lit):
    # MBB: I_nu ~ nu^beta B_nu(T), B_nu ~ nu^3/(e^x-1); brightness temperature ~ I_nu/nu^2 (textbook)
    for nu in gen.BANDS_GHZ:
        for bd, Td in ((1.54, 20.0), (2.2, 11.0)):
            B = lambda v: v ** 3 / np.expm1(H_OVER_K * v / Td)
            ref = (nu / 353.0) ** bd * B(nu) / B(353.0) * (353.0 / nu) ** 2
            assert abs(oracle.sed_dust(model_lit, nu, bd, Td) / ref - 1) < 1e-13


def test_sed_rayleigh_jeans_limit(model_lit):
    # T_d -> infinity: Planck ratio -> nu0/nu, so a_d -> (nu/nu0)^beta_d  (R1 pin)
    for nu in gen.BANDS_GHZ:
        a = oracle.sed_dust(model_lit, nu, 1.54, 1e9)
        assert abs(a / (nu / 353.0) ** 1.54 - 1) < 1e-7


def test_sed_sync_power_law(model_lit):
    for nu in gen.BANDS_GHZ:
        assert abs(oracle.sed_sync(model_lit, nu, -3.1) / (nu / 23.0) ** -3.1 - 1) < 1e-14


def test_units_factor(model, model_lit):
    # K_RJ -> K_CMB: u = (e^x-1)^2/(x^2 e^x) = (2 sinh(x/2)/x)^2 -> 1 for x -> 0   (R2)
    for nu in list(gen.BANDS_GHZ) + [23.0, 353.0]:
        x = H_OVER_K * nu / 2.7255
        assert abs(oracle.krj2kcmb(nu) / (2 * np.sinh(x / 2) / x) ** 2 - 1) < 1e-13
    assert abs(oracle.krj2kcmb(1e-3) - 1) < 1e-9
    for nu in gen.BANDS_GHZ:
        r_d = oracle.sed_dust(model, nu, 1.5, 21.0) / oracle.sed_dust(model_lit, nu, 1.5, 21.0)
        r_s = oracle.sed_sync(model, nu, -2.9) / oracle.sed_sync(model_lit, nu, -2.9)
        assert abs(r_d / (oracle.krj2kcmb(nu) / oracle.krj2kcmb(353.0)) - 1) < 1e-13
        assert abs(r_s / (oracle.krj2kcmb(nu) / oracle.krj2kcmb(23.0)) - 1) < 1e-13


def test_sed_matches_independent_forward_model(model):
    # gen/ holds an independently written numpy forward model; the two must agree
    a_d, a_s = gen.mixing_columns(gen.BANDS_GHZ, 1.61, 18.5, -2.8)
    for f, nu in enumerate(gen.BANDS_GHZ):
        assert abs(oracle.sed_dust(model, nu, 1.61, 18.5) / a_d[f] - 1) < 1e-12
        assert abs(oracle.sed_sync(model, nu, -2.8) / a_s[f] - 1) < 1e-12


def test_sed_derivatives_vs_central_differences(model):
    for nu in gen.BANDS_GHZ:
        bd, Td, bs = 1.6, 19.0, -3.1
        h = 1e-6
        fd = (oracle.sed_dust(model, nu, bd + h, Td) - oracle.sed_dust(model, nu, bd - h, Td)) / (2 * h)
        assert abs(oracle.dsed_dust_dbeta(model, nu, bd, Td) - fd) <= 1e-8 * abs(fd) + 1e-12
        h = 1e-4
        fd = (oracle.sed_dust(model, nu, bd, Td + h) - oracle.sed_dust(model, nu, bd, Td - h)) / (2 * h)
        assert abs(oracle.dsed_dust_dT(model, nu, bd, Td) - fd) <= 1e-7 * abs(fd) + 1e-12
        h = 1e-6
        fd = (oracle.sed_sync(model, nu, bs + h) - oracle.sed_sync(model, nu, bs - h)) / (2 * h)
        assert abs(oracle.dsed_sync_dbeta(model, nu, bs) - fd) <= 1e-8 * abs(fd) + 1e-12
    A, dA = oracle.mixing_matrix(model, 1.6, 19.0, -3.1)
    assert np.all(A[:, 0] == 1.0)                                   # A_cmb = 1
    assert abs(dA[1, :]).max() > 0 and A.shape == (15, 3) and dA.shape == (3, 15)


# ----------------------------------------------------------------------------- solve / maps (Eq. 5, 8, 11)

def test_W_A_is_identity(model):
    # [W A_cmb]_cmb = 1 (Eq. 11); more generally W A = I
    ninv = gen.ninv_f32(64).astype(np.float64)
    A, _ = oracle.mixing_matrix(model, 1.54, 20.0, -3.0)
    for j in range(3):
        r = oracle.pixel(model, ninv, A[:, j], -2.0 * A[:, j], 1.54, 20.0, -3.0)
        e = np.zeros(3); e[j] = 1
        np.testing.assert_allclose(r["s"][:, 0], e, atol=2e-13)
        np.testing.assert_allclose(r["s"][:, 1], -2 * e, atol=4e-13)


def test_normal_equations_and_ll(model):
    rng = np.random.default_rng(0)
    ninv = gen.ninv_f32(64).astype(np.float64)
    dq, du = rng.normal(size=15) * 30, rng.normal(size=15) * 30
    r = oracle.pixel(model, ninv, dq, du, 1.7, 17.0, -2.7)
    A, dA = oracle.mixing_matrix(model, 1.7, 17.0, -2.7)
    for S, d in enumerate((dq, du)):
        res = A.T @ (ninv * (d - A @ r["s"][:, S]))             # dL/ds = 0 (Eq. 4)
        assert np.abs(res).max() < 1e-9 * np.abs(A.T @ (ninv * d)).max()
    # numpy lstsq as the textbook GLS solution
    sw = np.sqrt(ninv)
    for S, d in enumerate((dq, du)):
        ref = np.linalg.lstsq(A * sw[:, None], d * sw, rcond=None)[0]
        np.testing.assert_allclose(r["s"][:, S], ref, rtol=1e-9, atol=1e-11)
    # chi^2 identity: (d-As)^T N^-1 (d-As) = d^T N^-1 d - b^T M^-1 b   =>  ll = -1/2 b.s
    chi2 = sum(np.sum(ninv * (d - A @ r["s"][:, S]) ** 2) for S, d in enumerate((dq, du)))
    dNd = np.sum(ninv * dq ** 2) + np.sum(ninv * du ** 2)
    assert abs((-2 * r["ll"]) - (dNd - chi2)) < 1e-10 * dNd


def test_noiseless_recovery_of_maps_and_optimum():
    # truth constant per cluster, data generated on the same patch grid: the optimum is the truth and the
    # maps equal the inputs ("true optimal configuration is known by construction")
    w = gen.make_config(0, noiseless=True, cluster_truth=True)
    m = oracle.Model(w.freqs)
    d, idx, K = _entry(w)
    ptrue = np.concatenate(w.truth["per_cluster"])
    r = oracle.nll_grad(m, d, w.ninv, idx, K, ptrue, want_maps=True, want_tol=True)
    assert r["rc"] == 0
    s_true = w.truth["s"]
    # d is stored in fp32, so recovery is limited by 6e-8 * |d| * conditioning
    assert np.abs(r["maps"] - s_true).max() < 2e-4 * np.abs(s_true).max()
    dNd = np.sum(w.ninv.astype(np.float64)[:, None, None] * d.astype(np.float64) ** 2)
    assert abs(r["nll"][0] + 0.5 * dNd) < 1e-9 * dNd               # chi^2 = 0 at the truth
    assert np.all(np.abs(r["grad"]) < 1e-6 * r["gscale"])           # stationary point
    rng = np.random.default_rng(1)
    for _ in range(20):
        pp = ptrue + rng.normal(size=ptrue.size) * np.array([0.02] * K[0] + [0.3] * K[1] + [0.02] * K[2])
        assert oracle.nll_grad(m, d, w.ninv, idx, K, pp, want_grad=False)["nll"][0] > r["nll"][0]


def test_nfreq_equal_ncomp_reduces_to_dNd():
    # with nfreq = ncomp, A is square and b^T M^-1 b = d^T N^-1 d for any parameters (north_star pin)
    w = gen.make_config(0)
    sel = [2, 8, 13]
    m3 = oracle.Model(w.freqs[sel])
    d, idx, K = _entry(w)
    d3, n3 = np.ascontiguousarray(d[sel]), w.ninv[sel]
    dNd = np.sum(n3.astype(np.float64)[:, None, None] * d3.astype(np.float64) ** 2)
    for seed in range(3):
        p = w.params_jittered(seed, 3.0)
        r = oracle.nll_grad(m3, d3, n3, idx, K, p)
        assert abs(r["nll"][0] + 0.5 * dNd) < 1e-10 * dNd
        assert np.abs(r["grad"]).max() < 1e-6 * dNd                 # flat in the parameters


def test_chi2_statistic_with_noise():
    # per-pixel clusters at the truth: 2 nll + d^T N^-1 d = chi^2 with 2 npix (F-3) dof
    ns = 16
    npix = 12 * ns * ns
    truth = gen.draw_truth(npix, 7)
    sigma = gen.noise_sigma(ns)
    d = gen.synthesize(truth, gen.BANDS_GHZ, sigma, (3,))[0]
    ninv = gen.ninv_f32(ns)
    idx = np.tile(np.arange(npix, dtype=np.int32), (3, 1))
    p = np.concatenate([truth["beta_d"], truth["T_d"], truth["beta_s"]])
    m = oracle.Model(gen.BANDS_GHZ)
    r = oracle.nll_grad(m, d, ninv, idx, [npix] * 3, p, want_grad=False)
    dNd = np.sum(ninv.astype(np.float64)[:, None, None] * d.astype(np.float64) ** 2)
    chi2 = 2 * r["nll"][0] + dNd
    dof = 2 * npix * (15 - 3)
    assert abs(chi2 - dof) < 5 * np.sqrt(2 * dof)


def test_ninv_scaling(model, c1):
    d, idx, K = _entry(c1)
    p = c1.params_jittered(2)
    r1 = oracle.nll_grad(model, d, c1.ninv, idx, K, p, want_maps=True)
    r4 = oracle.nll_grad(model, d, c1.ninv * np.float32(4.0), idx, K, p, want_maps=True)
    np.testing.assert_allclose(r4["nll"], 4 * r1["nll"], rtol=1e-13)
    np.testing.assert_allclose(r4["grad"], 4 * r1["grad"], rtol=1e-10, atol=1e-9 * np.abs(r1["grad"]).max())
    np.testing.assert_allclose(r4["maps"], r1["maps"], rtol=1e-10, atol=1e-12)


# ----------------------------------------------------------------------------- gradient (Eq. 17, R4)

def test_gradient_vs_central_differences_every_cluster(model, c1):
    d, idx, K = _entry(c1)
    p = c1.params_jittered(1)
    r = oracle.nll_grad(model, d, c1.ninv, idx, K, p, want_tol=True)
    f = lambda q: oracle.nll_grad(model, d, c1.ninv, idx, K, q, want_grad=False)["nll"][0]
    for k in range(p.size):
        h = 1e-5 * max(1.0, abs(p[k]))
        pp, pm = p.copy(), p.copy()
        pp[k] += h; pm[k] -= h
        fd = (f(pp) - f(pm)) / (2 * h)
        assert abs(fd - r["grad"][k]) <= 2e-6 * abs(fd) + 1e-9 * r["gscale"][k], (k, fd, r["grad"][k])


def test_single_cluster_gradient_is_sum_of_per_pixel_gradients(model, c1):
    d, _, _ = _entry(c1)
    npix = c1.npix
    one = np.zeros((3, npix), dtype=np.int32)
    per = np.tile(np.arange(npix, dtype=np.int32), (3, 1))
    r1 = oracle.nll_grad(model, d, c1.ninv, one, [1, 1, 1], np.array([1.5, 19.0, -3.1]))
    rp = oracle.nll_grad(model, d, c1.ninv, per, [npix] * 3,
                         np.concatenate([np.full(npix, 1.5), np.full(npix, 19.0), np.full(npix, -3.1)]))
    assert abs(r1["nll"][0] - rp["nll"][0]) < 1e-12 * abs(r1["nll"][0])
    for t in range(3):
        tot = rp["grad"][t * npix:(t + 1) * npix].sum()
        assert abs(r1["grad"][t] - tot) < 1e-10 * np.abs(rp["grad"][t * npix:(t + 1) * npix]).sum()


# ----------------------------------------------------------------------------- cluster reduction / indexing

def test_pixel_permutation_and_cluster_relabelling(model, c1):
    d, idx, K = _entry(c1)
    p = c1.params_jittered(3)
    r = oracle.nll_grad(model, d, c1.ninv, idx, K, p, want_maps=True)
    perm = np.random.default_rng(5).permutation(c1.npix)
    rp = oracle.nll_grad(model, np.ascontiguousarray(d[:, :, perm]), c1.ninv, idx[:, perm], K, p, want_maps=True)
    np.testing.assert_allclose(rp["nll"], r["nll"], rtol=1e-13)
    np.testing.assert_allclose(rp["grad"], r["grad"], rtol=1e-11, atol=1e-9)
    np.testing.assert_array_equal(rp["maps"], r["maps"][:, :, perm])
    # relabel beta_d clusters by a permutation sigma: parameters and gradient move with the labels
    sig = np.array([2, 0, 3, 1])
    idx2 = idx.copy(); idx2[0] = sig[idx[0]]
    p2 = p.copy(); p2[sig] = p[:4]
    r2 = oracle.nll_grad(model, d, c1.ninv, idx2, K, p2)
    np.testing.assert_allclose(r2["nll"], r["nll"], rtol=1e-14)
    np.testing.assert_allclose(r2["grad"][sig], r["grad"][:4], rtol=1e-13)
    np.testing.assert_allclose(r2["grad"][4:], r["grad"][4:], rtol=1e-13)


def test_empty_cluster_masked_pixels_and_regions(model, c1):
    d, idx, K = _entry(c1)
    # an extra, empty cluster per parameter gets gradient exactly 0 and changes nothing else (R9)
    K2 = [K[0] + 1, K[1] + 1, K[2] + 1]
    p = c1.params_jittered(4)
    p2 = np.concatenate([p[:4], [9.9], p[4:6], [33.0], p[6:], [-1.5]])
    r = oracle.nll_grad(model, d, c1.ninv, idx, K, p, want_maps=True)
    r2 = oracle.nll_grad(model, d, c1.ninv, idx, K2, p2)
    assert r2["grad"][4] == 0.0 and r2["grad"][7] == 0.0 and r2["grad"][11] == 0.0
    np.testing.assert_array_equal(np.delete(r2["grad"], [4, 7, 11]), r["grad"])
    # masked pixels (id -1 in ANY map) are skipped everywhere, maps are 0 there (R7)
    idxm = idx.copy()
    idxm[0, 10:50] = -1; idxm[1, 40:90] = -1; idxm[2, 700:] = -1
    masked = (idxm < 0).any(0)
    rm = oracle.nll_grad(model, d, c1.ninv, idxm, K, p, want_maps=True)
    keep = np.flatnonzero(~masked)
    rk = oracle.nll_grad(model, np.ascontiguousarray(d[:, :, keep]), c1.ninv, idx[:, keep], K, p, want_maps=True)
    np.testing.assert_allclose(rm["nll"], rk["nll"], rtol=1e-14)
    np.testing.assert_allclose(rm["grad"], rk["grad"], rtol=1e-12, atol=1e-9)
    assert np.all(rm["maps"][:, :, masked] == 0.0)
    np.testing.assert_array_equal(rm["maps"][:, :, keep], rk["maps"])
    # regions: nll per region equals separate runs with the other regions masked (R10)
    reg = (np.arange(c1.npix) * 3 // c1.npix).astype(np.uint8)
    rr = oracle.nll_grad(model, d, c1.ninv, idx, K, p, region=reg, nregion=3)
    assert abs(rr["nll"].sum() - r["nll"][0]) < 1e-12 * abs(r["nll"][0])
    gsum = np.zeros_like(p)
    for q in range(3):
        iq = np.where(reg[None, :] == q, idx, -1).astype(np.int32)
        rq = oracle.nll_grad(model, d, c1.ninv, iq, K, p)
        assert abs(rq["nll"][0] - rr["nll"][q]) < 1e-13 * abs(rr["nll"][q])
        gsum += rq["grad"]
    np.testing.assert_allclose(gsum, rr["grad"], rtol=1e-11, atol=1e-9)


def test_error_returns(model, c1):
    d, idx, K = _entry(c1)
    p = c1.params_const()
    bad = p.copy(); bad[K[0]] = 0.0                                   # T_d <= 0
    assert oracle.nll_grad(model, d, c1.ninv, idx, K, bad)["rc"] == -3
    bad = p.copy(); bad[0] = np.nan
    assert oracle.nll_grad(model, d, c1.ninv, idx, K, bad)["rc"] == -3
    ib = idx.copy(); ib[1, 5] = K[1]
    assert oracle.nll_grad(model, d, c1.ninv, ib, K, p)["rc"] == -2
    ib = idx.copy(); ib[2, 5] = -2
    assert oracle.nll_grad(model, d, c1.ninv, ib, K, p)["rc"] == -2
    r = oracle.nll_grad(model, d, np.zeros(15, np.float32), idx, K, p)   # M = 0: singular (R11)
    assert r["rc"] == -1 and np.isinf(r["nll"][0])


# ----------------------------------------------------------------------------- whole path

def test_brute_force_grid_recovers_truth():
    # K=(1,1,1), noiseless nside-8 sky whose (uniform) truth lies on the grid => argmin = truth
    npix = 768
    truth = gen.draw_truth(npix, 11)
    truth["beta_d"][:] = 1.54; truth["T_d"][:] = 20.0; truth["beta_s"][:] = -3.0
    d = gen.synthesize(truth, gen.BANDS_GHZ, None, (0,))[0]
    ninv = gen.ninv_f32(8)
    m = oracle.Model(gen.BANDS_GHZ)
    idx = np.zeros((3, npix), dtype=np.int32)
    gb = np.linspace(1.34, 1.74, 11); gT = np.linspace(16.0, 24.0, 11); gs = np.linspace(-3.4, -2.6, 11)
    vals = np.empty((11, 11, 11))
    for i, b in enumerate(gb):
        for j, T in enumerate(gT):
            for k, s in enumerate(gs):
                vals[i, j, k] = oracle.nll_grad(m, d, ninv, idx, [1, 1, 1], np.array([b, T, s]), want_grad=False)["nll"][0]
    i, j, k = np.unravel_index(np.argmin(vals), vals.shape)
    assert (i, j, k) == (5, 5, 5)
    dNd = np.sum(ninv.astype(np.float64)[:, None, None] * d.astype(np.float64) ** 2)
    assert abs(vals[5, 5, 5] + 0.5 * dNd) < 1e-3                    # chi^2 ~ 0 (fp32 rounding of d only)
    assert np.sort(vals.ravel())[1] - vals[5, 5, 5] > 1.0           # unique, well separated minimum


# ----------------------------------------------------------------------------- tolerance scales absg / gscale (T2)
# Every gradient bound of the GPU parity tests is built from these two oracle outputs (tests/helpers.py check_T2), so
# a mistake in them would silently loosen every gradient check.  They are pinned to things other than themselves.

def _dA_numpy(freqs, bd, Td, bs, h=1e-6):
    """d a_d/d beta_d, d a_d/d T_d, d a_s/d beta_s [F] by central differences of gen's independent forward model."""
    ad_p, _ = gen.mixing_columns(freqs, bd + h, Td, bs)
    ad_m, _ = gen.mixing_columns(freqs, bd - h, Td, bs)
    at_p, _ = gen.mixing_columns(freqs, bd, Td + h, bs)
    at_m, _ = gen.mixing_columns(freqs, bd, Td - h, bs)
    _, as_p = gen.mixing_columns(freqs, bd, Td, bs + h)
    _, as_m = gen.mixing_columns(freqs, bd, Td, bs - h)
    return np.stack([(ad_p - ad_m) / (2 * h), (at_p - at_m) / (2 * h), (as_p - as_m) / (2 * h)])


def test_gscale_of_one_pixel_against_a_numpy_restatement(model, c1):
    """gs_theta = sum_S |s_{S,c(theta)}| sum_f w_f |d_{S,f}| |da_f/dtheta|, restated with numpy
    from the definition: GLS solution by lstsq on gen's forward model, derivatives by central differences."""
    d, idx, K = _entry(c1)
    w = c1.ninv.astype(np.float64)
    comp_of = (1, 1, 2)
    for p, (bd, Td, bs) in ((3, (1.54, 20.0, -3.0)), (200, (1.7, 17.5, -2.8)), (767, (1.2, 31.0, -3.4))):
        dq, du = d[:, 0, p].astype(np.float64), d[:, 1, p].astype(np.float64)
        r = oracle.pixel(model, w, dq, du, bd, Td, bs)
        a_d, a_s = gen.mixing_columns(c1.freqs, bd, Td, bs)
        A = np.stack([np.ones_like(a_d), a_d, a_s], axis=1)
        sw = np.sqrt(w)
        s = np.stack([np.linalg.lstsq(A * sw[:, None], x * sw, rcond=None)[0] for x in (dq, du)], axis=1)   # [3, 2]
        dA = _dA_numpy(c1.freqs, bd, Td, bs)
        for t in range(3):
            want = sum(abs(s[comp_of[t], S]) * np.sum(w * np.abs(x) * np.abs(dA[t])) for S, x in enumerate((dq, du)))
            assert abs(r["gs"][t] - want) <= 2e-7 * want, (p, t, r["gs"][t], want)
            # and the gradient term itself, from the same restatement (Eq. 17, factor 1)
            g = -sum(s[comp_of[t], S] * np.sum(w * (x - A @ s[:, S]) * dA[t]) for S, x in enumerate((dq, du)))
            assert abs(r["g"][t] - g) <= 2e-6 * want


def test_absg_equals_abs_grad_when_every_pixel_is_its_own_cluster(model, c1):
    d, _, _ = _entry(c1)
    npix = c1.npix
    idx = np.tile(np.arange(npix, dtype=np.int32), (3, 1))
    params = np.concatenate([1.54 + 0.05 * np.sin(np.arange(npix)), 20.0 + np.cos(np.arange(npix)),
                             -3.0 + 0.05 * np.sin(0.3 * np.arange(npix))])
    r = oracle.nll_grad(model, d, c1.ninv, idx, [npix] * 3, params, want_tol=True)
    assert r["rc"] == 0
    assert np.array_equal(r["absg"], np.abs(r["grad"]))
    # per cluster = per pixel here: gscale is the one-pixel quantity pinned above
    w = c1.ninv.astype(np.float64)
    for p in (0, 411):
        one = oracle.pixel(model, w, d[:, 0, p].astype(np.float64), d[:, 1, p].astype(np.float64),
                           params[p], params[npix + p], params[2 * npix + p])
        assert np.allclose([r["gscale"][p], r["gscale"][npix + p], r["gscale"][2 * npix + p]], one["gs"], rtol=1e-14)


def test_absg_and_gscale_are_sums_over_the_clusters_pixels(model, c1):
    """absg_k = sum_{p in k} |g_p| and gscale_k = sum_{p in k} gs_p with the per-pixel terms of the K = npix run;
    hence absg >= |grad| (triangle inequality), with equality only without cancellation."""
    d, idx, K = _entry(c1)
    params = c1.params_jittered(seed=4)
    r = oracle.nll_grad(model, d, c1.ninv, idx, K, params, want_tol=True)
    npix = c1.npix
    own = np.tile(np.arange(npix, dtype=np.int32), (3, 1))
    pp = np.concatenate([params[:K[0]][idx[0]], params[K[0]:K[0] + K[1]][idx[1]], params[K[0] + K[1]:][idx[2]]])
    rp = oracle.nll_grad(model, d, c1.ninv, own, [npix] * 3, pp, want_tol=True)
    o = 0
    for t in range(3):
        gp, sp = rp["grad"][t * npix:(t + 1) * npix], rp["gscale"][t * npix:(t + 1) * npix]
        want_a = np.bincount(idx[t], weights=np.abs(gp), minlength=K[t])
        want_s = np.bincount(idx[t], weights=sp, minlength=K[t])
        assert np.allclose(r["absg"][o:o + K[t]], want_a, rtol=1e-12)
        assert np.allclose(r["gscale"][o:o + K[t]], want_s, rtol=1e-12)
        o += K[t]
    assert np.all(r["absg"] >= np.abs(r["grad"]) * (1 - 1e-12))
    assert np.all(r["gscale"] > 0)


def test_gscale_closed_form_on_noiseless_data_at_the_truth():
    """Noiseless cluster-constant sky at its true parameters: s = s*, d = A s*, the gradient vanishes but
    gscale_k = sum_{p in k} sum_S |s*_c| sum_f w_f |(A s*)_f| |da_f/dtheta| is a closed form of the inputs."""
    w = gen.make_config(0, noiseless=True, cluster_truth=True)
    model = oracle.Model(w.freqs)
    d, idx, K = _entry(w)
    truth = np.concatenate(w.truth["per_cluster"])
    r = oracle.nll_grad(model, d, w.ninv, idx, K, truth, want_tol=True)
    assert r["rc"] == 0
    wf = w.ninv.astype(np.float64)
    comp_of = (1, 1, 2)
    s = w.truth["s"]                                             # [3, 2, npix]
    gs = np.zeros((3, w.npix))
    for p in range(w.npix):
        dA = _dA_numpy(w.freqs, w.truth["beta_d"][p], w.truth["T_d"][p], w.truth["beta_s"][p])
        for t in range(3):
            gs[t, p] = sum(abs(s[comp_of[t], S, p]) * np.sum(wf * np.abs(d[:, S, p].astype(np.float64)) * np.abs(dA[t]))
                           for S in range(2))
    o = 0
    for t in range(3):
        want = np.bincount(idx[t], weights=gs[t], minlength=K[t])
        assert np.allclose(r["gscale"][o:o + K[t]], want, rtol=5e-6)     # fp32 rounding of d moves s by ~1e-7
        o += K[t]
    # the gradient is zero to the rounding of the fp32 data, many orders below the scale
    assert np.all(np.abs(r["grad"]) <= 1e-5 * r["gscale"])


def test_tolerance_scales_follow_the_scalings_of_the_gradient(model, c1):
    """Ninv -> c Ninv scales grad, absg and gscale by c; relabelling clusters permutes all three alike."""
    d, idx, K = _entry(c1)
    params = c1.params_jittered(seed=5)
    r1 = oracle.nll_grad(model, d, c1.ninv, idx, K, params, want_tol=True)
    r4 = oracle.nll_grad(model, d, (4.0 * c1.ninv).astype(np.float32), idx, K, params, want_tol=True)
    for key in ("grad", "absg", "gscale"):
        assert np.allclose(r4[key], 4.0 * r1[key], rtol=1e-13)
    perm = np.array([2, 0, 3, 1], dtype=np.int32)               # new label of old cluster k of the beta_d map
    idx2 = idx.copy()
    idx2[0] = perm[idx[0]]
    p2 = params.copy()
    p2[:K[0]][perm] = params[:K[0]]
    r2 = oracle.nll_grad(model, d, c1.ninv, idx2, K, p2, want_tol=True)
    for key in ("grad", "absg", "gscale"):
        assert np.allclose(r2[key][:K[0]][perm], r1[key][:K[0]], rtol=1e-13)
        assert np.allclose(r2[key][K[0]:], r1[key][K[0]:], rtol=1e-13)
