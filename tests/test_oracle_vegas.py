"""Pins for the oracle's Vegas pieces (SURVEY.md §8(c) G7 'Pins'): closed-form integrals, fixed end points,
alpha = 0 fixed point, <jac> = 1, quantile convergence.  The grid-update details (alpha = 1.5, 3-point smoothing)
are a READING of Lepage's algorithm (DESIGN.md R-G7), not fixed by the paper.  CPU only."""
import math

import numpy as np

from oracle import ref


def run_vegas(f, D, n_it, n_ev, alpha=1.5, nb=50, seed=4):
    edges = np.tile(np.linspace(0, 1, nb + 1), (D, 1))
    res = []
    for it in range(n_it):
        y = ref.philox_uniform(seed, it, 0, D, n_ev)
        x, jac, idx = ref.vegas_map(edges, y)
        fv = jac * f(x)
        sums = ref.vegas_accumulate(fv, idx, nb)
        I = sums[0] / n_ev
        var = (sums[1] / n_ev - I * I) / (n_ev - 1)
        res.append((I, var))
        edges = ref.vegas_refine(edges, sums[3:], alpha)
    return edges, res


def test_map_uniform_grid_is_identity():
    edges = np.tile(np.linspace(0, 1, 51), (3, 1))
    y = ref.philox_uniform(1, 0, 0, 3, 1000)
    x, jac, idx = ref.vegas_map(edges, y)
    assert np.max(np.abs(x - y)) < 1e-15 and np.max(np.abs(jac - 1)) < 1e-13
    assert np.array_equal(idx, np.minimum((y * 50).astype(int), 49))


def test_jacobian_averages_to_one_and_integral_of_one():
    """On any grid, int jac dy = 1 exactly per dimension: sample mean -> 1; integrand 1 integrates to 1."""
    rng = np.random.default_rng(0)
    e = np.sort(rng.uniform(size=(4, 49)), axis=1)
    edges = np.concatenate([np.zeros((4, 1)), e, np.ones((4, 1))], 1)
    y = ref.philox_uniform(2, 0, 0, 4, 400000)
    x, jac, idx = ref.vegas_map(edges, y)
    assert abs(jac.mean() - 1) < 5 * jac.std() / math.sqrt(len(jac))
    assert x.min() >= 0 and x.max() <= 1
    # x lies in the bin it claims
    for d in range(4):
        assert np.all(x[:, d] >= edges[d, idx[:, d]] - 1e-15) and np.all(x[:, d] <= edges[d, idx[:, d] + 1] + 1e-15)


def test_alpha_zero_is_a_fixed_point_and_endpoints_stay():
    f = lambda x: np.exp(-50 * ((x - 0.3) ** 2).sum(1))
    edges, _ = run_vegas(f, 2, 2, 20000, alpha=0.0)
    assert np.max(np.abs(edges - np.linspace(0, 1, 51))) < 1e-13
    edges, _ = run_vegas(f, 2, 4, 20000, alpha=1.5)
    assert np.all(edges[:, 0] == 0) and np.all(edges[:, -1] == 1)
    assert np.all(np.diff(edges, axis=1) > 0)


def test_separable_gaussian_closed_form():
    """int over [0,1]^4 of prod_d exp(-(x_d-mu)^2/(2 s^2)) = [s sqrt(2 pi) (Phi((1-mu)/s) - Phi(-mu/s))]^4."""
    mu, s, D = 0.4, 0.05, 4
    f = lambda x: np.exp(-((x - mu) ** 2).sum(1) / (2 * s * s))
    one = s * math.sqrt(2 * math.pi) * 0.5 * (math.erf((1 - mu) / s / math.sqrt(2)) - math.erf(-mu / s / math.sqrt(2)))
    exact = one ** D
    edges, res = run_vegas(f, D, 6, 40000)
    I = np.array([r[0] for r in res])
    var = np.array([r[1] for r in res])
    # each iteration is unbiased; adaptation shrinks the error by a large factor
    for Ij, vj in zip(I, var):
        assert abs(Ij - exact) < 5 * math.sqrt(vj)
    assert var[-1] < var[0] / 50
    comb = (I / var).sum() / (1 / var).sum()
    assert abs(comb - exact) < 5 * (1 / var).sum() ** -0.5


def test_edges_converge_to_quantiles_in_1d():
    """With alpha = 1 repeated refinement puts equal sum f^2 ... in 1-D for f ∝ density p the optimal Vegas grid
    equalises int |f| per bin; check the adapted grid's median edge against the |f|-quantile within a bin width."""
    f = lambda x: 3 * x[:, 0] ** 2
    edges, res = run_vegas(f, 1, 12, 100000, alpha=1.0, nb=50)
    # CDF of |f| is x^3 -> median at 0.5^(1/3)
    med = edges[0, 25]
    assert abs(med - 0.5 ** (1 / 3)) < 0.03
    assert abs(edges[0, 5] - 0.1 ** (1 / 3)) < 0.06
    I = res[-1][0]
    assert abs(I - 1) < 5 * math.sqrt(res[-1][1])
    assert res[-1][1] < res[0][1] / 20


def test_refine_hand_case():
    """Two bins, alpha = 1, S = (1, 3): smoothing gives s = (2, 2) -> weights equal -> edge stays at 0.5.
    Three bins, S = (0, 0, 6), alpha = 1: s = (0, 2, 3), r = (0, .4, .6), w = (0, (r-1)/ln r ...) by hand."""
    e = ref.vegas_refine(np.array([[0, 0.5, 1.0]]), np.array([[1.0, 3.0]]), 1.0)
    assert np.allclose(e, [[0, 0.5, 1.0]])
    S = np.array([[0.0, 0.0, 6.0]])
    e0 = np.array([[0, 1 / 3, 2 / 3, 1.0]])
    e = ref.vegas_refine(e0, S, 1.0)[0]
    r = np.array([0.0, 0.4, 0.6])
    w = np.array([0.0, (0.4 - 1) / math.log(0.4), (0.6 - 1) / math.log(0.6)])
    tgt = w.sum() / 3
    # new edge 1 at cumulative tgt: inside old bin 1 (bin 0 has zero weight)
    want1 = 1 / 3 + (tgt / w[1]) / 3
    want2 = (1 / 3 + (2 * tgt / w[1]) / 3) if 2 * tgt <= w[1] else (2 / 3 + ((2 * tgt - w[1]) / w[2]) / 3)
    assert abs(e[1] - want1) < 1e-14 and abs(e[2] - want2) < 1e-14 and e[0] == 0 and e[3] == 1


import pytest  # noqa: E402


@pytest.mark.parametrize("proc", ["gg_ttxgg", "qg_ttxqg", "qqx_ttxgg"])
def test_hadronic_mode_factorises_into_pinned_pieces(proc):
    """The beams of the quark-initiated channels (N1 x N3) carry their own DECLARED toy densities: quark
    2 x^-0.5 (1-x)^3, antiquark 0.3 x^-1.1 (1-x)^7 (checked by hand at x = 1/4).
    ps_mode 2 (DESIGN.md R-N3): f = jac g(x1) g(x2) x [the partonic integrand at sqrt(s_hat) =
    sqrt(x1 x2 S)].  Every factor on the right is produced by an already pinned routine called separately (vegas_map,
    rambo_generate in diet mode at sqrt(s_hat), cuts, tier-1 |M|^2); the toy density 3 x^-1.2 (1-x)^5 is the declared
    reading, checked at x = 1/4 where it is 3 * 4^1.2 * (3/4)^5 by hand.  Also: events below threshold give exactly 0."""
    import numpy as np
    from oracle import ref
    from paper_2211_14056_b200.workloads import PARAMS
    n, S = 400, 13000.0
    rng = np.random.default_rng(3)
    g = ref.GridRef(10, 50, 1.5, seed=9, ps_mode=2)
    e = np.sort(rng.uniform(size=(10, 51)), axis=1)
    e[:, 0], e[:, -1] = 0.0, 1.0
    g.edges[:] = e
    me = ref.MatrixElementRef(proc)
    sums, f = me.vegas_integrand(g, S, 5, n, want_f=True)
    y = ref.philox_uniform(9, 0, 5, 10, n)
    x, jac, idx = ref.vegas_map(e, y)
    glu = lambda t: 3.0 * t ** -1.2 * (1.0 - t) ** 5
    qrk = lambda t: 2.0 * t ** -0.5 * (1.0 - t) ** 3
    aqk = lambda t: 0.3 * t ** -1.1 * (1.0 - t) ** 7
    assert abs(glu(0.25) - 3 * 4 ** 1.2 * 0.75 ** 5) < 1e-12 and abs(qrk(0.25) - 2 * 2 * 0.75 ** 3) < 1e-12
    assert abs(aqk(0.25) - 0.3 * 4 ** 1.1 * 0.75 ** 7) < 1e-12
    dens1, dens2 = {"gg_ttxgg": (glu, glu), "qg_ttxqg": (qrk, glu), "qqx_ttxgg": (qrk, aqk)}[proc]
    masses = (173.0, 173.0, 0.0, 0.0)
    want = np.zeros(n)
    for i in range(n):
        rs = np.sqrt(x[i, 0] * x[i, 1]) * S
        if rs <= sum(masses):
            continue
        mom, w = ref.rambo_generate(x[i:i + 1, 2:], rs, masses, 1)
        if ref.cuts(mom, (0, 0, 1, 1), PARAMS["ptj_min"], PARAMS["dr_min"])[0]:
            want[i] = jac[i] * dens1(x[i, 0]) * dens2(x[i, 1]) * w[0] * me.eval(mom)[0] / (2 * rs * rs) * 0.3893793721e9
    assert np.array_equal(f != 0, want != 0) and (want == 0).any() and (want != 0).sum() > 100
    nz = want != 0
    assert np.max(np.abs(f[nz] / want[nz] - 1)) < 1e-12
    assert abs(sums[0] / f.sum() - 1) < 1e-12 and sums[2] == nz.sum()


# ---- the physics integrand and the iteration driver ------------------------------
def _sigma_gg_ttx_quadrature(sqrt_s, m, alpha_s, n_nodes=96):
    """sigma(gg -> t tbar) at fixed sqrt(s_hat) from pieces pinned elsewhere: the closed-form |M|^2 of config 1
    (tests/helpers.py, pinned against the definition tier in test_oracle_me.py) integrated over the two-body phase
    space d Phi_2 = beta/(16 pi) d cos(theta) (total beta/(8 pi): test_rambo_two_body_massive_weight) times the
    flux 1/(2 s_hat) and the conversion 0.3893793721e9 pb GeV^2."""
    from tests.helpers import closed_form_gg_ttx
    s = sqrt_s * sqrt_s
    beta = math.sqrt(1 - 4 * m * m / s)
    c, wq = np.polynomial.legendre.leggauss(n_nodes)
    e, p = sqrt_s / 2, beta * sqrt_s / 2
    st = np.sqrt(1 - c * c)
    mom = np.zeros((n_nodes, 4, 4))
    mom[:, 0] = [e, 0, 0, e]
    mom[:, 1] = [e, 0, 0, -e]
    mom[:, 2, 0], mom[:, 2, 1], mom[:, 2, 3] = e, p * st, p * c
    mom[:, 3, 0], mom[:, 3, 1], mom[:, 3, 3] = e, -p * st, -p * c
    integral = (wq * closed_form_gg_ttx(mom, alpha_s, m)).sum()
    return 0.3893793721e9 / (2 * s) * beta / (16 * math.pi) * integral


def test_total_cross_section_gg_ttx_pins_the_integrand_normalisation():
    """Pins flux 1/(2 s_hat), W_ps, jac, the conversion constant and |M|^2 TOGETHER through vegas_iterate_ref itself
    (VERDICT r1 'parity unpinned' item): sigma(gg -> t tbar, sqrt(s_hat) = 1 TeV, no cuts) from three oracle Vegas
    iterations (classic RAMBO, D = 8) against the 1-D quadrature above; the textbook total cross section
    pi alpha_s^2/(3 s)[(1 + rho + rho^2/16) ln((1+beta)/(1-beta)) - beta (7/4 + 31 rho/16)] is a second, independent
    check of the quadrature (it is verified here, not trusted)."""
    from paper_2211_14056_b200.workloads import PARAMS
    rs, m, a_s = 1000.0, PARAMS["m_top"], PARAMS["alpha_s"]
    quad = _sigma_gg_ttx_quadrature(rs, m, a_s)
    assert abs(_sigma_gg_ttx_quadrature(rs, m, a_s, 48) / quad - 1) < 1e-12      # the quadrature has converged
    s = rs * rs
    rho, beta = 4 * m * m / s, math.sqrt(1 - 4 * m * m / s)
    book = math.pi * a_s ** 2 / (3 * s) * ((1 + rho + rho ** 2 / 16) * math.log((1 + beta) / (1 - beta))
                                           - beta * (7 / 4 + 31 * rho / 16)) * 0.3893793721e9
    assert abs(book / quad - 1) < 1e-10
    me = ref.MatrixElementRef("gg_ttx")
    g = ref.GridRef(8, 50, 1.5, seed=11, ps_mode=0)
    res = [me.vegas_iterate(g, rs, 150000) for _ in range(3)]
    I = np.array([r["integral"] for r in res])
    var = np.array([r["variance"] for r in res])
    for Ij, vj in zip(I, var):      # every iteration is an unbiased estimate
        assert abs(Ij - quad) < 4.5 * math.sqrt(vj)
    comb, sig = (I / var).sum() / (1 / var).sum(), (1 / var).sum() ** -0.5
    assert sig / comb < 3e-3 and abs(comb - quad) < 4 * sig
    assert all(r["n_pass"] == 150000 for r in res)      # no cuts: every event contributes
    # a wrong flux (1/(2 sqrt(s)), 1/s, 1/(4 s)), a dropped 2 pi or a missing conversion would be off by >= 2x
    assert abs(comb / quad - 1) < 0.01


def test_vegas_iterate_ref_by_hand():
    """vegas_iterate_ref itself: I = (1/N) sum f, sigma^2 = [(1/N) sum f^2 - I^2]/(N-1)
    recomputed by hand from the per-event f of the same iteration (vegas_integrand_ref, pinned above), the grid
    refined with exactly the accumulated S_{d,i}, the iteration counter advanced (so the next call draws new points)."""
    me = ref.MatrixElementRef("gg_ttx")
    for n in (2, 7, 1000):
        g = ref.GridRef(8, 50, 1.5, seed=5, ps_mode=0)
        g2 = ref.GridRef(8, 50, 1.5, seed=5, ps_mode=0)
        sums, f = me.vegas_integrand(g2, 1000.0, 0, n, want_f=True)
        r = me.vegas_iterate(g, 1000.0, n)
        I = math.fsum(f) / n
        var = (math.fsum(f * f) / n - I * I) / (n - 1)
        assert abs(r["integral"] / I - 1) < 1e-14 and abs(r["variance"] / var - 1) < 1e-10 * max(1, I * I / (var * n))
        assert abs(r["sum_w"] / math.fsum(f) - 1) < 1e-14 and abs(r["sum_w2"] / math.fsum(f * f) - 1) < 1e-14
        assert r["n_pass"] == n and g.iteration == 1 and g2.iteration == 0
        want_edges = ref.vegas_refine(g2.edges, sums[3:].reshape(8, 50), 1.5)
        assert np.array_equal(g.edges, want_edges)
        # the second iteration uses the refined grid and a new random stream
        r2 = me.vegas_iterate(g, 1000.0, n)
        assert g.iteration == 2 and r2["integral"] != r["integral"]


# ---- unweighted events ------------------------------------------------------------------------
def test_unweighting_is_hit_or_miss_with_its_own_random_stream():
    """Pins of vegas_unweight_ref: the uniform comes from Philox counter (event, 0x7fffffff, iteration) — recomputed here
    from the pinned raw Philox —, the decision is u w_max < f, the accepted list is ascending and reproducible under
    sharding, overweight events are always kept and counted, and the acceptance rate is <f>/w_max within its binomial
    error (so the kept events carry unit weight)."""
    rng = np.random.default_rng(5)
    n = 40000
    f = rng.exponential(1.0, n) * (rng.uniform(size=n) < 0.8)        # 20 % cut events with f = 0
    w_max = 6.0
    acc, n_over = ref.vegas_unweight(f, w_max, seed=4, iteration=3, first_event=1000)
    assert n_over == int((f > w_max).sum()) and n_over > 0
    assert np.all(np.diff(acc) > 0) and acc.min() >= 1000 and acc.max() < 1000 + n
    keep = np.zeros(n, bool)
    keep[acc - 1000] = True
    assert not keep[f == 0].any() and keep[f > w_max].all()
    for e in list(range(0, 200)) + [n - 1]:                           # the decision, event by event, from raw Philox
        o = ref.philox_raw([(1000 + e) & 0xffffffff, (1000 + e) >> 32, 0x7fffffff, 3], [4, 0])
        u = (((int(o[0]) << 32 | int(o[1])) >> 11) + 0.5) / 2 ** 53
        assert keep[e] == (f[e] > 0 and u * w_max < f[e])
    p = np.minimum(f / w_max, 1.0)
    assert abs(keep.sum() - p.sum()) < 5 * math.sqrt((p * (1 - p)).sum())
    # sharding: two halves with their own first_event give the same list
    a1, _ = ref.vegas_unweight(f[:n // 2], w_max, 4, 3, 1000)
    a2, _ = ref.vegas_unweight(f[n // 2:], w_max, 4, 3, 1000 + n // 2)
    assert np.array_equal(np.concatenate([a1, a2]), acc)
    # another iteration or seed decides differently; the phase-space uniforms of the event do not enter
    assert not np.array_equal(ref.vegas_unweight(f, w_max, 4, 2, 1000)[0], acc)
    assert not np.array_equal(ref.vegas_unweight(f, w_max, 5, 3, 1000)[0], acc)


def test_generate_reproduces_the_integrand_kinematics():
    """vegas_generate_ref(ids) gives the momenta and the |M|^2-free weight of exactly the events vegas_integrand_ref
    integrates: f_e = weight_e x Theta_e x me2(momenta_e) with the pinned cuts and tier-1 |M|^2 called separately."""
    from paper_2211_14056_b200.workloads import PARAMS
    me = ref.MatrixElementRef("gg_ttxg")
    g = ref.GridRef(5, 50, 1.5, seed=8, ps_mode=1)
    rng = np.random.default_rng(1)
    e = np.sort(rng.uniform(size=(5, 51)), axis=1)
    e[:, 0], e[:, -1] = 0.0, 1.0
    g.edges[:] = e
    n = 300
    sums, f = me.vegas_integrand(g, 1000.0, 40, n, want_f=True)
    ids = np.arange(40, 40 + n)[::-1].copy()                           # any order, any subset
    mom, w = me.vegas_generate(g, 1000.0, ids)
    ok = ref.cuts(mom, (0, 0, 1), PARAMS["ptj_min"], PARAMS["dr_min"]).astype(bool)
    want = np.where(ok, w * me.eval(mom), 0.0)[::-1]
    nz = want != 0
    assert np.array_equal(nz, f != 0) and nz.sum() > 100
    assert np.max(np.abs(f[nz] / want[nz] - 1)) < 1e-12
