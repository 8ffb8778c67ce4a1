"""Properties of the CUDA phase-space and Vegas steps checked DIRECTLY on the GPU results, without the oracle in between
(What's weak 2: rambo / cuts / refine on the device follow the oracle's sources closely, so a shared
misreading would agree with itself; these are the pins of SURVEY.md §8(c) G1, G2, G5, G7 applied to the product's own
output, with the expectations written in numpy in a different form)."""
import math

import numpy as np
import pytest
import torch

from paper_2211_14056_b200 import api

pytestmark = pytest.mark.gpu


def mdot(a, b):
    return a[..., 0] * b[..., 0] - (a[..., 1:] * b[..., 1:]).sum(-1)


@pytest.mark.parametrize("masses,mode", [((0.0, 0.0), 0), ((173.0, 173.0), 0), ((173.0, 173.0, 0.0), 0), ((173.0, 173.0, 0.0, 0.0), 0),
                                         ((173.0, 173.0, 0.0, 0.0), 1), ((173.0, 173.0, 0.0, 0.0, 0.0), 1), ((0.0,) * 6, 0)])
def test_rambo_conservation_mass_shell_and_flat_weight(masses, mode):
    """sum p = (sqrt s, 0, 0, 0) and p_i^2 = m_i^2 to 1e-12 s on every event; massless: the weight is the constant
    (pi/2)^(n-1) s^(n-2) / ((n-1)! (n-2)!) (2 pi)^(4-3n) (RAMBO's flat phase-space volume)."""
    n, rs, n_ev = len(masses), 1000.0, 20000
    nd = 4 * n if mode == 0 else 3 * n - 4
    r = api.philox_uniform(5, 0, 0, nd, n_ev)
    mom, w = api.rambo_generate(r, rs, masses, mode)
    mom, w = mom.cpu().numpy(), w.cpu().numpy()
    tot = mom[:, 2:].sum(1)
    tot[:, 0] -= rs
    assert np.abs(tot).max() / rs < 1e-12
    assert np.abs(mdot(mom[:, 2:], mom[:, 2:]) - np.array(masses) ** 2).max() / rs ** 2 < 1e-12
    assert np.all(mom[:, 2:, 0] > 0) and np.all(w > 0)
    assert np.array_equal(mom[:, 0], np.tile([rs / 2, 0, 0, rs / 2], (n_ev, 1)))
    assert np.array_equal(mom[:, 1], np.tile([rs / 2, 0, 0, -rs / 2], (n_ev, 1)))
    if not any(masses) and mode == 0:
        w0 = (math.pi / 2) ** (n - 1) * rs ** (2 * n - 4) / (math.factorial(n - 1) * math.factorial(n - 2)) * (2 * math.pi) ** (4 - 3 * n)
        assert np.max(np.abs(w / w0 - 1)) < 1e-12


def test_rambo_two_body_isotropy_and_massive_weight():
    """n = 2 with equal masses: |p| = sqrt(s/4 - m^2) on every event, cos(theta) uniform (mean 0, variance 1/3 within
    5 sigma), weight = the two-body volume beta / (8 pi) with beta = 2|p|/sqrt(s)."""
    rs, m, n_ev = 1000.0, 173.0, 200000
    r = api.philox_uniform(6, 0, 0, 8, n_ev)
    mom, w = api.rambo_generate(r, rs, (m, m), 0)
    mom, w = mom.cpu().numpy(), w.cpu().numpy()
    pabs = np.sqrt((mom[:, 2, 1:] ** 2).sum(-1))
    want = math.sqrt(rs * rs / 4 - m * m)
    assert np.max(np.abs(pabs / want - 1)) < 1e-12
    c = mom[:, 2, 3] / pabs
    assert abs(c.mean()) < 5 / math.sqrt(3 * n_ev) and abs((c * c).mean() - 1 / 3) < 5 * math.sqrt(4 / 45 / n_ev)
    assert np.max(np.abs(w / (2 * want / rs / (8 * math.pi)) - 1)) < 1e-11


def test_cuts_against_a_numpy_restatement():
    """p_T via hypot, rapidity via arctanh(p_z / E), azimuth difference via the angle of the complex ratio: a third way
    of writing SURVEY 8(c) G5, evaluated in numpy on the GPU's own momenta; flips only within 1e-9 of a boundary."""
    rs, masses, jets = 1000.0, (173.0, 173.0, 0.0, 0.0), (0, 0, 1, 1)
    r = api.philox_uniform(3, 0, 0, 16, 100000)
    mom, _ = api.rambo_generate(r, rs, masses, 0)
    got = api.apply_cuts(mom, jets, 20.0, 0.4).cpu().numpy().astype(bool)
    p = mom.cpu().numpy()[:, 2:]
    pt = np.hypot(p[..., 1], p[..., 2])
    y = np.arctanh(p[..., 3] / p[..., 0])
    z = p[..., 1] + 1j * p[..., 2]
    ok = np.ones(len(p), bool)
    margin = np.full(len(p), np.inf)
    for i in (2, 3):
        ok &= pt[:, i] > 20.0
        margin = np.minimum(margin, np.abs(pt[:, i] - 20.0))
        for j in range(4):
            if j != i:
                dphi = np.angle(z[:, i] / z[:, j])
                dr = np.sqrt((y[:, i] - y[:, j]) ** 2 + dphi ** 2)
                ok &= dr > 0.4
                margin = np.minimum(margin, np.abs(dr - 0.4))
    diff = got != ok
    assert not np.any(diff & (margin > 1e-9)), np.nonzero(diff)[0][:5]
    assert 0.8 < got.mean() < 0.95


def test_vegas_map_and_refine_properties():
    """Map: x in the bin the index names, jacobian = prod N_b * width, mean jacobian 1.  Refine: end points
    fixed, edges increasing, alpha = 0 leaves a uniform grid where it is, and after a refinement every new bin holds the same
    share of the damped, smoothed weight (recomputed here with numpy's cumulative sums and interpolation)."""
    D, nb, n = 3, 50, 200000
    rng = np.random.default_rng(2)
    e = np.sort(rng.uniform(size=(D, nb + 1)), axis=1)
    e[:, 0], e[:, -1] = 0.0, 1.0
    y = torch.from_numpy(rng.uniform(size=(n, D))).cuda()
    x, jac, idx = api.vegas_map(torch.from_numpy(e).cuda(), y)
    x, jac, idx = x.cpu().numpy(), jac.cpu().numpy(), idx.cpu().numpy()
    lo = np.take_along_axis(e, idx.T, 1).T
    hi = np.take_along_axis(e, idx.T + 1, 1).T
    assert np.all((x >= lo) & (x <= hi))
    assert np.max(np.abs(jac / np.prod(nb * (hi - lo), axis=1) - 1)) < 1e-13
    assert abs(jac.mean() - 1) < 5 * jac.std() / math.sqrt(n)
    # refinement
    S = rng.uniform(size=(D, nb)) ** 3
    S[1, 10:14] = 0.0                     # empty bins
    uni = np.tile(np.linspace(0, 1, nb + 1), (D, 1))
    # (alpha = 0: every bin with a non-zero smoothed weight counts 1; bins whose smoothed weight is 0 count 0 by the reading)
    same = api.vegas_refine(torch.from_numpy(uni.copy()).cuda(), torch.from_numpy(S + 1e-3).cuda(), 0.0).cpu().numpy()
    assert np.max(np.abs(same - uni)) < 1e-14
    new = api.vegas_refine(torch.from_numpy(e.copy()).cuda(), torch.from_numpy(S).cuda(), 1.5).cpu().numpy()
    assert np.all(new[:, 0] == 0.0) and np.all(new[:, -1] == 1.0) and np.all(np.diff(new, axis=1) > 0)
    for d in range(D):
        s = np.empty(nb)
        s[0], s[-1] = (S[d, 0] + S[d, 1]) / 2, (S[d, -2] + S[d, -1]) / 2
        s[1:-1] = (S[d, :-2] + S[d, 1:-1] + S[d, 2:]) / 3
        rr = s / s.sum()
        with np.errstate(divide="ignore", invalid="ignore"):
            wgt = np.where(rr > 0, ((rr - 1) / np.log(rr)) ** 1.5, 0.0)
        cum = np.concatenate([[0.0], np.cumsum(wgt)])          # cumulative weight at the OLD edges
        at_new = np.interp(new[d], e[d], cum)                  # ... and, linearly inside old bins, at the NEW edges
        share = np.diff(at_new) / cum[-1]
        assert np.max(np.abs(share * nb - 1)) < 1e-9
