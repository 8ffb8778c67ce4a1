"""Test-side helpers: seeded inputs and Lorentz transformations (numpy).  No method arithmetic."""
import numpy as np


def mdot(a, b):
    return a[..., 0] * b[..., 0] - (a[..., 1:] * b[..., 1:]).sum(-1)


def random_lorentz(rng, beta_max=0.9):
    """A random proper orthochronous Lorentz transformation (rotation x boost) as a 4x4 matrix."""
    q, r = np.linalg.qr(rng.normal(size=(3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    R = np.eye(4)
    R[1:, 1:] = q
    n = rng.normal(size=3)
    n /= np.linalg.norm(n)
    beta = beta_max * rng.uniform()
    g = 1.0 / np.sqrt(1 - beta * beta)
    B = np.eye(4)
    B[0, 0] = g
    B[0, 1:] = B[1:, 0] = g * beta * n
    B[1:, 1:] += (g - 1) * np.outer(n, n)
    return B @ R


def transform(momenta, L):
    return np.einsum("mn,...n->...m", L, momenta)


def closed_form_epem_mupmum(mom, alpha_em):
    """(1/4) sum |M|^2 = 2 e^4 (t^2+u^2)/s^2  — BASELINE.json:configs[0], SURVEY.md §8(c) I."""
    s = mdot(mom[:, 0] + mom[:, 1], mom[:, 0] + mom[:, 1])
    t = mdot(mom[:, 0] - mom[:, 2], mom[:, 0] - mom[:, 2])
    u = mdot(mom[:, 0] - mom[:, 3], mom[:, 0] - mom[:, 3])
    e2 = 4 * np.pi * alpha_em
    return 2 * e2 ** 2 * (t ** 2 + u ** 2) / s ** 2


def closed_form_gg_ttx(mom, alpha_s, m):
    """g_s^4 [1/(6 tau1 tau2) - 3/8][tau1^2 + tau2^2 + rho - rho^2/(4 tau1 tau2)], spin/colour averaged —
    the textbook heavy-quark hadroproduction formula quoted in SURVEY.md §8(c) I (config 1)."""
    s = mdot(mom[:, 0] + mom[:, 1], mom[:, 0] + mom[:, 1])
    t = mdot(mom[:, 0] - mom[:, 2], mom[:, 0] - mom[:, 2])
    u = mdot(mom[:, 0] - mom[:, 3], mom[:, 0] - mom[:, 3])
    gs2 = 4 * np.pi * alpha_s
    t1, t2, rho = (m * m - t) / s, (m * m - u) / s, 4 * m * m / s
    return gs2 ** 2 * (1 / (6 * t1 * t2) - 3.0 / 8) * (t1 ** 2 + t2 ** 2 + rho - rho ** 2 / (4 * t1 * t2))


def momentum_violation(mom):
    """delta = max |sum k| / sqrt(s) of each event's own input.  |M|^2 is only defined on momentum-conserving on-shell
    input; the cancellation-free RAMBO boost (DESIGN.md R-G1b) keeps delta below 1e-12 on every event, so the
    1e-10 tolerance of BASELINE.json:north_star applies to every event without exception (tests assert both)."""
    tot = mom[:, :2].sum(1) - mom[:, 2:].sum(1)
    return np.abs(tot).max(1) / (mom[:, 0, 0] + mom[:, 1, 0])
