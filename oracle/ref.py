"""ORACLE — TEST INFRASTRUCTURE ONLY.

ctypes loader for oracle/liboracle_ref.so (numpy host arrays in, numpy host arrays out).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module; the product package never does.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class MeParams(C.Structure):
    _fields_ = [("alpha_s", C.c_double), ("alpha_em", C.c_double), ("m_top", C.c_double), ("w_top", C.c_double),
                ("ptj_min", C.c_double), ("dr_min", C.c_double)]


class VegasGrid(C.Structure):
    _fields_ = [("n_dim", C.c_int), ("n_bins", C.c_int), ("edges", C.c_void_p), ("alpha", C.c_double),
                ("seed", C.c_uint64), ("iteration", C.c_int), ("ps_mode", C.c_int)]


class VegasResult(C.Structure):
    _fields_ = [("integral", C.c_double), ("variance", C.c_double), ("sum_w", C.c_double), ("sum_w2", C.c_double),
                ("n_pass", C.c_longlong)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.me_init_ref.argtypes = [C.c_char_p, C.POINTER(MeParams), C.POINTER(C.c_void_p)]
        _lib.me_free_ref.argtypes = [C.c_void_p]
        _lib.me_free_ref.restype = None
        for name in ("me_n_external_ref", "me_n_final_ref"):
            getattr(_lib, name).argtypes = [C.c_void_p]
        _lib.me_eval_ref.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong]
        _lib.me_eval_def_ref.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong]
        _lib.me_eval_diag_ref.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong]
        _lib.me_amplitude_diag_ref.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.me_set_basis_ref.argtypes = [C.c_void_p, C.c_int, C.c_int]
        _lib.me_set_ward_leg_ref.argtypes = [C.c_void_p, C.c_int]
        _lib.me_info_ref.argtypes = [C.c_void_p, C.c_int]
        _lib.me_colour_matrix_ref.argtypes = [C.c_void_p, C.c_void_p]
        _lib.me_flow_perms_ref.argtypes = [C.c_void_p, C.c_void_p]
        _lib.me_amplitude_def_ref.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.me_flows_ref.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.me_open_tensor_ref.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.su3_generators_ref.argtypes = [C.c_void_p, C.c_void_p]
        _lib.wavefunction_ref.argtypes = [C.c_int, C.c_void_p, C.c_double, C.c_int, C.c_int, C.c_void_p]
        _lib.philox_raw_ref.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.philox_uniform_ref.argtypes = [C.c_uint64, C.c_uint64, C.c_longlong, C.c_int, C.c_void_p, C.c_longlong]
        _lib.rambo_generate_ref.argtypes = [C.c_void_p, C.c_double, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                            C.c_longlong]
        _lib.cuts_ref.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_longlong]
        _lib.vegas_map_ref.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_longlong]
        _lib.vegas_accumulate_ref.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_longlong, C.c_void_p]
        _lib.vegas_refine_ref.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_double]
        _lib.vegas_integrand_ref.argtypes = [C.c_void_p, C.POINTER(VegasGrid), C.c_double, C.c_longlong, C.c_longlong,
                                             C.c_void_p, C.c_void_p]
        _lib.vegas_iterate_ref.argtypes = [C.c_void_p, C.POINTER(VegasGrid), C.c_double, C.c_longlong,
                                           C.POINTER(VegasResult)]
        _lib.vegas_unweight_ref.argtypes = [C.c_void_p, C.c_longlong, C.c_double, C.c_uint64, C.c_uint64, C.c_longlong,
                                            C.c_void_p, C.c_void_p]
        _lib.vegas_generate_ref.argtypes = [C.c_void_p, C.POINTER(VegasGrid), C.c_double, C.c_void_p, C.c_longlong,
                                            C.c_void_p, C.c_void_p]
        _lib.oracle_set_threads_ref.argtypes = [C.c_int]
        _lib.oracle_set_threads_ref.restype = None
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def set_threads(n):
    lib().oracle_set_threads_ref(int(n))


def get_threads():
    return int(lib().oracle_get_threads_ref())


DEFAULT_PARAMS = dict(alpha_s=0.118, alpha_em=1.0 / 132.507, m_top=173.0, w_top=0.0, ptj_min=20.0, dr_min=0.4)


class MatrixElementRef:
    """me_init_ref / me_eval_ref: tier-1 oracle (tier 0 via eval_def)."""

    def __init__(self, process, **params):
        p = dict(DEFAULT_PARAMS)
        p.update(params)
        self.params = MeParams(**p)
        self.process = process
        self._h = C.c_void_p()
        rc = lib().me_init_ref(process.encode(), C.byref(self.params), C.byref(self._h))
        if rc:
            raise ValueError(f"me_init_ref({process!r}) failed with {rc}")
        self.n_external = lib().me_n_external_ref(self._h)
        self.n_final = lib().me_n_final_ref(self._h)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.me_free_ref(self._h)
            self._h = None

    def _mom(self, momenta):
        m = _f64(momenta).reshape(-1, self.n_external, 4)
        return m, m.shape[0]

    def eval(self, momenta):
        m, n = self._mom(momenta)
        out = np.empty(n)
        rc = lib().me_eval_ref(self._h, _p(m), _p(out), n)
        assert rc == 0, rc
        return out

    def eval_def(self, momenta):
        m, n = self._mom(momenta)
        out = np.empty(n)
        rc = lib().me_eval_def_ref(self._h, _p(m), _p(out), n)
        assert rc == 0, rc
        return out

    def eval_diag(self, momenta):
        """tier 1 in the diagram basis (me_tier1g.cpp)"""
        m, n = self._mom(momenta)
        out = np.empty(n)
        rc = lib().me_eval_diag_ref(self._h, _p(m), _p(out), n)
        assert rc == 0, rc
        return out

    def amplitude_diag(self, mom, hel, col):
        m = _f64(mom).reshape(self.n_external, 4)
        hel = np.ascontiguousarray(hel, dtype=np.int32)
        col = np.ascontiguousarray(col, dtype=np.int32)
        out = np.empty(2)
        assert lib().me_amplitude_diag_ref(self._h, _p(m), _p(hel), _p(col), _p(out)) == 0
        return complex(out[0], out[1])

    def info_diag(self):
        return dict(n_diag=lib().me_info_ref(self._h, 5), n_terms=lib().me_info_ref(self._h, 6),
                    n_diag_4g=lib().me_info_ref(self._h, 7))

    def set_basis(self, spin_basis, pol_basis):
        lib().me_set_basis_ref(self._h, spin_basis, pol_basis)

    def set_ward_leg(self, leg):
        lib().me_set_ward_leg_ref(self._h, leg)

    def info(self):
        return dict(n_diag=lib().me_info_ref(self._h, 0), n_terms=lib().me_info_ref(self._h, 1),
                    n_diag_4g=lib().me_info_ref(self._h, 2), n_flow=lib().me_info_ref(self._h, 3),
                    n_gluon=lib().me_info_ref(self._h, 4))

    def colour_matrix(self):
        nf = self.info()["n_flow"]
        cf = np.empty((nf, nf))
        assert lib().me_colour_matrix_ref(self._h, _p(cf)) == 0
        return cf

    def flow_perms(self):
        i = self.info()
        perms = np.empty((i["n_flow"], i["n_gluon"]), dtype=np.int32)
        assert lib().me_flow_perms_ref(self._h, _p(perms)) == 0
        return perms

    def amplitude_def(self, mom, hel, col):
        m = _f64(mom).reshape(self.n_external, 4)
        hel = np.ascontiguousarray(hel, dtype=np.int32)
        col = np.ascontiguousarray(col, dtype=np.int32)
        out = np.empty(2)
        assert lib().me_amplitude_def_ref(self._h, _p(m), _p(hel), _p(col), _p(out)) == 0
        return complex(out[0], out[1])

    def open_tensor(self, k, col):
        """tier-0 amplitude with unit wavefunctions: complex array of shape (4,) * n_external, all-incoming momenta k"""
        k = _f64(k).reshape(self.n_external, 4)
        col = np.ascontiguousarray(col, dtype=np.int32)
        T = np.empty((4 ** self.n_external, 2))
        assert lib().me_open_tensor_ref(self._h, _p(k), _p(col), _p(T)) == 0
        return (T[:, 0] + 1j * T[:, 1]).reshape((4,) * self.n_external)

    def flows(self, mom, hel):
        m = _f64(mom).reshape(self.n_external, 4)
        hel = np.ascontiguousarray(hel, dtype=np.int32)
        J = np.empty((self.info()["n_flow"], 2))
        assert lib().me_flows_ref(self._h, _p(m), _p(hel), _p(J)) == 0
        return J[:, 0] + 1j * J[:, 1]

    # --- Vegas over this process ---
    def vegas_integrand(self, grid, sqrt_s, first_event, n_ev, want_f=False):
        sums = np.zeros(3 + grid.n_dim * grid.n_bins)
        f = np.empty(n_ev) if want_f else None
        rc = lib().vegas_integrand_ref(self._h, C.byref(grid.c), sqrt_s, first_event, n_ev, _p(sums),
                                       _p(f) if want_f else None)
        assert rc == 0, rc
        return (sums, f) if want_f else sums

    def vegas_generate(self, grid, sqrt_s, ids):
        ids = np.ascontiguousarray(ids, dtype=np.int64)
        mom = np.empty((len(ids), lib().me_n_external_ref(self._h), 4))
        w = np.empty(len(ids))
        rc = lib().vegas_generate_ref(self._h, C.byref(grid.c), sqrt_s, _p(ids), len(ids), _p(mom), _p(w))
        assert rc == 0, rc
        return mom, w

    def vegas_iterate(self, grid, sqrt_s, n_ev):
        res = VegasResult()
        rc = lib().vegas_iterate_ref(self._h, C.byref(grid.c), sqrt_s, n_ev, C.byref(res))
        assert rc == 0, rc
        return dict(integral=res.integral, variance=res.variance, sum_w=res.sum_w, sum_w2=res.sum_w2, n_pass=res.n_pass)


def vegas_unweight(f, w_max, seed, iteration, first_event=0):
    """Hit-or-miss: returns (accepted global event indices, ascending; number of f > w_max)."""
    f = _f64(f)
    acc = np.empty(len(f), dtype=np.int64)
    counts = np.zeros(2, dtype=np.int64)
    assert lib().vegas_unweight_ref(_p(f), len(f), float(w_max), seed, iteration, first_event, _p(acc), _p(counts)) == 0
    return acc[:counts[0]].copy(), int(counts[1])


class GridRef:
    """Host Vegas grid [n_dim][n_bins+1], uniform at start (BASELINE.json:configs[4])."""

    def __init__(self, n_dim, n_bins=50, alpha=1.5, seed=4, ps_mode=1):
        self.edges = np.tile(np.linspace(0.0, 1.0, n_bins + 1), (n_dim, 1)).copy()
        self.c = VegasGrid(n_dim, n_bins, self.edges.ctypes.data, alpha, seed, 0, ps_mode)

    n_dim = property(lambda s: s.c.n_dim)
    n_bins = property(lambda s: s.c.n_bins)
    iteration = property(lambda s: s.c.iteration)


def su3_generators():
    T = np.empty((8, 3, 3, 2))
    f = np.empty((8, 8, 8))
    lib().su3_generators_ref(_p(T), _p(f))
    return T[..., 0] + 1j * T[..., 1], f


def wavefunction(kind, p, mass, s, basis):
    out = np.empty(8)
    p = _f64(p)
    assert lib().wavefunction_ref({"u": 0, "v": 1, "eps": 2}[kind], _p(p), float(mass), int(s), int(basis), _p(out)) == 0
    return out[0::2] + 1j * out[1::2]


def philox_raw(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    o = np.empty(4, dtype=np.uint32)
    lib().philox_raw_ref(_p(c), _p(k), _p(o))
    return o


def philox_uniform(seed, iteration, first_event, n_dim, n_ev):
    out = np.empty((n_ev, n_dim))
    assert lib().philox_uniform_ref(seed, iteration, first_event, n_dim, _p(out), n_ev) == 0
    return out


def rambo_generate(rand, sqrt_s, masses, ps_mode=0):
    masses = _f64(masses)
    n = len(masses)
    nd = 4 * n if ps_mode == 0 else 3 * n - 4
    r = _f64(rand).reshape(-1, nd)
    mom = np.empty((r.shape[0], n + 2, 4))
    w = np.empty(r.shape[0])
    assert lib().rambo_generate_ref(_p(r), float(sqrt_s), _p(masses), n, ps_mode, _p(mom), _p(w), r.shape[0]) == 0
    return mom, w


def cuts(momenta, is_gluon, ptj_min, dr_min):
    isg = np.ascontiguousarray(is_gluon, dtype=np.int32)
    n = len(isg)
    m = _f64(momenta).reshape(-1, n + 2, 4)
    out = np.empty(m.shape[0], dtype=np.int32)
    assert lib().cuts_ref(_p(m), n, _p(isg), float(ptj_min), float(dr_min), _p(out), m.shape[0]) == 0
    return out


def vegas_map(edges, y):
    e = _f64(edges)
    D, nb = e.shape[0], e.shape[1] - 1
    y = _f64(y).reshape(-1, D)
    x = np.empty_like(y)
    jac = np.empty(y.shape[0])
    idx = np.empty(y.shape, dtype=np.int32)
    lib().vegas_map_ref(_p(e), D, nb, _p(y), _p(x), _p(jac), _p(idx), y.shape[0])
    return x, jac, idx


def vegas_accumulate(f, idx, n_bins):
    f = _f64(f)
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    D = idx.shape[1]
    sums = np.empty(3 + D * n_bins)
    lib().vegas_accumulate_ref(_p(f), _p(idx), D, n_bins, f.shape[0], _p(sums))
    return sums


def vegas_refine(edges, S, alpha):
    e = _f64(edges).copy()
    D, nb = e.shape[0], e.shape[1] - 1
    S = _f64(S).reshape(D, nb)
    lib().vegas_refine_ref(_p(e), D, nb, _p(S), float(alpha))
    return e
