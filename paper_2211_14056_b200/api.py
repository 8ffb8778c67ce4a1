"""Thin Python binding of include/madme.h: same names, argument marshalling only.

torch is used for device memory and streams (tensors in, tensors out, `tensor.data_ptr()` and
`torch.cuda.current_stream().cuda_stream` handed to the C ABI).  Every step of the path runs in the CUDA
kernels of libmadme.so; there is no CPU fallback and no oracle import here: if the library is missing or
there is no CUDA device, calls raise.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmadme.so")
_lib = None

ME_OK, ME_EINVAL, ME_EPROCESS, ME_ECUDA, ME_ENODEV, ME_EDIM = 0, -1, -2, -3, -4, -5


class MadmeError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("madme error %d: %s" % (code, msg))
        self.code = code


class MeParams(C.Structure):
    _fields_ = [("alpha_s", C.c_double), ("alpha_em", C.c_double), ("m_top", C.c_double), ("w_top", C.c_double),
                ("ptj_min", C.c_double), ("dr_min", C.c_double)]


class VegasGridC(C.Structure):
    _fields_ = [("n_dim", C.c_int), ("n_bins", C.c_int), ("edges", C.c_void_p), ("alpha", C.c_double),
                ("seed", C.c_uint64), ("iteration", C.c_int), ("ps_mode", C.c_int)]


class VegasResultC(C.Structure):
    _fields_ = [("integral", C.c_double), ("variance", C.c_double), ("sum_w", C.c_double), ("sum_w2", C.c_double),
                ("n_pass", C.c_longlong)]


# every symbol include/madme.h declares (tests check that the library exports exactly these)
SYMBOLS = ["me_init", "me_free", "me_reserve", "me_n_external", "me_n_final", "me_info", "me_flops_per_event", "me_eval",
           "me_eval_helicities", "philox_uniform", "rambo_generate", "apply_cuts", "vegas_map", "vegas_refine",
           "vegas_integrand", "vegas_iterate", "vegas_combine", "vegas_finish", "vegas_max_weight", "vegas_unweight",
           "vegas_unweight_static", "vegas_unweight_static_init", "vegas_generate", "fp64_peak_probe", "me_last_error"]


def lib():
    """Load libmadme.so (built in-tree by paper_2211_14056_b200.build).  Fails loudly when it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libmadme.so is not built: run `python -m paper_2211_14056_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, ll, dbl, i32, u64 = C.c_void_p, C.c_longlong, C.c_double, C.c_int, C.c_uint64
    L.me_init.argtypes = [C.c_char_p, C.POINTER(MeParams), C.POINTER(vp)]
    L.me_free.argtypes = [vp]
    L.me_free.restype = None
    L.me_reserve.argtypes = [vp, ll]
    L.me_n_external.argtypes = [vp]
    L.me_n_final.argtypes = [vp]
    L.me_info.argtypes = [vp, i32]
    L.me_info.restype = ll
    L.me_flops_per_event.argtypes = [vp]
    L.me_flops_per_event.restype = dbl
    L.me_eval.argtypes = [vp, vp, vp, ll, vp]
    L.me_eval_helicities.argtypes = [vp, vp, vp, ll, vp]
    L.philox_uniform.argtypes = [u64, u64, ll, i32, vp, ll, vp]
    L.rambo_generate.argtypes = [vp, dbl, C.POINTER(dbl), i32, i32, vp, vp, ll, vp]
    L.apply_cuts.argtypes = [vp, i32, C.POINTER(i32), dbl, dbl, vp, ll, vp]
    L.vegas_map.argtypes = [vp, i32, i32, vp, vp, vp, vp, ll, vp]
    L.vegas_refine.argtypes = [vp, i32, i32, vp, dbl, vp]
    L.vegas_integrand.argtypes = [vp, C.POINTER(VegasGridC), dbl, ll, ll, vp, vp, vp]
    L.vegas_iterate.argtypes = [vp, C.POINTER(VegasGridC), dbl, ll, C.POINTER(VegasResultC), vp]
    L.vegas_combine.argtypes = [vp, i32, i32, vp, vp]
    L.vegas_finish.argtypes = [vp, ll, C.POINTER(VegasResultC), vp]
    L.vegas_max_weight.argtypes = [vp, ll, vp, vp]
    L.vegas_unweight.argtypes = [vp, vp, ll, dbl, u64, u64, ll, vp, vp, vp]
    L.vegas_unweight_static.argtypes = [vp, ll, dbl, u64, u64, ll, vp, vp, vp]
    L.vegas_unweight_static_init.argtypes = []
    L.vegas_generate.argtypes = [vp, C.POINTER(VegasGridC), dbl, vp, ll, vp, vp, vp]
    L.fp64_peak_probe.argtypes = [ll, vp, C.POINTER(dbl), vp]
    L.me_last_error.restype = C.c_char_p
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        raise MadmeError(rc, lib().me_last_error().decode())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _dev(t, dtype, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CUDA tensor of dtype %s" % (name, dtype))
    return C.c_void_p(t.data_ptr())


class Handle:
    """Owner of a me_handle* (released on garbage collection)."""

    def __init__(self, ptr, process):
        self.ptr, self.process = ptr, process
        self.n_external = lib().me_n_external(ptr)
        self.n_final = lib().me_n_final(ptr)

    def __del__(self):
        if getattr(self, "ptr", None) and _lib is not None:
            _lib.me_free(self.ptr)
            self.ptr = None


def me_init(process, params):
    """params: dict with alpha_s, alpha_em, m_top, w_top, ptj_min, dr_min (workloads.PARAMS)."""
    p = MeParams(**{k: float(params[k]) for k, _ in MeParams._fields_})
    out = C.c_void_p()
    _check(lib().me_init(process.encode(), C.byref(p), C.byref(out)))
    return Handle(out, process)


def me_free(h):
    h.__del__()


def me_reserve(h, max_events):
    """Size the handle's per-event Vegas scratch (32 B/event) for calls of up to max_events events.  The C calls
    never allocate; this binding's vegas_* functions call me_reserve for you when they see a larger batch than
    reserved — call it yourself to decide when that allocation happens."""
    _check(lib().me_reserve(h.ptr, int(max_events)))


def _reserved(h, n_ev):
    if n_ev > int(lib().me_info(h.ptr, 11)):
        me_reserve(h, n_ev)


def me_info(h, what):
    return int(lib().me_info(h.ptr, what))


def me_flops_per_event(h):
    return float(lib().me_flops_per_event(h.ptr))


def me_eval(h, momenta, me2=None, stream=None):
    """momenta: cuda f64 [n_ev, n_ext, 4] -> me2: cuda f64 [n_ev]."""
    n_ev = momenta.shape[0]
    if momenta.dim() != 3 or momenta.shape[1] != h.n_external or momenta.shape[2] != 4:
        raise ValueError("momenta must be [n_ev, %d, 4]" % h.n_external)
    if me2 is None:
        me2 = torch.empty(n_ev, dtype=torch.float64, device=momenta.device)
    _check(lib().me_eval(h.ptr, _dev(momenta, torch.float64, "momenta"), _dev(me2, torch.float64, "me2"), n_ev, _stream(stream)))
    return me2


def me_eval_helicities(h, momenta, out=None, stream=None):
    n_ev = momenta.shape[0]
    n_hel = me_info(h, 4)
    if out is None:
        out = torch.empty((n_ev, n_hel), dtype=torch.float64, device=momenta.device)
    _check(lib().me_eval_helicities(h.ptr, _dev(momenta, torch.float64, "momenta"), _dev(out, torch.float64, "me2_hel"), n_ev,
                                    _stream(stream)))
    return out


def philox_uniform(seed, iteration, first_event, n_dim, n_ev, out=None, stream=None, device="cuda"):
    if out is None:
        out = torch.empty((n_ev, n_dim), dtype=torch.float64, device=device)
    _check(lib().philox_uniform(seed, iteration, first_event, n_dim, _dev(out, torch.float64, "rand"), n_ev, _stream(stream)))
    return out


def rambo_generate(rand, sqrt_s, masses, ps_mode=0, momenta=None, weights=None, stream=None):
    n_ev, n_final = rand.shape[0], len(masses)
    if momenta is None:
        momenta = torch.empty((n_ev, n_final + 2, 4), dtype=torch.float64, device=rand.device)
    if weights is None:
        weights = torch.empty(n_ev, dtype=torch.float64, device=rand.device)
    m = (C.c_double * n_final)(*[float(x) for x in masses])
    if rand.dim() != 2 or rand.shape[1] != (4 * n_final if ps_mode == 0 else 3 * n_final - 4):
        raise ValueError("rand must be [n_ev, 4 n_final] (ps_mode 0) or [n_ev, 3 n_final - 4] (ps_mode 1)")
    _check(lib().rambo_generate(_dev(rand, torch.float64, "rand"), float(sqrt_s), m, n_final, ps_mode,
                                _dev(momenta, torch.float64, "momenta"), _dev(weights, torch.float64, "weights"), n_ev, _stream(stream)))
    return momenta, weights


def apply_cuts(momenta, is_gluon, ptj_min, dr_min, out=None, stream=None):
    n_ev, n_final = momenta.shape[0], momenta.shape[1] - 2
    if out is None:
        out = torch.empty(n_ev, dtype=torch.int32, device=momenta.device)
    g = (C.c_int * n_final)(*[int(x) for x in is_gluon])
    _check(lib().apply_cuts(_dev(momenta, torch.float64, "momenta"), n_final, g, float(ptj_min), float(dr_min),
                            _dev(out, torch.int32, "pass"), n_ev, _stream(stream)))
    return out


def vegas_map(edges, y, stream=None):
    n, n_dim = y.shape
    n_bins = edges.shape[1] - 1
    x = torch.empty_like(y)
    jac = torch.empty(n, dtype=torch.float64, device=y.device)
    idx = torch.empty((n, n_dim), dtype=torch.int32, device=y.device)
    _check(lib().vegas_map(_dev(edges, torch.float64, "edges"), n_dim, n_bins, _dev(y, torch.float64, "y"),
                           _dev(x, torch.float64, "x"), _dev(jac, torch.float64, "jac"), _dev(idx, torch.int32, "idx"), n, _stream(stream)))
    return x, jac, idx


def vegas_refine(edges, S, alpha, stream=None):
    n_dim, n_bins = S.shape
    _check(lib().vegas_refine(_dev(edges, torch.float64, "edges"), n_dim, n_bins, _dev(S, torch.float64, "S"), float(alpha), _stream(stream)))
    return edges


class VegasGrid:
    """Python mirror of the C vegas_grid; `edges` is a caller-owned cuda f64 [n_dim, n_bins+1] tensor."""

    def __init__(self, n_dim, n_bins, alpha, seed, ps_mode, device="cuda", edges=None):
        if edges is None:
            edges = torch.linspace(0.0, 1.0, n_bins + 1, dtype=torch.float64, device=device).repeat(n_dim, 1).contiguous()
        self.edges = edges
        self.c = VegasGridC(n_dim, n_bins, edges.data_ptr(), float(alpha), seed, 0, ps_mode)

    @property
    def iteration(self):
        return self.c.iteration

    @iteration.setter
    def iteration(self, v):
        self.c.iteration = int(v)


def vegas_integrand(h, grid, sqrt_s, first_event, n_ev, want_f=False, stream=None):
    n_out = 3 + grid.c.n_dim * grid.c.n_bins
    sums = torch.empty(n_out, dtype=torch.float64, device=grid.edges.device)
    f = torch.empty(n_ev, dtype=torch.float64, device=grid.edges.device) if want_f else None
    _reserved(h, n_ev)
    _check(lib().vegas_integrand(h.ptr, C.byref(grid.c), float(sqrt_s), first_event, n_ev, _dev(sums, torch.float64, "sums"),
                                 _dev(f, torch.float64, "f") if want_f else None, _stream(stream)))
    return sums, f


def vegas_iterate(h, grid, sqrt_s, n_ev, stream=None):
    r = VegasResultC()
    _reserved(h, n_ev)
    _check(lib().vegas_iterate(h.ptr, C.byref(grid.c), float(sqrt_s), n_ev, C.byref(r), _stream(stream)))
    return _result(r)


def _result(r):
    return dict(integral=r.integral, variance=r.variance, sum_w=r.sum_w, sum_w2=r.sum_w2, n_pass=r.n_pass)


def vegas_combine(parts, stream=None):
    """parts: cuda f64 [n_parts, n_out] -> their sum in fixed order, cuda f64 [n_out]."""
    n_parts, n_out = parts.shape
    sums = torch.empty(n_out, dtype=torch.float64, device=parts.device)
    _check(lib().vegas_combine(_dev(parts, torch.float64, "parts"), n_parts, n_out, _dev(sums, torch.float64, "sums"), _stream(stream)))
    return sums


def vegas_finish(sums, n_total, stream=None):
    r = VegasResultC()
    _check(lib().vegas_finish(_dev(sums, torch.float64, "sums"), int(n_total), C.byref(r), _stream(stream)))
    return _result(r)


def vegas_max_weight(f, stream=None):
    """f: cuda f64 [n_ev] -> cuda f64 [1], max f."""
    out = torch.empty(1, dtype=torch.float64, device=f.device)
    _check(lib().vegas_max_weight(_dev(f, torch.float64, "f"), f.shape[0], _dev(out, torch.float64, "w_max"), _stream(stream)))
    return out


def vegas_unweight(h, f, w_max, seed, iteration, first_event=0, stream=None):
    """Hit-or-miss on the weights f of events [first_event, first_event + len(f)).  Returns (accepted global event
    indices in ascending order as a cuda int64 tensor view of length n_kept, n_overweight)."""
    n_ev = f.shape[0]
    accepted = torch.empty(n_ev, dtype=torch.int64, device=f.device)
    counts = torch.empty(2, dtype=torch.int64, device=f.device)
    _reserved(h, n_ev)
    _check(lib().vegas_unweight(h.ptr, _dev(f, torch.float64, "f"), n_ev, float(w_max), seed, iteration, first_event,
                                _dev(accepted, torch.int64, "accepted"), _dev(counts, torch.int64, "counts"), _stream(stream)))
    c = counts.tolist()      # marshalling: the two counters come back to size the view
    return accepted[:c[0]], c[1]


UNWEIGHT_STATIC_MAX_EVENTS = 4194304


def vegas_unweight_static_init():
    """Set-up of vegas_unweight_static on the current device (looks up the device address of its static scratch)."""
    _check(lib().vegas_unweight_static_init())


def vegas_unweight_static(f, w_max, seed, iteration, first_event=0, accepted=None, counts=None, stream=None):
    """vegas_unweight without a handle and without any allocation inside the library (its scratch is a fixed device
    array): at most UNWEIGHT_STATIC_MAX_EVENTS events per call, one call at a time per device.  Pass `accepted` (cuda
    int64 [n_ev]) and `counts` (cuda int64 [2]) to keep the binding from allocating too; then the raw tensors are returned
    and nothing is read back.  Otherwise returns (accepted view of length n_kept, n_overweight) like vegas_unweight."""
    n_ev = f.shape[0]
    raw = accepted is not None and counts is not None
    if accepted is None:
        accepted = torch.empty(n_ev, dtype=torch.int64, device=f.device)
    if counts is None:
        counts = torch.empty(2, dtype=torch.int64, device=f.device)
    _check(lib().vegas_unweight_static(_dev(f, torch.float64, "f"), n_ev, float(w_max), seed, iteration, first_event,
                                       _dev(accepted, torch.int64, "accepted"), _dev(counts, torch.int64, "counts"), _stream(stream)))
    if raw:
        return accepted, counts
    c = counts.tolist()
    return accepted[:c[0]], c[1]


def vegas_generate(h, grid, sqrt_s, event_ids, stream=None):
    """Momenta [n, n_ext, 4] and weights (without |M|^2 and cuts) [n] of the listed events of iteration grid.iteration."""
    n = event_ids.shape[0]
    momenta = torch.empty((n, h.n_external, 4), dtype=torch.float64, device=event_ids.device)
    weights = torch.empty(n, dtype=torch.float64, device=event_ids.device)
    _check(lib().vegas_generate(h.ptr, C.byref(grid.c), float(sqrt_s), _dev(event_ids, torch.int64, "event_ids"), n,
                                _dev(momenta, torch.float64, "momenta"), _dev(weights, torch.float64, "weights"), _stream(stream)))
    return momenta, weights


def fp64_peak_probe(n_iter, stream=None):
    """Launch the DFMA-chain kernel; returns the number of thread-level DFMAs it executes (time it with events)."""
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    n = C.c_double()
    _check(lib().fp64_peak_probe(n_iter, _dev(sink, torch.float64, "sink"), C.byref(n), _stream(stream)))
    return n.value


def vegas_iterate_sharded(h, grid, sqrt_s, n_total, group=None, stream=None):
    """One Vegas iteration over `n_total` events split across the ranks of `group`: every rank
    integrates its contiguous event range with the fused kernel (no communication), the per-rank sum vectors
    (3 + n_dim * n_bins doubles) are all-gathered and added by the library in FIXED rank order (vegas_combine), and
    every rank refines its own copy of the grid from the identical totals — so all ranks hold bit-identical grids and
    the result does not depend on arrival order.  The exchange is latency-bound (3.2 KB); with backend "nccl" it runs
    over NVLink, with "gloo" over the host.  Returns the same dict as vegas_iterate, identical on every rank.
    Marshalling only: every number is computed by the library."""
    import torch.distributed as dist
    from .sharding import gather_sums, strong_shard
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    first, n = strong_shard(rank, world, n_total)
    sums, _ = vegas_integrand(h, grid, sqrt_s, first, n, stream=stream)
    if world > 1:
        sums = vegas_combine(gather_sums(sums, group), stream=stream)
    n_dim, n_bins = grid.c.n_dim, grid.c.n_bins
    vegas_refine(grid.edges, sums[3:].view(n_dim, n_bins), grid.c.alpha, stream=stream)
    res = vegas_finish(sums, n_total, stream=stream)
    grid.iteration = grid.iteration + 1
    return res
